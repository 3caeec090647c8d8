// Grouped, batched, segment-accumulating FP64 GEMM on the DMMA pipe (sm_100a), operands staged by
// cp.async producer warps into an mbarrier-synchronised shared-memory ring (gemm.cu).
//
// One launch executes a list of output tiles of ONE tile shape.  Each output matrix C (M x N) is
//     C (+)= sum_{seg in segs(C)} sum_{r < seg.count} alpha_seg * op(A_seg[r]) * op(B_seg[r])
// which is the shape of every dense contraction on the DMRG hot path (Eq. (8), :109):
//   phase 1 of a task group : Z     = [O_L,0; O_L,1; ..] * Psi_in   (operators of a term group stacked
//                                                                    along M: "segmented rows")
//   phase 2 of an output    : Psi' += sum_r alpha Z_r * O_R,r^T      (segments accumulate in registers,
//                                                                    no global atomics)
//   renormalisation         : O'   += A2^T (O A1)
//   complementary operators : P     = W * [stacked normal operator blocks]
// All dimensions are multiples of 8 (blocks are stored zero-padded), so no edge predication
// inside an 8x8x4 mma tile is needed.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dmrg {

struct GSeg {
  const double* A;
  const double* B;
  long long rsA, rsB;   // per-repeat strides in elements (repeats accumulate into one output)
  long long bsA, bsB;   // per-batch strides in elements (batch elements are separate outputs)
  // segmented rows / columns: row m of op(A) lives in operator (m / amr) at A + (m / amr) * ams, local
  // row m % amr (amr == 0: plain matrix).  Same for the columns of op(B) with bnr / bns.
  long long ams, bns;
  int amr, bnr;
  unsigned amr_inv, bnr_inv;   // floor(2^32 / d) + 1 for the division by amr / bnr
  int lda, ldb;
  int K;                // multiple of 8
  int count;            // repeats accumulated into the same output
  int flags;            // bit0: A stored K x M (op(A) = A^T); bit1: B stored N x K (op(B) = B^T)
  int pad_;
  double alpha;
};

struct GOut {
  double* C;
  long long bsC;            // batch stride of C in elements
  int M, N, ldc;
  int seg_begin, seg_end;
  int accumulate;           // 1: C += acc, 0: C = acc
};

struct GTile {
  int out, batch, m0, n0;   // output index, batch index, first row / column of the tile
};

// Tile shapes (rows x cols of C per CTA).  Index = 3 * row_class + col_class, classes {32, 64, 128}.
constexpr int GEMM_NSHAPES = 9;
constexpr int GEMM_DIMS[3] = {32, 64, 128};
inline int gemm_shape_rows(int s) { return GEMM_DIMS[s / 3]; }
inline int gemm_shape_cols(int s) { return GEMM_DIMS[s % 3]; }

// Launch `ntiles` tiles of shape `shape` (device arrays); every CTA takes `tiles_per_cta` consecutive
// tiles of the list.  Returns the cudaError of the launch.
cudaError_t launch_grouped_gemm(int shape, const GOut* d_outs, const GSeg* d_segs, const GTile* d_tiles,
                                int ntiles, int tiles_per_cta, cudaStream_t stream);
int gemm_shape_ctas_per_sm(int shape);   // resident CTAs per SM the shape's kernel is built for
cudaError_t grouped_gemm_init();

}  // namespace dmrg
