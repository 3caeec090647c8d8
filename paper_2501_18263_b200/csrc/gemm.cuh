// Grouped, batched, segment-accumulating FP64 GEMM on the DMMA pipe (sm_100a).
//
// One launch executes a list of output tiles.  Each output matrix C (M x N) is
//     C (+)= sum_{seg in segs(C)} sum_{r < seg.count} alpha_seg * op(A_seg[r]) * op(B_seg[r])
// which is the shape of every dense contraction on the DMRG hot path (Eq. (8), :109):
//   phase 1 of a task group : Z_r   = O_L,r * Psi_in            (batch over r, one segment)
//   phase 2 of an output    : Psi' += sum_r alpha Z_r * O_R,r^T  (segments accumulate in registers,
//                                                                no global atomics)
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
  int tile_m, tile_n;       // tile extents, multiples of 8, <= 128
  int accumulate;           // 1: C += acc, 0: C = acc
};

struct GTile {
  int out, batch, tm, tn;   // output index, batch index, tile row / column index
};

constexpr int GEMM_BM = 128, GEMM_BN = 128, GEMM_KC = 16, GEMM_STAGES = 4, GEMM_THREADS = 256;
constexpr int GEMM_STAGE_DOUBLES = 2 * GEMM_BM * (GEMM_KC + 4);
constexpr int GEMM_SMEM_BYTES = GEMM_STAGES * GEMM_STAGE_DOUBLES * 8;

// Launch over `ntiles` tiles (device arrays).  Returns the cudaError of the launch.
cudaError_t launch_grouped_gemm(const GOut* d_outs, const GSeg* d_segs, const GTile* d_tiles,
                                int ntiles, cudaStream_t stream);
cudaError_t grouped_gemm_init();

}  // namespace dmrg
