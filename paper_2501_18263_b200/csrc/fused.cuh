// Fused two-step contraction for small sectors (sm_100a): one warp owns a 16-row strip of an output block of psi'
// (or of any "C += alpha X Y W" item whose dimensions all fit the tile class) and runs the whole task list of that
// block,
//     C += alpha * op(A_r) * op(P_r) * W_r        (Eq. (8), :109:  psi'{out} += c O_L psi{in} O_R^T)
// task by task, with the intermediate Z = op(A) op(P) kept in REGISTERS: the accumulator fragments of the first
// DMMA are turned into the A fragments of the second one by quad shuffles, so neither Z nor partial sums of C ever
// leave the SM (no workspace round trip, no second launch, no global atomics; fused.cu).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace dmrg {

struct FTask {
  const double* A;      // left factor of repeat 0, stored row-major; nullptr: two-matrix task C += alpha op(P) W
  const double* P;      // middle factor (the psi block); two-matrix tasks: the left factor
  const double* B;      // right factor W (ni x no logical)
  long long rsA, rsP, rsB;   // per-repeat strides in elements (repeats accumulate into the same C)
  int lda, ldp, ldb;
  int count;            // repeats
  short mi, ni;         // contraction extents: op(A) is (M x mi), op(P) is (mi x ni) [two-matrix: (M x ni)], W is (ni x N)
  short pad0_, pad1_;
  int flags;            // bit0: A stored transposed (mi x M); bit1: P stored transposed; bit2: W stored transposed (N x ni)
  int pad2_;
  double alpha;
};

struct FOut {
  double* C;
  int ldc, M, N;        // multiples of 8; N <= FUSED_MAX_N
  int task_begin, task_end;
  int accumulate;       // 1: C += result, 0: C = result (split parts write partial sums to scratch)
  int pad_;
};

constexpr int FUSED_NCLASSES = 8;     // class c: outputs with N = 8 (c + 1) columns
constexpr int FUSED_MAX_N = 8 * FUSED_NCLASSES;
constexpr int FUSED_STRIP = 16;       // rows of an output strip (one warp)

// One warp per entry of `items` = (output index, first row of its strip), heaviest first; cls = tile class.
cudaError_t launch_fused(int cls, const FOut* d_outs, const FTask* d_tasks, const int2* d_items, int nitems, cudaStream_t st);
int fused_warps_per_sm(int cls);   // resident warps per SM of the class's kernel

}  // namespace dmrg
