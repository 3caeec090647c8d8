// Fused small-sector kernel (fused.cuh).  One WARP owns a 16-row strip of an output block and runs the whole task
// list of that block on it.  For every task repeat and every pair of 8-column tiles of the intermediate Z:
//   step 1   Z(16 x 16)  = op(A)[strip, :] op(P)[:, 16 columns]        DMMA m8n8k4, 4 accumulator fragments
//   step 2   C(16 x N)  += alpha Z W[16 rows, :]                       accumulators of C live for the whole task list
// where the accumulator fragments of Z serve directly as the A fragments of step 2 (see fused_task),
// so the intermediate never exists outside a few registers.  Rows are independent in an MMA, so strips never
// exchange data: there is no shared memory, no barrier and no producer warp.  The MMA fragments are loaded straight
// from global memory through L1 (a quad reads 32 contiguous bytes of an A row, eight lanes read 64 contiguous bytes
// of a B row: whole 32-byte sectors either way); A[strip, :] is re-read from L1 once per pair of Z tiles.  The
// kernel is specialised on N / 8 (the number of 8-column accumulator tiles), which is fixed per output, so that the
// hot loops carry no predication; everything else (M, the contraction extents) is a runtime loop bound.
// Two earlier versions are recorded in DESIGN.md: whole operand blocks staged in shared memory through an mbarrier
// ring (two tasks in flight per SM: latency-bound, 3-4 TFLOP/s) and a fully unrolled register version whose
// predicated fragment arrays cost 24 instructions per DMMA (3.5 TFLOP/s).
#include "fused.cuh"

namespace dmrg {

namespace {

__device__ __forceinline__ void f_dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ double f_ld(const double* p) { return __ldg(p); }

enum : int { FT_TA = 1, FT_TP = 2, FT_TB = 4 };

constexpr int FUSED_WARPS = 4;     // independent warps per CTA (neighbouring strips: they share operands in L1)

__device__ __forceinline__ double2 f_ld2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }

// One task (all its repeats) on one strip.  TA: A stored transposed (mi x M); TB: W stored transposed (N x ni).
// Contraction indices are taken in the order the accumulator fragments hold them: within an 8-wide slab the first
// MMA k-step uses k = 2 lk, the second k = 2 lk + 1 (any pairing of the k of op(A) with the same k of op(B) gives the
// same sum).  A row-major A (not TA) and a transposed W (TB) — the stored forms of O_L and O_R in H_eff.psi — are
// then read with 16-byte loads, and the accumulator fragments of Z ARE the A fragments of step 2: no shuffle.
template <int NTN, bool TA, bool TB>
__device__ __forceinline__ void fused_task(double (&acc)[2][NTN][2], const FTask& tk, int rA, int rA1, int lr, int lk) {
  const int ldb = tk.ldb;
  // W fragment pair (k = k0 + 2 lk, k0 + 2 lk + 1; column 8 n + lr) at Br + offB + n * stepB (+ ldb for the second if !TB)
  const int offB = TB ? lr * ldb + 2 * lk : 2 * lk * ldb + lr;
  const int stepB = TB ? 8 * ldb : 8;
  const int slabB = TB ? 8 : 8 * ldb;           // advance of k0 by 8
  if (tk.A) {
    const int lda = tk.lda;
    const int sPk = (tk.flags & FT_TP) ? 1 : tk.ldp, sPn = (tk.flags & FT_TP) ? tk.ldp : 1;
    const int offA0 = TA ? 2 * lk * lda + rA : rA * lda + 2 * lk;
    const int offA1 = TA ? 2 * lk * lda + rA1 : rA1 * lda + 2 * lk;
    const int slabA = TA ? 8 * lda : 8;
    const int offP = 2 * lk * sPk + lr * sPn;
    const int ns = tk.mi >> 3, ntI = tk.ni >> 3;
    for (int r = 0; r < tk.count; ++r) {
      const double* Ar = tk.A + r * tk.rsA;
      const double* Pr = tk.P + r * tk.rsP + offP;
      const double* Br = tk.B + r * tk.rsB + offB;
      for (int j0 = 0; j0 < ntI; j0 += 2) {
        const bool two = j0 + 1 < ntI;
        // ---- step 1: two 8-column tiles of Z = op(A)[strip, :] op(P) ----
        double z[2][2][2] = {{{0.0, 0.0}, {0.0, 0.0}}, {{0.0, 0.0}, {0.0, 0.0}}};   // [row fragment][tile][element]
        const double* pa0 = Ar + offA0;
        const double* pa1 = Ar + offA1;
        const double* pb0 = Pr + 8 * j0 * sPn;
        const double* pb1 = two ? pb0 + 8 * sPn : pb0;
        for (int s = 0; s < ns; ++s) {
          double a0x, a0y, a1x, a1y;
          if constexpr (TA) {
            a0x = f_ld(pa0); a0y = f_ld(pa0 + lda); a1x = f_ld(pa1); a1y = f_ld(pa1 + lda);
          } else {
            const double2 v0 = f_ld2(pa0), v1 = f_ld2(pa1);
            a0x = v0.x; a0y = v0.y; a1x = v1.x; a1y = v1.y;
          }
          const double b0x = f_ld(pb0), b0y = f_ld(pb0 + sPk), b1x = f_ld(pb1), b1y = f_ld(pb1 + sPk);
          f_dmma(z[0][0][0], z[0][0][1], a0x, b0x);
          f_dmma(z[1][0][0], z[1][0][1], a1x, b0x);
          f_dmma(z[0][1][0], z[0][1][1], a0x, b1x);
          f_dmma(z[1][1][0], z[1][1][1], a1x, b1x);
          f_dmma(z[0][0][0], z[0][0][1], a0y, b0y);
          f_dmma(z[1][0][0], z[1][0][1], a1y, b0y);
          f_dmma(z[0][1][0], z[0][1][1], a0y, b1y);
          f_dmma(z[1][1][0], z[1][1][1], a1y, b1y);
          pa0 += slabA; pa1 += slabA; pb0 += 8 * sPk; pb1 += 8 * sPk;
        }
        // ---- step 2: C += alpha Z W; the accumulator fragments of Z are the A fragments ----
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
          if (jj == 1 && !two) break;
          const double* q = Br + (j0 + jj) * slabB;
          double wx[NTN], wy[NTN];
#pragma unroll
          for (int n = 0; n < NTN; ++n) {
            if constexpr (TB) { const double2 v = f_ld2(q + n * stepB); wx[n] = v.x; wy[n] = v.y; }
            else { wx[n] = f_ld(q + n * stepB); wy[n] = f_ld(q + n * stepB + ldb); }
          }
          const double a0x = z[0][jj][0] * tk.alpha, a0y = z[0][jj][1] * tk.alpha;
          const double a1x = z[1][jj][0] * tk.alpha, a1y = z[1][jj][1] * tk.alpha;
#pragma unroll
          for (int n = 0; n < NTN; ++n) {
            f_dmma(acc[0][n][0], acc[0][n][1], a0x, wx[n]);
            f_dmma(acc[1][n][0], acc[1][n][1], a1x, wx[n]);
          }
#pragma unroll
          for (int n = 0; n < NTN; ++n) {
            f_dmma(acc[0][n][0], acc[0][n][1], a0y, wy[n]);
            f_dmma(acc[1][n][0], acc[1][n][1], a1y, wy[n]);
          }
        }
      }
    }
  } else {
    // ---- two-matrix task: C += alpha op(P)[strip, :] W ----
    const int sPm = (tk.flags & FT_TP) ? 1 : tk.ldp, sPk = (tk.flags & FT_TP) ? tk.ldp : 1;
    const int offA0 = rA * sPm + 2 * lk * sPk, offA1 = rA1 * sPm + 2 * lk * sPk;
    const int ns = tk.ni >> 3;
    for (int r = 0; r < tk.count; ++r) {
      const double* pa0 = tk.P + r * tk.rsP + offA0;
      const double* pa1 = tk.P + r * tk.rsP + offA1;
      const double* q = tk.B + r * tk.rsB + offB;
      for (int s = 0; s < ns; ++s) {
        const double a0x = f_ld(pa0) * tk.alpha, a0y = f_ld(pa0 + sPk) * tk.alpha;
        const double a1x = f_ld(pa1) * tk.alpha, a1y = f_ld(pa1 + sPk) * tk.alpha;
        double wx[NTN], wy[NTN];
#pragma unroll
        for (int n = 0; n < NTN; ++n) {
          if constexpr (TB) { const double2 v = f_ld2(q + n * stepB); wx[n] = v.x; wy[n] = v.y; }
          else { wx[n] = f_ld(q + n * stepB); wy[n] = f_ld(q + n * stepB + ldb); }
        }
#pragma unroll
        for (int n = 0; n < NTN; ++n) {
          f_dmma(acc[0][n][0], acc[0][n][1], a0x, wx[n]);
          f_dmma(acc[1][n][0], acc[1][n][1], a1x, wx[n]);
        }
#pragma unroll
        for (int n = 0; n < NTN; ++n) {
          f_dmma(acc[0][n][0], acc[0][n][1], a0y, wy[n]);
          f_dmma(acc[1][n][0], acc[1][n][1], a1y, wy[n]);
        }
        pa0 += 8 * sPk; pa1 += 8 * sPk; q += slabB;
      }
    }
  }
}

template <int NTN, int MINB>
__global__ void __launch_bounds__(32 * FUSED_WARPS, MINB)
k_fused(const FOut* __restrict__ outs, const FTask* __restrict__ tasks, const int2* __restrict__ items, int nitems) {
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * FUSED_WARPS + (threadIdx.x >> 5);
  if (gw >= nitems) return;
  const int2 item = items[gw];
  const FOut o = outs[item.x];
  const int r0 = item.y, lr = lane >> 2, lk = lane & 3;
  const bool row1 = r0 + 8 < o.M;                  // second 8-row fragment inside the block
  double acc[2][NTN][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int n = 0; n < NTN; ++n) acc[i][n][0] = acc[i][n][1] = 0.0;
  const int rA = r0 + lr, rA1 = row1 ? rA + 8 : rA;                  // (the second fragment of a ragged strip re-reads the first)

  for (int t = o.task_begin; t < o.task_end; ++t) {
    const FTask tk = tasks[t];
    switch (tk.flags & (FT_TA | FT_TB)) {
      case 0: fused_task<NTN, false, false>(acc, tk, rA, rA1, lr, lk); break;
      case FT_TA: fused_task<NTN, true, false>(acc, tk, rA, rA1, lr, lk); break;
      case FT_TB: fused_task<NTN, false, true>(acc, tk, rA, rA1, lr, lk); break;
      default: fused_task<NTN, true, true>(acc, tk, rA, rA1, lr, lk); break;
    }
  }

  double* Cw = o.C + (long long)(r0 + lr) * o.ldc + 2 * lk;
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    if (i == 0 || row1) {
      double2* row = reinterpret_cast<double2*>(Cw + (long long)(8 * i) * o.ldc);
#pragma unroll
      for (int n = 0; n < NTN; ++n) {
        double2 v = make_double2(acc[i][n][0], acc[i][n][1]);
        if (o.accumulate) { const double2 old = row[4 * n]; v.x += old.x; v.y += old.y; }
        row[4 * n] = v;
      }
    }
  }
}

template <int NTN>
cudaError_t launch_one(const FOut* o, const FTask* t, const int2* items, int n, cudaStream_t st) {
  constexpr int MINB = NTN <= 4 ? 4 : 3;      // <= 128 / <= 168 registers per thread
  k_fused<NTN, MINB><<<(n + FUSED_WARPS - 1) / FUSED_WARPS, 32 * FUSED_WARPS, 0, st>>>(o, t, items, n);
  return cudaGetLastError();
}

}  // namespace

int fused_warps_per_sm(int cls) { return FUSED_WARPS * (cls < 4 ? 4 : 3); }

cudaError_t launch_fused(int cls, const FOut* o, const FTask* t, const int2* items, int n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  switch (cls) {
    case 0: return launch_one<1>(o, t, items, n, st);
    case 1: return launch_one<2>(o, t, items, n, st);
    case 2: return launch_one<3>(o, t, items, n, st);
    case 3: return launch_one<4>(o, t, items, n, st);
    case 4: return launch_one<5>(o, t, items, n, st);
    case 5: return launch_one<6>(o, t, items, n, st);
    case 6: return launch_one<7>(o, t, items, n, st);
    case 7: return launch_one<8>(o, t, items, n, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace dmrg
