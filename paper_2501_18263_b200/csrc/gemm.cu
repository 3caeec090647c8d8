// Grouped FP64 GEMM kernels: one CTA per output tile, 8 or 16 warps, DMMA m8n8k4, multi-stage cp.async
// pipeline that runs across segment boundaries.  Nine tile shapes ({32,64,128}^2) are instantiated;
// the inner loop is branch-free with compile-time shared-memory offsets for each of the four
// operand-layout combinations.  See gemm.cuh for the contract.
#include "gemm.cuh"

namespace dmrg {

namespace {

constexpr int KC = 16;        // K extent of one pipeline stage
constexpr int PK = KC + 4;    // pitch of the K-contiguous tile format [x][k]   (conflict-free LDS.64)

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = static_cast<unsigned>(__cvta_generic_to_shared(smem));
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// Walks the flattened (segment, repeat, k-chunk) space of one output.
struct ChunkIter {
  int seg, seg_end, rep, k0, batch;
  const GSeg* segs;
  const double* A;
  const double* B;
  long long rsA, rsB, ams, bns;
  int lda, ldb, K, count, flags, amr, bnr;
  unsigned amr_inv, bnr_inv;
  double alpha;
  __device__ __forceinline__ void load_seg() {
    if (seg < seg_end) {
      const GSeg& s = segs[seg];
      A = s.A + batch * s.bsA; B = s.B + batch * s.bsB;
      rsA = s.rsA; rsB = s.rsB; ams = s.ams; bns = s.bns; amr = s.amr; bnr = s.bnr;
      amr_inv = s.amr_inv; bnr_inv = s.bnr_inv;
      lda = s.lda; ldb = s.ldb; K = s.K; count = s.count; flags = s.flags; alpha = s.alpha;
    }
  }
  __device__ __forceinline__ void init(const GSeg* sg, int b, int e, int bat) {
    segs = sg; seg = b; seg_end = e; rep = 0; k0 = 0; batch = bat;
    load_seg();
  }
  __device__ __forceinline__ bool valid() const { return seg < seg_end; }
  __device__ __forceinline__ void next() {
    k0 += KC;
    if (k0 >= K) {
      k0 = 0;
      if (++rep >= count) { rep = 0; ++seg; load_seg(); }
    }
  }
};

// element offset of logical row/col x (0-based in the whole operand) for a segmented operand
__device__ __forceinline__ long long seg_off(int x, int nr, unsigned inv, long long stride, int& local) {
  if (nr == 0) { local = x; return 0; }
  int b = (int)__umulhi((unsigned)x, inv);
  local = x - b * nr;
  return (long long)b * stride;
}

// Copy one operand tile into shared memory.  BX = tile extent in the non-K dimension.
//   xcontig == 0: element (x, k) at src[x*ld + k]  -> smem [x][k], pitch PK
//   xcontig == 1: element (x, k) at src[k*ld + x]  -> smem [k][x], pitch BX + 4
template <int BX, int NT>
__device__ __forceinline__ void load_tile(double* sm, const double* base, int ld, int x0, int ext, int k0,
                                          int kv, int xcontig, int nr, unsigned inv, long long stride, int tid) {
  constexpr int ITERS = (BX * KC / 2) / NT;
  static_assert(ITERS >= 1, "tile too small for the loader");
  if (!xcontig) {
#pragma unroll
    for (int it = 0; it < ITERS; ++it) {
      int c = tid + it * NT;
      int x = c / (KC / 2), kk = (c % (KC / 2)) * 2;
      if (x < ext && kk < kv) {
        int loc;
        long long o = seg_off(x0 + x, nr, inv, stride, loc);
        cp_async16(sm + x * PK + kk, base + o + (long long)loc * ld + k0 + kk);
      }
    }
  } else {
#pragma unroll
    for (int it = 0; it < ITERS; ++it) {
      int c = tid + it * NT;
      int kr = c / (BX / 2), xx = (c % (BX / 2)) * 2;
      if (kr < kv && xx < ext) {
        int loc;
        long long o = seg_off(x0 + xx, nr, inv, stride, loc);
        cp_async16(sm + kr * (BX + 4) + xx, base + o + (long long)(k0 + kr) * ld + loc);
      }
    }
  }
}

// One pipeline stage of MMAs with compile-time shared-memory offsets.
template <int BM, int BN, int FA, int FB, bool AX, bool BX>
__device__ __forceinline__ void compute_stage(double (&acc)[FA][FB][2], const double* sA, const double* sB,
                                              int wm0, int wn0, int lr, int lk, int kv, double alpha) {
  constexpr int SAM = AX ? 1 : PK, SAK = AX ? (BM + 4) : 1;
  constexpr int SBN = BX ? 1 : PK, SBK = BX ? (BN + 4) : 1;
  const double* pa = sA + (wm0 + lr) * SAM + lk * SAK;
  const double* pb = sB + (wn0 + lr) * SBN + lk * SBK;
  const bool scale = alpha != 1.0;
#pragma unroll
  for (int kk = 0; kk < KC; kk += 4) {
    if (kk < kv) {
      double af[FA], bf[FB];
#pragma unroll
      for (int i = 0; i < FA; ++i) af[i] = pa[(8 * i) * SAM + kk * SAK];
#pragma unroll
      for (int j = 0; j < FB; ++j) bf[j] = pb[(8 * j) * SBN + kk * SBK];
      if (scale) {
#pragma unroll
        for (int j = 0; j < FB; ++j) bf[j] *= alpha;
      }
#pragma unroll
      for (int i = 0; i < FA; ++i)
#pragma unroll
        for (int j = 0; j < FB; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
}

template <int BM, int BN, int WR, int WC, int STAGES, int MINB>
__global__ void __launch_bounds__(32 * WR * WC, MINB)
k_grouped_gemm(const GOut* __restrict__ outs, const GSeg* __restrict__ segs, const GTile* __restrict__ tiles) {
  constexpr int NT = 32 * WR * WC;   // threads per CTA
  constexpr int WM = BM / WR, WN = BN / WC, FA = WM / 8, FB = WN / 8;
  constexpr int TA = BM * PK, TB = BN * PK, STAGE = TA + TB;
  extern __shared__ __align__(16) double smem[];
  const GTile t = tiles[blockIdx.x];
  const GOut o = outs[t.out];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm0 = (warp / WC) * WM, wn0 = (warp % WC) * WN;
  const int m0 = t.m0, n0 = t.n0;
  const int em = min(BM, o.M - m0), en = min(BN, o.N - n0);   // tile extents (multiples of 8)
  const bool active = wm0 < em && wn0 < en;                    // warp-uniform

  double acc[FA][FB][2];
#pragma unroll
  for (int i = 0; i < FA; ++i)
#pragma unroll
    for (int j = 0; j < FB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  ChunkIter prod, cons;
  prod.init(segs, o.seg_begin, o.seg_end, t.batch);
  cons.init(segs, o.seg_begin, o.seg_end, t.batch);

  auto issue = [&](int stage) {
    if (prod.valid()) {
      double* sA = smem + stage * STAGE;
      double* sB = sA + TA;
      const int kv = min(KC, prod.K - prod.k0);
      const int ta = prod.flags & 1, tb = (prod.flags >> 1) & 1;
      // op(A)(m,k): !ta -> A[m*lda+k] (K-contig) ; ta -> A[k*lda+m] (X-contig)
      load_tile<BM, NT>(sA, prod.A + prod.rep * prod.rsA, prod.lda, m0, em, prod.k0, kv, ta, prod.amr,
                    prod.amr_inv, prod.ams, tid);
      // op(B)(k,n): !tb -> B[k*ldb+n] (X-contig) ; tb -> B[n*ldb+k] (K-contig)
      load_tile<BN, NT>(sB, prod.B + prod.rep * prod.rsB, prod.ldb, n0, en, prod.k0, kv, !tb, prod.bnr,
                    prod.bnr_inv, prod.bns, tid);
      prod.next();
    }
    cp_async_commit();
  };

#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) issue(s);

  int stage = 0;
  const int lr = lane >> 2, lk = lane & 3;
  while (cons.valid()) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    issue((stage + STAGES - 1) % STAGES);
    if (active) {
      const double* sA = smem + stage * STAGE;
      const double* sB = sA + TA;
      const int kv = min(KC, cons.K - cons.k0);
      const int ta = cons.flags & 1, tb = (cons.flags >> 1) & 1;
      if (!ta) {
        if (tb) compute_stage<BM, BN, FA, FB, false, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, cons.alpha);
        else compute_stage<BM, BN, FA, FB, false, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, cons.alpha);
      } else {
        if (tb) compute_stage<BM, BN, FA, FB, true, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, cons.alpha);
        else compute_stage<BM, BN, FA, FB, true, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, cons.alpha);
      }
    }
    cons.next();
    stage = (stage + 1) % STAGES;
  }
  cp_async_wait<0>();

  if (!active) return;
  double* C = o.C + (long long)t.batch * o.bsC;
#pragma unroll
  for (int i = 0; i < FA; ++i) {
    const int rl = wm0 + 8 * i;
    if (rl < em) {
#pragma unroll
      for (int j = 0; j < FB; ++j) {
        const int cl = wn0 + 8 * j;
        if (cl < en) {
          double2* p = reinterpret_cast<double2*>(C + (long long)(m0 + rl + lr) * o.ldc + n0 + cl + 2 * lk);
          double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
          if (o.accumulate) {
            double2 old = *p;
            v.x += old.x; v.y += old.y;
          }
          *p = v;
        }
      }
    }
  }
}

template <int BM, int BN, int WR, int WC, int STAGES, int MINB>
struct Cfg {
  static constexpr int smem = STAGES * (BM + BN) * PK * 8;
  static cudaError_t init() {
    return cudaFuncSetAttribute(k_grouped_gemm<BM, BN, WR, WC, STAGES, MINB>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  }
  static cudaError_t launch(const GOut* o, const GSeg* s, const GTile* t, int n, cudaStream_t st) {
    k_grouped_gemm<BM, BN, WR, WC, STAGES, MINB><<<n, 32 * WR * WC, smem, st>>>(o, s, t);
    return cudaGetLastError();
  }
};

//                 BM   BN  WR WC ST MINB
using S32x32   = Cfg<32, 32, 2, 4, 3, 4>;
using S32x64   = Cfg<32, 64, 2, 4, 3, 4>;
using S32x128  = Cfg<32, 128, 1, 8, 3, 3>;
using S64x32   = Cfg<64, 32, 4, 2, 3, 4>;
using S64x64   = Cfg<64, 64, 2, 4, 3, 3>;
using S64x128  = Cfg<64, 128, 2, 4, 3, 2>;
using S128x32  = Cfg<128, 32, 8, 1, 3, 3>;
using S128x64  = Cfg<128, 64, 4, 2, 3, 2>;
using S128x128 = Cfg<128, 128, 4, 4, 4, 1>;

}  // namespace

cudaError_t grouped_gemm_init() {
  cudaError_t e;
  if ((e = S32x32::init()) != cudaSuccess) return e;
  if ((e = S32x64::init()) != cudaSuccess) return e;
  if ((e = S32x128::init()) != cudaSuccess) return e;
  if ((e = S64x32::init()) != cudaSuccess) return e;
  if ((e = S64x64::init()) != cudaSuccess) return e;
  if ((e = S64x128::init()) != cudaSuccess) return e;
  if ((e = S128x32::init()) != cudaSuccess) return e;
  if ((e = S128x64::init()) != cudaSuccess) return e;
  return S128x128::init();
}

cudaError_t launch_grouped_gemm(int shape, const GOut* o, const GSeg* s, const GTile* t, int n, cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  switch (shape) {
    case 0: return S32x32::launch(o, s, t, n, st);
    case 1: return S32x64::launch(o, s, t, n, st);
    case 2: return S32x128::launch(o, s, t, n, st);
    case 3: return S64x32::launch(o, s, t, n, st);
    case 4: return S64x64::launch(o, s, t, n, st);
    case 5: return S64x128::launch(o, s, t, n, st);
    case 6: return S128x32::launch(o, s, t, n, st);
    case 7: return S128x64::launch(o, s, t, n, st);
    case 8: return S128x128::launch(o, s, t, n, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace dmrg
