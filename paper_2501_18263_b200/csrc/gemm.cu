// Grouped FP64 GEMM kernel: 128x128 output tile per CTA, 8 warps, DMMA m8n8k4, 4-stage cp.async
// pipeline that runs across segment boundaries.  See gemm.cuh for the contract.
#include "gemm.cuh"

namespace dmrg {

namespace {

constexpr int BM = GEMM_BM, BN = GEMM_BN, KC = GEMM_KC, STAGES = GEMM_STAGES;
constexpr int PK = KC + 4;   // pitch of the K-contiguous tile format  [x][k]
constexpr int PX = BM + 4;   // pitch of the X-contiguous tile format  [k][x]   (BM == BN)
constexpr int TILE_DOUBLES = BM * PK;  // >= KC * PX

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
  int seg, seg_end, rep, k0;
  const GSeg* segs;
  // current segment (valid when seg < seg_end)
  const double* A;
  const double* B;
  long long rsA, rsB;
  int lda, ldb, K, count, flags, batch;
  double alpha;
  __device__ __forceinline__ void load_seg() {
    if (seg < seg_end) {
      const GSeg& s = segs[seg];
      A = s.A + batch * s.bsA; B = s.B + batch * s.bsB;
      rsA = s.rsA; rsB = s.rsB; lda = s.lda; ldb = s.ldb;
      K = s.K; count = s.count; flags = s.flags; alpha = s.alpha;
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

// Copy one operand tile (X extent `ext`, K extent `kv`) into shared memory.
//   trans == 0 ("K-contiguous"): element (x, k) at src[x*ld + k]  -> smem [x][k], pitch PK
//   trans == 1 ("X-contiguous"): element (x, k) at src[k*ld + x]  -> smem [k][x], pitch PX
__device__ __forceinline__ void load_tile(double* sm, const double* src, int ld, int ext, int kv,
                                          int xcontig, int tid) {
  if (!xcontig) {
#pragma unroll
    for (int it = 0; it < (BM * KC / 2) / GEMM_THREADS; ++it) {
      int c = tid + it * GEMM_THREADS;
      int x = c / (KC / 2), kk = (c % (KC / 2)) * 2;
      if (x < ext && kk < kv) cp_async16(sm + x * PK + kk, src + (long long)x * ld + kk);
    }
  } else {
#pragma unroll
    for (int it = 0; it < (BM * KC / 2) / GEMM_THREADS; ++it) {
      int c = tid + it * GEMM_THREADS;
      int kr = c / (BM / 2), xx = (c % (BM / 2)) * 2;
      if (kr < kv && xx < ext) cp_async16(sm + kr * PX + xx, src + (long long)kr * ld + xx);
    }
  }
}

__global__ void __launch_bounds__(GEMM_THREADS, 1)
k_grouped_gemm(const GOut* __restrict__ outs, const GSeg* __restrict__ segs,
               const GTile* __restrict__ tiles) {
  extern __shared__ __align__(16) double smem[];
  const GTile t = tiles[blockIdx.x];
  const GOut o = outs[t.out];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wr = warp & 1, wc = warp >> 1;  // 2 warp rows x 4 warp columns, sub-tiles interleaved
  const int m0 = t.tm * o.tile_m, n0 = t.tn * o.tile_n;
  const int em = min(o.tile_m, o.M - m0), en = min(o.tile_n, o.N - n0);  // tile extents
  const int ntm = em >> 3, ntn = en >> 3;
  const int na = (ntm - wr + 1) >> 1;  // active 8-row sub-tiles of this warp (rows wr, wr+2, ..)
  const int nb = (ntn - wc + 3) >> 2;  // active 8-col sub-tiles (cols wc, wc+4, ..)

  double acc[8][4][2];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  ChunkIter prod, cons;
  prod.init(segs, o.seg_begin, o.seg_end, t.batch);
  cons.init(segs, o.seg_begin, o.seg_end, t.batch);

  auto issue = [&](int stage) {
    if (prod.valid()) {
      double* sA = smem + stage * GEMM_STAGE_DOUBLES;
      double* sB = sA + TILE_DOUBLES;
      const int kv = min(KC, prod.K - prod.k0);
      const int ta = prod.flags & 1, tb = (prod.flags >> 1) & 1;
      const double* a = prod.A + prod.rep * prod.rsA;
      const double* b = prod.B + prod.rep * prod.rsB;
      // op(A)(m,k): !ta -> A[m*lda+k] (K-contig) ; ta -> A[k*lda+m] (X-contig)
      a += ta ? ((long long)prod.k0 * prod.lda + m0) : ((long long)m0 * prod.lda + prod.k0);
      // op(B)(k,n): !tb -> B[k*ldb+n] (X-contig) ; tb -> B[n*ldb+k] (K-contig)
      b += tb ? ((long long)n0 * prod.ldb + prod.k0) : ((long long)prod.k0 * prod.ldb + n0);
      load_tile(sA, a, prod.lda, em, kv, ta, tid);
      load_tile(sB, b, prod.ldb, en, kv, !tb, tid);
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

    const double* sA = smem + stage * GEMM_STAGE_DOUBLES;
    const double* sB = sA + TILE_DOUBLES;
    const int kv = min(KC, cons.K - cons.k0);
    const int ta = cons.flags & 1, tb = (cons.flags >> 1) & 1;
    const int sAm = ta ? 1 : PK, sAk = ta ? PX : 1;
    const int sBn = tb ? PK : 1, sBk = tb ? 1 : PX;
    const double alpha = cons.alpha;
    const double* pa = sA + (wr * 8 + lr) * sAm + lk * sAk;
    const double* pb = sB + (wc * 8 + lr) * sBn + lk * sBk;
    for (int kk = 0; kk < kv; kk += 4) {
      double af[8], bf[4];
#pragma unroll
      for (int i = 0; i < 8; ++i)
        if (i < na) af[i] = alpha * pa[(16 * i) * sAm + kk * sAk];
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (j < nb) bf[j] = pb[(32 * j) * sBn + kk * sBk];
#pragma unroll
      for (int i = 0; i < 8; ++i)
        if (i < na) {
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (j < nb) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }
    cons.next();
    stage = (stage + 1) % STAGES;
  }
  cp_async_wait<0>();

  double* C = o.C + (long long)t.batch * o.bsC;
#pragma unroll
  for (int i = 0; i < 8; ++i)
    if (i < na) {
      const int row = m0 + (wr + 2 * i) * 8 + lr;
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (j < nb) {
          const int col = n0 + (wc + 4 * j) * 8 + 2 * lk;
          double2* p = reinterpret_cast<double2*>(C + (long long)row * o.ldc + col);
          double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
          if (o.accumulate) {
            double2 old = *p;
            v.x += old.x; v.y += old.y;
          }
          *p = v;
        }
    }
}

}  // namespace

cudaError_t grouped_gemm_init() {
  return cudaFuncSetAttribute(k_grouped_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              GEMM_SMEM_BYTES);
}

cudaError_t launch_grouped_gemm(const GOut* d_outs, const GSeg* d_segs, const GTile* d_tiles,
                                int ntiles, cudaStream_t stream) {
  if (ntiles <= 0) return cudaSuccess;
  k_grouped_gemm<<<ntiles, GEMM_THREADS, GEMM_SMEM_BYTES, stream>>>(d_outs, d_segs, d_tiles);
  return cudaGetLastError();
}

}  // namespace dmrg
