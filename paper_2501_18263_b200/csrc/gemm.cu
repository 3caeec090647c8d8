// Grouped FP64 GEMM kernels (sm_100a): warp-specialised, NP producer warps + WR*WC consumer warps.
//
//   producer warps: walk the (segment, repeat, k-chunk) list of the CTA's output tiles and stream the two
//                   operand tiles of every k-chunk into a ring of shared-memory stages with 16-byte
//                   cp.async copies whose completion is counted on the stage's "full" mbarrier
//                   (cp.async.mbarrier.arrive.noinc).  They never wait for the math and run ahead into
//                   the CTA's next tile.
//   consumer warps: wait on "full", run the k-chunk on the FP64 tensor pipe (DMMA m8n8k4, the only FP64
//                   MMA shape sm_100a has in SASS), release the stage on its "empty" mbarrier.  No
//                   __syncthreads, no global loads and no address arithmetic in the main loop.
// A CTA handles `tiles_per_cta` consecutive tiles of the launch's (heaviest-first) tile list, so the
// pipeline fill and the epilogue of short-K tiles overlap with the neighbouring tiles' loads.
// Measured on B200: with the copies issued by the MMA warps themselves and a
// __syncthreads per stage every tile shape topped out at 70 % of the DMMA peak; TMA bulk copies
// (cp.async.bulk) cost ~57 clk per copy per SM whatever their size, which starves the K-contiguous
// operand format (one 128-byte row per copy); dedicated cp.async warps reach 92-95 % in the same test.
#include "gemm.cuh"

namespace dmrg {

namespace {

constexpr int KC = 16;        // K extent of one pipeline stage
constexpr int PK = KC + 4;    // pitch of the K-contiguous tile format [x][k]   (conflict-free LDS.64)

__device__ __forceinline__ unsigned smem_u32(const void* p) { return static_cast<unsigned>(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra LAB_DONE;\n"
      "bra LAB_WAIT;\n"
      "LAB_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(smem)), "l"(gmem));
}
__device__ __forceinline__ void cp_async16s(unsigned smem_addr, const void* gmem) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem_addr), "l"(gmem));
}
// the mbarrier receives one (pre-counted) arrival once all prior cp.async of this thread have landed
__device__ __forceinline__ void cp_async_arrive(unsigned long long* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ double lds64(unsigned addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

constexpr int SEGW = sizeof(GSeg) / 8;   // 64-bit words per segment descriptor
constexpr int SEGCACHE = 32;             // descriptors staged in shared memory per producer warp
static_assert(sizeof(GSeg) % 8 == 0, "GSeg is copied as 64-bit words");

// Walks the flattened (segment, repeat, k-chunk) space of one output (producer warps only; all lanes of
// a warp walk in lockstep).  Segment descriptors are staged 32 at a time in a per-warp shared-memory
// cache with one coalesced read, so a list of short segments costs one global latency per 32 of them.
struct ChunkIter {
  int seg, seg_end, rep, k0, batch, cbase, lane;
  const GSeg* segs;
  unsigned long long* cache;
  const double* A;
  const double* B;
  long long rsA, rsB, ams, bns;
  int lda, ldb, K, count, flags, amr, bnr;
  unsigned amr_inv, bnr_inv;
  double alpha;
  __device__ __forceinline__ void load_seg() {
    if (seg < seg_end) {
      if (seg >= cbase + SEGCACHE) {
        __syncwarp();
        cbase = seg;
        const int nw = min(SEGCACHE, seg_end - seg) * SEGW;
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(segs + seg);
        for (int w = lane; w < nw; w += 32) cache[w] = src[w];
        __syncwarp();
      }
      const GSeg& s = *reinterpret_cast<const GSeg*>(cache + (seg - cbase) * SEGW);
      A = s.A + batch * s.bsA; B = s.B + batch * s.bsB;
      rsA = s.rsA; rsB = s.rsB; ams = s.ams; bns = s.bns; amr = s.amr; bnr = s.bnr;
      amr_inv = s.amr_inv; bnr_inv = s.bnr_inv;
      lda = s.lda; ldb = s.ldb; K = s.K; count = s.count; flags = s.flags; alpha = s.alpha;
    }
  }
  __device__ __forceinline__ void init(const GSeg* sg, int b, int e, int bat, unsigned long long* c, int ln) {
    segs = sg; seg = b; seg_end = e; rep = 0; k0 = 0; batch = bat; cache = c; lane = ln;
    cbase = b - SEGCACHE;   // forces the first fill
    load_seg();
  }
  __device__ __forceinline__ bool valid() const { return seg < seg_end; }
  __device__ __forceinline__ bool last() const { return k0 + KC >= K && rep + 1 >= count && seg + 1 >= seg_end; }
  __device__ __forceinline__ void next() {
    k0 += KC;
    if (k0 >= K) {
      k0 = 0;
      if (++rep >= count) { rep = 0; ++seg; load_seg(); }
    }
  }
};

// element offset of logical row/col x (0-based in the whole operand) for a segmented (stacked) operand
__device__ __forceinline__ long long seg_off(int x, int nr, unsigned inv, long long stride, int& local) {
  if (nr == 0) { local = x; return 0; }
  int b = (int)__umulhi((unsigned)x, inv);
  local = x - b * nr;
  return (long long)b * stride;
}

// Producer: copy one operand tile of a k-chunk into shared memory, 16 bytes per cp.async, NPT threads.
// BX = tile extent in the non-K dimension, ext = valid extent (multiple of 8), kv = valid k (8 or 16).
//   xcontig == 0: element (x, k) at src[x*ld + k]  -> smem [x][k], pitch PK
//   xcontig == 1: element (x, k) at src[k*ld + x]  -> smem [k][x], pitch BX + 4
// A thread keeps its 16-byte column (K-contiguous) or its x position (X-contiguous) for the whole tile and
// walks rows with constant strides, so a copy costs a compare, the cp.async and two adds.
template <int BX, int NPT>
__device__ __forceinline__ void produce_tile(double* sm, const double* base, int ld, int x0, int ext, int k0, int kv,
                                             int xcontig, int nr, unsigned inv, long long stride, int pt) {
  if (!xcontig) {
    constexpr int RS = NPT / 8;                  // rows per pass
    constexpr int ITERS = (BX + RS - 1) / RS;
    const int kk = (pt & 7) * 2;
    if (kk >= kv) return;
    int x = pt >> 3;
    unsigned s = smem_u32(sm + x * PK + kk);
    if (nr == 0) {
      const double* g = base + (long long)(x0 + x) * ld + (k0 + kk);
      const long long gs = (long long)RS * ld;
#pragma unroll
      for (int it = 0; it < ITERS; ++it) {
        if (x < ext) cp_async16s(s, g);
        x += RS; s += RS * PK * 8; g += gs;
      }
    } else {
#pragma unroll
      for (int it = 0; it < ITERS; ++it) {
        if (x < ext) {
          int loc;
          const long long o = seg_off(x0 + x, nr, inv, stride, loc);
          cp_async16s(s, base + o + (long long)loc * ld + (k0 + kk));
        }
        x += RS; s += RS * PK * 8;
      }
    }
  } else {
    constexpr int HX = BX / 2;                   // 16-byte columns per k row
    static_assert(NPT % HX == 0, "producer threads must cover whole k rows");
    constexpr int KS = NPT / HX;                 // k rows per pass
    constexpr int ITERS = (KC + KS - 1) / KS;
    const int xx = (pt % HX) * 2;
    if (xx >= ext) return;
    int kr = pt / HX;
    int loc;
    const long long o = seg_off(x0 + xx, nr, inv, stride, loc);
    const double* g = base + o + (long long)(k0 + kr) * ld + loc;
    const long long gs = (long long)KS * ld;
    unsigned s = smem_u32(sm + kr * (BX + 4) + xx);
#pragma unroll
    for (int it = 0; it < ITERS; ++it) {
      if (kr < kv) cp_async16s(s, g);
      kr += KS; s += KS * (BX + 4) * 8; g += gs;
    }
  }
}

// One pipeline stage of MMAs with compile-time shared-memory offsets.
// FAE x FBE (<= FA x FB) = the warp's 8x8 fragments that lie inside the tile's valid extent: a ragged tile
// runs the variant with half the fragment rows and/or columns and pays tensor-pipe time for that area only.
template <int BM, int BN, int FA, int FB, int FAE, int FBE, bool AX, bool BX, bool SCALE>
__device__ __forceinline__ void compute_stage(double (&acc)[FA][FB][2], const double* sA, const double* sB,
                                              int wm0, int wn0, int lr, int lk, int kv, double alpha) {
  constexpr int SAM = AX ? 1 : PK, SAK = AX ? (BM + 4) : 1;
  constexpr int SBN = BX ? 1 : PK, SBK = BX ? (BN + 4) : 1;
  // fragment loads as volatile asm: they keep their place before the (volatile) MMAs of the k-step, so the
  // shared-memory latency is paid once per k-step instead of once per MMA
  const unsigned pa = smem_u32(sA + (wm0 + lr) * SAM + lk * SAK);
  const unsigned pb = smem_u32(sB + (wn0 + lr) * SBN + lk * SBK);
#pragma unroll
  for (int kk = 0; kk < KC; kk += 4) {
    if (kk < kv) {
      double af[FAE], bf[FBE];
#pragma unroll
      for (int i = 0; i < FAE; ++i) af[i] = lds64(pa + ((8 * i) * SAM + kk * SAK) * 8);
#pragma unroll
      for (int j = 0; j < FBE; ++j) bf[j] = lds64(pb + ((8 * j) * SBN + kk * SBK) * 8);
      if (SCALE) {
#pragma unroll
        for (int j = 0; j < FBE; ++j) bf[j] *= alpha;
      }
#pragma unroll
      for (int i = 0; i < FAE; ++i)
#pragma unroll
        for (int j = 0; j < FBE; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }
  }
}

template <int BM, int BN, int FA, int FB, int FAE, int FBE>
__device__ __forceinline__ void compute_dispatch(double (&acc)[FA][FB][2], const double* sA, const double* sB, int wm0,
                                                 int wn0, int lr, int lk, int kv, double alpha, int flags) {
  switch (flags & 7) {   // bit0 ta, bit1 tb, bit2 alpha != 1
    case 0: compute_stage<BM, BN, FA, FB, FAE, FBE, false, true, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, 1.0); break;
    case 1: compute_stage<BM, BN, FA, FB, FAE, FBE, true, true, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, 1.0); break;
    case 2: compute_stage<BM, BN, FA, FB, FAE, FBE, false, false, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, 1.0); break;
    case 3: compute_stage<BM, BN, FA, FB, FAE, FBE, true, false, false>(acc, sA, sB, wm0, wn0, lr, lk, kv, 1.0); break;
    case 4: compute_stage<BM, BN, FA, FB, FAE, FBE, false, true, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, alpha); break;
    case 5: compute_stage<BM, BN, FA, FB, FAE, FBE, true, true, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, alpha); break;
    case 6: compute_stage<BM, BN, FA, FB, FAE, FBE, false, false, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, alpha); break;
    default: compute_stage<BM, BN, FA, FB, FAE, FBE, true, false, true>(acc, sA, sB, wm0, wn0, lr, lk, kv, alpha); break;
  }
}

// What the producers tell the consumers about a stage.  The first chunk of a tile also carries the
// tile itself, so the consumer warps never read a descriptor from global memory.
struct StageMeta {
  double alpha;
  double* C;      // first chunk of a tile: element (m0, n0) of the output (batch applied)
  int kv;
  int flags;      // bit0 ta, bit1 tb, bit2 alpha != 1, bit3 last chunk of the tile, bit4 first chunk of the
                  // tile, bit5 last chunk of the CTA, bit6 output accumulates
  int ldc, em, en, pad_;
};
enum : int { F_LAST = 8, F_FIRST = 16, F_FINAL = 32, F_ACC = 64 };

template <int BM, int BN, int WR, int WC, int NP, int STAGES, int MINB>
__global__ void __launch_bounds__(32 * (WR * WC + NP), MINB)
k_grouped_gemm(const GOut* __restrict__ outs, const GSeg* __restrict__ segs, const GTile* __restrict__ tiles,
               int ntiles, int tiles_per_cta) {
  constexpr int NCW = WR * WC;   // consumer warps
  constexpr int NPT = 32 * NP;   // producer threads
  constexpr int WM = BM / WR, WN = BN / WC, FA = WM / 8, FB = WN / 8;
  constexpr int TA = BM * PK, TB = BN * PK, STAGE = TA + TB;
  static_assert(KC * (BM + 4) <= TA && KC * (BN + 4) <= TB, "x-contiguous format must fit the stage buffer");
  extern __shared__ __align__(16) double smem[];
  __shared__ __align__(8) unsigned long long full_bar[STAGES], empty_bar[STAGES];
  __shared__ __align__(16) StageMeta meta[STAGES];
  __shared__ __align__(16) unsigned long long segcache[NP][SEGCACHE * SEGW];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid == 0) {
    // full: one counted cp.async arrival per producer thread + the explicit arrival that publishes meta
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], NPT + 1); mbar_init(&empty_bar[s], NCW); }
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::);
  }
  __syncthreads();
  int stage = 0;
  unsigned phase = 0;

  // Register split (instances with 64x32 warp tiles whose consumer and producer warps are whole warpgroups):
  // the producers hand most of their registers to the consumers, whose 128 accumulator registers otherwise
  // leave no room to keep the fragment addresses and a full set of fragments live (at the launch-time cap ptxas
  // re-derives the shared-memory addresses at every k-step and funnels the A fragments through one register).
  // The CTA's total stays what it was launched with: NP * (BASE - PREG) = NCW * (CREG - BASE).
  constexpr bool REGSPLIT = (WM == 64 && WN == 32 && NCW % 4 == 0 && NP % 4 == 0);
  constexpr int BASEREG = (65536 / (32 * (NCW + NP) * MINB)) / 8 * 8;   // what __launch_bounds__ lets ptxas use
  constexpr int PREG = BASEREG >= 160 ? 72 : 56;
  constexpr int CREG = (BASEREG + (BASEREG - PREG) * NP / NCW) / 8 * 8;
  static_assert(!REGSPLIT || (CREG <= 232 && NP * PREG + NCW * CREG <= (NCW + NP) * BASEREG), "register split");
  if (warp >= NCW) {
    if constexpr (REGSPLIT) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;\n" ::"n"(PREG));
    // ------------------------------------------------ producers ------------------------------------------------
    // (every tile of the list has at least one k-chunk: the planner emits no tiles for empty outputs)
    const int pt = tid - 32 * NCW;
    const int t_begin = blockIdx.x * tiles_per_cta, t_end = min(ntiles, t_begin + tiles_per_cta);
    GTile tn = tiles[t_begin];
    for (int ti = t_begin; ti < t_end; ++ti) {
      const GTile t = tn;
      if (ti + 1 < t_end) tn = tiles[ti + 1];   // in flight while this tile streams
      const GOut o = outs[t.out];
      const int em = min(BM, o.M - t.m0), en = min(BN, o.N - t.n0);
      ChunkIter it;
      it.init(segs, o.seg_begin, o.seg_end, t.batch, segcache[warp - NCW], lane);
      bool first = true;
      while (it.valid()) {
        mbar_wait(&empty_bar[stage], phase ^ 1);
        double* sA = smem + stage * STAGE;
        double* sB = sA + TA;
        const int kv = min(KC, it.K - it.k0);
        const int ta = it.flags & 1, tb = (it.flags >> 1) & 1;
        if (pt == 0) {
          const bool last = it.last();
          StageMeta m;
          m.alpha = it.alpha;
          m.C = o.C + (long long)t.batch * o.bsC + (long long)t.m0 * o.ldc + t.n0;
          m.kv = kv;
          m.flags = (it.flags & 3) | (it.alpha != 1.0 ? 4 : 0) | (last ? F_LAST : 0) | (first ? F_FIRST : 0) |
                    (last && ti + 1 == t_end ? F_FINAL : 0) | (o.accumulate ? F_ACC : 0);
          m.ldc = o.ldc; m.em = em; m.en = en; m.pad_ = 0;
          meta[stage] = m;
          mbar_arrive(&full_bar[stage]);
        }
        first = false;
        // op(A)(m,k): !ta -> A[m*lda+k] (K-contig) ; ta -> A[k*lda+m] (X-contig)
        produce_tile<BM, NPT>(sA, it.A + it.rep * it.rsA, it.lda, t.m0, em, it.k0, kv, ta, it.amr, it.amr_inv, it.ams, pt);
        // op(B)(k,n): !tb -> B[k*ldb+n] (X-contig) ; tb -> B[n*ldb+k] (K-contig)
        produce_tile<BN, NPT>(sB, it.B + it.rep * it.rsB, it.ldb, t.n0, en, it.k0, kv, !tb, it.bnr, it.bnr_inv, it.bns, pt);
        cp_async_arrive(&full_bar[stage]);
        it.next();
        if (++stage == STAGES) { stage = 0; phase ^= 1; }
      }
    }
    asm volatile("cp.async.wait_all;\n" ::);
    return;
  }

  // ---------------------------------------------------- consumers ----------------------------------------------------
  // One stream of stages; tile boundaries are flags in the stage meta.
  if constexpr (REGSPLIT) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;\n" ::"n"(CREG));
  const int wm0 = (warp / WC) * WM, wn0 = (warp % WC) * WN;
  const int lr = lane >> 2, lk = lane & 3;
  double acc[FA][FB][2];
  double* C = nullptr;
  int ldc = 0, em = 0, en = 0, accum = 0;
  bool active = false;
  int part = 0;
  while (true) {
    mbar_wait(&full_bar[stage], phase);
    const StageMeta mt = meta[stage];
    if (mt.flags & F_FIRST) {
      C = mt.C; ldc = mt.ldc; em = mt.em; en = mt.en; accum = mt.flags & F_ACC;
      active = wm0 < em && wn0 < en;   // warp-uniform
      part = (em - wm0 <= 4 * FA ? 1 : 0) | (en - wn0 <= 4 * FB ? 2 : 0);
#pragma unroll
      for (int i = 0; i < FA; ++i)
#pragma unroll
        for (int j = 0; j < FB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    }
    if (active) {
      const double* sA = smem + stage * STAGE;
      const double* sB = sA + TA;
      // 128x128 tiles are 94-97 % full in the measured workloads: that instance keeps one variant (the extra
      // variants cost it 4 % through code size); the narrower shapes (fill 25-85 %) get the half variants
      constexpr bool RAGGED = BM * BN < 128 * 128;
      if (!RAGGED || part == 0)
        compute_dispatch<BM, BN, FA, FB, FA, FB>(acc, sA, sB, wm0, wn0, lr, lk, mt.kv, mt.alpha, mt.flags);
      else if (part == 1)
        compute_dispatch<BM, BN, FA, FB, RAGGED ? FA / 2 : FA, FB>(acc, sA, sB, wm0, wn0, lr, lk, mt.kv, mt.alpha, mt.flags);
      else if (part == 2)
        compute_dispatch<BM, BN, FA, FB, FA, RAGGED ? FB / 2 : FB>(acc, sA, sB, wm0, wn0, lr, lk, mt.kv, mt.alpha, mt.flags);
      else
        compute_dispatch<BM, BN, FA, FB, RAGGED ? FA / 2 : FA, RAGGED ? FB / 2 : FB>(acc, sA, sB, wm0, wn0, lr, lk, mt.kv, mt.alpha, mt.flags);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty_bar[stage]);
    if (++stage == STAGES) { stage = 0; phase ^= 1; }
    if (!(mt.flags & F_LAST)) continue;

    if (active) {
      // epilogue: one 8-row fragment strip (FB double2 per thread) at a time; for accumulating outputs all
      // loads of a strip are issued before its adds and stores, so the read latency is paid once per strip
      double* Cw = C + (long long)(wm0 + lr) * ldc + wn0 + 2 * lk;
#pragma unroll
      for (int i = 0; i < FA; ++i) {
        if (wm0 + 8 * i < em) {
          double2* row = reinterpret_cast<double2*>(Cw + (long long)(8 * i) * ldc);
          double2 old[FB];
          if (accum) {
#pragma unroll
            for (int j = 0; j < FB; ++j)
              if (wn0 + 8 * j < en) old[j] = row[4 * j];
          }
#pragma unroll
          for (int j = 0; j < FB; ++j) {
            if (wn0 + 8 * j < en) {
              double2 v = make_double2(acc[i][j][0], acc[i][j][1]);
              if (accum) { v.x += old[j].x; v.y += old[j].y; }
              row[4 * j] = v;
            }
          }
        }
      }
    }
    if (mt.flags & F_FINAL) break;
  }
}

template <int BM, int BN, int WR, int WC, int NP, int STAGES, int MINB>
struct Cfg {
  static constexpr int smem = STAGES * (BM + BN) * PK * 8;
  static constexpr int threads = 32 * (WR * WC + NP);
  static constexpr int minb = MINB;
  static cudaError_t init() {
    return cudaFuncSetAttribute(k_grouped_gemm<BM, BN, WR, WC, NP, STAGES, MINB>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  }
  static cudaError_t launch(const GOut* o, const GSeg* s, const GTile* t, int n, int per, cudaStream_t st) {
    k_grouped_gemm<BM, BN, WR, WC, NP, STAGES, MINB><<<(n + per - 1) / per, threads, smem, st>>>(o, s, t, n, per);
    return cudaGetLastError();
  }
};

//                 BM   BN  WR WC NP ST MINB     warp tile
using S32x32   = Cfg<32, 32, 1, 1, 2, 6, 4>;   // 32x32
using S32x64   = Cfg<32, 64, 1, 2, 2, 6, 3>;   // 32x32
using S32x128  = Cfg<32, 128, 1, 4, 2, 4, 2>;  // 32x32
using S64x32   = Cfg<64, 32, 2, 1, 2, 6, 3>;   // 32x32
using S64x64   = Cfg<64, 64, 2, 2, 4, 4, 2>;   // 32x32
using S64x128  = Cfg<64, 128, 1, 4, 4, 3, 2>;  // 64x32, register split 56 / 200
using S128x32  = Cfg<128, 32, 4, 1, 2, 4, 2>;  // 32x32
using S128x64  = Cfg<128, 64, 2, 2, 4, 3, 2>;  // 64x32, register split 56 / 200
using S128x128 = Cfg<128, 128, 2, 4, 4, 5, 1>; // 64x32, register split 72 / 216

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

int gemm_shape_ctas_per_sm(int shape) {
  switch (shape) {
    case 0: return S32x32::minb;
    case 1: return S32x64::minb;
    case 2: return S32x128::minb;
    case 3: return S64x32::minb;
    case 4: return S64x64::minb;
    case 5: return S64x128::minb;
    case 6: return S128x32::minb;
    case 7: return S128x64::minb;
    default: return S128x128::minb;
  }
}

cudaError_t launch_grouped_gemm(int shape, const GOut* o, const GSeg* s, const GTile* t, int n, int tiles_per_cta,
                                cudaStream_t st) {
  if (n <= 0) return cudaSuccess;
  const int per = tiles_per_cta < 1 ? 1 : tiles_per_cta;
  switch (shape) {
    case 0: return S32x32::launch(o, s, t, n, per, st);
    case 1: return S32x64::launch(o, s, t, n, per, st);
    case 2: return S32x128::launch(o, s, t, n, per, st);
    case 3: return S64x32::launch(o, s, t, n, per, st);
    case 4: return S64x64::launch(o, s, t, n, per, st);
    case 5: return S64x128::launch(o, s, t, n, per, st);
    case 6: return S128x32::launch(o, s, t, n, per, st);
    case 7: return S128x64::launch(o, s, t, n, per, st);
    case 8: return S128x128::launch(o, s, t, n, per, st);
  }
  return cudaErrorInvalidValue;
}

}  // namespace dmrg
