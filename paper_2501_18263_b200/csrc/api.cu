// extern "C" boundary of the library (include/dmrg_b200.h).  Argument marshalling, input checks,
// the environment / renormalisation drivers and the Davidson loop; all arithmetic on vectors and
// operator blocks runs in the CUDA kernels of gemm.cu / kernels.cu.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "engine.h"
#include "su2.h"

using namespace dmrg;

#define API_BEGIN                                  \
  if (!ctx) return DMRG_ERR_ARG;                   \
  try {                                            \
    DMRG_CUDA(cudaSetDevice(ctx->cfg.device));
#define API_END                                    \
    return DMRG_OK;                                \
  } catch (const dmrg::Error& e) {                 \
    ctx->err = e.what();                           \
    return e.code;                                 \
  } catch (const std::exception& e) {              \
    ctx->err = e.what();                           \
    return DMRG_ERR_ARG;                           \
  }

namespace dmrg {
bool HostPool::get(size_t npages, std::vector<double*>* out) {
  out->clear();
  while (free_pages.size() < npages) {
    if (total + page_bytes > cap) return false;
    void* p = nullptr;
    if (cudaMallocHost(&p, page_bytes) != cudaSuccess) { cudaGetLastError(); return false; }
    total += page_bytes;
    free_pages.push_back(static_cast<double*>(p));
  }
  out->assign(free_pages.end() - npages, free_pages.end());
  free_pages.resize(free_pages.size() - npages);
  return true;
}
HostPool::~HostPool() { for (double* p : free_pages) cudaFreeHost(p); }
}  // namespace dmrg

extern "C" {

int dmrg_create(const dmrg_config* cfg, dmrg_ctx** out) {
  if (!cfg || !out) return DMRG_ERR_ARG;
  *out = nullptr;
  if (cfg->symmetry != 0 && cfg->symmetry != 1) return DMRG_ERR_UNSUPPORTED;
  if (cfg->symmetry == 1 && cfg->n_up != cfg->n_dn) return DMRG_ERR_UNSUPPORTED;   // SU(2): total spin 0 only
  if (!cfg->alloc || !cfg->free || cfg->L < 2 || cfg->L > 64 || cfg->n_up < 0 || cfg->n_dn < 0 ||
      cfg->n_up > cfg->L || cfg->n_dn > cfg->L)
    return DMRG_ERR_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || cfg->device < 0 || cfg->device >= ndev) return DMRG_ERR_CUDA;
  if (cudaSetDevice(cfg->device) != cudaSuccess) return DMRG_ERR_CUDA;
  if (grouped_gemm_init() != cudaSuccess) return DMRG_ERR_CUDA;
  dmrg_ctx* c = new dmrg_ctx();
  c->cfg = *cfg;
  c->al.alloc = cfg->alloc;
  c->al.free_ = cfg->free;
  c->al.user = cfg->alloc_user;
  c->L = cfg->L;
  c->site.resize(cfg->L + 2);
  c->site_ops.build_products();
  if (cfg->env_host_bytes) {
    c->host_pool = std::make_shared<dmrg::HostPool>();
    c->host_pool->cap = cfg->env_host_bytes;
    // 256 MiB pages for real problems; small caps (tests) get 64 pages
    uint64_t pb = std::min<uint64_t>(1ull << 28, std::max<uint64_t>(1ull << 16, cfg->env_host_bytes / 64));
    c->host_pool->page_bytes = pb & ~7ull;
  }
  try {
    if (!std::getenv("DMRG_B200_SERIAL")) c->exec.init();   // debugging aid: every launch in order on one stream
  } catch (const dmrg::Error&) {
    delete c;
    return DMRG_ERR_CUDA;
  }
  *out = c;
  return DMRG_OK;
}

int dmrg_destroy(dmrg_ctx* ctx) {
  if (!ctx) return DMRG_ERR_ARG;
  cudaSetDevice(ctx->cfg.device);
  cudaDeviceSynchronize();
  delete ctx;
  return DMRG_OK;
}

const char* dmrg_last_error(const dmrg_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int dmrg_load_integrals(dmrg_ctx* ctx, int32_t L, const double* h_T, const double* h_V, double e_core) {
  API_BEGIN
  DMRG_REQUIRE(L == ctx->L && h_T && h_V, DMRG_ERR_ARG, "load_integrals: bad arguments");
  const size_t n = (size_t)L;
  for (size_t i = 0; i < n; ++i)
    for (size_t j = 0; j < i; ++j)
      DMRG_REQUIRE(std::fabs(h_T[i * n + j] - h_T[j * n + i]) <= 1e-12, DMRG_ERR_INPUT, "T is not symmetric");
  auto V = [&](size_t i, size_t j, size_t k, size_t l) { return h_V[((i * n + j) * n + k) * n + l]; };
  for (size_t i = 0; i < n; ++i) for (size_t j = 0; j < n; ++j) for (size_t k = 0; k < n; ++k) for (size_t l = 0; l < n; ++l)
    DMRG_REQUIRE(std::fabs(V(i, j, k, l) - V(k, l, i, j)) <= 1e-12, DMRG_ERR_INPUT, "V_ijkl != V_klij");
  ctx->drop_term_groups();                             // (waits for builders that still read the old integrals)
  ctx->T.assign(h_T, h_T + n * n);
  ctx->w.resize(n * n * n * n);
  for (size_t i = 0; i < n; ++i) for (size_t j = 0; j < n; ++j) for (size_t k = 0; k < n; ++k) for (size_t l = 0; l < n; ++l)
    ctx->w[((i * n + j) * n + k) * n + l] = 0.5 * (V(i, j, k, l) + V(j, i, l, k));
  ctx->e_core = e_core;
  ctx->have_integrals = true;
  ctx->left_cache.clear(); ctx->right_cache.clear();   // every operator depends on the integrals
  ctx->left.reset(); ctx->right.reset();
  ctx->k = 0;
  API_END
}

int dmrg_mps_set_sectors(dmrg_ctx* ctx, const int32_t* off, const int32_t* qu, const int32_t* qd, const int32_t* dim) {
  API_BEGIN
  DMRG_REQUIRE(off && qu && qd && dim, DMRG_ERR_ARG, "set_sectors: null pointer");
  const int L = ctx->L;
  std::vector<Sectors> bond(L + 1);
  for (int b = 0; b <= L; ++b) {
    DMRG_REQUIRE(off[b + 1] > off[b], DMRG_ERR_INPUT, "set_sectors: empty bond");
    for (int i = off[b]; i < off[b + 1]; ++i) {
      DMRG_REQUIRE(dim[i] > 0 && qu[i] >= 0 && qd[i] >= 0, DMRG_ERR_INPUT, "set_sectors: bad sector");
      if (i > off[b])
        DMRG_REQUIRE(qu[i - 1] < qu[i] || (qu[i - 1] == qu[i] && qd[i - 1] < qd[i]), DMRG_ERR_INPUT,
                     "set_sectors: sectors not sorted");
      bond[b].add(qu[i], qd[i], dim[i]);
    }
  }
  DMRG_REQUIRE(bond[0].size() == 1 && bond[0].qu[0] == 0 && bond[0].qd[0] == 0 && bond[0].dim[0] == 1,
               DMRG_ERR_INPUT, "set_sectors: bond 0 must be {(0,0):1}");
  if (ctx->su2())
    DMRG_REQUIRE(bond[L].size() == 1 && bond[L].qu[0] == ctx->cfg.n_up + ctx->cfg.n_dn && bond[L].qd[0] == 0 &&
                     bond[L].dim[0] == 1, DMRG_ERR_INPUT, "set_sectors: bond L must be {(N, 2S=0):1}");
  else
    DMRG_REQUIRE(bond[L].size() == 1 && bond[L].qu[0] == ctx->cfg.n_up && bond[L].qd[0] == ctx->cfg.n_dn &&
                     bond[L].dim[0] == 1, DMRG_ERR_INPUT, "set_sectors: bond L must be {(n_up,n_dn):1}");
  ctx->bond = std::move(bond);
  ctx->centre.clear();
  for (auto& s : ctx->site) { s.canonical = -1; s.blks.clear(); s.find.clear(); s.find3.clear(); s.data.release(); }
  ctx->left_cache.clear(); ctx->right_cache.clear();
  ctx->left.reset(); ctx->right.reset();
  ctx->k = 0;
  API_END
}

static int set_site_impl(dmrg_ctx* ctx, int32_t site, int32_t canonical, int32_t nblocks, const int32_t* qin,
                         const int32_t* s, const int32_t* qout_su2, const int64_t* blk_off, const double* h_data,
                         void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE((qout_su2 != nullptr) == ctx->su2(), DMRG_ERR_ARG,
               "set_site: use dmrg_mps_set_site for U(1)xU(1) and dmrg_mps_set_site_su2 for SU(2) contexts");
  DMRG_REQUIRE(!ctx->bond.empty(), DMRG_ERR_ARG, "set_site: call dmrg_mps_set_sectors first");
  DMRG_REQUIRE(site >= 1 && site <= ctx->L && (canonical == 0 || canonical == 1) && nblocks > 0 && qin && s &&
                   blk_off && h_data, DMRG_ERR_ARG, "set_site: bad arguments");
  const Sectors& bi = ctx->bond[site - 1];
  const Sectors& bo = ctx->bond[site];
  SiteTensor t;
  t.canonical = canonical;
  long long off = 0;
  for (int n = 0; n < nblocks; ++n) {
    DMRG_REQUIRE(qin[n] >= 0 && qin[n] < bi.size() && s[n] >= 0 && s[n] < (qout_su2 ? 3 : 4), DMRG_ERR_INPUT,
                 "set_site: bad block label");
    int qo;
    if (qout_su2) {   // SU(2): (N, 2S) + multiplet m -> (N + n(m), 2S or 2S +- 1)
      qo = qout_su2[n];
      DMRG_REQUIRE(qo >= 0 && qo < bo.size(), DMRG_ERR_INPUT, "set_site: bad q_out");
      const int dN = bo.qu[qo] - bi.qu[qin[n]], dS = bo.qd[qo] - bi.qd[qin[n]];
      DMRG_REQUIRE(dN == su2::MULT_N[s[n]] && (su2::MULT_S2[s[n]] == 0 ? dS == 0 : (dS == 1 || dS == -1)), DMRG_ERR_INPUT,
                   "set_site: q_out is not a coupling of q_in with the site multiplet");
    } else {
      qo = bo.find(bi.qu[qin[n]] + SITE_QU[s[n]], bi.qd[qin[n]] + SITE_QD[s[n]]);
      DMRG_REQUIRE(qo >= 0, DMRG_ERR_INPUT, "set_site: q_in + q(s) is not a sector of the next bond");
    }
    SiteBlk b{qin[n], s[n], qo, bi.dim[qin[n]], bo.dim[qo], pad8(bi.dim[qin[n]]), pad8(bo.dim[qo]), off};
    off += (long long)b.dinp * b.doutp;
    if (qout_su2)
      DMRG_REQUIRE(t.find3.emplace(std::array<int, 3>{b.qin, b.s, b.qout}, n).second, DMRG_ERR_INPUT, "set_site: duplicate block");
    else
      DMRG_REQUIRE(t.find.emplace(std::make_pair(b.qin, b.s), n).second, DMRG_ERR_INPUT, "set_site: duplicate block");
    t.blks.push_back(b);
  }
  // isometry check on the host (input validation only)
  if (canonical == 0) {
    for (int qo = 0; qo < bo.size(); ++qo) {
      const int d = bo.dim[qo];
      std::vector<double> g((size_t)d * d, 0.0);
      for (int n = 0; n < nblocks; ++n) {
        if (t.blks[n].qout != qo) continue;
        const double* a = h_data + blk_off[n];
        for (int r = 0; r < t.blks[n].din; ++r)
          for (int i = 0; i < d; ++i) {
            const double ai = a[(size_t)r * d + i];
            if (ai == 0.0) continue;
            for (int j = 0; j < d; ++j) g[(size_t)i * d + j] += ai * a[(size_t)r * d + j];
          }
      }
      for (int i = 0; i < d; ++i) for (int j = 0; j < d; ++j)
        DMRG_REQUIRE(std::fabs(g[(size_t)i * d + j] - (i == j ? 1.0 : 0.0)) <= 1e-10, DMRG_ERR_INPUT,
                     "set_site: tensor is not left-canonical");
    }
  } else {
    for (int qi = 0; qi < bi.size(); ++qi) {
      const int d = bi.dim[qi];
      std::vector<double> g((size_t)d * d, 0.0);
      for (int n = 0; n < nblocks; ++n) {
        if (t.blks[n].qin != qi) continue;
        const double* a = h_data + blk_off[n];
        const int c = t.blks[n].dout;
        for (int i = 0; i < d; ++i) for (int j = 0; j < d; ++j) {
          double sum = 0;
          for (int q = 0; q < c; ++q) sum += a[(size_t)i * c + q] * a[(size_t)j * c + q];
          g[(size_t)i * d + j] += sum;
        }
      }
      for (int i = 0; i < d; ++i) for (int j = 0; j < d; ++j)
        DMRG_REQUIRE(std::fabs(g[(size_t)i * d + j] - (i == j ? 1.0 : 0.0)) <= 1e-10, DMRG_ERR_INPUT,
                     "set_site: tensor is not right-canonical");
    }
  }
  std::vector<double> padded((size_t)std::max<long long>(off, 8), 0.0);
  for (int n = 0; n < nblocks; ++n) {
    const SiteBlk& b = t.blks[n];
    const double* a = h_data + blk_off[n];
    for (int r = 0; r < b.din; ++r)
      std::memcpy(&padded[(size_t)b.off + (size_t)r * b.doutp], a + (size_t)r * b.dout, sizeof(double) * b.dout);
  }
  t.data.upload(&ctx->al, padded, st);
  DMRG_CUDA(cudaStreamSynchronize(st));
  ctx->invalidate_site(site);
  ctx->site[site] = std::move(t);
  API_END
}

int dmrg_mps_update_bond(dmrg_ctx* ctx, int32_t b, int32_t nsec, const int32_t* qu, const int32_t* qd, const int32_t* dim) {
  API_BEGIN
  DMRG_REQUIRE(!ctx->bond.empty() && b >= 1 && b <= ctx->L - 1 && nsec > 0 && qu && qd && dim, DMRG_ERR_ARG,
               "update_bond: bad arguments");
  Sectors s;
  for (int i = 0; i < nsec; ++i) {
    DMRG_REQUIRE(dim[i] > 0 && qu[i] >= 0 && qd[i] >= 0, DMRG_ERR_INPUT, "update_bond: bad sector");
    if (i > 0)
      DMRG_REQUIRE(qu[i - 1] < qu[i] || (qu[i - 1] == qu[i] && qd[i - 1] < qd[i]), DMRG_ERR_INPUT, "update_bond: sectors not sorted");
    s.add(qu[i], qd[i], dim[i]);
  }
  ctx->bond[b] = std::move(s);
  ctx->centre.clear();                      // (a centre factor of dmrg_truncate_bond refers to the old sectors)
  for (int i : {b, b + 1}) {
    SiteTensor& t = ctx->site[i];
    t.canonical = -1; t.blks.clear(); t.find.clear(); t.find3.clear(); t.data.release();
  }
  ctx->invalidate_site(b);
  ctx->invalidate_site(b + 1);
  API_END
}

int dmrg_mps_set_site(dmrg_ctx* ctx, int32_t site, int32_t canonical, int32_t nblocks, const int32_t* qin,
                      const int32_t* s, const int64_t* blk_off, const double* h_data, void* stream) {
  return set_site_impl(ctx, site, canonical, nblocks, qin, s, nullptr, blk_off, h_data, stream);
}

int dmrg_mps_set_site_su2(dmrg_ctx* ctx, int32_t site, int32_t canonical, int32_t nblocks, const int32_t* qin,
                          const int32_t* m, const int32_t* qout, const int64_t* blk_off, const double* h_data,
                          void* stream) {
  if (!qout) return DMRG_ERR_ARG;
  return set_site_impl(ctx, site, canonical, nblocks, qin, m, qout, blk_off, h_data, stream);
}

// dmrg_env_build / dmrg_renormalize: while the environments and the plan are being replaced there is no prepared
// problem; if the call fails half way the context stays in that state (k = 0) instead of pointing at stale blocks.
struct PreparedGuard {
  dmrg_ctx* ctx;
  bool ok = false;
  ~PreparedGuard() {
    if (ok) return;
    ctx->k = 0;
    ctx->apply_plan.clear();
    ctx->left.reset();
    ctx->right.reset();
  }
};

static uint64_t env_cache_cap(const dmrg_ctx* ctx) {
  if (ctx->cfg.env_cache_bytes) return ctx->cfg.env_cache_bytes;
  size_t fr = 0, tot = 0;
  if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) return 0;
  return tot / 8;
}

// ---- host tier of the environment cache (cfg.env_host_bytes) ----
// copies `n` doubles between a device array and the page list, starting at element `pos` of the paged stream
static void paged_copy(std::vector<double*>& pages, uint64_t page_elems, uint64_t pos, double* dev, size_t n, bool to_host,
                       cudaStream_t st) {
  size_t done = 0;
  while (done < n) {
    const uint64_t pg = (pos + done) / page_elems, off = (pos + done) % page_elems;
    const size_t m = (size_t)std::min<uint64_t>(n - done, page_elems - off);
    if (to_host) DMRG_CUDA(cudaMemcpyAsync(pages[pg] + off, dev + done, m * 8, cudaMemcpyDeviceToHost, st));
    else DMRG_CUDA(cudaMemcpyAsync(dev + done, pages[pg] + off, m * 8, cudaMemcpyHostToDevice, st));
    done += m;
  }
}

static bool spill_block(dmrg_ctx* ctx, BlockSide& b, cudaStream_t st) {
  if (b.spilled) return true;
  if (!ctx->host_pool) return false;
  HostPool& hp = *ctx->host_pool;
  uint64_t elems = 0;
  for (auto& c : b.cls) if (c && c->data.p) elems += c->data.n;
  const uint64_t pe = hp.page_bytes / 8;
  if (!hp.get((size_t)((elems + pe - 1) / pe), &b.host_pages)) return false;
  b.host_n.assign(b.cls.size(), 0);
  uint64_t pos = 0;
  for (size_t i = 0; i < b.cls.size(); ++i) {
    OpClass* c = b.cls[i].get();
    if (!c || !c->data.p) continue;
    paged_copy(b.host_pages, pe, pos, c->data.p, c->data.n, true, st);
    b.host_n[i] = c->data.n;
    pos += c->data.n;
  }
  DMRG_CUDA(cudaStreamSynchronize(st));
  for (auto& c : b.cls) if (c) c->data.release();
  b.pool = ctx->host_pool; b.spilled = true;
  ++ctx->n_spills;
  return true;
}

static void fetch_block(dmrg_ctx* ctx, BlockSide& b, cudaStream_t st) {
  if (!b.spilled) return;
  const uint64_t pe = b.pool->page_bytes / 8;
  uint64_t pos = 0;
  for (size_t i = 0; i < b.cls.size(); ++i) {
    OpClass* c = b.cls[i].get();
    if (!c || !b.host_n[i]) continue;
    c->data.allocate(&ctx->al, b.host_n[i]);
    paged_copy(b.host_pages, pe, pos, c->data.p, b.host_n[i], false, st);
    pos += b.host_n[i];
  }
  DMRG_CUDA(cudaStreamSynchronize(st));
  b.pool->put(b.host_pages);
  b.pool.reset(); b.spilled = false;
  ++ctx->n_fetches;
}

// Keeps the device-resident part of the cache under its cap: the resident block farthest from the two-site problem
// at bond (kb, kb+1) the caller is heading for — left blocks measured from kb-1, right blocks from kb+2 — goes to the
// host tier, or is dropped when there is none (or it is full).  The blocks in use are never touched.
static void cache_enforce(dmrg_ctx* ctx, int kb, cudaStream_t st) {
  const uint64_t cap = env_cache_cap(ctx);
  while (true) {
    uint64_t res = 0;
    std::shared_ptr<BlockSide> far;
    bool far_left = true; int far_key = 0, far_dist = -1;
    for (int side = 0; side < 2; ++side)
      for (auto& kv : (side == 0 ? ctx->left_cache : ctx->right_cache)) {
        if (kv.second->spilled) continue;
        if (kv.second == ctx->left || kv.second == ctx->right) continue;    // in use: neither counted nor moved
        res += kv.second->bytes();
        const int dist = std::abs(kv.first - (side == 0 ? kb - 1 : kb + 2));
        if (dist > far_dist) { far_dist = dist; far = kv.second; far_left = side == 0; far_key = kv.first; }
      }
    if (res <= cap || !far) return;
    drop_presummed(*far, ctx->su2());
    if (!spill_block(ctx, *far, st)) (far_left ? ctx->left_cache : ctx->right_cache).erase(far_key);
  }
}

// kb: the bond the caller is heading for (distances decide which cached block leaves the device first)
static void cache_put(dmrg_ctx* ctx, bool left, int key, const std::shared_ptr<BlockSide>& b, cudaStream_t st, int kb) {
  (left ? ctx->left_cache : ctx->right_cache)[key] = b;
  cache_enforce(ctx, kb, st);
}

static void build_side(dmrg_ctx* ctx, bool left, int upto, cudaStream_t st, double* flops_last) {
  // left: sites 1..upto ; right: sites L..upto (descending).  Starts from the nearest cached block.
  const bool su = ctx->su2();
  std::shared_ptr<BlockSide> blk;
  int from = left ? 0 : ctx->L + 1;     // block covers sites 1..from (left) or from..L (right)
  if (left) {
    for (auto& kv : ctx->left_cache) if (kv.first <= upto && kv.first >= from) { from = kv.first; blk = kv.second; }
  } else {
    for (auto& kv : ctx->right_cache) if (kv.first >= upto && kv.first <= from) { from = kv.first; blk = kv.second; }
  }
  if (!blk) blk = su ? su2e::vacuum_block_su2(ctx, left, st) : vacuum_block(ctx, left, st);
  if (blk->spilled) {
    // make room first: the block about to come back counts as needed
    fetch_block(ctx, *blk, st);
    (left ? ctx->left : ctx->right) = blk;
    cache_enforce(ctx, left ? upto + 1 : upto - 2, st);
  }
  auto step = [&](int i) {
    std::shared_ptr<BlockSide> nb = su ? renormalize_block_su2(ctx, *blk, i, st, flops_last)
                                       : renormalize_block(ctx, *blk, i, st, flops_last);
    (left ? ctx->left : ctx->right) = nb;     // in use: the cache must not move it to the host tier
    cache_put(ctx, left, i, nb, st, left ? upto + 1 : upto - 2);   // keep what is close to the bond being prepared
    return nb;
  };
  if (left) for (int i = from + 1; i <= upto; ++i) blk = step(i);
  else for (int i = from - 1; i >= upto; --i) blk = step(i);
  (left ? ctx->left : ctx->right) = blk;
}

int dmrg_env_build(dmrg_ctx* ctx, int32_t k, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->have_integrals && !ctx->bond.empty(), DMRG_ERR_ARG, "env_build: integrals and sectors first");
  DMRG_REQUIRE(k >= 1 && k + 1 <= ctx->L, DMRG_ERR_ARG, "env_build: bond out of range");
  auto t0 = std::chrono::steady_clock::now();
  PreparedGuard guard{ctx};   // no prepared problem unless this call succeeds
  ctx->apply_plan.clear();
  if (ctx->left) drop_presummed(*ctx->left, ctx->su2());      // they may stay in the cache: carried operators only
  if (ctx->right) drop_presummed(*ctx->right, ctx->su2());
  ctx->left.reset();
  ctx->right.reset();
  double fl = 0;
  build_side(ctx, true, k - 1, st, &fl);
  build_side(ctx, false, k + 2, st, &fl);
  ctx->stats.flops_renorm = fl;
  ctx->k = k;
  if (ctx->su2()) prepare_superblock_su2(ctx, st); else prepare_superblock(ctx, st);
  ctx->stats.last_build_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  guard.ok = true;
  API_END
}

int dmrg_renormalize(dmrg_ctx* ctx, int32_t direction, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && ctx->left && ctx->right, DMRG_ERR_ARG, "renormalize: call dmrg_env_build first");
  auto t0 = std::chrono::steady_clock::now();
  const int k = ctx->k;
  double fl = 0;
  DMRG_REQUIRE(direction == 0 || direction == 1, DMRG_ERR_ARG, "renormalize: direction must be 0 or 1");
  DMRG_REQUIRE(direction == 0 ? k + 2 <= ctx->L : k - 1 >= 1, DMRG_ERR_ARG, "renormalize: already at the end of the chain");
  PreparedGuard guard{ctx};   // no prepared problem unless this call succeeds
  ctx->apply_plan.clear();
  drop_presummed(*ctx->left, ctx->su2());
  drop_presummed(*ctx->right, ctx->su2());
  if (direction == 0) {
    DMRG_REQUIRE(k + 2 <= ctx->L, DMRG_ERR_ARG, "renormalize: already at the right end");
    auto r0 = std::chrono::steady_clock::now();
    ctx->left = ctx->su2() ? renormalize_block_su2(ctx, *ctx->left, k, st, &fl) : renormalize_block(ctx, *ctx->left, k, st, &fl);
    cache_put(ctx, true, k, ctx->left, st, k + 1);
    ctx->stats.renorm_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - r0).count();
    double f2 = 0;
    ctx->right.reset();
    build_side(ctx, false, k + 3, st, &f2);
    ctx->k = k + 1;
  } else if (direction == 1) {
    DMRG_REQUIRE(k - 1 >= 1, DMRG_ERR_ARG, "renormalize: already at the left end");
    auto r0 = std::chrono::steady_clock::now();
    ctx->right = ctx->su2() ? renormalize_block_su2(ctx, *ctx->right, k + 1, st, &fl)
                            : renormalize_block(ctx, *ctx->right, k + 1, st, &fl);
    cache_put(ctx, false, k + 1, ctx->right, st, k - 1);
    ctx->stats.renorm_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - r0).count();
    double f2 = 0;
    ctx->left.reset();
    build_side(ctx, true, k - 2, st, &f2);
    ctx->k = k - 1;
  } else {
    throw Error(DMRG_ERR_ARG, "renormalize: direction must be 0 or 1");
  }
  ctx->stats.flops_renorm = fl;
  if (ctx->su2()) prepare_superblock_su2(ctx, st); else prepare_superblock(ctx, st);
  ctx->stats.last_build_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  guard.ok = true;
  API_END
}

int dmrg_psi_layout(dmrg_ctx* ctx, int32_t* nblocks, dmrg_psi_block* out, int64_t* n) {
  API_BEGIN
  DMRG_REQUIRE(ctx->k > 0, DMRG_ERR_ARG, "psi_layout: no two-site problem prepared");
  if (nblocks) *nblocks = (int32_t)ctx->psi.size();
  if (n) *n = ctx->psi_n;
  if (out) {
    const Sectors& sl = ctx->left->sec;
    const Sectors& sr = ctx->right->sec;
    for (size_t i = 0; i < ctx->psi.size(); ++i) {
      const PsiBlk& b = ctx->psi[i];
      if (ctx->su2())   // (N, 2S) labels; qR = left label of bond k+1
        out[i] = dmrg_psi_block{sl.qu[b.qL], sl.qd[b.qL], b.s1, b.s2, ctx->cfg.n_up + ctx->cfg.n_dn - sr.qu[b.qR],
                                sr.qd[b.qR], b.dL, b.dR, b.off_c, b.SLp, 0};
      else
        out[i] = dmrg_psi_block{sl.qu[b.qL], sl.qd[b.qL], b.s1, b.s2, ctx->cfg.n_up - sr.qu[b.qR],
                                ctx->cfg.n_dn - sr.qd[b.qR], b.dL, b.dR, b.off_c, 0, 0};
    }
  }
  API_END
}

// sharded contexts: sum of the ranks' disjoint psi' blocks (padded layout), through the caller's collective
static void shard_reduce(dmrg_ctx* ctx, cudaStream_t st) {
  if (ctx->shard_count <= 1 || !ctx->reduce_cb) return;
  const int rc = ctx->reduce_cb(ctx->reduce_user, ctx->psi_out_p.p, (int64_t)ctx->psi_np, (void*)st);
  DMRG_REQUIRE(rc == 0, DMRG_ERR_ARG, "heff_apply: the reduce callback of dmrg_set_shard failed");
}
// e_core.psi is added once: by every rank after a reduce, by rank 0 alone when the caller sums partial results
static double shard_e_core(const dmrg_ctx* ctx) {
  return (ctx->shard_count > 1 && !ctx->reduce_cb && ctx->shard_rank != 0) ? 0.0 : ctx->e_core;
}

// psi_out_p = H_eff psi_in_p on the padded internal buffers
static void apply_padded(dmrg_ctx* ctx, cudaStream_t st) {
  DMRG_CUDA(cudaMemsetAsync(ctx->psi_out_p.p, 0, (size_t)ctx->psi_np * 8, st));
  ++ctx->launches;
  ctx->apply_plan.run(st, &ctx->launches, ctx->ex());
  shard_reduce(ctx, st);
}

int dmrg_heff_apply(dmrg_ctx* ctx, const double* d_in, double* d_out, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_in && d_out, DMRG_ERR_ARG, "heff_apply: no problem prepared or null pointer");
  launch_pack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), d_in, ctx->psi_in_p.p, st);
  apply_padded(ctx, st);
  launch_unpack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), ctx->psi_out_p.p, d_out, shard_e_core(ctx), d_in, st);
  ctx->launches += 2;
  DMRG_CUDA(cudaGetLastError());
  API_END
}

int dmrg_heff_diag(dmrg_ctx* ctx, double* d_diag, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_diag, DMRG_ERR_ARG, "heff_diag: no problem prepared or null pointer");
  launch_unpack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), ctx->diag_p.p, d_diag, 0.0, nullptr, st);
  ++ctx->launches;
  if (ctx->e_core != 0.0) { launch_add_const(ctx->e_core, d_diag, ctx->psi_n, st); ++ctx->launches; }
  DMRG_CUDA(cudaGetLastError());
  API_END
}

// symmetric eigenproblem of the small Rayleigh-Ritz matrix (cyclic Jacobi), lowest pair
static void jacobi_lowest(std::vector<double> a, int n, double* theta, std::vector<double>* y) {
  std::vector<double> v((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) v[(size_t)i * n + i] = 1.0;
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0;
    for (int p = 0; p < n; ++p) for (int q = p + 1; q < n; ++q) off += a[(size_t)p * n + q] * a[(size_t)p * n + q];
    if (off < 1e-60) break;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) {
        double apq = a[(size_t)p * n + q];
        if (std::fabs(apq) < 1e-300) continue;
        double tau = (a[(size_t)q * n + q] - a[(size_t)p * n + p]) / (2 * apq);
        double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1 + tau * tau));
        double c = 1 / std::sqrt(1 + t * t), s = t * c;
        for (int r = 0; r < n; ++r) {
          double arp = a[(size_t)r * n + p], arq = a[(size_t)r * n + q];
          a[(size_t)r * n + p] = c * arp - s * arq;
          a[(size_t)r * n + q] = s * arp + c * arq;
        }
        for (int r = 0; r < n; ++r) {
          double apr = a[(size_t)p * n + r], aqr = a[(size_t)q * n + r];
          a[(size_t)p * n + r] = c * apr - s * aqr;
          a[(size_t)q * n + r] = s * apr + c * aqr;
        }
        for (int r = 0; r < n; ++r) {
          double vrp = v[(size_t)r * n + p], vrq = v[(size_t)r * n + q];
          v[(size_t)r * n + p] = c * vrp - s * vrq;
          v[(size_t)r * n + q] = s * vrp + c * vrq;
        }
      }
  }
  int best = 0;
  for (int i = 1; i < n; ++i) if (a[(size_t)i * n + i] < a[(size_t)best * n + best]) best = i;
  *theta = a[(size_t)best * n + best];
  y->resize(n);
  for (int i = 0; i < n; ++i) (*y)[i] = v[(size_t)i * n + best];
}

// Davidson-Liu on padded device vectors (DESIGN.md App. E).  x_p: start vector in / Ritz vector out.
static void davidson_padded(dmrg_ctx* ctx, double* x_p, double tol, int max_iter, int max_basis, double* energy,
                            int* iters, double* resid, cudaStream_t st) {
  const long long n = ctx->psi_np;
  DMRG_REQUIRE(max_basis >= 2 && max_basis <= 60 && max_iter >= 1, DMRG_ERR_ARG, "davidson: bad max_basis / max_iter");
  ctx->dav_V.allocate(&ctx->al, (size_t)n * max_basis);
  ctx->dav_W.allocate(&ctx->al, (size_t)n * max_basis);
  ctx->dav_tmp.allocate(&ctx->al, (size_t)n * 3);
  ctx->dav_small.allocate(&ctx->al, 256);
  ctx->dav_partials.allocate(&ctx->al, (size_t)DOT_BLOCKS * 64);
  double* V = ctx->dav_V.p; double* W = ctx->dav_W.p;
  double* xr = ctx->dav_tmp.p; double* hx = xr + n; double* t = hx + n;
  double* d_small = ctx->dav_small.p;
  std::vector<double> hs(64);
  auto dots = [&](const double* x, const double* Y, int m, double* out) {
    launch_multidot(x, Y, n, m, n, ctx->dav_partials.p, d_small, st);
    ctx->launches += 2;
    DMRG_CUDA(cudaMemcpyAsync(out, d_small, sizeof(double) * m, cudaMemcpyDeviceToHost, st));
    DMRG_CUDA(cudaStreamSynchronize(st));
  };
  auto applyH = [&](const double* v, double* w) {
    DMRG_CUDA(cudaMemcpyAsync(ctx->psi_in_p.p, v, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
    apply_padded(ctx, st);
    DMRG_CUDA(cudaMemcpyAsync(w, ctx->psi_out_p.p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
    if (ctx->e_core != 0.0) { launch_axpy(ctx->e_core, v, w, n, st); ++ctx->launches; }
  };
  // v1 = x / |x|
  double nrm2;
  dots(x_p, x_p, 1, &nrm2);
  DMRG_REQUIRE(nrm2 > 0, DMRG_ERR_INPUT, "davidson: zero start vector");
  DMRG_CUDA(cudaMemcpyAsync(V, x_p, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
  launch_scale(1.0 / std::sqrt(nrm2), V, n, st); ++ctx->launches;
  applyH(V, W);
  int m = 1, napply = 1;
  std::vector<double> G((size_t)max_basis * max_basis, 0.0);
  dots(W, V, 1, hs.data());
  G[0] = hs[0];
  double theta = G[0], rn = 0;
  std::vector<double> y;
  while (true) {
    std::vector<double> Gm((size_t)m * m);
    for (int i = 0; i < m; ++i) for (int j = 0; j < m; ++j) Gm[(size_t)i * m + j] = 0.5 * (G[(size_t)i * max_basis + j] + G[(size_t)j * max_basis + i]);
    jacobi_lowest(Gm, m, &theta, &y);
    DMRG_CUDA(cudaMemcpyAsync(d_small + 64, y.data(), sizeof(double) * m, cudaMemcpyHostToDevice, st));
    launch_combine(V, n, d_small + 64, m, n, xr, st);
    launch_combine(W, n, d_small + 64, m, n, hx, st);
    double* r = ctx->psi_in_p.p;   // scratch: overwritten by the next apply anyway
    launch_residual_precond(xr, hx, ctx->diag_p.p, theta, theta - ctx->e_core, r, t, n, st);
    ctx->launches += 3;
    double r2;
    dots(r, r, 1, &r2);
    rn = std::sqrt(r2);
    if (rn <= tol || napply >= max_iter) break;
    if (m >= max_basis) {   // restart with the Ritz vector
      double x2;
      dots(xr, xr, 1, &x2);
      double sc = 1.0 / std::sqrt(x2);
      DMRG_CUDA(cudaMemcpyAsync(V, xr, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
      DMRG_CUDA(cudaMemcpyAsync(W, hx, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
      launch_scale(sc, V, n, st); launch_scale(sc, W, n, st); ctx->launches += 2;
      m = 1;
      G[0] = theta;
    }
    for (int pass = 0; pass < 2; ++pass) {   // classical Gram-Schmidt, twice
      dots(t, V, m, hs.data());
      DMRG_CUDA(cudaMemcpyAsync(d_small + 128, hs.data(), sizeof(double) * m, cudaMemcpyHostToDevice, st));
      launch_project_out(V, n, d_small + 128, m, n, t, st); ++ctx->launches;
    }
    double t2;
    dots(t, t, 1, &t2);
    if (std::sqrt(t2) < 1e-14) break;
    double* vn = V + (size_t)m * n; double* wn = W + (size_t)m * n;
    DMRG_CUDA(cudaMemcpyAsync(vn, t, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
    launch_scale(1.0 / std::sqrt(t2), vn, n, st); ++ctx->launches;
    applyH(vn, wn);
    ++napply;
    dots(wn, V, m + 1, hs.data());
    for (int i = 0; i <= m; ++i) G[(size_t)i * max_basis + m] = G[(size_t)m * max_basis + i] = hs[i];
    ++m;
  }
  double x2;
  dots(xr, xr, 1, &x2);
  DMRG_CUDA(cudaMemcpyAsync(x_p, xr, (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
  launch_scale(1.0 / std::sqrt(x2), x_p, n, st); ++ctx->launches;
  DMRG_CUDA(cudaStreamSynchronize(st));
  *energy = theta; *iters = napply; *resid = rn;
}

int dmrg_davidson(dmrg_ctx* ctx, double* d_psi, double tol, int32_t max_iter, int32_t max_basis, double* h_energy,
                  int32_t* h_iters, double* h_resid, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_psi && h_energy && h_iters && h_resid, DMRG_ERR_ARG, "davidson: bad arguments");
  DMRG_REQUIRE(ctx->shard_count <= 1 || ctx->reduce_cb, DMRG_ERR_ARG, "davidson: a sharded context needs the reduce callback");
  DevArray<double> xp;
  xp.allocate(&ctx->al, (size_t)ctx->psi_np);
  DMRG_CUDA(cudaMemsetAsync(xp.p, 0, (size_t)ctx->psi_np * 8, st));
  launch_pack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), d_psi, xp.p, st); ++ctx->launches;
  int it = 0;
  davidson_padded(ctx, xp.p, tol, max_iter, max_basis, h_energy, &it, h_resid, st);
  *h_iters = it;
  launch_unpack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), xp.p, d_psi, 0.0, nullptr, st); ++ctx->launches;
  DMRG_CUDA(cudaStreamSynchronize(st));
  API_END
}

int dmrg_heff_apply_host(dmrg_ctx* ctx, const double* h_in, double* h_out, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && h_in && h_out, DMRG_ERR_ARG, "heff_apply_host: bad arguments");
  DevArray<double> a, b;
  a.allocate(&ctx->al, (size_t)ctx->psi_n);
  b.allocate(&ctx->al, (size_t)ctx->psi_n);
  DMRG_CUDA(cudaMemcpyAsync(a.p, h_in, (size_t)ctx->psi_n * 8, cudaMemcpyHostToDevice, st));
  int rc = dmrg_heff_apply(ctx, a.p, b.p, stream);
  if (rc != DMRG_OK) return rc;
  DMRG_CUDA(cudaMemcpyAsync(h_out, b.p, (size_t)ctx->psi_n * 8, cudaMemcpyDeviceToHost, st));
  DMRG_CUDA(cudaStreamSynchronize(st));
  API_END
}

int dmrg_davidson_host(dmrg_ctx* ctx, double* h_psi, double tol, int32_t max_iter, int32_t max_basis, double* h_energy,
                       int32_t* h_iters, double* h_resid, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && h_psi, DMRG_ERR_ARG, "davidson_host: bad arguments");
  DevArray<double> a;
  a.allocate(&ctx->al, (size_t)ctx->psi_n);
  DMRG_CUDA(cudaMemcpyAsync(a.p, h_psi, (size_t)ctx->psi_n * 8, cudaMemcpyHostToDevice, st));
  int rc = dmrg_davidson(ctx, a.p, tol, max_iter, max_basis, h_energy, h_iters, h_resid, stream);
  if (rc != DMRG_OK) return rc;
  DMRG_CUDA(cudaMemcpyAsync(h_psi, a.p, (size_t)ctx->psi_n * 8, cudaMemcpyDeviceToHost, st));
  DMRG_CUDA(cudaStreamSynchronize(st));
  API_END
}

int dmrg_set_shard(dmrg_ctx* ctx, int32_t rank, int32_t count, dmrg_reduce_fn reduce, void* user) {
  API_BEGIN
  DMRG_REQUIRE(count >= 1 && rank >= 0 && rank < count, DMRG_ERR_ARG, "set_shard: need 0 <= rank < count");
  ctx->shard_rank = rank;
  ctx->shard_count = count;
  ctx->reduce_cb = count > 1 ? reduce : nullptr;
  ctx->reduce_user = user;
  // a prepared problem belongs to the old sharding
  ctx->k = 0;
  ctx->apply_plan.clear();
  API_END
}

int dmrg_shard_info(dmrg_ctx* ctx, int32_t* h_owner, double* h_flops) {
  API_BEGIN
  DMRG_REQUIRE(ctx->k > 0, DMRG_ERR_ARG, "shard_info: no problem prepared");
  if (h_owner) for (size_t i = 0; i < ctx->psi.size(); ++i) h_owner[i] = ctx->psi_owner[i];
  if (h_flops) for (int r = 0; r < ctx->shard_count; ++r) h_flops[r] = r < (int)ctx->shard_flops.size() ? ctx->shard_flops[r] : 0.0;
  API_END
}

int dmrg_block_flops(dmrg_ctx* ctx, double* h_flops) {
  API_BEGIN
  DMRG_REQUIRE(ctx->k > 0 && h_flops && ctx->blk_flops.size() == ctx->psi.size(), DMRG_ERR_ARG, "block_flops: no problem prepared");
  for (size_t i = 0; i < ctx->psi.size(); ++i) h_flops[i] = ctx->blk_flops[i];
  API_END
}

int dmrg_stats(dmrg_ctx* ctx, dmrg_stats_t* out) {
  API_BEGIN
  DMRG_REQUIRE(out, DMRG_ERR_ARG, "stats: null pointer");
  ctx->stats.total_launches = ctx->launches;
  ctx->stats.env_spills = ctx->n_spills;
  ctx->stats.env_fetches = ctx->n_fetches;
  ctx->stats.env_host_bytes = ctx->host_pool ? (double)ctx->host_pool->total : 0.0;
  ctx->stats.env_device_bytes = (double)ctx->cache_bytes();
  *out = ctx->stats;
  API_END
}

int dmrg_env_export(dmrg_ctx* ctx, int32_t side, int32_t kind, int32_t i, int32_t j, double* h_out, int64_t* Dout) {
  API_BEGIN
  DMRG_REQUIRE(ctx->k > 0 && (side == 0 || side == 1) && kind >= 0 && kind <= 10, DMRG_ERR_ARG, "env_export: bad arguments");
  DMRG_REQUIRE(!ctx->su2(), DMRG_ERR_UNSUPPORTED, "env_export: U(1)xU(1) contexts only");
  const BlockSide& B = side == 0 ? *ctx->left : *ctx->right;
  static const int kmap[11] = {K_H, K_CU, K_CD, K_AUU, K_AUD, K_ADD, K_BUU, K_BUD, K_BDD, K_SU, K_SD};
  const int kk = kmap[kind];
  const OpClass& C = *B.cls[kk];
  const int n = B.norb();
  int idx = 0;
  auto inb = [&](int o) { return o >= B.lo && o < B.hi; };
  switch (kk) {
    case K_H: idx = 0; break;
    case K_CU: case K_CD: DMRG_REQUIRE(inb(i), DMRG_ERR_ARG, "env_export: orbital not in block"); idx = i - B.lo; break;
    case K_AUU: case K_ADD:
      DMRG_REQUIRE(inb(i) && inb(j) && i < j, DMRG_ERR_ARG, "env_export: need i<j in block");
      idx = (i - B.lo) * n - (i - B.lo) * (i - B.lo + 1) / 2 + (j - i - 1); break;
    case K_SU: case K_SD:
      DMRG_REQUIRE(i >= 0 && i < ctx->L && !inb(i), DMRG_ERR_ARG, "env_export: orbital must be outside the block");
      idx = B.is_left ? i - B.hi : i; break;
    default: DMRG_REQUIRE(inb(i) && inb(j), DMRG_ERR_ARG, "env_export: orbitals not in block"); idx = (i - B.lo) * n + (j - B.lo);
  }
  const long long D = B.sec.total();
  if (Dout) *Dout = D;
  if (h_out) {
    std::vector<long long> start(B.sec.size());
    long long o = 0;
    for (int s = 0; s < B.sec.size(); ++s) { start[s] = o; o += B.sec.dim[s]; }
    std::fill(h_out, h_out + D * D, 0.0);
    for (size_t b = 0; b < C.blocks.size(); ++b) {
      const ClsBlock& cb = C.blocks[b];
      std::vector<double> h((size_t)cb.rp * cb.cp);
      DMRG_CUDA(cudaMemcpy(h.data(), C.ptr((int)b, idx), h.size() * 8, cudaMemcpyDeviceToHost));
      for (int r = 0; r < cb.rows; ++r)
        for (int c = 0; c < cb.cols; ++c)
          h_out[(start[cb.so] + r) * D + start[cb.si] + c] = h[(size_t)r * cb.cp + c];
    }
  }
  API_END
}

int dmrg_env_export_block(dmrg_ctx* ctx, int32_t side, int32_t kind, int32_t d2S, int32_t qa, int32_t qb, int32_t* nops,
                          int32_t* rows, int32_t* cols, double* h_out) {
  API_BEGIN
  DMRG_REQUIRE(ctx->k > 0 && side >= 0 && side <= 3 && nops && rows && cols, DMRG_ERR_ARG, "env_export_block: bad arguments");
  const BlockSide* Bp = side == 0 ? ctx->left.get() : side == 1 ? ctx->right.get() : nullptr;
  if (side >= 2) {
    auto& cache = side == 2 ? ctx->left_cache : ctx->right_cache;
    auto f = cache.find(side == 2 ? ctx->k - 2 : ctx->k + 3);
    DMRG_REQUIRE(f != cache.end() && !f->second->spilled, DMRG_ERR_ARG,
                 "env_export_block: the predecessor block is not in the device tier of the environment cache");
    Bp = f->second.get();
    side -= 2;
  }
  const BlockSide& B = *Bp;
  const OpClass* C = nullptr;
  int ca = qa, cb = qb;     // the block's own content
  if (ctx->su2()) {
    DMRG_REQUIRE(kind >= 0 && kind <= 6, DMRG_ERR_ARG, "env_export_block: kind out of range");
    const auto& kr = B.kinds[kind + 1];                 // su2e::SKind without SK_ID
    DMRG_REQUIRE(d2S >= -kr.k2 && d2S <= kr.k2 && !((d2S + kr.k2) & 1), DMRG_ERR_ARG, "env_export_block: d2S is not a spin change of this kind");
    C = B.cls[kr.cids[(d2S + kr.k2) / 2]].get();
    if (side == 1) ca = ctx->cfg.n_up + ctx->cfg.n_dn - qa;
  } else {
    static const int kmap[11] = {K_H, K_CU, K_CD, K_AUU, K_AUD, K_ADD, K_BUU, K_BUD, K_BDD, K_SU, K_SD};
    DMRG_REQUIRE(kind >= 0 && kind <= 10, DMRG_ERR_ARG, "env_export_block: kind out of range");
    C = B.cls[kmap[kind]].get();
    if (side == 1) { ca = ctx->cfg.n_up - qa; cb = ctx->cfg.n_dn - qb; }
  }
  DMRG_REQUIRE(C && C->data.p, DMRG_ERR_ARG, "env_export_block: class not resident");
  *nops = C->nops; *rows = 0; *cols = 0;
  const int si = B.sec.find(ca, cb);
  const int b = si >= 0 ? C->blk_of_in[si] : -1;
  if (b < 0) return DMRG_OK;
  const ClsBlock& cb_ = C->blocks[b];
  *rows = cb_.rows; *cols = cb_.cols;
  if (h_out && C->nops > 0) {
    std::vector<double> h((size_t)C->nops * cb_.rp * cb_.cp);
    DMRG_CUDA(cudaMemcpy(h.data(), C->ptr(b, 0), h.size() * 8, cudaMemcpyDeviceToHost));
    for (int o = 0; o < C->nops; ++o)
      for (int r = 0; r < cb_.rows; ++r)
        std::memcpy(h_out + ((size_t)o * cb_.rows + r) * cb_.cols, h.data() + ((size_t)o * cb_.rp + r) * cb_.cp,
                    sizeof(double) * cb_.cols);
  }
  API_END
}

int dmrg_apply_profile(dmrg_ctx* ctx, const double* d_in, double* d_out, int32_t cap, dmrg_launch_info* h_out,
                       int32_t* n, void* stream) {
  API_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_in && d_out && n, DMRG_ERR_ARG, "apply_profile: bad arguments");
  launch_pack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), d_in, ctx->psi_in_p.p, st);
  DMRG_CUDA(cudaMemsetAsync(ctx->psi_out_p.p, 0, (size_t)ctx->psi_np * 8, st));
  std::vector<LaunchRecord> rec;
  ctx->apply_plan.run_profiled(st, &rec);
  shard_reduce(ctx, st);
  launch_unpack(ctx->d_psi_blocks.p, (int)ctx->psi.size(), ctx->psi_out_p.p, d_out, shard_e_core(ctx), d_in, st);
  ctx->launches += 3 + (int64_t)rec.size();
  DMRG_CUDA(cudaStreamSynchronize(st));
  *n = (int32_t)rec.size();
  for (int i = 0; i < (int)rec.size() && i < cap && h_out; ++i)
    h_out[i] = dmrg_launch_info{rec[i].chunk, rec[i].phase, rec[i].shape, rec[i].ntiles, rec[i].flops, (double)rec[i].ms};
  API_END
}

int dmrg_su2_f_factor(int32_t twoSa, int32_t twoSk, int32_t twoSg, int32_t twokL, int32_t twokk, int32_t twok,
               int32_t twoSa_out, int32_t twoSk_out, int32_t twoSg_out, double* h_F_ninej, double* h_F_contraction) {
  if (!h_F_ninej || !h_F_contraction) return DMRG_ERR_ARG;
  *h_F_ninej = su2::F_ninej(twoSa, twoSk, twoSg, twokL, twokk, twok, twoSa_out, twoSk_out, twoSg_out);
  // the same factor from the library's own contraction (su2::phi_blocking) for site spins 0 / 1/2 is not a
  // product form; here: direct sum over magnetic quantum numbers with the library's CG table
  double tot = 0.0;
  for (int Mg_ = -twoSg_out; Mg_ <= twoSg_out; Mg_ += 2)
    for (int q = -twok; q <= twok; q += 2) {
      const int Mg = Mg_ - q;
      const double wo = su2::cg(twoSg, Mg, twok, q, twoSg_out, Mg_);
      if (wo == 0.0) continue;
      for (int qL = -twokL; qL <= twokL; qL += 2) {
        const int qk = q - qL;
        const double cop = su2::cg(twokL, qL, twokk, qk, twok, q);
        if (cop == 0.0) continue;
        for (int Ma = -twoSa; Ma <= twoSa; Ma += 2) {
          const int Mk = Mg - Ma;
          const double cin = su2::cg(twoSa, Ma, twoSk, Mk, twoSg, Mg);
          if (cin == 0.0) continue;
          tot += wo * cop * cin * su2::cg(twoSa_out, Ma + qL, twoSk_out, Mk + qk, twoSg_out, Mg_) *
                 su2::cg(twoSa, Ma, twokL, qL, twoSa_out, Ma + qL) * su2::cg(twoSk, Mk, twokk, qk, twoSk_out, Mk + qk);
        }
      }
    }
  *h_F_contraction = tot / (twoSg_out + 1);
  return DMRG_OK;
}

int dmrg_fp64_peak(dmrg_ctx* ctx, double* h_tflops, void* stream) {
  API_BEGIN
  DMRG_REQUIRE(h_tflops, DMRG_ERR_ARG, "fp64_peak: null pointer");
  DevArray<double> scratch;
  scratch.allocate(&ctx->al, 64);
  DMRG_CUDA(measure_dmma_peak(scratch.p, h_tflops, (cudaStream_t)stream));
  ctx->launches += 2;
  API_END
}

int dmrg_dfma_peak(dmrg_ctx* ctx, double* h_tflops, void* stream) {
  API_BEGIN
  DMRG_REQUIRE(h_tflops, DMRG_ERR_ARG, "dfma_peak: null pointer");
  DevArray<double> scratch;
  scratch.allocate(&ctx->al, 64);
  DMRG_CUDA(measure_dfma_peak(scratch.p, h_tflops, (cudaStream_t)stream));
  ctx->launches += 2;
  API_END
}

}  // extern "C"
