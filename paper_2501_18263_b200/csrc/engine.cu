#include "engine.h"
#include "su2.h"

#include <algorithm>
#include <chrono>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <set>
#include <tuple>
#include <unordered_map>

namespace dmrg {

// ------------------------------------------------------------------------------------------------
// class storage
// ------------------------------------------------------------------------------------------------
void OpClass::layout(const Sectors& sec, int du_, int dd_, int nops_) {
  du = du_; dd = dd_; nops = nops_;
  nalloc = pad8(std::max(nops, 1));   // whole multiples of 8 operators: a class block is a valid GEMM operand
  blocks.clear();
  blk_of_in.assign(sec.size(), -1);
  blk_of_out.assign(sec.size(), -1);
  long long off = 0;
  for (int si = 0; si < sec.size(); ++si) {
    int so = sec.find(sec.qu[si] + du, sec.qd[si] + dd);
    if (so < 0) continue;
    ClsBlock b{so, si, sec.dim[so], sec.dim[si], pad8(sec.dim[so]), pad8(sec.dim[si]), off};
    off += (long long)nalloc * b.rp * b.cp;
    blk_of_in[si] = (int)blocks.size();
    blk_of_out[so] = (int)blocks.size();
    blocks.push_back(b);
  }
  elems = off;
}

void OpClass::allocate(Allocator* al, cudaStream_t st) {
  data.allocate(al, (size_t)std::max<long long>(elems, 8));
  DMRG_CUDA(cudaMemsetAsync(data.p, 0, (size_t)std::max<long long>(elems, 8) * 8, st));
}

// ------------------------------------------------------------------------------------------------
// site operators (4x4, rows = out state); |3> = a+_up a+_dn |0>
// ------------------------------------------------------------------------------------------------
static void site_elem(bool cre, int spin, double* m) {
  std::memset(m, 0, 16 * sizeof(double));
  if (spin == 0) { m[2 * 4 + 0] = 1.0; m[3 * 4 + 1] = 1.0; }     // a+_up : 0->up, dn->updn
  else           { m[1 * 4 + 0] = 1.0; m[3 * 4 + 2] = -1.0; }    // a+_dn : 0->dn, up-> -updn
  if (!cre) {
    double t[16];
    for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) t[r * 4 + c] = m[c * 4 + r];
    std::memcpy(m, t, sizeof(t));
  }
}
static void mat4_mul(const double* a, const double* b, double* c) {
  double t[16];
  for (int r = 0; r < 4; ++r)
    for (int q = 0; q < 4; ++q) {
      double s = 0;
      for (int k = 0; k < 4; ++k) s += a[r * 4 + k] * b[k * 4 + q];
      t[r * 4 + q] = s;
    }
  std::memcpy(c, t, sizeof(t));
}

SiteOpTable::SiteOpTable() {
  std::array<double, 16> id{};
  for (int i = 0; i < 4; ++i) id[i * 4 + i] = 1.0;
  mats.push_back(id);
}
int SiteOpTable::intern(const double* m) {
  bool zero = true;
  for (int i = 0; i < 16; ++i) if (m[i] != 0.0) zero = false;
  if (zero) return -1;
  for (size_t i = 0; i < mats.size(); ++i)
    if (std::memcmp(mats[i].data(), m, 16 * sizeof(double)) == 0) return (int)i;
  std::array<double, 16> a;
  std::memcpy(a.data(), m, sizeof(double) * 16);
  mats.push_back(a);
  return (int)mats.size() - 1;
}
int SiteOpTable::parity(int id) const {
  for (int r = 0; r < 4; ++r)
    for (int c = 0; c < 4; ++c)
      if (mats[id][r * 4 + c] != 0.0)
        return (SITE_QU[r] + SITE_QD[r] - SITE_QU[c] - SITE_QD[c]) & 1;
  return 0;
}

// product of the elementary site operators in `ops` (leftmost first); returns interned id or -1.
// All strings of up to four elementary operators are interned when the table is built, so this is a
// read-only lookup (the term enumeration calls it from several threads).
static inline int site_code(const EOp* ops, int n) {
  int code = 0, base = 0;
  for (int i = 0; i < n; ++i) { code |= ((ops[i].cre ? 2 : 0) | ops[i].spin) << (2 * i); base = base * 4 + 1; }
  return base + code;      // base = (4^n - 1) / 3
}
static int site_product_slow(SiteOpTable& tab, const EOp* ops, int n) {
  double m[16];
  std::memset(m, 0, sizeof(m));
  for (int i = 0; i < 4; ++i) m[i * 4 + i] = 1.0;
  for (int i = 0; i < n; ++i) {
    double e[16];
    site_elem(ops[i].cre, ops[i].spin, e);
    mat4_mul(m, e, m);
  }
  return tab.intern(m);
}
void SiteOpTable::build_products() {
  prod.assign(341, -1);
  for (int n = 0; n <= 4; ++n)
    for (int c = 0; c < (1 << (2 * n)); ++c) {
      EOp ops[4];
      for (int i = 0; i < n; ++i) { int b = (c >> (2 * i)) & 3; ops[i] = EOp{(b & 2) != 0, 0, b & 1}; }
      prod[site_code(ops, n)] = site_product_slow(*this, ops, n);
    }
}
static inline int site_product(const SiteOpTable& tab, const EOp* ops, int n) { return tab.prod[site_code(ops, n)]; }

// ------------------------------------------------------------------------------------------------
// naming of block operators
// ------------------------------------------------------------------------------------------------
static int nops_of(const BlockSide& B, int kind, int L) {
  const int n = B.norb();
  switch (kind) {
    case K_ID: case K_H: return 1;
    case K_CU: case K_CD: return n;
    case K_AUU: case K_ADD: return n * (n - 1) / 2;
    case K_AUD: case K_BUU: case K_BUD: case K_BDD: return n * n;
    case K_SU: case K_SD: return B.is_left ? (L - B.hi) : B.lo;
  }
  return 0;
}
static const int KIND_DU[K_NSTD] = {0, 0, 1, 0, 2, 1, 0, 0, 1, 0, -1, 0};
static const int KIND_DD[K_NSTD] = {0, 0, 0, 1, 0, 1, 2, 0, -1, 0, 0, -1};

static inline int idx_tri(const BlockSide& B, int i, int j) {   // i < j
  int a = i - B.lo, b = j - B.lo, n = B.norb();
  return a * n - a * (a + 1) / 2 + (b - a - 1);
}
static inline int idx_sq(const BlockSide& B, int i, int j) { return (i - B.lo) * B.norb() + (j - B.lo); }
static inline int idx_S(const BlockSide& B, int x) { return B.is_left ? x - B.hi : x; }

// Names the product ops[0] ops[1] .. (all orbitals inside B).  Returns 0 ok, 1 vanishes, 2 too long.
static int name_block_ops(const BlockSide& B, const EOp* ops, int n, OpRef& ref, double& sign) {
  sign = 1.0;
  ref = OpRef{};
  if (n == 0) { ref.cls = K_ID; ref.idx = 0; return 0; }
  if (n == 1) {
    ref.cls = ops[0].spin == 0 ? K_CU : K_CD;
    ref.idx = ops[0].orb - B.lo;
    ref.tr = !ops[0].cre;
    return 0;
  }
  if (n > 2) return 2;
  EOp p = ops[0], q = ops[1];
  if (p.cre == q.cre) {       // a+ a+  or  a a = (a+_q a+_p)^T
    bool tr = !p.cre;
    if (tr) std::swap(p, q);  // now the string is a+_p a+_q
    if (p.spin == q.spin) {
      if (p.orb == q.orb) return 1;
      ref.cls = p.spin == 0 ? K_AUU : K_ADD;
      if (p.orb < q.orb) ref.idx = idx_tri(B, p.orb, q.orb);
      else { ref.idx = idx_tri(B, q.orb, p.orb); sign = -1.0; }
    } else if (p.spin == 0) {
      ref.cls = K_AUD; ref.idx = idx_sq(B, p.orb, q.orb);
    } else {                  // a+_{i dn} a+_{j up} = - a+_{j up} a+_{i dn}
      ref.cls = K_AUD; ref.idx = idx_sq(B, q.orb, p.orb); sign = -1.0;
    }
    ref.tr = tr;
    return 0;
  }
  if (!p.cre) return 2;       // a a+ never appears in a normal-ordered string
  if (p.spin == q.spin) {
    ref.cls = p.spin == 0 ? K_BUU : K_BDD; ref.idx = idx_sq(B, p.orb, q.orb);
  } else if (p.spin == 0) {
    ref.cls = K_BUD; ref.idx = idx_sq(B, p.orb, q.orb);
  } else {                    // a+_{i dn} a_{j up} = (a+_{j up} a_{i dn})^T
    ref.cls = K_BUD; ref.idx = idx_sq(B, q.orb, p.orb); ref.tr = true;
  }
  return 0;
}

// ------------------------------------------------------------------------------------------------
// runs and pre-summation
// ------------------------------------------------------------------------------------------------
struct Entry { int a, b; double c; };            // a: partner / destination index, b: source operator
struct Run { int a0, b0, cnt; double c; };

static std::vector<Run> make_runs(std::vector<Entry> e, const std::set<int>* cuts = nullptr) {
  std::sort(e.begin(), e.end(), [](const Entry& x, const Entry& y) { return x.a != y.a ? x.a < y.a : x.b < y.b; });
  std::vector<Run> r;
  for (const Entry& x : e) {
    if (!r.empty()) {
      Run& l = r.back();
      if (x.a == l.a0 + l.cnt && x.b == l.b0 + l.cnt && x.c == l.c && !(cuts && cuts->count(x.a))) {
        ++l.cnt;
        continue;
      }
    }
    r.push_back(Run{x.a, x.b, 1, x.c});
  }
  return r;
}

// K[x] = sum_b W[x][b] * src[b] for the distinct partner indices x of `e` (sorted).  Creates the class
// (same block structure as src), queues the stacked GEMMs, rewrites e as (a, K index, 1).
struct Presummer {
  dmrg_ctx* ctx;
  cudaStream_t st;
  Planner planner;
  std::vector<DevArray<double>> coefs;
  Presummer(dmrg_ctx* c, cudaStream_t s) : ctx(c), st(s), planner(&c->al, ~0ull >> 8) {}
  std::unique_ptr<OpClass> make(const Sectors& sec, const OpClass& src, std::vector<Entry>& e) {
    std::vector<int> rows;
    for (auto& x : e) rows.push_back(x.a);
    std::sort(rows.begin(), rows.end());
    rows.erase(std::unique(rows.begin(), rows.end()), rows.end());
    auto K = std::make_unique<OpClass>();
    K->kind = K_NSTD;
    K->layout(sec, src.du, src.dd, (int)rows.size());
    K->allocate(&ctx->al, st);
    const int Mp = K->nalloc, Kp = src.nalloc;
    std::vector<double> W((size_t)Mp * Kp, 0.0);
    for (auto& x : e) {
      int r = (int)(std::lower_bound(rows.begin(), rows.end(), x.a) - rows.begin());
      W[(size_t)r * Kp + x.b] += x.c;
    }
    coefs.emplace_back();
    coefs.back().upload(&ctx->al, W, st);
    for (size_t b = 0; b < K->blocks.size(); ++b) {
      const ClsBlock& kb = K->blocks[b];
      int sb = src.blk_of_in[kb.si];
      const int N = kb.rp * kb.cp;
      Item it;
      it.C = K->ptr((int)b, 0); it.ldc = N; it.strideC = 0; it.count = 1; it.alpha = 1.0; it.nmat = 2;
      it.X = Mat{coefs.back().p, Kp, false, 0, Mp, Kp, (int)rows.size(), src.nops};
      it.Y = Mat{src.ptr(sb, 0), N, false, 0, Kp, N, src.nops, kb.rows * kb.cols};
      planner.add(it);
    }
    std::vector<Entry> out;
    for (size_t r = 0; r < rows.size(); ++r) out.push_back(Entry{rows[r], (int)r, 1.0});
    e.swap(out);
    return K;
  }
  void run() {
    Plan p;
    planner.finish(&p, st);
    p.run(st, &ctx->launches, ctx->ex());
    DMRG_CUDA(cudaStreamSynchronize(st));
    coefs.clear();
  }
};

// ------------------------------------------------------------------------------------------------
// helpers shared by the renormalisation step and the two-site problem
// ------------------------------------------------------------------------------------------------
static inline double W4(const dmrg_ctx* c, int i, int j, int k, int l) {
  const int L = c->L;
  return c->w[(((size_t)i * L + j) * L + k) * L + l];
}
static inline double T2(const dmrg_ctx* c, int i, int j) { return c->T[(size_t)i * c->L + j]; }

static void fill_identity(OpClass& id, cudaStream_t st) {
  std::vector<double> h((size_t)id.elems, 0.0);
  for (auto& b : id.blocks)
    for (int r = 0; r < b.rows; ++r) h[(size_t)b.off + (size_t)r * b.cp + r] = 1.0;
  if (!h.empty()) DMRG_CUDA(cudaMemcpyAsync(id.data.p, h.data(), h.size() * 8, cudaMemcpyHostToDevice, st));
}

static void layout_standard(dmrg_ctx* ctx, BlockSide& B, cudaStream_t st) {
  B.cls.clear();
  for (int k = 0; k < K_NSTD; ++k) {
    auto c = std::make_unique<OpClass>();
    c->kind = k;
    c->layout(B.sec, KIND_DU[k], KIND_DD[k], nops_of(B, k, ctx->L));
    c->allocate(&ctx->al, st);
    B.cls.push_back(std::move(c));
  }
  fill_identity(*B.cls[K_ID], st);
}

std::unique_ptr<BlockSide> vacuum_block(dmrg_ctx* ctx, bool is_left, cudaStream_t st) {
  auto B = std::make_unique<BlockSide>();
  B->is_left = is_left;
  B->lo = B->hi = is_left ? 0 : ctx->L;
  B->sec.add(0, 0, 1);
  layout_standard(ctx, *B, st);
  return B;
}

// Workspace cap for the O_L.psi intermediates: the caller's, else 40 % of the device memory this context
// has not allocated itself (1..64 GB).  Fewer, larger chunks mean fewer under-filled launch tails per
// apply.  (cudaMemGetInfo is no guide here: the caller's allocator may cache freed blocks.)
static uint64_t workspace_cap(const dmrg_ctx* ctx) {
  if (ctx->cfg.workspace_bytes) return ctx->cfg.workspace_bytes;
  size_t fr = 0, tot = 0;
  if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) return 16ull << 30;
  // the context's workspace arena is what the cap is about: it does not count as memory taken (while no plan holds it)
  const uint64_t arena = ctx->ws_arena.in_use ? 0 : 8ull * ctx->ws_arena.buf.n;
  const uint64_t mine = ctx->al.live_bytes > arena ? ctx->al.live_bytes - arena : 0;
  const uint64_t rest = tot > mine ? tot - mine : 0;
  const uint64_t cap = std::min<uint64_t>(std::max<uint64_t>(rest / 5 * 2, 1ull << 30), 64ull << 30);
  // an arena of 60-100 % of that is kept as it is: plans are then cut to fit it and it is never reallocated in a sweep
  if (arena >= cap / 5 * 3 && arena <= cap) return arena;
  return cap;
}

static inline uint64_t pack_key(int a, int b, int c, int d, int e, int f) {
  return ((uint64_t)a << 40) | ((uint64_t)b << 28) | ((uint64_t)c << 22) | ((uint64_t)d << 10) |
         ((uint64_t)e << 9) | (uint64_t)f;
}

// ------------------------------------------------------------------------------------------------
// renormalisation step: operators of old (+) site, projected by the MPS tensor
// ------------------------------------------------------------------------------------------------
std::unique_ptr<BlockSide> renormalize_block(dmrg_ctx* ctx, const BlockSide& old, int site,
                                             cudaStream_t st, double* flops_out) {
  const int L = ctx->L;
  const bool left = old.is_left;
  const int s_orb = site - 1;
  DMRG_REQUIRE(left ? (old.hi == s_orb) : (old.lo == s_orb + 1), DMRG_ERR_ARG, "renormalize: site not adjacent");
  const SiteTensor& A = ctx->site[site];
  DMRG_REQUIRE(A.canonical == (left ? 0 : 1), DMRG_ERR_ARG,
               "renormalize: site tensor " + std::to_string(site) + " missing or of the wrong canonical form");
  auto nb = std::make_unique<BlockSide>();
  BlockSide& B = *nb;
  B.is_left = left;
  B.lo = left ? old.lo : s_orb;
  B.hi = left ? s_orb + 1 : old.hi;
  const Sectors& bsec = ctx->bond[left ? site : site - 1];
  for (int i = 0; i < bsec.size(); ++i) {
    if (left) B.sec.add(bsec.qu[i], bsec.qd[i], bsec.dim[i]);
    else B.sec.add(ctx->cfg.n_up - bsec.qu[i], ctx->cfg.n_dn - bsec.qd[i], bsec.dim[i]);
  }
  layout_standard(ctx, B, st);

  PhaseTimer pt("renormalize");
  // ---- contributions: new operator = sum coef * (old operator (x) site operator) ----
  std::unordered_map<uint64_t, double> acc;
  auto in_old = [&](int orb) { return orb >= old.lo && orb < old.hi; };
  auto add_named = [&](int dk, int di, OpRef src, int sop, double coef) {
    if (sop < 0 || coef == 0.0) return;
    acc[pack_key(dk, di, src.cls, src.idx, src.tr ? 1 : 0, sop)] += coef;
  };
  auto add_ops = [&](int dk, int di, const EOp* ops, int n, double coef) {
    EOp bo[4], so[4];
    int nb_ = 0, ns = 0, inv = 0;
    for (int i = 0; i < n; ++i) {
      if (in_old(ops[i].orb)) { bo[nb_++] = ops[i]; if (!left) inv += 0; if (left) inv += ns; }
      else { so[ns++] = ops[i]; if (!left) inv += nb_; }
    }
    OpRef src; double sg;
    int rc = name_block_ops(old, bo, nb_, src, sg);
    if (rc == 1) return;
    DMRG_REQUIRE(rc == 0, DMRG_ERR_ARG, "internal: unnamed block operator string");
    int sop = site_product(ctx->site_ops, so, ns);
    add_named(dk, di, src, sop, coef * sg * ((inv & 1) ? -1.0 : 1.0));
  };
  std::vector<int> orbs;
  for (int i = B.lo; i < B.hi; ++i) orbs.push_back(i);
  // normal operators
  for (int i : orbs)
    for (int s = 0; s < 2; ++s) {
      EOp o[1] = {{true, i, s}};
      add_ops(s == 0 ? K_CU : K_CD, i - B.lo, o, 1, 1.0);
    }
  for (int i : orbs)
    for (int j : orbs) {
      if (i < j) {
        EOp uu[2] = {{true, i, 0}, {true, j, 0}};
        add_ops(K_AUU, idx_tri(B, i, j), uu, 2, 1.0);
        EOp dd[2] = {{true, i, 1}, {true, j, 1}};
        add_ops(K_ADD, idx_tri(B, i, j), dd, 2, 1.0);
      }
      EOp ud[2] = {{true, i, 0}, {true, j, 1}};
      add_ops(K_AUD, idx_sq(B, i, j), ud, 2, 1.0);
      EOp buu[2] = {{true, i, 0}, {false, j, 0}};
      add_ops(K_BUU, idx_sq(B, i, j), buu, 2, 1.0);
      EOp bud[2] = {{true, i, 0}, {false, j, 1}};
      add_ops(K_BUD, idx_sq(B, i, j), bud, 2, 1.0);
      EOp bdd[2] = {{true, i, 1}, {false, j, 1}};
      add_ops(K_BDD, idx_sq(B, i, j), bdd, 2, 1.0);
    }
  // S_x for x outside the new block:  S = 1/2 sum_j T_xj a_j + sum_jkl w_xjkl a+_jt a_lt a_ks
  for (int x = 0; x < L; ++x) {
    if (x >= B.lo && x < B.hi) continue;
    for (int s = 0; s < 2; ++s) {
      const int dk = s == 0 ? K_SU : K_SD, di = idx_S(B, x);
      add_named(dk, di, OpRef{dk, idx_S(old, x), false}, 0, 1.0);      // all operators in the old block
      EOp a1[1] = {{false, s_orb, s}};
      add_ops(dk, di, a1, 1, 0.5 * T2(ctx, x, s_orb));
      for (int j : orbs) for (int k : orbs) for (int l : orbs) {
        if (in_old(j) && in_old(k) && in_old(l)) continue;
        double wv = W4(ctx, x, j, k, l);
        if (wv == 0.0) continue;
        for (int t = 0; t < 2; ++t) {
          EOp o[3] = {{true, j, t}, {false, l, t}, {false, k, s}};
          add_ops(dk, di, o, 3, wv);
        }
      }
    }
  }
  // H of the new block
  add_named(K_H, 0, OpRef{K_H, 0, false}, 0, 1.0);
  for (int s = 0; s < 2; ++s) {
    // a+_s S^old_s + h.c.  (S^old carries three operators of the old block)
    const int sk = s == 0 ? K_SU : K_SD, si = idx_S(old, s_orb);
    double mc[16], ma[16];
    site_elem(true, s, mc);
    site_elem(false, s, ma);
    int oc = ctx->site_ops.intern(mc), oa = ctx->site_ops.intern(ma);
    // left: block factor first, a+_s S = -S a+_s ; S^T a_s already ordered.  right: site first.
    add_named(K_H, 0, OpRef{sk, si, false}, oc, left ? -1.0 : 1.0);
    add_named(K_H, 0, OpRef{sk, si, true}, oa, left ? 1.0 : -1.0);
  }
  for (int i : orbs) for (int j : orbs) {
    if (in_old(i) && in_old(j)) continue;
    double f = (in_old(i) || in_old(j)) ? 0.5 : 1.0;   // the other half sits in a+_s S^old_s + h.c.
    double tv = f * T2(ctx, i, j);
    if (tv == 0.0) continue;
    for (int s = 0; s < 2; ++s) {
      EOp o[2] = {{true, i, s}, {false, j, s}};
      add_ops(K_H, 0, o, 2, tv);
    }
  }
  for (int i : orbs) for (int j : orbs) for (int k : orbs) for (int l : orbs) {
    int nin = (int)in_old(i) + in_old(j) + in_old(k) + in_old(l);
    if (nin >= 3) continue;
    double wv = 0.5 * W4(ctx, i, j, k, l);
    if (wv == 0.0) continue;
    for (int s = 0; s < 2; ++s) for (int t = 0; t < 2; ++t) {
      EOp o[4] = {{true, i, s}, {true, j, t}, {false, l, t}, {false, k, s}};
      add_ops(K_H, 0, o, 4, wv);
    }
  }

  pt.lap("enumerate strings");
  // ---- group by (dst kind, src class, transpose, site op), pre-sum where a destination has several sources
  struct GKey { int dk, sc, tr, sop; bool operator<(const GKey& o) const { return std::tie(dk, sc, tr, sop) < std::tie(o.dk, o.sc, o.tr, o.sop); } };
  std::map<GKey, std::vector<Entry>> groups;
  for (auto& kv : acc) {
    if (std::fabs(kv.second) < 1e-300) continue;
    uint64_t k = kv.first;
    GKey g{(int)(k >> 40), (int)((k >> 22) & 63), (int)((k >> 9) & 1), (int)(k & 511)};
    groups[g].push_back(Entry{(int)((k >> 28) & 4095), (int)((k >> 10) & 4095), kv.second});
  }
  Presummer pre(ctx, st);
  std::vector<std::unique_ptr<OpClass>> temps;
  struct FG { GKey g; const OpClass* src; std::vector<Entry> e; };
  std::vector<FG> fgs;
  for (auto& kv : groups) {
    FG f{kv.first, old.cls[kv.first.sc].get(), kv.second};
    std::vector<int> cnt;
    bool multi = false;
    { std::map<int, int> c; for (auto& e : f.e) if (++c[e.a] > 1) multi = true; }
    if (multi && f.g.sc != K_ID) {
      temps.push_back(pre.make(old.sec, *f.src, f.e));
      f.src = temps.back().get();
    }
    fgs.push_back(std::move(f));
  }
  pre.run();

  // canonical partition of each destination class, so that batched outputs never overlap
  std::map<int, std::set<int>> cuts;
  for (auto& f : fgs)
    for (auto& r : make_runs(f.e)) { cuts[f.g.dk].insert(r.a0); cuts[f.g.dk].insert(r.a0 + r.cnt); }

  pt.lap("group + pre-sum");
  // ---- emit the triple products  new(q2' <- q1') += alpha * W2^T op(S)(q2 <- q1) W1 ----
  const uint64_t cap = workspace_cap(ctx);
  Planner planner(&ctx->al, cap, &ctx->ws_arena);
  for (auto& f : fgs) {
    OpClass& D = *B.cls[f.g.dk];
    const OpClass& S = *f.src;
    const auto& sm = ctx->site_ops.mats[f.g.sop];
    const int spar = ctx->site_ops.parity(f.g.sop);
    const int cpar = (S.du + S.dd) & 1;
    auto runs = make_runs(f.e, &cuts[f.g.dk]);
    for (size_t bd = 0; bd < D.blocks.size(); ++bd) {
      const ClsBlock& db = D.blocks[bd];
      for (int s2 = 0; s2 < 4; ++s2) for (int s1 = 0; s1 < 4; ++s1) {
        const double sv = sm[s2 * 4 + s1];
        if (sv == 0.0) continue;
        const int q1 = old.sec.find(B.sec.qu[db.si] - SITE_QU[s1], B.sec.qd[db.si] - SITE_QD[s1]);
        const int q2 = old.sec.find(B.sec.qu[db.so] - SITE_QU[s2], B.sec.qd[db.so] - SITE_QD[s2]);
        if (q1 < 0 || q2 < 0) continue;
        // site tensor blocks: left (qin = old sector, qout = new); right (qin = new sector, qout = old)
        auto f1 = A.find.find(left ? std::make_pair(q1, s1) : std::make_pair(db.si, s1));
        auto f2 = A.find.find(left ? std::make_pair(q2, s2) : std::make_pair(db.so, s2));
        if (f1 == A.find.end() || f2 == A.find.end()) continue;
        const SiteBlk& w1 = A.blks[f1->second];
        const SiteBlk& w2 = A.blks[f2->second];
        int sb;
        if (f.g.sc == K_ID) { if (q1 != q2) continue; sb = S.blk_of_in[q1]; }
        else if (!f.g.tr) { sb = S.blk_of_in[q1]; if (sb < 0 || S.blocks[sb].so != q2) continue; }
        else { sb = S.blk_of_out[q1]; if (sb < 0 || S.blocks[sb].si != q2) continue; }
        double sign = 1.0;
        if (left) { if (spar && ((old.sec.qu[q1] + old.sec.qd[q1]) & 1)) sign = -1.0; }
        else { if (cpar && ((SITE_QU[s1] + SITE_QD[s1]) & 1)) sign = -1.0; }
        const ClsBlock& sbk = S.blocks[sb];
        const int d1 = old.sec.dim[q1], d2 = old.sec.dim[q2];
        for (auto& r : runs) {
          Item it;
          it.C = D.ptr((int)bd, r.a0); it.ldc = db.cp; it.strideC = D.op_stride((int)bd);
          it.count = r.cnt; it.alpha = r.c * sv * sign;
          Mat X, Wm;
          if (left) {   // W2^T (d2' x d2), W1 (d1 x d1')
            X = Mat{A.data.p + w2.off, w2.doutp, true, 0, db.rp, pad8(d2), db.rows, d2};
            Wm = Mat{A.data.p + w1.off, w1.doutp, false, 0, pad8(d1), db.cp, d1, db.cols};
          } else {      // B2 (d2' x d2), B1^T (d1 x d1')
            X = Mat{A.data.p + w2.off, w2.doutp, false, 0, db.rp, pad8(d2), db.rows, d2};
            Wm = Mat{A.data.p + w1.off, w1.doutp, true, 0, pad8(d1), db.cp, d1, db.cols};
          }
          if (f.g.sc == K_ID) {
            it.nmat = 2; it.X = X; it.Y = Wm;
          } else {
            it.nmat = 3; it.X = X; it.W = Wm;
            it.Y = Mat{S.ptr(sb, r.b0), sbk.cp, f.g.tr != 0, S.op_stride(sb), pad8(d2), pad8(d1), d2, d1};
          }
          planner.add(it);
        }
      }
    }
  }
  pt.lap("items");
  Plan plan;
  planner.finish(&plan, st);
  pt.lap("planner.finish");
  plan.run(st, &ctx->launches, ctx->ex());
  DMRG_CUDA(cudaStreamSynchronize(st));
  pt.lap("run");
  if (flops_out) *flops_out = plan.flops_analytic;
  return nb;
}

// ------------------------------------------------------------------------------------------------
// two-site problem at bond (k, k+1): parts L | site k | site k+1 | R
// ------------------------------------------------------------------------------------------------
static inline uint64_t pack_key4(const OpRef& l, int o1, int o2, const OpRef& r) {
  return ((uint64_t)l.cls << 50) | ((uint64_t)l.idx << 38) | ((uint64_t)(l.tr ? 1 : 0) << 37) |
         ((uint64_t)o1 << 28) | ((uint64_t)o2 << 19) | ((uint64_t)r.cls << 13) | ((uint64_t)r.idx << 1) |
         (uint64_t)(r.tr ? 1 : 0);
}

// Four-part term groups of one bond: (left class, transpose, site op 1, site op 2, right class, transpose) ->
// coefficient entries (left operator, right operator, coefficient).  They depend on the bond and the
// integrals only, so sweeps re-use them (dmrg_ctx::term_cache).
struct TermGroups : TermGroupsBase {
  struct GKey {
    int lc, lt, o1, o2, rc, rt;
    bool operator<(const GKey& o) const { return std::tie(lc, lt, o1, o2, rc, rt) < std::tie(o.lc, o.lt, o.o1, o.o2, o.rc, o.rt); }
  };
  std::map<GKey, std::vector<Entry>> groups;
  size_t bytes() const override { size_t b = 0; for (auto& kv : groups) b += kv.second.size() * sizeof(Entry); return b; }
};

// Open-addressing accumulator  key -> sum of coefficients  for the term enumeration (linear probing; pack_key4 uses
// bits 0-55 only, so ~0 marks a free slot).  Iteration is in slot order: whoever needs a fixed order sorts afterwards.
struct FlatAcc {
  static constexpr uint64_t FREE = ~0ull;
  std::vector<uint64_t> keys;
  std::vector<double> vals;
  size_t n = 0, mask = 0;
  explicit FlatAcc(size_t cap = 256) { keys.assign(cap, FREE); vals.assign(cap, 0.0); mask = cap - 1; }
  static inline uint64_t mix(uint64_t x) {
    x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
    return x;
  }
  void grow() {
    FlatAcc big((mask + 1) * 2);
    for (size_t i = 0; i <= mask; ++i) if (keys[i] != FREE) big[keys[i]] = vals[i];
    *this = std::move(big);
  }
  double& operator[](uint64_t key) {
    if ((n + 1) * 10 > (mask + 1) * 7) grow();
    size_t i = mix(key) & mask;
    while (keys[i] != FREE && keys[i] != key) i = (i + 1) & mask;
    if (keys[i] == FREE) { keys[i] = key; vals[i] = 0.0; ++n; }
    return vals[i];
  }
  template <class F> void for_each(F&& f) const {
    for (size_t i = 0; i <= mask; ++i) if (keys[i] != FREE) f(keys[i], vals[i]);
  }
};

// Four-part term groups of bond k (Eq. (6)), pre-summation not yet applied: a function of (L, k, T, V) only --
// no block data, no device work, nothing of the context written -- so it can run on a host thread ahead of the step
// that needs it (prefetch_term_groups).
static std::shared_ptr<TermGroups> build_term_groups(const dmrg_ctx* ctx, int k) {
  PhaseTimer pt("term groups");
  using GKey = TermGroups::GKey;
  const int L = ctx->L;
  const int o_s1 = k - 1, o_s2 = k;
  BlockSide BL, BR;                     // for the naming of block operators only: the orbital ranges of the two blocks
  BL.is_left = true; BL.lo = 0; BL.hi = k - 1;
  BR.is_left = false; BR.lo = k + 1; BR.hi = L;
  const SiteOpTable& site_ops = ctx->site_ops;   // read-only: every product of <= 4 elementary operators is interned
  // ---- four-part terms  coef * O_L (x) o_1 (x) o_2 (x) O_R ----
  constexpr int NB = 8;                 // buckets of the parallel enumeration = partitions of the key space
  FlatAcc acc;
  auto part_of = [&](int orb) { return orb < o_s1 ? 0 : (orb == o_s1 ? 1 : (orb == o_s2 ? 2 : 3)); };
  auto add_named = [&](const OpRef& l, int o1, int o2, const OpRef& r, double coef) {
    if (o1 < 0 || o2 < 0 || coef == 0.0) return;
    acc[pack_key4(l, o1, o2, r)] += coef;
  };
  // returns false if the string cannot be named (internal error); key = 0 with c = 0 for a vanishing string
  auto key_of = [&](const EOp* ops, int n, double coef, uint64_t& key, double& c) {
    EOp po[4][4];
    int np[4] = {0, 0, 0, 0}, inv = 0;
    c = 0.0;
    for (int i = 0; i < n; ++i) {
      int p = part_of(ops[i].orb);
      for (int q = p + 1; q < 4; ++q) inv += np[q];   // operators of later parts already seen
      po[p][np[p]++] = ops[i];
    }
    OpRef l, r; double sl, sr;
    int rc = name_block_ops(BL, po[0], np[0], l, sl);
    if (rc == 1) return true;
    if (rc != 0) return false;
    rc = name_block_ops(BR, po[3], np[3], r, sr);
    if (rc == 1) return true;
    if (rc != 0) return false;
    const int o1 = site_product(site_ops, po[1], np[1]);
    const int o2 = site_product(site_ops, po[2], np[2]);
    const double cc = coef * sl * sr * ((inv & 1) ? -1.0 : 1.0);
    if (o1 < 0 || o2 < 0 || cc == 0.0) return true;
    key = pack_key4(l, o1, o2, r);
    c = cc;
    return true;
  };
  auto add_ops = [&](const EOp* ops, int n, double coef) {
    uint64_t key; double c;
    DMRG_REQUIRE(key_of(ops, n, coef, key, c), DMRG_ERR_ARG, "internal: unnamed operator string");
    if (c != 0.0) acc[key] += c;
  };
  const OpRef ID{K_ID, 0, false};
  add_named(OpRef{K_H, 0, false}, 0, 0, ID, 1.0);
  add_named(ID, 0, 0, OpRef{K_H, 0, false}, 1.0);
  for (int s = 0; s < 2; ++s) {
    const EOp ec{true, 0, s}, ea{false, 0, s};
    const int oc_ = site_product(site_ops, &ec, 1), oa_ = site_product(site_ops, &ea, 1);
    const int sk = s == 0 ? K_SU : K_SD, ck = s == 0 ? K_CU : K_CD;
    // x outside L:  a+_x S^L_x = - S^L_x a+_x ,  h.c. = (S^L_x)^T a_x
    for (int x = o_s1; x < L; ++x) {
      OpRef S{sk, idx_S(BL, x), false}, St{sk, idx_S(BL, x), true};
      if (x == o_s1) { add_named(S, oc_, 0, ID, -1.0); add_named(St, oa_, 0, ID, 1.0); }
      else if (x == o_s2) { add_named(S, 0, oc_, ID, -1.0); add_named(St, 0, oa_, ID, 1.0); }
      else { add_named(S, 0, 0, OpRef{ck, x - BR.lo, false}, -1.0); add_named(St, 0, 0, OpRef{ck, x - BR.lo, true}, 1.0); }
    }
    // x outside R:  a+_x S^R_x ,  h.c. = (S^R_x)^T a_x = - a_x (S^R_x)^T
    for (int x = 0; x <= o_s2; ++x) {
      OpRef S{sk, idx_S(BR, x), false}, St{sk, idx_S(BR, x), true};
      if (x == o_s1) { add_named(ID, oc_, 0, S, 1.0); add_named(ID, oa_, 0, St, -1.0); }
      else if (x == o_s2) { add_named(ID, 0, oc_, S, 1.0); add_named(ID, 0, oa_, St, -1.0); }
      else { add_named(OpRef{ck, x - BL.lo, false}, 0, 0, S, 1.0); add_named(OpRef{ck, x - BL.lo, true}, 0, 0, St, -1.0); }
    }
  }
  auto is_block = [&](int p) { return p == 0 || p == 3; };
  for (int i = 0; i < L; ++i) for (int j = 0; j < L; ++j) {
    int pi = part_of(i), pj = part_of(j);
    if (pi == pj && is_block(pi)) continue;                        // inside H^L / H^R
    double f = 1.0;
    if (pi != pj) f -= 0.5 * (is_block(pi) ? 1 : 0) + 0.5 * (is_block(pj) ? 1 : 0);   // halves carried by S^L, S^R
    double tv = f * T2(ctx, i, j);
    if (tv == 0.0) continue;
    for (int s = 0; s < 2; ++s) {
      EOp o[2] = {{true, i, s}, {false, j, s}};
      add_ops(o, 2, tv);
    }
  }
  pt.lap("one-body + S strings");
  // The L^4 two-body strings: NB buckets (i mod NB), each with one private map per key partition (key mod NB), filled
  // in parallel; partition p then sums its maps in bucket order, so the coefficient sums do not depend on the
  // number of threads.
  std::vector<FlatAcc> loc((size_t)NB * NB);
  std::vector<FlatAcc> parts(NB);
  {
    int err_any = 0;
#pragma omp parallel for num_threads(NB) schedule(static, 1)
    for (int b = 0; b < NB; ++b) {
      int err = 0;
      FlatAcc* mine = &loc[(size_t)b * NB];
      for (int i = b; i < L; i += NB)
        for (int j = 0; j < L; ++j) for (int kk = 0; kk < L; ++kk) for (int l = 0; l < L; ++l) {
          int cnt[4] = {0, 0, 0, 0};
          ++cnt[part_of(i)]; ++cnt[part_of(j)]; ++cnt[part_of(kk)]; ++cnt[part_of(l)];
          if (cnt[0] >= 3 || cnt[3] >= 3) continue;                      // inside H^L/H^R or a+ S + h.c.
          const double wv = 0.5 * W4(ctx, i, j, kk, l);
          if (wv == 0.0) continue;
          for (int s = 0; s < 2; ++s) for (int t = 0; t < 2; ++t) {
            EOp o[4] = {{true, i, s}, {true, j, t}, {false, l, t}, {false, kk, s}};
            uint64_t key; double c;
            if (!key_of(o, 4, wv, key, c)) { err = 1; continue; }
            if (c != 0.0) mine[key % NB][key] += c;
          }
        }
      if (err) {
#pragma omp atomic write
        err_any = 1;
      }
    }
    DMRG_REQUIRE(!err_any, DMRG_ERR_ARG, "internal: unnamed operator string");
    pt.lap("two-body strings (parallel)");
#pragma omp parallel for num_threads(NB) schedule(static, 1)
    for (int p = 0; p < NB; ++p) {
      FlatAcc& out = parts[p];
      acc.for_each([&](uint64_t key, double v) { if ((int)(key % NB) == p) out[key] += v; });   // one-body, S, H strings
      for (int b = 0; b < NB; ++b) loc[(size_t)b * NB + p].for_each([&](uint64_t key, double v) { out[key] += v; });
    }
    loc.clear();
  }
  pt.lap("merge");
  // ---- group the terms by (left class, transpose, site operators, right class, transpose) ----
  auto tg = std::make_shared<TermGroups>();
  std::map<GKey, std::vector<Entry>>& groups = tg->groups;   // Entry: a = left index, b = right index
  {
    std::unordered_map<uint64_t, std::vector<Entry>*> fast;   // group bits of the key -> its entry list
    const uint64_t gmask = ~((0xFFFull << 38) | (0xFFFull << 1));
    for (auto& part : parts)
      part.for_each([&](uint64_t q, double v) {
        if (std::fabs(v) < 1e-300) return;
        std::vector<Entry>*& e = fast[q & gmask];
        if (!e) {
          GKey g{(int)(q >> 50) & 63, (int)(q >> 37) & 1, (int)(q >> 28) & 511, (int)(q >> 19) & 511,
                 (int)(q >> 13) & 63, (int)(q & 1)};
          e = &groups[g];
        }
        e->push_back(Entry{(int)(q >> 38) & 4095, (int)(q >> 1) & 4095, v});
      });
    // a fixed entry order inside every group (the maps iterate in slot order)
    std::vector<std::vector<Entry>*> gv;
    for (auto& kv : groups) gv.push_back(&kv.second);
#pragma omp parallel for num_threads(NB) schedule(dynamic, 1)
    for (int g = 0; g < (int)gv.size(); ++g)
      std::sort(gv[g]->begin(), gv[g]->end(), [](const Entry& x, const Entry& y) { return x.a != y.a ? x.a < y.a : x.b < y.b; });
  }
  pt.lap("group");
  return tg;
}

static void cache_term_groups(dmrg_ctx* ctx, int k, const std::shared_ptr<TermGroupsBase>& tg) {
  size_t cached = 0;
  for (auto& kv : ctx->term_cache) cached += kv.second->bytes();
  if (cached + tg->bytes() <= (size_t)1 << 30) ctx->term_cache[k] = tg;   // host memory cap: 1 GiB
}

static std::shared_ptr<TermGroupsBase> build_term_groups_su2(const dmrg_ctx* ctx, int k);   // engine_su2.inc

// Starts building the term groups of bond k on a host thread unless they are cached or on their way.  Called when a
// two-site problem has been prepared, for its two neighbours: a sweep needs one of them next, and the build (an
// O(L^4) enumeration) then runs while the eigensolver keeps the GPU busy instead of in front of the next step
// ("Tables": host work that should not show up in the sweep time).  DMRG_B200_NO_PREFETCH=1 turns it off.
static void prefetch_term_groups(dmrg_ctx* ctx, int k) {
  static const bool off = std::getenv("DMRG_B200_NO_PREFETCH") != nullptr;
  if (off || k < 1 || k + 1 > ctx->L || ctx->term_cache.count(k) || ctx->term_prefetch.count(k)) return;
  const dmrg_ctx* c = ctx;
  ctx->term_prefetch[k] = std::async(std::launch::async, [c, k]() -> std::shared_ptr<TermGroupsBase> {
                            if (c->su2()) return build_term_groups_su2(c, k);
                            return build_term_groups(c, k);
                          }).share();
}

static void harvest_term_prefetch(dmrg_ctx* ctx);
static void prefetch_neighbour_term_groups(dmrg_ctx* ctx) {
  harvest_term_prefetch(ctx);
  prefetch_term_groups(ctx, ctx->k + 1);
  prefetch_term_groups(ctx, ctx->k - 1);
}

// The term groups of bond k if a host thread is building (or has built) them; waits for it.  Null if none is.
static std::shared_ptr<TermGroupsBase> take_prefetched_term_groups(dmrg_ctx* ctx, int k) {
  auto pf = ctx->term_prefetch.find(k);
  if (pf == ctx->term_prefetch.end()) return nullptr;
  auto fut = pf->second;
  ctx->term_prefetch.erase(pf);
  return fut.get();     // (rethrows what the builder threw)
}

// Moves finished builds into the cache (the ones of the direction the sweep did not take).
static void harvest_term_prefetch(dmrg_ctx* ctx) {
  for (auto it = ctx->term_prefetch.begin(); it != ctx->term_prefetch.end();) {
    if (it->second.wait_for(std::chrono::seconds(0)) != std::future_status::ready) { ++it; continue; }
    try { cache_term_groups(ctx, it->first, it->second.get()); } catch (...) {}   // (a failed build is simply not cached)
    it = ctx->term_prefetch.erase(it);
  }
}

// Output-block sharding of H_eff.psi over ranks ("independent operations"): every psi'
// block is computed completely by one rank, so the exchange is a sum with exact zeros.  Longest-processing-time
// assignment on the analytic flops per output block; ties by block index and rank, so all ranks agree.
static void assign_shard_owners(dmrg_ctx* ctx, const std::vector<double>& blk_flops) {
  const size_t nb = ctx->psi.size();
  ctx->psi_owner.assign(nb, 0);
  ctx->shard_flops.assign((size_t)std::max(1, ctx->shard_count), 0.0);
  if (ctx->shard_count <= 1) return;
  std::vector<int> order(nb);
  for (size_t i = 0; i < nb; ++i) order[i] = (int)i;
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return blk_flops[a] > blk_flops[b]; });
  for (int b : order) {
    int best = 0;
    for (int r = 1; r < ctx->shard_count; ++r) if (ctx->shard_flops[r] < ctx->shard_flops[best]) best = r;
    ctx->psi_owner[b] = best;
    ctx->shard_flops[best] += blk_flops[b];
  }
}

// diag(H_eff) from the diagonal tasks, and the statistics of the prepared two-site problem
static void finish_superblock(dmrg_ctx* ctx, std::vector<std::vector<DiagTask>>& dtasks, int64_t n_terms,
                              int64_t n_tasks, int64_t n_groups, cudaStream_t st) {
  BlockSide& BL = *ctx->left;
  BlockSide& BR = *ctx->right;
  // ---- diagonal of H_eff ----
  {
    std::vector<DiagTask> flat;
    std::vector<int> begin(ctx->psi.size() + 1, 0);
    for (size_t b = 0; b < ctx->psi.size(); ++b) {
      begin[b] = (int)flat.size();
      flat.insert(flat.end(), dtasks[b].begin(), dtasks[b].end());
    }
    begin[ctx->psi.size()] = (int)flat.size();
    DevArray<DiagTask> d_tasks;
    DevArray<int> d_begin;
    d_tasks.upload(&ctx->al, flat, st);
    d_begin.upload(&ctx->al, begin, st);
    launch_diag(ctx->d_psi_blocks.p, (int)ctx->psi.size(), d_tasks.p, d_begin.p, ctx->diag_p.p, st);
    ++ctx->launches;
    DMRG_CUDA(cudaStreamSynchronize(st));
  }

  // ---- statistics ----
  dmrg_stats_t& s = ctx->stats;
  s.n_terms = n_terms;
  s.n_tasks = n_tasks;
  s.n_groups = n_groups;
  s.flops_apply = ctx->apply_plan.flops_analytic;
  s.flops_executed = ctx->apply_plan.flops_executed;
  s.flops_shared = ctx->apply_plan.flops_shared;
  s.bytes_intermediate = ctx->apply_plan.bytes_intermediate;
  s.psi_size = ctx->psi_n;
  s.op_bytes_left = (int64_t)BL.bytes();
  s.op_bytes_right = (int64_t)BR.bytes();
  s.bytes_unique = (double)(s.op_bytes_left + s.op_bytes_right) + 16.0 * (double)ctx->psi_n;
  s.n_chunks = (int)ctx->apply_plan.chunks.size();
  s.launches_per_apply = ctx->apply_plan.launches() + 2;
}


void prepare_superblock(dmrg_ctx* ctx, cudaStream_t st) {
  const int k = ctx->k;
  BlockSide& BL = *ctx->left;
  BlockSide& BR = *ctx->right;
  DMRG_REQUIRE(BL.lo == 0 && BL.hi == k - 1 && BR.lo == k + 1 && BR.hi == ctx->L, DMRG_ERR_ARG,
               "superblock: environments do not match the bond");
  const int NU = ctx->cfg.n_up, ND = ctx->cfg.n_dn;
  // drop pre-summed classes of an earlier bond
  BL.cls.resize(K_NSTD);
  BR.cls.resize(K_NSTD);
  ctx->apply_plan.clear();

  // ---- psi layout: blocks (qL lexicographic, s1, s2) ----
  ctx->psi.clear();
  ctx->psi_find.clear();
  long long oc = 0, op = 0;
  for (int ql = 0; ql < BL.sec.size(); ++ql)
    for (int s1 = 0; s1 < 4; ++s1)
      for (int s2 = 0; s2 < 4; ++s2) {
        int ru = NU - BL.sec.qu[ql] - SITE_QU[s1] - SITE_QU[s2];
        int rd = ND - BL.sec.qd[ql] - SITE_QD[s1] - SITE_QD[s2];
        int qr = BR.sec.find(ru, rd);
        if (qr < 0) continue;
        PsiBlk b{ql, s1, s2, qr, BL.sec.dim[ql], BR.sec.dim[qr], pad8(BL.sec.dim[ql]), pad8(BR.sec.dim[qr]), oc, op};
        oc += (long long)b.dL * b.dR;
        op += (long long)b.dLp * b.dRp;
        ctx->psi_find[{ql, s1, s2}] = (int)ctx->psi.size();
        ctx->psi.push_back(b);
      }
  ctx->psi_n = oc;
  ctx->psi_np = op;
  {
    std::vector<PsiBlockDev> hb;
    for (auto& b : ctx->psi) hb.push_back(PsiBlockDev{b.off_c, b.off_p, b.dL, b.dR, b.dLp, b.dRp});
    ctx->d_psi_blocks.upload(&ctx->al, hb, st);
    ctx->psi_in_p.allocate(&ctx->al, (size_t)std::max<long long>(op, 8));
    ctx->psi_out_p.allocate(&ctx->al, (size_t)std::max<long long>(op, 8));
    ctx->diag_p.allocate(&ctx->al, (size_t)std::max<long long>(op, 8));
    DMRG_CUDA(cudaMemsetAsync(ctx->psi_in_p.p, 0, (size_t)std::max<long long>(op, 8) * 8, st));
    DMRG_CUDA(cudaMemsetAsync(ctx->psi_out_p.p, 0, (size_t)std::max<long long>(op, 8) * 8, st));
    DMRG_CUDA(cudaMemsetAsync(ctx->diag_p.p, 0, (size_t)std::max<long long>(op, 8) * 8, st));
  }

  PhaseTimer pt("superblock");
  using GKey = TermGroups::GKey;
  // The term groups depend on the bond and the integrals only: a sweep that comes back to this bond re-uses them.
  std::shared_ptr<TermGroups> tg;
  {
    auto f = ctx->term_cache.find(k);
    if (f != ctx->term_cache.end()) tg = std::static_pointer_cast<TermGroups>(f->second);
  }
  if (!tg) {
    auto got = take_prefetched_term_groups(ctx, k);
    if (got) {
      tg = std::static_pointer_cast<TermGroups>(got);
      pt.lap("term groups from the prefetch thread");
    } else {
      tg = build_term_groups(ctx, k);
      pt.lap("term groups built here");
    }
    cache_term_groups(ctx, k, tg);
  } else {
    pt.lap("term groups from cache");
  }
  const auto& groups = tg->groups;
  Presummer pre(ctx, st);
  struct FG { GKey g; int lcls, rcls; std::vector<Entry> e; };
  std::vector<FG> fgs;
  int64_t n_terms = 0;
  for (auto& kv : groups) {
    FG f{kv.first, kv.first.lc, kv.first.rc, kv.second};
    size_t nrows = 0, ncols = 0;
    {
      std::vector<char> sr(4096, 0), sc(4096, 0);
      for (auto& e : f.e) {
        if (!sr[e.a]) { sr[e.a] = 1; ++nrows; }
        if (!sc[e.b]) { sc[e.b] = 1; ++ncols; }
      }
    }
    const size_t nnz = f.e.size();
    const bool canL = f.g.lc != K_ID, canR = f.g.rc != K_ID;
    size_t costL = canL ? ncols : nnz + 1, costR = canR ? nrows : nnz + 1;
    size_t best = std::min(costL, costR);
    if (best * 4 <= nnz * 3) {
      if (costL <= costR) {     // K^L[b] = sum_a coef * O_L[a]  for each right partner b
        std::vector<Entry> t;
        for (auto& e : f.e) t.push_back(Entry{e.b, e.a, e.c});
        BL.cls.push_back(pre.make(BL.sec, *BL.cls[f.g.lc], t));
        f.lcls = (int)BL.cls.size() - 1;
        f.e.clear();
        for (auto& e : t) f.e.push_back(Entry{e.b, e.a, 1.0});
      } else {
        std::vector<Entry> t = f.e;
        BR.cls.push_back(pre.make(BR.sec, *BR.cls[f.g.rc], t));
        f.rcls = (int)BR.cls.size() - 1;
        f.e = t;
      }
    }
    n_terms += (int64_t)f.e.size();
    fgs.push_back(std::move(f));
  }
  pt.lap("pre-sum: coefficient matrices, classes, items");
  pre.run();
  pt.lap("pre-sum: plan + launches + sync");

  // ---- tasks of PAPER.md Eq. (8): (term group x psi block) -> contraction items + diagonal tasks ----
  const uint64_t cap = workspace_cap(ctx);
  Planner planner(&ctx->al, cap, &ctx->ws_arena);
  std::vector<std::vector<DiagTask>> dtasks(ctx->psi.size());
  int64_t n_tasks = 0, n_groups = 0;
  // psi blocks outermost: the items that apply the same operator run to the same psi block (different term
  // groups) are then neighbours and land in the same workspace chunk, where they share the intermediate
  std::vector<std::vector<Run>> all_runs;
  for (auto& f : fgs) all_runs.push_back(make_runs(f.e));
  // Sharded contexts (dmrg_set_shard) run the loop twice: pass 0 only adds up the analytic flops per OUTPUT block,
  // from which every rank derives the same block -> rank map; pass 1 emits the items of the blocks this rank owns.
  std::vector<double> blk_flops(ctx->psi.size(), 0.0);
  for (int pass = ctx->shard_count > 1 ? 0 : 1; pass < 2; ++pass) {
  if (pass == 1) { assign_shard_owners(ctx, blk_flops); ctx->blk_flops.assign(ctx->psi.size(), 0.0); }
  for (size_t bi = 0; bi < ctx->psi.size(); ++bi) {
    for (size_t gi = 0; gi < fgs.size(); ++gi) {
      const auto& f = fgs[gi];
      const OpClass& CL = *BL.cls[f.lcls];
      const OpClass& CR = *BR.cls[f.rcls];
      const auto& m1 = ctx->site_ops.mats[f.g.o1];
      const auto& m2 = ctx->site_ops.mats[f.g.o2];
      const int p1 = ctx->site_ops.parity(f.g.o1), p2 = ctx->site_ops.parity(f.g.o2);
      const int pR = (CR.du + CR.dd) & 1;
      const auto& runs = all_runs[gi];
      const PsiBlk& in = ctx->psi[bi];
      // left operator block acting on sector in.qL
      int lb = -1, qLo = in.qL;
      if (f.g.lc != K_ID) {
        lb = f.g.lt ? CL.blk_of_out[in.qL] : CL.blk_of_in[in.qL];
        if (lb < 0) continue;
        qLo = f.g.lt ? CL.blocks[lb].si : CL.blocks[lb].so;
      }
      int rb = -1, qRo = in.qR;
      if (f.g.rc != K_ID) {
        rb = f.g.rt ? CR.blk_of_out[in.qR] : CR.blk_of_in[in.qR];
        if (rb < 0) continue;
        qRo = f.g.rt ? CR.blocks[rb].si : CR.blocks[rb].so;
      }
      for (int s1o = 0; s1o < 4; ++s1o) {
        const double v1 = m1[s1o * 4 + in.s1];
        if (v1 == 0.0) continue;
        for (int s2o = 0; s2o < 4; ++s2o) {
          const double v2 = m2[s2o * 4 + in.s2];
          if (v2 == 0.0) continue;
          auto fo = ctx->psi_find.find({qLo, s1o, s2o});
          if (fo == ctx->psi_find.end()) continue;
          const PsiBlk& out = ctx->psi[fo->second];
          if (out.qR != qRo) continue;
          // fermion sign: operators right of a part pass that part's input state
          int nL = BL.sec.qu[in.qL] + BL.sec.qd[in.qL];
          int n1 = SITE_QU[in.s1] + SITE_QD[in.s1], n2 = SITE_QU[in.s2] + SITE_QD[in.s2];
          int ph = nL * (p1 + p2 + pR) + n1 * (p2 + pR) + n2 * pR;
          const double sgn = (ph & 1) ? -1.0 : 1.0;
          const bool mine = ctx->psi_owner[fo->second] == ctx->shard_rank;
          if (pass == 1 && mine) ++n_groups;
          for (auto& r : runs) {
            if (pass == 1 && mine) n_tasks += r.cnt;
            Item it;
            it.C = ctx->psi_out_p.p + out.off_p; it.ldc = out.dRp; it.strideC = 0;
            it.count = r.cnt; it.alpha = r.c * v1 * v2 * sgn;
            Mat Xp{ctx->psi_in_p.p + in.off_p, in.dRp, false, 0, in.dLp, in.dRp, in.dL, in.dR};
            Mat ML, MR;
            if (lb >= 0) {
              const ClsBlock& b = CL.blocks[lb];
              ML = Mat{CL.ptr(lb, r.a0), b.cp, f.g.lt != 0, CL.op_stride(lb), out.dLp, in.dLp, out.dL, in.dL};
            }
            if (rb >= 0) {    // W = op(R)^T : (n x n')
              const ClsBlock& b = CR.blocks[rb];
              MR = Mat{CR.ptr(rb, r.b0), b.cp, f.g.rt == 0, CR.op_stride(rb), in.dRp, out.dRp, in.dR, out.dR};
            }
            if (lb >= 0 && rb >= 0) { it.nmat = 3; it.X = ML; it.Y = Xp; it.W = MR; }
            else if (lb >= 0) { it.nmat = 2; it.X = ML; it.Y = Xp; }
            else if (rb >= 0) { it.nmat = 2; it.X = Xp; it.Y = MR; }
            else {
              const OpClass& I = *BR.cls[K_ID];
              int ib = I.blk_of_in[in.qR];
              it.nmat = 2; it.X = Xp;
              it.Y = Mat{I.ptr(ib, 0), I.blocks[ib].cp, false, 0, in.dRp, in.dRp, in.dR, in.dR};
            }
            if (pass == 0) { blk_flops[fo->second] += item_flops(it); continue; }
            ctx->blk_flops[fo->second] += item_flops(it);     // analytic flops per OUTPUT block (dmrg_block_flops)
            if (mine) planner.add(it);
            if (fo->second == (int)bi) {      // the diagonal is kept whole on every rank
              DiagTask d{};
              d.L = lb >= 0 ? CL.ptr(lb, r.a0) : nullptr;
              d.R = rb >= 0 ? CR.ptr(rb, r.b0) : nullptr;
              d.rsL = lb >= 0 ? CL.op_stride(lb) : 0;
              d.rsR = rb >= 0 ? CR.op_stride(rb) : 0;
              d.ldl = lb >= 0 ? CL.blocks[lb].cp : 0;
              d.ldr = rb >= 0 ? CR.blocks[rb].cp : 0;
              d.count = r.cnt;
              d.alpha = it.alpha;
              dtasks[bi].push_back(d);
            }
          }
        }
      }
    }
  }
  }
  pt.lap("tasks -> items");
  planner.finish(&ctx->apply_plan, st);
  pt.lap("planner.finish");
  finish_superblock(ctx, dtasks, n_terms, n_tasks, n_groups, st);
  pt.lap("diag + stats");
  // the sweep goes to one of the neighbouring bonds next: their term groups are built while the eigensolver runs
  prefetch_neighbour_term_groups(ctx);
}

#include "engine_su2.inc"

void drop_presummed(BlockSide& b, bool su2) {
  if (!su2) {
    if ((int)b.cls.size() > K_NSTD) b.cls.resize(K_NSTD);
  } else if ((int)b.kinds.size() > su2e::SK_N) {
    b.cls.resize(b.kinds[su2e::SK_N - 1].cids.back() + 1);
    b.kinds.resize(su2e::SK_N);
  }
}

}  // namespace dmrg
