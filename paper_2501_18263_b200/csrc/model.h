// Host-side model: sectors, block-sparse operator classes, MPS tensors, and the context.
//
// Operator storage ("class storage"): operators of one kind on one
// block share q_out - q_in = (du, dd) and therefore their block structure.  A class
// stores, for each non-zero block (q_out, q_in), ALL its operators contiguously:
//     data[ block.off + op * rp * cp + r * cp + c ],   rp, cp = dims padded to multiples of 8
// so that "one block of every operator in a term group" is a strided batch for the GEMM kernel.
#pragma once
#include <array>
#include <future>
#include <map>
#include <memory>

#include "common.h"
#include "kernels.cuh"
#include "plan.h"

namespace dmrg {

static const int SITE_QU[4] = {0, 0, 1, 1};   // s = 0, dn, up, up+dn
static const int SITE_QD[4] = {0, 1, 0, 1};

struct Sectors {
  std::vector<int> qu, qd, dim;
  std::unordered_map<int, int> index;
  static int key(int u, int d) { return (u + 256) * 4096 + (d + 256); }
  int size() const { return (int)dim.size(); }
  int find(int u, int d) const {
    auto it = index.find(key(u, d));
    return it == index.end() ? -1 : it->second;
  }
  void add(int u, int d, int n) {
    index[key(u, d)] = size();
    qu.push_back(u); qd.push_back(d); dim.push_back(n);
  }
  long long total() const { long long t = 0; for (int x : dim) t += x; return t; }
};

enum Kind : int { K_ID = 0, K_H, K_CU, K_CD, K_AUU, K_AUD, K_ADD, K_BUU, K_BUD, K_BDD, K_SU, K_SD, K_NSTD };

struct ClsBlock {
  int so, si;          // out / in sector index
  int rows, cols, rp, cp;
  long long off;       // element offset of operator 0 of this block
};

struct OpClass {
  int kind = 0, du = 0, dd = 0, nops = 0, nalloc = 0;
  std::vector<ClsBlock> blocks;
  std::vector<int> blk_of_in, blk_of_out;
  DevArray<double> data;
  long long elems = 0;
  void layout(const Sectors& sec, int du_, int dd_, int nops_);
  void allocate(Allocator* al, cudaStream_t st);
  double* ptr(int b, int r) const { return data.p + blocks[b].off + (long long)r * blocks[b].rp * blocks[b].cp; }
  long long op_stride(int b) const { return (long long)blocks[b].rp * blocks[b].cp; }
};

// Pinned host memory of the environment cache's host tier (api.cu): fixed-size pages, pinned on first use and kept
// until the context dies (pinning costs ~0.3 s per GB, a copy into a pinned page runs at PCIe speed), so any free
// page fits any block.
struct HostPool {
  std::vector<double*> free_pages;
  uint64_t page_bytes = 0, total = 0, cap = 0;      // bytes pinned so far / allowed
  bool get(size_t npages, std::vector<double*>* out);
  void put(std::vector<double*>& pages) { for (double* p : pages) free_pages.push_back(p); pages.clear(); }
  ~HostPool();
};

struct BlockSide {
  bool is_left = true;
  int lo = 0, hi = 0;          // orbitals [lo, hi)
  Sectors sec;                 // labelled by the block's own electron content
  std::vector<std::unique_ptr<OpClass>> cls;   // [0, K_NSTD) standard kinds, then pre-summed classes
  // SU(2): an operator kind (tensor operator of doubled rank k2 changing N by dN) owns one class per
  // spin change d2S = dd of the class; kinds[0..SK_N) are the carried ones, pre-summed kinds follow.
  struct KindRef { int k2 = 0, dN = 0; std::vector<int> cids; };
  std::vector<KindRef> kinds;
  int norb() const { return hi - lo; }
  uint64_t bytes() const { uint64_t b = 0; for (auto& c : cls) if (c) b += (uint64_t)c->elems * 8; return b; }
  // host tier: a spilled block keeps its layout; the data of all classes sit back to back in pinned pages
  bool spilled = false;
  std::vector<double*> host_pages;
  std::vector<size_t> host_n;         // elements per class in the host copy
  std::shared_ptr<HostPool> pool;
  ~BlockSide() { if (pool) pool->put(host_pages); }
};

struct SiteBlk {
  int qin, s, qout;            // sector indices in bond i-1 / bond i
  int din, dout, dinp, doutp;
  long long off;               // element offset in the padded device array
};

struct SiteTensor {
  int canonical = -1;          // 0 left, 1 right, -1 unset
  std::vector<SiteBlk> blks;
  std::map<std::pair<int, int>, int> find;   // (qin, s) -> block            (U(1)xU(1))
  std::map<std::array<int, 3>, int> find3;   // (qin, m, qout) -> block      (SU(2): s holds the multiplet m)
  DevArray<double> data;
};

struct OpRef { int cls = K_ID; int idx = 0; bool tr = false; };

struct SiteOpTable {
  std::vector<std::array<double, 16>> mats;
  std::vector<int> prod;       // id of every product of <= 4 elementary site operators (engine.cu site_code)
  void build_products();
  SiteOpTable();
  int intern(const double* m);
  int parity(int id) const;
};

// Term groups of the two-site problem of one bond (engine.cu, engine_su2.inc): a function of the bond and the integrals.
struct TermGroupsBase {
  virtual ~TermGroupsBase() = default;
  virtual size_t bytes() const = 0;
};

// What dmrg_truncate_bond leaves behind for dmrg_start_vector (truncate.cu): per kept sector of the truncated bond the
// centre factor, c rows in descending order of the singular values: Sigma V^T (row length = columns of the sector) when
// the sweep moves right, (U Sigma)^T (row length = rows of the sector) when it moves left.
struct CentreFactor {
  int bond = 0, direction = -1;            // bond == 0: none
  DevArray<double> C;
  struct Sec {
    int c = 0, len = 0;                    // kept states, row length
    long long off = 0;                     // first element in C
    std::map<std::pair<int, int>, std::pair<int, int>> groups;   // (s2, q_R) or (q_L, s1) -> (first position, width) in a row
  };
  std::map<std::pair<int, int>, Sec> sec;  // label (n_up, n_dn) of the kept bond sector
  void clear() { bond = 0; direction = -1; C.release(); sec.clear(); }
};

struct PsiBlk { int qL, s1, s2, qR; int dL, dR, dLp, dRp; long long off_c, off_p; int qLp = -1; /* SU(2): (N, 2S) of L' */ int NLp = 0, SLp = 0; };

}  // namespace dmrg

// The opaque context of the C ABI.
struct dmrg_ctx {
  dmrg_config cfg;
  dmrg::Allocator al;
  std::string err;
  int L = 0;
  std::vector<double> T, w;    // T (L*L), w_ijkl = (V_ijkl + V_jilk)/2 (L^4)
  double e_core = 0;
  bool have_integrals = false;
  std::vector<dmrg::Sectors> bond;          // bond sectors, label = electrons left of the bond
  std::vector<dmrg::SiteTensor> site;       // 1-based
  int k = 0;                                // current bond (k, k+1); 0 = none
  std::shared_ptr<dmrg::BlockSide> left, right;
  // environment cache for sweeps: left_cache[i] = block of sites 1..i, right_cache[i] = block of sites i..L.
  // Entries are dropped when a site tensor or bond they depend on changes; total size is capped.
  std::map<int, std::shared_ptr<dmrg::BlockSide>> left_cache, right_cache;
  std::map<int, std::shared_ptr<dmrg::TermGroupsBase>> term_cache;   // bond k -> term groups of the two-site problem
  // Term groups of neighbouring bonds being built ahead of time on host threads (engine.cu prefetch_term_groups).
  // The builders read L, T, w and site_ops: whoever changes those calls drop_term_groups() first.
  std::map<int, std::shared_future<std::shared_ptr<dmrg::TermGroupsBase>>> term_prefetch;
  void drop_term_groups() {
    for (auto& kv : term_prefetch) if (kv.second.valid()) kv.second.wait();
    term_prefetch.clear();
    term_cache.clear();
  }
  ~dmrg_ctx() { for (auto& kv : term_prefetch) if (kv.second.valid()) kv.second.wait(); }
  std::shared_ptr<dmrg::HostPool> host_pool;         // host tier (cfg.env_host_bytes > 0)
  int64_t n_spills = 0, n_fetches = 0;
  uint64_t cache_bytes() const {      // device-resident bytes of the cached blocks
    uint64_t b = 0;
    for (auto& kv : left_cache) if (!kv.second->spilled) b += kv.second->bytes();
    for (auto& kv : right_cache) if (!kv.second->spilled) b += kv.second->bytes();
    return b;
  }
  void invalidate_site(int i) {     // site tensor i changed
    if (k > 0 && (i <= k - 1 || i >= k + 2)) {   // it lies inside a block of the prepared problem: that problem is gone
      k = 0; left.reset(); right.reset(); apply_plan.clear();
    }
    for (auto it = left_cache.begin(); it != left_cache.end();) it = it->first >= i ? left_cache.erase(it) : std::next(it);
    for (auto it = right_cache.begin(); it != right_cache.end();) it = it->first <= i ? right_cache.erase(it) : std::next(it);
  }
  dmrg::SiteOpTable site_ops;
  dmrg::CentreFactor centre;                    // dmrg_truncate_bond -> dmrg_start_vector
  // two-site problem
  std::vector<dmrg::PsiBlk> psi;
  std::map<std::array<int, 3>, int> psi_find;   // (qL, s1, s2) -> block
  std::map<std::array<int, 5>, int> psi_find5;  // SU(2): (qL, m1, 2S of L', m2, qR) -> block
  bool su2() const { return cfg.symmetry == 1; }
  long long psi_n = 0, psi_np = 0;
  dmrg::DevArray<dmrg::PsiBlockDev> d_psi_blocks;
  dmrg::DevArray<double> psi_in_p, psi_out_p, diag_p;
  dmrg::WsArena ws_arena;                       // declared before every plan that may lease it (destroyed after them)
  dmrg::Plan apply_plan;
  // output-block sharding of the apply over ranks (dmrg_set_shard); psi_owner[block] = rank that computes it
  int shard_rank = 0, shard_count = 1;
  dmrg_reduce_fn reduce_cb = nullptr;
  void* reduce_user = nullptr;
  std::vector<int> psi_owner;
  std::vector<double> shard_flops;               // analytic flops per rank of the prepared problem
  std::vector<double> blk_flops;                 // analytic flops per output block of the prepared problem (all ranks' tasks)
  dmrg::Exec exec;                              // worker streams (plan.h)
  dmrg::Exec* ex() { return exec.ok ? &exec : nullptr; }
  dmrg_stats_t stats{};
  int64_t launches = 0;
  // Davidson workspace
  dmrg::DevArray<double> dav_V, dav_W, dav_tmp, dav_small, dav_partials;
  int dav_basis = 0;
};
