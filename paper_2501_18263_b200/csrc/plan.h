// Contraction planner: turns "C += alpha * X*Y*W" items (Eq. (8) tasks and the
// renormalisation triple products of PAPER.md:99) into launches of the grouped GEMM kernel.
//
// A three-matrix item is executed in two phases inside one workspace chunk:
//   phase 1:  Z[b] = X[b]*Y[b]   (or Y[b]*W[b], whichever order is cheaper)   -> workspace
//   phase 2:  C   += alpha * Z[b]*W[b]   (or X[b]*Z[b])
// Items that accumulate into the same output become K-segments of ONE output tile, so the sum over
// terms stays in registers (no global atomics).  Chunks bound the workspace; outputs accumulate
// across chunks (they are zeroed by the caller before the plan runs).
#pragma once
#include <cstdlib>
#include <map>
#include <memory>
#include <tuple>

#include "common.h"
#include "fused.cuh"
#include "gemm.cuh"
#include "kernels.cuh"

namespace dmrg {

// A matrix operand.  Logical shape is (rows x cols) AFTER the optional transpose; `p` points to the
// stored row-major array with leading dimension ld; element b of a batch is at p + b*stride.
struct Mat {
  const double* p = nullptr;
  int ld = 0;
  bool tr = false;          // stored array is the transpose of the logical matrix
  long long stride = 0;
  int rows = 0, cols = 0;   // padded logical dims (multiples of 8)
  int urows = 0, ucols = 0; // unpadded logical dims (for the analytic flop count)
};

struct Item {
  double* C = nullptr;
  int ldc = 0;
  long long strideC = 0;    // 0: all `count` products accumulate into the same C; else batch of outputs
  int count = 1;
  double alpha = 1.0;
  int nmat = 2;             // C += alpha X*Y (2) or alpha X*Y*W (3)
  Mat X, Y, W;
};

// analytic flops of an item: the cheaper contraction order on the true (unpadded) dims
inline double item_flops(const Item& it) {
  auto fl = [](double m, double k, double n) { return 2.0 * m * k * n; };
  if (it.nmat == 2) return it.count * fl(it.X.urows, it.X.ucols, it.Y.ucols);
  const double left = fl(it.X.urows, it.X.ucols, it.Y.ucols) + fl(it.X.urows, it.Y.ucols, it.W.ucols);
  const double right = fl(it.Y.urows, it.Y.ucols, it.W.ucols) + fl(it.X.urows, it.X.ucols, it.W.ucols);
  return it.count * std::min(left, right);
}

struct Phase {
  DevArray<GOut> outs;
  DevArray<GSeg> segs;
  DevArray<GTile> tiles[GEMM_NSHAPES];   // one tile list per tile shape, heaviest tiles first
  int ntiles[GEMM_NSHAPES] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  double shape_flops[GEMM_NSHAPES] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // flops the tiles of each launch execute
  double shape_flops_full[GEMM_NSHAPES] = {0, 0, 0, 0, 0, 0, 0, 0, 0};   // same with every tile counted at its full BM x BN
  DevArray<RedDesc> red;                  // split-K partial sums to fold into the outputs afterwards
  int nred = 0, red_max_batch = 1;
  int launches() const { int n = nred > 0; for (int s = 0; s < GEMM_NSHAPES; ++s) n += ntiles[s] > 0; return n; }
};

struct Chunk {
  Phase p1, p2;
};

// Outputs whose whole task list runs in the fused small-sector kernel (fused.cuh): one launch per tile class,
// before the two-phase chunks (both accumulate into the same outputs, so the stages run one after the other).
struct FusedPhase {
  DevArray<FOut> outs;
  DevArray<FTask> tasks;
  DevArray<int2> order[FUSED_NCLASSES];     // (output, first row of the strip) work items of each class, heaviest first
  int nouts[FUSED_NCLASSES] = {};           // number of work items (warps)
  double cls_flops[FUSED_NCLASSES] = {};    // flops the launch of each class executes (padded dims)
  DevArray<RedDesc> red;
  int nred = 0;
  int64_t ntasks = 0;
  int launches() const { int n = nred > 0; for (int c = 0; c < FUSED_NCLASSES; ++c) n += nouts[c] > 0; return n; }
  void clear() { outs.release(); tasks.release(); red.release(); nred = 0; ntasks = 0;
                 for (int c = 0; c < FUSED_NCLASSES; ++c) { order[c].release(); nouts[c] = 0; cls_flops[c] = 0; } }
};

// Worker streams for running the independent launches of a plan stage concurrently (fork/join with
// events around the caller's stream).  Kernels of different tile shapes have very different grid
// sizes; run back to back each one ends in its own under-filled tail, run side by side they fill it.
struct Exec {
  static constexpr int NW = 6;
  cudaStream_t w[NW] = {};
  cudaEvent_t fork = nullptr, join[NW] = {};
  std::vector<cudaEvent_t> pool;      // per-chunk events of Plan::run's two lanes (created on first use, kept)
  cudaEvent_t event(size_t i);
  bool ok = false;
  void init();
  ~Exec();
};

// Workspace arena of a context: the intermediates of one plan at a time live in ONE device block that outlasts the
// plans (a blocking step, then the two-site problem of the next bond, ...), instead of one allocation of tens of GB
// per plan through the caller's allocator (measured: 90 ms of cudaMalloc per fresh workspace behind torch, and
// fragmentation over a sweep).  A plan leases it; a second plan built while the lease is out allocates its own.
struct WsArena {
  DevArray<double> buf;
  bool in_use = false;
};
struct WsArenaRelease { void operator()(WsArena* a) const { if (a) a->in_use = false; } };
using WsLease = std::unique_ptr<WsArena, WsArenaRelease>;

// One kernel launch of a plan, timed with CUDA events (dmrg_apply_profile).
struct LaunchRecord { int chunk, phase, shape, ntiles; double flops; float ms; };

struct Plan {
  std::vector<Chunk> chunks;
  FusedPhase fused;
  DevArray<double> workspace, scratch;   // workspace: only when the plan could not lease the context's arena
  WsLease lease;                         // the arena this plan's intermediates live in (released with the plan)
  bool print_stats = false;   // DMRG_B200_PLAN_STATS: per-shape tile fill printed when a plan is built
  long long ws_half = 0;   // elements per workspace half (two halves when there are several chunks)
  double flops_analytic = 0, flops_executed = 0, bytes_intermediate = 0;
  double flops_shared = 0;   // phase-1 flops saved by sharing intermediates between term groups
  int64_t n_items = 0, n_products = 0;
  int launches() const;
  // Two lanes on the worker streams of `ex` (nullptr: everything in order on `st`): lane A runs phase 1 of the
  // chunks, lane B phase 2 and the split-K reductions.  Dependencies are per chunk, by events: phase 1 of chunk c
  // needs workspace half c&1 back (phase 2 of chunk c-2 done), phase 2 of chunk c needs phase 1 of chunk c and
  // phase 2 of chunk c-1 (outputs accumulate in chunk order: no atomics, fixed order).  No stage-wide joins:
  // the tail of one launch is filled by whatever the other lane has ready.
  void run(cudaStream_t st, int64_t* launch_counter, Exec* ex = nullptr) const;
  // Same launches, each bracketed by events (shape -1 = split-K reduction).  Synchronises `st`.
  void run_profiled(cudaStream_t st, std::vector<LaunchRecord>* out) const;
  void clear() { chunks.clear(); fused.clear(); workspace.release(); scratch.release(); lease.reset(); }
};

class Planner {
 public:
  // A chunk may use half the cap: consecutive chunks alternate between two workspace halves.
  Planner(Allocator* al, uint64_t workspace_cap_bytes, WsArena* arena = nullptr)
      : al_(al), cap_(workspace_cap_bytes / 16), arena_(arena) {}
  void add(const Item& it);
  // Uploads descriptors, allocates the workspace and patches workspace-relative pointers.
  void finish(Plan* plan, cudaStream_t st);

 private:
  struct HSeg { GSeg s; bool a_ws, b_ws; };          // *_ws: pointer is a workspace offset
  struct HOut { GOut o; bool c_ws; std::vector<HSeg> segs; int batch; double work; bool c_sc = false; };
  // identity of a phase-1 product (operands, shapes, batch): equal keys give the same intermediate
  struct ZKey {
    const double* a; const double* b; long long sa, sb; int lda, ldb, rows, k, cols, cnt, flags;
    bool operator==(const ZKey& o) const {
      return a == o.a && b == o.b && sa == o.sa && sb == o.sb && lda == o.lda && ldb == o.ldb && rows == o.rows && k == o.k &&
             cols == o.cols && cnt == o.cnt && flags == o.flags;
    }
  };
  struct ZHash {
    size_t operator()(const ZKey& z) const {
      uint64_t h = (uint64_t)(uintptr_t)z.a * 0x9E3779B97F4A7C15ull ^ ((uint64_t)(uintptr_t)z.b + 0x7F4A7C15ull) * 0xC2B2AE3D27D4EB4Full;
      h ^= ((uint64_t)z.cnt << 40) ^ ((uint64_t)z.rows << 20) ^ (uint64_t)z.cols ^ ((uint64_t)z.flags << 60) ^ ((uint64_t)z.k << 8);
      return (size_t)(h ^ (h >> 29));
    }
  };
  struct P2Key {
    const double* c; int batch; long long stride;
    bool operator==(const P2Key& o) const { return c == o.c && batch == o.batch && stride == o.stride; }
  };
  struct P2Hash {
    size_t operator()(const P2Key& k) const {
      uint64_t h = (uint64_t)(uintptr_t)k.c * 0x9E3779B97F4A7C15ull ^ ((uint64_t)k.batch << 48) ^ (uint64_t)k.stride;
      return (size_t)(h ^ (h >> 31));
    }
  };
  struct HChunk {
    std::unordered_map<ZKey, long long, ZHash> zmap;     // intermediates already in this chunk's workspace
    std::vector<HOut> p1;
    std::vector<HOut> p2;
    std::unordered_map<P2Key, int, P2Hash> p2_index;     // (C, batch, strideC) -> p2 slot
    std::map<const double*, const double*> batched_out;   // [begin, end) of the batched outputs of this chunk
    long long ws_used = 0;
  };
  void add_piece(const Item& it, int b0, int cnt);
  bool add_fused(const Item& it);
  struct HFOut { double* C; int ldc, M, N; std::vector<FTask> tasks; };
  std::vector<HFOut> fused_;
  std::unordered_map<const double*, int> fused_index_;
  bool fused_on_ = std::getenv("DMRG_B200_NO_FUSED") == nullptr;
  // largest output dimension / largest contraction extent routed to the fused kernel (measured: DESIGN.md §7)
  int fused_max_ = std::getenv("DMRG_B200_FUSED_MAX") ? std::atoi(std::getenv("DMRG_B200_FUSED_MAX")) : 64;
  int fused_maxk_ = std::getenv("DMRG_B200_FUSED_MAXK") ? std::atoi(std::getenv("DMRG_B200_FUSED_MAXK")) : 64;
  HOut& p2_out(HChunk& ch, const Item& it, int b0, int cnt, int M, int N);
  Allocator* al_;
  long long cap_;
  WsArena* arena_ = nullptr;
  std::vector<HChunk> chunks_;
  long long ws_max_ = 0;
  double fa_ = 0, fe_ = 0, bi_ = 0, fshared_ = 0;
  bool share_z_ = std::getenv("DMRG_B200_NO_ZSHARE") == nullptr;
  int64_t n_items_ = 0, n_products_ = 0;
};

}  // namespace dmrg
