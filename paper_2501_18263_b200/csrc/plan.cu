#include "plan.h"

#include <algorithm>
#include <cstdlib>
#include <numeric>

namespace dmrg {

int Plan::launches() const {
  int n = fused.launches();
  for (const auto& c : chunks) n += c.p1.launches() + c.p2.launches();
  return n;
}

void Exec::init() {
  if (ok) return;
  for (int i = 0; i < NW; ++i) {
    DMRG_CUDA(cudaStreamCreateWithFlags(&w[i], cudaStreamNonBlocking));
    DMRG_CUDA(cudaEventCreateWithFlags(&join[i], cudaEventDisableTiming));
  }
  DMRG_CUDA(cudaEventCreateWithFlags(&fork, cudaEventDisableTiming));
  ok = true;
}
cudaEvent_t Exec::event(size_t i) {
  while (pool.size() <= i) {
    cudaEvent_t e;
    DMRG_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    pool.push_back(e);
  }
  return pool[i];
}
Exec::~Exec() {
  for (auto e : pool) cudaEventDestroy(e);
  if (!ok) return;
  for (int i = 0; i < NW; ++i) { cudaStreamDestroy(w[i]); cudaEventDestroy(join[i]); }
  cudaEventDestroy(fork);
}

namespace {
// Tiles per CTA: long lists of short tiles are batched so that the producer warp's prefetch runs across
// tile boundaries; keep >= 16 CTAs per resident slot for load balance.
int tiles_per_cta(int shape, int ntiles) {
  const int slots = 148 * gemm_shape_ctas_per_sm(shape);
  return std::max(1, std::min(16, ntiles / (slots * 16)));
}
cudaError_t launch_shape(const Phase& ph, int s, cudaStream_t st) {
  return launch_grouped_gemm(s, ph.outs.p, ph.segs.p, ph.tiles[s].p, ph.ntiles[s], tiles_per_cta(s, ph.ntiles[s]), st);
}
struct Launch { const Phase* ph; int shape; double work; };
void collect(const Phase& ph, std::vector<Launch>& v) {
  for (int s = GEMM_NSHAPES - 1; s >= 0; --s)
    if (ph.ntiles[s] > 0) v.push_back(Launch{&ph, s, ph.shape_flops[s]});
}
}  // namespace

// fused small-sector stage: the launches of the tile classes are independent (disjoint outputs)
static void run_fused(const FusedPhase& f, cudaStream_t st, int64_t* launch_counter, Exec* ex) {
  int nl = 0;
  for (int c = 0; c < FUSED_NCLASSES; ++c) nl += f.nouts[c] > 0;
  if (nl == 0) return;
  if (launch_counter) *launch_counter += nl + (f.nred > 0);
  if (!ex || nl == 1) {
    for (int c = FUSED_NCLASSES - 1; c >= 0; --c)
      DMRG_CUDA(launch_fused(c, f.outs.p, f.tasks.p, f.order[c].p, f.nouts[c], st));
  } else {
    DMRG_CUDA(cudaEventRecord(ex->fork, st));
    const int nw = std::min<int>(Exec::NW, nl);
    for (int i = 0; i < nw; ++i) DMRG_CUDA(cudaStreamWaitEvent(ex->w[i], ex->fork, 0));
    int w = 0;
    for (int c = FUSED_NCLASSES - 1; c >= 0; --c) {
      if (f.nouts[c] <= 0) continue;
      DMRG_CUDA(launch_fused(c, f.outs.p, f.tasks.p, f.order[c].p, f.nouts[c], ex->w[w % nw]));
      ++w;
    }
    for (int i = 0; i < nw; ++i) {
      DMRG_CUDA(cudaEventRecord(ex->join[i], ex->w[i]));
      DMRG_CUDA(cudaStreamWaitEvent(st, ex->join[i], 0));
    }
  }
  if (f.nred > 0) launch_reduce_partials(f.red.p, f.nred, 1, st);
}

void Plan::run(cudaStream_t st, int64_t* launch_counter, Exec* ex) const {
  const int n = (int)chunks.size();
  run_fused(fused, st, launch_counter, ex);
  if (n == 0) return;
  if (!ex) {
    for (int c = 0; c < n; ++c)
      for (int p = 0; p < 2; ++p) {
        const Phase& ph = p ? chunks[c].p2 : chunks[c].p1;
        std::vector<Launch> ls;
        collect(ph, ls);
        if (launch_counter) *launch_counter += (int64_t)ls.size() + (ph.nred > 0);
        for (auto& l : ls) DMRG_CUDA(launch_shape(*l.ph, l.shape, st));
        if (ph.nred > 0) launch_reduce_partials(ph.red.p, ph.nred, ph.red_max_batch, st);
      }
    return;
  }
  constexpr int LA = Exec::NW / 2, LB = Exec::NW - LA;        // streams of lane A (phase 1) / lane B (phase 2)
  auto evA = [&](int c, int i) { return ex->event((size_t)c * (LA + LB + 1) + i); };
  auto evB = [&](int c, int j) { return ex->event((size_t)c * (LA + LB + 1) + LA + j); };
  auto evDone = [&](int c) { return ex->event((size_t)c * (LA + LB + 1) + LA + LB); };
  DMRG_CUDA(cudaEventRecord(ex->fork, st));
  for (int c = 0; c < n; ++c) {
    // ---- lane A: phase 1 of chunk c ----
    {
      std::vector<Launch> ls;
      collect(chunks[c].p1, ls);
      std::stable_sort(ls.begin(), ls.end(), [](const Launch& a, const Launch& b) { return a.work > b.work; });
      if (launch_counter) *launch_counter += (int64_t)ls.size();
      for (int i = 0; i < LA; ++i)
        DMRG_CUDA(cudaStreamWaitEvent(ex->w[i], c < 2 ? ex->fork : evDone(c - 2), 0));
      for (size_t q = 0; q < ls.size(); ++q) DMRG_CUDA(launch_shape(*ls[q].ph, ls[q].shape, ex->w[q % LA]));
      for (int i = 0; i < LA; ++i) DMRG_CUDA(cudaEventRecord(evA(c, i), ex->w[i]));
    }
    // ---- lane B: phase 2 of chunk c, then its split-K reduction ----
    {
      const Phase& ph = chunks[c].p2;
      std::vector<Launch> ls;
      collect(ph, ls);
      std::stable_sort(ls.begin(), ls.end(), [](const Launch& a, const Launch& b) { return a.work > b.work; });
      if (launch_counter) *launch_counter += (int64_t)ls.size() + (ph.nred > 0);
      for (int j = 0; j < LB; ++j) {
        for (int i = 0; i < LA; ++i) DMRG_CUDA(cudaStreamWaitEvent(ex->w[LA + j], evA(c, i), 0));
        if (c > 0) DMRG_CUDA(cudaStreamWaitEvent(ex->w[LA + j], evDone(c - 1), 0));
      }
      for (size_t q = 0; q < ls.size(); ++q) DMRG_CUDA(launch_shape(*ls[q].ph, ls[q].shape, ex->w[LA + q % LB]));
      for (int j = 1; j < LB; ++j) {
        DMRG_CUDA(cudaEventRecord(evB(c, j), ex->w[LA + j]));
        DMRG_CUDA(cudaStreamWaitEvent(ex->w[LA], evB(c, j), 0));
      }
      if (ph.nred > 0) launch_reduce_partials(ph.red.p, ph.nred, ph.red_max_batch, ex->w[LA]);
      DMRG_CUDA(cudaEventRecord(evDone(c), ex->w[LA]));
    }
  }
  DMRG_CUDA(cudaStreamWaitEvent(st, evDone(n - 1), 0));
  for (int i = 0; i < LA; ++i) DMRG_CUDA(cudaStreamWaitEvent(st, evA(n - 1, i), 0));
}

void Plan::run_profiled(cudaStream_t st, std::vector<LaunchRecord>* out) const {
  std::vector<cudaEvent_t> ev;
  auto mark = [&]() {
    cudaEvent_t e;
    DMRG_CUDA(cudaEventCreate(&e));
    DMRG_CUDA(cudaEventRecord(e, st));
    ev.push_back(e);
  };
  out->clear();
  mark();
  for (int c = FUSED_NCLASSES - 1; c >= 0; --c) {     // phase 3 = fused small-sector kernel, shape = tile class
    if (fused.nouts[c] <= 0) continue;
    DMRG_CUDA(launch_fused(c, fused.outs.p, fused.tasks.p, fused.order[c].p, fused.nouts[c], st));
    mark();
    out->push_back(LaunchRecord{0, 3, c, fused.nouts[c], fused.cls_flops[c], 0.f});
  }
  if (fused.nred > 0) {
    launch_reduce_partials(fused.red.p, fused.nred, 1, st);
    mark();
    out->push_back(LaunchRecord{0, 3, -1, fused.nred, 0.0, 0.f});
  }
  for (size_t c = 0; c < chunks.size(); ++c)
    for (int p = 0; p < 2; ++p) {
      const Phase& ph = p == 0 ? chunks[c].p1 : chunks[c].p2;
      for (int s = GEMM_NSHAPES - 1; s >= 0; --s) {
        if (ph.ntiles[s] <= 0) continue;
        DMRG_CUDA(launch_shape(ph, s, st));
        mark();
        out->push_back(LaunchRecord{(int)c, p + 1, s, ph.ntiles[s], ph.shape_flops[s], 0.f});
      }
      if (ph.nred > 0) {
        launch_reduce_partials(ph.red.p, ph.nred, ph.red_max_batch, st);
        mark();
        out->push_back(LaunchRecord{(int)c, p + 1, -1, ph.nred, 0.0, 0.f});
      }
    }
  DMRG_CUDA(cudaStreamSynchronize(st));
  for (size_t i = 0; i < out->size(); ++i) DMRG_CUDA(cudaEventElapsedTime(&(*out)[i].ms, ev[i], ev[i + 1]));
  for (auto e : ev) cudaEventDestroy(e);
}

static inline double fl(double a, double b, double c) { return 2.0 * a * b * c; }

// Splits an extent (multiple of 8) into tile rows/cols of class 0/1/2 = 32/64/128: (start, class).
static void split_dim(int n, std::vector<std::pair<int, int>>& out) {
  int pos = 0;
  while (pos < n) {
    int rem = n - pos;
    if (rem > 96) { out.push_back({pos, 2}); pos += 128; }
    else if (rem > 32) { out.push_back({pos, 1}); pos += 64; }
    else { out.push_back({pos, 0}); pos += 32; }
  }
}

void Planner::add(const Item& it) {
  DMRG_REQUIRE(it.count >= 1, DMRG_ERR_ARG, "planner: empty item");
  ++n_items_;
  n_products_ += it.count;
  if (add_fused(it)) return;
  if (it.nmat == 2) {
    fa_ += item_flops(it);
    add_piece(it, 0, it.count);
    return;
  }
  // analytic flops: the cheaper order on the true (unpadded) dims
  fa_ += item_flops(it);
  // workspace per product, in the order the kernels will use (padded dims)
  double pl = fl(it.X.rows, it.X.cols, it.Y.cols) + fl(it.X.rows, it.Y.cols, it.W.cols);
  double pr = fl(it.Y.rows, it.Y.cols, it.W.cols) + fl(it.X.rows, it.X.cols, it.W.cols);
  long long zsz = (pl <= pr) ? (long long)it.X.rows * it.Y.cols : (long long)it.Y.rows * it.W.cols;
  DMRG_REQUIRE(zsz <= cap_, DMRG_ERR_ALLOC, "planner: workspace cap smaller than one intermediate block");
  int per = (int)std::min<long long>(it.count, cap_ / zsz);
  for (int b0 = 0; b0 < it.count; b0 += per) add_piece(it, b0, std::min(per, it.count - b0));
}

// Items whose every dimension fits one tile of the fused kernel (<= 64 after padding) and that accumulate into one
// output (not a batch of outputs) join that output's task list; the intermediate X*Y never leaves the SM.
bool Planner::add_fused(const Item& it) {
  if (!fused_on_ || it.strideC != 0) return false;
  const int DMAX = fused_max_, KMAX = fused_maxk_;
  FTask t{};
  int M, N;
  if (it.nmat == 3) {
    M = it.X.rows; N = it.W.cols;
    if (N > FUSED_MAX_N || M > DMAX || N > DMAX || it.X.cols > KMAX || it.Y.cols > KMAX) return false;
    t.A = it.X.p; t.rsA = it.X.stride; t.lda = it.X.ld;
    t.P = it.Y.p; t.rsP = it.Y.stride; t.ldp = it.Y.ld;
    t.B = it.W.p; t.rsB = it.W.stride; t.ldb = it.W.ld;
    t.mi = (short)it.X.cols; t.ni = (short)it.Y.cols;
    t.flags = (it.X.tr ? 1 : 0) | (it.Y.tr ? 2 : 0) | (it.W.tr ? 4 : 0);
    fe_ += it.count * (fl(M, it.X.cols, it.Y.cols) + fl(M, it.Y.cols, N));
  } else {
    M = it.X.rows; N = it.Y.cols;
    if (N > FUSED_MAX_N || M > DMAX || N > DMAX || it.X.cols > KMAX) return false;
    t.A = nullptr; t.rsA = 0; t.lda = 0;
    t.P = it.X.p; t.rsP = it.X.stride; t.ldp = it.X.ld;
    t.B = it.Y.p; t.rsB = it.Y.stride; t.ldb = it.Y.ld;
    t.mi = 0; t.ni = (short)it.X.cols;
    t.flags = (it.X.tr ? 2 : 0) | (it.Y.tr ? 4 : 0);
    fe_ += it.count * fl(M, it.X.cols, N);
  }
  t.count = it.count; t.alpha = it.alpha;
  fa_ += item_flops(it);
  auto f = fused_index_.find(it.C);
  if (f == fused_index_.end()) {
    f = fused_index_.emplace(it.C, (int)fused_.size()).first;
    fused_.push_back(HFOut{it.C, it.ldc, M, N, {}});
  }
  HFOut& o = fused_[f->second];
  DMRG_REQUIRE(o.M == M && o.N == N && o.ldc == it.ldc, DMRG_ERR_ARG, "planner: one output with two shapes");
  o.tasks.push_back(t);
  return true;
}

Planner::HOut& Planner::p2_out(HChunk& ch, const Item& it, int b0, int cnt, int M, int N) {
  const bool batched = it.strideC != 0;
  double* C = it.C + (batched ? b0 * it.strideC : 0);
  const P2Key key{(const double*)C, batched ? cnt : 1, it.strideC};
  auto f = ch.p2_index.find(key);
  if (f != ch.p2_index.end()) return ch.p2[f->second];
  HOut o{};
  o.o.C = C; o.o.bsC = batched ? it.strideC : 0;
  o.o.M = M; o.o.N = N; o.o.ldc = it.ldc; o.o.accumulate = 1;
  o.c_ws = false; o.batch = batched ? cnt : 1; o.work = 0;
  ch.p2_index[key] = (int)ch.p2.size();
  ch.p2.push_back(std::move(o));
  return ch.p2.back();
}

void Planner::add_piece(const Item& it, int b0, int cnt) {
  if (chunks_.empty()) chunks_.emplace_back();
  const bool batched = it.strideC != 0;
  if (batched) {
    // Batched outputs of one chunk must be identical or disjoint: each becomes its own list of output tiles, and two
    // lists that overlap would read-modify-write the same C tiles from different CTAs of one launch.  The callers'
    // runs are disjoint-or-identical, but the workspace split of Planner::add cuts different items at different
    // places; a piece that overlaps an output of the current chunk without being equal to it opens a new chunk
    // (phase 2 of consecutive chunks runs in order).
    const double* lo = it.C + (long long)b0 * it.strideC;
    const double* hi = lo + (long long)cnt * it.strideC;
    auto conflict = [&](const HChunk& ch) {
      auto f = ch.batched_out.lower_bound(lo);
      if (f != ch.batched_out.begin()) {
        auto pv = std::prev(f);
        if (pv->second > lo) return true;                       // starts earlier, reaches into [lo, hi)
      }
      if (f != ch.batched_out.end() && f->first < hi && !(f->first == lo && f->second == hi)) return true;
      return false;
    };
    if (conflict(chunks_.back())) chunks_.emplace_back();
    chunks_.back().batched_out[lo] = hi;
  }
  auto mkseg = [](const double* A, int lda, bool ta, const double* B, int ldb, bool tb, int K) {
    HSeg h{};
    h.s.A = A; h.s.B = B; h.s.lda = lda; h.s.ldb = ldb; h.s.K = K; h.s.count = 1;
    h.s.flags = (ta ? 1 : 0) | (tb ? 2 : 0); h.s.alpha = 1.0;
    h.s.rsA = h.s.rsB = h.s.bsA = h.s.bsB = 0; h.a_ws = h.b_ws = false;
    h.s.ams = h.s.bns = 0; h.s.amr = h.s.bnr = 0; h.s.amr_inv = h.s.bnr_inv = 0;
    return h;
  };
  if (it.nmat == 2) {
    HOut& o = p2_out(chunks_.back(), it, b0, cnt, it.X.rows, it.Y.cols);
    HSeg h = mkseg(it.X.p + b0 * it.X.stride, it.X.ld, it.X.tr, it.Y.p + b0 * it.Y.stride, it.Y.ld,
                   it.Y.tr, it.X.cols);
    h.s.alpha = it.alpha;
    if (batched) { h.s.bsA = it.X.stride; h.s.bsB = it.Y.stride; }
    else { h.s.count = cnt; h.s.rsA = it.X.stride; h.s.rsB = it.Y.stride; }
    o.segs.push_back(h);
    fe_ += cnt * fl(it.X.rows, it.X.cols, it.Y.cols);
    return;
  }
  double pl = fl(it.X.rows, it.X.cols, it.Y.cols) + fl(it.X.rows, it.Y.cols, it.W.cols);
  double pr = fl(it.Y.rows, it.Y.cols, it.W.cols) + fl(it.X.rows, it.X.cols, it.W.cols);
  const bool left_first = pl <= pr;
  const int zr = left_first ? it.X.rows : it.Y.rows;
  const int zc = left_first ? it.Y.cols : it.W.cols;
  const long long zsz = (long long)zr * zc;
  bool shared = false;
  long long zoff_shared = 0;
  // phase 1: Z[b] = X[b] Y[b]  or  Y[b] W[b].  When only one operand varies with b the `cnt` products
  // are ONE GEMM: operators stacked along M (segmented rows of op(A)) or along N (segmented columns of
  // op(B)); the class storage keeps them contiguous per block, so no copy is needed.
  const Mat& A1 = left_first ? it.X : it.Y;
  const Mat& B1 = left_first ? it.Y : it.W;
  const double p1f = fl(A1.rows, A1.cols, B1.cols);
  // The same intermediate is needed by every term group that applies the same operator run to the same psi
  // block (e.g. a+_l psi for the G5, G12 and G13 patterns): inside a chunk it is computed once.
  const ZKey zkey{A1.p + b0 * A1.stride, B1.p + b0 * B1.stride, A1.stride, B1.stride, A1.ld, B1.ld, A1.rows, A1.cols,
                  B1.cols, cnt, (A1.tr ? 1 : 0) | (B1.tr ? 2 : 0)};
  if (share_z_) {
    auto f = chunks_.back().zmap.find(zkey);
    if (f != chunks_.back().zmap.end()) {
      shared = true;
      zoff_shared = f->second;
    }
  }
  if (!shared && chunks_.back().ws_used + zsz * cnt > cap_) chunks_.emplace_back();
  HChunk& ch = chunks_.back();
  const long long zoff = shared ? zoff_shared : ch.ws_used;
  // (the kernel divides a stacked row index x < cnt * zr by zr with one umulhi, exact for x * zr < 2^32)
  const bool mergeM = cnt > 1 && A1.stride != 0 && B1.stride == 0 && (unsigned long long)cnt * zr * zr < (1ull << 32);
  const bool mergeN = cnt > 1 && A1.stride == 0 && B1.stride != 0 && (unsigned long long)cnt * zc * zc < (1ull << 32);
  const long long zld = mergeN ? (long long)cnt * zc : zc;       // leading dimension of Z
  const long long zstep = mergeN ? zc : zsz;                      // offset of Z[b] relative to Z[0]
  if (shared) {
    fe_ += cnt * (std::min(pl, pr) - p1f);
    bi_ += 8.0 * zsz * cnt;                                       // read once more in phase 2
    fshared_ += cnt * p1f;
  } else {
    ch.ws_used += zsz * cnt;
    ws_max_ = std::max(ws_max_, ch.ws_used);
    bi_ += 2.0 * 8.0 * zsz * cnt;
    fe_ += cnt * std::min(pl, pr);
    if (share_z_) ch.zmap.emplace(zkey, zoff);
    HOut z{};
    z.o.C = reinterpret_cast<double*>(zoff); z.c_ws = true;
    z.o.bsC = zsz; z.o.M = mergeM ? cnt * zr : zr; z.o.N = mergeN ? cnt * zc : zc; z.o.ldc = (int)zld;
    z.o.accumulate = 0;
    z.batch = (mergeM || mergeN) ? 1 : cnt; z.work = 0;
    HSeg h = mkseg(A1.p + b0 * A1.stride, A1.ld, A1.tr, B1.p + b0 * B1.stride, B1.ld, B1.tr, A1.cols);
    if (mergeM) {
      h.s.amr = zr; h.s.ams = A1.stride; h.s.amr_inv = (unsigned)(0x100000000ull / (unsigned)zr) + 1u;
    } else if (mergeN) {
      h.s.bnr = zc; h.s.bns = B1.stride; h.s.bnr_inv = (unsigned)(0x100000000ull / (unsigned)zc) + 1u;
    } else {
      h.s.bsA = A1.stride; h.s.bsB = B1.stride;
    }
    z.segs.push_back(h);
    ch.p1.push_back(std::move(z));
  }
  // phase 2: C += alpha Z[b] W[b]  or  alpha X[b] Z[b]
  HOut& o = p2_out(ch, it, b0, cnt, it.X.rows, it.W.cols);
  HSeg h;
  if (left_first) {
    h = mkseg(reinterpret_cast<const double*>(zoff), (int)zld, false, it.W.p + b0 * it.W.stride, it.W.ld,
              it.W.tr, zc);
    h.a_ws = true;
    if (batched) { h.s.bsA = zstep; h.s.bsB = it.W.stride; }
    else { h.s.count = cnt; h.s.rsA = zstep; h.s.rsB = it.W.stride; }
  } else {
    h = mkseg(it.X.p + b0 * it.X.stride, it.X.ld, it.X.tr, reinterpret_cast<const double*>(zoff), (int)zld,
              false, zr);
    h.b_ws = true;
    if (batched) { h.s.bsA = it.X.stride; h.s.bsB = zstep; }
    else { h.s.count = cnt; h.s.rsA = it.X.stride; h.s.rsB = zstep; }
  }
  h.s.alpha = it.alpha;
  o.segs.push_back(h);
}

void Planner::finish(Plan* plan, cudaStream_t st) {
  PhaseTimer pt("  planner.finish");
  plan->clear();
  plan->flops_analytic = fa_;
  plan->flops_executed = fe_;
  plan->bytes_intermediate = bi_;
  plan->flops_shared = fshared_;
  plan->n_items = n_items_;
  plan->n_products = n_products_;
  const bool two_halves = chunks_.size() > 1;
  plan->ws_half = ws_max_;
  double* ws = nullptr;
  if (ws_max_ > 0) {
    const size_t need = (size_t)ws_max_ * (two_halves ? 2 : 1);
    if (arena_ && !arena_->in_use) {
      // grow when the plan needs more; give the block back when it is far larger than what this plan may use at all
      // (the cap follows the memory the context has left: environment blocks may have grown since)
      const size_t limit = std::max<size_t>(need, 2 * (size_t)cap_);
      if (arena_->buf.n < need || arena_->buf.n > limit + limit / 4) {
        arena_->buf.release();
        arena_->buf.allocate(al_, need);
      }
      arena_->in_use = true;
      plan->lease.reset(arena_);
      ws = arena_->buf.p;
    } else {
      plan->workspace.allocate(al_, need);
      ws = plan->workspace.p;
    }
  }
  pt.lap("workspace allocation (the caller's allocator)");
  if (std::getenv("DMRG_B200_PLAN_STATS")) plan->print_stats = true;

  // ---- split-K: heavy outputs are cut into parts along their (segment, repeat) list so that one launch
  // has several CTAs per SM of comparable length.  Part 0 accumulates into C; the others write partial
  // sums to scratch, which a reduction kernel folds into C in a fixed order afterwards.
  struct HRed { RedDesc d; long long p_off; };
  std::vector<std::vector<HRed>> reds(chunks_.size());
  long long scratch_max = 0;
  for (size_t ci = 0; ci < chunks_.size(); ++ci) {
    std::vector<HOut>& hv = chunks_[ci].p2;
    // cost model of one tile: k-chunks x max(tile area, 8192) -- a narrow tile is latency-bound and takes
    // about as long per k-chunk as a 64x128 one.  Outputs are cut so that no tile part exceeds 1/64 of
    // the per-SM share of the chunk (at most 32 parts per output).
    double total = 0;
    std::vector<double> ks(hv.size()), mxa(hv.size()), contrib(hv.size());
    const long long nhv = (long long)hv.size();
    // (per-output terms in parallel, summed in index order below: the plan does not depend on the thread count)
#pragma omp parallel for schedule(static) if (nhv > 4096)
    for (long long i = 0; i < nhv; ++i) {
      double k = 0;
      for (auto& hs : hv[i].segs) k += (double)hs.s.K * hs.s.count;
      ks[i] = k;
      static thread_local std::vector<std::pair<int, int>> rs, cs;
      rs.clear(); cs.clear();
      split_dim(hv[i].o.M, rs); split_dim(hv[i].o.N, cs);
      double mx = 0, sum = 0;
      for (auto& r : rs) for (auto& c : cs) {
        double t = std::max(8192.0, (double)GEMM_DIMS[r.second] * GEMM_DIMS[c.second]);
        sum += k * t * hv[i].batch;
        mx = std::max(mx, t);
      }
      mxa[i] = mx;
      contrib[i] = sum;
    }
    for (long long i = 0; i < nhv; ++i) total += contrib[i];
    // (measured at 1/8, 1/16, 1/32, 1/64, 1/96, 1/128 of the per-SM share: configs[3] 527.9 / 496.8 / 488.4-489.3 /
    // 486.2-487.2 / 488.6 / 491.0 ms; configs[2] and SU(2) configs[3] are 1 % faster at 1/64 than at 1/32 as well)
    const double wstar = total / (148.0 * 64.0);
    // the parts of every heavy output are built on host threads (scratch offsets relative to the output's own
    // partial tiles), then appended in output order with the running scratch offset
    struct Split { long long out; int ns; std::vector<HOut> parts; HRed rd; long long sc_need = 0; };
    std::vector<Split> sp;                      // the outputs that are cut, in output order
    for (long long i = 0; i < nhv; ++i) {
      long long units = 0;
      for (auto& hs : hv[i].segs) units += hs.s.count;
      int ns = wstar > 0 ? (int)std::ceil(ks[i] * mxa[i] / wstar) : 1;
      ns = (int)std::min<long long>(std::min(ns, 32), units);
      if (ns > 1) { sp.emplace_back(); sp.back().out = i; sp.back().ns = ns; }
    }
    const long long nsp = (long long)sp.size();
#pragma omp parallel for schedule(dynamic, 64) if (nsp > 1024)
    for (long long q = 0; q < nsp; ++q) {
      Split& S = sp[q];
      const long long i = S.out;
      const int ns = S.ns;
      HOut& h = hv[i];
      const long long mn = (long long)h.o.M * h.o.N;
      S.rd.d.C = h.o.C; S.rd.d.bsC = h.o.bsC; S.rd.d.M = h.o.M; S.rd.d.N = h.o.N; S.rd.d.ldc = h.o.ldc;
      S.rd.d.nparts = ns - 1; S.rd.d.batch = h.batch; S.rd.p_off = 0;
      const double target = ks[i] / ns;
      size_t si = 0; int rep = 0;      // cursor into the (segment, repeat) list
      for (int p = 0; p < ns; ++p) {
        HOut part{};
        part.o = h.o; part.c_ws = false; part.batch = h.batch; part.work = 0;
        if (p > 0) {
          part.c_sc = true;
          part.o.C = reinterpret_cast<double*>((long long)(p - 1) * h.batch * mn);
          part.o.bsC = mn; part.o.ldc = h.o.N; part.o.accumulate = 0;
        }
        double got = 0;
        while (si < h.segs.size() && (p == ns - 1 || got < target)) {
          const HSeg& hs = h.segs[si];
          const int left = hs.s.count - rep;
          int take = left;
          if (p != ns - 1) {
            double room = target - got;
            take = (int)std::min<double>(left, std::max(1.0, std::floor(room / hs.s.K + 0.5)));
          }
          HSeg sub = hs;
          sub.s.count = take;
          if (rep > 0) {
            if (hs.a_ws) sub.s.A = reinterpret_cast<const double*>(reinterpret_cast<long long>(hs.s.A) + rep * hs.s.rsA);
            else sub.s.A = hs.s.A + rep * hs.s.rsA;
            if (hs.b_ws) sub.s.B = reinterpret_cast<const double*>(reinterpret_cast<long long>(hs.s.B) + rep * hs.s.rsB);
            else sub.s.B = hs.s.B + rep * hs.s.rsB;
          }
          part.segs.push_back(sub);
          got += (double)take * hs.s.K;
          rep += take;
          if (rep >= hs.s.count) { rep = 0; ++si; }
        }
        if (!part.segs.empty() || p == 0) S.parts.push_back(std::move(part));
        else S.rd.d.nparts = std::min(S.rd.d.nparts, p - 1);
      }
      S.sc_need = (long long)(ns - 1) * h.batch * mn;
    }
    std::vector<HOut> ex;
    ex.reserve(hv.size());
    long long sc_used = 0;
    size_t nq = 0;
    for (size_t i = 0; i < hv.size(); ++i) {
      if (nq >= sp.size() || sp[nq].out != (long long)i) { ex.push_back(std::move(hv[i])); continue; }
      Split& S = sp[nq++];
      S.rd.p_off = sc_used;
      reds[ci].push_back(S.rd);
      for (auto& part : S.parts) {
        if (part.c_sc) part.o.C = reinterpret_cast<double*>(reinterpret_cast<long long>(part.o.C) + sc_used);
        ex.push_back(std::move(part));
      }
      sc_used += S.sc_need;
    }
    hv.swap(ex);
    scratch_max = std::max(scratch_max, sc_used);
  }
  pt.lap("split-K");
  // ---- fused small-sector outputs: tile class, split of heavy task lists into parts, launch order ----
  struct FPart { int out; bool partial; long long sc_off; std::vector<FTask> tasks; double cost; int cls; };
  std::vector<FPart> fparts;
  struct FRed { int out; long long sc_off; int nparts; };
  std::vector<FRed> freds;
  long long fsc_used = 0;
  {
    // cost of one repeat for ONE strip (a warp): MACs + an overhead per task (descriptor, first-fragment latency)
    auto unit_cost = [](const HFOut& o, const FTask& t, int rows) {
      return rows * ((t.A ? (double)t.mi * t.ni : 0.0) + (double)t.ni * o.N) + 2048.0;
    };
    std::vector<int> cls(fused_.size());
    std::vector<double> cost(fused_.size(), 0.0);
    double cls_total[FUSED_NCLASSES] = {};
    for (size_t i = 0; i < fused_.size(); ++i) {
      const HFOut& o = fused_[i];
      const int c = o.N / 8 - 1;
      cls[i] = c;
      const int rows = FUSED_STRIP;
      for (auto& t : o.tasks) cost[i] += t.count * unit_cost(o, t, rows);
      cls_total[c] += cost[i] * ((o.M + rows - 1) / rows);
    }
    for (size_t i = 0; i < fused_.size(); ++i) {
      HFOut& o = fused_[i];
      // aim at ~6 work items per resident warp of the class, all of about the same length (measured at 1.5 / 3 / 6 /
      // 12 / 24: configs[1] 0.598 / 0.543 / 0.532 / 0.531 / 0.533 ms, configs[2] 13.49 / 13.33 / 13.25 / 13.25 / 13.25 ms)
      const int rows = FUSED_STRIP;
      const double target = std::max(cls_total[cls[i]] / (148.0 * fused_warps_per_sm(cls[i]) * 6.0), 1.0);
      long long units = 0;
      for (auto& t : o.tasks) units += t.count;
      int ns = (int)std::min<long long>(std::min<long long>((long long)std::ceil(cost[i] / target), 64), units);
      if (ns < 1) ns = 1;
      const long long mn = (long long)o.M * o.N;
      if (ns > 1) { freds.push_back(FRed{(int)i, fsc_used, ns - 1}); }
      const double per = cost[i] / ns;
      size_t ti = 0; int rep = 0;
      int made = 0;
      for (int p = 0; p < ns; ++p) {
        FPart part{(int)i, p > 0, p > 0 ? fsc_used + (long long)(p - 1) * mn : 0, {}, 0.0, cls[i]};
        while (ti < o.tasks.size() && (p == ns - 1 || part.cost < per)) {
          const FTask& t = o.tasks[ti];
          const double uc = unit_cost(o, t, rows);
          const int left = t.count - rep;
          int take = left;
          if (p != ns - 1) take = (int)std::min<double>(left, std::max(1.0, std::floor((per - part.cost) / uc + 0.5)));
          FTask sub = t;
          sub.count = take;
          if (sub.A) sub.A += (long long)rep * t.rsA;
          sub.P += (long long)rep * t.rsP;
          sub.B += (long long)rep * t.rsB;
          part.tasks.push_back(sub);
          part.cost += take * uc;
          rep += take;
          if (rep >= t.count) { rep = 0; ++ti; }
        }
        if (!part.tasks.empty()) { fparts.push_back(std::move(part)); ++made; }
      }
      if (ns > 1) {
        // parts that came out empty are at the end: the reduction folds only the partial tiles that were written
        freds.back().nparts = std::max(0, made - 1);
        fsc_used += (long long)(ns - 1) * mn;
      }
    }
    scratch_max = std::max(scratch_max, fsc_used);
  }
  pt.lap("fused parts");
  if (scratch_max > 0) plan->scratch.allocate(al_, (size_t)scratch_max);
  double* sc = plan->scratch.p;
  if (!fparts.empty()) {
    FusedPhase& F = plan->fused;
    std::vector<FOut> outs;
    std::vector<FTask> tasks;
    std::vector<std::pair<double, int>> ord[FUSED_NCLASSES];
    for (auto& pt : fparts) {
      const HFOut& o = fused_[pt.out];
      FOut fo{};
      fo.C = pt.partial ? sc + pt.sc_off : o.C;
      fo.ldc = pt.partial ? o.N : o.ldc;
      fo.M = o.M; fo.N = o.N;
      fo.accumulate = pt.partial ? 0 : 1;
      fo.task_begin = (int)tasks.size();
      for (auto& t : pt.tasks) {
        tasks.push_back(t);
        F.cls_flops[pt.cls] += t.count * ((t.A ? fl(o.M, t.mi, t.ni) : 0.0) + fl(o.M, t.ni, o.N));
      }
      fo.task_end = (int)tasks.size();
      ord[pt.cls].push_back({pt.cost, (int)outs.size()});
      outs.push_back(fo);
    }
    for (int c = 0; c < FUSED_NCLASSES; ++c) {
      std::stable_sort(ord[c].begin(), ord[c].end(), [](const std::pair<double, int>& a, const std::pair<double, int>& b) { return a.first > b.first; });
      std::vector<int2> o;
      for (auto& x : ord[c])
        for (int r0 = 0; r0 < outs[x.second].M; r0 += FUSED_STRIP) o.push_back(make_int2(x.second, r0));
      F.nouts[c] = (int)o.size();
      if (!o.empty()) F.order[c].upload(al_, o, st);
    }
    F.ntasks = (int64_t)tasks.size();
    F.outs.upload(al_, outs, st);
    F.tasks.upload(al_, tasks, st);
    std::vector<RedDesc> rd;
    for (auto& r : freds) {
      if (r.nparts <= 0) continue;
      const HFOut& o = fused_[r.out];
      RedDesc d{};
      d.C = o.C; d.P = sc + r.sc_off; d.bsC = 0; d.M = o.M; d.N = o.N; d.ldc = o.ldc; d.nparts = r.nparts; d.batch = 1;
      rd.push_back(d);
    }
    F.nred = (int)rd.size();
    if (!rd.empty()) F.red.upload(al_, rd, st);
    if (plan->print_stats)
      for (int c = 0; c < FUSED_NCLASSES; ++c)
        if (F.nouts[c])
          fprintf(stderr, "plan fused N = %d: %d warps, flops %.4g\n", 8 * (c + 1), F.nouts[c], F.cls_flops[c]);
  }
  fused_.clear();
  fused_index_.clear();
  // host side of one phase of one chunk: descriptors and per-shape tile lists (heaviest first).  Independent of every
  // other (chunk, phase), so all of them are built on host threads at once; the uploads follow in order.
  struct Built { std::vector<GOut> outs; std::vector<GSeg> segs; std::vector<GTile> tiles[GEMM_NSHAPES]; };
  auto build_host = [&](std::vector<HOut>& hv, Phase& ph, double* ws, Built& bt) {
    std::vector<GOut>& outs = bt.outs;
    std::vector<GSeg>& segs = bt.segs;
    struct TW { GTile t; double w; };
    std::vector<TW> tw[GEMM_NSHAPES];
    outs.reserve(hv.size());
    size_t nseg = 0;
    for (auto& h : hv) nseg += h.segs.size();
    segs.reserve(nseg);
    std::vector<std::pair<int, int>> rs, cs;
    for (size_t oi = 0; oi < hv.size(); ++oi) {
      HOut& h = hv[oi];
      GOut o = h.o;
      if (h.c_ws) o.C = ws + reinterpret_cast<long long>(h.o.C);
      if (h.c_sc) o.C = sc + reinterpret_cast<long long>(h.o.C);
      o.seg_begin = (int)segs.size();
      double ksum = 0;
      for (auto& hs : h.segs) {
        GSeg s = hs.s;
        if (hs.a_ws) s.A = ws + reinterpret_cast<long long>(hs.s.A);
        if (hs.b_ws) s.B = ws + reinterpret_cast<long long>(hs.s.B);
        ksum += (double)s.K * s.count;
        segs.push_back(s);
      }
      o.seg_end = (int)segs.size();
      outs.push_back(o);
      if (o.seg_begin == o.seg_end) continue;   // nothing to add: the kernel needs >= 1 k-chunk per tile
      rs.clear(); cs.clear();
      split_dim(o.M, rs);
      split_dim(o.N, cs);
      for (int b = 0; b < h.batch; ++b)
        for (auto& r : rs)
          for (auto& c : cs) {
            int shape = 3 * r.second + c.second;
            double w = ksum * GEMM_DIMS[r.second] * GEMM_DIMS[c.second];
            tw[shape].push_back({GTile{(int)oi, b, r.first, c.first}, w});
            ph.shape_flops[shape] += 2.0 * ksum * std::min(GEMM_DIMS[r.second], o.M - r.first) *
                                     std::min(GEMM_DIMS[c.second], o.N - c.first);
            ph.shape_flops_full[shape] += 2.0 * w;
          }
    }
    for (int s = 0; s < GEMM_NSHAPES; ++s) {
      std::stable_sort(tw[s].begin(), tw[s].end(), [](const TW& a, const TW& b) { return a.w > b.w; });
      bt.tiles[s].resize(tw[s].size());
      for (size_t i = 0; i < tw[s].size(); ++i) bt.tiles[s][i] = tw[s][i].t;
      ph.ntiles[s] = (int)bt.tiles[s].size();
    }
  };
  auto upload_built = [&](Built& bt, Phase& ph) {
    for (int s = 0; s < GEMM_NSHAPES; ++s)
      if (!bt.tiles[s].empty()) ph.tiles[s].upload(al_, bt.tiles[s], st);
    ph.outs.upload(al_, bt.outs, st);
    ph.segs.upload(al_, bt.segs, st);
    bt = Built{};
  };
  pt.lap("fused upload");
  plan->chunks.resize(chunks_.size());
  struct PS { double act = 0, full = 0; long long tiles = 0; } ps[2][GEMM_NSHAPES];
  std::vector<Built> built(2 * chunks_.size());
  const long long nbuild = (long long)built.size();
#pragma omp parallel for schedule(dynamic, 1) if (nbuild > 2)
  for (long long i = 0; i < nbuild; ++i) {
    const size_t c = (size_t)i / 2;
    double* wsc = ws + ((c & 1) ? ws_max_ : 0);   // chunk c works in workspace half c & 1
    if (i & 1) build_host(chunks_[c].p2, plan->chunks[c].p2, wsc, built[i]);
    else build_host(chunks_[c].p1, plan->chunks[c].p1, wsc, built[i]);
  }
  pt.lap("chunk tile lists (host threads)");
  for (size_t c = 0; c < chunks_.size(); ++c) {
    upload_built(built[2 * c], plan->chunks[c].p1);
    upload_built(built[2 * c + 1], plan->chunks[c].p2);
    if (!reds[c].empty()) {
      std::vector<RedDesc> rd;
      int mb = 1;
      for (auto& r : reds[c]) {
        if (r.d.nparts <= 0) continue;
        RedDesc d = r.d;
        d.P = sc + r.p_off;
        mb = std::max(mb, d.batch);
        rd.push_back(d);
      }
      plan->chunks[c].p2.nred = (int)rd.size();
      plan->chunks[c].p2.red_max_batch = mb;
      if (!rd.empty()) plan->chunks[c].p2.red.upload(al_, rd, st);
    }
    for (int p = 0; p < 2; ++p) {
      const Phase& ph = p ? plan->chunks[c].p2 : plan->chunks[c].p1;
      for (int sh = 0; sh < GEMM_NSHAPES; ++sh) {
        ps[p][sh].act += ph.shape_flops[sh]; ps[p][sh].full += ph.shape_flops_full[sh]; ps[p][sh].tiles += ph.ntiles[sh];
      }
    }
  }
  if (plan->print_stats)
    for (int p = 0; p < 2; ++p)
      for (int sh = 0; sh < GEMM_NSHAPES; ++sh)
        if (ps[p][sh].tiles)
          fprintf(stderr, "plan phase %d shape %dx%d tiles %lld flops %.4g full-tile flops %.4g (fill %.3f)\n", p + 1,
                  GEMM_DIMS[sh / 3], GEMM_DIMS[sh % 3], ps[p][sh].tiles, ps[p][sh].act, ps[p][sh].full,
                  ps[p][sh].act / ps[p][sh].full);
  pt.lap("chunk uploads");
  chunks_.clear();
  pt.lap("free host items");
}

}  // namespace dmrg
