#include "plan.h"

#include <algorithm>
#include <numeric>

namespace dmrg {

int Plan::launches() const {
  int n = 0;
  for (const auto& c : chunks) n += (c.p1.ntiles > 0) + (c.p2.ntiles > 0);
  return n;
}

void Plan::run(cudaStream_t st, int64_t* launch_counter) const {
  for (const auto& c : chunks) {
    if (c.p1.ntiles > 0) {
      DMRG_CUDA(launch_grouped_gemm(c.p1.outs.p, c.p1.segs.p, c.p1.tiles.p, c.p1.ntiles, st));
      if (launch_counter) ++*launch_counter;
    }
    if (c.p2.ntiles > 0) {
      DMRG_CUDA(launch_grouped_gemm(c.p2.outs.p, c.p2.segs.p, c.p2.tiles.p, c.p2.ntiles, st));
      if (launch_counter) ++*launch_counter;
    }
  }
}

static inline double fl(double a, double b, double c) { return 2.0 * a * b * c; }

void Planner::add(const Item& it) {
  DMRG_REQUIRE(it.count >= 1, DMRG_ERR_ARG, "planner: empty item");
  ++n_items_;
  n_products_ += it.count;
  if (it.nmat == 2) {
    fa_ += it.count * fl(it.X.urows, it.X.ucols, it.Y.ucols);
    add_piece(it, 0, it.count);
    return;
  }
  // analytic flops: the cheaper order on the true (unpadded) dims
  double left = fl(it.X.urows, it.X.ucols, it.Y.ucols) + fl(it.X.urows, it.Y.ucols, it.W.ucols);
  double right = fl(it.Y.urows, it.Y.ucols, it.W.ucols) + fl(it.X.urows, it.X.ucols, it.W.ucols);
  fa_ += it.count * std::min(left, right);
  // workspace per product, in the order the kernels will use (padded dims)
  double pl = fl(it.X.rows, it.X.cols, it.Y.cols) + fl(it.X.rows, it.Y.cols, it.W.cols);
  double pr = fl(it.Y.rows, it.Y.cols, it.W.cols) + fl(it.X.rows, it.X.cols, it.W.cols);
  long long zsz = (pl <= pr) ? (long long)it.X.rows * it.Y.cols : (long long)it.Y.rows * it.W.cols;
  DMRG_REQUIRE(zsz <= cap_, DMRG_ERR_ALLOC, "planner: workspace cap smaller than one intermediate block");
  int per = (int)std::min<long long>(it.count, cap_ / zsz);
  for (int b0 = 0; b0 < it.count; b0 += per) add_piece(it, b0, std::min(per, it.count - b0));
}

Planner::HOut& Planner::p2_out(HChunk& ch, const Item& it, int b0, int cnt, int M, int N) {
  const bool batched = it.strideC != 0;
  double* C = it.C + (batched ? b0 * it.strideC : 0);
  auto key = std::make_tuple((const double*)C, batched ? cnt : 1, it.strideC);
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
  auto mkseg = [](const double* A, int lda, bool ta, const double* B, int ldb, bool tb, int K) {
    HSeg h{};
    h.s.A = A; h.s.B = B; h.s.lda = lda; h.s.ldb = ldb; h.s.K = K; h.s.count = 1;
    h.s.flags = (ta ? 1 : 0) | (tb ? 2 : 0); h.s.alpha = 1.0;
    h.s.rsA = h.s.rsB = h.s.bsA = h.s.bsB = 0; h.a_ws = h.b_ws = false;
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
  if (chunks_.back().ws_used + zsz * cnt > cap_) chunks_.emplace_back();
  HChunk& ch = chunks_.back();
  const long long zoff = ch.ws_used;
  ch.ws_used += zsz * cnt;
  ws_max_ = std::max(ws_max_, ch.ws_used);
  bi_ += 2.0 * 8.0 * zsz * cnt;
  fe_ += cnt * std::min(pl, pr);
  // phase 1: Z[b] = X[b] Y[b]  or  Y[b] W[b]
  {
    HOut z{};
    z.o.C = reinterpret_cast<double*>(zoff); z.c_ws = true;
    z.o.bsC = zsz; z.o.M = zr; z.o.N = zc; z.o.ldc = zc; z.o.accumulate = 0;
    z.batch = cnt; z.work = 0;
    const Mat& A = left_first ? it.X : it.Y;
    const Mat& B = left_first ? it.Y : it.W;
    HSeg h = mkseg(A.p + b0 * A.stride, A.ld, A.tr, B.p + b0 * B.stride, B.ld, B.tr, A.cols);
    h.s.bsA = A.stride; h.s.bsB = B.stride;
    z.segs.push_back(h);
    ch.p1.push_back(std::move(z));
  }
  // phase 2: C += alpha Z[b] W[b]  or  alpha X[b] Z[b]
  HOut& o = p2_out(ch, it, b0, cnt, it.X.rows, it.W.cols);
  HSeg h;
  if (left_first) {
    h = mkseg(reinterpret_cast<const double*>(zoff), zc, false, it.W.p + b0 * it.W.stride, it.W.ld,
              it.W.tr, zc);
    h.a_ws = true;
    if (batched) { h.s.bsA = zsz; h.s.bsB = it.W.stride; }
    else { h.s.count = cnt; h.s.rsA = zsz; h.s.rsB = it.W.stride; }
  } else {
    h = mkseg(it.X.p + b0 * it.X.stride, it.X.ld, it.X.tr, reinterpret_cast<const double*>(zoff), zc,
              false, zr);
    h.b_ws = true;
    if (batched) { h.s.bsA = it.X.stride; h.s.bsB = zsz; }
    else { h.s.count = cnt; h.s.rsA = it.X.stride; h.s.rsB = zsz; }
  }
  h.s.alpha = it.alpha;
  o.segs.push_back(h);
}

void Planner::finish(Plan* plan, cudaStream_t st) {
  plan->clear();
  plan->flops_analytic = fa_;
  plan->flops_executed = fe_;
  plan->bytes_intermediate = bi_;
  plan->n_items = n_items_;
  plan->n_products = n_products_;
  if (ws_max_ > 0) plan->workspace.allocate(al_, (size_t)ws_max_);
  double* ws = plan->workspace.p;
  auto build = [&](std::vector<HOut>& hv, Phase& ph) {
    std::vector<GOut> outs;
    std::vector<GSeg> segs;
    struct TW { GTile t; double w; };
    std::vector<TW> tw;
    outs.reserve(hv.size());
    for (size_t oi = 0; oi < hv.size(); ++oi) {
      HOut& h = hv[oi];
      GOut o = h.o;
      if (h.c_ws) o.C = ws + reinterpret_cast<long long>(h.o.C);
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
      int tm = (o.M + GEMM_BM - 1) / GEMM_BM, tn = (o.N + GEMM_BN - 1) / GEMM_BN;
      o.tile_m = pad8((o.M + tm - 1) / tm);
      o.tile_n = pad8((o.N + tn - 1) / tn);
      tm = (o.M + o.tile_m - 1) / o.tile_m;
      tn = (o.N + o.tile_n - 1) / o.tile_n;
      outs.push_back(o);
      for (int b = 0; b < h.batch; ++b)
        for (int i = 0; i < tm; ++i)
          for (int j = 0; j < tn; ++j) {
            int em = std::min(o.tile_m, o.M - i * o.tile_m), en = std::min(o.tile_n, o.N - j * o.tile_n);
            double w = ksum * ((em + 15) / 16) * ((en + 31) / 32);
            tw.push_back({GTile{(int)oi, b, i, j}, w});
          }
    }
    std::stable_sort(tw.begin(), tw.end(), [](const TW& a, const TW& b) { return a.w > b.w; });
    std::vector<GTile> tiles(tw.size());
    for (size_t i = 0; i < tw.size(); ++i) tiles[i] = tw[i].t;
    ph.ntiles = (int)tiles.size();
    ph.outs.upload(al_, outs, st);
    ph.segs.upload(al_, segs, st);
    ph.tiles.upload(al_, tiles, st);
  };
  plan->chunks.resize(chunks_.size());
  for (size_t c = 0; c < chunks_.size(); ++c) {
    build(chunks_[c].p1, plan->chunks[c].p1);
    build(chunks_[c].p2, plan->chunks[c].p2);
  }
  chunks_.clear();
}

}  // namespace dmrg
