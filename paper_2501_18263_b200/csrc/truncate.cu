// The truncation step of a two-site micro-iteration behind the C ABI ("keeping only the D largest singular
// values in SVD"; Fig. 1, :63): SVD of the optimised wavefunction per sector of bond k, selection of the D largest
// singular values over all sectors, the new canonical site tensor written straight into the library's MPS store, and
// the wave-function transformation that gives the next bond's start vector.  U(1)xU(1) contexts.  Sector matrices
// that fit the shared memory of one CTA (~165 x 165: the regime of the paper's mode optimisation, D <= 256) are
// decomposed there; larger ones are rotated in place in global memory (correct at any size, slow).
//
//   dmrg_truncate_bond   k_sector_svd (one CTA per bond sector, one-sided Jacobi with the rotations accumulated),
//                        selection on the host (one small D2H of the singular values), k_write_isometry
//   dmrg_start_vector    k_start_vector: psi_next{block} = (Sigma V^T)[kept, columns] . R-site   (sweep to the right)
//                                                         = L-site . (U Sigma)[rows, kept]       (sweep to the left)
//   dmrg_bond_sectors    the sectors of a bond as the library holds them (host query)
//
// One-sided Jacobi on the shorter side of Psi_q: with its ROWS as the vectors (rotations G from the left: R <- G R,
// Psi' = R Psi has orthogonal rows = Sigma V^T, U = R^T), with its COLUMNS (Psi' = Psi R^T = U Sigma, V^T = R).  When the
// vectors lie on the side of the isometry the new site tensor needs, that isometry is the accumulated R, orthogonal to
// rounding whatever the singular values are, and the rotated vectors are the centre factor; otherwise the isometry is
// the normalised rotated vectors (orthonormal to the convergence threshold 1e-14) and the centre factor is Sigma R.
#include <algorithm>
#include <cmath>
#include <map>

#include "engine.h"

using namespace dmrg;

namespace {

constexpr size_t SMEM_CAP = 220 * 1024;                         // dynamic shared memory one CTA may ask for

struct TrPlace { long long off; int dL, dR, row0, col0; };     // one psi block inside Psi_q[(a s1), (s2 b)]
struct TrSector {
  int place_begin, place_end;
  int n, m;                 // n vectors of length m
  int by_cols, pad_;        // the vectors are the columns of Psi_q (else its rows)
  int sig_off, in_smem;     // first singular value / permutation entry of this sector; in shared memory: 2 = vectors
                            // and R, 1 = vectors only, 0 = nothing (both rotated in place in global memory)
  long long r_off, v_off;   // R (n x n) and the rotated vectors (n x m) in the work arrays
};

// Singular values (sorted descending, with the permutation that sorts them), accumulated rotations R and rotated
// vectors of one sector.  Round-robin pairing, one warp per pair, fixed order: deterministic.
constexpr int SVD_THREADS = 1024;                                // 32 warps: one pair of vectors per warp and round

__global__ void __launch_bounds__(SVD_THREADS) k_sector_svd(const TrSector* __restrict__ secs, const TrPlace* __restrict__ places,
                                                    const double* __restrict__ psi,
                                                    double* __restrict__ sigma, int* __restrict__ perm,
                                                    double* __restrict__ Rall, double* __restrict__ Vall,
                                                    double* __restrict__ norms) {
  extern __shared__ double Vs[];                      // n vectors of length m (pitch m + 1) if the sector fits
  __shared__ int rotated;
  const TrSector sc = secs[blockIdx.x];
  const int n = sc.n, m = sc.m, pitch = sc.in_smem ? m + 1 : m;
  // a sector too large for shared memory is rotated in place in its output array (L2-resident: slower, any size)
  double* V = sc.in_smem ? Vs : Vall + sc.v_off;
  double* nrm = norms + sc.sig_off;
  const int rpitch = sc.in_smem == 2 ? n + 1 : n;
  double* R = sc.in_smem == 2 ? Vs + (size_t)n * pitch : Rall + sc.r_off;
  for (int i = threadIdx.x; i < n * pitch; i += blockDim.x) V[i] = 0.0;
  for (int i = threadIdx.x; i < n * n; i += blockDim.x) R[(i / n) * rpitch + i % n] = (i / n == i % n) ? 1.0 : 0.0;
  __syncthreads();
  for (int p = sc.place_begin; p < sc.place_end; ++p) {
    const TrPlace pl = places[p];
    for (int e = threadIdx.x; e < pl.dL * pl.dR; e += blockDim.x) {
      const int r = pl.row0 + e / pl.dR, c = pl.col0 + e % pl.dR;
      const double v = psi[pl.off + e];
      if (sc.by_cols) V[c * pitch + r] = v; else V[r * pitch + c] = v;
    }
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
  // One pair of vectors per group of EIGHT lanes: 128 pairs in flight per CTA, so a round of the tournament is a single
  // pass for n <= 256 and its cost is one latency chain (dots, reduction, rotation) rather than several in sequence.
  const int grp = threadIdx.x >> 3, l8 = threadIdx.x & 7, ngrp = blockDim.x >> 3;
  const unsigned gmask = 0xFFu << (threadIdx.x & 24);   // the lanes of this group inside its warp
  const int np = (n + 1) & ~1;                        // players of the round-robin tournament (one bye if n is odd)
  for (int sweep = 0; sweep < 60; ++sweep) {
    if (threadIdx.x == 0) rotated = 0;
    __syncthreads();
    for (int round = 0; round < np - 1; ++round) {
      for (int g = grp; g < np / 2; g += ngrp) {
        int a = g == 0 ? np - 1 : (round + g) % (np - 1);   // circle method: player np-1 is fixed, the others rotate
        int b = (round + np - 1 - g) % (np - 1);
        if (a > b) { const int t = a; a = b; b = t; }
        if (b >= n) continue;                         // bye
        double* va = V + a * pitch;
        double* vb = V + b * pitch;
        double al = 0.0, be = 0.0, ga = 0.0;
        for (int i = l8; i < m; i += 8) { const double x = va[i], y = vb[i]; al = fma(x, x, al); be = fma(y, y, be); ga = fma(x, y, ga); }
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
          al += __shfl_xor_sync(gmask, al, o, 8); be += __shfl_xor_sync(gmask, be, o, 8); ga += __shfl_xor_sync(gmask, ga, o, 8);
        }
        if (ga * ga > 1e-28 * (al * be)) {            // |cos(a, b)| > 1e-14
          // tan of the rotation angle: t = sign(tau) g / (|tau| + sqrt(tau^2 + g^2)), tau = |b|^2 - |a|^2, g = 2 a.b
          const double tau = be - al, g2 = 2.0 * ga;
          const double t = (tau >= 0.0 ? g2 : -g2) / (fabs(tau) + sqrt(fma(tau, tau, g2 * g2)));
          const double c = rsqrt(fma(t, t, 1.0)), s = c * t;
          for (int i = l8; i < m; i += 8) {
            const double x = va[i], y = vb[i];
            va[i] = c * x - s * y;
            vb[i] = s * x + c * y;
          }
          // rows a, b of R (in global memory for the larger sectors): all loads of a 64-wide slab are issued before
          // the first use, so that a slab costs one memory latency
          double* ra = R + (size_t)a * rpitch;
          double* rb = R + (size_t)b * rpitch;
          for (int base = 0; base < n; base += 64) {
            double xr[8], yr[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int i = base + l8 + 8 * u;
              if (i < n) { xr[u] = ra[i]; yr[u] = rb[i]; }
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
              const int i = base + l8 + 8 * u;
              if (i < n) { ra[i] = c * xr[u] - s * yr[u]; rb[i] = s * xr[u] + c * yr[u]; }
            }
          }
          if (l8 == 0) rotated = 1;
        }
      }
      __syncthreads();
    }
    const int any = rotated;
    __syncthreads();
    if (!any) break;
  }
  for (int v = warp; v < n; v += nwarps) {
    double s = 0.0;
    for (int i = lane; i < m; i += 32) { const double x = V[v * pitch + i]; s = fma(x, x, s); }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) nrm[v] = sqrt(s);
  }
  __syncthreads();
  // descending order; equal values keep their index order
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double si = nrm[i];
    int rank = 0;
    for (int j = 0; j < n; ++j) { const double sj = nrm[j]; rank += (sj > si) || (sj == si && j < i); }
    sigma[sc.sig_off + rank] = si;
    perm[sc.sig_off + rank] = i;
  }
  if (sc.in_smem) {
    double* Vo = Vall + sc.v_off;
    for (int i = threadIdx.x; i < n * m; i += blockDim.x) Vo[i] = V[(i / m) * pitch + i % m];
  }
  if (sc.in_smem == 2) {
    double* Ro = Rall + sc.r_off;
    for (int i = threadIdx.x; i < n * n; i += blockDim.x) Ro[i] = R[(i / n) * rpitch + i % n];
  }
}

// After the selection: per kept sector, the c kept isometry rows and centre rows in descending order of the singular
// values.  normal (the vectors were taken on the isometry side): isometry row j = R[perm[j], :], centre row j = rotated
// vector perm[j].  Otherwise (the vectors were taken on the centre side, the shorter one): isometry row j = rotated
// vector perm[j] / sigma_j (orthonormal to the convergence threshold of the Jacobi iteration), centre row j =
// sigma_j R[perm[j], :].
struct FinSec { long long r_off, v_off, iso_off, cen_off; int n, m, c, sig_off, normal, pad_; };

__global__ void k_finalize(const FinSec* __restrict__ secs, const double* __restrict__ Rall, const double* __restrict__ Vall,
                           const double* __restrict__ sigma, const int* __restrict__ perm, double* __restrict__ iso,
                           double* __restrict__ cen) {
  const FinSec f = secs[blockIdx.x];
  const double* R = Rall + f.r_off;
  const double* V = Vall + f.v_off;
  const int li = f.normal ? f.n : f.m, lc = f.normal ? f.m : f.n;
  for (int e = threadIdx.x; e < f.c * li; e += blockDim.x) {
    const int j = e / li, p = e % li, v = perm[f.sig_off + j];
    iso[f.iso_off + e] = f.normal ? R[(size_t)v * f.n + p] : V[(size_t)v * f.m + p] / sigma[f.sig_off + j];
  }
  for (int e = threadIdx.x; e < f.c * lc; e += blockDim.x) {
    const int j = e / lc, p = e % lc, v = perm[f.sig_off + j];
    cen[f.cen_off + e] = f.normal ? V[(size_t)v * f.m + p] : sigma[f.sig_off + j] * R[(size_t)v * f.n + p];
  }
}

// One block of the new site tensor from the isometry rows I (c x len) of its sector: dst[i, j] = I[j, base + i]
// (left-canonical: i = row of the old block, j = kept state) or I[i, base + j] (right-canonical).
struct IsoBlk { long long dst_off, src_off; int din, dout, doutp, len, base, right; };

__global__ void k_write_isometry(const IsoBlk* __restrict__ blks, const double* __restrict__ iso, double* __restrict__ dst) {
  const IsoBlk b = blks[blockIdx.x];
  const double* I = iso + b.src_off;
  for (int e = threadIdx.x; e < b.din * b.dout; e += blockDim.x) {
    const int i = e / b.dout, j = e % b.dout;
    dst[b.dst_off + (long long)i * b.doutp + j] = b.right ? I[(size_t)i * b.len + b.base + j] : I[(size_t)j * b.len + b.base + i];
  }
}

// One block of the next start vector from the centre rows C (c x len) of its sector and a site block S.
// right == 0 (sweep to the right): out[i, j] = sum_t C[i, base + t] S[t, j];  right == 1: out[i, j] = sum_t S[i, t] C[j, base + t].
struct StBlk { long long out_off, c_off, s_off; int dL, dR, len, base, w, lds, right, pad_; };

__global__ void k_start_vector(const StBlk* __restrict__ blks, const double* __restrict__ cen, const double* __restrict__ site,
                               double* __restrict__ out) {
  const StBlk b = blks[blockIdx.x];
  const double* C = cen + b.c_off;
  const double* S = site + b.s_off;
  for (int e = threadIdx.x + blockIdx.y * blockDim.x; e < b.dL * b.dR; e += blockDim.x * gridDim.y) {
    const int i = e / b.dR, j = e % b.dR;
    double s = 0.0;
    if (!b.right) {
      const double* c = C + (size_t)i * b.len + b.base;
      for (int t = 0; t < b.w; ++t) s = fma(c[t], S[(size_t)t * b.lds + j], s);
    } else {
      const double* c = C + (size_t)j * b.len + b.base;
      for (int t = 0; t < b.w; ++t) s = fma(S[(size_t)i * b.lds + t], c[t], s);
    }
    out[b.out_off + e] = s;
  }
}

#define TR_BEGIN                                   \
  if (!ctx) return DMRG_ERR_ARG;                   \
  try {                                            \
    DMRG_CUDA(cudaSetDevice(ctx->cfg.device));
#define TR_END                                     \
    return DMRG_OK;                                \
  } catch (const dmrg::Error& e) {                 \
    ctx->err = e.what();                           \
    return e.code;                                 \
  } catch (const std::exception& e) {              \
    ctx->err = e.what();                           \
    return DMRG_ERR_ARG;                           \
  }

}  // namespace

extern "C" {

int dmrg_truncate_bond(dmrg_ctx* ctx, const double* d_psi, int32_t direction, int32_t D, double* h_discarded,
                       int32_t* h_kept, void* stream) {
  TR_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && ctx->left && ctx->right && d_psi, DMRG_ERR_ARG, "truncate_bond: no problem prepared or null pointer");
  DMRG_REQUIRE((direction == 0 || direction == 1) && D >= 1, DMRG_ERR_ARG, "truncate_bond: direction is 0 or 1, D >= 1");
  DMRG_REQUIRE(!ctx->su2(), DMRG_ERR_UNSUPPORTED, "truncate_bond: U(1)xU(1) contexts only");
  const int k = ctx->k;
  const Sectors& SL = ctx->left->sec;      // index = sector index of bond k-1
  const Sectors& SR = ctx->right->sec;     // index = sector index of bond k+1
  const Sectors& bl = ctx->bond[k - 1];
  const Sectors& br = ctx->bond[k + 1];
  DMRG_REQUIRE(SL.size() == bl.size() && SR.size() == br.size(), DMRG_ERR_ARG, "truncate_bond: blocks and bonds disagree");
  // ---- sectors of bond k: q = q_L + q(s1); rows (q_L, s1), columns (s2, q_R); lexicographic in q ----
  struct Tmp {
    std::map<std::pair<int, int>, std::pair<int, int>> row, col;     // group -> (first position, width)
    int rows = 0, cols = 0;
    std::vector<TrPlace> pl;
  };
  std::map<std::pair<int, int>, Tmp> by_q;
  for (auto& b : ctx->psi) {
    Tmp& t = by_q[{SL.qu[b.qL] + SITE_QU[b.s1], SL.qd[b.qL] + SITE_QD[b.s1]}];
    auto r = t.row.find({b.qL, b.s1});
    if (r == t.row.end()) { r = t.row.emplace(std::make_pair(b.qL, b.s1), std::make_pair(t.rows, b.dL)).first; t.rows += b.dL; }
    auto c = t.col.find({b.s2, b.qR});
    if (c == t.col.end()) { c = t.col.emplace(std::make_pair(b.s2, b.qR), std::make_pair(t.cols, b.dR)).first; t.cols += b.dR; }
    t.pl.push_back(TrPlace{b.off_c, b.dL, b.dR, r->second.first, c->second.first});
  }
  std::vector<TrSector> secs;
  std::vector<TrPlace> places;
  std::vector<std::pair<int, int>> labels;
  long long nsig = 0, r_elems = 0, v_elems = 0;
  size_t smem_max = 0;
  for (auto& kv : by_q) {
    Tmp& t = kv.second;
    // the vectors are taken on the shorter side (fewer of them, and no rank-deficient set); on a tie on the side of
    // the isometry: rows when the sweep moves right, columns when it moves left
    const bool by_cols = direction == 0 ? t.cols < t.rows : t.cols <= t.rows;
    const int n = by_cols ? t.cols : t.rows, m = by_cols ? t.rows : t.cols;
    TrSector s{(int)places.size(), 0, n, m, by_cols ? 1 : 0, 0, (int)nsig, 0, r_elems, v_elems};
    places.insert(places.end(), t.pl.begin(), t.pl.end());
    s.place_end = (int)places.size();
    const size_t need1 = (size_t)n * (m + 1) * 8, need2 = need1 + (size_t)n * (n + 1) * 8;
    s.in_smem = need2 <= SMEM_CAP ? 2 : (need1 <= SMEM_CAP ? 1 : 0);
    if (s.in_smem) smem_max = std::max(smem_max, s.in_smem == 2 ? need2 : need1);
    nsig += n; r_elems += (long long)n * n; v_elems += (long long)n * m;
    secs.push_back(s);
    labels.push_back(kv.first);
  }
  DMRG_REQUIRE(!secs.empty(), DMRG_ERR_ARG, "truncate_bond: the two-site problem has no blocks");
  DevArray<TrSector> d_secs;
  DevArray<TrPlace> d_places;
  DevArray<double> d_sigma, d_R, d_V, d_norms;
  DevArray<int> d_perm;
  d_secs.upload(&ctx->al, secs, st);
  d_places.upload(&ctx->al, places, st);
  d_sigma.allocate(&ctx->al, (size_t)nsig);
  d_perm.allocate(&ctx->al, (size_t)nsig);
  d_R.allocate(&ctx->al, (size_t)r_elems);
  d_V.allocate(&ctx->al, (size_t)v_elems);
  d_norms.allocate(&ctx->al, (size_t)nsig);
  DMRG_CUDA(cudaFuncSetAttribute(k_sector_svd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
  k_sector_svd<<<(unsigned)secs.size(), SVD_THREADS, smem_max, st>>>(d_secs.p, d_places.p, d_psi, d_sigma.p, d_perm.p, d_R.p, d_V.p, d_norms.p);
  ++ctx->launches;
  DMRG_CUDA(cudaGetLastError());
  std::vector<double> sig((size_t)nsig);
  DMRG_CUDA(cudaMemcpyAsync(sig.data(), d_sigma.p, sizeof(double) * nsig, cudaMemcpyDeviceToHost, st));
  DMRG_CUDA(cudaStreamSynchronize(st));
  // ---- the D largest over all sectors (R23: equal values in lexicographic sector order; <= 1e-14 never) ----
  struct SV { double s; int sec; };
  std::vector<SV> all;
  all.reserve((size_t)nsig);
  for (size_t si = 0; si < secs.size(); ++si)
    for (int i = 0; i < secs[si].n; ++i) all.push_back(SV{sig[secs[si].sig_off + i], (int)si});
  std::stable_sort(all.begin(), all.end(), [](const SV& a, const SV& b) { return a.s > b.s; });
  std::vector<int> kept(secs.size(), 0);
  int nkept = 0;
  for (size_t i = 0; i < all.size() && i < (size_t)D; ++i)
    if (all[i].s > 1e-14) { ++kept[all[i].sec]; ++nkept; }
  double weight = 0.0;
  for (size_t i = (size_t)D; i < all.size(); ++i) weight += all[i].s * all[i].s;
  DMRG_REQUIRE(nkept > 0, DMRG_ERR_INPUT, "truncate_bond: the wavefunction is zero");
  if (h_discarded) *h_discarded = weight;
  if (h_kept) *h_kept = nkept;
  // ---- kept isometry and centre rows of every kept sector, in descending order of the singular values ----
  Sectors nb;
  std::vector<int> new_index(secs.size(), -1);
  std::vector<FinSec> fin;
  std::vector<long long> iso_off(secs.size(), 0), cen_off(secs.size(), 0);
  long long iso_elems = 0, cen_elems = 0;
  {
    size_t si = 0;
    for (auto& kv : by_q) {
      const Tmp& tm = kv.second;
      if (kept[si] > 0) {
        new_index[si] = nb.size();
        nb.add(labels[si].first, labels[si].second, kept[si]);
        const bool normal = (secs[si].by_cols != 0) == (direction == 1);
        iso_off[si] = iso_elems; cen_off[si] = cen_elems;
        fin.push_back(FinSec{secs[si].r_off, secs[si].v_off, iso_elems, cen_elems, secs[si].n, secs[si].m, kept[si],
                             secs[si].sig_off, normal ? 1 : 0, 0});
        iso_elems += (long long)kept[si] * (direction == 0 ? tm.rows : tm.cols);
        cen_elems += (long long)kept[si] * (direction == 0 ? tm.cols : tm.rows);
      }
      ++si;
    }
  }
  DevArray<FinSec> d_fin;
  DevArray<double> d_iso, d_cen;
  d_fin.upload(&ctx->al, fin, st);
  d_iso.allocate(&ctx->al, (size_t)iso_elems);
  d_cen.allocate(&ctx->al, (size_t)cen_elems);
  k_finalize<<<(unsigned)fin.size(), 256, 0, st>>>(d_fin.p, d_R.p, d_V.p, d_sigma.p, d_perm.p, d_iso.p, d_cen.p);
  ++ctx->launches;
  DMRG_CUDA(cudaGetLastError());
  // ---- the new canonical site tensor, written on the device ----
  const int site = direction == 0 ? k : k + 1;
  SiteTensor t;
  t.canonical = direction;
  std::vector<IsoBlk> iso;
  long long off = 0;
  {
    size_t si = 0;
    for (auto& kv : by_q) {
      const Tmp& tm = kv.second;
      const int c = kept[si];
      if (c > 0) {
        if (direction == 0) {
          for (auto& g : tm.row) {        // (q_L, s1) -> rows [first, first + d_L)
            SiteBlk b{g.first.first, g.first.second, new_index[si], g.second.second, c, pad8(g.second.second), pad8(c), off};
            iso.push_back(IsoBlk{off, iso_off[si], b.din, b.dout, b.doutp, tm.rows, g.second.first, 0});
            off += (long long)b.dinp * b.doutp;
            t.find.emplace(std::make_pair(b.qin, b.s), (int)t.blks.size());
            t.blks.push_back(b);
          }
        } else {
          for (auto& g : tm.col) {        // (s2, q_R) -> columns [first, first + d_R)
            SiteBlk b{new_index[si], g.first.first, g.first.second, c, g.second.second, pad8(c), pad8(g.second.second), off};
            iso.push_back(IsoBlk{off, iso_off[si], b.din, b.dout, b.doutp, tm.cols, g.second.first, 1});
            off += (long long)b.dinp * b.doutp;
            t.find.emplace(std::make_pair(b.qin, b.s), (int)t.blks.size());
            t.blks.push_back(b);
          }
        }
      }
      ++si;
    }
  }
  t.data.allocate(&ctx->al, (size_t)std::max<long long>(off, 8));
  DMRG_CUDA(cudaMemsetAsync(t.data.p, 0, (size_t)std::max<long long>(off, 8) * 8, st));
  DevArray<IsoBlk> d_isoblk;
  d_isoblk.upload(&ctx->al, iso, st);
  k_write_isometry<<<(unsigned)iso.size(), 128, 0, st>>>(d_isoblk.p, d_iso.p, t.data.p);
  ++ctx->launches;
  DMRG_CUDA(cudaGetLastError());
  // ---- the centre factor for dmrg_start_vector ----
  CentreFactor& cf = ctx->centre;
  cf.clear();
  cf.bond = k; cf.direction = direction;
  {
    size_t si = 0;
    for (auto& kv : by_q) {
      if (kept[si] > 0) {
        CentreFactor::Sec s;
        s.c = kept[si]; s.len = direction == 0 ? kv.second.cols : kv.second.rows; s.off = cen_off[si];
        s.groups = direction == 0 ? kv.second.col : kv.second.row;
        cf.sec.emplace(kv.first, std::move(s));
      }
      ++si;
    }
  }
  cf.C = std::move(d_cen);
  DMRG_CUDA(cudaStreamSynchronize(st));      // the descriptor arrays and R die with this call
  // ---- install: bond k, then the site tensor (what dmrg_mps_update_bond + dmrg_mps_set_site do from host data) ----
  ctx->bond[k] = std::move(nb);
  for (int i : {k, k + 1}) {
    SiteTensor& o = ctx->site[i];
    o.canonical = -1; o.blks.clear(); o.find.clear(); o.find3.clear(); o.data.release();
  }
  ctx->invalidate_site(k);
  ctx->invalidate_site(k + 1);
  ctx->site[site] = std::move(t);
  TR_END
}

int dmrg_bond_sectors(dmrg_ctx* ctx, int32_t b, int32_t* nsec, int32_t* h_q_up, int32_t* h_q_dn, int32_t* h_dim) {
  TR_BEGIN
  DMRG_REQUIRE(!ctx->bond.empty() && b >= 0 && b <= ctx->L && nsec, DMRG_ERR_ARG, "bond_sectors: sectors first, 0 <= b <= L");
  const Sectors& s = ctx->bond[b];
  *nsec = s.size();
  for (int i = 0; i < s.size(); ++i) {
    if (h_q_up) h_q_up[i] = s.qu[i];
    if (h_q_dn) h_q_dn[i] = s.qd[i];
    if (h_dim) h_dim[i] = s.dim[i];
  }
  TR_END
}

int dmrg_start_vector(dmrg_ctx* ctx, double* d_out, void* stream) {
  TR_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  const CentreFactor& cf = ctx->centre;
  DMRG_REQUIRE(ctx->k > 0 && d_out, DMRG_ERR_ARG, "start_vector: no problem prepared or null pointer");
  DMRG_REQUIRE(cf.bond > 0 && ctx->k == cf.bond + (cf.direction == 0 ? 1 : -1), DMRG_ERR_ARG,
               "start_vector: needs dmrg_truncate_bond at the neighbouring bond followed by dmrg_renormalize in the same direction");
  const int kb = cf.bond;
  const Sectors& mid = ctx->bond[kb];
  const SiteTensor& S = ctx->site[cf.direction == 0 ? kb + 2 : kb - 1];
  DMRG_REQUIRE(S.canonical == (cf.direction == 0 ? 1 : 0) && S.data.p, DMRG_ERR_ARG, "start_vector: the neighbouring site tensor is not set");
  std::vector<StBlk> blks;
  for (auto& b : ctx->psi) {
    StBlk sb{};
    if (cf.direction == 0) {
      // new block (q_mid, s_{k+1}, s_{k+2}, q_R'): C_q[:, columns (s_{k+1}, q_{k+1})] . R-site[(q_{k+1}, s_{k+2}) -> q_R']
      auto f = cf.sec.find({mid.qu[b.qL], mid.qd[b.qL]});
      if (f == cf.sec.end()) continue;
      const int q1 = ctx->bond[kb + 1].find(mid.qu[b.qL] + SITE_QU[b.s1], mid.qd[b.qL] + SITE_QD[b.s1]);
      if (q1 < 0) continue;
      auto g = f->second.groups.find({b.s1, q1});
      auto sf = S.find.find({q1, b.s2});
      if (g == f->second.groups.end() || sf == S.find.end()) continue;
      const SiteBlk& w = S.blks[sf->second];
      DMRG_REQUIRE(w.qout == b.qR && w.din == g->second.second && w.dout == b.dR && f->second.c == b.dL, DMRG_ERR_ARG,
                   "start_vector: the centre factor does not match the prepared problem");
      sb = StBlk{b.off_c, f->second.off, w.off, b.dL, b.dR, f->second.len, g->second.first, w.din, w.doutp, 0, 0};
    } else {
      // new block (q_L', s_{k-1}, s_k, q_mid): L-site[(q_L', s_{k-1}) -> q_{k-1}] . (U Sigma)_q[rows (q_{k-1}, s_k), :]
      auto f = cf.sec.find({mid.qu[b.qR], mid.qd[b.qR]});
      if (f == cf.sec.end()) continue;
      const int q1 = ctx->bond[kb - 1].find(mid.qu[b.qR] - SITE_QU[b.s2], mid.qd[b.qR] - SITE_QD[b.s2]);
      if (q1 < 0) continue;
      auto g = f->second.groups.find({q1, b.s2});
      auto sf = S.find.find({b.qL, b.s1});
      if (g == f->second.groups.end() || sf == S.find.end()) continue;
      const SiteBlk& w = S.blks[sf->second];
      if (w.qout != q1) continue;
      DMRG_REQUIRE(w.dout == g->second.second && w.din == b.dL && f->second.c == b.dR, DMRG_ERR_ARG,
                   "start_vector: the centre factor does not match the prepared problem");
      sb = StBlk{b.off_c, f->second.off, w.off, b.dL, b.dR, f->second.len, g->second.first, w.dout, w.doutp, 1, 0};
    }
    blks.push_back(sb);
  }
  DMRG_CUDA(cudaMemsetAsync(d_out, 0, (size_t)ctx->psi_n * 8, st));
  if (!blks.empty()) {
    DevArray<StBlk> d_blks;
    d_blks.upload(&ctx->al, blks, st);
    k_start_vector<<<dim3((unsigned)blks.size(), 4), 128, 0, st>>>(d_blks.p, cf.C.p, S.data.p, d_out);
    ++ctx->launches;
    DMRG_CUDA(cudaGetLastError());
    DMRG_CUDA(cudaStreamSynchronize(st));    // the descriptor array dies with this call
  }
  TR_END
}

}  // extern "C"
