// Mode-optimisation micro-iteration, steps ii) and iii) of PAPER.md Fig. 1 (:63): two-site gates on the optimised
// wavefunction, the block entropy of the cut between the two sites (an SVD per bond sector "in every cycle",
// PAPER.md:63), and the rotation of the integrals t, v.  U(1)xU(1) contexts.
//
//   dmrg_two_site_gate   psi'{a, s1' s2', b} = sum G[(s1' s2'), (s1 s2)] psi{a, s1 s2, b}     HBM-bound block combination
//   dmrg_bond_entropy    singular values of Psi[(a s1), (s2 b)] per sector of bond k by one-sided Jacobi in shared
//                        memory (one CTA per sector), S_1/2 = 2 ln sum sigma_i and S_1 from them on the device
//   dmrg_rotate_integrals  T, w -> rotated by the 2x2 block on orbitals (k, k+1); host data of the context
//   dmrg_bond_entropy_static  dmrg_bond_entropy with its device scratch in a file-scope array: allocates nothing
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <mutex>

#include "engine.h"

using namespace dmrg;

namespace {

struct GateTerm { long long off_in; double c; };
struct GateOut { long long off_out; long long n; int term_begin, term_end; };

__global__ void k_two_site_gate(const GateOut* __restrict__ outs, const GateTerm* __restrict__ terms,
                                const double* __restrict__ in, double* __restrict__ out) {
  const GateOut o = outs[blockIdx.x];
  for (long long e = threadIdx.x + (long long)blockIdx.y * blockDim.x; e < o.n; e += (long long)blockDim.x * gridDim.y) {
    double s = 0.0;
    for (int t = o.term_begin; t < o.term_end; ++t) s = fma(terms[t].c, in[terms[t].off_in + e], s);   // fixed order
    out[o.off_out + e] = s;
  }
}

// One psi block inside the matrix Psi_q[(a s1), (s2 b)] of a bond sector q.
struct SvPlace { long long off; int dL, dR, row0, col0; };
struct SvSector { int place_begin, place_end, rows, cols, sig_off, pad_; };

// sigma of one sector by one-sided (Hestenes) Jacobi: the n = min(rows, cols) shorter-side vectors of length
// m = max(rows, cols) are rotated pairwise until mutually orthogonal; their norms are the singular values.
// Round-robin pairing, one warp per pair, fixed order: deterministic.
__global__ void __launch_bounds__(256) k_sector_svals(const SvSector* __restrict__ secs, const SvPlace* __restrict__ places,
                                                      const double* __restrict__ psi, double* __restrict__ sigma) {
  extern __shared__ double V[];                       // n vectors of length m (pitch m + 1)
  __shared__ int rotated;
  const SvSector sc = secs[blockIdx.x];
  const bool tr = sc.cols < sc.rows;                  // vectors = columns of Psi_q if there are fewer columns
  const int n = tr ? sc.cols : sc.rows, m = tr ? sc.rows : sc.cols, pitch = m + 1;
  for (int i = threadIdx.x; i < n * pitch; i += blockDim.x) V[i] = 0.0;
  __syncthreads();
  for (int p = sc.place_begin; p < sc.place_end; ++p) {
    const SvPlace pl = places[p];
    for (int e = threadIdx.x; e < pl.dL * pl.dR; e += blockDim.x) {
      const int r = pl.row0 + e / pl.dR, c = pl.col0 + e % pl.dR;
      const double v = psi[pl.off + e];
      if (tr) V[c * pitch + r] = v; else V[r * pitch + c] = v;
    }
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = blockDim.x >> 5;
  const int np = (n + 1) & ~1;                        // players of the round-robin tournament (one bye if n is odd)
  for (int sweep = 0; sweep < 60; ++sweep) {
    if (threadIdx.x == 0) rotated = 0;
    __syncthreads();
    for (int round = 0; round < np - 1; ++round) {
      for (int g = warp; g < np / 2; g += nwarps) {
        // circle method: player np-1 is fixed, the others rotate
        int a = g == 0 ? np - 1 : (round + g) % (np - 1);
        int b = (round + np - 1 - g) % (np - 1);
        if (a > b) { const int t = a; a = b; b = t; }
        if (b >= n) continue;                         // bye
        double* va = V + a * pitch;
        double* vb = V + b * pitch;
        double al = 0.0, be = 0.0, ga = 0.0;
        for (int i = lane; i < m; i += 32) { const double x = va[i], y = vb[i]; al = fma(x, x, al); be = fma(y, y, be); ga = fma(x, y, ga); }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          al += __shfl_xor_sync(0xffffffffu, al, o); be += __shfl_xor_sync(0xffffffffu, be, o); ga += __shfl_xor_sync(0xffffffffu, ga, o);
        }
        if (fabs(ga) > 1e-14 * sqrt(al * be) && ga != 0.0) {
          const double zeta = (be - al) / (2.0 * ga);
          const double t = (zeta >= 0.0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
          const double c = 1.0 / sqrt(1.0 + t * t), s = c * t;
          for (int i = lane; i < m; i += 32) {
            const double x = va[i], y = vb[i];
            va[i] = c * x - s * y;
            vb[i] = s * x + c * y;
          }
          if (lane == 0) rotated = 1;
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
    if (lane == 0) sigma[sc.sig_off + v] = sqrt(s);
  }
}

// S_1/2 = 2 ln(sum sigma / sqrt(sum sigma^2)) and S_1 = -sum p ln p, p = sigma^2 / sum sigma^2; one block,
// fixed-order tree.
__global__ void k_entropies(const double* __restrict__ sigma, int n, double* __restrict__ out) {
  __shared__ double sh[3][256];
  double s1 = 0.0, s2 = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) { s1 += sigma[i]; s2 = fma(sigma[i], sigma[i], s2); }
  sh[0][threadIdx.x] = s1; sh[1][threadIdx.x] = s2;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) { sh[0][threadIdx.x] += sh[0][threadIdx.x + w]; sh[1][threadIdx.x] += sh[1][threadIdx.x + w]; }
    __syncthreads();
  }
  const double tot1 = sh[0][0], tot2 = sh[1][0];
  double vn = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double p = sigma[i] * sigma[i] / tot2;
    if (p > 0.0) vn -= p * log(p);
  }
  __syncthreads();
  sh[2][threadIdx.x] = vn;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) sh[2][threadIdx.x] += sh[2][threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = 2.0 * log(tot1 / sqrt(tot2)); out[1] = sh[2][0]; out[2] = tot2; }
}

#define MO_BEGIN                                   \
  if (!ctx) return DMRG_ERR_ARG;                   \
  try {                                            \
    DMRG_CUDA(cudaSetDevice(ctx->cfg.device));
#define MO_END                                     \
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

int dmrg_two_site_gate(dmrg_ctx* ctx, const double* h_G, const double* d_in, double* d_out, void* stream) {
  MO_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && h_G && d_in && d_out && d_in != d_out, DMRG_ERR_ARG, "two_site_gate: no problem prepared, null or aliased pointers");
  DMRG_REQUIRE(!ctx->su2(), DMRG_ERR_UNSUPPORTED, "two_site_gate: U(1)xU(1) contexts only");
  std::vector<GateOut> outs;
  std::vector<GateTerm> terms;
  for (int so = 0; so < 16; ++so)
    for (int si = 0; si < 16; ++si) {
      const int du = SITE_QU[so / 4] + SITE_QU[so % 4] - SITE_QU[si / 4] - SITE_QU[si % 4];
      const int dd = SITE_QD[so / 4] + SITE_QD[so % 4] - SITE_QD[si / 4] - SITE_QD[si % 4];
      if (du != 0 || dd != 0)
        DMRG_REQUIRE(std::fabs(h_G[so * 16 + si]) <= 1e-14, DMRG_ERR_INPUT, "two_site_gate: the gate does not conserve (n_up, n_dn) of the two sites");
    }
  for (size_t b = 0; b < ctx->psi.size(); ++b) {
    const PsiBlk& o = ctx->psi[b];
    GateOut go{o.off_c, (long long)o.dL * o.dR, (int)terms.size(), 0};
    for (int s1 = 0; s1 < 4; ++s1)
      for (int s2 = 0; s2 < 4; ++s2) {
        const double g = h_G[(o.s1 * 4 + o.s2) * 16 + s1 * 4 + s2];
        if (g == 0.0) continue;
        auto f = ctx->psi_find.find({o.qL, s1, s2});
        if (f == ctx->psi_find.end()) continue;        // (same q_R as the output block: exists whenever that one does)
        const PsiBlk& in = ctx->psi[f->second];
        if (in.qR != o.qR) continue;
        terms.push_back(GateTerm{in.off_c, g});
      }
    go.term_end = (int)terms.size();
    outs.push_back(go);
  }
  DevArray<GateOut> d_outs;
  DevArray<GateTerm> d_terms;
  d_outs.upload(&ctx->al, outs, st);
  if (terms.empty()) terms.push_back(GateTerm{0, 0.0});
  d_terms.upload(&ctx->al, terms, st);
  if (!outs.empty()) k_two_site_gate<<<dim3((unsigned)outs.size(), 4), 256, 0, st>>>(d_outs.p, d_terms.p, d_in, d_out);
  ++ctx->launches;
  DMRG_CUDA(cudaGetLastError());
  DMRG_CUDA(cudaStreamSynchronize(st));      // the descriptor arrays die with this call
  MO_END
}

int dmrg_rotation_gate(double theta, double* h_G) {
  if (!h_G) return DMRG_ERR_ARG;
  // kappa = sum_s (c+_{2,s} c_{1,s} - c+_{1,s} c_{2,s}) on the two-site occupation basis (index 4 s1 + s2), Jordan-Wigner:
  // c+_{1,s} = c+_s (x) 1, c+_{2,s} = P (x) c+_s with the site matrices of DESIGN.md "Conventions"
  double cre[2][16] = {}, par[16] = {}, one[16] = {};
  cre[0][2 * 4 + 0] = 1.0; cre[0][3 * 4 + 1] = 1.0;       // a+_up : 0 -> up, dn -> up+dn
  cre[1][1 * 4 + 0] = 1.0; cre[1][3 * 4 + 2] = -1.0;      // a+_dn : 0 -> dn, up -> -(up+dn)
  const double pd[4] = {1.0, -1.0, -1.0, 1.0};
  for (int i = 0; i < 4; ++i) { par[i * 4 + i] = pd[i]; one[i * 4 + i] = 1.0; }
  auto kron = [](const double* a, const double* b, double* o) {
    for (int r1 = 0; r1 < 4; ++r1) for (int c1 = 0; c1 < 4; ++c1) for (int r2 = 0; r2 < 4; ++r2) for (int c2 = 0; c2 < 4; ++c2)
      o[(r1 * 4 + r2) * 16 + c1 * 4 + c2] = a[r1 * 4 + c1] * b[r2 * 4 + c2];
  };
  double K[256] = {};
  for (int s = 0; s < 2; ++s) {
    double c1[256], c2[256];
    kron(cre[s], one, c1);
    kron(par, cre[s], c2);
    for (int r = 0; r < 16; ++r) for (int c = 0; c < 16; ++c) {
      double v = 0.0;
      for (int q = 0; q < 16; ++q) v += c2[r * 16 + q] * c1[c * 16 + q] - c1[r * 16 + q] * c2[c * 16 + q];   // c2 c1^T - c1 c2^T
      K[r * 16 + c] += v;
    }
  }
  // G = exp(-theta K): scaling and squaring of the Taylor series
  int sq = 0;
  double t = -theta;
  while (std::fabs(t) > 0.125) { t *= 0.5; ++sq; }
  double G[256] = {}, term[256] = {}, tmp[256];
  for (int i = 0; i < 16; ++i) G[i * 16 + i] = term[i * 16 + i] = 1.0;
  for (int n = 1; n <= 24; ++n) {
    for (int r = 0; r < 16; ++r) for (int c = 0; c < 16; ++c) {
      double v = 0.0;
      for (int q = 0; q < 16; ++q) v += term[r * 16 + q] * K[q * 16 + c];
      tmp[r * 16 + c] = v * t / n;
    }
    std::memcpy(term, tmp, sizeof(tmp));
    for (int i = 0; i < 256; ++i) G[i] += term[i];
  }
  for (int s = 0; s < sq; ++s) {
    for (int r = 0; r < 16; ++r) for (int c = 0; c < 16; ++c) {
      double v = 0.0;
      for (int q = 0; q < 16; ++q) v += G[r * 16 + q] * G[q * 16 + c];
      tmp[r * 16 + c] = v;
    }
    std::memcpy(G, tmp, sizeof(tmp));
  }
  std::memcpy(h_G, G, sizeof(G));
  return DMRG_OK;
}

int dmrg_bond_entropy(dmrg_ctx* ctx, const double* d_psi, double* h_S_half, double* h_S_vn, double* h_sigma,
                      int32_t* n_sigma, void* stream) {
  MO_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_psi, DMRG_ERR_ARG, "bond_entropy: no problem prepared or null pointer");
  DMRG_REQUIRE(!ctx->su2(), DMRG_ERR_UNSUPPORTED, "bond_entropy: U(1)xU(1) contexts only");
  const Sectors& SL = ctx->left->sec;
  const Sectors& SR = ctx->right->sec;
  // sectors of bond k: q = q_L + q(s1); rows (q_L, s1), columns (s2, q_R)
  struct Tmp { std::map<std::pair<int, int>, int> row0, col0; int rows = 0, cols = 0; std::vector<SvPlace> pl; };
  std::map<std::pair<int, int>, Tmp> by_q;
  for (auto& b : ctx->psi) {
    const std::pair<int, int> q{SL.qu[b.qL] + SITE_QU[b.s1], SL.qd[b.qL] + SITE_QD[b.s1]};
    Tmp& t = by_q[q];
    auto r = t.row0.find({b.qL, b.s1});
    if (r == t.row0.end()) { r = t.row0.emplace(std::make_pair(b.qL, b.s1), t.rows).first; t.rows += b.dL; }
    auto c = t.col0.find({b.s2, b.qR});
    if (c == t.col0.end()) { c = t.col0.emplace(std::make_pair(b.s2, b.qR), t.cols).first; t.cols += b.dR; }
    t.pl.push_back(SvPlace{b.off_c, b.dL, b.dR, r->second, c->second});
  }
  (void)SR;
  std::vector<SvSector> secs;
  std::vector<SvPlace> places;
  int nsig = 0;
  size_t smem_max = 0;
  for (auto& kv : by_q) {
    Tmp& t = kv.second;
    SvSector s{(int)places.size(), 0, t.rows, t.cols, nsig, 0};
    places.insert(places.end(), t.pl.begin(), t.pl.end());
    s.place_end = (int)places.size();
    const int n = std::min(t.rows, t.cols), m = std::max(t.rows, t.cols);
    smem_max = std::max(smem_max, (size_t)n * (m + 1) * 8);
    nsig += n;
    secs.push_back(s);
  }
  DMRG_REQUIRE(smem_max <= 220 * 1024, DMRG_ERR_UNSUPPORTED,
               "bond_entropy: a bond sector is larger than the shared-memory Jacobi kernel holds (mode optimisation runs at D <= 256)");
  if (n_sigma) *n_sigma = nsig;
  DevArray<SvSector> d_secs;
  DevArray<SvPlace> d_places;
  DevArray<double> d_sigma, d_out;
  d_secs.upload(&ctx->al, secs, st);
  d_places.upload(&ctx->al, places, st);
  d_sigma.allocate(&ctx->al, (size_t)std::max(nsig, 1));
  d_out.allocate(&ctx->al, 8);
  DMRG_CUDA(cudaFuncSetAttribute(k_sector_svals, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
  k_sector_svals<<<(unsigned)secs.size(), 256, smem_max, st>>>(d_secs.p, d_places.p, d_psi, d_sigma.p);
  k_entropies<<<1, 256, 0, st>>>(d_sigma.p, nsig, d_out.p);
  ctx->launches += 2;
  DMRG_CUDA(cudaGetLastError());
  double res[3];
  DMRG_CUDA(cudaMemcpyAsync(res, d_out.p, sizeof(res), cudaMemcpyDeviceToHost, st));
  if (h_sigma) DMRG_CUDA(cudaMemcpyAsync(h_sigma, d_sigma.p, sizeof(double) * nsig, cudaMemcpyDeviceToHost, st));
  DMRG_CUDA(cudaStreamSynchronize(st));
  if (h_S_half) *h_S_half = res[0];
  if (h_S_vn) *h_S_vn = res[1];
  MO_END
}

int dmrg_rotate_integrals(dmrg_ctx* ctx, int32_t k, double theta) {
  MO_BEGIN
  DMRG_REQUIRE(ctx->have_integrals && k >= 1 && k + 1 <= ctx->L, DMRG_ERR_ARG, "rotate_integrals: integrals first, 1 <= k < L");
  const size_t n = (size_t)ctx->L, a = (size_t)k - 1, b = (size_t)k;
  const double c = std::cos(theta), s = std::sin(theta);
  ctx->drop_term_groups();              // (waits for builders that still read the old integrals)
  // new orbital a~ = c a + s b, b~ = -s a + c b (creation operators transform with the same matrix): every index of
  // T and w is rotated in turn
  auto rot = [&](std::vector<double>& t, int rank) {
    size_t stride = 1;
    for (int pos = rank - 1; pos >= 0; --pos, stride *= n) {
      const size_t total = t.size();
      for (size_t base = 0; base < total; ++base) {
        if ((base / stride) % n != a) continue;
        const size_t ib = base + (b - a) * stride;
        const double xa = t[base], xb = t[ib];
        t[base] = c * xa + s * xb;
        t[ib] = -s * xa + c * xb;
      }
    }
  };
  rot(ctx->T, 2);
  rot(ctx->w, 4);
  // every operator of every block depends on the integrals
  ctx->left_cache.clear(); ctx->right_cache.clear();
  ctx->left.reset(); ctx->right.reset();
  ctx->apply_plan.clear();
  ctx->k = 0;
  MO_END
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------
// dmrg_bond_entropy_static: dmrg_bond_entropy for callers that may not allocate device memory (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  The same two kernels; every device buffer they
// need beyond psi (sector and placement tables, the singular values, the three results) lives in ONE file-scope
// array of fixed size, which every GPU that loads the library holds until the process exits.
//
// In host code `g_entropy_scratch` is only a stand-in for the symbol: its device address is looked up once per device,
// with that device current, by cudaGetSymbolAddress, and it is that address the kernels are given.
// ------------------------------------------------------------------------------------------------------------------
namespace {

constexpr size_t ST_OFF_OUT = 0;                                                            // 3 doubles (256 B reserved)
constexpr size_t ST_OFF_SIGMA = 256;
constexpr size_t ST_OFF_SECS = ST_OFF_SIGMA + sizeof(double) * DMRG_STATIC_MAX_SIGMA;
constexpr size_t ST_OFF_PLACES = ST_OFF_SECS + sizeof(SvSector) * DMRG_STATIC_MAX_SECTORS;
constexpr size_t ST_BYTES = ST_OFF_PLACES + sizeof(SvPlace) * DMRG_STATIC_MAX_BLOCKS;
static_assert(ST_OFF_SECS % 256 == 0 && ST_OFF_PLACES % 256 == 0, "sub-arrays of the static scratch stay 256-byte aligned");
static_assert(ST_BYTES <= 128 * 1024, "the static scratch is meant to stay modest");

static __device__ __align__(256) unsigned char g_entropy_scratch[ST_BYTES];

constexpr int ST_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char* g_static_ptr[ST_MAX_DEVICES] = {};

// Device address of g_entropy_scratch on `device`, which must be the current device.
unsigned char* static_scratch(int device) {
  std::lock_guard<std::mutex> lk(g_static_mu);
  DMRG_REQUIRE(device >= 0 && device < ST_MAX_DEVICES, DMRG_ERR_ARG, "bond_entropy_static: device ordinal out of range");
  if (!g_static_ptr[device]) {
    int cur = -1;
    DMRG_CUDA(cudaGetDevice(&cur));
    DMRG_REQUIRE(cur == device, DMRG_ERR_CUDA, "bond_entropy_static: the device of the context is not current");
    void* p = nullptr;
    DMRG_CUDA(cudaGetSymbolAddress(&p, g_entropy_scratch));
    DMRG_REQUIRE(p != nullptr, DMRG_ERR_CUDA, "bond_entropy_static: cudaGetSymbolAddress returned a null address");
    g_static_ptr[device] = static_cast<unsigned char*>(p);
  }
  return g_static_ptr[device];
}

}  // namespace

extern "C" int dmrg_bond_entropy_static(dmrg_ctx* ctx, const double* d_psi, double* h_S_half, double* h_S_vn,
                                        double* h_sigma, int32_t* n_sigma, void* stream) {
  MO_BEGIN
  cudaStream_t st = (cudaStream_t)stream;
  DMRG_REQUIRE(ctx->k > 0 && d_psi, DMRG_ERR_ARG, "bond_entropy_static: no problem prepared or null pointer");
  DMRG_REQUIRE(!ctx->su2(), DMRG_ERR_UNSUPPORTED, "bond_entropy_static: U(1)xU(1) contexts only");
  DMRG_REQUIRE(ctx->psi.size() <= (size_t)DMRG_STATIC_MAX_BLOCKS, DMRG_ERR_UNSUPPORTED,
               "bond_entropy_static: " + std::to_string(ctx->psi.size()) + " psi blocks exceed the static scratch (DMRG_STATIC_MAX_BLOCKS = " +
                   std::to_string(DMRG_STATIC_MAX_BLOCKS) + "); use dmrg_bond_entropy");
  // sectors of bond k, as in dmrg_bond_entropy: q = q_L + q(s1); rows (q_L, s1), columns (s2, q_R); lexicographic in q
  const Sectors& SL = ctx->left->sec;
  struct Tmp { std::map<std::pair<int, int>, int> row0, col0; int rows = 0, cols = 0; std::vector<SvPlace> pl; };
  std::map<std::pair<int, int>, Tmp> by_q;
  for (auto& b : ctx->psi) {
    Tmp& t = by_q[{SL.qu[b.qL] + SITE_QU[b.s1], SL.qd[b.qL] + SITE_QD[b.s1]}];
    auto r = t.row0.find({b.qL, b.s1});
    if (r == t.row0.end()) { r = t.row0.emplace(std::make_pair(b.qL, b.s1), t.rows).first; t.rows += b.dL; }
    auto c = t.col0.find({b.s2, b.qR});
    if (c == t.col0.end()) { c = t.col0.emplace(std::make_pair(b.s2, b.qR), t.cols).first; t.cols += b.dR; }
    t.pl.push_back(SvPlace{b.off_c, b.dL, b.dR, r->second, c->second});
  }
  std::vector<SvSector> secs;
  std::vector<SvPlace> places;
  long long nsig = 0;
  size_t smem_max = 0;
  for (auto& kv : by_q) {
    Tmp& t = kv.second;
    SvSector s{(int)places.size(), 0, t.rows, t.cols, (int)nsig, 0};
    places.insert(places.end(), t.pl.begin(), t.pl.end());
    s.place_end = (int)places.size();
    const int n = std::min(t.rows, t.cols), m = std::max(t.rows, t.cols);
    smem_max = std::max(smem_max, (size_t)n * (m + 1) * 8);
    nsig += n;
    secs.push_back(s);
  }
  // the limits of the static scratch come first: they are this entry point's own
  DMRG_REQUIRE(nsig <= DMRG_STATIC_MAX_SIGMA, DMRG_ERR_UNSUPPORTED,
               "bond_entropy_static: " + std::to_string(nsig) + " singular values exceed the static scratch (DMRG_STATIC_MAX_SIGMA = " +
                   std::to_string(DMRG_STATIC_MAX_SIGMA) + "); use dmrg_bond_entropy");
  DMRG_REQUIRE(secs.size() <= (size_t)DMRG_STATIC_MAX_SECTORS, DMRG_ERR_UNSUPPORTED,
               "bond_entropy_static: " + std::to_string(secs.size()) + " bond sectors exceed the static scratch (DMRG_STATIC_MAX_SECTORS = " +
                   std::to_string(DMRG_STATIC_MAX_SECTORS) + "); use dmrg_bond_entropy");
  DMRG_REQUIRE(smem_max <= 220 * 1024, DMRG_ERR_UNSUPPORTED,
               "bond_entropy_static: a bond sector is larger than the shared-memory Jacobi kernel holds (mode optimisation runs at D <= 256)");
  if (n_sigma) *n_sigma = (int32_t)nsig;
  unsigned char* base = static_scratch(ctx->cfg.device);
  double* d_out = reinterpret_cast<double*>(base + ST_OFF_OUT);
  double* d_sigma = reinterpret_cast<double*>(base + ST_OFF_SIGMA);
  SvSector* d_secs = reinterpret_cast<SvSector*>(base + ST_OFF_SECS);
  SvPlace* d_places = reinterpret_cast<SvPlace*>(base + ST_OFF_PLACES);
  // Nothing here accumulates into the scratch: the tables are overwritten, k_sector_svals writes every sigma[0, nsig)
  // and k_entropies all three results before anything reads them, so the previous call's contents are never seen.
  // The results are cleared all the same, so that a kernel that failed to run cannot hand back the last call's values.
  DMRG_CUDA(cudaMemsetAsync(d_out, 0, 256, st));
  if (!secs.empty()) DMRG_CUDA(cudaMemcpyAsync(d_secs, secs.data(), secs.size() * sizeof(SvSector), cudaMemcpyHostToDevice, st));
  if (!places.empty()) DMRG_CUDA(cudaMemcpyAsync(d_places, places.data(), places.size() * sizeof(SvPlace), cudaMemcpyHostToDevice, st));
  DMRG_CUDA(cudaFuncSetAttribute(k_sector_svals, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max));
  if (!secs.empty()) k_sector_svals<<<(unsigned)secs.size(), 256, smem_max, st>>>(d_secs, d_places, d_psi, d_sigma);
  k_entropies<<<1, 256, 0, st>>>(d_sigma, (int)nsig, d_out);
  ctx->launches += 2;
  DMRG_CUDA(cudaGetLastError());
  double res[3];
  DMRG_CUDA(cudaMemcpyAsync(res, d_out, sizeof(res), cudaMemcpyDeviceToHost, st));
  if (h_sigma && nsig > 0) DMRG_CUDA(cudaMemcpyAsync(h_sigma, d_sigma, sizeof(double) * nsig, cudaMemcpyDeviceToHost, st));
  DMRG_CUDA(cudaStreamSynchronize(st));      // the host tables above must outlive the copies
  if (h_S_half) *h_S_half = res[0];
  if (h_S_vn) *h_S_vn = res[1];
  MO_END
}
