// Host-side SU(2) coefficients (see su2.h).  Plain C++; compiled by nvcc with the rest of the library.
#include "su2.h"

#include <cmath>
#include <cstdlib>
#include <mutex>

namespace dmrg {
namespace su2 {

namespace {

struct FactTable {
  long double t[81];
  FactTable() {
    t[0] = 1.0L;
    for (int i = 1; i <= 80; ++i) t[i] = t[i - 1] * (long double)i;
  }
};
long double fact(int n) {   // n! for 0 <= n <= 80
  static const FactTable tab;   // function-local static: initialised once, thread-safe (C++11)
  return (n < 0 || n > 80) ? 0.0L : tab.t[n];
}
inline long double fh(int twice) { return fact(twice / 2); }   // (twice/2)!

double cg_raw(int j1, int m1, int j2, int m2, int J, int M) {
  if (m1 + m2 != M || J < std::abs(j1 - j2) || J > j1 + j2 || ((j1 + j2 + J) & 1)) return 0.0;
  if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(M) > J || ((j1 + m1) & 1) || ((j2 + m2) & 1) || ((J + M) & 1))
    return 0.0;
  long double pref = (long double)(J + 1) * fh(J + j1 - j2) * fh(J - j1 + j2) * fh(j1 + j2 - J) / fh(j1 + j2 + J + 2);
  pref *= fh(J + M) * fh(J - M) * fh(j1 - m1) * fh(j1 + m1) * fh(j2 - m2) * fh(j2 + m2);
  long double s = 0.0L;
  for (int k2 = 0; k2 <= j1 + j2 - J; k2 += 2) {
    const int a[6] = {k2, j1 + j2 - J - k2, j1 - m1 - k2, j2 + m2 - k2, J - j2 + m1 + k2, J - j1 - m2 + k2};
    bool ok = true;
    long double den = 1.0L;
    for (int x : a) {
      if (x < 0) { ok = false; break; }
      den *= fh(x);
    }
    if (!ok) continue;
    s += (((k2 / 2) & 1) ? -1.0L : 1.0L) / den;
  }
  return (double)(s * std::sqrt(pref));
}

std::mutex g_mu;
std::unordered_map<uint64_t, double> g_cg;

}  // namespace

double cg(int j1, int m1, int j2, int m2, int J, int M) {
  if (m1 + m2 != M) return 0.0;
  // spins stay far below 64 (doubled) in every supported problem
  const uint64_t key = ((uint64_t)(j1 & 127) << 35) | ((uint64_t)((m1 + 64) & 127) << 28) | ((uint64_t)(j2 & 127) << 21) |
                       ((uint64_t)((m2 + 64) & 127) << 14) | ((uint64_t)(J & 127) << 7) | (uint64_t)((M + 64) & 127);
  {
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_cg.find(key);
    if (it != g_cg.end()) return it->second;
  }
  const double v = cg_raw(j1, m1, j2, m2, J, M);
  std::lock_guard<std::mutex> lk(g_mu);
  g_cg[key] = v;
  return v;
}

double sixj(int a, int b, int c, int d, int e, int f) {
  auto tri = [](int x, int y, int z, long double* out) {
    if (((x + y + z) & 1) || z < std::abs(x - y) || z > x + y) return false;
    *out = fh(x + y - z) * fh(x - y + z) * fh(-x + y + z) / fh(x + y + z + 2);
    return true;
  };
  long double t1, t2, t3, t4;
  if (!tri(a, b, c, &t1) || !tri(a, e, f, &t2) || !tri(d, b, f, &t3) || !tri(d, e, c, &t4)) return 0.0;
  const int lo = std::max(std::max(a + b + c, a + e + f), std::max(d + b + f, d + e + c));
  const int hi = std::min(std::min(a + b + d + e, b + c + e + f), a + c + d + f);
  long double s = 0.0L;
  for (int t = lo; t <= hi; t += 2) {
    long double den = fh(t - a - b - c) * fh(t - a - e - f) * fh(t - d - b - f) * fh(t - d - e - c) *
                      fh(a + b + d + e - t) * fh(b + c + e + f - t) * fh(a + c + d + f - t);
    s += (((t / 2) & 1) ? -1.0L : 1.0L) * fh(t + 2) / den;
  }
  return (double)(s * std::sqrt(t1 * t2 * t3 * t4));
}

double ninej(int a, int b, int c, int d, int e, int f, int g, int h, int i) {
  double s = 0.0;
  const int lo = std::max(std::max(std::abs(a - i), std::abs(d - h)), std::abs(b - f));
  const int hi = std::min(std::min(a + i, d + h), b + f);
  for (int x = lo; x <= hi; ++x) {
    if ((x + a + i) & 1) continue;
    s += ((x & 1) ? -1.0 : 1.0) * (x + 1) * sixj(a, b, c, f, i, x) * sixj(d, e, f, b, x, h) * sixj(g, h, i, x, a, d);
  }
  return s;
}

double F_ninej(int Sa, int Sk, int Sg, int kL, int kk, int kop, int Sa_, int Sk_, int Sg_) {
  return std::sqrt((double)(Sa_ + 1) * (Sk_ + 1) * (Sg + 1) * (kop + 1)) * ninej(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_);
}

// <S2 M2| X_q or (X_q)^T |S1 M1> per unit reduced element (Wigner-Eckart, Clebsch-Gordan form)
static inline double we(bool is_id, bool tr, int k2, int q2, int S1, int M1, int S2, int M2) {
  if (is_id) return (S1 == S2 && M1 == M2) ? 1.0 : 0.0;
  return tr ? cg(S2, M2, k2, q2, S1, M1) : cg(S1, M1, k2, q2, S2, M2);
}

double phi_blocking(bool left, int k2, int S1, int m1, int S1p, int S2, int m2, int S2p, int ko2, int qo2, bool tr,
                    bool src_is_identity, const double* site, int n_old1, bool src_odd) {
  // new operator defined by its highest-weight component q = k; evaluate at M2' = S2', M1' = S2' - k
  const int M2p = S2p, M1p = S2p - k2;
  if (std::abs(M1p) > S1p) return 0.0;
  const double den = cg(S1p, M1p, k2, k2, S2p, M2p);
  if (den == 0.0) return 0.0;
  const int s1m = MULT_S2[m1], s2m = MULT_S2[m2];
  double tot = 0.0;
  for (int mu1 = -s1m; mu1 <= s1m; mu1 += 2) {
    const int M1 = M1p - mu1;
    if (std::abs(M1) > S1) continue;
    const double c1 = left ? cg(S1, M1, s1m, mu1, S1p, M1p) : cg(s1m, mu1, S1, M1, S1p, M1p);
    if (c1 == 0.0) continue;
    const int st1 = site_state(m1, mu1);
    for (int st2 = 0; st2 < 4; ++st2) {
      const double sv = site[st2 * 4 + st1];
      if (sv == 0.0 || STATE_M[st2] != m2) continue;
      const int mu2 = STATE_MU[st2];
      const int M2 = M2p - mu2;
      if (std::abs(M2) > S2) continue;
      const double c2 = left ? cg(S2, M2, s2m, mu2, S2p, M2p) : cg(s2m, mu2, S2, M2, S2p, M2p);
      if (c2 == 0.0) continue;
      const double w = we(src_is_identity, tr, ko2, qo2, S1, M1, S2, M2);
      if (w == 0.0) continue;
      double sg = 1.0;
      if (left) {   // block.site: the site operator passes the old block's input state
        const int spar = (MULT_N[m2] - MULT_N[m1]) & 1;
        if (spar && (n_old1 & 1)) sg = -1.0;
      } else {      // site.block: the block operator passes the site's input state
        if (src_odd && (MULT_N[m1] & 1)) sg = -1.0;
      }
      tot += c1 * c2 * w * sv * sg;
    }
  }
  return tot / den;
}

double phi_task(const TaskKey& K, const double* o1, const double* o2) {
  const int s1m = MULT_S2[K.m1], s2m = MULT_S2[K.m2], s1m_ = MULT_S2[K.m1_], s2m_ = MULT_S2[K.m2_];
  const int p1 = (MULT_N[K.m1_] - MULT_N[K.m1]) & 1, p2 = (MULT_N[K.m2_] - MULT_N[K.m2]) & 1;
  double tot = 0.0;
  for (int Mp = -K.Sp; Mp <= K.Sp; Mp += 2) {
    const double ct = cg(K.Sp, Mp, K.Sp, -Mp, 0, 0);
    for (int mu1 = -s1m; mu1 <= s1m; mu1 += 2) {
      const int Ma = Mp - mu1;
      if (std::abs(Ma) > K.Sa) continue;
      const double c1 = cg(K.Sa, Ma, s1m, mu1, K.Sp, Mp);
      if (c1 == 0.0) continue;
      const int st1 = site_state(K.m1, mu1);
      for (int mu2 = -s2m; mu2 <= s2m; mu2 += 2) {
        const int Mb = -Mp - mu2;
        if (std::abs(Mb) > K.Sb) continue;
        const double c2 = cg(s2m, mu2, K.Sb, Mb, K.Sp, -Mp);
        if (c2 == 0.0) continue;
        const int st2 = site_state(K.m2, mu2);
        // fermion sign: operators right of a part pass that part's input state
        const int n1 = MULT_N[K.m1], n2 = MULT_N[K.m2];
        const int ph = K.nLodd * (p1 + p2 + K.pR) + n1 * (p2 + K.pR) + n2 * K.pR;
        const double sg = (ph & 1) ? -1.0 : 1.0;
        for (int mu1_ = -s1m_; mu1_ <= s1m_; mu1_ += 2) {
          const int st1_ = site_state(K.m1_, mu1_);
          const double v1 = o1[st1_ * 4 + st1];
          if (v1 == 0.0) continue;
          for (int mu2_ = -s2m_; mu2_ <= s2m_; mu2_ += 2) {
            const int st2_ = site_state(K.m2_, mu2_);
            const double v2 = o2[st2_ * 4 + st2];
            if (v2 == 0.0) continue;
            const int Ma_ = K.idL ? Ma : (K.trL ? Ma - K.qL : Ma + K.qL);
            const int Mb_ = K.idR ? Mb : (K.trR ? Mb - K.qR : Mb + K.qR);
            if (std::abs(Ma_) > K.Sa_ || std::abs(Mb_) > K.Sb_) continue;
            const int Mp_ = Ma_ + mu1_;
            if (Mb_ + mu2_ != -Mp_ || std::abs(Mp_) > K.Sp_) continue;
            const double wl = we(K.idL, K.trL, K.kL, K.qL, K.Sa, Ma, K.Sa_, Ma_);
            if (wl == 0.0) continue;
            const double wr = we(K.idR, K.trR, K.kR, K.qR, K.Sb, Mb, K.Sb_, Mb_);
            if (wr == 0.0) continue;
            const double co = cg(K.Sp_, Mp_, K.Sp_, -Mp_, 0, 0) * cg(K.Sa_, Ma_, s1m_, mu1_, K.Sp_, Mp_) *
                              cg(s2m_, mu2_, K.Sb_, Mb_, K.Sp_, -Mp_);
            tot += ct * c1 * c2 * co * wl * wr * v1 * v2 * sg;
          }
        }
      }
    }
  }
  return tot;
}

}  // namespace su2
}  // namespace dmrg
