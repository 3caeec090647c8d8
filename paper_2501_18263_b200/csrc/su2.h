// SU(2) spin adaptation, host side: Clebsch-Gordan table, the rescaled 9j factor F of
// PAPER.md Eq. (10)-(11), and the task prefactors F_tau of Eq. (9).
//
// How prefactors are obtained here.  Every carried operator is an irreducible tensor
// operator X^k stored by its reduced elements, <S'M'|X^k_q|SM> = <S M; k q|S' M'> X_red[S',S]
// (Wigner-Eckart in Clebsch-Gordan form, reading R11).  The term engine enumerates the elementary strings
// of PAPER.md Eq. (1) exactly as in the U(1) case and names every block factor as a COMPONENT q of one of
// these tensor operators (or the transpose of a component); the coefficient a (term, sector) task carries
// is then the contraction of the Clebsch-Gordan tensors of the coupled states with the Wigner-Eckart
// coefficients of the factors, summed over all magnetic quantum numbers — the construction of PAPER.md
// Fig. 4 (:150), applied to the whole task (`phi_task`) or to one blocking step (`phi_blocking`).  The values
// are tabulated in hash maps keyed by the quantum numbers ("efficiently searchable lookup table",
// PAPER.md:142).  For a product of two tensor operators the same contraction equals F of Eq. (11);
// `F_ninej` is the closed form, exported through dmrg_su2_f_factor so that tests can compare the two.
#pragma once
#include <array>
#include <cstdint>
#include <unordered_map>
#include <vector>

namespace dmrg {
namespace su2 {

// site multiplets m = 0,1,2 = (N=0,S=0), (N=1,S=1/2), (N=2,S=0); doubled spins
static const int MULT_N[3] = {0, 1, 2};
static const int MULT_S2[3] = {0, 1, 0};
// U(1) site state (0, dn, up, updn) -> (multiplet, doubled S_z)
static const int STATE_M[4] = {0, 1, 1, 2};
static const int STATE_MU[4] = {0, -1, 1, 0};
inline int site_state(int m, int mu) { return m == 0 ? 0 : (m == 2 ? 3 : (mu > 0 ? 2 : 1)); }

// <j1 m1; j2 m2 | J M>, doubled integer arguments, Condon-Shortley phases (Racah's formula), memoised.
double cg(int j1, int m1, int j2, int m2, int J, int M);
double sixj(int a, int b, int c, int d, int e, int f);
double ninej(int a, int b, int c, int d, int e, int f, int g, int h, int i);
// PAPER.md Eq. (11): sqrt((2Sa'+1)(2Sk'+1)(2Sg+1)(2k+1)) * 9j{Sa Sk Sg; kL kk k; Sa' Sk' Sg'}
double F_ninej(int Sa, int Sk, int Sg, int kL, int kk, int kop, int Sa_, int Sk_, int Sg_);

// A block factor of an elementary string, named as a component of a carried tensor operator.
struct Comp {
  int kind;     // SKind
  int idx;      // operator index inside the kind
  int k2, q2;   // doubled rank and component
  bool tr;      // the factor is the TRANSPOSE of that component
  double coef;
};

// One blocking step: reduced element of the new operator (rank k2, defined by its highest-weight
// component) between new multiplets |(S1, m1) S1p> -> |(S2, m2) S2p>, per unit reduced element of the old
// operator block (S2 <- S1, or its transpose), for the site matrix `site` (4x4, rows = out).
// left = true: states |(block, site)>, operator order block.site; false: |(site, block)>, site.block.
// n_old1 = particle number of the old block's input sector; src_odd = the old operator changes N by an odd
// number.
double phi_blocking(bool left, int k2, int S1, int m1, int S1p, int S2, int m2, int S2p, int ko2, int qo2, bool tr,
                    bool src_is_identity, const double* site, int n_old1, bool src_odd);

// One task of PAPER.md Eq. (9) for total spin 0: <out| X_L (x) o1 (x) o2 (x) Y_R |in> per unit reduced elements,
// in = |((Sa, m1) Sp, (m2, Sb) Sp) 0>, out likewise (primed).  L/R: doubled rank, component, transpose flag,
// identity flag.  nL = particle number of the left input sector; pR = right operator is fermionic.
struct TaskKey {
  int Sa, m1, Sp, m2, Sb, Sa_, m1_, Sp_, m2_, Sb_;
  int kL, qL, trL, idL, kR, qR, trR, idR, o1, o2, nLodd, pR;
};
double phi_task(const TaskKey& key, const double* o1, const double* o2);

}  // namespace su2
}  // namespace dmrg
