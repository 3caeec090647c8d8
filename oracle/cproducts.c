/* TEST INFRASTRUCTURE ONLY (oracle/): never linked, loaded or called by the product path.
 *
 * The contraction loop of the CPU oracle in plain C: psi'{out} += sg * op(mL) . psi{in} . op(mR)^T, one product per
 * (term, sector) task of PAPER.md Eq. (8) (:109-113: "the two-step contraction O_L psi O_R^T"), written as the two
 * triple loops of the definition -- no BLAS, no blocking, no reordering.  The list of products is made by
 * oracle/clevel.py from the SAME term list oracle/dmrg.py:TwoSiteOracle._accumulate walks (the C side has no term
 * enumeration of its own); this file only replaces numpy's `mL @ x @ mR.T`.  Pinned in tests/test_oracle_clevel.py
 * against that numpy loop and, through it, against P^T H_FCI P.
 *
 * Shares nothing with paper_2501_18263_b200/csrc/.  Built by oracle/clevel.py (gcc -O2 -fopenmp).
 */
#include <stdlib.h>
#include <string.h>

typedef struct {
  long long a_off, x_off, b_off; /* offsets (in doubles) of mL, the psi block and mR in `pool` */
  int a_rows, a_cols;            /* stored shape of mL */
  int x_rows, x_cols;            /* shape of the psi block */
  int b_rows, b_cols;            /* stored shape of mR */
  int ta, tb;                    /* ta: use mL^T; tb: use mR (i.e. op(mR)^T = mR) instead of mR^T */
  double sg;
} product_t;

/* out_off[o] .. : output block o is out_rows[o] x out_cols[o] at outpool + out_off[o];
 * its products are prods[first[o] .. first[o+1]) and are added in that order (fixed order: deterministic).
 * Returns 0, or -1 if a shape does not fit (nothing is written for that product's output from there on). */
int heff_products(const product_t* prods, const long long* first, long long nout, const long long* out_off,
                  const int* out_rows, const int* out_cols, const double* pool, double* outpool) {
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (long long o = 0; o < nout; ++o) {
    const int M = out_rows[o], N = out_cols[o];
    double* O = outpool + out_off[o];
    double* Y = NULL;
    long long ycap = 0;
    for (long long t = first[o]; t < first[o + 1]; ++t) {
      const product_t* p = &prods[t];
      const double* A = pool + p->a_off;
      const double* X = pool + p->x_off;
      const double* B = pool + p->b_off;
      const int am = p->ta ? p->a_cols : p->a_rows; /* rows of op(mL) */
      const int ak = p->ta ? p->a_rows : p->a_cols; /* = rows of psi block */
      const int bn = p->tb ? p->b_cols : p->b_rows; /* rows of op(mR) = columns of the output */
      const int bk = p->tb ? p->b_rows : p->b_cols; /* = columns of psi block */
      if (am != M || bn != N || ak != p->x_rows || bk != p->x_cols) {
#pragma omp atomic write
        bad = 1;
        break;
      }
      const int K1 = ak, K2 = bk;
      if ((long long)M * K2 > ycap) {
        free(Y);
        ycap = (long long)M * K2;
        Y = (double*)malloc(sizeof(double) * (size_t)ycap);
      }
      /* step 1: Y = op(mL) . psi   (M x K2) */
      for (int i = 0; i < M; ++i)
        for (int q = 0; q < K2; ++q) {
          double s = 0.0;
          for (int k = 0; k < K1; ++k) {
            const double a = p->ta ? A[(long long)k * p->a_cols + i] : A[(long long)i * p->a_cols + k];
            s += a * X[(long long)k * p->x_cols + q];
          }
          Y[(long long)i * K2 + q] = s;
        }
      /* step 2: O += sg * Y . op(mR)^T   (M x N) */
      for (int i = 0; i < M; ++i)
        for (int j = 0; j < N; ++j) {
          double s = 0.0;
          for (int q = 0; q < K2; ++q) {
            const double b = p->tb ? B[(long long)q * p->b_cols + j] : B[(long long)j * p->b_cols + q];
            s += Y[(long long)i * K2 + q] * b;
          }
          O[(long long)i * N + j] += p->sg * s;
        }
    }
    free(Y);
  }
  return bad ? -1 : 0;
}
