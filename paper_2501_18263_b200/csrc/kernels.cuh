// Auxiliary kernels: psi pack/unpack between the compact C-ABI layout and the zero-padded internal
// layout, the HBM-bound Davidson vector operations (DESIGN.md App. E), the H_eff diagonal, and the
// DMMA peak probe.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace dmrg {

struct PsiBlockDev {
  long long off_c;   // offset in the compact vector
  long long off_p;   // offset in the padded vector
  int rows, cols, rows_p, cols_p;
};

struct DiagTask {
  const double* L;   // block of the left operator (or nullptr = identity)
  const double* R;
  long long rsL, rsR;
  int ldl, ldr;
  int count;
  int pad_;
  double alpha;
};

// padded[blocks] = compact (pads untouched: caller keeps them zero)
void launch_pack(const PsiBlockDev* blocks, int nblocks, const double* compact, double* padded, cudaStream_t st);
// compact = padded + shift * x_compact  (x_compact may be nullptr when shift == 0)
void launch_unpack(const PsiBlockDev* blocks, int nblocks, const double* padded, double* compact,
                   double shift, const double* x_compact, cudaStream_t st);

constexpr int DOT_BLOCKS = 592;   // 4 per SM, fixed => deterministic reduction tree
// out[j] = sum_i x[i] * Y[j*ldy + i], j < m   (two kernels; `partials` holds m*DOT_BLOCKS doubles)
void launch_multidot(const double* x, const double* Y, long long ldy, int m, long long n,
                     double* partials, double* out, cudaStream_t st);
// y = sum_j c[j] * V[j*ldv + i]  (c on device, m <= 64)
void launch_combine(const double* V, long long ldv, const double* c, int m, long long n, double* y, cudaStream_t st);
// y += a * x
void launch_axpy(double a, const double* x, double* y, long long n, cudaStream_t st);
// y -= sum_j c[j] * V[j]   (c on device)
void launch_project_out(const double* V, long long ldv, const double* c, int m, long long n, double* y, cudaStream_t st);
// y += a (every element)
void launch_add_const(double a, double* y, long long n, cudaStream_t st);
// y = a * y
void launch_scale(double a, double* y, long long n, cudaStream_t st);
// r = hx - theta*x ; t = r / clamp(theta_d - d) with |theta_d - d| >= 1e-12, sign kept.  theta is the Ritz value of
// the operator hx was made with (e_core included), theta_d the same value on the scale of the diagonal d
// (which is stored without e_core).
void launch_residual_precond(const double* x, const double* hx, const double* d, double theta, double theta_d,
                             double* r, double* t, long long n, cudaStream_t st);
// diag(H_eff): out_p[block] = sum_tasks alpha * diag(L) (x) diag(R)
void launch_diag(const PsiBlockDev* blocks, int nblocks, const DiagTask* tasks, const int* task_begin,
                 double* out_p, cudaStream_t st);
// split-K partial sums: C[b] += P[0][b] + P[1][b] + ... (fixed order => deterministic)
struct RedDesc {
  double* C;
  const double* P;           // part p, batch b at P + (p * batch + b) * M * N, row-major with ld = N
  long long bsC;
  int M, N, ldc, nparts, batch, pad_;
};
void launch_reduce_partials(const RedDesc* d, int n, int max_batch, cudaStream_t st);
// register-only DMMA loop; returns achieved TFLOP/s
constexpr int DIAG_MAX_DIM = 640;
cudaError_t measure_dmma_peak(double* d_scratch, double* tflops, cudaStream_t st);
// register-only DFMA loop (FP64 vector pipe); returns achieved TFLOP/s
cudaError_t measure_dfma_peak(double* d_scratch, double* tflops, cudaStream_t st);

}  // namespace dmrg
