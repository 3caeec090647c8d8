#include "kernels.cuh"

namespace dmrg {

namespace {

__global__ void k_pack(const PsiBlockDev* __restrict__ blocks, const double* __restrict__ compact,
                       double* __restrict__ padded) {
  const PsiBlockDev b = blocks[blockIdx.x];
  const long long n = (long long)b.rows * b.cols;
  for (long long e = threadIdx.x + (long long)blockIdx.y * blockDim.x; e < n;
       e += (long long)blockDim.x * gridDim.y) {
    int r = (int)(e / b.cols), c = (int)(e % b.cols);
    padded[b.off_p + (long long)r * b.cols_p + c] = compact[b.off_c + e];
  }
}

__global__ void k_unpack(const PsiBlockDev* __restrict__ blocks, const double* __restrict__ padded,
                         double* __restrict__ compact, double shift, const double* __restrict__ x) {
  const PsiBlockDev b = blocks[blockIdx.x];
  const long long n = (long long)b.rows * b.cols;
  for (long long e = threadIdx.x + (long long)blockIdx.y * blockDim.x; e < n;
       e += (long long)blockDim.x * gridDim.y) {
    int r = (int)(e / b.cols), c = (int)(e % b.cols);
    double v = padded[b.off_p + (long long)r * b.cols_p + c];
    if (x) v += shift * x[b.off_c + e];
    compact[b.off_c + e] = v;
  }
}

// stage 1: per-block partial sums in a fixed order (thread-strided, then shared-memory tree)
__global__ void k_multidot1(const double* __restrict__ x, const double* __restrict__ Y, long long ldy,
                            long long n, double* __restrict__ partials) {
  __shared__ double sh[256];
  const double* y = Y + (long long)blockIdx.y * ldy;
  double s = 0.0;
  const long long n2 = n >> 1;   // n is even (padded layout)
  const double2* x2 = reinterpret_cast<const double2*>(x);
  const double2* y2 = reinterpret_cast<const double2*>(y);
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n2;
       i += (long long)blockDim.x * gridDim.x) {
    double2 a = x2[i], b = y2[i];
    s = fma(a.x, b.x, s);
    s = fma(a.y, b.y, s);
  }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) partials[(long long)blockIdx.y * gridDim.x + blockIdx.x] = sh[0];
}

__global__ void k_multidot2(const double* __restrict__ partials, int nb, double* __restrict__ out) {
  __shared__ double sh[256];
  double s = 0.0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) s += partials[(long long)blockIdx.x * nb + i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int w = 128; w > 0; w >>= 1) {
    if (threadIdx.x < w) sh[threadIdx.x] += sh[threadIdx.x + w];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[blockIdx.x] = sh[0];
}

__global__ void k_combine(const double* __restrict__ V, long long ldv, const double* __restrict__ c,
                          int m, long long n, double* __restrict__ y, int subtract) {
  __shared__ double cs[64];
  if (threadIdx.x < m) cs[threadIdx.x] = c[threadIdx.x];
  __syncthreads();
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n;
       i += (long long)blockDim.x * gridDim.x) {
    double s = 0.0;
    for (int j = 0; j < m; ++j) s = fma(cs[j], V[(long long)j * ldv + i], s);
    y[i] = subtract ? (y[i] - s) : s;
  }
}

__global__ void k_axpy(double a, const double* __restrict__ x, double* __restrict__ y, long long n) {
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n;
       i += (long long)blockDim.x * gridDim.x)
    y[i] = fma(a, x[i], y[i]);
}

__global__ void k_scale(double a, double* __restrict__ y, long long n) {
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n;
       i += (long long)blockDim.x * gridDim.x)
    y[i] *= a;
}

__global__ void k_add_const(double a, double* __restrict__ y, long long n) {
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n;
       i += (long long)blockDim.x * gridDim.x)
    y[i] += a;
}

__global__ void k_resid(const double* __restrict__ x, const double* __restrict__ hx,
                        const double* __restrict__ d, double theta, double theta_d, double* __restrict__ r,
                        double* __restrict__ t, long long n) {
  for (long long i = threadIdx.x + (long long)blockIdx.x * blockDim.x; i < n;
       i += (long long)blockDim.x * gridDim.x) {
    double rv = hx[i] - theta * x[i];
    double den = theta_d - d[i];
    if (fabs(den) < 1e-12) den = den < 0 ? -1e-12 : 1e-12;
    r[i] = rv;
    t[i] = rv / den;
  }
}

constexpr int DIAG_T = 4, DIAG_MAXD = 640;   // 40 KB of static shared memory
__global__ void k_diag(const PsiBlockDev* __restrict__ blocks, const DiagTask* __restrict__ tasks,
                       const int* __restrict__ task_begin, double* __restrict__ out) {
  __shared__ double dl[DIAG_T][DIAG_MAXD];
  __shared__ double dr[DIAG_T][DIAG_MAXD];
  const PsiBlockDev b = blocks[blockIdx.x];
  const int t0 = task_begin[blockIdx.x], t1 = task_begin[blockIdx.x + 1];
  // sectors larger than DIAG_MAXD are covered by (row range) x (column range) panels
  for (int r0 = 0; r0 < b.rows; r0 += DIAG_MAXD)
    for (int q0 = 0; q0 < b.cols; q0 += DIAG_MAXD) {
      const int nr = min(DIAG_MAXD, b.rows - r0), nq = min(DIAG_MAXD, b.cols - q0);
      const int n = nr * nq;
      for (int e = threadIdx.x; e < n; e += blockDim.x)
        out[b.off_p + (long long)(r0 + e / nq) * b.cols_p + (q0 + e % nq)] = 0.0;
      __syncthreads();
      for (int t = t0; t < t1; ++t) {
        const DiagTask tk = tasks[t];
        for (int c0 = 0; c0 < tk.count; c0 += DIAG_T) {
          const int nc = min(DIAG_T, tk.count - c0);
          for (int idx = threadIdx.x; idx < nc * nr; idx += blockDim.x) {
            int c = idx / nr, a = r0 + idx % nr;
            dl[c][idx % nr] = tk.L ? tk.L[(long long)(c0 + c) * tk.rsL + (long long)a * tk.ldl + a] : 1.0;
          }
          for (int idx = threadIdx.x; idx < nc * nq; idx += blockDim.x) {
            int c = idx / nq, a = q0 + idx % nq;
            dr[c][idx % nq] = tk.R ? tk.R[(long long)(c0 + c) * tk.rsR + (long long)a * tk.ldr + a] : 1.0;
          }
          __syncthreads();
          for (int e = threadIdx.x; e < n; e += blockDim.x) {
            int r = e / nq, c = e % nq;
            double s = 0.0;
            for (int q = 0; q < nc; ++q) s = fma(dl[q][r], dr[q][c], s);
            out[b.off_p + (long long)(r0 + r) * b.cols_p + (q0 + c)] += tk.alpha * s;
          }
          __syncthreads();
        }
      }
    }
}

__global__ void k_reduce_partials(const RedDesc* __restrict__ ds) {
  const RedDesc d = ds[blockIdx.x];
  const int b = blockIdx.y;
  if (b >= d.batch) return;
  const long long mn = (long long)d.M * d.N;
  double* C = d.C + (long long)b * d.bsC;
  for (long long e = threadIdx.x; e < mn; e += blockDim.x) {
    const int r = (int)(e / d.N), c = (int)(e % d.N);
    double s = C[(long long)r * d.ldc + c];
    for (int p = 0; p < d.nparts; ++p) s += d.P[((long long)p * d.batch + b) * mn + e];
    C[(long long)r * d.ldc + c] = s;
  }
}

__global__ void k_dmma_peak(double* out, int iters, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;   // keeps the loop alive without a store on the normal path
}

__global__ void k_dfma_peak(double* out, int iters, double a, double b) {
  double c[16];
#pragma unroll
  for (int i = 0; i < 16; i++) c[i] = threadIdx.x + i;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) c[i] = fma(c[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += c[i];
  if (s == 12345.678) out[0] = s;
}

inline int grid_for(long long n) {
  long long g = (n + 255) / 256;
  return (int)(g < 1 ? 1 : (g > 1184 ? 1184 : g));
}

}  // namespace

void launch_pack(const PsiBlockDev* blocks, int nblocks, const double* compact, double* padded, cudaStream_t st) {
  if (nblocks > 0) k_pack<<<dim3(nblocks, 4), 256, 0, st>>>(blocks, compact, padded);
}
void launch_unpack(const PsiBlockDev* blocks, int nblocks, const double* padded, double* compact,
                   double shift, const double* x, cudaStream_t st) {
  if (nblocks > 0) k_unpack<<<dim3(nblocks, 4), 256, 0, st>>>(blocks, padded, compact, shift, x);
}
void launch_multidot(const double* x, const double* Y, long long ldy, int m, long long n,
                     double* partials, double* out, cudaStream_t st) {
  if (m <= 0) return;
  k_multidot1<<<dim3(DOT_BLOCKS, m), 256, 0, st>>>(x, Y, ldy, n, partials);
  k_multidot2<<<m, 256, 0, st>>>(partials, DOT_BLOCKS, out);
}
void launch_combine(const double* V, long long ldv, const double* c, int m, long long n, double* y, cudaStream_t st) {
  k_combine<<<grid_for(n), 256, 0, st>>>(V, ldv, c, m, n, y, 0);
}
void launch_project_out(const double* V, long long ldv, const double* c, int m, long long n, double* y, cudaStream_t st) {
  k_combine<<<grid_for(n), 256, 0, st>>>(V, ldv, c, m, n, y, 1);
}
void launch_axpy(double a, const double* x, double* y, long long n, cudaStream_t st) {
  k_axpy<<<grid_for(n), 256, 0, st>>>(a, x, y, n);
}
void launch_scale(double a, double* y, long long n, cudaStream_t st) {
  k_scale<<<grid_for(n), 256, 0, st>>>(a, y, n);
}
void launch_add_const(double a, double* y, long long n, cudaStream_t st) {
  k_add_const<<<grid_for(n), 256, 0, st>>>(a, y, n);
}
void launch_residual_precond(const double* x, const double* hx, const double* d, double theta, double theta_d,
                             double* r, double* t, long long n, cudaStream_t st) {
  k_resid<<<grid_for(n), 256, 0, st>>>(x, hx, d, theta, theta_d, r, t, n);
}
void launch_diag(const PsiBlockDev* blocks, int nblocks, const DiagTask* tasks, const int* task_begin,
                 double* out_p, cudaStream_t st) {
  if (nblocks > 0) k_diag<<<nblocks, 256, 0, st>>>(blocks, tasks, task_begin, out_p);
}

void launch_reduce_partials(const RedDesc* d, int n, int max_batch, cudaStream_t st) {
  if (n > 0) k_reduce_partials<<<dim3(n, max_batch), 256, 0, st>>>(d);
}

cudaError_t measure_dmma_peak(double* dummy, double* tflops, cudaStream_t st) {
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaError_t e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 20000, threads = 512;
  k_dmma_peak<<<sms, threads, 0, st>>>(dummy, 2000, 1.0000001, 1e-9);
  cudaEventRecord(e0, st);
  k_dmma_peak<<<sms, threads, 0, st>>>(dummy, iters, 1.0000001, 1e-9);
  cudaEventRecord(e1, st);
  e = cudaEventSynchronize(e1);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  double fl = 2.0 * 8 * 8 * 4 * 8.0 * iters * (threads / 32.0) * sms;
  *tflops = fl / (ms * 1e-3) * 1e-12;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return e;
}

cudaError_t measure_dfma_peak(double* dummy, double* tflops, cudaStream_t st) {
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 20000, threads = 1024;
  k_dfma_peak<<<2 * sms, threads, 0, st>>>(dummy, 2000, 1.0000001, 1e-9);
  cudaEventRecord(e0, st);
  k_dfma_peak<<<2 * sms, threads, 0, st>>>(dummy, iters, 1.0000001, 1e-9);
  cudaEventRecord(e1, st);
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  const double fl = 2.0 * 16.0 * iters * threads * 2.0 * sms;
  *tflops = fl / (ms * 1e-3) * 1e-12;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return e;
}

}  // namespace dmrg
