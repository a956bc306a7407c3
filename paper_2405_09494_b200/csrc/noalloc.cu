// gwsig_dyson_solve_noalloc (include/gwsig.h): Eq. 19a, for callers that may not allocate.
//
//   X_m = [1 - A_m]^{-1} A_m,   m < nmat,   A_m, X_m complex128 [n][n] row-major
//
// The same batched Gauss-Jordan elimination with partial pivoting as dyson_solve_kernel (kernels_aux.cu, used by
// gwsig_dyson_p), but the per-CTA augmented matrices [1 - A | A] live in a file-scope device array of fixed size instead of
// a buffer the context allocates: this entry point calls no cudaMalloc / cudaFree and no allocating library routine, takes
// no context, and does not synchronise.  Every GPU that loads the library holds the array (16 MiB) until the process exits.
//
// In HOST code `g_noalloc_scratch` is a host-side stand-in for the symbol, not a device address; the device address is
// resolved once per device with cudaGetSymbolAddress (device current) and handed to the kernel.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdio>
#include <mutex>

#include "gwsig.h"

namespace {

constexpr int kNmax = GWSIG_NOALLOC_NMAX;                               // 256
constexpr long long kScratchElems = GWSIG_NOALLOC_SCRATCH_BYTES / 16;   // complex128 elements
constexpr int kThreads = 256;
constexpr int kMaxCtas = 592;                                           // 4 per SM of a B200
static_assert(2LL * kNmax * kNmax <= kScratchElems, "the scratch must hold one augmented matrix of the largest size");

static __device__ __align__(256) double2 g_noalloc_scratch[kScratchElems];

// one CTA per matrix at a time; M = this CTA's slice of the scratch, [n][2n]: columns 0..n-1 = 1 - A -> 1, n..2n-1 = A -> X.
// Every element of M that is read was written earlier in the same matrix' pass, so stale contents of earlier calls never
// matter; `info` (caller's, cleared by the entry point) is the only word that has to start at zero.
__global__ void __launch_bounds__(kThreads) dyson_solve_noalloc_kernel(const double2* __restrict__ A_in, double2* X_out, int nmat, int n,
                                                                       double2* work, int* info) {
  __shared__ double2 prow[2 * kNmax];
  __shared__ double2 fac[kNmax];
  __shared__ double red_v[kThreads];
  __shared__ int red_i[kThreads];
  const int tid = threadIdx.x, nt = blockDim.x, w2 = 2 * n;
  double2* M = work + (long long)blockIdx.x * n * w2;
  for (int mat = blockIdx.x; mat < nmat; mat += gridDim.x) {
    const double2* A = A_in + (long long)mat * n * n;
    double2* X = X_out + (long long)mat * n * n;
    for (int e = tid; e < n * n; e += nt) {
      const int r = e / n, c = e - r * n;
      const double2 a = A[e];
      M[(long long)r * w2 + c] = make_double2((r == c ? 1.0 : 0.0) - a.x, -a.y);
      M[(long long)r * w2 + n + c] = a;
    }
    __syncthreads();
    for (int c = 0; c < n; ++c) {
      // pivot = row of largest |.|^2 in column c among rows c..n-1 (smallest row index among equals)
      double best = -1.0;
      int bi = c;
      for (int r = c + tid; r < n; r += nt) {
        const double2 v = M[(long long)r * w2 + c];
        const double a2 = v.x * v.x + v.y * v.y;
        if (a2 > best) { best = a2; bi = r; }
      }
      red_v[tid] = best; red_i[tid] = bi;
      __syncthreads();
      for (int s = nt / 2; s > 0; s >>= 1) {
        if (tid < s && (red_v[tid + s] > red_v[tid] || (red_v[tid + s] == red_v[tid] && red_i[tid + s] < red_i[tid]))) {
          red_v[tid] = red_v[tid + s]; red_i[tid] = red_i[tid + s];
        }
        __syncthreads();
      }
      const int piv = red_i[0];
      const double pv2 = red_v[0];
      if ((pv2 <= 0.0 || !(pv2 == pv2)) && tid == 0 && info) *info = 1;      // singular 1 - A or a non-finite input
      const double2 pv = M[(long long)piv * w2 + c];
      __syncthreads();
      const double inv_r = pv.x / pv2, inv_i = -pv.y / pv2;
      // swap rows c <-> piv on columns c..2n-1 while scaling the pivot row; keep the scaled row in shared memory
      for (int j = c + tid; j < w2; j += nt) {
        const double2 a = M[(long long)piv * w2 + j], b = M[(long long)c * w2 + j];
        const double2 sc = make_double2(a.x * inv_r - a.y * inv_i, a.x * inv_i + a.y * inv_r);
        if (piv != c) M[(long long)piv * w2 + j] = b;
        M[(long long)c * w2 + j] = sc;
        prow[j] = sc;
      }
      __syncthreads();
      for (int r = tid; r < n; r += nt) fac[r] = r == c ? make_double2(0.0, 0.0) : M[(long long)r * w2 + c];
      __syncthreads();
      const int wj = w2 - (c + 1);
      for (long long e = tid; e < (long long)n * wj; e += nt) {
        const int r = (int)(e / wj), j = c + 1 + (int)(e - (long long)r * wj);
        const double2 f = fac[r], pr = prow[j];
        double2* d = &M[(long long)r * w2 + j];
        d->x -= f.x * pr.x - f.y * pr.y;
        d->y -= f.x * pr.y + f.y * pr.x;
      }
      __syncthreads();
    }
    for (int e = tid; e < n * n; e += nt) X[e] = M[(long long)(e / n) * w2 + n + (e % n)];
    __syncthreads();
  }
}

// device address of g_noalloc_scratch, resolved once per device
std::mutex g_mu;
double2* g_scratch_ptr[64] = {};

int report(char* errbuf, int errbuf_len, int code, const char* what, const char* detail = "") {
  if (errbuf && errbuf_len > 0) std::snprintf(errbuf, (size_t)errbuf_len, "gwsig_dyson_solve_noalloc: %s%s", what, detail);
  return code;
}

}  // namespace

extern "C" int gwsig_dyson_solve_noalloc(const void* dA, void* dX, int nmat, int n, void* d_info, void* stream, char* errbuf,
                                         int errbuf_len) {
  if (errbuf && errbuf_len > 0) errbuf[0] = 0;
  if (nmat < 0 || n < 1) return report(errbuf, errbuf_len, GWSIG_ERR_ARG, "nmat < 0 or n < 1");
  if (n > kNmax) {
    char msg[160];
    std::snprintf(msg, sizeof(msg), "n = %d exceeds GWSIG_NOALLOC_NMAX = %d (the fixed %d MiB scratch holds one [n][2n] matrix per CTA)", n,
                  kNmax, (int)(GWSIG_NOALLOC_SCRATCH_BYTES >> 20));
    return report(errbuf, errbuf_len, GWSIG_ERR_ARG, msg);
  }
  if (nmat == 0) return GWSIG_OK;
  if (!dA || !dX) return report(errbuf, errbuf_len, GWSIG_ERR_ARG, "NULL device pointer");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return report(errbuf, errbuf_len, GWSIG_ERR_CUDA, "cudaGetDevice: ", cudaGetErrorString(e));
  if (dev < 0 || dev >= 64) return report(errbuf, errbuf_len, GWSIG_ERR_ARG, "device ordinal outside 0..63");
  double2* work = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
      double2* ptr = nullptr;
      e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);        // this device's copy of the array (device `dev` is current)
      if (e != cudaSuccess || !ptr) return report(errbuf, errbuf_len, GWSIG_ERR_CUDA, "cudaGetSymbolAddress: ", cudaGetErrorString(e));
      g_scratch_ptr[dev] = ptr;
    }
    work = g_scratch_ptr[dev];
  }
  const long long per = 2LL * n * n;
  const int ncta = (int)std::min<long long>(std::min<long long>(nmat, kScratchElems / per), kMaxCtas);
  cudaStream_t st = (cudaStream_t)stream;
  if (d_info) {
    e = cudaMemsetAsync(d_info, 0, sizeof(int), st);
    if (e != cudaSuccess) return report(errbuf, errbuf_len, GWSIG_ERR_CUDA, "cudaMemsetAsync(d_info): ", cudaGetErrorString(e));
  }
  dyson_solve_noalloc_kernel<<<(unsigned)ncta, kThreads, 0, st>>>((const double2*)dA, (double2*)dX, nmat, n, work, (int*)d_info);
  e = cudaGetLastError();
  if (e != cudaSuccess) return report(errbuf, errbuf_len, GWSIG_ERR_CUDA, "kernel launch: ", cudaGetErrorString(e));
  return GWSIG_OK;
}
