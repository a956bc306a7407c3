// HBM-bound helper kernels of the hot path: structured unfold (Eq. 22 / 25), the Sigma
// epilogue (scale, optional Hermitise), and the FP64 issue-rate probes used by bench.py.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "kernels_aux.cuh"

namespace {

// out[r,c] = sum_{m in nz(r)} sum_{n in nz(c)} P[r,m] ph[m] X[m,n] P[c,n] conj(ph[n])
// O^k(alpha^) = P . diag(ph) is never formed densely: P = (atom permutation) x (real Wigner D) has at
// most 2l+1 <= 9 entries per row (Eq. 3-4).  X^{k~} = O X^k O^dagger (Eq. 22).
__global__ void __launch_bounds__(256) unfold_sparse_kernel(UnfoldParams p) {
  const int tgt = blockIdx.x / p.ntau, t = blockIdx.x % p.ntau;      // (target, tau) on grid.x: Nk * ntau exceeds 65535 at cfg5
  const int e = blockIdx.y * blockDim.x + threadIdx.x;
  const int n = p.n;
  if (e >= n * n) return;
  const int r = e / n, c = e - r * n;
  const int op = p.tgt_op[tgt];
  const double2* X = p.src + ((long long)p.tgt_src[tgt] * p.ntau + t) * n * n;
  const double2* ph = p.colphase + (long long)tgt * n;
  const int* rc = p.ell_cols + ((long long)op * n + r) * p.maxnz;
  const double* rv = p.ell_vals + ((long long)op * n + r) * p.maxnz;
  const int* cc = p.ell_cols + ((long long)op * n + c) * p.maxnz;
  const double* cv = p.ell_vals + ((long long)op * n + c) * p.maxnz;
  const int nr = p.ell_cnt[op * n + r], nc = p.ell_cnt[op * n + c];
  double sr = 0.0, si = 0.0;
  for (int a = 0; a < nr; ++a) {
    const int m = rc[a];
    const double2 pm = ph[m];
    const double wr = rv[a] * pm.x, wi = rv[a] * pm.y;        // P[r,m] ph[m]
    double tr = 0.0, ti = 0.0;                                // sum_n X[m,n] P[c,n] conj(ph[n])
    for (int b = 0; b < nc; ++b) {
      const int nn = cc[b];
      const double2 x = X[(long long)m * n + nn];
      const double2 pn = ph[nn];
      const double ur = cv[b] * pn.x, ui = -cv[b] * pn.y;
      tr += x.x * ur - x.y * ui;
      ti += x.x * ui + x.y * ur;
    }
    sr += wr * tr - wi * ti;
    si += wr * ti + wi * tr;
  }
  p.dst[((long long)tgt * p.ntau + t) * n * n + e] = make_double2(sr, si);
}

// Sigma = scale * acc, optionally (Sigma + Sigma^dagger)/2, for a list of square-matrix batches.
__global__ void __launch_bounds__(256) epilogue_kernel(EpilogueParams p) {
  const int d = blockIdx.y;
  const EpiDesc D = p.desc[d];
  const long long total = (long long)D.count * D.n * D.n;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const int nn = D.n * D.n;
    const long long t = e / nn;
    const int ij = (int)(e - t * nn);
    const int i = ij / D.n, j = ij - i * D.n;
    const long long base = D.off + t * D.stride;
    double2 v = p.acc[base + ij];
    if (p.hermitize) {
      const double2 w = p.acc[base + (long long)j * D.n + i];
      v.x = 0.5 * (v.x + w.x);
      v.y = 0.5 * (v.y - w.y);
    }
    p.out[base + ij] = make_double2(p.scale * v.x, p.scale * v.y);
  }
}

// deterministic stage 3: one thread per element of a Sigma block, the block's split-K partial tiles added in part order
__global__ void __launch_bounds__(256) reduce_parts_kernel(const RedGroupDev* groups, const double2* partial, double2* acc, int t0) {
  const RedGroupDev g = groups[blockIdx.y];
  const long long total = (long long)g.M * g.ni;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
    const double2* src = partial + g.part_off + e;
    double sr = 0.0, si = 0.0;
    for (int p = 0; p < g.nparts; ++p) {
      const double2 v = src[(long long)p * total];
      sr += v.x; si += v.y;
    }
    const int row = (int)(e / g.ni), j = (int)(e - (long long)row * g.ni);      // row = (tau, i)
    const int tau = row / g.ni, i = row - tau * g.ni;
    double2* dst = acc + g.c_off + (long long)(t0 + tau) * g.sts + (long long)i * g.ni + j;
    dst->x += sr; dst->y += si;
  }
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// register-only issue-rate probes: NACC independent accumulator chains per warp
template <int NACC>
__global__ void probe_dmma_kernel(long long iters, double* sink) {
  double c0[NACC], c1[NACC];
#pragma unroll
  for (int a = 0; a < NACC; ++a) { c0[a] = threadIdx.x * 1e-9; c1[a] = a * 1e-9; }
  double x = 1.0 + 1e-12 * threadIdx.x, y = 1.0 - 1e-12 * threadIdx.x;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int a = 0; a < NACC; ++a) dmma884(c0[a], c1[a], x, y);
  }
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < NACC; ++a) s += c0[a] + c1[a];
  if (s == 123.456) sink[0] = s;
}

template <int NACC>
__global__ void probe_dfma_kernel(long long iters, double* sink) {
  double c[NACC];
#pragma unroll
  for (int a = 0; a < NACC; ++a) c[a] = threadIdx.x * 1e-9 + a;
  double x = 1.0 + 1e-12 * threadIdx.x, y = 1e-9;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int a = 0; a < NACC; ++a) c[a] = fma(c[a], x, y);
  }
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < NACC; ++a) s += c[a];
  if (s == 123.456) sink[0] = s;
}

// both pipes' instructions interleaved in every warp: if DMMA and DFMA were separate pipes the sum of the
// two rates would exceed either probe alone
template <int NACC>
__global__ void probe_mixed_kernel(long long iters, double* sink) {
  double c0[NACC], c1[NACC], c[NACC];
#pragma unroll
  for (int a = 0; a < NACC; ++a) { c0[a] = threadIdx.x * 1e-9; c1[a] = a * 1e-9; c[a] = threadIdx.x * 1e-9 + a; }
  double x = 1.0 + 1e-12 * threadIdx.x, y = 1.0 - 1e-12 * threadIdx.x, z = 1e-9;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int a = 0; a < NACC; ++a) {
      dmma884(c0[a], c1[a], x, y);
#pragma unroll
      for (int r = 0; r < 8; ++r) c[(a + r) % NACC] = fma(c[(a + r) % NACC], x, z);    // 8 DFMA (256 lane-FMAs) per DMMA (256 FMAs)
    }
  }
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < NACC; ++a) s += c0[a] + c1[a] + c[a];
  if (s == 123.456) sink[0] = s;
}

}  // namespace

cudaError_t launch_unfold_sparse(const UnfoldParams& p, int ntarget, cudaStream_t stream) {
  if (ntarget <= 0) return cudaSuccess;
  dim3 grid((unsigned)((long long)ntarget * p.ntau), (unsigned)((p.n * p.n + 255) / 256));
  unfold_sparse_kernel<<<grid, 256, 0, stream>>>(p);
  return cudaGetLastError();
}

// P0 (Eq. 20): dst[k][n] = src[k][reverse ? ntau-1-n : n]^T for square matrices of side nao.  Stages 1 and 2 of Algorithm 3
// contract G over its SECOND index (X1 = sum_d G[c,d] T[d,..]); the transposed copy makes the tile rows (c) the contiguous index
// of the A operand, as in stage 1 of the Sigma path.  One CTA per (k, tau); the matrices are small (nao <= a few hundred).
__global__ void __launch_bounds__(256) transpose_tau_kernel(const double2* src, double2* dst, int ntau, int nao, int reverse) {
  const long long kt = blockIdx.x;                       // k * ntau + n   (grid.x: Nk * ntau exceeds 65535 at config 5)
  const long long k = kt / ntau, n = kt % ntau;
  const long long elems = (long long)nao * nao;
  const double2* s_ = src + (k * ntau + (reverse ? ntau - 1 - n : n)) * elems;
  double2* d_ = dst + kt * elems;
  for (long long e = threadIdx.x; e < elems; e += blockDim.x) {
    const int r = (int)(e / nao), c = (int)(e - (long long)r * nao);
    d_[e] = s_[(long long)c * nao + r];
  }
}

cudaError_t launch_transpose_tau(const double2* src, double2* dst, int nk, int ntau, int nao, bool reverse, cudaStream_t stream) {
  if (nk <= 0 || ntau <= 0) return cudaSuccess;
  transpose_tau_kernel<<<(unsigned)((long long)nk * ntau), 256, 0, stream>>>(src, dst, ntau, nao, reverse ? 1 : 0);
  return cudaGetLastError();
}

// Eq. 19a: P = [1 - P0]^{-1} P0 for one (q, Omega) per CTA at a time: Gauss-Jordan elimination with partial
// pivoting on the augmented matrix [1 - P0 | P0] kept in a per-CTA global scratch (L2-resident: 2.9 MB at naux = 300); the pivot
// row and the factor column of a step sit in shared memory.  2 n^3 complex multiply-adds per matrix: 0.2 % of one pair's
// contraction, so plain FP64 FMAs.
constexpr int DYS_NMAX = 512;
__global__ void __launch_bounds__(256) dyson_solve_kernel(double2* X, int nmat, int n, double2* work, int* fail_flag) {
  __shared__ double2 prow[2 * DYS_NMAX];
  __shared__ double2 fac[DYS_NMAX];
  __shared__ double red_v[256];
  __shared__ int red_i[256];
  const int tid = threadIdx.x, nt = blockDim.x, w2 = 2 * n;
  double2* M = work + (long long)blockIdx.x * n * w2;
  for (int mat = blockIdx.x; mat < nmat; mat += gridDim.x) {
    double2* A = X + (long long)mat * n * n;
    for (int e = tid; e < n * n; e += nt) {
      const int r = e / n, c = e - r * n;
      const double2 a = A[e];
      M[(long long)r * w2 + c] = make_double2((r == c ? 1.0 : 0.0) - a.x, -a.y);
      M[(long long)r * w2 + n + c] = a;
    }
    __syncthreads();
    for (int c = 0; c < n; ++c) {
      double best = -1.0; int bi = c;
      for (int r = c + tid; r < n; r += nt) {
        const double2 v = M[(long long)r * w2 + c];
        const double a2 = v.x * v.x + v.y * v.y;
        if (a2 > best) { best = a2; bi = r; }
      }
      red_v[tid] = best; red_i[tid] = bi;
      __syncthreads();
      for (int s_ = nt / 2; s_ > 0; s_ >>= 1) {
        if (tid < s_ && (red_v[tid + s_] > red_v[tid] || (red_v[tid + s_] == red_v[tid] && red_i[tid + s_] < red_i[tid]))) {
          red_v[tid] = red_v[tid + s_]; red_i[tid] = red_i[tid + s_];
        }
        __syncthreads();
      }
      const int piv = red_i[0];
      const double pv2 = red_v[0];
      if (pv2 <= 0.0 || !(pv2 == pv2)) { if (tid == 0) *fail_flag = 1; }           // singular 1 - P0 (or NaN input): flagged, result undefined
      const double2 pv = M[(long long)piv * w2 + c];
      __syncthreads();
      const double inv_r = pv.x / pv2, inv_i = -pv.y / pv2;                          // 1 / pivot
      // swap rows c <-> piv on columns c .. 2n-1 while scaling the pivot row; keep it in shared memory
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
    for (int e = tid; e < n * n; e += nt) A[e] = M[(long long)(e / n) * w2 + n + (e % n)];
    __syncthreads();
  }
}

cudaError_t launch_dyson_solve(double2* X, int nmat, int n, double2* work, int ncta, int* fail_flag, cudaStream_t stream) {
  if (nmat <= 0) return cudaSuccess;
  if (n > DYS_NMAX || ncta < 1) return cudaErrorInvalidValue;
  dyson_solve_kernel<<<(unsigned)std::min(ncta, nmat), 256, 0, stream>>>(X, nmat, n, work, fail_flag);
  return cudaGetLastError();
}

// Eq. 21b, first factor: rho_Q = scale * sum_k sum_{ab} gamma^k[a][b] V^{kk}[Q][b][a], one CTA per Q.  The thread
// index runs over (k, b, a) with a fastest, so V is read in contiguous runs; every thread sums its terms in a fixed order and the
// block reduction is a fixed tree: the result is bit-reproducible.  HBM-bound: V^{kk} is read once (nk naux nao^2 16 bytes).
__global__ void __launch_bounds__(256) hartree_rho_kernel(const double2* __restrict__ gamma, const double2* __restrict__ Vd, double2* rho,
                                                          int nk, int nao, int naux, double scale) {
  __shared__ double red_r[256], red_i[256];
  const int Q = blockIdx.x, tid = threadIdx.x, n2 = nao * nao;
  double sr = 0.0, si = 0.0;
  for (long long e = tid; e < (long long)nk * n2; e += blockDim.x) {
    const int k = (int)(e / n2), ba = (int)(e - (long long)k * n2);
    const int b = ba / nao, a = ba - b * nao;
    const double2 v = Vd[((long long)k * naux + Q) * n2 + ba];          // V^{kk}[Q][b][a]
    const double2 g = gamma[(long long)k * n2 + a * nao + b];           // gamma^k[a][b]
    sr += g.x * v.x - g.y * v.y;
    si += g.x * v.y + g.y * v.x;
  }
  red_r[tid] = sr; red_i[tid] = si;
  __syncthreads();
  for (int s_ = blockDim.x / 2; s_ > 0; s_ >>= 1) {
    if (tid < s_) { red_r[tid] += red_r[tid + s_]; red_i[tid] += red_i[tid + s_]; }
    __syncthreads();
  }
  if (tid == 0) rho[Q] = make_double2(scale * red_r[0], scale * red_i[0]);
}

// Eq. 21b, second factor: J^k[i][j] = sum_Q V^{kk}[Q][i][j] rho_Q, one thread per (k, i, j), Q ascending.  HBM-bound: the second
// read of V^{kk}.
__global__ void __launch_bounds__(256) hartree_j_kernel(const double2* __restrict__ Vd, const double2* __restrict__ rho, double2* J, int nk,
                                                        int nao, int naux) {
  const int n2 = nao * nao;
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (long long)nk * n2) return;
  const int k = (int)(e / n2), ij = (int)(e - (long long)k * n2);
  const double2* v = Vd + (long long)k * naux * n2 + ij;
  double sr = 0.0, si = 0.0;
  for (int Q = 0; Q < naux; ++Q) {
    const double2 x = v[(long long)Q * n2], r = rho[Q];
    sr += x.x * r.x - x.y * r.y;
    si += x.x * r.y + x.y * r.x;
  }
  J[e] = make_double2(sr, si);
}

cudaError_t launch_hartree(const double2* gamma, const double2* Vd, double2* rho, double2* J, int nk, int nao, int naux, cudaStream_t stream) {
  if (nk <= 0 || nao <= 0 || naux <= 0) return cudaSuccess;
  hartree_rho_kernel<<<(unsigned)naux, 256, 0, stream>>>(gamma, Vd, rho, nk, nao, naux, 1.0 / (double)nk);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const long long tot = (long long)nk * nao * nao;
  hartree_j_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, stream>>>(Vd, rho, J, nk, nao, naux);
  return cudaGetLastError();
}

// Allowed-block detection ("only non-zero blocks are considered"): max |.| of every candidate block (p, alpha, iota)
// of the block-basis tensors T3[pair][P][a][i] (Eq. 27).  One CTA per (pair, slab of auxiliary rows): a shared-memory table of the
// pair's candidates (non-negative doubles order like their bit patterns: integer atomicMax), flushed to global once.
__global__ void __launch_bounds__(256) block_maxabs_kernel(const double2* __restrict__ T3, const int* __restrict__ lab_aux, const int* __restrict__ lab_ao,
                                                           const int* __restrict__ pair_qkk, unsigned long long* out, int naux, int nao, int mb_ao,
                                                           int ncand, int rows_per_cta) {
  extern __shared__ unsigned long long cand[];
  const int pair = blockIdx.x, P0 = blockIdx.y * rows_per_cta, tid = threadIdx.x;
  for (int c = tid; c < ncand; c += blockDim.x) cand[c] = 0ULL;
  __syncthreads();
  const int q = pair_qkk[3 * pair], k2 = pair_qkk[3 * pair + 1], k1 = pair_qkk[3 * pair + 2];
  const int n2 = nao * nao;
  const int P1 = min(naux, P0 + rows_per_cta);
  const double2* T = T3 + (long long)pair * naux * n2;
  for (long long e = (long long)P0 * n2 + tid; e < (long long)P1 * n2; e += blockDim.x) {
    const int P = (int)(e / n2), ai = (int)(e - (long long)P * n2);
    const int a = ai / nao, i = ai - a * nao;
    const double2 v = T[e];
    const double m = sqrt(v.x * v.x + v.y * v.y);
    const int c = (lab_aux[q * naux + P] * mb_ao + lab_ao[k2 * nao + a]) * mb_ao + lab_ao[k1 * nao + i];
    atomicMax(&cand[c], (unsigned long long)__double_as_longlong(m));
  }
  __syncthreads();
  for (int c = tid; c < ncand; c += blockDim.x)
    if (cand[c]) atomicMax(&out[(long long)pair * ncand + c], cand[c]);
}

cudaError_t launch_block_maxabs(const double2* T3, const int* lab_aux, const int* lab_ao, const int* pair_qkk, double* out, int npairs, int naux,
                                int nao, int mb_aux, int mb_ao, cudaStream_t stream) {
  if (npairs <= 0) return cudaSuccess;
  const int ncand = mb_aux * mb_ao * mb_ao;
  if ((size_t)ncand * sizeof(unsigned long long) > 48 * 1024) return cudaErrorInvalidValue;
  const int rows_per_cta = 8;
  for (int p0 = 0; p0 < npairs; p0 += 65535) {                     // (pairs on grid.x would do; kept symmetric with the other launchers)
    const int np = std::min(65535, npairs - p0);
    dim3 grid((unsigned)np, (unsigned)((naux + rows_per_cta - 1) / rows_per_cta));
    block_maxabs_kernel<<<grid, 256, (size_t)ncand * sizeof(unsigned long long), stream>>>(T3 + (long long)p0 * naux * nao * nao, lab_aux, lab_ao,
                                                                                           pair_qkk + 3LL * p0, (unsigned long long*)out + (long long)p0 * ncand,
                                                                                           naux, nao, mb_ao, ncand, rows_per_cta);
  }
  return cudaGetLastError();
}

// P0 (Eq. 20): the pair tensors arrive as T[Q][x][y] (auxiliary index first, like every dense V of the interface); stages 1 and 2
// of Algorithm 3 want the auxiliary index LAST -- T'[x][y][Q] -- so that both the tile rows of X1 / X2 and the operand rows they are
// made from are contiguous in Q.  One tiled transpose [naux][nao^2] -> [nao^2][naux] per pair per push (read + write of V once).
__global__ void __launch_bounds__(256) aux_last_kernel(const double2* __restrict__ src, double2* __restrict__ dst, int naux, int n2) {
  __shared__ double2 tile[32][33];
  const long long base = (long long)blockIdx.z * naux * n2;
  const int x0 = blockIdx.x * 32, q0 = blockIdx.y * 32;            // x = (x, y) flattened, q = auxiliary index
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;          // 32 x 8 threads
  for (int j = ty; j < 32; j += 8) {
    const int q = q0 + j, x = x0 + tx;
    if (q < naux && x < n2) tile[j][tx] = src[base + (long long)q * n2 + x];
  }
  __syncthreads();
  for (int j = ty; j < 32; j += 8) {
    const int x = x0 + j, q = q0 + tx;
    if (q < naux && x < n2) dst[base + (long long)x * naux + q] = tile[tx][j];
  }
}

cudaError_t launch_aux_last(const double2* src, double2* dst, long long npairs, int naux, int n2, cudaStream_t stream) {
  for (long long p0 = 0; p0 < npairs; p0 += 65535) {
    const int np = (int)std::min<long long>(65535, npairs - p0);
    dim3 grid((unsigned)((n2 + 31) / 32), (unsigned)((naux + 31) / 32), (unsigned)np);
    aux_last_kernel<<<grid, 256, 0, stream>>>(src + p0 * (long long)naux * n2, dst + p0 * (long long)naux * n2, naux, n2);
  }
  return cudaGetLastError();
}

cudaError_t launch_reduce_parts(const RedGroupDev* groups, int ngroups, const double2* partial, double2* acc, int t0, cudaStream_t stream) {
  if (ngroups <= 0) return cudaSuccess;
  for (int g0 = 0; g0 < ngroups; g0 += 65535) {
    dim3 grid(8, (unsigned)std::min(65535, ngroups - g0));
    reduce_parts_kernel<<<grid, 256, 0, stream>>>(groups + g0, partial, acc, t0);
  }
  return cudaGetLastError();
}

cudaError_t launch_epilogue(const EpilogueParams& p, int ndesc, int num_sms, cudaStream_t stream) {
  if (ndesc <= 0) return cudaSuccess;
  dim3 grid((unsigned)(num_sms > 0 ? 4 : 1), (unsigned)ndesc);
  epilogue_kernel<<<grid, 256, 0, stream>>>(p);
  return cudaGetLastError();
}

cudaError_t launch_probe(int kind, int warps_per_block, int blocks, long long iters, double* sink, cudaStream_t stream,
                         double* flops_out) {
  constexpr int NACC = 16;
  if (kind == 0) {
    probe_dmma_kernel<NACC><<<blocks, warps_per_block * 32, 0, stream>>>(iters, sink);
    *flops_out = (double)blocks * warps_per_block * (double)iters * NACC * 512.0;       // 8*8*4*2 per DMMA
  } else if (kind == 1) {
    probe_dfma_kernel<NACC><<<blocks, warps_per_block * 32, 0, stream>>>(iters, sink);
    *flops_out = (double)blocks * warps_per_block * 32.0 * (double)iters * NACC * 2.0;
  } else if (kind == 3) {      // ONE dependent chain per warp: with 1 warp per sub-partition this is the DMMA latency
    probe_dmma_kernel<1><<<blocks, warps_per_block * 32, 0, stream>>>(iters * NACC, sink);
    *flops_out = (double)blocks * warps_per_block * (double)iters * NACC * 512.0;
  } else {
    probe_mixed_kernel<NACC><<<blocks, warps_per_block * 32, 0, stream>>>(iters, sink);
    *flops_out = (double)blocks * warps_per_block * (double)iters * NACC * (512.0 + 8 * 32 * 2.0);
  }
  return cudaGetLastError();
}
