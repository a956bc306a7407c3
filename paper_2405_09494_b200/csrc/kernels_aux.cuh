// Declarations of the helper kernels (unfold, epilogue, FP64 probes).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct UnfoldParams {
  const double2* src;       // [nsrc][ntau][n][n]   wedge data
  double2* dst;             // [ntarget][ntau][n][n]
  const int* tgt_src;       // [ntarget] wedge index of the star representative
  const int* tgt_op;        // [ntarget] operation alpha with alpha k_I = k'
  const double2* colphase;  // [ntarget][n]  exp(-2 pi i k' . s_atom(c))   (Eq. 3)
  const int* ell_cols;      // [nops][n][maxnz]  non-zeros of the real representation matrix
  const double* ell_vals;   // [nops][n][maxnz]
  const int* ell_cnt;       // [nops][n]
  int n, ntau, maxnz;
};

struct EpiDesc {
  long long off;     // first element of the batch
  long long stride;  // elements between consecutive matrices (tau)
  int n, count;      // n x n matrices, `count` of them
};

struct EpilogueParams {
  const double2* acc;
  double2* out;
  const EpiDesc* desc;  // device
  double scale;
  int hermitize;
};

struct RedGroupDev {      // = gwsig::RedGroup (plan.hpp)
  long long c_off, sts, part_off;
  int ni, M, nparts, pad_;
};
// acc[block] += sum over the block's partial tiles IN PART ORDER (deterministic stage 3)
cudaError_t launch_reduce_parts(const RedGroupDev* groups, int ngroups, const double2* partial, double2* acc, int t0, cudaStream_t stream);
// Eq. 19a per matrix: X <- [1 - X]^{-1} X in place, nmat matrices [n][n] back to back; work = per-CTA scratch [ncta][n][2n]
cudaError_t launch_block_maxabs(const double2* T3, const int* lab_aux, const int* lab_ao, const int* pair_qkk, double* out, int npairs, int naux,
                                int nao, int mb_aux, int mb_ao, cudaStream_t stream);
cudaError_t launch_aux_last(const double2* src, double2* dst, long long npairs, int naux, int n2, cudaStream_t stream);
cudaError_t launch_hartree(const double2* gamma, const double2* Vd, double2* rho, double2* J, int nk, int nao, int naux, cudaStream_t stream);
cudaError_t launch_dyson_solve(double2* X, int nmat, int n, double2* work, int ncta, int* fail_flag, cudaStream_t stream);
// dst[k][n] = src[k][ntau-1-n] for nk matrices-over-tau of `elems` complex numbers each (G(beta - tau) for Eq. 20)
cudaError_t launch_transpose_tau(const double2* src, double2* dst, int nk, int ntau, int nao, bool reverse, cudaStream_t stream);
cudaError_t launch_unfold_sparse(const UnfoldParams& p, int ntarget, cudaStream_t stream);
cudaError_t launch_epilogue(const EpilogueParams& p, int ndesc, int num_sms, cudaStream_t stream);
cudaError_t launch_probe(int kind, int warps_per_block, int blocks, long long iters, double* sink, cudaStream_t stream,
                         double* flops_out);
