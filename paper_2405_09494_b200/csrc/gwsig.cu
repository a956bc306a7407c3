// C-ABI of the gwsig library (include/gwsig.h): context, device buffers, launch orchestration.
// Order of work per evaluation:
//   sigma_begin : [a1] unfold G to the full zone (IBZ mode)            -> Gbz
//   sigma_push  : [a2] unfold W for the q of the pushed pairs (IBZ)    -> W ring
//                 per sub-batch of whole q's, per tau chunk:
//                 [a3] X^T = G^T conj(V2), [a4] Y^T = X^T W, [a5] Sigma_acc += Y V2   (grouped GEMM engine)
//   sigma_end   : [a6] Sigma = -(1/Nk) Sigma_acc (optional Hermitise)
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <tuple>
#include <vector>

#include "gwsig.h"
#include "kernels_aux.cuh"
#include "plan.hpp"
#include "zgemm_grouped.cuh"

using gwsig::cplx;
using gwsig::Plan;
using gwsig::StagePlan;

namespace {

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  cudaError_t ensure(size_t need) {
    if (need <= bytes) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr; bytes = 0;
    cudaError_t e = cudaMalloc(&p, need);
    if (e == cudaSuccess) bytes = need;
    return e;
  }
  void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
};

struct DevStage {
  DevBuf prob, seg, bucket, red;
  int nprob = 0, nred = 0;
  long long ntiles = 0, partial_elems = 0;
};
struct DevPlan { DevStage st[3]; };

}  // namespace

struct gwsig_ctx {
  Plan plan;
  int device = -1;
  bool cuda_ready = false;
  int num_sms = 0;
  std::string err;
  // options
  int engine = GWSIG_ENGINE_DMMA;
  int hermitize = 0;
  long long scratch_mib = 8192;
  long long v_ring_mib = 1024;
  int tau_chunk = 0;
  int bulk_copies = 0;
  // evaluation state
  bool in_eval = false;
  bool exchange = false;        // evaluation opened by exchange_begin: no W, stage 2 skipped (Eq. 21c)
  const double2* dG = nullptr;
  const double2* dW = nullptr;
  double2* dSigma = nullptr;
  cudaStream_t stream = nullptr;
  long long next_pair = 0;
  long long launches = 0;
  // device buffers
  DevBuf gbz, wring, xbuf, ybuf, sigacc, counters, epidesc, probe_sink;
  DevBuf oblk_ao, oblk_aux, unf_tmp, partial;
  DevBuf dys_flag;                               // N3: singular-matrix flag of the Eq. 19 solve
  DevBuf hart_rho;                               // N2: auxiliary density rho_Q of the Hartree term (Eq. 21b)
  DevBuf p0vt;                                   // N1: aux-last copy T'[x][y][Q] of the pushed pair tensors (stages 1, 2 of Algorithm 3)
  DevBuf u_ao_dev, u_aux_dev;                    // N4: the adapted bases on the device (set_blocks with U)
  DevBuf grev, p0acc, p0desc;                    // N1 (Eq. 20): G(beta - tau) on the full zone, the P0 accumulator, its epilogue descriptors
  bool in_p0 = false;
  double2* dP0 = nullptr;
  std::map<std::tuple<long long, long long, int>, std::unique_ptr<DevPlan>> p0_cache;    // partial: split-K partial tiles of deterministic stage 3
  DevBuf __unused_;             // Eq. 28: O_block tables and the scratch T of the two-step block unfold
  DevBuf h_g, h_w, h_sig, h_vslot[2];           // device side of sigma_eval_host
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_freed[2] = {nullptr, nullptr};
  DevBuf tgt_src, tgt_op, colphase_ao, ell_cols_ao, ell_vals_ao, ell_cnt_ao;     // unfold tables (ao)
  DevBuf wtgt_src, wtgt_op, colphase_aux, ell_cols_aux, ell_vals_aux, ell_cnt_aux;
  int maxnz_ao = 0, maxnz_aux = 0;
  bool tables_ready = false;
  int n_epidesc = 0;
  std::map<std::tuple<long long, long long, int, int>, std::unique_ptr<DevPlan>> plan_cache;
  int counter_slot = 0;
  static constexpr int kCounterSlots = 8192;
  // optional per-kernel device timing (option "timing"): event pairs on the launching stream
  int timing = 0;
  std::vector<cudaEvent_t> ev_pool;
  std::vector<std::pair<int, int>> ev_used;     // (kind, pool index of the start event; stop = +1)
  double kind_ms[GWSIG_NKINDS] = {0};
  long long kind_launches[GWSIG_NKINDS] = {0};
};

namespace {

int fail(gwsig_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
int cuda_fail(gwsig_ctx* c, cudaError_t e, const char* where) {
  return fail(c, GWSIG_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                                   \
  do {                                                             \
    cudaError_t e__ = (call);                                      \
    if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);     \
  } while (0)

int ensure_cuda(gwsig_ctx* ctx) {
  if (ctx->cuda_ready) return GWSIG_OK;
  if (ctx->device < 0) return fail(ctx, GWSIG_ERR_CUDA, "host-only context (device < 0): no CUDA device; there is no CPU fallback");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev <= ctx->device)
    return fail(ctx, GWSIG_ERR_CUDA, std::string("no usable CUDA device (there is no CPU fallback): ") + cudaGetErrorString(e));
  CU(cudaSetDevice(ctx->device));
  CU(cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, ctx->device));
  ctx->cuda_ready = true;
  return GWSIG_OK;
}

template <class T>
int upload(gwsig_ctx* ctx, DevBuf& b, const std::vector<T>& v) {
  size_t bytes = std::max<size_t>(v.size() * sizeof(T), 16);
  CU(b.ensure(bytes));
  if (!v.empty()) CU(cudaMemcpyAsync(b.p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, ctx->stream));
  // the host vector may be a temporary: make the copy complete before returning
  CU(cudaStreamSynchronize(ctx->stream));
  return GWSIG_OK;
}

// ELL form of the real representation matrices (non-zeros per row <= 2l+1)
void build_ell(const std::vector<double>& D, int nops, int n, std::vector<int>& cols, std::vector<double>& vals,
               std::vector<int>& cnt, int& maxnz) {
  maxnz = 1;
  cnt.assign((size_t)nops * n, 0);
  for (int g = 0; g < nops; ++g)
    for (int r = 0; r < n; ++r) {
      int c = 0;
      for (int j = 0; j < n; ++j)
        if (std::fabs(D[((size_t)g * n + r) * n + j]) > 1e-13) ++c;
      cnt[(size_t)g * n + r] = c;
      maxnz = std::max(maxnz, c);
    }
  cols.assign((size_t)nops * n * maxnz, 0);
  vals.assign((size_t)nops * n * maxnz, 0.0);
  for (int g = 0; g < nops; ++g)
    for (int r = 0; r < n; ++r) {
      int c = 0;
      for (int j = 0; j < n; ++j) {
        double v = D[((size_t)g * n + r) * n + j];
        if (std::fabs(v) > 1e-13) {
          cols[((size_t)g * n + r) * maxnz + c] = j;
          vals[((size_t)g * n + r) * maxnz + c] = v;
          ++c;
        }
      }
    }
}

// exp(-2 pi i k' . s_atom(c)(g)) for target k' reached with operation g   (Eq. 3)
void column_phases(const Plan& P, const std::vector<int>& targets, const std::vector<int>& atom_of, int n,
                   std::vector<double2>& out) {
  out.resize(targets.size() * (size_t)n);
  for (size_t t = 0; t < targets.size(); ++t) {
    int k = targets[t], g = P.op_of[k], nn[3];
    P.kcoords(k, nn);
    for (int c = 0; c < n; ++c) {
      const int* s = &P.shift[((size_t)g * P.natom + atom_of[c]) * 3];
      double ph = -2.0 * M_PI * ((double)nn[0] * s[0] / P.N[0] + (double)nn[1] * s[1] / P.N[1] + (double)nn[2] * s[2] / P.N[2]);
      out[t * n + c] = make_double2(std::cos(ph), std::sin(ph));
    }
  }
}

int prepare_tables(gwsig_ctx* ctx) {
  if (ctx->tables_ready) return GWSIG_OK;
  const Plan& P = ctx->plan;
  if (P.mode == GWSIG_IBZ) {
    std::vector<int> cols, cnt;
    std::vector<double> vals;
    build_ell(P.D_ao, P.nops, P.nao, cols, vals, cnt, ctx->maxnz_ao);
    int rc;
    if ((rc = upload(ctx, ctx->ell_cols_ao, cols))) return rc;
    if ((rc = upload(ctx, ctx->ell_vals_ao, vals))) return rc;
    if ((rc = upload(ctx, ctx->ell_cnt_ao, cnt))) return rc;
    build_ell(P.D_aux, P.nops, P.naux, cols, vals, cnt, ctx->maxnz_aux);
    if ((rc = upload(ctx, ctx->ell_cols_aux, cols))) return rc;
    if ((rc = upload(ctx, ctx->ell_vals_aux, vals))) return rc;
    if ((rc = upload(ctx, ctx->ell_cnt_aux, cnt))) return rc;
    std::vector<int> targets(P.nk), src(P.nk), op(P.nk);
    for (int k = 0; k < P.nk; ++k) { targets[k] = k; src[k] = P.ir_index[P.ir_of[k]]; op[k] = P.op_of[k]; }
    std::vector<double2> ph;
    column_phases(P, targets, P.ao_atom, P.nao, ph);
    if ((rc = upload(ctx, ctx->colphase_ao, ph))) return rc;
    column_phases(P, targets, P.aux_atom, P.naux, ph);
    if ((rc = upload(ctx, ctx->colphase_aux, ph))) return rc;
    if ((rc = upload(ctx, ctx->tgt_src, src))) return rc;
    if ((rc = upload(ctx, ctx->tgt_op, op))) return rc;
  }
  if (P.mode == GWSIG_IBZ_BLOCK && P.have_U) {
    int rc;
    if ((rc = upload(ctx, ctx->u_ao_dev, P.U_ao))) return rc;
    if ((rc = upload(ctx, ctx->u_aux_dev, P.U_aux))) return rc;
  }
  if (P.mode == GWSIG_IBZ_BLOCK && P.general_gauge) {
    int rc;
    if ((rc = upload(ctx, ctx->oblk_ao, P.oblk_ao))) return rc;
    if ((rc = upload(ctx, ctx->oblk_aux, P.oblk_aux))) return rc;
  }
  // epilogue descriptors: one batch of ntau square matrices per (output k, block)
  std::vector<EpiDesc> ed;
  for (int i = 0; i < P.nk1; ++i) {
    const std::vector<int>& off = P.ao_off[P.out_list[i]];
    long long stride = P.mode == GWSIG_IBZ_BLOCK ? gwsig::sumsq(off) : (long long)P.nao * P.nao;
    long long o = P.sig_off[i];
    for (size_t b = 0; b + 1 < off.size(); ++b) {
      int n = off[b + 1] - off[b];
      ed.push_back(EpiDesc{o, stride, n, P.ntau});
      o += (long long)n * n;
    }
  }
  ctx->n_epidesc = (int)ed.size();
  int rc = upload(ctx, ctx->epidesc, ed);
  if (rc) return rc;
  ctx->tables_ready = true;
  return GWSIG_OK;
}

int get_dev_plan(gwsig_ctx* ctx, long long p0, long long np, int nt, int q_first, DevPlan** out) {
  auto key = std::make_tuple(p0, np, nt, q_first);
  auto it = ctx->plan_cache.find(key);
  if (it != ctx->plan_cache.end()) { *out = it->second.get(); return GWSIG_OK; }
  if (ctx->plan_cache.size() >= 256) {          // callers that push ever-changing ranges must not grow the cache without bound
    CU(cudaStreamSynchronize(ctx->stream));      // (a cached plan may still be read by kernels in flight)
    for (auto& kv : ctx->plan_cache)
      for (int s = 0; s < 3; ++s) { kv.second->st[s].prob.release(); kv.second->st[s].seg.release(); kv.second->st[s].bucket.release(); kv.second->st[s].red.release(); }
    ctx->plan_cache.clear();
  }
  std::unique_ptr<DevPlan> dp(new DevPlan());
  for (int s = 0; s < 3; ++s) {
    StagePlan sp;
    int rc = ctx->plan.build_stage(p0, np, nt, s + 1, q_first, sp, ctx->num_sms > 0 ? ctx->num_sms : 148);
    if (rc) return fail(ctx, rc, "internal: build_stage failed");
    DevStage& d = dp->st[s];
    d.nprob = (int)sp.prob.size();
    d.ntiles = sp.ntiles;
    if ((rc = upload(ctx, d.prob, sp.prob))) return rc;
    if ((rc = upload(ctx, d.seg, sp.seg))) return rc;
    if ((rc = upload(ctx, d.bucket, sp.bucket))) return rc;
    d.nred = (int)sp.red.size();
    d.partial_elems = sp.partial_elems;
    if (d.nred && (rc = upload(ctx, d.red, sp.red))) return rc;
  }
  *out = dp.get();
  ctx->plan_cache[key] = std::move(dp);
  return GWSIG_OK;
}

int tic(gwsig_ctx* ctx, int kind) {
  if (!ctx->timing) return GWSIG_OK;
  size_t need = 2 * (ctx->ev_used.size() + 1);
  while (ctx->ev_pool.size() < need) {
    cudaEvent_t e;
    CU(cudaEventCreate(&e));
    ctx->ev_pool.push_back(e);
  }
  int idx = (int)(2 * ctx->ev_used.size());
  ctx->ev_used.push_back(std::make_pair(kind, idx));
  CU(cudaEventRecord(ctx->ev_pool[idx], ctx->stream));
  return GWSIG_OK;
}
int toc(gwsig_ctx* ctx) {
  if (!ctx->timing) return GWSIG_OK;
  CU(cudaEventRecord(ctx->ev_pool[ctx->ev_used.back().second + 1], ctx->stream));
  return GWSIG_OK;
}

// which kernel runs launch kind st (0 = Eq. 28 unfold, 1..3 = contraction stage) under engine option e:
// GWSIG_ENGINE_DMMA (default) = the 3M kernel where it is the faster one on B200 (stages 1 and 2: 86 % of the flops) and the
// 4-product kernel for stage 3 (two-level k index, narrow N, atomic accumulation) and the unfold (measured)
int stage_engine(int e, int st) {
  if (e == GWSIG_ENGINE_DMMA) return (st == 1 || st == 2) ? GWSIG_ENGINE_DMMA_3M : GWSIG_ENGINE_DMMA_4M;
  return e;
}
void set_tile_heights(gwsig_ctx* ctx) {
  for (int st = 0; st < 4; ++st) ctx->plan.tile_m[st] = stage_engine(ctx->engine, st) == GWSIG_ENGINE_DMMA_3M ? ZG_BM3 : ZG_BM;
}

int run_stage(gwsig_ctx* ctx, int kind, const DevStage& d, const double2* A, const double2* B, double2* C, int t0) {
  if (d.ntiles <= 0) return GWSIG_OK;
  if (ctx->counter_slot >= gwsig_ctx::kCounterSlots) {
    CU(cudaMemsetAsync(ctx->counters.p, 0, gwsig_ctx::kCounterSlots * sizeof(unsigned long long), ctx->stream));
    ctx->counter_slot = 0;
  }
  ZgParams zp;
  zp.A = A; zp.B = B; zp.C = C;
  zp.prob = (const gwsig_problem*)d.prob.p;
  zp.seg = (const gwsig_seg*)d.seg.p;
  zp.bucket = (const int*)d.bucket.p;
  zp.nprob = d.nprob;
  zp.total_tiles = d.ntiles;
  zp.t0 = t0;
  zp.use_bulk = ctx->bulk_copies;
  const int st = kind == GWSIG_KIND_STAGE1 ? 1 : kind == GWSIG_KIND_STAGE2 ? 2 : kind == GWSIG_KIND_STAGE3 ? 3 : 0;
  zp.bm = ctx->plan.tile_m[st];
  zp.counter = (unsigned long long*)ctx->counters.p + ctx->counter_slot++;
  int rc = tic(ctx, kind);
  if (rc) return rc;
  CU(zg_launch(stage_engine(ctx->engine, st), zp, ctx->num_sms, ctx->stream));
  if ((rc = toc(ctx))) return rc;
  ctx->launches++;
  return GWSIG_OK;
}

// Eq. 28: X_blk^{k'}(tau) = O_block X_blk^{k_I}(tau) O_block^dagger for mesh points [k_first, k_first + k_count),
// two launches of the grouped engine (step 1 into the scratch T, step 2 into dst).  aux: W with the auxiliary blocks.
int run_block_unfold(gwsig_ctx* ctx, bool aux, int k_first, int k_count, const double2* src, double2* dst) {
  const Plan& P = ctx->plan;
  const long long elems = P.unfolded_elems(aux, k_first, k_count);
  CU(ctx->unf_tmp.ensure(std::max<size_t>((size_t)elems * sizeof(double2), 16)));
  const double2* O = (const double2*)(aux ? ctx->oblk_aux.p : ctx->oblk_ao.p);
  for (int step = 1; step <= 2; ++step) {
    StagePlan sp;
    int rc = P.build_unfold(aux, k_first, k_count, step, sp);
    if (rc) return fail(ctx, rc, "internal: build_unfold failed");
    DevStage d;
    d.nprob = (int)sp.prob.size();
    d.ntiles = sp.ntiles;
    if ((rc = upload(ctx, d.prob, sp.prob))) return rc;
    if ((rc = upload(ctx, d.seg, sp.seg))) return rc;
    if ((rc = upload(ctx, d.bucket, sp.bucket))) return rc;
    rc = run_stage(ctx, aux ? GWSIG_KIND_UNFOLD_W : GWSIG_KIND_UNFOLD_G, d, step == 1 ? src : (const double2*)ctx->unf_tmp.p, O,
                   step == 1 ? (double2*)ctx->unf_tmp.p : dst, 0);
    // the descriptor tables are read by the kernel just enqueued: free them only after it has run
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    d.prob.release(); d.seg.release(); d.bucket.release();
    if (rc) return rc;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "block unfold");
  }
  return GWSIG_OK;
}

}  // namespace

static void invalidate(gwsig_ctx* ctx) {
  ctx->tables_ready = false;
  for (auto& kv : ctx->plan_cache)
    for (int s = 0; s < 3; ++s) { kv.second->st[s].prob.release(); kv.second->st[s].seg.release(); kv.second->st[s].bucket.release(); kv.second->st[s].red.release(); }
  ctx->plan_cache.clear();
  for (auto& kv : ctx->p0_cache)
    for (int s = 0; s < 3; ++s) { kv.second->st[s].prob.release(); kv.second->st[s].seg.release(); kv.second->st[s].bucket.release(); }
  ctx->p0_cache.clear();
  ctx->in_eval = false;
  ctx->in_p0 = false;
}

// =============================================================================================
extern "C" {

int gwsig_create(gwsig_ctx** out, int device) {
  if (!out) return GWSIG_ERR_ARG;
  *out = new gwsig_ctx();
  (*out)->device = device;
  set_tile_heights(*out);
  return GWSIG_OK;
}

int gwsig_destroy(gwsig_ctx* ctx) {
  if (!ctx) return GWSIG_ERR_ARG;
  if (ctx->cuda_ready) {
    cudaSetDevice(ctx->device);
    DevBuf* bufs[] = {&ctx->gbz, &ctx->wring, &ctx->xbuf, &ctx->ybuf, &ctx->sigacc, &ctx->counters, &ctx->epidesc,
                      &ctx->probe_sink, &ctx->oblk_ao, &ctx->oblk_aux, &ctx->unf_tmp, &ctx->partial, &ctx->grev, &ctx->p0acc, &ctx->p0desc, &ctx->u_ao_dev, &ctx->u_aux_dev, &ctx->dys_flag, &ctx->hart_rho, &ctx->p0vt, &ctx->tgt_src, &ctx->tgt_op, &ctx->colphase_ao, &ctx->ell_cols_ao,
                      &ctx->ell_vals_ao, &ctx->ell_cnt_ao, &ctx->wtgt_src, &ctx->wtgt_op, &ctx->colphase_aux,
                      &ctx->ell_cols_aux, &ctx->ell_vals_aux, &ctx->ell_cnt_aux, &ctx->h_g, &ctx->h_w, &ctx->h_sig,
                      &ctx->h_vslot[0], &ctx->h_vslot[1]};
    for (DevBuf* b : bufs) b->release();
    for (int i = 0; i < 2; ++i) {
      if (ctx->ev_copied[i]) cudaEventDestroy(ctx->ev_copied[i]);
      if (ctx->ev_freed[i]) cudaEventDestroy(ctx->ev_freed[i]);
    }
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    for (auto& kv : ctx->plan_cache)
      for (int s = 0; s < 3; ++s) { kv.second->st[s].prob.release(); kv.second->st[s].seg.release(); kv.second->st[s].bucket.release(); kv.second->st[s].red.release(); }
  }
  delete ctx;
  return GWSIG_OK;
}

const char* gwsig_last_error(const gwsig_ctx* ctx) { return ctx ? ctx->err.c_str() : "NULL context"; }


int gwsig_set_lattice(gwsig_ctx* ctx, const double a[9], const int mesh[3], int nao, int naux, int ntau, double beta) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_lattice(a, mesh, nao, naux, ntau, beta);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_set_atoms(gwsig_ctx* ctx, int natom, const double* pos, const int* ao_atom, const int* aux_atom) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_atoms(natom, pos, ao_atom, aux_atom);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_set_symmetry(gwsig_ctx* ctx, int nops, const int* rot, const double* trans, const double* D_ao,
                       const double* D_aux, const int* shift, int mode) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_symmetry(nops, rot, trans, D_ao, D_aux, shift, mode);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_set_blocks(gwsig_ctx* ctx, const int* nblk_ao, const int* ao_block_off, const int* nblk_aux,
                     const int* aux_block_off, const double* U_ao, const double* U_aux) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_blocks(nblk_ao, ao_block_off, nblk_aux, aux_block_off, U_ao, U_aux);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_set_output_points(gwsig_ctx* ctx, int n, const int* k_list) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_output_points(n, k_list);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_set_triples(gwsig_ctx* ctx, int64_t npairs, const int64_t* triple_ptr, const int32_t* triples) {
  if (!ctx) return GWSIG_ERR_ARG;
  invalidate(ctx);
  int rc = ctx->plan.set_triples(npairs, triple_ptr, triples);
  return rc ? fail(ctx, rc, ctx->plan.err) : rc;
}

int gwsig_get_ibz(gwsig_ctx* ctx, int* nik, int* ir_list, int* ir_of, int* op_of) {
  if (!ctx) return GWSIG_ERR_ARG;
  const Plan& P = ctx->plan;
  if (!P.have_sym) return fail(ctx, GWSIG_ERR_ARG, "get_ibz: call set_symmetry first");
  if (nik) *nik = (int)P.ir_list.size();
  if (ir_list) std::copy(P.ir_list.begin(), P.ir_list.end(), ir_list);
  if (ir_of) std::copy(P.ir_of.begin(), P.ir_of.end(), ir_of);
  if (op_of) std::copy(P.op_of.begin(), P.op_of.end(), op_of);
  return GWSIG_OK;
}

int gwsig_pair_count(gwsig_ctx* ctx, int64_t* npairs, int* nk1) {
  if (!ctx) return GWSIG_ERR_ARG;
  if (!ctx->plan.have_sym) return fail(ctx, GWSIG_ERR_ARG, "pair_count: call set_symmetry first");
  if (npairs) *npairs = ctx->plan.npairs;
  if (nk1) *nk1 = ctx->plan.nk1;
  return GWSIG_OK;
}

int gwsig_pair_info(gwsig_ctx* ctx, int64_t pair, int* k1, int* k2, int* q, int64_t* v_offset, int64_t* v_elems) {
  if (!ctx) return GWSIG_ERR_ARG;
  const Plan& P = ctx->plan;
  if (!P.have_sym || pair < 0 || pair >= P.npairs) return fail(ctx, GWSIG_ERR_ARG, "pair_info: bad pair index or no symmetry set");
  int a, b, c, d;
  P.pair(pair, a, b, c, d);
  if (k1) *k1 = a;
  if (k2) *k2 = b;
  if (q) *q = c;
  if (v_offset || v_elems) {
    if (P.v_off.empty()) return fail(ctx, GWSIG_ERR_ARG, "pair_info: V layout needs set_triples in IBZ_BLOCK mode");
    if (v_offset) *v_offset = P.v_off[pair];
    if (v_elems) *v_elems = P.v_off[pair + 1] - P.v_off[pair];
  }
  return GWSIG_OK;
}

int gwsig_buffer_sizes(gwsig_ctx* ctx, int64_t* g_elems, int64_t* w_elems, int64_t* sigma_elems, int64_t* v_elems) {
  if (!ctx) return GWSIG_ERR_ARG;
  const Plan& P = ctx->plan;
  if (!P.have_sym) return fail(ctx, GWSIG_ERR_ARG, "buffer_sizes: call set_symmetry first");
  if (g_elems) *g_elems = P.g_elems;
  if (w_elems) *w_elems = P.w_elems;
  if (sigma_elems) *sigma_elems = P.sig_elems;
  if (v_elems) *v_elems = P.v_off.empty() ? -1 : P.v_off.back();
  return GWSIG_OK;
}

int gwsig_set_option(gwsig_ctx* ctx, const char* key, int64_t value) {
  if (!ctx || !key) return GWSIG_ERR_ARG;
  std::string k(key);
  if (k == "engine") {
    if (value != GWSIG_ENGINE_DMMA && value != GWSIG_ENGINE_REFERENCE && value != GWSIG_ENGINE_DMMA_4M && value != GWSIG_ENGINE_DMMA_3M) return fail(ctx, GWSIG_ERR_ARG, "set_option: bad engine");
    if (ctx->engine != (int)value) invalidate(ctx);       // the tile height is part of the plan
    ctx->engine = (int)value;
    set_tile_heights(ctx);
  } else if (k == "hermitize") ctx->hermitize = value != 0;
  else if (k == "scratch_mib") { if (value < 1) return fail(ctx, GWSIG_ERR_ARG, "set_option: scratch_mib < 1"); ctx->scratch_mib = value; }
  else if (k == "v_ring_mib") { if (value < 1) return fail(ctx, GWSIG_ERR_ARG, "set_option: v_ring_mib < 1"); ctx->v_ring_mib = value; }
  else if (k == "timing") ctx->timing = value != 0;
  else if (k == "bulk_copies") ctx->bulk_copies = value != 0;
  else if (k == "deterministic") { invalidate(ctx); ctx->plan.deterministic = value != 0; }
  else if (k == "tau_chunk") { if (value < 0) return fail(ctx, GWSIG_ERR_ARG, "set_option: tau_chunk < 0"); ctx->tau_chunk = (int)value; }
  else return fail(ctx, GWSIG_ERR_ARG, "set_option: unknown key " + k);
  return GWSIG_OK;
}

int gwsig_flop_counts(gwsig_ctx* ctx, double* full_bz_equiv, double* executed) {
  if (!ctx) return GWSIG_ERR_ARG;
  if (!ctx->plan.have_sym) return fail(ctx, GWSIG_ERR_ARG, "flop_counts: call set_symmetry first");
  double f, e;
  ctx->plan.flop_counts(f, e);
  if (full_bz_equiv) *full_bz_equiv = f;
  if (executed) *executed = e;
  return GWSIG_OK;
}

int gwsig_last_launch_count(gwsig_ctx* ctx, int64_t* launches) {
  if (!ctx || !launches) return GWSIG_ERR_ARG;
  *launches = ctx->launches;
  return GWSIG_OK;
}

int gwsig_kernel_times(gwsig_ctx* ctx, double* ms, int64_t* launches) {
  if (!ctx || !ms || !launches) return GWSIG_ERR_ARG;
  if (!ctx->timing) return fail(ctx, GWSIG_ERR_ARG, "kernel_times: set option timing = 1 before sigma_begin");
  for (int i = 0; i < GWSIG_NKINDS; ++i) { ms[i] = 0; launches[i] = 0; }
  if (!ctx->ev_used.empty()) {
    CU(cudaEventSynchronize(ctx->ev_pool[ctx->ev_used.back().second + 1]));
    for (auto& u : ctx->ev_used) {
      float t = 0;
      CU(cudaEventElapsedTime(&t, ctx->ev_pool[u.second], ctx->ev_pool[u.second + 1]));
      ms[u.first] += t;
      launches[u.first] += 1;
    }
  }
  return GWSIG_OK;
}

int gwsig_plan_counts(gwsig_ctx* ctx, int64_t p0, int64_t np, int nt, int stage, int64_t* nproblems, int64_t* nsegs,
                      int64_t* ntiles) {
  if (!ctx) return GWSIG_ERR_ARG;
  const Plan& P = ctx->plan;
  if (!P.have_sym || (P.v_off.empty() && stage < 30)) return fail(ctx, GWSIG_ERR_ARG, "plan_counts: plan incomplete");
  StagePlan sp;
  int rc = stage == 51 ? P.build_gridtransform(P.nk1, (int)np, nt, sp)                          // 51: grid transform, np = n_in, nt = n_out
         : stage >= 40 ? P.build_vtransform(p0, np, stage - 40, sp)                             // 41, 42, 43: Eq. 27 steps
         : stage >= 30 ? P.build_p0_stage(p0, np, nt, stage - 30, sp)                           // 31, 32, 33: P0 stages (Eq. 20)
         : stage >= 10 ? P.build_unfold(stage / 10 == 2, (int)p0, (int)np, stage % 10, sp)      // 11, 12: G unfold steps; 21, 22: W
                       : P.build_stage(p0, np, nt, stage, (int)(p0 / P.nk1), sp);
  if (rc) return fail(ctx, rc, "plan_counts: bad range / stage");
  if (nproblems) *nproblems = (int64_t)sp.prob.size();
  if (nsegs) *nsegs = (int64_t)sp.seg.size();
  if (ntiles) *ntiles = sp.ntiles;
  return GWSIG_OK;
}

int gwsig_plan_get(gwsig_ctx* ctx, int64_t p0, int64_t np, int nt, int stage, void* problems_out, void* segs_out) {
  if (!ctx || !problems_out || !segs_out) return GWSIG_ERR_ARG;
  const Plan& P = ctx->plan;
  if (!P.have_sym || (P.v_off.empty() && stage < 30)) return fail(ctx, GWSIG_ERR_ARG, "plan_get: plan incomplete");
  StagePlan sp;
  int rc = stage == 51 ? P.build_gridtransform(P.nk1, (int)np, nt, sp)                          // 51: grid transform, np = n_in, nt = n_out
         : stage >= 40 ? P.build_vtransform(p0, np, stage - 40, sp)                             // 41, 42, 43: Eq. 27 steps
         : stage >= 30 ? P.build_p0_stage(p0, np, nt, stage - 30, sp)                           // 31, 32, 33: P0 stages (Eq. 20)
         : stage >= 10 ? P.build_unfold(stage / 10 == 2, (int)p0, (int)np, stage % 10, sp)      // 11, 12: G unfold steps; 21, 22: W
                       : P.build_stage(p0, np, nt, stage, (int)(p0 / P.nk1), sp);
  if (rc) return fail(ctx, rc, "plan_get: bad range / stage");
  std::memcpy(problems_out, sp.prob.data(), sp.prob.size() * sizeof(gwsig_problem));
  std::memcpy(segs_out, sp.seg.data(), sp.seg.size() * sizeof(gwsig_seg));
  return GWSIG_OK;
}

// ---------------------------------------------------------------------------------------------
int gwsig_sigma_begin(gwsig_ctx* ctx, const void* dG, const void* dW, void* dSigma, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!P.have_sym) return fail(ctx, GWSIG_ERR_ARG, "sigma_begin: call set_symmetry first");
  if (P.mode == GWSIG_IBZ_BLOCK && (!P.have_blocks || !P.have_triples))
    return fail(ctx, GWSIG_ERR_ARG, "sigma_begin: IBZ_BLOCK mode needs set_blocks and set_triples");
  if (!dG || (!dW && !ctx->exchange) || !dSigma) return fail(ctx, GWSIG_ERR_ARG, "sigma_begin: NULL device pointer");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  ctx->stream = (cudaStream_t)stream;
  ctx->dG = (const double2*)dG;
  ctx->dW = (const double2*)dW;
  ctx->dSigma = (double2*)dSigma;
  if ((rc = prepare_tables(ctx))) return rc;
  CU(ctx->sigacc.ensure(std::max<size_t>(P.sig_elems * sizeof(double2), 16)));
  CU(cudaMemsetAsync(ctx->sigacc.p, 0, P.sig_elems * sizeof(double2), ctx->stream));
  CU(ctx->counters.ensure(gwsig_ctx::kCounterSlots * sizeof(unsigned long long)));
  CU(cudaMemsetAsync(ctx->counters.p, 0, gwsig_ctx::kCounterSlots * sizeof(unsigned long long), ctx->stream));
  ctx->counter_slot = 0;
  ctx->launches = 0;
  ctx->ev_used.clear();
  if (P.mode == GWSIG_IBZ) {
    // [a1] G(k') = O G(k_I) O^dagger for every mesh point (Eq. 22; Algorithm 2 step 2)
    CU(ctx->gbz.ensure((size_t)P.nk * P.ntau * P.nao * P.nao * sizeof(double2)));
    UnfoldParams up;
    up.src = ctx->dG; up.dst = (double2*)ctx->gbz.p;
    up.tgt_src = (const int*)ctx->tgt_src.p; up.tgt_op = (const int*)ctx->tgt_op.p;
    up.colphase = (const double2*)ctx->colphase_ao.p;
    up.ell_cols = (const int*)ctx->ell_cols_ao.p; up.ell_vals = (const double*)ctx->ell_vals_ao.p;
    up.ell_cnt = (const int*)ctx->ell_cnt_ao.p;
    up.n = P.nao; up.ntau = P.ntau; up.maxnz = ctx->maxnz_ao;
    if ((rc = tic(ctx, GWSIG_KIND_UNFOLD_G))) return rc;
    CU(launch_unfold_sparse(up, P.nk, ctx->stream));
    if ((rc = toc(ctx))) return rc;
    ctx->launches++;
  }
  if (P.mode == GWSIG_IBZ_BLOCK && P.general_gauge) {
    // [a1] block basis, explicit gauge: G_blk(k') = O_block G_blk(k_I) O_block^dagger for every mesh point (Eq. 28)
    CU(ctx->gbz.ensure(std::max<size_t>((size_t)P.gu_off[P.nk] * sizeof(double2), 16)));
    if ((rc = run_block_unfold(ctx, false, 0, P.nk, ctx->dG, (double2*)ctx->gbz.p))) return rc;
  }
  ctx->next_pair = 0;
  ctx->in_eval = true;
  return GWSIG_OK;
}

int gwsig_sigma_push_pairs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!ctx->in_eval) return fail(ctx, GWSIG_ERR_ORDER, "sigma_push_pairs: call sigma_begin first");
  if (np < 1 || p0 != ctx->next_pair || p0 + np > P.npairs)
    return fail(ctx, GWSIG_ERR_ORDER, "sigma_push_pairs: ranges must be pushed in increasing order without gaps");
  if (!dV) return fail(ctx, GWSIG_ERR_ARG, "sigma_push_pairs: NULL device pointer");
  CU(cudaSetDevice(ctx->device));
  const double2* Vbase = (const double2*)dV;
  const int nk1 = P.nk1;

  const double2* Wsrc = P.mode == GWSIG_IBZ ? nullptr : ctx->dW;     // IBZ: the ring, filled per sub-batch below
  const bool blk_unfold = P.mode == GWSIG_IBZ_BLOCK && P.general_gauge;
  const double2* Gsrc = (P.mode == GWSIG_IBZ || blk_unfold) ? (const double2*)ctx->gbz.p : ctx->dG;

  // sub-batches of pairs (whole q's where possible) and tau chunks sized to the scratch budget
  // X + Y scratch: the option, but never more than 40 % of what the device has free (+ what the scratch already holds)
  size_t free_b = 0, total_b = 0;
  CU(cudaMemGetInfo(&free_b, &total_b));
  const double avail = 0.4 * ((double)free_b + (double)ctx->xbuf.bytes + (double)ctx->ybuf.bytes);
  const double budget = std::min((double)ctx->scratch_mib * 1048576.0, std::max(avail, 64.0 * 1048576.0)) / (2.0 * sizeof(double2));   // elements of X (= of Y)
  long long s0 = p0;
  while (s0 < p0 + np) {
    // grow the sub-batch by whole q's while X for all tau still fits
    long long s1 = std::min<long long>(p0 + np, (s0 / nk1 + 1) * nk1);
    while (s1 < p0 + np) {
      long long s2 = std::min<long long>(p0 + np, s1 + nk1);
      if ((double)(P.v_off[s2] - P.v_off[s0]) * P.ntau > budget) break;
      s1 = s2;
    }
    const long long ns = s1 - s0;
    const double per_tau = (double)(P.v_off[s1] - P.v_off[s0]);
    int nt_max = ctx->tau_chunk > 0 ? ctx->tau_chunk : (int)std::max(1.0, std::floor(budget / std::max(per_tau, 1.0)));
    nt_max = std::min(nt_max, P.ntau);
    const int nchunks = (P.ntau + nt_max - 1) / nt_max;
    const int nt = (P.ntau + nchunks - 1) / nchunks;
    const size_t xbytes = (size_t)std::max(per_tau * nt, 1.0) * sizeof(double2);
    CU(ctx->xbuf.ensure(xbytes));
    if (!ctx->exchange) CU(ctx->ybuf.ensure(xbytes));
    const double2* Vsub = Vbase + (P.v_off[s0] - P.v_off[p0]);
    const int q_sub = (int)(s0 / nk1);                 // first q of this sub-batch = first q held by the W ring
    if (ctx->exchange) {
      // Eq. 21c: W -> delta, nothing to unfold
    } else if (P.mode == GWSIG_IBZ) {
      // [a2] unfold W for the q of this sub-batch only (Eq. 25; Algorithm 4 line 6): the ring holds a few
      // q, never the whole zone (100 GB at cfg5)
      const int nq = (int)((s1 - 1) / nk1) - q_sub + 1;
      CU(ctx->wring.ensure((size_t)nq * P.ntau * P.naux * P.naux * sizeof(double2)));
      UnfoldParams up;
      up.src = ctx->dW; up.dst = (double2*)ctx->wring.p;
      up.tgt_src = (const int*)ctx->tgt_src.p + q_sub; up.tgt_op = (const int*)ctx->tgt_op.p + q_sub;
      up.colphase = (const double2*)ctx->colphase_aux.p + (size_t)q_sub * P.naux;
      up.ell_cols = (const int*)ctx->ell_cols_aux.p; up.ell_vals = (const double*)ctx->ell_vals_aux.p;
      up.ell_cnt = (const int*)ctx->ell_cnt_aux.p;
      up.n = P.naux; up.ntau = P.ntau; up.maxnz = ctx->maxnz_aux;
      int rc = tic(ctx, GWSIG_KIND_UNFOLD_W);
      if (rc) return rc;
      CU(launch_unfold_sparse(up, nq, ctx->stream));
      if ((rc = toc(ctx))) return rc;
      ctx->launches++;
      Wsrc = (const double2*)ctx->wring.p;
    } else if (blk_unfold) {
      // [a2] block basis, explicit gauge: W_blk(q) = O_block W_blk(q_I) O_block^dagger for the q of this sub-batch (Eq. 28 / 25)
      const int nq = (int)((s1 - 1) / nk1) - q_sub + 1;
      CU(ctx->wring.ensure(std::max<size_t>((size_t)P.unfolded_elems(true, q_sub, nq) * sizeof(double2), 16)));
      int rc = run_block_unfold(ctx, true, q_sub, nq, ctx->dW, (double2*)ctx->wring.p);
      if (rc) return rc;
      Wsrc = (const double2*)ctx->wring.p;
    }
    for (int t0 = 0; t0 < P.ntau; t0 += nt) {
      const int ntc = std::min(nt, P.ntau - t0);
      DevPlan* dp = nullptr;
      int rc = get_dev_plan(ctx, s0, ns, ntc, q_sub, &dp);
      if (rc) return rc;
      if ((rc = run_stage(ctx, GWSIG_KIND_STAGE1, dp->st[0], Gsrc, Vsub, (double2*)ctx->xbuf.p, t0))) return rc;                     // [a3]
      if (!ctx->exchange &&
          (rc = run_stage(ctx, GWSIG_KIND_STAGE2, dp->st[1], (const double2*)ctx->xbuf.p, Wsrc, (double2*)ctx->ybuf.p, t0))) return rc;  // [a4]
      const double2* Ysrc = (const double2*)(ctx->exchange ? ctx->xbuf.p : ctx->ybuf.p);     // Eq. 21c: Y = X (W = delta)
      if (dp->st[2].nred) {
        // deterministic accumulation: parts write private tiles, then one ordered reduction into the accumulator
        CU(ctx->partial.ensure(std::max<size_t>((size_t)dp->st[2].partial_elems * sizeof(double2), 16)));
        if ((rc = run_stage(ctx, GWSIG_KIND_STAGE3, dp->st[2], Ysrc, Vsub, (double2*)ctx->partial.p, t0))) return rc;
        CU(launch_reduce_parts((const RedGroupDev*)dp->st[2].red.p, dp->st[2].nred, (const double2*)ctx->partial.p, (double2*)ctx->sigacc.p, t0,
                               ctx->stream));
        ctx->launches++;
      } else if ((rc = run_stage(ctx, GWSIG_KIND_STAGE3, dp->st[2], Ysrc, Vsub, (double2*)ctx->sigacc.p, t0))) return rc; // [a5]
    }
    s0 = s1;
  }
  ctx->next_pair = p0 + np;
  return GWSIG_OK;
}

int gwsig_sigma_end(gwsig_ctx* ctx) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!ctx->in_eval) return fail(ctx, GWSIG_ERR_ORDER, "sigma_end: call sigma_begin first");
  if (ctx->next_pair != P.npairs) return fail(ctx, GWSIG_ERR_ORDER, "sigma_end: not all pairs were pushed");
  CU(cudaSetDevice(ctx->device));
  // [a6] Sigma = -(1/Nk) sum_q Sigma^{k,q}   (Eq. 16 prefactor)
  EpilogueParams ep;
  ep.acc = (const double2*)ctx->sigacc.p;
  ep.out = ctx->dSigma;
  ep.desc = (const EpiDesc*)ctx->epidesc.p;
  ep.scale = -1.0 / (double)P.nk;
  ep.hermitize = ctx->hermitize;
  int rc = tic(ctx, GWSIG_KIND_EPILOGUE);
  if (rc) return rc;
  CU(launch_epilogue(ep, ctx->n_epidesc, ctx->num_sms, ctx->stream));
  if ((rc = toc(ctx))) return rc;
  ctx->launches++;
  ctx->in_eval = false;
  ctx->exchange = false;
  return GWSIG_OK;
}

int gwsig_sigma_eval(gwsig_ctx* ctx, const void* dG, const void* dV_all, const void* dW, void* dSigma, void* stream) {
  int rc = gwsig_sigma_begin(ctx, dG, dW, dSigma, stream);
  if (rc) return rc;
  rc = gwsig_sigma_push_pairs(ctx, 0, ctx->plan.npairs, dV_all);
  if (rc) return rc;
  return gwsig_sigma_end(ctx);
}

int gwsig_sigma_abort(gwsig_ctx* ctx) {
  if (!ctx) return GWSIG_ERR_ARG;
  if (!ctx->in_eval) return fail(ctx, GWSIG_ERR_ORDER, "sigma_abort: no evaluation is open");
  ctx->in_eval = false;
  ctx->exchange = false;
  return GWSIG_OK;
}

/* ---- N2: Hartree-Fock exchange K^k (Eq. 21c) = Eq. 16 with W -> delta_{QQ'} and G(tau) -> gamma --------- */
int gwsig_exchange_begin(gwsig_ctx* ctx, const void* dGamma, void* dK, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  if (ctx->in_eval) return fail(ctx, GWSIG_ERR_ORDER, "exchange_begin: an evaluation is already open");
  ctx->exchange = true;
  int rc = gwsig_sigma_begin(ctx, dGamma, nullptr, dK, stream);
  if (rc) ctx->exchange = false;
  return rc;
}

int gwsig_exchange_eval(gwsig_ctx* ctx, const void* dGamma, const void* dV_all, void* dK, void* stream) {
  int rc = gwsig_exchange_begin(ctx, dGamma, dK, stream);
  if (rc) return rc;
  rc = gwsig_sigma_push_pairs(ctx, 0, ctx->plan.npairs, dV_all);
  if (rc) { ctx->in_eval = false; ctx->exchange = false; return rc; }
  return gwsig_sigma_end(ctx);
}

/* ---- N2: Hartree J, Eq. 21b ---------------------------------------------------------------------------------- */
int gwsig_hartree_eval(gwsig_ctx* ctx, const void* dGamma, const void* dVdiag, void* dJ, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!P.have_lattice) return fail(ctx, GWSIG_ERR_ARG, "hartree_eval: call set_lattice first");
  if (ctx->in_eval || ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "hartree_eval: an evaluation is open");
  if (!dGamma || !dVdiag || !dJ) return fail(ctx, GWSIG_ERR_ARG, "hartree_eval: NULL device pointer");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  ctx->stream = (cudaStream_t)stream;
  ctx->ev_used.clear();
  ctx->launches = 0;
  CU(ctx->hart_rho.ensure((size_t)P.naux * sizeof(double2)));
  if ((rc = tic(ctx, GWSIG_KIND_HARTREE))) return rc;
  CU(launch_hartree((const double2*)dGamma, (const double2*)dVdiag, (double2*)ctx->hart_rho.p, (double2*)dJ, P.nk, P.nao, P.naux, ctx->stream));
  if ((rc = toc(ctx))) return rc;
  ctx->launches += 2;
  return GWSIG_OK;
}

/* ---- N3: P^q(tau) from the bare bubble, Eq. 19 ------------------------------------------------------- */
int gwsig_dyson_p(gwsig_ctx* ctx, const void* dP0, const void* dTf, const void* dTb, int nw, void* dP, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!P.have_sym) return fail(ctx, GWSIG_ERR_ARG, "dyson_p: call set_symmetry first");
  if (P.mode == GWSIG_IBZ_BLOCK) return fail(ctx, GWSIG_ERR_ARG, "dyson_p: built for the dense layouts (FULL_BZ, IBZ) only");
  if (ctx->in_eval || ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "dyson_p: an evaluation is open");
  if (!dP0 || !dTf || !dTb || !dP || nw < 1) return fail(ctx, GWSIG_ERR_ARG, "dyson_p: NULL pointer or nw < 1");
  if (P.naux > 512) return fail(ctx, GWSIG_ERR_ARG, "dyson_p: naux > 512");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  ctx->stream = (cudaStream_t)stream;
  CU(ctx->counters.ensure(gwsig_ctx::kCounterSlots * sizeof(unsigned long long)));
  CU(cudaMemsetAsync(ctx->counters.p, 0, gwsig_ctx::kCounterSlots * sizeof(unsigned long long), ctx->stream));
  ctx->counter_slot = 0;
  ctx->ev_used.clear();
  ctx->launches = 0;
  const int nq = P.nk1;
  const long long n2 = (long long)P.naux * P.naux;
  const int ncta = 2 * std::max(ctx->num_sms, 1);
  CU(ctx->xbuf.ensure((size_t)nq * nw * n2 * sizeof(double2)));                       // P0(i Omega), then P(i Omega) in place
  CU(ctx->ybuf.ensure((size_t)ncta * P.naux * 2 * P.naux * sizeof(double2)));         // per-CTA augmented matrices
  CU(ctx->dys_flag.ensure(16));
  CU(cudaMemsetAsync(ctx->dys_flag.p, 0, 16, ctx->stream));
  auto xform = [&](const double2* src, const double2* T, double2* dst, int nin, int nout) -> int {
    StagePlan sp;
    int r = P.build_gridtransform(nq, nin, nout, sp);
    if (r) return fail(ctx, r, "internal: build_gridtransform failed");
    DevStage d;
    d.nprob = (int)sp.prob.size(); d.ntiles = sp.ntiles;
    if ((r = upload(ctx, d.prob, sp.prob))) return r;
    if ((r = upload(ctx, d.seg, sp.seg))) return r;
    if ((r = upload(ctx, d.bucket, sp.bucket))) return r;
    r = run_stage(ctx, GWSIG_KIND_GRIDXFORM, d, src, T, dst, 0);
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    d.prob.release(); d.seg.release(); d.bucket.release();
    if (r) return r;
    if (e != cudaSuccess) return cuda_fail(ctx, e, "dyson_p transform");
    return GWSIG_OK;
  };
  // P0(i Omega_n) = sum_t Tf[n,t] P0(tau_t)
  if ((rc = xform((const double2*)dP0, (const double2*)dTf, (double2*)ctx->xbuf.p, P.ntau, nw))) return rc;
  // P(i Omega) = [1 - P0(i Omega)]^{-1} P0(i Omega)                                   (Eq. 19a)
  if ((rc = tic(ctx, GWSIG_KIND_DYSON))) return rc;
  CU(launch_dyson_solve((double2*)ctx->xbuf.p, nq * nw, P.naux, (double2*)ctx->ybuf.p, ncta, (int*)ctx->dys_flag.p, ctx->stream));
  if ((rc = toc(ctx))) return rc;
  ctx->launches++;
  // P(tau_t) = sum_n Tb[t,n] P(i Omega_n)                                             (Eq. 19b)
  if ((rc = xform((const double2*)ctx->xbuf.p, (const double2*)dTb, (double2*)dP, nw, P.ntau))) return rc;
  int flag = 0;
  CU(cudaMemcpyAsync(&flag, ctx->dys_flag.p, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (flag) return fail(ctx, GWSIG_ERR_ARG, "dyson_p: 1 - P0(i Omega) is singular (or an input is not finite) for at least one (q, Omega)");
  return GWSIG_OK;
}

/* ---- N4: Eq. 27 on the device --------------------------------------------------------------------------- */
int gwsig_block_transform_v(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV_dense, void* dV_packed, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (P.mode != GWSIG_IBZ_BLOCK || !P.have_blocks || !P.have_triples)
    return fail(ctx, GWSIG_ERR_ARG, "block_transform_v: needs GWSIG_IBZ_BLOCK with set_blocks and set_triples");
  if (!P.have_U) return fail(ctx, GWSIG_ERR_ARG, "block_transform_v: set_blocks must be given the adapted bases U_ao, U_aux");
  // V prepared on demand ("copied on demand"): the call is allowed between the pushes of an open Sigma evaluation,
  // on that evaluation's stream (it shares the X / Y scratch and the tile counters with it, in stream order)
  if (ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "block_transform_v: a P0 evaluation is open");
  if (ctx->in_eval && (cudaStream_t)stream != ctx->stream) return fail(ctx, GWSIG_ERR_ARG, "block_transform_v: inside an open evaluation the stream must be the evaluation's");
  if (np < 1 || p0 < 0 || p0 + np > P.npairs) return fail(ctx, GWSIG_ERR_ARG, "block_transform_v: bad pair range");
  if (!dV_dense || !dV_packed) return fail(ctx, GWSIG_ERR_ARG, "block_transform_v: NULL device pointer");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  ctx->stream = (cudaStream_t)stream;
  if ((rc = prepare_tables(ctx))) return rc;
  CU(ctx->counters.ensure(gwsig_ctx::kCounterSlots * sizeof(unsigned long long)));
  CU(cudaMemsetAsync(ctx->counters.p, 0, gwsig_ctx::kCounterSlots * sizeof(unsigned long long), ctx->stream));
  ctx->counter_slot = 0;
  const long long xs = (long long)P.naux * P.nao * P.nao;
  size_t free_b = 0, total_b = 0;
  CU(cudaMemGetInfo(&free_b, &total_b));
  const double avail = 0.4 * ((double)free_b + (double)ctx->xbuf.bytes + (double)ctx->ybuf.bytes);
  const double budget = std::min((double)ctx->scratch_mib * 1048576.0, std::max(avail, 64.0 * 1048576.0)) / (2.0 * sizeof(double2));
  const long long ns_max = std::max<long long>(1, (long long)(budget / (double)xs));
  for (long long s0 = p0; s0 < p0 + np; s0 += ns_max) {
    const long long ns = std::min<long long>(ns_max, p0 + np - s0);
    CU(ctx->xbuf.ensure((size_t)xs * ns * sizeof(double2)));
    CU(ctx->ybuf.ensure((size_t)xs * ns * sizeof(double2)));
    const double2* Vsub = (const double2*)dV_dense + (s0 - p0) * xs;
    double2* Out = (double2*)dV_packed + (P.v_off[s0] - P.v_off[p0]);
    for (int step = 1; step <= 3; ++step) {
      StagePlan sp;
      rc = P.build_vtransform(s0, ns, step, sp);
      if (rc) return fail(ctx, rc, "internal: build_vtransform failed");
      DevStage d;
      d.nprob = (int)sp.prob.size(); d.ntiles = sp.ntiles;
      if ((rc = upload(ctx, d.prob, sp.prob))) return rc;
      if ((rc = upload(ctx, d.seg, sp.seg))) return rc;
      if ((rc = upload(ctx, d.bucket, sp.bucket))) return rc;
      const double2* A = step == 1 ? Vsub : step == 2 ? (const double2*)ctx->xbuf.p : (const double2*)ctx->ybuf.p;
      const double2* Bm = (const double2*)(step == 1 ? ctx->u_aux_dev.p : ctx->u_ao_dev.p);
      double2* C = step == 1 ? (double2*)ctx->xbuf.p : step == 2 ? (double2*)ctx->ybuf.p : Out;
      rc = run_stage(ctx, GWSIG_KIND_VTRANSFORM, d, A, Bm, C, 0);
      cudaError_t e = cudaStreamSynchronize(ctx->stream);      // the descriptor tables are freed below
      d.prob.release(); d.seg.release(); d.bucket.release();
      if (rc) return rc;
      if (e != cudaSuccess) return cuda_fail(ctx, e, "block_transform_v");
    }
  }
  return GWSIG_OK;
}

/* ---- N4: allowed-block detection on the device (Eq. 27) ------------------------------------------------------ */
int gwsig_block_maxabs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV_dense, int mb_aux, int mb_ao, void* d_maxabs, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (P.mode != GWSIG_IBZ_BLOCK || !P.have_blocks) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: needs GWSIG_IBZ_BLOCK with set_blocks");
  if (!P.have_U) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: set_blocks must be given the adapted bases U_ao, U_aux");
  if (ctx->in_eval || ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "block_maxabs: an evaluation is open");
  if (np < 1 || p0 < 0 || p0 + np > P.npairs) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: bad pair range");
  if (!dV_dense || !d_maxabs) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: NULL device pointer");
  int nb_aux = 0, nb_ao = 0;
  for (int k = 0; k < P.nk; ++k) {
    nb_aux = std::max(nb_aux, (int)P.aux_off[k].size() - 1);
    nb_ao = std::max(nb_ao, (int)P.ao_off[k].size() - 1);
  }
  if (mb_aux < nb_aux || mb_ao < nb_ao) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: mb_aux / mb_ao smaller than the largest block count of a mesh point");
  const long long ncand = (long long)mb_aux * mb_ao * mb_ao;
  if (ncand * 8 > 48 * 1024) return fail(ctx, GWSIG_ERR_ARG, "block_maxabs: more than 6144 candidate blocks per pair");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  ctx->stream = (cudaStream_t)stream;
  if ((rc = prepare_tables(ctx))) return rc;
  CU(ctx->counters.ensure(gwsig_ctx::kCounterSlots * sizeof(unsigned long long)));
  CU(cudaMemsetAsync(ctx->counters.p, 0, gwsig_ctx::kCounterSlots * sizeof(unsigned long long), ctx->stream));
  ctx->counter_slot = 0;
  ctx->ev_used.clear();
  ctx->launches = 0;
  // block label of every basis function at every mesh point
  std::vector<int> lab_aux((size_t)P.nk * P.naux), lab_ao((size_t)P.nk * P.nao);
  for (int k = 0; k < P.nk; ++k) {
    for (size_t b = 0; b + 1 < P.aux_off[k].size(); ++b)
      for (int i = P.aux_off[k][b]; i < P.aux_off[k][b + 1]; ++i) lab_aux[(size_t)k * P.naux + i] = (int)b;
    for (size_t b = 0; b + 1 < P.ao_off[k].size(); ++b)
      for (int i = P.ao_off[k][b]; i < P.ao_off[k][b + 1]; ++i) lab_ao[(size_t)k * P.nao + i] = (int)b;
  }
  DevBuf d_lab_aux, d_lab_ao, d_qkk;
  auto cleanup = [&]() { d_lab_aux.release(); d_lab_ao.release(); d_qkk.release(); };
  if ((rc = upload(ctx, d_lab_aux, lab_aux)) || (rc = upload(ctx, d_lab_ao, lab_ao))) { cleanup(); return rc; }
  cudaError_t e = cudaMemsetAsync(d_maxabs, 0, (size_t)np * ncand * sizeof(double), ctx->stream);
  if (e != cudaSuccess) { cleanup(); return cuda_fail(ctx, e, "block_maxabs memset"); }
  const long long xs = (long long)P.naux * P.nao * P.nao;
  size_t free_b = 0, total_b = 0;
  e = cudaMemGetInfo(&free_b, &total_b);
  if (e != cudaSuccess) { cleanup(); return cuda_fail(ctx, e, "cudaMemGetInfo"); }
  const double avail = 0.4 * ((double)free_b + (double)ctx->xbuf.bytes + (double)ctx->ybuf.bytes);
  const double budget = std::min((double)ctx->scratch_mib * 1048576.0, std::max(avail, 64.0 * 1048576.0)) / (2.0 * sizeof(double2));
  const long long ns_max = std::max<long long>(1, (long long)(budget / (double)xs));
  for (long long s0 = p0; s0 < p0 + np; s0 += ns_max) {
    const long long ns = std::min<long long>(ns_max, p0 + np - s0);
    if ((e = ctx->xbuf.ensure((size_t)xs * ns * sizeof(double2))) != cudaSuccess || (e = ctx->ybuf.ensure((size_t)xs * ns * sizeof(double2))) != cudaSuccess) {
      cleanup();
      return cuda_fail(ctx, e, "block_maxabs scratch");
    }
    const double2* Vsub = (const double2*)dV_dense + (s0 - p0) * xs;
    const int steps[3] = {1, 2, 4};                  // T1 -> xbuf, T2 -> ybuf, T3 (dense, every block) -> xbuf
    for (int si = 0; si < 3; ++si) {
      StagePlan sp;
      rc = P.build_vtransform(s0, ns, steps[si], sp);
      if (rc) { cleanup(); return fail(ctx, rc, "internal: build_vtransform failed"); }
      DevStage d;
      d.nprob = (int)sp.prob.size(); d.ntiles = sp.ntiles;
      if ((rc = upload(ctx, d.prob, sp.prob)) || (rc = upload(ctx, d.seg, sp.seg)) || (rc = upload(ctx, d.bucket, sp.bucket))) { cleanup(); return rc; }
      const double2* A = si == 0 ? Vsub : si == 1 ? (const double2*)ctx->xbuf.p : (const double2*)ctx->ybuf.p;
      const double2* Bm = (const double2*)(si == 0 ? ctx->u_aux_dev.p : ctx->u_ao_dev.p);
      double2* C = si == 1 ? (double2*)ctx->ybuf.p : (double2*)ctx->xbuf.p;
      rc = run_stage(ctx, GWSIG_KIND_VTRANSFORM, d, A, Bm, C, 0);
      e = cudaStreamSynchronize(ctx->stream);      // the descriptor tables are freed below
      d.prob.release(); d.seg.release(); d.bucket.release();
      if (rc) { cleanup(); return rc; }
      if (e != cudaSuccess) { cleanup(); return cuda_fail(ctx, e, "block_maxabs"); }
    }
    std::vector<int> qkk((size_t)3 * ns);
    for (long long l = 0; l < ns; ++l) {
      int k1, k2, q, i1;
      P.pair(s0 + l, k1, k2, q, i1);
      qkk[3 * l] = q; qkk[3 * l + 1] = k2; qkk[3 * l + 2] = k1;
    }
    if ((rc = upload(ctx, d_qkk, qkk))) { cleanup(); return rc; }
    e = launch_block_maxabs((const double2*)ctx->xbuf.p, (const int*)d_lab_aux.p, (const int*)d_lab_ao.p, (const int*)d_qkk.p,
                            (double*)d_maxabs + (s0 - p0) * ncand, (int)ns, P.naux, P.nao, mb_aux, mb_ao, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { cleanup(); return cuda_fail(ctx, e, "block_maxabs reduction"); }
    ctx->launches++;
  }
  cleanup();
  return GWSIG_OK;
}

/* ---- N1: bare bubble P0^q(tau) (Eq. 20, Algorithm 3), dense modes ---------------------------- */
int gwsig_p0_begin(gwsig_ctx* ctx, const void* dG, void* dP0, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!P.have_sym) return fail(ctx, GWSIG_ERR_ARG, "p0_begin: call set_symmetry first");
  if (P.mode == GWSIG_IBZ_BLOCK) return fail(ctx, GWSIG_ERR_ARG, "p0_begin: the bare bubble is built for the dense modes (FULL_BZ, IBZ) only");
  if (ctx->in_eval || ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "p0_begin: an evaluation is already open");
  if (!dG || !dP0) return fail(ctx, GWSIG_ERR_ARG, "p0_begin: NULL device pointer");
  // reuse sigma_begin for the device set-up and the unfold of G (Eq. 22); it needs no W for that
  ctx->exchange = true;
  int rc = gwsig_sigma_begin(ctx, dG, nullptr, dP0, stream);
  ctx->exchange = false;
  ctx->in_eval = false;
  if (rc) return rc;
  const double2* Gsrc = P.mode == GWSIG_IBZ ? (const double2*)ctx->gbz.p : ctx->dG;
  const long long n2 = (long long)P.nao * P.nao;
  // two transposed copies of G on the whole zone (Algorithm 3 contracts G over its second index: the transposes make the tile
  // rows the contiguous index of the A operand): grev[0 .. ) = G(beta - tau)^T and, behind it, G(tau)^T.
  // G(-tau_n) = -G(beta - tau_n) = -G[ntau-1-n] (fermionic antiperiodicity, uniform grid); the sign goes into the epilogue
  // (-(1/Nk) of Eq. 20 becomes +1/Nk)
  const size_t gelems = (size_t)P.nk * P.ntau * n2;
  CU(ctx->grev.ensure(2 * gelems * sizeof(double2)));
  CU(launch_transpose_tau(Gsrc, (double2*)ctx->grev.p, P.nk, P.ntau, P.nao, true, ctx->stream));
  CU(launch_transpose_tau(Gsrc, (double2*)ctx->grev.p + gelems, P.nk, P.ntau, P.nao, false, ctx->stream));
  ctx->launches += 2;
  const size_t pe = (size_t)P.nk1 * P.ntau * P.naux * P.naux;
  CU(ctx->p0acc.ensure(std::max<size_t>(pe * sizeof(double2), 16)));
  CU(cudaMemsetAsync(ctx->p0acc.p, 0, pe * sizeof(double2), ctx->stream));
  ctx->dP0 = (double2*)dP0;
  ctx->next_pair = 0;
  ctx->in_p0 = true;
  return GWSIG_OK;
}

int gwsig_p0_push_pairs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "p0_push_pairs: call p0_begin first");
  const long long npairs = (long long)P.nk * P.nk1;
  if (np < 1 || p0 != ctx->next_pair || p0 + np > npairs)
    return fail(ctx, GWSIG_ERR_ORDER, "p0_push_pairs: ranges must be pushed in increasing order without gaps");
  if (!dV) return fail(ctx, GWSIG_ERR_ARG, "p0_push_pairs: NULL device pointer");
  CU(cudaSetDevice(ctx->device));
  const long long xs = (long long)P.naux * P.nao * P.nao;
  size_t free_b = 0, total_b = 0;
  CU(cudaMemGetInfo(&free_b, &total_b));
  const double avail = 0.4 * ((double)free_b + (double)ctx->xbuf.bytes + (double)ctx->ybuf.bytes);
  const double budget = std::min((double)ctx->scratch_mib * 1048576.0, std::max(avail, 64.0 * 1048576.0)) / (2.0 * sizeof(double2));
  const double2* Gsrc = P.mode == GWSIG_IBZ ? (const double2*)ctx->gbz.p : ctx->dG;
  const double2* Vbase = (const double2*)dV;
  long long s0 = p0;
  while (s0 < p0 + np) {
    // sub-batch: as many pairs as fit the X1 / X2 scratch for at least one tau; then as many tau as fit
    long long ns = std::max<long long>(1, std::min<long long>(p0 + np - s0, (long long)(budget / (double)xs)));
    int nt_max = ctx->tau_chunk > 0 ? ctx->tau_chunk : (int)std::max(1.0, std::floor(budget / ((double)xs * (double)ns)));
    nt_max = std::min(nt_max, P.ntau);
    const int nchunks = (P.ntau + nt_max - 1) / nt_max;
    const int nt = (P.ntau + nchunks - 1) / nchunks;
    const size_t xbytes = (size_t)xs * ns * nt * sizeof(double2);
    CU(ctx->xbuf.ensure(xbytes));
    CU(ctx->ybuf.ensure(xbytes));
    // the sub-batch's pair tensors with the auxiliary index last (what the stage-1 / stage-2 descriptors address)
    CU(ctx->p0vt.ensure((size_t)xs * ns * sizeof(double2)));
    CU(launch_aux_last(Vbase + (s0 - p0) * xs, (double2*)ctx->p0vt.p, ns, P.naux, P.nao * P.nao, ctx->stream));
    ctx->launches++;
    const double2* Vsub = (const double2*)ctx->p0vt.p;
    for (int t0 = 0; t0 < P.ntau; t0 += nt) {
      const int ntc = std::min(nt, P.ntau - t0);
      auto key = std::make_tuple((long long)s0, (long long)ns, ntc);
      DevPlan* dp = nullptr;
      auto it = ctx->p0_cache.find(key);
      if (it != ctx->p0_cache.end()) dp = it->second.get();
      else {
        std::unique_ptr<DevPlan> np_(new DevPlan());
        for (int s = 0; s < 3; ++s) {
          StagePlan sp;
          int rc = P.build_p0_stage(s0, ns, ntc, s + 1, sp, ctx->num_sms > 0 ? ctx->num_sms : 148);
          if (rc) return fail(ctx, rc, "internal: build_p0_stage failed");
          DevStage& d = np_->st[s];
          d.nprob = (int)sp.prob.size(); d.ntiles = sp.ntiles;
          if ((rc = upload(ctx, d.prob, sp.prob))) return rc;
          if ((rc = upload(ctx, d.seg, sp.seg))) return rc;
          if ((rc = upload(ctx, d.bucket, sp.bucket))) return rc;
        }
        dp = np_.get();
        ctx->p0_cache[key] = std::move(np_);
      }
      int rc;
      if ((rc = run_stage(ctx, GWSIG_KIND_STAGE1, dp->st[0], (const double2*)ctx->grev.p, Vsub, (double2*)ctx->xbuf.p, t0))) return rc;   // X1
      if ((rc = run_stage(ctx, GWSIG_KIND_STAGE2, dp->st[1], (const double2*)ctx->grev.p + (size_t)P.nk * P.ntau * P.nao * P.nao, Vsub, (double2*)ctx->ybuf.p, t0))) return rc;   // X2
      if ((rc = run_stage(ctx, GWSIG_KIND_STAGE3, dp->st[2], (const double2*)ctx->xbuf.p, (const double2*)ctx->ybuf.p, (double2*)ctx->p0acc.p, t0))) return rc;
    }
    s0 += ns;
  }
  ctx->next_pair = p0 + np;
  return GWSIG_OK;
}

int gwsig_p0_end(gwsig_ctx* ctx) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!ctx->in_p0) return fail(ctx, GWSIG_ERR_ORDER, "p0_end: call p0_begin first");
  if (ctx->next_pair != (long long)P.nk * P.nk1) return fail(ctx, GWSIG_ERR_ORDER, "p0_end: not all pairs were pushed");
  CU(cudaSetDevice(ctx->device));
  std::vector<EpiDesc> ed;
  for (int iq = 0; iq < P.nk1; ++iq) ed.push_back(EpiDesc{(long long)iq * P.ntau * P.naux * P.naux, (long long)P.naux * P.naux, P.naux, P.ntau});
  int rc = upload(ctx, ctx->p0desc, ed);
  if (rc) return rc;
  EpilogueParams ep;
  ep.acc = (const double2*)ctx->p0acc.p;
  ep.out = ctx->dP0;
  ep.desc = (const EpiDesc*)ctx->p0desc.p;
  ep.scale = 1.0 / (double)P.nk;          // -(1/Nk) of Eq. 20 times the -1 of G(-tau) = -G(beta - tau)
  ep.hermitize = ctx->hermitize;
  if ((rc = tic(ctx, GWSIG_KIND_EPILOGUE))) return rc;
  CU(launch_epilogue(ep, (int)ed.size(), ctx->num_sms, ctx->stream));
  if ((rc = toc(ctx))) return rc;
  ctx->launches++;
  ctx->in_p0 = false;
  return GWSIG_OK;
}

int gwsig_p0_eval(gwsig_ctx* ctx, const void* dG, const void* dV_all, void* dP0, void* stream) {
  int rc = gwsig_p0_begin(ctx, dG, dP0, stream);
  if (rc) return rc;
  rc = gwsig_p0_push_pairs(ctx, 0, (int64_t)ctx->plan.nk * ctx->plan.nk1, dV_all);
  if (rc) { ctx->in_p0 = false; return rc; }
  return gwsig_p0_end(ctx);
}

int gwsig_sigma_eval_host(gwsig_ctx* ctx, const void* hG, const void* hV_all, const void* hW, void* hSigma, void* stream) {
  if (!ctx) return GWSIG_ERR_ARG;
  Plan& P = ctx->plan;
  if (!P.have_sym || P.v_off.empty()) return fail(ctx, GWSIG_ERR_ARG, "sigma_eval_host: plan incomplete (set_symmetry / set_triples)");
  if (!hG || !hV_all || !hW || !hSigma) return fail(ctx, GWSIG_ERR_ARG, "sigma_eval_host: NULL host pointer");
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  cudaStream_t st = (cudaStream_t)stream;
  if (!ctx->copy_stream) {
    CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CU(cudaEventCreateWithFlags(&ctx->ev_copied[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&ctx->ev_freed[i], cudaEventDisableTiming));
    }
  }
  const size_t cb = sizeof(double2);
  CU(ctx->h_g.ensure(std::max<size_t>(P.g_elems * cb, 16)));
  CU(ctx->h_w.ensure(std::max<size_t>(P.w_elems * cb, 16)));
  CU(ctx->h_sig.ensure(std::max<size_t>(P.sig_elems * cb, 16)));
  // batches of whole q (nk1 pairs each) that fit one ring slot; a single q larger than the slot grows the slot
  const int nk1 = P.nk1;
  const long long slot_elems_opt = ctx->v_ring_mib * 1048576LL / (long long)cb;
  std::vector<long long> cuts{0};
  long long need = 0;
  for (long long p = 0; p < P.npairs;) {
    long long e = p + nk1;
    while (e < P.npairs && P.v_off[e + nk1] - P.v_off[p] <= slot_elems_opt) e += nk1;
    need = std::max(need, P.v_off[e] - P.v_off[p]);
    cuts.push_back(e);
    p = e;
  }
  const int nslots = cuts.size() > 2 ? 2 : 1;
  for (int i = 0; i < nslots; ++i) CU(ctx->h_vslot[i].ensure(std::max<size_t>(need * cb, 16)));
  CU(cudaMemcpyAsync(ctx->h_g.p, hG, P.g_elems * cb, cudaMemcpyHostToDevice, st));
  CU(cudaMemcpyAsync(ctx->h_w.p, hW, P.w_elems * cb, cudaMemcpyHostToDevice, st));
  if ((rc = gwsig_sigma_begin(ctx, ctx->h_g.p, ctx->h_w.p, ctx->h_sig.p, stream))) return rc;
  const double2* hV = (const double2*)hV_all;
  for (size_t b = 0; b + 1 < cuts.size(); ++b) {
    const int slot = (int)(b % nslots);
    const long long p0 = cuts[b], p1 = cuts[b + 1];
    if (b >= (size_t)nslots) CU(cudaStreamWaitEvent(ctx->copy_stream, ctx->ev_freed[slot], 0));   // slot consumed?
    CU(cudaMemcpyAsync(ctx->h_vslot[slot].p, hV + P.v_off[p0], (size_t)(P.v_off[p1] - P.v_off[p0]) * cb, cudaMemcpyHostToDevice,
                       ctx->copy_stream));
    CU(cudaEventRecord(ctx->ev_copied[slot], ctx->copy_stream));
    CU(cudaStreamWaitEvent(st, ctx->ev_copied[slot], 0));
    if ((rc = gwsig_sigma_push_pairs(ctx, p0, p1 - p0, ctx->h_vslot[slot].p))) { ctx->in_eval = false; return rc; }
    CU(cudaEventRecord(ctx->ev_freed[slot], st));
  }
  if ((rc = gwsig_sigma_end(ctx))) return rc;
  CU(cudaMemcpyAsync(hSigma, ctx->h_sig.p, P.sig_elems * cb, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return GWSIG_OK;
}

int gwsig_probe_fp64(gwsig_ctx* ctx, int kind, int warps_per_block, int blocks_per_sm, int64_t iters, double* tflops,
                     double* ms) {
  if (!ctx || !tflops || kind < 0 || kind > 3 || warps_per_block < 1 || warps_per_block > 32 || blocks_per_sm < 1 || iters < 1) return GWSIG_ERR_ARG;
  int rc = ensure_cuda(ctx);
  if (rc) return rc;
  CU(cudaSetDevice(ctx->device));
  CU(ctx->probe_sink.ensure(64));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0));
  CU(cudaEventCreate(&e1));
  double flops = 0;
  CU(launch_probe(kind, warps_per_block, ctx->num_sms * blocks_per_sm, iters / 8 + 1, (double*)ctx->probe_sink.p, nullptr, &flops));  // warm-up
  CU(cudaEventRecord(e0, nullptr));
  CU(launch_probe(kind, warps_per_block, ctx->num_sms * blocks_per_sm, iters, (double*)ctx->probe_sink.p, nullptr, &flops));
  CU(cudaEventRecord(e1, nullptr));
  CU(cudaEventSynchronize(e1));
  float t = 0;
  CU(cudaEventElapsedTime(&t, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  *tflops = flops / (t * 1e-3) / 1e12;
  if (ms) *ms = t;
  return GWSIG_OK;
}

}  // extern "C"
