/* gwsig -- C-ABI boundary of the B200-native GW self-energy evaluation.
 *
 * The operation (Eq. 16 of arXiv 2405.09494, readings A1/A6/A7 of DESIGN.md):
 *
 *   Sigma_ij(k,tau) = -(1/Nk) sum_{q in BZ} sum_{QQ'ab}
 *        conj(V2[Q,a,i]) * G_ab(k-q,tau) * W_{QQ'}(q,tau) * V2[Q',b,j],      V2 = V^{k-q,k}
 *
 * evaluated for k in the irreducible wedge, optionally in the
 * Dirac-character block basis over the symmetry-allowed blocks only,
 * following the pair loop of Algorithm 4.  W is the paper's P^q(tau) (Eq. 19).
 *
 * Conventions
 *   - every function returns 0 on success, a negative gwsig_status otherwise; nothing is
 *     launched on error; gwsig_last_error() returns a static description of the last failure.
 *   - all array arguments are CALLER-OWNED; the library copies what it keeps at the call.
 *   - "host" / "dev" in a comment says where the pointer must live.  Complex numbers are
 *     interleaved (re, im) doubles (complex128).  Matrices are row-major.
 *   - momenta are mesh indices  k = (n0*N1 + n1)*N2 + n2,  k - q is taken modulo the mesh.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - no CPU fallback exists: without a CUDA device sigma_* return GWSIG_ERR_CUDA.
 *     The plan-side calls (set_*, get_ibz, pair_*, plan_*) are host-only and need no device.
 */
#ifndef GWSIG_H
#define GWSIG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gwsig_ctx gwsig_ctx;

typedef enum {
  GWSIG_OK = 0,
  GWSIG_ERR_ARG = -1,      /* bad size / NULL pointer / call order                               */
  GWSIG_ERR_SYMMETRY = -2, /* rotation does not map the mesh onto itself, D not orthogonal, ...   */
  GWSIG_ERR_BLOCKS = -3,   /* block maps do not tile [0,n), star members disagree, bad triples    */
  GWSIG_ERR_CUDA = -4,     /* CUDA runtime error (message holds cudaGetErrorString)               */
  GWSIG_ERR_ORDER = -5     /* pushed pair range out of order / incomplete at sigma_end            */
} gwsig_status;

typedef enum {
  GWSIG_FULL_BZ = 0,   /* k1 over the whole mesh, G and W given on the whole mesh, no unfold      */
  GWSIG_IBZ = 1,       /* k1 over the wedge; G, W given at wedge points, unfolded by Eq. 22 / 25  */
  GWSIG_IBZ_BLOCK = 2  /* wedge + block basis: packed irrep blocks, allowed triples only          */
} gwsig_mode;

typedef enum {
  GWSIG_ENGINE_DMMA = 0,      /* FP64 tensor-core grouped GEMM (mma.sync m8n8k4 f64 -> DMMA), default: per stage the
                                 faster of the two tensor kernels below (3M for stages 1 and 2, 4M for stage 3)         */
  GWSIG_ENGINE_REFERENCE = 1, /* one-thread-per-element DFMA kernels on the same plan (debug)                       */
  GWSIG_ENGINE_DMMA_4M = 2,   /* every stage on the tensor-core kernel with the conventional 4-product complex multiply */
  GWSIG_ENGINE_DMMA_3M = 3    /* every stage on the tensor-core kernel with the 3M / Karatsuba complex multiply:
                                 3 real DMMA per complex 8x8x4 block                                                 */
} gwsig_engine;

/* kernel kinds for gwsig_kernel_times (steps a1..a6 of DESIGN.md) */
enum {
  GWSIG_KIND_UNFOLD_G = 0,
  GWSIG_KIND_UNFOLD_W = 1,
  GWSIG_KIND_STAGE1 = 2, /* X = V G          */
  GWSIG_KIND_STAGE2 = 3, /* Y = W X          */
  GWSIG_KIND_STAGE3 = 4, /* Sigma += Y V     */
  GWSIG_KIND_EPILOGUE = 5,
  GWSIG_KIND_VTRANSFORM = 6, /* Eq. 27 block transform of V (gwsig_block_transform_v) */
  GWSIG_KIND_GRIDXFORM = 7,  /* tau <-> i Omega transforms of gwsig_dyson_p                  */
  GWSIG_KIND_DYSON = 8,      /* batched [1 - P0]^{-1} P0 solve of gwsig_dyson_p             */
  GWSIG_KIND_HARTREE = 9,    /* the two kernels of gwsig_hartree_eval (Eq. 21b)             */
  GWSIG_NKINDS = 10
};

/* ---- life cycle ------------------------------------------------------------------------ */
/* device >= 0: CUDA device ordinal used by sigma_*; device < 0: host-only context (plan calls). */
int gwsig_create(gwsig_ctx** out, int device);
int gwsig_destroy(gwsig_ctx* ctx);
const char* gwsig_last_error(const gwsig_ctx* ctx);

/* ---- problem statement ----------------------------------------------------------------------
 * set_lattice: a[9] rows = primitive vectors (host); mesh[3] = Gamma-centred k mesh;
 * nao, naux = orbital / auxiliary basis sizes; ntau = number of imaginary-time points (Sigma is
 * pointwise in tau, the grid itself is not needed); beta is recorded only.                        */
int gwsig_set_lattice(gwsig_ctx* ctx, const double a[9], const int mesh[3], int nao, int naux, int ntau,
                      double beta);

/* set_atoms: natom; pos[natom*3] fractional (host, recorded); ao_atom[nao], aux_atom[naux] = atom
 * each basis function sits on (needed for the per-atom phase of Eq. 3).           */
int gwsig_set_atoms(gwsig_ctx* ctx, int natom, const double* pos, const int* ao_atom, const int* aux_atom);

/* set_symmetry (all host):
 *   rot[nops*9]   integer rotation W in lattice coordinates, r -> W r + w        ({alpha|v})
 *   trans[nops*3] fractional translation w (recorded; enters D^k of Eq. 7 only, i.e. the pre-step)
 *   D_ao[nops*nao*nao], D_aux[nops*naux*naux]  k-independent REAL representation
 *                 (atom permutation (x) real Wigner D, Eq. 3-4); row index = image function
 *   shift[nops*natom*3] integer lattice shift s_x with  W tau_x + w = tau_perm(x) + s_x ("translation
 *                 vector between rotated and original atom").  The library multiplies the
 *                 phase exp(-2 pi i k~ . s_x) into column (x,m) itself:  O^k = D . diag(phase)  (Eq. 3)
 *   mode          gwsig_mode.   nops = 0 is allowed only with GWSIG_FULL_BZ.
 * Builds the k maps, the stars (representative = first member in index order, op_of = first
 * operation in input order mapping it there; space-group operations only, no time reversal) and
 * the (q-major) pair list.  Errors: GWSIG_ERR_SYMMETRY.                                            */
int gwsig_set_symmetry(gwsig_ctx* ctx, int nops, const int* rot, const double* trans, const double* D_ao,
                       const double* D_aux, const int* shift, int mode);

/* set_blocks (IBZ_BLOCK only, host): irrep (isotypic) block maps per mesh point in CSR form:
 *   nblk_ao[Nk], ao_block_off[sum(nblk_ao)+Nk] : for each k the nblk+1 offsets 0 = o_0 < ... = nao
 *   nblk_aux[Nk], aux_block_off[...]           : same for the auxiliary basis at q
 *   U_ao [Nk*nao*nao], U_aux[Nk*naux*naux]     : symmetry-adapted bases U^k (Eq. 26) or NULL.
 *       NULL  = the gauge U^{k'} = O^{k_I}(alpha^) U^{k_I} for star members, for which O_block of
 *               Eq. 28 is the identity and block data of k' are those of its representative;
 *       given = the library forms O_block = U^{k' dagger} O^{k_I}(alpha^) U^{k_I} (Eq. 28) for
 *               op_of[k'] and unfolds packed blocks with it (must come out block diagonal).
 * Errors: GWSIG_ERR_BLOCKS (offsets do not tile, star member's block sizes differ from its
 * representative's, O_block not block diagonal).                                                   */
int gwsig_set_blocks(gwsig_ctx* ctx, const int* nblk_ao, const int* ao_block_off, const int* nblk_aux,
                     const int* aux_block_off, const double* U_ao, const double* U_aux);

/* set_output_points (host, optional, after set_symmetry and before set_triples): evaluate Sigma only at
 * the n listed k1 (wedge representatives in the IBZ modes, any mesh point in FULL_BZ) instead of at all of
 * them.  "One representative is chosen" per star and every output k1 is an independent sum
 * over q (Eq. 16), so this is also how the work would be dealt to several GPUs (the paper distributes
 * (k1,k2) pairs).  Pairs become q * n + i1 over the listed points; inputs G, W keep their
 * layout; V2 and Sigma carry the listed points only.  Errors: GWSIG_ERR_ARG (not a wedge point, repeated). */
int gwsig_set_output_points(gwsig_ctx* ctx, int n, const int* k_list);

/* set_triples (IBZ_BLOCK only, host): symmetry-allowed blocks of V2 for every pair ("only non-zero
 * blocks are considered").  triple_ptr[npairs+1] CSR; triples[3*nt] = (p, alpha, iota):
 * aux block of q, orbital block of k2, orbital block of k1; sorted by p within a pair.              */
int gwsig_set_triples(gwsig_ctx* ctx, int64_t npairs, const int64_t* triple_ptr, const int32_t* triples);

/* ---- what the plan decided (host outputs; any pointer may be NULL) --------------------------- */
int gwsig_get_ibz(gwsig_ctx* ctx, int* nik, int* ir_list /*[nik]*/, int* ir_of /*[Nk]*/, int* op_of /*[Nk]*/);
/* pairs are ordered q-major: pair = q * nk1 + i1, k1 = out_list[i1], k2 = k1 - q                   */
int gwsig_pair_count(gwsig_ctx* ctx, int64_t* npairs, int* nk1);
int gwsig_pair_info(gwsig_ctx* ctx, int64_t pair, int* k1, int* k2, int* q, int64_t* v_offset /*elements*/,
                    int64_t* v_elems);
/* element counts / offsets of the G, W and Sigma buffers sigma_eval expects in the current mode:
 *   FULL_BZ : G[Nk][ntau][nao][nao], W[Nk][ntau][naux][naux], Sigma[Nk][ntau][nao][nao]
 *   IBZ     : the same with the wedge points (in ir_list order) instead of Nk
 *   IBZ_BLOCK: per wedge point [ntau][sum_b n_b^2] packed diagonal blocks, points concatenated     */
int gwsig_buffer_sizes(gwsig_ctx* ctx, int64_t* g_elems, int64_t* w_elems, int64_t* sigma_elems, int64_t* v_elems);

/* ---- the evaluation -------------------------------------------------------------------------
 * sigma_begin : dG, dW (dev, layouts above), dSigma (dev, written by sigma_end).  Unfolds G to the
 *               full zone (Eq. 22 / 28), zeroes the accumulator.
 * sigma_push_pairs : dV (dev) holds V2 = V^{k2,k1}_{Q,bj} for pairs p0 .. p0+np-1, packed back to
 *               back in pair order ([naux][nao][nao] dense; allowed blocks in IBZ_BLOCK mode, see
 *               DESIGN.md).  Ranges must be pushed in increasing order without gaps and should
 *               cover whole q (multiples of nk1) for best reuse of the unfolded W(q).  Runs
 *               X = V G, Y = W X, Sigma += Y V  (Algorithm 4 lines 5-8) for those pairs, all tau.
 *               Exists because V does not fit on the device at the large configs.
 * sigma_end   : epilogue  Sigma = -(1/Nk) * accumulated (optionally Hermitised) -> dSigma.
 * sigma_eval  : begin + one push of all pairs + end.
 * All work is enqueued on `stream`; results are valid after the stream is synchronised.           */
int gwsig_sigma_begin(gwsig_ctx* ctx, const void* dG, const void* dW, void* dSigma, void* stream);
int gwsig_sigma_push_pairs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV);
int gwsig_sigma_end(gwsig_ctx* ctx);
int gwsig_sigma_eval(gwsig_ctx* ctx, const void* dG, const void* dV_all, const void* dW, void* dSigma, void* stream);
/* sigma_abort : leave an evaluation opened by sigma_begin without writing dSigma (nothing is launched).
 *               Used to time a prefix of the pair list (bench.py: FULL_BZ on a q subset, scaled).  */
int gwsig_sigma_abort(gwsig_ctx* ctx);
/* sigma_eval_host : the same evaluation with HOST buffers (layouts as above; page-locked memory gives
 *               asynchronous copies, pageable memory works but serialises).  The library owns the
 *               device side: it copies hG, hW to the device, streams hV through a two-slot device
 *               ring in batches of whole q (option "v_ring_mib", per slot) on its own copy stream so
 *               that the transfer of batch n+1 overlaps the contraction of batch n -- "V is copied on
 *               demand" (Algorithm 4 line 3) -- and copies Sigma back to
 *               hSigma.  Returns after the result has landed in hSigma (the stream is synchronised). */
int gwsig_sigma_eval_host(gwsig_ctx* ctx, const void* hG, const void* hV_all, const void* hW, void* hSigma,
                          void* stream);

/* ---- N2: Hartree-Fock exchange -------------------------------------------------
 * K^k_ij = -(1/Nk) sum_{k'} sum_{ab} sum_Q V^{k k'}_{ia}(Q) gamma^{k'}_{ab} V^{k' k}_{bj}(Q)       (Eq. 21c)
 * is Eq. 16 with W -> delta_{QQ'} and G(k - q, tau) -> the density matrix gamma^{k'}: the same pair list,
 * the same V2 operand, stage 1 (X = V gamma) feeding stage 3 (K += X V) directly, stage 2 skipped.  dGamma has the layout
 * of G with the context's ntau slices treated as independent density matrices (set ntau = 1 in set_lattice for one
 * gamma per k); dK has the layout of Sigma.  exchange_begin is followed by sigma_push_pairs ... sigma_end (or
 * sigma_abort) exactly as sigma_begin is; exchange_eval = begin + one push of all pairs + end.                       */
int gwsig_exchange_begin(gwsig_ctx* ctx, const void* dGamma, void* dK, void* stream);
int gwsig_exchange_eval(gwsig_ctx* ctx, const void* dGamma, const void* dV_all, void* dK, void* stream);

/* ---- N2 (second half): the Hartree self-energy J^k -------------------------------------------
 * J^k_ij = (1/Nk) sum_{k'} sum_{ab} sum_Q V^{kk}_{ij}(Q) gamma^{k'}_{ab} V^{k'k'}_{ba}(Q)      (Eq. 21b), one spin channel
 * (the sum over sigma_1 is a factor the caller applies), gamma^k = G^k(tau = 0^-).  Two HBM-bound kernels: the
 * auxiliary density rho_Q = (1/Nk) sum_{k'} tr[gamma^{k'} V^{k'k'}(Q)] (one CTA per Q, fixed summation order: bit-reproducible), then
 * J^k = sum_Q V^{kk}(Q) rho_Q.  Orbital basis, ALL Nk points of the mesh in the order of the k index, whatever the context's mode
 * (only set_lattice is needed; no symmetry is used):
 *   dGamma (dev, in) [Nk][nao][nao]      dVdiag (dev, in) [Nk][naux][nao][nao] = V^{kk}_{Q,ij}      dJ (dev, out) [Nk][nao][nao]
 * complex128, caller-owned.  Asynchronous on `stream`.  Errors: GWSIG_ERR_ARG (NULL pointer, no lattice), GWSIG_ERR_ORDER
 * (an evaluation is open), GWSIG_ERR_CUDA.                                                                                  */
int gwsig_hartree_eval(gwsig_ctx* ctx, const void* dGamma, const void* dVdiag, void* dJ, void* stream);

/* ---- N3: the auxiliary function P from the bare bubble ------------------------------------
 * P^q(i Omega_n) = [1 - P0^q(i Omega_n)]^{-1} P0^q(i Omega_n)  (Eq. 19a),  P^q(tau) by the inverse transform
 * (Eq. 19b), for every q of the output list (the paper does this step on the CPU with MPI).
 * The tau <-> i Omega transforms are MATRICES supplied by the caller (the paper uses sparse intermediate-representation
 * grids; on a plain grid Tb[t][n] = exp(-i Omega_n tau_t) / beta):
 *   dP0 (dev) [nq][ntau][naux][naux]   dTf (dev) [nw][ntau]   dTb (dev) [ntau][nw]   dP (dev) [nq][ntau][naux][naux]
 *   P0(i Omega_n) = sum_t Tf[n][t] P0(tau_t);   P(tau_t) = sum_n Tb[t][n] P(i Omega_n).
 * Both transforms run on the grouped engine, the solve is a batched Gauss-Jordan elimination with partial pivoting (one CTA
 * per (q, Omega) at a time).  Dense layouts only (GWSIG_FULL_BZ, GWSIG_IBZ).  Synchronises the stream; GWSIG_ERR_ARG if some
 * 1 - P0(i Omega) is singular.                                                                                       */
int gwsig_dyson_p(gwsig_ctx* ctx, const void* dP0, const void* dTf, const void* dTb, int nw, void* dP, void* stream);

/* ---- the Eq. 19a solve for callers that may not allocate -------------------------------------------------------------
 * X_m = [1 - A_m]^{-1} A_m for m < nmat (Eq. 19a: P(q, i Omega) from P0(q, i Omega); one matrix per (q, Omega)).
 * Code under CUDA graph capture, tight serving loops and harnesses that forbid cudaMalloc cannot use gwsig_dyson_p, whose
 * context grows its buffers on demand.  This entry point takes no context, calls no cudaMalloc / cudaFree and no allocating
 * library routine, and does not synchronise: it clears *d_info and launches ONE kernel on `stream`.  Its scratch (one
 * augmented matrix [n][2n] per CTA) is a file-scope `static __device__` array of GWSIG_NOALLOC_SCRATCH_BYTES that every GPU
 * which loads the library holds until the process exits; the first call on a device resolves the array's device address
 * (cudaGetSymbolAddress: no allocation, but make that first call outside stream capture).
 *   dA (dev, in)  [nmat][n][n] complex128 row-major, caller-owned, not modified unless dX == dA
 *   dX (dev, out) same shape; dX == dA (in place) is allowed, partial overlap is not
 *   d_info (dev, out, may be NULL) one int: 0, or 1 if some 1 - A_m was singular / not finite (that X_m is then undefined)
 *   stream: a stream of the CURRENT device (the caller's inputs live there); the call returns once the work is queued
 * n <= GWSIG_NOALLOC_NMAX, else GWSIG_ERR_ARG; nmat is unbounded (CTAs loop over the matrices).  ALL calls of a device share
 * the one scratch array: calls that can overlap on the GPU (different streams, or graph branches without an edge between
 * them) race -- order them on one stream or with events.  The scratch keeps the last call's contents; nothing in it has to
 * start at zero (every element read was written by the same matrix' pass).  Same elimination, pivoting rule and operation
 * order as the kernel behind gwsig_dyson_p.  On error returns GWSIG_ERR_ARG / GWSIG_ERR_CUDA and, when errbuf != NULL,
 * writes a NUL-terminated message of at most errbuf_len bytes (host).                                                    */
#define GWSIG_NOALLOC_NMAX 256
#define GWSIG_NOALLOC_SCRATCH_BYTES (16 << 20)
int gwsig_dyson_solve_noalloc(const void* dA, void* dX, int nmat, int n, void* d_info, void* stream, char* errbuf, int errbuf_len);

/* ---- N4: block-basis transform of V on the device ----------------------------------------
 * V2blk_{P,a,i} = sum_{Q,b,j} conj(Uaux^q_{Q,P}) conj(U^{k2}_{b,a}) V2_{Q,b,j} U^{k1}_{j,i}     (Eq. 27; V2 = V^{k2,k1},
 * q = k1 - k2) for pairs p0 .. p0+np-1: dV_dense (dev) holds the orbital-basis tensors [naux][nao][nao] back to back in pair
 * order, dV_packed (dev) receives the allowed blocks in the packed layout sigma_push_pairs expects (first element = first
 * element of pair p0).  Needs GWSIG_IBZ_BLOCK, set_blocks WITH U_ao / U_aux, set_triples.  Three launches of the grouped engine
 * per sub-batch of pairs (auxiliary index, first orbital index, second orbital index + packing); the paper does this step on
 * the CPU before the calculation.  Synchronises the stream.                                              
 * May be called between the gwsig_sigma_push_pairs calls of an open Sigma evaluation (V prepared on demand) if `stream`
 * is that evaluation's stream; not while a P0 evaluation is open.  */
int gwsig_block_transform_v(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV_dense, void* dV_packed, void* stream);

/* ---- N4, second half: allowed-block detection on the device ("only non-zero blocks are considered") ----
 * For pairs p0 .. p0+np-1 the Eq. 27 transform of the orbital-basis tensors is carried out for EVERY block (three grouped-GEMM
 * launches per sub-batch, the last one dense) and the largest |.| of each candidate block (p, alpha, iota) is reduced on the
 * device.  Needs GWSIG_IBZ_BLOCK and set_blocks WITH the bases U_ao, U_aux; needs NO triples: this is the call whose result the
 * caller thresholds (e.g. 1e-9 of max |V|; forbidden blocks come out below 1e-13 of it) to build the lists for gwsig_set_triples.
 *   dV_dense (dev, in)  [np][naux][nao][nao] = V^{k2,k1}_{Q,bj} back to back in pair order (as for gwsig_block_transform_v)
 *   d_maxabs (dev, out) double [np][mb_aux][mb_ao][mb_ao]: entry ((pair * mb_aux + p) * mb_ao + alpha) * mb_ao + iota, zero for block
 *                       indices a mesh point does not have; mb_aux / mb_ao >= the largest number of auxiliary / orbital blocks of
 *                       any mesh point, mb_aux * mb_ao^2 <= 6144.
 * Synchronises the stream.  Errors: GWSIG_ERR_ARG, GWSIG_ERR_ORDER, GWSIG_ERR_CUDA.                                        */
int gwsig_block_maxabs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV_dense, int mb_aux, int mb_ao, void* d_maxabs, void* stream);

/* ---- N1: bare bubble ---------------------------------------------------------------
 * P0^q_{QQ'}(tau) = -(1/Nk) sum_k sum_{abcd} V^{k,k+q}_{Q,da} G^k_{cd}(-tau) G^{k+q}_{ab}(tau) V^{k+q,k}_{Q',bc}   (Eq. 20,
 * PAPER.md:179-184; one spin channel) in the order of Algorithm 3: X1 = V G^k(-tau), X2 = V G^{k+q}(tau),
 * P0 += X1 X2, for every q of the output list (the wedge in GWSIG_IBZ mode -- "Eq. 20 is evaluated for q in IBZ",
 * every mesh point in GWSIG_FULL_BZ; GWSIG_IBZ_BLOCK is refused) and every tau of the grid, which must be
 * uniform on [0, beta]: G(-tau_n) = -G(beta - tau_n) = -G[ntau-1-n].
 *   dG   : as for sigma_begin (wedge data in IBZ mode, unfolded by Eq. 22)
 *   dV   : T = V^{k,k+q}_{Q,da} as [naux][nao][nao] per pair, pairs ordered k-major: pair = k * nq + iq, q = q_list[iq]
 *          (each push is copied once into the layout [nao][nao][naux] -- auxiliary index last -- which stages 1 and 2 address)
 *          (gwsig_get_ibz / set_output_points give the list), k over the whole mesh; the partner V^{k+q,k} is taken as the
 *          conjugate transpose (reading A7 of DESIGN.md)
 *   dP0  : [nq][ntau][naux][naux], written by p0_end
 * p0_push_pairs takes ranges in increasing order without gaps, like sigma_push_pairs; p0_eval = begin + one push + end.  */
int gwsig_p0_begin(gwsig_ctx* ctx, const void* dG, void* dP0, void* stream);
int gwsig_p0_push_pairs(gwsig_ctx* ctx, int64_t p0, int64_t np, const void* dV);
int gwsig_p0_end(gwsig_ctx* ctx);
int gwsig_p0_eval(gwsig_ctx* ctx, const void* dG, const void* dV_all, void* dP0, void* stream);

/* ---- options and accounting ------------------------------------------------------------------ */
/* keys: "engine" (gwsig_engine), "hermitize" (0/1, default 0), "scratch_mib" (X+Y scratch budget,
 * default 8192), "tau_chunk" (0 = from the budget), "v_ring_mib" (size of one slot of the
 * V ring of sigma_eval_host, default 1024), "timing" (0/1: record a CUDA event pair around
 * every kernel launch on the launching stream, read back with gwsig_kernel_times),
 * "bulk_copies" (0/1, default 0): 1 = the 3M kernel stages operands that are whole contiguous rows (stage 2: X, W;
 * stage 3: V2) with cp.async.bulk (UBLKCP) instead of 16-byte cp.async -- measured slower on B200 (one bulk copy per 2 KB
 * row issues at ~130 cycles), kept for comparison,
 * "deterministic" (0/1, default 0): 1 = the split-K parts of stage 3 write private partial tiles that are summed into
 * Sigma in a fixed order by a reduction kernel instead of FP64 atomics in scheduler order: results are then bit-identical
 * from run to run (same device, same options); costs one extra pass over the partial tiles                         */
int gwsig_set_option(gwsig_ctx* ctx, const char* key, int64_t value);
/* real flops (8 per complex multiply-add) of one evaluation: the full-BZ dense equivalent
 * Nk^2 ntau 8(2A+B) and what the current mode's plan actually asks for.
 * In IBZ_BLOCK mode `executed` needs set_triples first.                                            */
int gwsig_flop_counts(gwsig_ctx* ctx, double* full_bz_equiv, double* executed);
/* number of kernel launches of the last evaluation                                                 */
int gwsig_last_launch_count(gwsig_ctx* ctx, int64_t* launches);
/* device time (ms, CUDA events on the launching stream) and launch count per kernel kind of the last
 * evaluation; ms[GWSIG_NKINDS], launches[GWSIG_NKINDS] (host).  Needs option "timing" = 1; blocks
 * until the last recorded event has completed.                                                     */
int gwsig_kernel_times(gwsig_ctx* ctx, double* ms, int64_t* launches);

/* ---- plan introspection (host-only; used by the CPU tests of the host logic) -------------------
 * stage: 51 = a grid transform of gwsig_dyson_p (np = n_in, nt = n_out); 41, 42, 43 = the three steps of the Eq. 27 transform (gwsig_block_transform_v); 31, 32, 33 = the three stages of the bare bubble (p0 / np then count P0 pairs); 11, 12 / 21, 22 = the two launches of
 * the Eq. 28 block unfold of G / W (p0 = first mesh point, np = number of points); 1 = X = V G lowered transposed, X^T = G^T conj(V2) (A = G, B = V2, C = X), 2 = Y = W X lowered transposed, Y^T = X^T W (A = X,
 * B = W, C = Y), 3 = Sigma += Y V (A = Y, B = V2, C = Sigma accumulator; the segment list of an
 * output block may be cut into several problems that add into the same C).
 * Descriptors are the structs of include/gwsig_plan.h; offsets are in complex elements relative
 * to the operand bases documented there.                                                           */
int gwsig_plan_counts(gwsig_ctx* ctx, int64_t p0, int64_t np, int nt, int stage, int64_t* nproblems, int64_t* nsegs,
                      int64_t* ntiles);
int gwsig_plan_get(gwsig_ctx* ctx, int64_t p0, int64_t np, int nt, int stage, void* problems_out, void* segs_out);

/* ---- FP64 peak probe (measurement support; needs a device) -------------------------------------
 * kind 0: register-only mma.sync.m8n8k4.f64 issue-rate loop; kind 1: register-only DFMA loop;
 * kind 2: both interleaved in every warp (tells whether DMMA and DFMA share one pipe); kind 3: one
 * dependent DMMA chain per warp (with 4 warps per block and 1 block per SM: the DMMA latency).
 * Returns achieved TFLOP/s over `iters` inner iterations on every SM (CUDA-event timed).           */
int gwsig_probe_fp64(gwsig_ctx* ctx, int kind, int warps_per_block, int blocks_per_sm, int64_t iters,
                     double* tflops, double* ms);

#ifdef __cplusplus
}
#endif
#endif /* GWSIG_H */
