// Host plan of the GW self-energy evaluation (step a0 of DESIGN.md): k maps, stars, pair list,
// packed layouts, and the lowering of Algorithm 4 to grouped-GEMM descriptors.
// Pure host C++ (no CUDA calls) so that it can be exercised without a device.
#pragma once
#include <complex>
#include <cstdint>
#include <string>
#include <vector>

#include "gwsig.h"
#include "gwsig_plan.h"

namespace gwsig {

typedef std::complex<double> cplx;

// deterministic stage 3: the split-K parts of one Sigma block write private partial tiles [part][M][N] (contiguous),
// summed into the accumulator in part order by reduce_parts_kernel
struct RedGroup {
  long long c_off;      // Sigma accumulator offset of the block (before t0 * sts)
  long long sts;        // elements per tau in the accumulator
  long long part_off;   // first partial tile in the scratch buffer
  int ni, M, nparts, pad_;
};

struct StagePlan {
  std::vector<RedGroup> red;      // only for stage 3 in deterministic mode
  long long partial_elems = 0;
  std::vector<gwsig_problem> prob;
  std::vector<gwsig_seg> seg;
  std::vector<int> bucket;    // bucket[t >> 6] = problem holding tile (t & ~63)   (zgemm_grouped.cuh)
  long long ntiles = 0;
};

struct Plan {
  // ---- lattice / sizes -------------------------------------------------------------------
  double a[9] = {0};
  int N[3] = {0, 0, 0};
  int nk = 0, nao = 0, naux = 0, ntau = 0, natom = 0;
  double beta = 0;
  std::vector<double> pos;
  std::vector<int> ao_atom, aux_atom;
  bool have_lattice = false, have_atoms = false, have_sym = false, have_blocks = false, have_triples = false;

  // ---- symmetry ---------------------------------------------------------------------------
  int nops = 0, mode = GWSIG_FULL_BZ;
  int tile_m[4] = {128, 128, 128, 128};   // tile height per launch kind: [0] Eq. 28 unfold, [1..3] contraction stage (the engine
                                          // chosen for that stage fixes it: zgemm_grouped.cuh)
  bool deterministic = false;  // stage 3 without atomics: private partial tiles + an ordered reduction (option "deterministic")
  std::vector<int> rot;        // [nops][9]
  std::vector<double> trans;   // [nops][3]
  std::vector<double> D_ao, D_aux;
  std::vector<int> shift;      // [nops][natom][3]
  std::vector<int> rotk;       // [nops][nk]   k~ = k W^-1
  std::vector<int> ir_list, ir_of, op_of, ir_index;   // ir_index[k] = position in ir_list or -1
  std::vector<int> out_list;   // k1 values Sigma is produced for (wedge or all k)
  int nk1 = 0;
  long long npairs = 0;

  // ---- blocks (IBZ_BLOCK) -------------------------------------------------------------------
  std::vector<std::vector<int>> ao_off, aux_off;     // per k: nblk+1 offsets (trivial {0,n} in dense modes)
  std::vector<cplx> U_ao, U_aux;                     // optional explicit gauge (set_blocks with U)
  bool general_gauge = false;                        // O_block != 1 somewhere: packed G / W must be unfolded (Eq. 28)
  bool have_U = false;                               // set_blocks was given U (needed by the Eq. 27 transform, N4)
  // O_block = U^{k'}^dagger O^{k_I}(alpha^) U^{k_I} (Eq. 28) for op_of[k'], packed diagonal blocks per mesh
  // point (block b of point k at oblk_*_off[k] + blk_off(b), row-major); only in the explicit gauge
  std::vector<cplx> oblk_ao, oblk_aux;
  std::vector<long long> oblk_ao_off, oblk_aux_off;  // [nk + 1]
  std::vector<long long> gu_off;                     // [nk + 1] unfolded packed G over the whole mesh (elements, all tau)
  std::vector<long long> triple_ptr;                 // [npairs+1]
  std::vector<int32_t> triples;                      // [3*nt]

  // ---- packed layouts (complex elements) --------------------------------------------------------
  std::vector<long long> g_in_off, w_in_off;   // per wedge/mesh point of the INPUT G / W buffers
  std::vector<long long> sig_off;              // per out_list entry
  std::vector<long long> v_off;                // [npairs+1]
  long long g_elems = 0, w_elems = 0, sig_elems = 0;

  std::string err;

  // mesh arithmetic
  int kindex(int n0, int n1, int n2) const;
  int ksub(int k, int q) const;
  void kcoords(int k, int n[3]) const;

  int set_lattice(const double a_[9], const int mesh[3], int nao_, int naux_, int ntau_, double beta_);
  int set_atoms(int natom_, const double* pos_, const int* ao_atom_, const int* aux_atom_);
  int set_symmetry(int nops_, const int* rot_, const double* trans_, const double* D_ao_, const double* D_aux_,
                   const int* shift_, int mode_);
  int set_blocks(const int* nblk_ao, const int* ao_block_off, const int* nblk_aux, const int* aux_block_off,
                 const double* U_ao_, const double* U_aux_);
  int set_output_points(int n, const int* k_list);
  int set_triples(int64_t npairs_, const int64_t* triple_ptr_, const int32_t* triples_);
  int finalize_layouts();

  // pair decomposition (q-major)
  void pair(long long p, int& k1, int& k2, int& q, int& i1) const {
    q = (int)(p / nk1);
    i1 = (int)(p % nk1);
    k1 = out_list[i1];
    k2 = ksub(k1, q);
  }
  // triples of a pair: explicit in block mode, the single dense triple (0,0,0) otherwise
  int pair_ntriples(long long p) const { return mode == GWSIG_IBZ_BLOCK ? (int)(triple_ptr[p + 1] - triple_ptr[p]) : 1; }
  void pair_triple(long long p, int t, int& bp, int& ba, int& bi) const {
    if (mode == GWSIG_IBZ_BLOCK) {
      const int32_t* T = &triples[3 * (triple_ptr[p] + t)];
      bp = T[0]; ba = T[1]; bi = T[2];
    } else { bp = ba = bi = 0; }
  }
  long long xsize(long long p) const { return v_off[p + 1] - v_off[p]; }   // X, Y and V2 share the shape

  // where the contraction reads G(k2) / W(q) from and with what tau stride.  q_first: first q held by
  // the W ring (IBZ dense mode).
  void g_source(int k2, long long& off, long long& tstride) const;
  void w_source(int q, int q_first, long long& off, long long& tstride) const;

  // lowering to descriptors; stage 1..3 as in gwsig_plan_get()
  // split_k > 1 cuts the segment list of every stage-3 problem into that many parts (separate problems that add
  // into the same Sigma block); 0 = choose so that the launch has enough tiles for `num_sms` SMs
  int build_stage(long long p0, long long np, int nt, int stage, int q_first, StagePlan& out, int num_sms = 148) const;
  // Eq. 28 unfold of packed diagonal blocks for mesh points [k_first, k_first + k_count), all tau, as two grouped GEMMs:
  //   step 1  T(tau) = X^{k_I}(tau) O_block^dagger     (A = packed wedge input, B = O_block, C = scratch T)
  //   step 2  X^{k'}(tau) = O_block T(tau)             (A = T, B = O_block, C = unfolded buffer)
  // aux = false: G with the orbital blocks, true: W with the auxiliary blocks.  T and the unfolded buffer share one layout:
  // point-major from k_first, [tau][packed blocks].
  int build_unfold(bool aux, int k_first, int k_count, int step, StagePlan& out) const;
  long long unfolded_elems(bool aux, int k_first, int k_count) const;
  int compute_oblock(bool aux);
  void flop_counts(double& full_equiv, double& executed) const;

  // ---- N1: bare bubble P0^q(tau), Eq. 20 / Algorithm 3, dense modes -------------------------
  // pairs are k-major: pair = k * nk1 + iq, q = out_list[iq] (the wedge in the IBZ mode), kq = k + q; the caller supplies
  // T = V^{k,k+q}_{Q,da} [naux][nao][nao] per pair (its partner V^{k+q,k} is the conjugate transpose, reading A7)
  int kadd(int k, int q) const;
  void p0_pair(long long p, int& k, int& q, int& kq, int& iq) const {
    k = (int)(p / nk1); iq = (int)(p % nk1); q = out_list[iq]; kq = kadd(k, q);
  }
  // stage 1: X1[(c,a)][Q] = sum_d Grev^k[c,d] T[Q,d,a]   (Grev(tau_n) = G(beta - tau_n): G(-tau) = -Grev, sign in the epilogue)
  // stage 2: X2[(c,a)][Q'] = sum_b G^{kq}[a,b] conj(T[Q',c,b])
  // stage 3: P0acc[iq][tau][Q][Q'] += sum over the pairs of the range with that q, sum_{(c,a)} X1[(c,a)][Q] X2[(c,a)][Q']
  // ---- N4: Eq. 27 on the device: dense orbital-basis V2 of pairs p0.. -> packed block-basis V2 (allowed triples)
  //   step 1  T1[P][(b,j)] = sum_Q conj(Uaux^q[Q,P]) V2[Q][(b,j)]      step 2  T2[P][a][j] = sum_b conj(U^{k2}[b,a]) T1[P][b][j]
  //   step 3  packed(P,a,i) = sum_j T2[P][a][j] U^{k1}[j,i]   for the allowed triples only, written in the packed layout
  // A: dense V2 / T1 / T2 (pair l at l * naux * nao^2), B: the U_aux table (step 1) or the U_ao table (steps 2, 3), [Nk][n][n]
  int build_vtransform(long long p0, long long np, int step, StagePlan& out) const;
  // ---- N3 (Eq. 19): dst[q][o][m] = sum_i T[o][i] src[q][i][m] for nq momenta, m over naux^2 (tau <-> i Omega transforms as GEMMs)
  int build_gridtransform(int nq, int nin, int nout, StagePlan& out) const;
  int build_p0_stage(long long p0, long long np, int nt, int stage, StagePlan& out, int num_sms = 148) const;
};

static inline long long sumsq(const std::vector<int>& off) {
  long long s = 0;
  for (size_t b = 0; b + 1 < off.size(); ++b) s += (long long)(off[b + 1] - off[b]) * (off[b + 1] - off[b]);
  return s;
}

}  // namespace gwsig
