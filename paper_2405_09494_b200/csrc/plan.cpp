// Host plan (step a0): see plan.hpp.  Citations are PAPER.md lines of arXiv 2405.09494.
#include "plan.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

#include "zgemm_grouped.cuh"

namespace gwsig {

int Plan::kindex(int n0, int n1, int n2) const {
  auto md = [](int v, int m) { int r = v % m; return r < 0 ? r + m : r; };
  return (md(n0, N[0]) * N[1] + md(n1, N[1])) * N[2] + md(n2, N[2]);
}
void Plan::kcoords(int k, int n[3]) const {
  n[2] = k % N[2];
  n[1] = (k / N[2]) % N[1];
  n[0] = k / (N[1] * N[2]);
}
int Plan::ksub(int k, int q) const {
  int a_[3], b_[3];
  kcoords(k, a_);
  kcoords(q, b_);
  return kindex(a_[0] - b_[0], a_[1] - b_[1], a_[2] - b_[2]);
}

int Plan::kadd(int k, int q) const {
  int a_[3], b_[3];
  kcoords(k, a_);
  kcoords(q, b_);
  return kindex(a_[0] + b_[0], a_[1] + b_[1], a_[2] + b_[2]);
}

int Plan::set_lattice(const double a_[9], const int mesh[3], int nao_, int naux_, int ntau_, double beta_) {
  if (!a_ || !mesh) { err = "set_lattice: NULL argument"; return GWSIG_ERR_ARG; }
  if (mesh[0] < 1 || mesh[1] < 1 || mesh[2] < 1 || nao_ < 1 || naux_ < 1 || ntau_ < 1) {
    err = "set_lattice: mesh, nao, naux and ntau must be positive"; return GWSIG_ERR_ARG;
  }
  if ((long long)mesh[0] * mesh[1] * mesh[2] > (1 << 20)) { err = "set_lattice: mesh too large"; return GWSIG_ERR_ARG; }
  std::memcpy(a, a_, sizeof(a));
  for (int i = 0; i < 3; ++i) N[i] = mesh[i];
  nk = mesh[0] * mesh[1] * mesh[2];
  nao = nao_; naux = naux_; ntau = ntau_; beta = beta_;
  have_lattice = true;
  have_atoms = have_sym = have_blocks = have_triples = false;
  return GWSIG_OK;
}

int Plan::set_atoms(int natom_, const double* pos_, const int* ao_atom_, const int* aux_atom_) {
  if (!have_lattice) { err = "set_atoms: call set_lattice first"; return GWSIG_ERR_ARG; }
  if (natom_ < 1 || !pos_ || !ao_atom_ || !aux_atom_) { err = "set_atoms: bad argument"; return GWSIG_ERR_ARG; }
  for (int i = 0; i < nao; ++i)
    if (ao_atom_[i] < 0 || ao_atom_[i] >= natom_) { err = "set_atoms: ao_atom out of range"; return GWSIG_ERR_ARG; }
  for (int i = 0; i < naux; ++i)
    if (aux_atom_[i] < 0 || aux_atom_[i] >= natom_) { err = "set_atoms: aux_atom out of range"; return GWSIG_ERR_ARG; }
  natom = natom_;
  pos.assign(pos_, pos_ + 3 * natom_);
  ao_atom.assign(ao_atom_, ao_atom_ + nao);
  aux_atom.assign(aux_atom_, aux_atom_ + naux);
  have_atoms = true;
  have_sym = have_blocks = have_triples = false;
  return GWSIG_OK;
}

static bool int_inverse(const int* W, int* Winv) {
  long long d = (long long)W[0] * (W[4] * W[8] - W[5] * W[7]) - (long long)W[1] * (W[3] * W[8] - W[5] * W[6]) +
                (long long)W[2] * (W[3] * W[7] - W[4] * W[6]);
  if (d != 1 && d != -1) return false;
  int c[9] = {W[4] * W[8] - W[5] * W[7], W[2] * W[7] - W[1] * W[8], W[1] * W[5] - W[2] * W[4],
              W[5] * W[6] - W[3] * W[8], W[0] * W[8] - W[2] * W[6], W[2] * W[3] - W[0] * W[5],
              W[3] * W[7] - W[4] * W[6], W[1] * W[6] - W[0] * W[7], W[0] * W[4] - W[1] * W[3]};
  for (int i = 0; i < 9; ++i) Winv[i] = (int)(c[i] * d);
  return true;
}

static bool orthogonal(const double* D, int n) {
  for (int i = 0; i < n; ++i)
    for (int j = i; j < n; ++j) {
      double s = 0;
      for (int k = 0; k < n; ++k) s += D[(size_t)i * n + k] * D[(size_t)j * n + k];
      if (std::fabs(s - (i == j ? 1.0 : 0.0)) > 1e-8) return false;
    }
  return true;
}

int Plan::set_symmetry(int nops_, const int* rot_, const double* trans_, const double* D_ao_, const double* D_aux_,
                       const int* shift_, int mode_) {
  if (!have_lattice) { err = "set_symmetry: call set_lattice first"; return GWSIG_ERR_ARG; }
  if (mode_ != GWSIG_FULL_BZ && mode_ != GWSIG_IBZ && mode_ != GWSIG_IBZ_BLOCK) { err = "set_symmetry: bad mode"; return GWSIG_ERR_ARG; }
  if (nops_ < 0 || (nops_ == 0 && mode_ != GWSIG_FULL_BZ)) { err = "set_symmetry: nops = 0 needs GWSIG_FULL_BZ"; return GWSIG_ERR_ARG; }
  if (nops_ > 0 && (!rot_ || !trans_ || !D_ao_ || !D_aux_ || !shift_ || !have_atoms)) {
    err = "set_symmetry: NULL argument or set_atoms not called"; return GWSIG_ERR_ARG;
  }
  mode = mode_;
  if (nops_ == 0) {            // no symmetry: identity only
    nops = 1;
    rot = {1, 0, 0, 0, 1, 0, 0, 0, 1};
    trans = {0, 0, 0};
    if (!have_atoms) { natom = 1; ao_atom.assign(nao, 0); aux_atom.assign(naux, 0); pos = {0, 0, 0}; have_atoms = true; }
    shift.assign((size_t)3 * natom, 0);
    D_ao.assign((size_t)nao * nao, 0.0);
    for (int i = 0; i < nao; ++i) D_ao[(size_t)i * nao + i] = 1.0;
    D_aux.assign((size_t)naux * naux, 0.0);
    for (int i = 0; i < naux; ++i) D_aux[(size_t)i * naux + i] = 1.0;
  } else {
    nops = nops_;
    rot.assign(rot_, rot_ + 9 * (size_t)nops);
    trans.assign(trans_, trans_ + 3 * (size_t)nops);
    D_ao.assign(D_ao_, D_ao_ + (size_t)nops * nao * nao);
    D_aux.assign(D_aux_, D_aux_ + (size_t)nops * naux * naux);
    shift.assign(shift_, shift_ + (size_t)nops * natom * 3);
    for (int g = 0; g < nops; ++g) {
      if (!orthogonal(&D_ao[(size_t)g * nao * nao], nao) || !orthogonal(&D_aux[(size_t)g * naux * naux], naux)) {
        err = "set_symmetry: representation matrix of operation " + std::to_string(g) + " is not orthogonal";
        return GWSIG_ERR_SYMMETRY;
      }
    }
  }
  // k~ = k W^-1 (row vector) on mesh indices; must stay on the mesh
  rotk.assign((size_t)nops * nk, 0);
  for (int g = 0; g < nops; ++g) {
    int Winv[9];
    if (!int_inverse(&rot[9 * g], Winv)) { err = "set_symmetry: rotation " + std::to_string(g) + " is not unimodular"; return GWSIG_ERR_SYMMETRY; }
    for (int k = 0; k < nk; ++k) {
      int n[3], out[3];
      kcoords(k, n);
      for (int j = 0; j < 3; ++j) {
        long long acc = 0;
        for (int i = 0; i < 3; ++i) {
          long long t = (long long)n[i] * Winv[3 * i + j] * N[j];
          if (t % N[i] != 0) { err = "set_symmetry: rotation " + std::to_string(g) + " does not map the k mesh onto itself"; return GWSIG_ERR_SYMMETRY; }
          acc += t / N[i];
        }
        long long r = acc % N[j];
        out[j] = (int)(r < 0 ? r + N[j] : r);
      }
      rotk[(size_t)g * nk + k] = kindex(out[0], out[1], out[2]);
    }
    // a rotation must permute the mesh
    std::vector<char> seen(nk, 0);
    for (int k = 0; k < nk; ++k) seen[rotk[(size_t)g * nk + k]] = 1;
    for (int k = 0; k < nk; ++k)
      if (!seen[k]) { err = "set_symmetry: rotation " + std::to_string(g) + " is not a permutation of the mesh"; return GWSIG_ERR_SYMMETRY; }
  }
  // stars: representative = first member in index order; op_of = first op mapping it there
  ir_of.assign(nk, -1); op_of.assign(nk, -1); ir_index.assign(nk, -1); ir_list.clear();
  for (int k = 0; k < nk; ++k) {
    if (ir_of[k] >= 0) continue;
    ir_index[k] = (int)ir_list.size();
    ir_list.push_back(k);
    for (int g = 0; g < nops; ++g) {
      int kp = rotk[(size_t)g * nk + k];
      if (ir_of[kp] < 0) { ir_of[kp] = k; op_of[kp] = g; }
    }
  }
  if (op_of[ir_list[0]] != 0 && nops > 0) {
    // the first operation must be the identity for op_of[representative] to be the identity
    for (int k : ir_list)
      if (rotk[(size_t)op_of[k] * nk + k] != k) { err = "set_symmetry: internal star error"; return GWSIG_ERR_SYMMETRY; }
  }
  out_list.clear();
  if (mode == GWSIG_FULL_BZ) { out_list.resize(nk); std::iota(out_list.begin(), out_list.end(), 0); }
  else out_list = ir_list;
  nk1 = (int)out_list.size();
  npairs = (long long)nk * nk1;
  // trivial (one-block) maps; set_blocks overrides them in IBZ_BLOCK mode
  ao_off.assign(nk, std::vector<int>{0, nao});
  aux_off.assign(nk, std::vector<int>{0, naux});
  U_ao.clear(); U_aux.clear(); general_gauge = false; have_U = false;
  have_sym = true;
  have_blocks = have_triples = false;
  triple_ptr.clear(); triples.clear();
  return finalize_layouts();
}

int Plan::set_output_points(int n, const int* k_list) {
  if (!have_sym) { err = "set_output_points: call set_symmetry first"; return GWSIG_ERR_ARG; }
  if (n < 1 || n > nk || !k_list) { err = "set_output_points: bad count or NULL list"; return GWSIG_ERR_ARG; }
  std::vector<char> seen(nk, 0);
  for (int i = 0; i < n; ++i) {
    const int k = k_list[i];
    if (k < 0 || k >= nk || seen[k]) { err = "set_output_points: point out of range or repeated"; return GWSIG_ERR_ARG; }
    if (mode != GWSIG_FULL_BZ && ir_index[k] < 0) { err = "set_output_points: point " + std::to_string(k) + " is not a wedge representative"; return GWSIG_ERR_ARG; }
    seen[k] = 1;
  }
  out_list.assign(k_list, k_list + n);
  nk1 = n;
  npairs = (long long)nk * nk1;
  have_triples = false;
  triple_ptr.clear(); triples.clear();
  return finalize_layouts();
}

int Plan::set_blocks(const int* nblk_ao, const int* ao_block_off, const int* nblk_aux, const int* aux_block_off,
                     const double* U_ao_, const double* U_aux_) {
  if (!have_sym || mode != GWSIG_IBZ_BLOCK) { err = "set_blocks: needs set_symmetry with GWSIG_IBZ_BLOCK"; return GWSIG_ERR_ARG; }
  if (!nblk_ao || !ao_block_off || !nblk_aux || !aux_block_off) { err = "set_blocks: NULL argument"; return GWSIG_ERR_ARG; }
  if ((U_ao_ == nullptr) != (U_aux_ == nullptr)) { err = "set_blocks: give both U_ao and U_aux or neither"; return GWSIG_ERR_ARG; }
  auto read = [&](const int* nblk, const int* offs, int n, std::vector<std::vector<int>>& out, const char* what) -> int {
    out.assign(nk, {});
    size_t pos_ = 0;
    for (int k = 0; k < nk; ++k) {
      if (nblk[k] < 1 || nblk[k] > n) { err = std::string("set_blocks: bad block count (") + what + ")"; return GWSIG_ERR_BLOCKS; }
      out[k].assign(offs + pos_, offs + pos_ + nblk[k] + 1);
      pos_ += nblk[k] + 1;
      if (out[k].front() != 0 || out[k].back() != n) { err = std::string("set_blocks: blocks do not tile [0,n) (") + what + ")"; return GWSIG_ERR_BLOCKS; }
      for (size_t b = 0; b + 1 < out[k].size(); ++b)
        if (out[k][b + 1] <= out[k][b]) { err = std::string("set_blocks: block offsets not increasing (") + what + ")"; return GWSIG_ERR_BLOCKS; }
    }
    for (int k = 0; k < nk; ++k)
      if (out[k] != out[ir_of[k]]) { err = std::string("set_blocks: star member's blocks differ from its representative's (") + what + ")"; return GWSIG_ERR_BLOCKS; }
    return GWSIG_OK;
  };
  int rc = read(nblk_ao, ao_block_off, nao, ao_off, "ao");
  if (rc) return rc;
  rc = read(nblk_aux, aux_block_off, naux, aux_off, "aux");
  if (rc) return rc;
  general_gauge = U_ao_ != nullptr;
  if (general_gauge) {
    const cplx* ua = reinterpret_cast<const cplx*>(U_ao_);
    const cplx* ux = reinterpret_cast<const cplx*>(U_aux_);
    U_ao.assign(ua, ua + (size_t)nk * nao * nao);
    U_aux.assign(ux, ux + (size_t)nk * naux * naux);
    if ((rc = compute_oblock(false))) return rc;
    if ((rc = compute_oblock(true))) return rc;
    // U given in the gauge U^{k'} = O U^{k_I}: every O_block is the identity and nothing has to be unfolded
    auto is_identity = [&](const std::vector<cplx>& ob, const std::vector<long long>& oo, const std::vector<std::vector<int>>& offs) {
      for (int k = 0; k < nk; ++k) {
        long long o = oo[k];
        for (size_t b = 0; b + 1 < offs[k].size(); ++b) {
          const int nb = offs[k][b + 1] - offs[k][b];
          for (int r = 0; r < nb; ++r)
            for (int c = 0; c < nb; ++c)
              if (std::abs(ob[(size_t)o + (size_t)r * nb + c] - cplx(r == c ? 1.0 : 0.0, 0.0)) > 1e-10) return false;
          o += (long long)nb * nb;
        }
      }
      return true;
    };
    if (is_identity(oblk_ao, oblk_ao_off, ao_off) && is_identity(oblk_aux, oblk_aux_off, aux_off)) general_gauge = false;
  } else { U_ao.clear(); U_aux.clear(); oblk_ao.clear(); oblk_aux.clear(); }
  have_U = U_ao_ != nullptr;
  have_blocks = true;
  have_triples = false;
  triple_ptr.clear(); triples.clear();
  return finalize_layouts();
}

int Plan::set_triples(int64_t npairs_, const int64_t* triple_ptr_, const int32_t* triples_) {
  if (!have_blocks || mode != GWSIG_IBZ_BLOCK) { err = "set_triples: needs set_blocks in GWSIG_IBZ_BLOCK mode"; return GWSIG_ERR_ARG; }
  if (npairs_ != npairs || !triple_ptr_ || (!triples_ && triple_ptr_[npairs_] > 0)) { err = "set_triples: wrong pair count or NULL argument"; return GWSIG_ERR_ARG; }
  if (triple_ptr_[0] != 0) { err = "set_triples: triple_ptr[0] must be 0"; return GWSIG_ERR_BLOCKS; }
  for (long long p = 0; p < npairs; ++p) {
    if (triple_ptr_[p + 1] < triple_ptr_[p]) { err = "set_triples: triple_ptr not monotone"; return GWSIG_ERR_BLOCKS; }
    int k1, k2, q, i1;
    pair(p, k1, k2, q, i1);
    int prev = -1;
    for (long long t = triple_ptr_[p]; t < triple_ptr_[p + 1]; ++t) {
      const int32_t* T = triples_ + 3 * t;
      if (T[0] < 0 || T[0] >= (int)aux_off[q].size() - 1 || T[1] < 0 || T[1] >= (int)ao_off[k2].size() - 1 || T[2] < 0 ||
          T[2] >= (int)ao_off[k1].size() - 1) { err = "set_triples: block index out of range at pair " + std::to_string(p); return GWSIG_ERR_BLOCKS; }
      if (T[0] < prev) { err = "set_triples: triples of a pair must be sorted by aux block"; return GWSIG_ERR_BLOCKS; }
      prev = T[0];
    }
  }
  triple_ptr.assign(triple_ptr_, triple_ptr_ + npairs + 1);
  triples.assign(triples_, triples_ + 3 * triple_ptr_[npairs]);
  have_triples = true;
  return finalize_layouts();
}

int Plan::finalize_layouts() {
  const bool blk = mode == GWSIG_IBZ_BLOCK;
  // input G / W: per wedge point (IBZ modes) or per mesh point (FULL_BZ), packed blocks in block mode
  std::vector<int> all_k(nk);
  std::iota(all_k.begin(), all_k.end(), 0);
  const std::vector<int>& pts = mode == GWSIG_FULL_BZ ? all_k : ir_list;     // inputs do not depend on the output points
  g_in_off.assign(pts.size() + 1, 0);
  w_in_off.assign(pts.size() + 1, 0);
  for (size_t i = 0; i < pts.size(); ++i) {
    long long gs = blk ? sumsq(ao_off[pts[i]]) : (long long)nao * nao;
    long long ws = blk ? sumsq(aux_off[pts[i]]) : (long long)naux * naux;
    g_in_off[i + 1] = g_in_off[i] + gs * ntau;
    w_in_off[i + 1] = w_in_off[i] + ws * ntau;
  }
  g_elems = g_in_off.back();
  w_elems = w_in_off.back();
  gu_off.assign(nk + 1, 0);
  for (int k = 0; k < nk; ++k) gu_off[k + 1] = gu_off[k] + (blk ? sumsq(ao_off[k]) : (long long)nao * nao) * ntau;
  sig_off.assign(nk1 + 1, 0);
  for (int i = 0; i < nk1; ++i)
    sig_off[i + 1] = sig_off[i] + (blk ? sumsq(ao_off[out_list[i]]) : (long long)nao * nao) * ntau;
  sig_elems = sig_off.back();
  v_off.clear();
  if (!blk) {
    v_off.resize(npairs + 1);
    for (long long p = 0; p <= npairs; ++p) v_off[p] = p * (long long)naux * nao * nao;
  } else if (have_triples) {
    v_off.assign(npairs + 1, 0);
    for (long long p = 0; p < npairs; ++p) {
      int k1, k2, q, i1;
      pair(p, k1, k2, q, i1);
      long long s = 0;
      for (long long t = triple_ptr[p]; t < triple_ptr[p + 1]; ++t) {
        const int32_t* T = &triples[3 * t];
        s += (long long)(aux_off[q][T[0] + 1] - aux_off[q][T[0]]) * (ao_off[k2][T[1] + 1] - ao_off[k2][T[1]]) *
             (ao_off[k1][T[2] + 1] - ao_off[k1][T[2]]);
      }
      v_off[p + 1] = v_off[p] + s;
    }
  }
  return GWSIG_OK;
}

void Plan::g_source(int k2, long long& off, long long& tstride) const {
  if (mode == GWSIG_IBZ_BLOCK) {
    tstride = sumsq(ao_off[k2]);
    if (general_gauge) off = gu_off[k2];                  // unfolded packed buffer over the whole mesh, mesh order (Eq. 28)
    else off = g_in_off[ir_index[ir_of[k2]]];            // S5 gauge: data of the representative
  } else {
    tstride = (long long)nao * nao;
    off = (long long)k2 * ntau * tstride;               // dG itself (FULL_BZ) or the unfolded buffer (IBZ)
  }
}

void Plan::w_source(int q, int q_first, long long& off, long long& tstride) const {
  if (mode == GWSIG_IBZ_BLOCK) {
    tstride = sumsq(aux_off[q]);
    if (general_gauge) {
      off = 0;
      for (int k = q_first; k < q; ++k) off += sumsq(aux_off[k]) * ntau;
    } else off = w_in_off[ir_index[ir_of[q]]];
  } else {
    tstride = (long long)naux * naux;
    off = (long long)(mode == GWSIG_FULL_BZ ? q : q - q_first) * ntau * tstride;
  }
}

static inline gwsig_idx2 lvl1(long long lo) { gwsig_idx2 d; d.hi = 0; d.lo = lo; d.div = GWSIG_NODIV; d.pad_ = 0; return d; }
static inline gwsig_idx2 lvl2(int div, long long hi, long long lo) { gwsig_idx2 d; d.hi = hi; d.lo = lo; d.div = div; d.pad_ = 0; return d; }

// ranges the tensor kernels rely on: the element offset of a tile COLUMN (relative to the tile's C base) fits 32 bits, and
// every index that goes through a TWO-LEVEL map (rows, columns, k) is below 2^22 (the kernels divide with a float reciprocal);
// single-level maps carry no such limit
static bool kernel_ranges_ok(const std::vector<gwsig_problem>& prob, const std::vector<gwsig_seg>& seg) {
  const long long lim = 1LL << 22;
  auto two = [](const gwsig_idx2& d) { return d.div != GWSIG_NODIV; };
  for (const auto& P : prob) {
    if (P.N <= 0) continue;
    if ((two(P.cm) && P.M >= lim) || (two(P.cn) && P.N >= lim)) return false;
    for (int s = P.seg_begin; s < P.seg_begin + P.seg_count; ++s) {
      const gwsig_seg& S = seg[s];
      if ((two(S.am) && P.M >= lim) || (two(S.bn) && P.N >= lim) || ((two(S.ak) || two(S.bk)) && S.K >= lim)) return false;
    }
    const long long n = P.N - 1;
    const long long off = P.cn.div == GWSIG_NODIV ? n * P.cn.lo : (n / P.cn.div) * P.cn.hi + std::min<long long>(P.cn.div - 1, n) * P.cn.lo;
    if (off < 0 || off >= (1LL << 31)) return false;
  }
  return true;
}

int Plan::build_stage(long long p0, long long np, int nt, int stage, int q_first, StagePlan& out, int num_sms) const {
  out.prob.clear(); out.seg.clear(); out.bucket.clear(); out.ntiles = 0; out.red.clear(); out.partial_elems = 0;
  if (p0 < 0 || np < 1 || p0 + np > npairs || nt < 1 || nt > ntau || stage < 1 || stage > 3) return GWSIG_ERR_ARG;
  if (v_off.empty()) return GWSIG_ERR_ARG;

  // chunk-local X / Y offsets: [pair][tau in chunk][xsize(pair)]
  std::vector<long long> xoff(np + 1, 0);
  for (long long l = 0; l < np; ++l) xoff[l + 1] = xoff[l] + xsize(p0 + l) * nt;

  struct TripleLay { int p, al, io, np_, na, ni; long long c0, poff, Np; };
  auto pair_layout = [&](long long p, std::vector<TripleLay>& T, std::vector<long long>& Np, std::vector<long long>& poff, int& k1,
                         int& k2, int& q, int& i1) {
    pair(p, k1, k2, q, i1);
    const std::vector<int>&oq = aux_off[q], &o2 = ao_off[k2], &o1 = ao_off[k1];
    int nb = (int)oq.size() - 1;
    Np.assign(nb, 0); poff.assign(nb + 1, 0);
    int ntr = pair_ntriples(p);
    T.resize(ntr);
    for (int t = 0; t < ntr; ++t) {
      int bp, ba, bi;
      pair_triple(p, t, bp, ba, bi);
      TripleLay& L = T[t];
      L.p = bp; L.al = ba; L.io = bi;
      L.np_ = oq[bp + 1] - oq[bp]; L.na = o2[ba + 1] - o2[ba]; L.ni = o1[bi + 1] - o1[bi];
      L.c0 = Np[bp];
      Np[bp] += (long long)L.na * L.ni;
    }
    for (int b = 0; b < nb; ++b) poff[b + 1] = poff[b] + (long long)(oq[b + 1] - oq[b]) * Np[b];
    for (auto& L : T) { L.poff = poff[L.p]; L.Np = Np[L.p]; }
  };
  auto blk_off = [](const std::vector<int>& off, int b) {     // offset of diagonal block b in the packed layout
    long long s = 0;
    for (int c = 0; c < b; ++c) s += (long long)(off[c + 1] - off[c]) * (off[c + 1] - off[c]);
    return s;
  };

  std::vector<TripleLay> T;
  std::vector<long long> Np, poff;
  std::vector<long long> cost;       // per problem: total K (tiles of one launch share the tile area)

  if (stage == 1 || stage == 2) {
    for (long long l = 0; l < np; ++l) {
      const long long p = p0 + l;
      int k1, k2, q, i1;
      pair_layout(p, T, Np, poff, k1, k2, q, i1);
      const long long vrel = v_off[p] - v_off[p0];
      const long long xs = xsize(p);
      if (stage == 1) {
        long long goff, gts;
        g_source(k2, goff, gts);
        for (const auto& L : T) {
          gwsig_seg S; std::memset(&S, 0, sizeof(S));
          gwsig_problem P; std::memset(&P, 0, sizeof(P));
          // X[P,i,b](tau) = sum_a conj(V2[P,a,i]) G[a,b](tau)          (Algorithm 4 line 5)
          // lowered TRANSPOSED, X^T[(tau,b),(P,i)] = sum_a G^T[(tau,b),a] conj(V2)[a,(P,i)]: tau folds into the long row
          // index (each V2 tile is read once for all tau of the chunk) and V2 is the narrow operand
          S.a_off = goff + blk_off(ao_off[k2], L.al);
          S.am = lvl2(L.na, gts, 1);                      // m = (tau, b)
          S.ak = lvl1(L.na);                              // k = a
          S.b_off = vrel + L.poff + L.c0;
          S.bk = lvl1(L.ni);
          S.bn = lvl2(L.ni, L.Np, 1);                     // n = (P, i)
          S.K = L.na;
          P.M = nt * L.na; P.N = L.np_ * L.ni;
          P.c_off = xoff[l] + L.poff + L.c0;
          // X (and Y) segments are stored [P][b][i], i fastest -- the transpose of V2's [P][a][i] in the middle index only:
          // every operand of every stage is then contiguous along its tile dimension (runs of n_alpha or n_iota elements,
          // whole rows in stage 2), which is what the bulk-copy loader wants
          P.cm = lvl2(L.na, xs, L.ni);
          P.cn = lvl2(L.ni, L.Np, 1);
          P.a_tstride = gts;
          P.nbatch = 1;
          P.flags = GWSIG_FLAG_CONJ_B;
          P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
          out.seg.push_back(S); out.prob.push_back(P); cost.push_back(S.K);
        }
      } else {
        long long woff, wts;
        w_source(q, q_first, woff, wts);
        const std::vector<int>& oq = aux_off[q];
        for (int b = 0; b + 1 < (int)oq.size(); ++b) {
          if (Np[b] == 0) continue;
          const int npb = oq[b + 1] - oq[b];
          gwsig_seg S; std::memset(&S, 0, sizeof(S));
          gwsig_problem P; std::memset(&P, 0, sizeof(P));
          // Y[P',n](tau) = sum_P W[P,P'](tau) X[P,n](tau)                (Algorithm 4 line 7)
          // lowered TRANSPOSED, Y^T[n,P'] = sum_P X^T[n,P] W[P,P']: the long index n = (iota, alpha, i, b) fills the
          // 128-row tiles and the ragged block size n_p only meets the 8-column granularity
          S.a_off = xoff[l] + poff[b];
          S.am = lvl1(1); S.ak = lvl1(Np[b]);              // A = X^T: m = column of X (contiguous), k = P
          S.b_off = woff + blk_off(oq, b);
          S.bk = lvl1(npb); S.bn = lvl1(1);                // B = W[P,P'] row-major
          S.K = npb;
          P.M = (int)Np[b]; P.N = npb;
          P.c_off = xoff[l] + poff[b];
          P.cm = lvl1(1); P.cn = lvl1(Np[b]);              // C = Y^T: element (n, P') at Y[P'][n]
          P.b_bstride = wts; P.b_tstride = wts;
          P.a_bstride = xs; P.c_bstride = xs;
          P.nbatch = nt;
          P.flags = 0;
          P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
          out.seg.push_back(S); out.prob.push_back(P); cost.push_back(S.K);
        }
      }
    }
  } else {
    // stage 3: Sigma_iota[i,j](tau) += sum over the pairs of this range with the same k1 and their triples
    //          with output block iota of  sum_{P',b} Y[P',i,b] V2[P',b,j]      (Algorithm 4 line 8, PAPER.md:347;
    //          only diagonal (iota,iota) blocks: the others cancel in the q sum -- DESIGN.md A8)
    // split-K: the segment lists are long (all pairs of the range x their triples) and the outputs few and small, so each
    // problem's list is cut into `parts` pieces of about equal K that add into the same Sigma block (FP64 atomics)
    struct P3 { gwsig_problem P; std::vector<gwsig_seg> segs; long long kt; };
    std::vector<P3> p3;
    long long tiles1 = 0;
    for (int i1 = 0; i1 < nk1; ++i1) {
      const int k1 = out_list[i1];
      const std::vector<int>& o1 = ao_off[k1];
      const int nb1 = (int)o1.size() - 1;
      std::vector<std::vector<gwsig_seg>> segs(nb1);
      long long lfirst = ((long long)i1 - (p0 % nk1) + nk1) % nk1;
      for (long long l = lfirst; l < np; l += nk1) {
        const long long p = p0 + l;
        int k1_, k2, q, i1_;
        pair_layout(p, T, Np, poff, k1_, k2, q, i1_);
        const long long vrel = v_off[p] - v_off[p0];
        const long long xs = xsize(p);
        if (xs * nt >= (1LL << 31)) return GWSIG_ERR_ARG;   // the per-element loader path keeps 32-bit row offsets
        for (const auto& L : T) {
          gwsig_seg S; std::memset(&S, 0, sizeof(S));
          S.a_off = xoff[l] + L.poff + L.c0;               // Y, same layout as X: [P'][b][i]
          S.am = lvl2(L.ni, xs, 1);                        // m = (tau, i)
          S.ak = lvl2(L.na, L.Np, L.ni);                   // k = (P', b)
          S.b_off = vrel + L.poff + L.c0;
          S.bk = lvl2(L.na, L.Np, L.ni);
          S.bn = lvl1(1);
          S.K = L.np_ * L.na;
          segs[L.io].push_back(S);
        }
      }
      long long sts = mode == GWSIG_IBZ_BLOCK ? sumsq(o1) : (long long)nao * nao;
      for (int b = 0; b < nb1; ++b) {
        if (segs[b].empty()) continue;
        const int ni = o1[b + 1] - o1[b];
        P3 x;
        std::memset(&x.P, 0, sizeof(x.P));
        x.P.M = nt * ni; x.P.N = ni;
        x.P.c_off = sig_off[i1] + blk_off(o1, b);
        x.P.cm = lvl2(ni, sts, ni); x.P.cn = lvl1(1);
        x.P.c_tstride = sts;
        x.P.nbatch = 1;
        x.P.flags = GWSIG_FLAG_ACCUM;
        x.kt = 0;
        for (auto& S : segs[b]) x.kt += S.K;
        x.segs.swap(segs[b]);
        tiles1 += (long long)zg_tiles_m(x.P.M, tile_m[3]) * zg_tiles_n(x.P.N);
        p3.push_back(std::move(x));
      }
    }
    // enough tiles for ~12 rounds of 2 CTAs per SM, pieces of at least ~512 k (measured on cfg3, ms of stage 3 for 4 / 8 / 12 / 20 /
    // 32 tiles per SM: 211 / 167 / 163 / 154.5 / 153.7)
    const long long want = 24LL * std::max(num_sms, 1);
    for (auto& x : p3) {
      long long parts = tiles1 > 0 ? (want + tiles1 - 1) / tiles1 : 1;
      parts = std::max(1LL, std::min<long long>(parts, std::max(1LL, x.kt / 512)));
      if ((long long)x.segs.size() < parts) {
        // too few segments to deal out: cut every segment along P' (k = (P', b): both operands advance by N_p per P')
        const long long r = (parts + (long long)x.segs.size() - 1) / (long long)x.segs.size();
        std::vector<gwsig_seg> cut;
        for (const auto& S : x.segs) {
          const int na = S.ak.div, npp = S.K / na;
          const long long pieces = std::min<long long>(r, npp);
          for (long long c = 0; c < pieces; ++c) {
            const int P0 = (int)(npp * c / pieces), P1 = (int)(npp * (c + 1) / pieces);
            gwsig_seg Sc = S;
            Sc.a_off += (long long)P0 * S.ak.hi;
            Sc.b_off += (long long)P0 * S.bk.hi;
            Sc.K = (P1 - P0) * na;
            cut.push_back(Sc);
          }
        }
        x.segs.swap(cut);
      }
      parts = std::min<long long>(parts, (long long)x.segs.size());
      size_t s0 = 0;
      long long kdone = 0;
      RedGroup rg;
      rg.c_off = x.P.c_off; rg.sts = x.P.c_tstride; rg.part_off = out.partial_elems; rg.ni = x.P.N; rg.M = x.P.M; rg.nparts = 0; rg.pad_ = 0;
      for (long long part = 0; part < parts; ++part) {
        const long long target = x.kt * (part + 1) / parts;
        gwsig_problem P = x.P;
        if (deterministic) {            // private partial tile [M][N], plain stores; summed in part order afterwards
          P.flags &= ~GWSIG_FLAG_ACCUM;
          P.c_off = out.partial_elems;
          P.cm = lvl1(x.P.N); P.cn = lvl1(1);
          P.c_tstride = 0;
        }
        P.seg_begin = (int)out.seg.size();
        long long kt = 0;
        while (s0 < x.segs.size() && (kdone < target || part == parts - 1)) {
          out.seg.push_back(x.segs[s0]);
          kdone += x.segs[s0].K; kt += x.segs[s0].K;
          ++s0;
        }
        P.seg_count = (int)out.seg.size() - P.seg_begin;
        if (P.seg_count == 0) continue;
        out.prob.push_back(P); cost.push_back(kt);
        if (deterministic) { out.partial_elems += (long long)x.P.M * x.P.N; ++rg.nparts; }
      }
      if (deterministic && rg.nparts > 0) out.red.push_back(rg);
    }
  }

  // range checks the kernels rely on: element offsets of A inside a tile fit 32 bits (the 4-product kernel keeps them in int),
  // a problem has fewer than 2^31 tiles, every problem has work (a C = tile without any K would never be written)
  auto span = [](const gwsig_idx2& d, long long n) -> long long {
    if (n <= 0) return 0;
    if (d.div == GWSIG_NODIV) return (n - 1) * d.lo;
    return ((n - 1) / d.div) * d.hi + std::min<long long>(d.div - 1, n - 1) * d.lo;
  };
  for (const auto& P : out.prob) {
    long long ktot = 0;
    for (int s = P.seg_begin; s < P.seg_begin + P.seg_count; ++s) {
      const gwsig_seg& S = out.seg[s];
      ktot += S.K;
      if (span(S.am, P.M) >= (1LL << 31) || span(S.bn, P.N) >= (1LL << 31)) { return GWSIG_ERR_ARG; }
    }
    if (ktot <= 0) return GWSIG_ERR_ARG;
    const long long nt_ = (long long)P.nbatch * zg_tiles_m(P.M, tile_m[stage]) * zg_tiles_n(P.N);
    if (nt_ >= (1LL << 31)) return GWSIG_ERR_ARG;
  }

  // heaviest problems first (dynamic scheduler takes tiles in order), then the tile prefix and the bucket table
  std::vector<int> order(out.prob.size());
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return cost[x] > cost[y]; });
  std::vector<gwsig_problem> sorted(out.prob.size());
  long long tb = 0;
  for (size_t i = 0; i < order.size(); ++i) {
    gwsig_problem P = out.prob[order[i]];
    P.tiles_m = zg_tiles_m(P.M, tile_m[stage]);
    P.tiles_n = zg_tiles_n(P.N);
    P.tile_begin = tb;
    tb += (long long)P.nbatch * P.tiles_m * P.tiles_n;
    sorted[i] = P;
  }
  out.prob.swap(sorted);
  if (!kernel_ranges_ok(out.prob, out.seg)) return GWSIG_ERR_ARG;
  out.ntiles = tb;
  out.bucket.assign((size_t)((tb + (1 << ZG_BUCKET_SHIFT) - 1) >> ZG_BUCKET_SHIFT) + 1, 0);
  {
    size_t pi = 0;
    for (size_t bkt = 0; bkt < out.bucket.size(); ++bkt) {
      const long long t = (long long)bkt << ZG_BUCKET_SHIFT;
      while (pi + 1 < out.prob.size() && out.prob[pi + 1].tile_begin <= t) ++pi;
      out.bucket[bkt] = (int)pi;
    }
  }
  return GWSIG_OK;
}

// O_block = U^{k'}^dagger O^{k_I}(alpha^) U^{k_I} for alpha = op_of[k']  (Eq. 28), with
// O^{k_I}(alpha^) = D(alpha) . diag(exp(-2 pi i k' . s_x))  (Eq. 3; column (x,m) carries the phase of its atom).
// Must come out block diagonal in the supplied block map; only the diagonal blocks are kept.
int Plan::compute_oblock(bool aux) {
  const int n = aux ? naux : nao;
  const std::vector<cplx>& U = aux ? U_aux : U_ao;
  const std::vector<double>& D = aux ? D_aux : D_ao;
  const std::vector<int>& atom = aux ? aux_atom : ao_atom;
  const std::vector<std::vector<int>>& offs = aux ? aux_off : ao_off;
  std::vector<cplx>& ob = aux ? oblk_aux : oblk_ao;
  std::vector<long long>& oo = aux ? oblk_aux_off : oblk_ao_off;
  oo.assign(nk + 1, 0);
  for (int k = 0; k < nk; ++k) oo[k + 1] = oo[k] + sumsq(offs[k]);
  ob.assign((size_t)oo[nk], cplx(0, 0));
  std::vector<cplx> OU((size_t)n * n), R((size_t)n * n);
  for (int kp = 0; kp < nk; ++kp) {
    const int kI = ir_of[kp], g = op_of[kp];
    int nn[3];
    kcoords(kp, nn);
    const cplx* UI = &U[(size_t)kI * n * n];
    const cplx* UP = &U[(size_t)kp * n * n];
    const double* Dg = &D[(size_t)g * n * n];
    // OU = D diag(phase) U^{k_I}   (D is sparse: skip zeros)
    std::fill(OU.begin(), OU.end(), cplx(0, 0));
    for (int r = 0; r < n; ++r)
      for (int m = 0; m < n; ++m) {
        const double d = Dg[(size_t)r * n + m];
        if (d == 0.0) continue;
        const int* sx = &shift[((size_t)g * natom + atom[m]) * 3];
        const double ph = -2.0 * M_PI * ((double)nn[0] * sx[0] / N[0] + (double)nn[1] * sx[1] / N[1] + (double)nn[2] * sx[2] / N[2]);
        const cplx w = d * cplx(std::cos(ph), std::sin(ph));
        for (int c = 0; c < n; ++c) OU[(size_t)r * n + c] += w * UI[(size_t)m * n + c];
      }
    // R = U^{k'}^dagger OU
    std::fill(R.begin(), R.end(), cplx(0, 0));
    for (int m = 0; m < n; ++m)
      for (int r = 0; r < n; ++r) {
        const cplx u = std::conj(UP[(size_t)m * n + r]);
        if (u == cplx(0, 0)) continue;
        for (int c = 0; c < n; ++c) R[(size_t)r * n + c] += u * OU[(size_t)m * n + c];
      }
    const std::vector<int>& off = offs[kp];
    double in_blk = 0, off_blk = 0;
    long long o = oo[kp];
    for (size_t b = 0; b + 1 < off.size(); ++b) {
      const int nb = off[b + 1] - off[b];
      for (int r = 0; r < nb; ++r)
        for (int c = 0; c < nb; ++c) ob[(size_t)o + (size_t)r * nb + c] = R[(size_t)(off[b] + r) * n + off[b] + c];
      o += (long long)nb * nb;
    }
    std::vector<int> lab(n);
    for (size_t b = 0; b + 1 < off.size(); ++b)
      for (int i = off[b]; i < off[b + 1]; ++i) lab[i] = (int)b;
    for (int r = 0; r < n; ++r)
      for (int c = 0; c < n; ++c) {
        const double a_ = std::abs(R[(size_t)r * n + c]);
        if (lab[r] == lab[c]) in_blk = std::max(in_blk, a_); else off_blk = std::max(off_blk, a_);
      }
    if (off_blk > 1e-8 * std::max(in_blk, 1e-300)) {
      err = std::string("set_blocks: O_block = U^dagger O U of mesh point ") + std::to_string(kp) + " is not block diagonal in the " +
            (aux ? "auxiliary" : "orbital") + " block map (Eq. 28)";
      return GWSIG_ERR_BLOCKS;
    }
  }
  return GWSIG_OK;
}

long long Plan::unfolded_elems(bool aux, int k_first, int k_count) const {
  long long s = 0;
  for (int k = k_first; k < k_first + k_count; ++k) s += sumsq(aux ? aux_off[k] : ao_off[k]) * ntau;
  return s;
}

int Plan::build_unfold(bool aux, int k_first, int k_count, int step, StagePlan& out) const {
  out.prob.clear(); out.seg.clear(); out.bucket.clear(); out.ntiles = 0;
  if (!general_gauge || k_first < 0 || k_count < 1 || k_first + k_count > nk || step < 1 || step > 2) return GWSIG_ERR_ARG;
  const std::vector<std::vector<int>>& offs = aux ? aux_off : ao_off;
  const std::vector<long long>& in_off = aux ? w_in_off : g_in_off;
  const std::vector<long long>& oo = aux ? oblk_aux_off : oblk_ao_off;
  long long uoff = 0;                                   // offset of point k in T / the unfolded buffer
  for (int k = k_first; k < k_first + k_count; ++k) {
    const std::vector<int>& off = offs[k];
    const long long ts = sumsq(off);                    // elements per tau
    long long bo = 0;
    for (size_t b = 0; b + 1 < off.size(); ++b) {
      const int nb = off[b + 1] - off[b];
      gwsig_seg S; std::memset(&S, 0, sizeof(S));
      gwsig_problem P; std::memset(&P, 0, sizeof(P));
      if (step == 1) {
        // T[(tau, r), c] = sum_m X^{k_I}[(tau, r), m] conj(O[c, m])
        S.a_off = in_off[ir_index[ir_of[k]]] + bo;
        S.am = lvl2(nb, ts, nb); S.ak = lvl1(1);
        S.b_off = oo[k] + bo;
        S.bk = lvl1(1); S.bn = lvl1(nb);                 // B[m, c] = O[c, m]
        S.K = nb;
        P.M = ntau * nb; P.N = nb;
        P.c_off = uoff + bo;
        P.cm = lvl2(nb, ts, nb); P.cn = lvl1(1);
        P.flags = GWSIG_FLAG_CONJ_B | GWSIG_FLAG_A_KMAJOR;
      } else {
        // X^{k'}[(tau), r, c] = sum_m O[r, m] T[(tau), m, c], lowered transposed: rows (tau, c), columns r
        S.a_off = uoff + bo;
        S.am = lvl2(nb, ts, 1); S.ak = lvl1(nb);         // A[(tau, c), m] = T[tau][m][c]
        S.b_off = oo[k] + bo;
        S.bk = lvl1(1); S.bn = lvl1(nb);                 // B[m, r] = O[r, m]
        S.K = nb;
        P.M = ntau * nb; P.N = nb;
        P.c_off = uoff + bo;
        P.cm = lvl2(nb, ts, 1); P.cn = lvl1(nb);         // C[(tau, c), r] = X[tau][r][c]
        P.flags = 0;
      }
      P.nbatch = 1;
      P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
      out.seg.push_back(S); out.prob.push_back(P);
      bo += (long long)nb * nb;
    }
    uoff += ts * ntau;
  }
  long long tb = 0;
  for (auto& P : out.prob) {
    P.tiles_m = zg_tiles_m(P.M, tile_m[0]);
    P.tiles_n = zg_tiles_n(P.N);
    P.tile_begin = tb;
    tb += (long long)P.nbatch * P.tiles_m * P.tiles_n;
  }
  if (!kernel_ranges_ok(out.prob, out.seg)) return GWSIG_ERR_ARG;
  out.ntiles = tb;
  out.bucket.assign((size_t)((tb + (1 << ZG_BUCKET_SHIFT) - 1) >> ZG_BUCKET_SHIFT) + 1, 0);
  size_t pi = 0;
  for (size_t bkt = 0; bkt < out.bucket.size(); ++bkt) {
    const long long t = (long long)bkt << ZG_BUCKET_SHIFT;
    while (pi + 1 < out.prob.size() && out.prob[pi + 1].tile_begin <= t) ++pi;
    out.bucket[bkt] = (int)pi;
  }
  return GWSIG_OK;
}

int Plan::build_vtransform(long long p0, long long np, int step, StagePlan& out) const {
  out.prob.clear(); out.seg.clear(); out.bucket.clear(); out.ntiles = 0; out.red.clear(); out.partial_elems = 0;
  // steps 1, 2: the dense transforms over the auxiliary and the first orbital index; step 3: the second orbital index, allowed
  // triples only, written into the packed layout (needs set_triples); step 4: the second orbital index for EVERY block, dense
  // (what the allowed-block detection looks at: gwsig_block_maxabs, before any triples exist)
  if (mode != GWSIG_IBZ_BLOCK || !have_U || (step == 3 && !have_triples)) return GWSIG_ERR_ARG;
  if (p0 < 0 || np < 1 || p0 + np > npairs || step < 1 || step > 4) return GWSIG_ERR_ARG;
  const long long n2 = (long long)nao * nao, xs = (long long)naux * n2;
  for (long long l = 0; l < np; ++l) {
    const long long p = p0 + l;
    int k1, k2, q, i1;
    pair(p, k1, k2, q, i1);
    if (step == 4) {          // T3[(P,a), i] = sum_j T2[P][a][j] U^{k1}[j, i]      (Eq. 27, last factor; no conjugation)
      gwsig_seg S; std::memset(&S, 0, sizeof(S));
      gwsig_problem P; std::memset(&P, 0, sizeof(P));
      S.a_off = l * xs; P.c_off = l * xs;
      S.am = lvl1(nao); S.ak = lvl1(1);
      S.b_off = (long long)k1 * n2; S.bk = lvl1(nao); S.bn = lvl1(1);
      S.K = nao;
      P.M = naux * nao; P.N = nao;
      P.cm = lvl1(nao); P.cn = lvl1(1);
      P.flags = 0;
      P.nbatch = 1;
      P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
      out.seg.push_back(S); out.prob.push_back(P);
    } else if (step < 3) {
      gwsig_seg S; std::memset(&S, 0, sizeof(S));
      gwsig_problem P; std::memset(&P, 0, sizeof(P));
      S.a_off = l * xs; P.c_off = l * xs;
      if (step == 1) {        // T1^T[(b,j), P] = sum_Q V2^T[(b,j), Q] conj(Uaux^q)[Q, P]
        S.am = lvl1(1); S.ak = lvl1(n2);
        S.b_off = (long long)q * naux * naux; S.bk = lvl1(naux); S.bn = lvl1(1);
        S.K = naux;
        P.M = (int)n2; P.N = naux;
        P.cm = lvl1(1); P.cn = lvl1(n2);
      } else {                // T2[(P,j), a] = sum_b T1[P][b][j] conj(U^{k2})[b, a]
        S.am = lvl2(nao, n2, 1); S.ak = lvl1(nao);
        S.b_off = (long long)k2 * n2; S.bk = lvl1(nao); S.bn = lvl1(1);
        S.K = nao;
        P.M = naux * nao; P.N = nao;
        P.cm = lvl2(nao, n2, 1); P.cn = lvl1(nao);
      }
      P.flags = GWSIG_FLAG_CONJ_B;
      P.nbatch = 1;
      P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
      out.seg.push_back(S); out.prob.push_back(P);
    } else {
      const std::vector<int>&oq = aux_off[q], &o2 = ao_off[k2], &o1 = ao_off[k1];
      const int nb = (int)oq.size() - 1;
      std::vector<long long> Np(nb, 0), c0s;
      const int ntr = pair_ntriples(p);
      c0s.resize(ntr);
      for (int t = 0; t < ntr; ++t) {
        int bp, ba, bi;
        pair_triple(p, t, bp, ba, bi);
        c0s[t] = Np[bp];
        Np[bp] += (long long)(o2[ba + 1] - o2[ba]) * (o1[bi + 1] - o1[bi]);
      }
      std::vector<long long> poff(nb + 1, 0);
      for (int b = 0; b < nb; ++b) poff[b + 1] = poff[b] + (long long)(oq[b + 1] - oq[b]) * Np[b];
      for (int t = 0; t < ntr; ++t) {
        int bp, ba, bi;
        pair_triple(p, t, bp, ba, bi);
        const int n_p = oq[bp + 1] - oq[bp], na = o2[ba + 1] - o2[ba], ni = o1[bi + 1] - o1[bi];
        gwsig_seg S; std::memset(&S, 0, sizeof(S));
        gwsig_problem P; std::memset(&P, 0, sizeof(P));
        // packed(P,a,i) = sum_j T2[oq+P][o2+a][j] U^{k1}[j][o1+i]
        S.a_off = l * xs + (long long)oq[bp] * n2 + (long long)o2[ba] * nao;
        S.am = lvl2(na, n2, nao); S.ak = lvl1(1);
        S.b_off = (long long)k1 * n2 + o1[bi]; S.bk = lvl1(nao); S.bn = lvl1(1);
        S.K = nao;
        P.M = n_p * na; P.N = ni;
        P.c_off = (v_off[p] - v_off[p0]) + poff[bp] + c0s[t];
        P.cm = lvl2(na, Np[bp], ni); P.cn = lvl1(1);
        P.flags = 0;
        P.nbatch = 1;
        P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
        out.seg.push_back(S); out.prob.push_back(P);
      }
    }
  }
  long long tb = 0;
  for (auto& P : out.prob) {
    P.tiles_m = zg_tiles_m(P.M, tile_m[0]);
    P.tiles_n = zg_tiles_n(P.N);
    P.tile_begin = tb;
    tb += (long long)P.nbatch * P.tiles_m * P.tiles_n;
  }
  if (!kernel_ranges_ok(out.prob, out.seg)) return GWSIG_ERR_ARG;
  out.ntiles = tb;
  out.bucket.assign((size_t)((tb + (1 << ZG_BUCKET_SHIFT) - 1) >> ZG_BUCKET_SHIFT) + 1, 0);
  size_t pi = 0;
  for (size_t bkt = 0; bkt < out.bucket.size(); ++bkt) {
    const long long t = (long long)bkt << ZG_BUCKET_SHIFT;
    while (pi + 1 < out.prob.size() && out.prob[pi + 1].tile_begin <= t) ++pi;
    out.bucket[bkt] = (int)pi;
  }
  return GWSIG_OK;
}

int Plan::build_gridtransform(int nq, int nin, int nout, StagePlan& out) const {
  out.prob.clear(); out.seg.clear(); out.bucket.clear(); out.ntiles = 0; out.red.clear(); out.partial_elems = 0;
  if (nq < 1 || nin < 1 || nout < 1) return GWSIG_ERR_ARG;
  const long long n2 = (long long)naux * naux;
  if (n2 >= (1LL << 31)) return GWSIG_ERR_ARG;
  long long tb = 0;
  for (int q = 0; q < nq; ++q) {
    gwsig_seg S; std::memset(&S, 0, sizeof(S));
    gwsig_problem P; std::memset(&P, 0, sizeof(P));
    S.a_off = (long long)q * nin * n2; S.am = lvl1(1); S.ak = lvl1(n2);       // A[m, i] = src[q][i][m]
    S.b_off = 0; S.bk = lvl1(1); S.bn = lvl1(nin);                            // B[i, o] = T[o][i]
    S.K = nin;
    P.M = (int)n2; P.N = nout;
    P.c_off = (long long)q * nout * n2; P.cm = lvl1(1); P.cn = lvl1(n2);      // C[m, o] = dst[q][o][m]
    P.nbatch = 1; P.flags = 0;
    P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
    P.tiles_m = zg_tiles_m(P.M, tile_m[0]); P.tiles_n = zg_tiles_n(P.N);
    P.tile_begin = tb;
    tb += (long long)P.tiles_m * P.tiles_n;
    out.seg.push_back(S); out.prob.push_back(P);
  }
  if (!kernel_ranges_ok(out.prob, out.seg)) return GWSIG_ERR_ARG;
  out.ntiles = tb;
  out.bucket.assign((size_t)((tb + (1 << ZG_BUCKET_SHIFT) - 1) >> ZG_BUCKET_SHIFT) + 1, 0);
  size_t pi = 0;
  for (size_t bkt = 0; bkt < out.bucket.size(); ++bkt) {
    const long long t = (long long)bkt << ZG_BUCKET_SHIFT;
    while (pi + 1 < out.prob.size() && out.prob[pi + 1].tile_begin <= t) ++pi;
    out.bucket[bkt] = (int)pi;
  }
  return GWSIG_OK;
}

int Plan::build_p0_stage(long long p0, long long np, int nt, int stage, StagePlan& out, int num_sms) const {
  out.prob.clear(); out.seg.clear(); out.bucket.clear(); out.ntiles = 0; out.red.clear(); out.partial_elems = 0;
  if (mode == GWSIG_IBZ_BLOCK) return GWSIG_ERR_ARG;                // dense modes only
  if (p0 < 0 || np < 1 || p0 + np > (long long)nk * nk1 || nt < 1 || nt > ntau || stage < 1 || stage > 3) return GWSIG_ERR_ARG;
  const long long n2 = (long long)nao * nao, xs = (long long)naux * n2, gts = n2, wts = (long long)naux * naux;
  std::vector<long long> cost;
  if (stage == 1 || stage == 2) {
    for (long long l = 0; l < np; ++l) {
      int k, q, kq, iq;
      p0_pair(p0 + l, k, q, kq, iq);
      gwsig_seg S; std::memset(&S, 0, sizeof(S));
      gwsig_problem P; std::memset(&P, 0, sizeof(P));
      S.K = nao;
      P.M = nt * nao; P.N = naux * nao;
      P.c_off = l * xs * nt;
      P.a_tstride = gts;
      P.nbatch = 1;
      if (stage == 1) {
        // X1^T[(tau,c),(a,Q)] = sum_d Grev^k[(tau,c),d] T[d,(a,Q)]                    (Algorithm 3 line 6)
        // column index n = (a, Q) with Q fastest: a tile row of C is then CONTIGUOUS in X1[tau][(c,a)][Q] (full-sector stores;
        // and so is the operand row, read from the aux-last copy of T the library makes per push)
        S.a_off = (long long)k * ntau * gts;
        S.am = lvl2(nao, gts, 1); S.ak = lvl1(nao);          // A = the library's transposed copy Grev^T[tau][d][c]: c contiguous
        S.b_off = l * xs;
        S.bk = lvl1((long long)nao * naux); S.bn = lvl1(1);  // n = (a, Q): the library's aux-last copy T'[d][a][Q] = T[Q][d][a]
        P.cm = lvl2(nao, xs, (long long)nao * naux);         // X1[tau][(c,a)][Q]
        P.cn = lvl1(1);                                      // a * naux + Q = n
        P.flags = 0;
      } else {
        // X2^T[(tau,a),(c,Q')] = sum_b G^{kq}[(tau,a),b] conj(T[Q'][c][b])              (Algorithm 3 line 7)
        // n = (c, Q') with Q' fastest, for the same reason: runs of naux contiguous elements of X2[tau][(c,a)][Q'] per tile row
        S.a_off = (long long)kq * ntau * gts;
        S.am = lvl2(nao, gts, 1); S.ak = lvl1(nao);          // A = the transposed copy G^T[tau][b][a]: a contiguous
        S.b_off = l * xs;
        S.bk = lvl1(naux); S.bn = lvl2(naux, (long long)nao * naux, 1);   // n = (c, Q'): the aux-last copy T'[c][b][Q'] = T[Q'][c][b]
        P.cm = lvl2(nao, xs, naux);                          // X2[tau][(c,a)][Q']: a * naux
        P.cn = lvl2(naux, (long long)nao * naux, 1);         // c * nao * naux + Q'
        P.flags = GWSIG_FLAG_CONJ_B;
      }
      P.seg_begin = (int)out.seg.size(); P.seg_count = 1;
      out.seg.push_back(S); out.prob.push_back(P); cost.push_back(S.K);
    }
  } else {
    // P0acc[iq][tau][Q][Q'] += sum_pairs sum_{(c,a)} X1[(c,a)][Q] X2[(c,a)][Q']       (Algorithm 3 line 8); the pairs
    // (k) of one q are the segments, cut into parts that add into the same block (FP64 atomics), one batch entry per tau
    long long tiles1 = 0;
    std::vector<std::vector<gwsig_seg>> segs(nk1);
    for (long long l = 0; l < np; ++l) {
      int k, q, kq, iq;
      p0_pair(p0 + l, k, q, kq, iq);
      gwsig_seg S; std::memset(&S, 0, sizeof(S));
      S.a_off = l * xs * nt; S.am = lvl1(1); S.ak = lvl1(naux);       // A[m = Q, k = (c,a)] = X1[(c,a)][Q]
      S.b_off = l * xs * nt; S.bk = lvl1(naux); S.bn = lvl1(1);       // B[k = (c,a), n = Q'] = X2[(c,a)][Q']
      S.K = (int)n2;
      segs[iq].push_back(S);
    }
    for (int iq = 0; iq < nk1; ++iq)
      if (!segs[iq].empty()) tiles1 += (long long)nt * zg_tiles_m(naux, tile_m[3]) * zg_tiles_n(naux);
    const long long want = 12LL * std::max(num_sms, 1);
    for (int iq = 0; iq < nk1; ++iq) {
      if (segs[iq].empty()) continue;
      long long parts = tiles1 > 0 ? (want + tiles1 - 1) / tiles1 : 1;
      parts = std::max(1LL, std::min<long long>(parts, (long long)segs[iq].size()));
      const size_t nsg = segs[iq].size();
      for (long long part = 0; part < parts; ++part) {
        const size_t s0 = nsg * part / parts, s1 = nsg * (part + 1) / parts;
        if (s1 <= s0) continue;
        gwsig_problem P; std::memset(&P, 0, sizeof(P));
        P.M = naux; P.N = naux;
        P.c_off = (long long)iq * ntau * wts;
        P.cm = lvl1(naux); P.cn = lvl1(1);
        P.a_bstride = xs; P.b_bstride = xs; P.c_bstride = wts; P.c_tstride = wts;
        P.nbatch = nt;
        P.flags = GWSIG_FLAG_ACCUM;
        P.seg_begin = (int)out.seg.size();
        for (size_t s_ = s0; s_ < s1; ++s_) out.seg.push_back(segs[iq][s_]);
        P.seg_count = (int)(s1 - s0);
        out.prob.push_back(P); cost.push_back((long long)(s1 - s0) * n2);
      }
    }
  }
  std::vector<int> order(out.prob.size());
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return cost[x] > cost[y]; });
  std::vector<gwsig_problem> sorted(out.prob.size());
  long long tb = 0;
  for (size_t i = 0; i < order.size(); ++i) {
    gwsig_problem P = out.prob[order[i]];
    P.tiles_m = zg_tiles_m(P.M, tile_m[stage]);
    P.tiles_n = zg_tiles_n(P.N);
    P.tile_begin = tb;
    tb += (long long)P.nbatch * P.tiles_m * P.tiles_n;
    sorted[i] = P;
  }
  out.prob.swap(sorted);
  if (!kernel_ranges_ok(out.prob, out.seg)) return GWSIG_ERR_ARG;
  out.ntiles = tb;
  out.bucket.assign((size_t)((tb + (1 << ZG_BUCKET_SHIFT) - 1) >> ZG_BUCKET_SHIFT) + 1, 0);
  size_t pi = 0;
  for (size_t bkt = 0; bkt < out.bucket.size(); ++bkt) {
    const long long t = (long long)bkt << ZG_BUCKET_SHIFT;
    while (pi + 1 < out.prob.size() && out.prob[pi + 1].tile_begin <= t) ++pi;
    out.bucket[bkt] = (int)pi;
  }
  return GWSIG_OK;
}

void Plan::flop_counts(double& full_equiv, double& executed) const {
  const double A = (double)naux * nao * nao * nao, B = (double)naux * naux * nao * nao;
  full_equiv = (double)nk * nk * ntau * 8.0 * (2.0 * A + B);
  if (mode != GWSIG_IBZ_BLOCK) { executed = (double)npairs * ntau * 8.0 * (2.0 * A + B); return; }
  executed = 0;
  if (!have_triples) return;
  double macs = 0;
  for (long long p = 0; p < npairs; ++p) {
    int k1, k2, q, i1;
    pair(p, k1, k2, q, i1);
    const std::vector<int>&oq = aux_off[q], &o2 = ao_off[k2], &o1 = ao_off[k1];
    std::vector<double> Np(oq.size() - 1, 0.0);
    for (long long t = triple_ptr[p]; t < triple_ptr[p + 1]; ++t) {
      const int32_t* T = &triples[3 * t];
      double np_ = oq[T[0] + 1] - oq[T[0]], na = o2[T[1] + 1] - o2[T[1]], ni = o1[T[2] + 1] - o1[T[2]];
      macs += np_ * ni * na * na + np_ * na * ni * ni;      // stage 1 + stage 3
      Np[T[0]] += na * ni;
    }
    for (size_t b = 0; b < Np.size(); ++b) { double npb = oq[b + 1] - oq[b]; macs += npb * npb * Np[b]; }   // stage 2
  }
  executed = 8.0 * ntau * macs;
}

}  // namespace gwsig
