"""Seeded synthetic tensors G, V, W~ (inputs only).

Recipe (stated again in DESIGN.md):
  * real-space operators H(R), A_m(R) (two-index) and V(R1,R2) (three-index) are
    drawn from per-object counter-based Philox streams, given the required
    index symmetries, and averaged over the space group with the real
    representation matrices (perm (x) Wigner D) and the lattice shifts;
  * Bloch sums follow Eq. 2:  H(k) = sum_R e^{+2 pi i k.R} H(R),
    V^{k1,k2}_{Q,ij} = sum_{R1,R2} e^{-2 pi i k1.R1 + 2 pi i k2.R2} V_{Q,i,j}(R1,R2);
  * G(k,tau) is the closed form -U diag(e^{-eps tau}/(1+e^{-beta eps})) U^dagger;
  * W~(q,tau) = sum_m e^{-w_m min(tau, beta-tau)} A_m(q) A_m(q)^dagger, w = (0.5, 1, 2).
"""
from __future__ import annotations

import os

import numpy as np

from .crystal import Crystal
from .group import KMesh

OMEGAS = (0.5, 1.0, 2.0)


def tau_grid(ntau: int, beta: float) -> np.ndarray:
    """uniform grid on [0, beta], endpoints included."""
    return np.arange(ntau) * (beta / (ntau - 1))


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[seed, stream]))


def fermi_factor(eps: np.ndarray, tau: float, beta: float) -> np.ndarray:
    """e^{-eps tau}/(1+e^{-beta eps}), overflow-free."""
    pos = eps >= 0
    out = np.empty_like(eps)
    out[pos] = np.exp(-eps[pos] * tau) / (1.0 + np.exp(-beta * eps[pos]))
    out[~pos] = np.exp(eps[~pos] * (beta - tau)) / (1.0 + np.exp(beta * eps[~pos]))
    return out


def green_closed_form(Hk: np.ndarray, mu: float, tau: np.ndarray, beta: float) -> np.ndarray:
    """G(tau) = -U diag(f(eps, tau)) U^dagger for one Hermitian H(k)  ->  [ntau, n, n]."""
    eps, U = np.linalg.eigh(Hk - mu * np.eye(Hk.shape[0]))
    f = np.stack([fermi_factor(eps, t, beta) for t in tau])           # [ntau, n]
    return -np.einsum("ia,ta,ja->tij", U, f, U.conj())


def chemical_potential(eigs: np.ndarray, nocc_total: int) -> float:
    """midpoint between the nocc_total-th and the next eigenvalue over all k (A11)."""
    e = np.sort(eigs.ravel())
    return 0.5 * (e[nocc_total - 1] + e[nocc_total])


def screened_from_A(A: np.ndarray, tau: np.ndarray, beta: float) -> np.ndarray:
    """W~(tau) = sum_m e^{-w_m min(tau, beta - tau)} A_m A_m^dagger ; A: [3, n, n] -> [ntau, n, n]."""
    AA = np.einsum("mij,mkj->mik", A, A.conj())
    t = np.minimum(tau, beta - tau)
    wgt = np.exp(-np.outer(t, np.array(OMEGAS)))                      # [ntau, 3]
    return np.einsum("tm,mik->tik", wgt, AA)


# ==========================================================================
# config 1: no symmetry, everything random per k
# ==========================================================================


class RandomC1Inputs:
    """BASELINE.json config 1 (C1, full BZ).  Readings A11, A12."""

    def __init__(self, mesh=(2, 2, 2), nao=8, naux=32, ntau=16, beta=10.0, nocc=4, seed=20240510):
        self.kmesh = KMesh(mesh)
        self.nk, self.nao, self.naux, self.ntau, self.beta = self.kmesh.nk, nao, naux, ntau, beta
        self.tau = tau_grid(ntau, beta)
        self.seed = seed
        r = _rng(seed, 1)
        A = r.standard_normal((self.nk, nao, nao)) + 1j * r.standard_normal((self.nk, nao, nao))
        self.Hk = 0.5 * (A + A.conj().transpose(0, 2, 1)) + 2.0 * np.diag(np.linspace(-1, 1, nao))[None]
        self.mu = chemical_potential(np.linalg.eigvalsh(self.Hk), nocc * self.nk)
        r = _rng(seed, 2)
        # V[k1,k2,Q,i,j]: free for k1<k2, conj-transposed partner for k1>k2, Hermitian in ij for k1==k2
        V = (r.standard_normal((self.nk, self.nk, naux, nao, nao))
             + 1j * r.standard_normal((self.nk, self.nk, naux, nao, nao))) / np.sqrt(naux)
        for k1 in range(self.nk):
            V[k1, k1] = 0.5 * (V[k1, k1] + V[k1, k1].conj().transpose(0, 2, 1))
            for k2 in range(k1):
                V[k1, k2] = V[k2, k1].conj().transpose(0, 2, 1)
        self._V = V
        r = _rng(seed, 3)
        self._A = 0.1 * (r.standard_normal((self.nk, 3, naux, naux)) + 1j * r.standard_normal((self.nk, 3, naux, naux)))

    def G_full(self) -> np.ndarray:
        return np.stack([green_closed_form(self.Hk[k], self.mu, self.tau, self.beta) for k in range(self.nk)])

    def W_full(self, qs=None) -> np.ndarray:
        qs = range(self.nk) if qs is None else qs
        return np.stack([screened_from_A(self._A[q], self.tau, self.beta) for q in qs])

    def V_pair(self, k1: int, k2: int) -> np.ndarray:
        """V^{k1,k2}_{Q,ij}  [naux, nao, nao]"""
        return self._V[k1, k2]

    def V2_rows(self, k1: int, k2s) -> np.ndarray:
        """V^{k2,k1}_{Q,bj} for every k2 in k2s  [len, naux, nao, nao]"""
        return np.stack([self._V[k2, k1] for k2 in k2s])

    def V_pairs(self, k1s, k2s) -> np.ndarray:
        """V^{k1,k2}_{Q,ij} for a list of pairs  [len, naux, nao, nao]"""
        return np.stack([self._V[a, b] for a, b in zip(k1s, k2s)])

    def V1_rows(self, k1: int, k2s) -> np.ndarray:
        """V^{k1,k2}_{Q,ia} for every k2 in k2s  [len, naux, nao, nao]"""
        return np.stack([self._V[k1, k2] for k2 in k2s])


# ==========================================================================
# configs 2-5: group-averaged real-space operators
# ==========================================================================


def lattice_shells(a: np.ndarray, nshell: int):
    """lattice vectors R (integer triples) up to the nshell-th distinct non-zero
    length, and d1 = nearest-neighbour lattice distance (A13)."""
    rng = np.arange(-4, 5)
    R = np.array(np.meshgrid(rng, rng, rng, indexing="ij")).reshape(3, -1).T
    d = np.linalg.norm(R @ a, axis=1)
    lens = np.unique(np.round(d, 9))
    lens = lens[lens > 0]
    keep = d <= lens[nshell - 1] + 1e-9
    order = np.lexsort((R[keep][:, 2], R[keep][:, 1], R[keep][:, 0], np.round(d[keep], 9)))
    return R[keep][order], d[keep][order], lens[0]


def _encode(R: np.ndarray) -> np.ndarray:
    """integer rows [..., m] (|entries| < 16) -> one int64 key each."""
    key = np.zeros(R.shape[:-1], dtype=np.int64)
    for c in range(R.shape[-1]):
        key = key * 33 + (R[..., c] + 16)
    return key


def _group_average(cr: Crystal, keys: np.ndarray, M: np.ndarray, reps, starts, nleg: int):
    """Shared bookkeeping of the group average (G7/G8).  ``keys`` [n, 3*(nleg-1)]
    are the lattice vectors R (two-index) or (R1, R2) (three-index) of the
    stacked real-space blocks ``M`` [n, ...]; leg 0 sits in cell 0, leg j>0 in
    cell R_j.  Under g an atom block (x_0, .., x_m) at (R_1, ..) moves to
    (perm x_0, .., perm x_m) at (W R_j + s_{x_j} - s_{x_0}) and every leg j is
    multiplied by the real representation matrix ``reps[j][g]`` (perm (x) Wigner D).
    The representation matrices only connect atom x to perm x, so each atom block
    is transformed on its own with the matching sub-matrices (same result as
    transforming the whole tensor, a fraction of the work)."""
    import threading
    sg = cr.sg
    nat = cr.natom
    nR = nleg - 1
    combos = np.array(np.meshgrid(*[np.arange(nat)] * nleg, indexing="ij")).reshape(nleg, -1).T
    Rs = keys.reshape(len(keys), nR, 3)

    def new_keys(g, combo):
        W, s = sg.W[g], sg.shift[g]
        Rn = Rs @ W.T + (s[combo[1:]] - s[combo[0]])[None, :, :]
        return Rn.reshape(len(keys), 3 * nR)

    allk = np.concatenate([new_keys(g, c) for g in range(sg.nops) for c in combos])
    uniq = np.unique(_encode(allk))
    del allk
    out = np.zeros((len(uniq),) + M.shape[1:])
    out_keys = np.zeros((len(uniq), 3 * nR), dtype=np.int64)
    lock = threading.Lock()

    def one_op(g):
        perm = sg.perm[g]
        for c in combos:
            sin = tuple(slice(starts[j][c[j]], starts[j][c[j] + 1]) for j in range(nleg))
            sout = tuple(slice(starts[j][perm[c[j]]], starts[j][perm[c[j]] + 1]) for j in range(nleg))
            B = np.ascontiguousarray(M[(slice(None),) + sin])
            for j in range(nleg):                                   # leg j: D[out rows, in cols] on axis 1 + j
                D = np.ascontiguousarray(reps[j][g][sout[j], sin[j]])
                if j == nleg - 1:
                    B = (B.reshape(-1, B.shape[-1]) @ D.T).reshape(B.shape)
                elif j == 0:
                    B = np.matmul(D, B.reshape(B.shape[0], B.shape[1], -1)).reshape(B.shape)
                else:
                    B = np.matmul(D[None, None], B)
            nk_ = new_keys(g, c)
            idx = np.searchsorted(uniq, _encode(nk_))
            with lock:
                out_keys[idx] = nk_
                out[(idx,) + sout] += B

    # serial over the operations: concurrent calls into the multi-threaded BLAS from several Python threads corrupted the
    # result for the larger bases (config 5: V lost its transposition symmetry); the BLAS calls are threaded by themselves
    for g in range(sg.nops):
        one_op(g)
    out /= sg.nops
    keep = np.abs(out).reshape(len(uniq), -1).max(axis=1) > 0
    if keep.all():
        return out_keys, out
    return out_keys[keep], out[keep]


def average_two_index(cr: Crystal, Xr: dict, P: np.ndarray, start: np.ndarray) -> dict:
    """(1/|G|) sum_g g.X with
    (g.X)_{(pi(x) i'),(pi(y) j')}(W R + s_y - s_x) += D_{i'i} D_{j'j} X_{(x i),(y j)}(R)   (G7)."""
    keys = np.array(list(Xr.keys()), dtype=np.int64)
    M = np.stack([Xr[tuple(k)] for k in keys])
    ok, om = _group_average(cr, keys, M, (P, P), (start, start), 2)
    return {tuple(int(v) for v in k): m for k, m in zip(ok, om)}


def average_three_index(cr: Crystal, Vr: dict) -> dict:
    """(1/|G|) sum_g g.V with
    (g.V)_{(pi(z)Q'),(pi(x)i'),(pi(y)j')}(W R1 + s_x - s_z, W R2 + s_y - s_z)
        += Daux_{Q'Q} D_{i'i} D_{j'j} V_{Q,i,j}(R1,R2)                                (G8).
    Returns (keys, blocks) rather than a dict: the table is 15 GB at config 5."""
    klist = list(Vr.keys())
    keys = np.array([list(k[0]) + list(k[1]) for k in klist], dtype=np.int64)
    M = np.stack([Vr[k] for k in klist])
    ok, om = _group_average(cr, keys, M, (cr.P_aux, cr.P_ao, cr.P_ao), (cr.aux_start, cr.ao_start, cr.ao_start), 3)
    return [tuple(int(v) for v in k) for k in ok], om          # keys (R1, R2) as 6-tuples, blocks [n, naux, nao, nao]


def _cdot_real(f: np.ndarray, X: np.ndarray, axis: int) -> np.ndarray:
    """sum_r f[r] X[..r..] over `axis` of the REAL table X with complex weights f, as two real contractions
    (np.tensordot would first cast the whole table to complex: 30 GB at config 5)."""
    return np.tensordot(f.real, X, axes=(0, axis)) + 1j * np.tensordot(f.imag, X, axes=(0, axis))


class SymmetricInputs:
    """BASELINE.json configs 2-5 (and the toys): symmetric random crystal."""

    def __init__(self, cr: Crystal, v_shells: int = 1):
        self.cr = cr
        self.kmesh = cr.kmesh
        self.nk, self.nao, self.naux = cr.kmesh.nk, cr.nao, cr.naux
        self.ntau, self.beta = cr.ntau, cr.beta
        self.tau = tau_grid(cr.ntau, cr.beta)
        seed = cr.seed
        a = cr.a

        # ---- H(R): Hermitian, decaying, group-averaged -------------------
        Rs, d, d1 = lattice_shells(a, cr.h_shells)
        r = _rng(seed, 1)
        raw = {tuple(R): r.standard_normal((cr.nao, cr.nao)) * np.exp(-dd / d1) for R, dd in zip(Rs, d)}
        raw = {R: 0.5 * (M + raw[tuple(-np.array(R))].T) for R, M in raw.items()}        # H_ab(R) = H_ba(-R)
        self.Hr = average_two_index(cr, raw, cr.P_ao, cr.ao_start)

        # ---- A_m(R), m = 1..3: N(0, 0.1), not Hermitian ------------------
        self.Ar = []
        for m in range(3):
            r = _rng(seed, 10 + m)
            raw = {tuple(R): 0.1 * r.standard_normal((cr.naux, cr.naux)) * np.exp(-dd / d1) for R, dd in zip(Rs, d)}
            self.Ar.append(average_two_index(cr, raw, cr.P_aux, cr.aux_start))

        # ---- V(R1,R2): three-centre, V_{Q,j,i}(R2,R1) = V_{Q,i,j}(R1,R2) -
        Rv, dv, _ = lattice_shells(a, v_shells)
        r = _rng(seed, 20)
        raw = {}
        for R1, d1_ in zip(Rv, dv):
            for R2, d2_ in zip(Rv, dv):
                raw[(tuple(R1), tuple(R2))] = (r.standard_normal((cr.naux, cr.nao, cr.nao))
                                               * np.exp(-(d1_ + d2_) / d1) / np.sqrt(cr.naux))
        raw = {K: 0.5 * (M + raw[(K[1], K[0])].transpose(0, 2, 1)) for K, M in raw.items()}
        vkeys, vvals = average_three_index(cr, raw)
        del raw
        # dense [nR1, nR2, naux*nao*nao] table for fast Bloch sums
        R1s, R2s = [tuple(k[:3]) for k in vkeys], [tuple(k[3:]) for k in vkeys]
        self.vR1 = sorted(set(R1s))
        self.vR2 = sorted(set(R2s))
        i1 = {R: i for i, R in enumerate(self.vR1)}
        i2 = {R: i for i, R in enumerate(self.vR2)}
        self.Vd = np.zeros((len(self.vR1), len(self.vR2), cr.naux * cr.nao * cr.nao))
        self.Vd[[i1[R] for R in R1s], [i2[R] for R in R2s]] = vvals.reshape(len(vvals), -1)
        del vvals
        self.vR1 = np.array(self.vR1)
        self.vR2 = np.array(self.vR2)

        # ---- H(k), mu -----------------------------------------------------
        self.Hk = np.stack([self.bloch_two_index(self.Hr, k) for k in range(self.nk)])
        self.mu = chemical_potential(np.linalg.eigvalsh(self.Hk), cr.nocc * self.nk)

    # ---- Bloch sums -------------------------------------------------------
    def bloch_two_index(self, Xr: dict, k: int) -> np.ndarray:
        kf = self.kmesh.frac[k]
        out = 0
        for R, M in Xr.items():
            out = out + np.exp(2j * np.pi * np.dot(kf, R)) * M
        return out

    def A_q(self, q: int) -> np.ndarray:
        return np.stack([self.bloch_two_index(Ar, q) for Ar in self.Ar])

    def G_k(self, k: int) -> np.ndarray:
        return green_closed_form(self.Hk[k], self.mu, self.tau, self.beta)

    def G_full(self, ks=None) -> np.ndarray:
        ks = range(self.nk) if ks is None else ks
        return np.stack([self.G_k(k) for k in ks])

    def W_full(self, qs=None) -> np.ndarray:
        qs = range(self.nk) if qs is None else qs
        return np.stack([screened_from_A(self.A_q(q), self.tau, self.beta) for q in qs])

    def V_pair(self, k1: int, k2: int) -> np.ndarray:
        """V^{k1,k2}_{Q,ij}  [naux, nao, nao]"""
        f1 = np.exp(-2j * np.pi * (self.vR1 @ self.kmesh.frac[k1]))
        f2 = np.exp(+2j * np.pi * (self.vR2 @ self.kmesh.frac[k2]))
        T = _cdot_real(f2, self.Vd, 1)                               # [nR1, nel]
        return (f1 @ T).reshape(self.naux, self.nao, self.nao)

    def V2_rows(self, k1: int, k2s) -> np.ndarray:
        """V^{k2,k1}_{Q,bj} for every k2 in k2s  [len, naux, nao, nao]
        (first momentum k2 carries e^{-2 pi i k2.R1}, second k1 carries e^{+2 pi i k1.R2})."""
        k2s = np.asarray(list(k2s))
        f2 = np.exp(+2j * np.pi * (self.vR2 @ self.kmesh.frac[k1]))
        T = _cdot_real(f2, self.Vd, 1)                               # [nR1, nel]
        f1 = np.exp(-2j * np.pi * (self.kmesh.frac[k2s] @ self.vR1.T))   # [nk2, nR1]
        return (f1 @ T).reshape(len(k2s), self.naux, self.nao, self.nao)


    def V_pairs(self, k1s, k2s) -> np.ndarray:
        """V^{k1,k2}_{Q,ij} for a LIST of pairs (k1s[n], k2s[n])  [len, naux, nao, nao]: the Bloch sum of V_pair with the two
        phase vectors multiplied out per pair, as two real products against the real-space table."""
        k1s, k2s = np.asarray(list(k1s)), np.asarray(list(k2s))
        f1 = np.exp(-2j * np.pi * (self.kmesh.frac[k1s] @ self.vR1.T))         # [n, nR1]
        f2 = np.exp(+2j * np.pi * (self.kmesh.frac[k2s] @ self.vR2.T))         # [n, nR2]
        F = (f1[:, :, None] * f2[:, None, :]).reshape(len(k1s), -1)
        Vd = self.Vd.reshape(F.shape[1], -1)
        out = (F.real @ Vd) + 1j * (F.imag @ Vd)
        return out.reshape(len(k1s), self.naux, self.nao, self.nao)

    def V1_rows(self, k1: int, k2s) -> np.ndarray:
        """V^{k1,k2}_{Q,ia} for every k2 in k2s  [len, naux, nao, nao]  (same Bloch sum as V_pair, batched over k2)."""
        k2s = np.asarray(list(k2s))
        f1 = np.exp(-2j * np.pi * (self.vR1 @ self.kmesh.frac[k1]))
        T = _cdot_real(f1, self.Vd, 0)                               # [nR2, nel]
        f2 = np.exp(+2j * np.pi * (self.kmesh.frac[k2s] @ self.vR2.T))   # [nk2, nR2]
        return (f2 @ T).reshape(len(k2s), self.naux, self.nao, self.nao)


def make_inputs(name: str, **over):
    """inputs object for 'cfg1'..'cfg5' or a toy crystal name."""
    from .crystal import make_crystal
    if name == "cfg1":
        return RandomC1Inputs(**over)
    v_shells = over.pop("v_shells", 1)
    return SymmetricInputs(make_crystal(name, **over), v_shells=v_shells)
