"""Host pre-step (Algorithm 1, and Eq. 26-27).

The paper block-diagonalises its integrals "before starting the self-consistent
GW calculation"; this module is that pre-step for callers of the
C-ABI library: it produces what ``gwsig_set_blocks`` / ``gwsig_set_triples`` and
``sigma_eval`` in IBZ_BLOCK mode take as INPUTS (U^k, the irrep block maps, the
allowed (p, alpha, iota) triples per pair and the packed block-basis tensors).
It is numpy host code, runs once per crystal, and is not part of the timed
hot path.  Nothing here evaluates Sigma.

Steps:
  S1 little group of k: operations with k~ = k
  S2 D^k(alpha) = e^{2 pi i k.w(alpha)} O^k(alpha^)                  (Eq. 7)
  S3 Dirac characters  Omega_gamma = (1/h) sum_beta D(beta) D(gamma) D(beta)^-1
     (first form of Eq. 10, read as a conjugation sum -- DESIGN.md A2)
  S4 one random Hermitian combination of them, eigh, clusters of equal
     eigenvalue = isotypic blocks, eigenvectors = U^k
  S5 star members: U^{k'} = O^{k_I}(alpha^) U^{k_I}  (so O_block of Eq. 28 is 1)
  S6 block-basis inputs by Eq. 26-27 and the packed ragged layout.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass
class BlockBasis:
    """U^k and the irrep (isotypic) block offsets for every k of the full mesh."""
    U: np.ndarray               # [nk, n, n] complex
    off: list                   # per k: int array [nblk+1], block b = off[b]:off[b+1]

    def nblk(self, k):
        return len(self.off[k]) - 1

    def sizes(self, k):
        return np.diff(self.off[k])

    def sumsq(self, k):
        return int((np.diff(self.off[k]) ** 2).sum())


class SymSetup:
    """Group data of one crystal + mesh, and Algorithm 1 on top of it."""

    def __init__(self, mesh, W, w, shift, P_ao, P_aux, ao_atom, aux_atom, seed: int = 7):
        self.N = np.array(mesh, dtype=np.int64)
        self.nk = int(np.prod(self.N))
        self.W = np.asarray(W, dtype=np.int64)
        self.w = np.asarray(w, float)
        self.shift = np.asarray(shift, dtype=np.int64)
        self.P = {"ao": np.asarray(P_ao, float), "aux": np.asarray(P_aux, float)}
        self.atom = {"ao": np.asarray(ao_atom, dtype=np.int64), "aux": np.asarray(aux_atom, dtype=np.int64)}
        self.nops = self.W.shape[0]
        self.seed = seed
        g0, g1, g2 = np.meshgrid(*[np.arange(m) for m in self.N], indexing="ij")
        self.n = np.stack([g0.ravel(), g1.ravel(), g2.ravel()], axis=1)
        self.frac = self.n / self.N[None, :]
        self.rot = np.stack([self._rotate(self.W[g]) for g in range(self.nops)])       # [nops, nk]
        # stars: representative = first member in index order; op_of = first op in input order
        self.ir_of = -np.ones(self.nk, dtype=np.int64)
        self.op_of = -np.ones(self.nk, dtype=np.int64)
        ir = []
        for k in range(self.nk):
            if self.ir_of[k] >= 0:
                continue
            ir.append(k)
            for g in range(self.nops):
                kp = self.rot[g, k]
                if self.ir_of[kp] < 0:
                    self.ir_of[kp] = k
                    self.op_of[kp] = g
        self.ir_list = np.array(ir, dtype=np.int64)
        self.ir_index = {int(k): i for i, k in enumerate(self.ir_list)}

    # ---- mesh arithmetic ---------------------------------------------------
    def index(self, n):
        n = np.mod(np.asarray(n, dtype=np.int64), self.N)
        return (n[..., 0] * self.N[1] + n[..., 1]) * self.N[2] + n[..., 2]

    def sub(self, k, q):
        return int(self.index(self.n[k] - self.n[q]))

    def _rotate(self, W):
        Winv = np.rint(np.linalg.inv(W)).astype(np.int64)
        num = np.zeros_like(self.n)
        for j in range(3):
            for i in range(3):
                t = self.n[:, i] * Winv[i, j] * self.N[j]
                if np.any(t % self.N[i] != 0):
                    raise ValueError("rotation does not map the k mesh onto itself")
                num[:, j] += t // self.N[i]
        return self.index(num)

    # ---- representation matrices (Eq. 3) --------------------
    def O(self, kind: str, k: int, g: int) -> np.ndarray:
        """O^k(alpha^_g), maps k -> rot[g, k];  = P_g . diag(exp(-2 pi i k~ . s_x))."""
        kt = self.frac[self.rot[g, k]]
        ph = np.exp(-2j * np.pi * (self.shift[g] @ kt))
        return self.P[kind][g] * ph[self.atom[kind]][None, :]

    def little_group(self, k: int):
        return [g for g in range(self.nops) if self.rot[g, k] == k]

    def D(self, kind: str, k: int, g: int) -> np.ndarray:
        """projective representation D^k(alpha) of Eq. 7 (g in the little group of k)."""
        return np.exp(2j * np.pi * np.dot(self.frac[k], self.w[g])) * self.O(kind, k, g)

    # ---- Algorithm 1 --------------------------------------------------------
    def dirac_characters(self, kind: str, k: int):
        """all Omega_gamma of the little group of k (S3)."""
        lg = self.little_group(k)
        Ds = [self.D(kind, k, g) for g in lg]
        h = len(lg)
        return [sum(Db @ Dg @ Db.conj().T for Db in Ds) / h for Dg in Ds]

    def adapt_one(self, kind: str, k: int, tol: float = 1e-8):
        """U^k and block offsets at one k (S3-S4).  The random Hermitian
        combination sum_gamma (c_gamma Omega_gamma + h.c.) is formed as
        (1/h) sum_beta D(beta) [sum_gamma c_gamma D(gamma)] D(beta)^dagger + h.c."""
        lg = self.little_group(k)
        Ds = [self.D(kind, k, g) for g in lg]
        n = Ds[0].shape[0]
        if len(lg) == 1:
            return np.eye(n, dtype=complex), np.array([0, n])
        rng = np.random.Generator(np.random.Philox(key=[self.seed, 1000 * k + (0 if kind == "ao" else 1)]))
        c = rng.standard_normal(len(lg)) + 1j * rng.standard_normal(len(lg))
        M = sum(ci * Di for ci, Di in zip(c, Ds))
        S = sum(Db @ M @ Db.conj().T for Db in Ds) / len(lg)
        Hc = S + S.conj().T
        ev, U = np.linalg.eigh(Hc)
        scale = max(np.abs(ev).max(), 1.0)
        cuts = [0] + [i for i in range(1, n) if ev[i] - ev[i - 1] > tol * scale] + [n]
        return U, np.array(cuts)

    def adapt(self, kind: str) -> BlockBasis:
        """U^k for every k: Algorithm 1 at the star representatives, S5 gauge elsewhere."""
        n = self.P[kind].shape[1]
        U = np.zeros((self.nk, n, n), dtype=complex)
        off = [None] * self.nk
        for kI in self.ir_list:
            U[kI], off[kI] = self.adapt_one(kind, int(kI))
        for k in range(self.nk):
            kI = self.ir_of[k]
            if k != kI:
                U[k] = self.O(kind, int(kI), int(self.op_of[k])) @ U[kI]
                off[k] = off[kI]
        return BlockBasis(U=U, off=off)

    def scramble(self, basis: BlockBasis, seed: int) -> BlockBasis:
        """an equally valid symmetry-adapted basis in a GENERAL gauge: U'^k = U^k . blockdiag(random unitaries), drawn
        independently at EVERY mesh point (the adapted basis is only fixed up to a unitary inside each isotypic block,
        PAPER.md:112-116).  Star members then no longer satisfy U^{k'} = O U^{k_I}, and O_block of Eq. 28
         is a genuine block-diagonal unitary instead of the identity."""
        U = np.empty_like(basis.U)
        for k in range(self.nk):
            rng = np.random.Generator(np.random.Philox(key=[seed, k]))
            R = np.zeros(basis.U[k].shape, dtype=complex)
            off = basis.off[k]
            for b in range(len(off) - 1):
                nb = off[b + 1] - off[b]
                Q, _ = np.linalg.qr(rng.standard_normal((nb, nb)) + 1j * rng.standard_normal((nb, nb)))
                R[off[b]:off[b + 1], off[b]:off[b + 1]] = Q
            U[k] = basis.U[k] @ R
        return BlockBasis(U=U, off=basis.off)

    # ---- Eq. 26-27: block-basis inputs, packed --------------------------------
    @staticmethod
    def pack_diag_blocks(X: np.ndarray, U: np.ndarray, off: np.ndarray, check: float = 1e-9):
        """X: [..., n, n] in the orbital basis -> packed diagonal blocks of U^dagger X U,
        [..., sum n_b^2] (block-major, row-major inside a block).  Off-block
        entries must vanish (they are exact zeros by symmetry)."""
        Xb = U.conj().T @ X @ U
        parts = []
        mask = np.ones(Xb.shape[-2:], dtype=bool)
        for b in range(len(off) - 1):
            s = slice(off[b], off[b + 1])
            parts.append(Xb[..., s, s].reshape(*Xb.shape[:-2], -1))
            mask[s, s] = False
        lead = np.abs(Xb).max()
        if mask.any() and np.abs(Xb[..., mask]).max() > check * max(lead, 1e-300):
            raise ValueError("input is not block diagonal in the symmetry-adapted basis")
        return np.concatenate(parts, axis=-1)

    @staticmethod
    def unpack_diag_blocks(packed: np.ndarray, off: np.ndarray) -> np.ndarray:
        """inverse of pack_diag_blocks' layout: [..., sum n_b^2] -> [..., n, n] block-diagonal."""
        n = off[-1]
        out = np.zeros(packed.shape[:-1] + (n, n), dtype=packed.dtype)
        o = 0
        for b in range(len(off) - 1):
            nb = off[b + 1] - off[b]
            out[..., off[b]:off[b + 1], off[b]:off[b + 1]] = packed[..., o:o + nb * nb].reshape(*packed.shape[:-1], nb, nb)
            o += nb * nb
        return out

    def block_V2(self, V2: np.ndarray, k1: int, k2: int, ao: BlockBasis, aux: BlockBasis,
                 thresh: float = 1e-9, vmax: float | None = None, triples=None):
        """V2 = V^{k2,k1}_{Q,bj} [naux,nao,nao] (orbital basis) ->
        (triples [nt,3] of (p, alpha, iota), packed block-basis tensor).

        V2blk_{P,a,i} = sum conj(Uaux^q_{Q,P}) conj(U^{k2}_{b,a}) V2_{Q,bj} U^{k1}_{j,i}
        (Eq. 27, with q = k1 - k2 the auxiliary momentum of V^{k2,k1}).
        A triple is allowed iff its block has an entry above thresh * max|V| (S6).
        Packed layout: aux block p major; inside p a matrix [n_p][N_p] whose
        columns are the allowed (alpha, iota) segments in triple order, each
        segment [a][i] row-major."""
        q = self.sub(k1, k2)
        T = np.einsum("QP,Qbj->Pbj", aux.U[q].conj(), V2, optimize=True)
        T = np.einsum("ba,Pbj->Paj", ao.U[k2].conj(), T, optimize=True)
        T = T @ ao.U[k1]
        op, o2, o1 = aux.off[q], ao.off[k2], ao.off[k1]
        if vmax is None:
            vmax = np.abs(T).max()
        if triples is None:
            triples = []
            for p in range(len(op) - 1):
                for al in range(len(o2) - 1):
                    for io in range(len(o1) - 1):
                        blk = T[op[p]:op[p + 1], o2[al]:o2[al + 1], o1[io]:o1[io + 1]]
                        if np.abs(blk).max() > thresh * vmax:
                            triples.append((p, al, io))
            triples = np.array(triples, dtype=np.int32).reshape(-1, 3)
        chunks = []
        for p in range(len(op) - 1):
            segs = [T[op[p]:op[p + 1], o2[al]:o2[al + 1], o1[io]:o1[io + 1]].reshape(op[p + 1] - op[p], -1)
                    for (pp, al, io) in triples if pp == p]
            if segs:
                chunks.append(np.concatenate(segs, axis=1).ravel())
        packed = np.concatenate(chunks) if chunks else np.zeros(0, dtype=complex)
        return triples, packed
