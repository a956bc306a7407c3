"""CPU ORACLE for the bare bubble P0^q(tau) (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  It shares no code with the CUDA path and imports nothing from it.

What it computes -- the plain definition, Eq. 20 of the paper, one spin channel (the spin sums of
Eq. 20 are a factor the caller applies), ORBITAL basis, FULL Brillouin zone, no symmetry:

    P0^q_{QQ'}(tau_n) = -(1/Nk) sum_k sum_{abcd}  V^{k,k+q}_{Q,da}  G^k_{cd}(-tau_n)  G^{k+q}_{ab}(tau_n)  V^{k+q,k}_{Q',bc}

Readings (A23): Eq. 20 is typeset with scrambled indices; the index pattern above is the one Algorithm 3
executes (X1 = V^{k,k+q} G^k(-tau), X2 = V^{k+q,k} G^{k+q}(tau), P0 = X1 X2).  G(-tau) is not an input of its
own: fermionic antiperiodicity, G(-tau) = -G(beta - tau), which on the uniform grid tau_n = n beta/(ntau-1) is the reversed
grid index, G(-tau_n) = -G[ntau-1-n].  Both V tensors are independent inputs (``V_pair(k1, k2)`` -> V^{k1,k2}_{Q,ij}).

``p0_brute`` is the sum as explicit loops (tiny inputs); ``p0_ref`` follows Algorithm 3: two products with G, then the
contraction over the orbital pair.  Pins (tests/test_oracle_pins.py): brute force, an independent einsum statement, the
single-level closed form P0 = |v|^2 n_F (1 - n_F) (tau-independent static susceptibility of one level), invariance under
orbital gauge changes and covariance under auxiliary ones, Hermiticity.
Parity status: pinned by those; absolute values for the synthetic crystals have no external reference.
"""
from __future__ import annotations

from typing import Callable, Sequence

import numpy as np


def g_minus_tau(G: np.ndarray) -> np.ndarray:
    """G(-tau_n) = -G(beta - tau_n) = -G[ntau-1-n] on the uniform grid (first axis = tau)."""
    return -G[::-1]


def p0_brute(nk: int, add: Callable[[int, int], int], G: np.ndarray, V_pair: Callable[[int, int], np.ndarray],
             qs: Sequence[int]) -> np.ndarray:
    """Eq. 20 by explicit loops.  G: [nk, ntau, nao, nao] on the full uniform grid.  Returns [len(qs), ntau, naux, naux]."""
    ntau, nao = G.shape[1], G.shape[2]
    out = None
    for iq, q in enumerate(qs):
        for k in range(nk):
            kq = int(add(k, q))
            Va = V_pair(k, kq)          # V^{k,k+q}_{Q,da}
            Vb = V_pair(kq, k)          # V^{k+q,k}_{Q',bc}
            naux = Va.shape[0]
            if out is None:
                out = np.zeros((len(qs), ntau, naux, naux), dtype=complex)
            for n in range(ntau):
                Gm = -G[k, ntau - 1 - n]                 # G^k(-tau_n)
                Gp = G[kq, n]                            # G^{k+q}(tau_n)
                for Q in range(naux):
                    for Qp in range(naux):
                        acc = 0.0 + 0.0j
                        for a in range(nao):
                            for b in range(nao):
                                for c in range(nao):
                                    for d in range(nao):
                                        acc += Va[Q, d, a] * Gm[c, d] * Gp[a, b] * Vb[Qp, b, c]
                        out[iq, n, Q, Qp] += acc
    return -out / nk


def p0_ref(nk: int, add: Callable[[int, int], int], G_of: Callable[[int], np.ndarray],
           V_pair: Callable[[int, int], np.ndarray], qs: Sequence[int], tau_idx: Sequence[int] | None = None) -> np.ndarray:
    """Eq. 20 in the order of Algorithm 3: per (q, k)
        X1[t, Q, c, a] = sum_d G^k_{cd}(-tau_t) V^{k,k+q}_{Q,da},   X2[t, Q', a, c] = sum_b G^{k+q}_{ab}(tau_t) V^{k+q,k}_{Q',bc},
        P0^{q,k}[t, Q, Q'] = sum_{a,c} X1[t, Q, c, a] X2[t, Q', a, c];  then the k sum and the -1/Nk prefactor.
    G_of(k) -> [ntau, nao, nao] on the FULL grid (the reversal for G(-tau) needs it); tau_idx selects the outputs.
    Returns [len(qs), len(tau_idx), naux, naux]."""
    out = None
    for iq, q in enumerate(qs):
        for k in range(nk):
            kq = int(add(k, q))
            Va, Vb = V_pair(k, kq), V_pair(kq, k)
            Gk, Gq = G_of(k), G_of(kq)
            ntau, nao = Gk.shape[0], Gk.shape[1]
            naux = Va.shape[0]
            ti = np.arange(ntau) if tau_idx is None else np.asarray(tau_idx)
            if out is None:
                out = np.zeros((len(qs), len(ti), naux, naux), dtype=complex)
            Gm = g_minus_tau(Gk)[ti]                                     # [t, c, d]
            Gp = Gq[ti]                                                  # [t, a, b]
            X1 = np.matmul(Gm[:, None], Va[None])                        # [t, Q, c, a]
            X2 = np.matmul(Gp[:, None], Vb[None])                        # [t, Q', a, c]
            A = X1.reshape(len(ti), naux, nao * nao)                     # (c, a)
            Bm = X2.transpose(0, 1, 3, 2).reshape(len(ti), naux, nao * nao)   # (c, a)
            out[iq] += np.matmul(A, Bm.transpose(0, 2, 1))
    return -out / nk
