"""CPU ORACLE for the GW self-energy (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this module.  It shares no code with the
CUDA path (``paper_2405_09494_b200/``) and imports nothing from it.

What it computes -- the plain definition, Eq. 16 of the paper,
in the ORBITAL basis, on the FULL Brillouin zone, with NO symmetry used anywhere:

    Sigma_ij(k, tau) = -(1/Nk) sum_{q in BZ} sum_{Q,Q'} sum_{a,b}
          V^{k,k-q}_{Q,ia}  G_ab(k-q, tau)  W~_{QQ'}(q, tau)  V^{k-q,k}_{Q',bj}

Readings of the garbled typesetting of Eq. 16 (A1/A6): W~ is the
paper's P^q(tau) (Eq. 19); Q belongs to the first V
(momenta k, k-q; auxiliary momentum -q), Q' to the second (auxiliary momentum
+q = k - (k-q)); one spin channel.

Both V tensors are taken from the caller as independent inputs (``V_pair(k1,k2)``
returns V^{k1,k2}_{Q,ij} as [naux, nao, nao]); the oracle does NOT assume the
conjugation relation between them.

Two implementations:
  * ``sigma_brute``  -- seven explicit nested Python loops (tiny inputs only);
  * ``sigma_ref``    -- the same sum as three plain matrix products per (k,q),
                        vectorised over tau with numpy.matmul (library primitive
                        as a step; no blocking / fusion / reordering).  This is
                        the timed CPU baseline.
Pins: tests/test_oracle_pins.py (brute force, scalar closed forms, bilinearity,
gauge covariance, symmetry covariance, Hermiticity, irrep-block zeros).
Parity status: pinned by closed forms / invariants; absolute values of Sigma for
the synthetic crystals have no external reference (the paper prints none).
"""
from __future__ import annotations

from typing import Callable, Sequence

import numpy as np


def sigma_brute(nk: int, sub: Callable[[int, int], int], G: np.ndarray, W: np.ndarray,
                V_pair: Callable[[int, int], np.ndarray], ks: Sequence[int]) -> np.ndarray:
    """Eq. 16 by explicit loops.  G: [nk, ntau, nao, nao], W: [nk, ntau, naux, naux].
    Returns [len(ks), ntau, nao, nao]."""
    ntau, nao = G.shape[1], G.shape[2]
    naux = W.shape[2]
    out = np.zeros((len(ks), ntau, nao, nao), dtype=complex)
    for ik, k in enumerate(ks):
        for q in range(nk):
            kq = int(sub(k, q))
            Va = V_pair(k, kq)          # V^{k,k-q}_{Q,ia}
            Vb = V_pair(kq, k)          # V^{k-q,k}_{Q',bj}
            for t in range(ntau):
                for i in range(nao):
                    for j in range(nao):
                        acc = 0.0 + 0.0j
                        for Q in range(naux):
                            for Qp in range(naux):
                                w = W[q, t, Q, Qp]
                                for a in range(nao):
                                    for b in range(nao):
                                        acc += Va[Q, i, a] * G[kq, t, a, b] * w * Vb[Qp, b, j]
                        out[ik, t, i, j] += acc
    return -out / nk


def sigma_ref(nk: int, sub: Callable[[int, int], int],
              G_of: Callable[[int], np.ndarray], W_of: Callable[[int], np.ndarray],
              V_pair: Callable[[int, int], np.ndarray], ks: Sequence[int]) -> np.ndarray:
    """Eq. 16 as three matrix products per (k, q) -- the order of Algorithm 4
    (PAPER.md:340-347): X1 = V G, X2 = X1 P, Sigma^{k,q} = X2 V; then the q sum
    and the -1/Nk prefactor.

    G_of(k) -> [nt, nao, nao] and W_of(q) -> [nt, naux, naux] return the tau
    points wanted (any subset: Sigma is pointwise in tau).
    Returns [len(ks), nt, nao, nao]."""
    out = None
    for ik, k in enumerate(ks):
        for q in range(nk):
            kq = int(sub(k, q))
            Va = V_pair(k, kq)                                   # [Q, i, a]
            Vb = V_pair(kq, k)                                   # [Q', b, j]
            g = G_of(kq)                                         # [t, a, b]
            w = W_of(q)                                          # [t, Q, Q']
            nt, nao = g.shape[0], g.shape[1]
            naux = w.shape[1]
            if out is None:
                out = np.zeros((len(ks), nt, nao, nao), dtype=complex)
            # X1[t, Q, i, b] = sum_a Va[Q, i, a] G[t, a, b]
            X1 = np.matmul(Va.reshape(1, naux * nao, nao), g).reshape(nt, naux, nao * nao)
            # X2[t, Q', i, b] = sum_Q W[t, Q, Q'] X1[t, Q, i, b]
            X2 = np.matmul(w.transpose(0, 2, 1), X1).reshape(nt, naux, nao, nao)
            # S[t, i, j] = sum_{Q', b} X2[t, Q', i, b] Vb[Q', b, j]
            X2 = X2.transpose(0, 2, 1, 3).reshape(nt, nao, naux * nao)
            out[ik] += np.matmul(X2, Vb.reshape(1, naux * nao, nao))
    return -out / nk


def flops_per_output(nk: int, nao: int, naux: int) -> float:
    """real flops sigma_ref spends per (k, tau) output: Nk * 8 (2A + B),
    A = naux nao^3, B = naux^2 nao^2 (8 flop per complex multiply-add)."""
    return nk * 8.0 * (2.0 * naux * nao ** 3 + float(naux) ** 2 * nao ** 2)
