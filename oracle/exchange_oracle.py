"""CPU ORACLE for the Hartree-Fock exchange self-energy (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  It shares no code with the CUDA path and imports nothing from it.

What it computes -- the plain definition, Eq. 21c of the paper, one spin channel, in the ORBITAL
basis, on the FULL Brillouin zone, no symmetry used:

    K^k_ij = -(1/Nk) sum_{k'} sum_{a,b} sum_Q  V^{k k'}_{ia}(Q)  gamma^{k'}_{ab}  V^{k' k}_{bj}(Q)

with gamma^k = G^k(tau = 0^-) the density matrix.  Both V tensors are independent inputs
(``V_pair(k1, k2)`` -> V^{k1,k2}_{Q,ij} as [naux, nao, nao]); the conjugation relation is not assumed.

``exchange_brute`` is the sum as explicit loops (tiny inputs); ``exchange_ref`` is two matrix products per (k, k').
Pins (tests/test_oracle_pins.py): brute force, the scalar closed form K = -|v|^2 <gamma>, the paper's own relation
"Eq. 16 with W -> delta and G -> gamma" against the separately pinned ``sigma_ref``, gauge covariance, Hermiticity.
Parity status: pinned by those; absolute values for the synthetic crystals have no external reference.
"""
from __future__ import annotations

from typing import Callable, Sequence

import numpy as np


def exchange_brute(nk: int, gamma: np.ndarray, V_pair: Callable[[int, int], np.ndarray], ks: Sequence[int]) -> np.ndarray:
    """Eq. 21c by explicit loops.  gamma: [nk, nao, nao].  Returns [len(ks), nao, nao]."""
    nao = gamma.shape[1]
    out = np.zeros((len(ks), nao, nao), dtype=complex)
    for ik, k in enumerate(ks):
        for kp in range(nk):
            Va = V_pair(k, kp)           # V^{k k'}_{Q, i a}
            Vb = V_pair(kp, k)           # V^{k' k}_{Q, b j}
            naux = Va.shape[0]
            for i in range(nao):
                for j in range(nao):
                    acc = 0.0 + 0.0j
                    for Q in range(naux):
                        for a in range(nao):
                            for b in range(nao):
                                acc += Va[Q, i, a] * gamma[kp, a, b] * Vb[Q, b, j]
                    out[ik, i, j] += acc
    return -out / nk


def exchange_ref(nk: int, gamma_of: Callable[[int], np.ndarray], V_pair: Callable[[int, int], np.ndarray],
                 ks: Sequence[int]) -> np.ndarray:
    """Eq. 21c as two matrix products per (k, k'): X[Q,i,b] = sum_a V^{k k'}[Q,i,a] gamma^{k'}[a,b], then
    K += sum_{Q,b} X[Q,i,b] V^{k' k}[Q,b,j]; finally the k' sum and the -1/Nk prefactor.
    gamma_of(k) -> [nao, nao].  Returns [len(ks), nao, nao]."""
    out = None
    for ik, k in enumerate(ks):
        for kp in range(nk):
            Va = V_pair(k, kp)
            Vb = V_pair(kp, k)
            g = gamma_of(kp)
            naux, nao = Va.shape[0], Va.shape[1]
            if out is None:
                out = np.zeros((len(ks), nao, nao), dtype=complex)
            X = np.matmul(Va.reshape(naux * nao, nao), g).reshape(naux, nao, nao)          # [Q, i, b]
            out[ik] += np.matmul(X.transpose(1, 0, 2).reshape(nao, naux * nao), Vb.reshape(naux * nao, nao))
    return -out / nk
