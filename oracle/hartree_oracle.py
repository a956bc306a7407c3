"""CPU ORACLE for the Hartree self-energy (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  It shares no code with the CUDA path and imports nothing from it.

What it computes -- the plain definition, Eq. 21b of the paper, ONE spin channel (the sum over sigma_1
is a factor the caller applies, as for Eq. 16 / 20 / 21c: DESIGN.md readings A21, A23), in the ORBITAL basis, on the FULL
Brillouin zone, no symmetry used:

    J^k_ij = (1/Nk) sum_{k'} sum_{a,b} sum_Q  V^{k k}_{ij}(Q)  gamma^{k'}_{ab}  V^{k' k'}_{ba}(Q)

with gamma^k = G^k(tau = 0^-) the density matrix.  Only the momentum-diagonal pair tensors enter
(``V_diag(k)`` -> V^{k,k}_{Q,ij} as [naux, nao, nao]).

``hartree_brute`` is the sum as explicit loops (tiny inputs); ``hartree_ref`` follows the factorisation the formula
states -- the auxiliary density rho_Q = (1/Nk) sum_{k'} tr[gamma^{k'} V^{k'k'}(Q)], then J^k = sum_Q V^{kk}(Q) rho_Q.
Pins (tests/test_oracle_pins.py): brute force, the scalar closed form, an independent einsum statement, the Hartree energy
identity (1/Nk) sum_k tr[gamma^k J^k] = sum_Q rho_Q^2, invariance under orbital unitaries and real orthogonal auxiliary
rotations, and on a symmetric crystal: rho real, J Hermitian, J(gk) = O J(k) O^dagger.
Parity status: pinned by those; absolute values for the synthetic crystals have no external reference.
"""
from __future__ import annotations

from typing import Callable, Sequence

import numpy as np


def hartree_brute(nk: int, gamma: np.ndarray, V_diag: Callable[[int], np.ndarray], ks: Sequence[int]) -> np.ndarray:
    """Eq. 21b by explicit loops.  gamma: [nk, nao, nao].  Returns [len(ks), nao, nao]."""
    nao = gamma.shape[1]
    out = np.zeros((len(ks), nao, nao), dtype=complex)
    for ik, k in enumerate(ks):
        Vk = V_diag(k)
        naux = Vk.shape[0]
        for kp in range(nk):
            Vp = V_diag(kp)
            for i in range(nao):
                for j in range(nao):
                    acc = 0.0 + 0.0j
                    for Q in range(naux):
                        for a in range(nao):
                            for b in range(nao):
                                acc += Vk[Q, i, j] * gamma[kp, a, b] * Vp[Q, b, a]
                    out[ik, i, j] += acc
    return out / nk


def aux_density(nk: int, gamma_of: Callable[[int], np.ndarray], V_diag: Callable[[int], np.ndarray]) -> np.ndarray:
    """rho_Q = (1/Nk) sum_{k'} sum_{ab} gamma^{k'}_{ab} V^{k'k'}_{ba}(Q)  -> [naux]  (the k'-dependent factor of Eq. 21b)."""
    rho = None
    for kp in range(nk):
        Vp = V_diag(kp)
        g = gamma_of(kp)
        naux, nao = Vp.shape[0], Vp.shape[1]
        if rho is None:
            rho = np.zeros(naux, dtype=complex)
        # tr[gamma V(Q)] = sum_ab gamma_ab V_ba(Q)
        rho += np.matmul(Vp.transpose(0, 2, 1).reshape(naux, nao * nao), g.reshape(nao * nao))
    return rho / nk


def hartree_ref(nk: int, gamma_of: Callable[[int], np.ndarray], V_diag: Callable[[int], np.ndarray], ks: Sequence[int]) -> np.ndarray:
    """Eq. 21b as its two factors: rho (above), then J^k_ij = sum_Q V^{kk}_{ij}(Q) rho_Q.  Returns [len(ks), nao, nao]."""
    rho = aux_density(nk, gamma_of, V_diag)
    out = []
    for k in ks:
        Vk = V_diag(k)
        naux, nao = Vk.shape[0], Vk.shape[1]
        out.append(np.matmul(rho, Vk.reshape(naux, nao * nao)).reshape(nao, nao))
    return np.stack(out)
