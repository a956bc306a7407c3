"""CPU ORACLE for the block-basis transform of the three-index tensor (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  It shares no code with the CUDA path and imports nothing from it.

What it computes -- Eq. 27 of the paper, C_block = U^{ki dagger} U^{q dagger} C U^{kj}, written for the one
stored tensor of this build, V2 = V^{k2,k1}_{Q,bj} (first momentum k2, second k1, auxiliary momentum q = k1 - k2):

    V2blk_{P,a,i} = sum_{Q,b,j}  conj(Uaux^q_{Q,P})  conj(U^{k2}_{b,a})  V2_{Q,b,j}  U^{k1}_{j,i}

(the first orbital index transforms with U^dagger like a bra, the second with U like a ket, the auxiliary index with
U_aux^dagger; Eq. 26 is the two-index case X_block = U^dagger X U).  ``block_transform_brute`` is the sum as loops,
``block_transform_ref`` three tensor contractions.  Pins (tests/test_oracle_pins.py): brute force, the inverse transform,
norm preservation, and -- the pin that fixes which index gets which conjugation -- Sigma evaluated by the separately pinned
``sigma_ref`` from block-basis G, W and V equals U^dagger Sigma U.
"""
from __future__ import annotations

import numpy as np


def block_transform_brute(V2: np.ndarray, Uaux_q: np.ndarray, U_k2: np.ndarray, U_k1: np.ndarray) -> np.ndarray:
    naux, nao = V2.shape[0], V2.shape[1]
    out = np.zeros_like(V2, dtype=complex)
    for P in range(naux):
        for a in range(nao):
            for i in range(nao):
                acc = 0.0 + 0.0j
                for Q in range(naux):
                    for b in range(nao):
                        for j in range(nao):
                            acc += np.conj(Uaux_q[Q, P]) * np.conj(U_k2[b, a]) * V2[Q, b, j] * U_k1[j, i]
                out[P, a, i] = acc
    return out


def block_transform_ref(V2: np.ndarray, Uaux_q: np.ndarray, U_k2: np.ndarray, U_k1: np.ndarray) -> np.ndarray:
    """Eq. 27 as three contractions, one index at a time: aux, first orbital, second orbital."""
    T = np.tensordot(Uaux_q.conj().T, V2, axes=(1, 0))            # [P, b, j]
    T = np.matmul(U_k2.conj().T[None], T)                          # [P, a, j]
    return np.matmul(T, U_k1[None])                                # [P, a, i]
