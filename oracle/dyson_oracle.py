"""CPU ORACLE for the auxiliary function P^q(tau) from the bare bubble (TEST INFRASTRUCTURE -- not a product path).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may
import this module.  It shares no code with the CUDA path and imports nothing from it.

What it computes -- Eq. 19 of the paper, per momentum q:

    P0(i Omega_n) = sum_t  Tf[n, t] P0(tau_t)                      (tau -> i Omega, the transform matrix is an INPUT)
    P(i Omega_n)  = [1 - P0(i Omega_n)]^{-1} P0(i Omega_n)          (Eq. 19a, the geometric series summed)
    P(tau_t)      = sum_n  Tb[t, n] P(i Omega_n)                   (Eq. 19b: Tb[t, n] = e^{-i Omega_n tau_t} / beta on a plain grid)

The paper works on sparse intermediate-representation grids; those transforms are matrices of exactly this
shape, so the grids never enter: Tf [nw, ntau] and Tb [ntau, nw] are supplied by the caller (reading A24 of DESIGN.md).
``dyson_p_loops`` spells the solve out by Gauss-Jordan elimination with partial pivoting in explicit loops (small inputs),
``dyson_p_ref`` uses numpy.linalg.solve.  Pins (tests/test_oracle_pins.py): loops vs ref, the scalar closed form
p0 / (1 - p0), the geometric series sum_{n>=1} P0^n for small ||P0||, the resolvent identity P - P0 = P0 P = P P0, and the
commuting-diagonal case.
"""
from __future__ import annotations

import numpy as np


def dyson_p_ref(P0: np.ndarray, Tf: np.ndarray, Tb: np.ndarray) -> np.ndarray:
    """P0: [nq, ntau, n, n]; Tf: [nw, ntau]; Tb: [ntau, nw].  Returns P [nq, ntau, n, n]."""
    n = P0.shape[-1]
    P0w = np.einsum("wt,qtab->qwab", Tf, P0)
    Pw = np.linalg.solve(np.eye(n)[None, None] - P0w, P0w)
    return np.einsum("tw,qwab->qtab", Tb, Pw)


def dyson_p_loops(P0: np.ndarray, Tf: np.ndarray, Tb: np.ndarray) -> np.ndarray:
    nq, ntau, n, _ = P0.shape
    nw = Tf.shape[0]
    out = np.zeros_like(P0, dtype=complex)
    for q in range(nq):
        Pw = np.zeros((nw, n, n), dtype=complex)
        for w in range(nw):
            A0 = np.zeros((n, n), dtype=complex)
            for t in range(ntau):
                A0 += Tf[w, t] * P0[q, t]
            M = np.concatenate([np.eye(n) - A0, A0], axis=1)          # [1 - P0 | P0]
            for c in range(n):
                piv = c + int(np.argmax(np.abs(M[c:, c])))
                M[[c, piv]] = M[[piv, c]]
                M[c] = M[c] / M[c, c]
                for r in range(n):
                    if r != c:
                        M[r] = M[r] - M[r, c] * M[c]
            Pw[w] = M[:, n:]
        for t in range(ntau):
            for w in range(nw):
                out[q, t] += Tb[t, w] * Pw[w]
    return out
