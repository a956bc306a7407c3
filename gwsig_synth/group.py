"""Space-group machinery for the synthetic crystals (input generation only).

Conventions (checked against PAPER.md Eq. 2-3, lines 39-67):
  * rows of ``a`` are the primitive vectors; a fractional column vector r has
    cartesian image a^T r; k.R = 2 pi sum_i k_i R_i with k, R fractional.
  * a space-group element acts on fractional coordinates as r -> W r + w
    ({alpha | v(alpha)}); its cartesian rotation is R = a^T W a^-T.
  * atom x (cell 0) is sent to atom perm[x] in cell shift[x] (integer):
    W tau_x + w = tau_perm[x] + shift[x]   ("translation vector between rotated
    and original atom").
  * k transforms as a row vector: k~ = k W^-1 (mod 1)  (alpha k = k~ + K).
  * real Wigner matrices: Y_m(R^-1 r) = sum_m' Y_m'(r) D_m'm   (PAPER.md:65,
    Eq. 4; improper operations need no special case because the harmonics are
    evaluated on the rotated point directly, which yields the (-1)^l of line 67).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass
from functools import lru_cache

import numpy as np

# --------------------------------------------------------------------------
# real harmonic polynomials, l = 0..4, explicit (mutually orthogonal on S^2)
# --------------------------------------------------------------------------


def _raw_harmonics(l: int, p: np.ndarray) -> np.ndarray:
    x, y, z = p[:, 0], p[:, 1], p[:, 2]
    r2 = x * x + y * y + z * z
    if l == 0:
        f = [np.ones_like(x)]
    elif l == 1:
        f = [x, y, z]
    elif l == 2:
        f = [x * y, y * z, 3 * z * z - r2, x * z, x * x - y * y]
    elif l == 3:
        f = [z * (5 * z * z - 3 * r2),
             x * (5 * z * z - r2), y * (5 * z * z - r2),
             z * (x * x - y * y), x * y * z,
             x * (x * x - 3 * y * y), y * (3 * x * x - y * y)]
    elif l == 4:
        f = [35 * z ** 4 - 30 * z * z * r2 + 3 * r2 * r2,
             x * z * (7 * z * z - 3 * r2), y * z * (7 * z * z - 3 * r2),
             (x * x - y * y) * (7 * z * z - r2), x * y * (7 * z * z - r2),
             x * z * (x * x - 3 * y * y), y * z * (3 * x * x - y * y),
             x ** 4 - 6 * x * x * y * y + y ** 4, x * y * (x * x - y * y)]
    else:
        raise ValueError("l up to 4 only")
    return np.stack(f, axis=1)


@lru_cache(maxsize=None)
def _sphere_quadrature():
    """Gauss-Legendre in cos(theta) x uniform in phi; exact for polynomials of
    degree <= 23 in (x,y,z) restricted to the unit sphere.  Weights sum to 1."""
    nu, nphi = 16, 32
    u, wu = np.polynomial.legendre.leggauss(nu)
    phi = 2 * np.pi * (np.arange(nphi) + 0.5) / nphi
    s = np.sqrt(1 - u * u)
    pts = np.stack([np.outer(s, np.cos(phi)).ravel(),
                    np.outer(s, np.sin(phi)).ravel(),
                    np.repeat(u, nphi)], axis=1)
    w = np.repeat(wu, nphi) / (2.0 * nphi)
    return pts, w


@lru_cache(maxsize=None)
def _harmonic_norms(l: int) -> np.ndarray:
    pts, w = _sphere_quadrature()
    f = _raw_harmonics(l, pts)
    gram = (f * w[:, None]).T @ f
    off = gram - np.diag(np.diag(gram))
    assert np.abs(off).max() < 1e-12 * np.abs(gram).max(), "harmonics not orthogonal"
    return 1.0 / np.sqrt(np.diag(gram))


def real_harmonics(l: int, pts: np.ndarray) -> np.ndarray:
    """[npts, 2l+1] real harmonic polynomials of degree l, orthonormal under the
    sphere average.  For l=1 the order is (x, y, z) so that D^1 = R."""
    return _raw_harmonics(l, np.asarray(pts, float)) * _harmonic_norms(l)[None, :]


def wigner_D_real(l: int, R: np.ndarray) -> np.ndarray:
    """D[m', m] with Y_m(R^-1 r) = sum_m' Y_m'(r) D[m', m]  (Eq. 4).
    Computed by exact quadrature of <Y_m' | Y_m o R^-1> on the sphere."""
    pts, w = _sphere_quadrature()
    Rinv = np.linalg.inv(R)
    ya = real_harmonics(l, pts)
    yb = real_harmonics(l, pts @ Rinv.T)          # rows are R^-1 r
    return (ya * w[:, None]).T @ yb


# --------------------------------------------------------------------------
# lattice point group and space group
# --------------------------------------------------------------------------


def lattice_point_group(a: np.ndarray) -> list[np.ndarray]:
    """All integer W (entries in {-1,0,1}, |det W| = 1) with W^T g W = g, g = a a^T
    (SURVEY 8(c) G2).  Identity first, otherwise itertools.product order."""
    g = a @ a.T
    out = []
    for ent in itertools.product((-1, 0, 1), repeat=9):
        W = np.array(ent, dtype=np.int64).reshape(3, 3)
        if abs(round(np.linalg.det(W))) != 1:
            continue
        if np.abs(W.T @ g @ W - g).max() < 1e-9 * np.abs(g).max():
            out.append(W)
    ident = [i for i, W in enumerate(out) if np.array_equal(W, np.eye(3, dtype=np.int64))]
    out.insert(0, out.pop(ident[0]))
    return out


@dataclass
class SpaceGroup:
    """Space-group operations of a crystal, in input order (identity first)."""
    a: np.ndarray            # [3,3] rows = primitive vectors
    W: np.ndarray            # [nops,3,3] int, fractional rotation parts
    w: np.ndarray            # [nops,3] fractional translations in [0,1)
    perm: np.ndarray         # [nops,natom] atom x -> perm[x]
    shift: np.ndarray        # [nops,natom,3] int lattice shift s_x
    Rcart: np.ndarray        # [nops,3,3] cartesian rotations

    @property
    def nops(self) -> int:
        return self.W.shape[0]

    def rep_real(self, func_atom: np.ndarray, func_shells: list[list[int]]) -> np.ndarray:
        """k-independent real representation [nops, n, n]:
        P[(perm[x], shell, m'), (x, shell, m)] = D^l_{m'm}(alpha)   (Eq. 3-4).
        ``func_shells[x]`` lists the l of every shell on atom x (atom-major,
        shell-major, m in harmonic order); ``func_atom`` gives the atom of each
        basis function and fixes n."""
        natom = len(func_shells)
        n = len(func_atom)
        start = np.zeros(natom + 1, dtype=int)
        for x in range(natom):
            start[x + 1] = start[x] + sum(2 * l + 1 for l in func_shells[x])
        assert start[-1] == n
        P = np.zeros((self.nops, n, n))
        for g in range(self.nops):
            Dl = {}
            for x in range(natom):
                y = self.perm[g, x]
                assert func_shells[x] == func_shells[y], "mapped atoms must carry equal shells"
                o = 0
                for l in func_shells[x]:
                    if l not in Dl:
                        Dl[l] = wigner_D_real(l, self.Rcart[g])
                    d = 2 * l + 1
                    P[g, start[y] + o:start[y] + o + d, start[x] + o:start[x] + o + d] = Dl[l]
                    o += d
        return P


def find_space_group(a: np.ndarray, pos: np.ndarray, species: np.ndarray) -> SpaceGroup:
    """Space group of (a, pos, species) by trial."""
    a = np.asarray(a, float)
    pos = np.asarray(pos, float)
    species = np.asarray(species)
    natom = len(pos)
    Ws, ws, perms, shifts = [], [], [], []
    for W in lattice_point_group(a):
        found = False
        for x0 in range(natom):
            if species[x0] != species[0]:
                continue
            w = pos[x0] - W @ pos[0]
            w = w - np.floor(w + 1e-9)
            perm = np.zeros(natom, dtype=int)
            shift = np.zeros((natom, 3), dtype=int)
            ok = True
            for x in range(natom):
                img = W @ pos[x] + w
                hit = -1
                for y in range(natom):
                    if species[y] != species[x]:
                        continue
                    d = img - pos[y]
                    dr = np.round(d)
                    if np.abs(d - dr).max() < 1e-7:
                        hit = y
                        shift[x] = dr.astype(int)
                        break
                if hit < 0:
                    ok = False
                    break
                perm[x] = hit
            if ok:
                if found:
                    raise ValueError("cell is not primitive: two translations for one rotation")
                found = True
                Ws.append(W)
                ws.append(w)
                perms.append(perm)
                shifts.append(shift)
    W = np.array(Ws, dtype=np.int64)
    ainvT = np.linalg.inv(a).T
    Rc = np.array([a.T @ Wi @ ainvT for Wi in W])
    return SpaceGroup(a=a, W=W, w=np.array(ws), perm=np.array(perms), shift=np.array(shifts), Rcart=Rc)


# --------------------------------------------------------------------------
# k mesh
# --------------------------------------------------------------------------


class KMesh:
    """Gamma-centred N1 x N2 x N3 mesh; k = n / N, index
    (n0*N1 + n1)*N2 + n2; all momentum arithmetic is exact on integers."""

    def __init__(self, mesh):
        self.N = np.array(mesh, dtype=np.int64)
        self.nk = int(np.prod(self.N))
        n0, n1, n2 = np.meshgrid(*[np.arange(m) for m in self.N], indexing="ij")
        self.n = np.stack([n0.ravel(), n1.ravel(), n2.ravel()], axis=1)   # [nk,3] ints
        self.frac = self.n / self.N[None, :]

    def index(self, n) -> np.ndarray:
        n = np.mod(np.asarray(n, dtype=np.int64), self.N)
        return (n[..., 0] * self.N[1] + n[..., 1]) * self.N[2] + n[..., 2]

    def sub(self, k, q):
        """index of k - q."""
        return self.index(self.n[k] - self.n[q])

    def rotate(self, W: np.ndarray) -> np.ndarray:
        """[nk] index of k~ = k W^-1 for every k."""
        Winv = np.rint(np.linalg.inv(W)).astype(np.int64)
        assert np.array_equal(Winv @ W, np.eye(3, dtype=np.int64))
        # k~_j N_j = sum_i n_i Winv[i,j] N_j / N_i must be an integer
        num = np.zeros_like(self.n)
        for j in range(3):
            acc = np.zeros(self.nk, dtype=np.int64)
            for i in range(3):
                t = self.n[:, i] * Winv[i, j] * self.N[j]
                if np.any(t % self.N[i] != 0):
                    raise ValueError("rotation does not map the k mesh onto itself")
                acc += t // self.N[i]
            num[:, j] = acc
        return self.index(num)

    def stars(self, sg: SpaceGroup):
        """(ir_list, ir_of, op_of): representative = first star member in index
        order, op_of[k'] = first operation in input order with alpha k_I = k'
        (SURVEY 8(c) A4).  Space-group operations only, no time reversal (A3)."""
        rot = np.stack([self.rotate(sg.W[g]) for g in range(sg.nops)])     # [nops, nk]
        ir_of = -np.ones(self.nk, dtype=np.int64)
        op_of = -np.ones(self.nk, dtype=np.int64)
        ir_list = []
        for k in range(self.nk):
            if ir_of[k] >= 0:
                continue
            ir_list.append(k)
            for g in range(sg.nops):
                kp = rot[g, k]
                if ir_of[kp] < 0:
                    ir_of[kp] = k
                    op_of[kp] = g
        return np.array(ir_list), ir_of, op_of, rot


def rep_at_k(P: np.ndarray, func_atom: np.ndarray, shift: np.ndarray, ktilde_frac: np.ndarray) -> np.ndarray:
    """O^k(alpha^) = P . diag(exp(-2 pi i k~ . s_x))  for one operation (Eq. 3,
    PAPER.md:58-61): column (x, m) carries the phase of its atom x; the result
    maps k -> k~ (X^{k~} = O X^k O^dagger, Eq. 22)."""
    ph = np.exp(-2j * np.pi * (shift @ ktilde_frac))        # [natom]
    return P * ph[func_atom][None, :]
