"""Crystal structures of BASELINE.json's configs (shapes only).

Every structure stands in for one of the paper's solids (Table 1):
the real pySCF integrals are not available, so the orbital / auxiliary shell
lists only fix nao, naux and the representation content.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from .group import KMesh, SpaceGroup, find_space_group

_FCC = 0.5 * np.array([[0.0, 1.0, 1.0], [1.0, 0.0, 1.0], [1.0, 1.0, 0.0]])
_SC = np.eye(3)


def _hex(c_over_a: float) -> np.ndarray:
    return np.array([[1.0, 0.0, 0.0], [-0.5, np.sqrt(3.0) / 2.0, 0.0], [0.0, 0.0, c_over_a]])


def _shells(spec: str) -> list[int]:
    """'s2 p2 d1' -> [0,0,1,1,2]"""
    out = []
    for tok in spec.split():
        l = "spdfg".index(tok[0])
        out += [l] * int(tok[1:])
    return out


@dataclass
class Crystal:
    name: str
    a: np.ndarray                      # [3,3] rows = primitive vectors
    pos: np.ndarray                    # [natom,3] fractional
    species: np.ndarray                # [natom]
    ao_shells: list[list[int]]         # per atom, list of l
    aux_shells: list[list[int]]
    mesh: tuple[int, int, int]
    ntau: int
    beta: float
    nocc: int                          # occupied orbitals per k (A11)
    h_shells: int = 2                  # H(R), A_m(R): lattice-vector shells kept (A13)
    seed: int = 20240509
    sg: SpaceGroup = field(init=False)
    kmesh: KMesh = field(init=False)

    def __post_init__(self):
        self.a = np.asarray(self.a, float)
        self.pos = np.asarray(self.pos, float)
        self.species = np.asarray(self.species)
        self.sg = find_space_group(self.a, self.pos, self.species)
        self.kmesh = KMesh(self.mesh)
        self.ao_atom = np.concatenate([[x] * sum(2 * l + 1 for l in sh) for x, sh in enumerate(self.ao_shells)])
        self.aux_atom = np.concatenate([[x] * sum(2 * l + 1 for l in sh) for x, sh in enumerate(self.aux_shells)])
        self.nao = len(self.ao_atom)
        self.naux = len(self.aux_atom)
        self.natom = len(self.pos)
        self.P_ao = self.sg.rep_real(self.ao_atom, self.ao_shells)       # [nops,nao,nao] real
        self.P_aux = self.sg.rep_real(self.aux_atom, self.aux_shells)
        self.ao_start = np.concatenate([[0], np.cumsum([sum(2 * l + 1 for l in sh) for sh in self.ao_shells])])
        self.aux_start = np.concatenate([[0], np.cumsum([sum(2 * l + 1 for l in sh) for sh in self.aux_shells])])


CONFIG_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")


def make_crystal(name: str, **over) -> Crystal:
    """Structures of configs 2-5 plus small toys used by the CPU tests.
    (config 1 has no crystal: C1, random H(k) -- see tensors.RandomC1Inputs.)"""
    u = 3.0 / 8.0
    wz_pos = [[1 / 3, 2 / 3, 0.0], [2 / 3, 1 / 3, 0.5], [1 / 3, 2 / 3, u], [2 / 3, 1 / 3, 0.5 + u]]
    table = {
        # config 2: simple cubic, Oh, 1 atom, s+p+d, aux (s,p,d)x2
        "cfg2": dict(a=_SC, pos=[[0, 0, 0]], species=[0], ao=["s1 p1 d1"], aux=["s2 p2 d2"],
                     mesh=(4, 4, 4), ntau=64, beta=50.0, nocc=4, h_shells=2, seed=20240511),
        # config 3: diamond, Fd-3m, stands in for Si 6x6x6
        "cfg3": dict(a=_FCC, pos=[[0, 0, 0], [0.25, 0.25, 0.25]], species=[0, 0],
                     ao=["s2 p2 d1"] * 2, aux=["s6 p6 d4 f2"] * 2,
                     mesh=(6, 6, 6), ntau=104, beta=100.0, nocc=13, h_shells=3, seed=20240512),
        # config 4: wurtzite, P6_3mc, BN-like
        "cfg4": dict(a=_hex(1.633), pos=wz_pos, species=[0, 0, 1, 1],
                     ao=["s2 p2 d1"] * 4, aux=["s6 p6 d4 f2"] * 4,
                     mesh=(6, 6, 4), ntau=128, beta=100.0, nocc=26, h_shells=3, seed=20240513),
        # config 5: rock salt, Fm-3m, two species; aux list per SURVEY A14 (150 / atom)
        "cfg5": dict(a=_FCC, pos=[[0, 0, 0], [0.5, 0.5, 0.5]], species=[0, 1],
                     ao=["s3 p3 d2 f1"] * 2, aux=["s8 p8 d6 f10 g2"] * 2,
                     mesh=(8, 8, 8), ntau=136, beta=200.0, nocc=29, h_shells=3, seed=20240514),
        # ---- toys for fast CPU tests -------------------------------------
        "toy_sc": dict(a=_SC, pos=[[0, 0, 0]], species=[0], ao=["s1 p1"], aux=["s1 p1 d1"],
                       mesh=(2, 2, 2), ntau=3, beta=5.0, nocc=2, h_shells=2, seed=11),
        "toy_diamond": dict(a=_FCC, pos=[[0, 0, 0], [0.25, 0.25, 0.25]], species=[0, 0],
                            ao=["s1 p1"] * 2, aux=["s1 p1"] * 2,
                            mesh=(2, 2, 2), ntau=3, beta=8.0, nocc=4, h_shells=2, seed=12),
        "toy_diamond4": dict(a=_FCC, pos=[[0, 0, 0], [0.25, 0.25, 0.25]], species=[0, 0],
                             ao=["s1 p1"] * 2, aux=["s1 p1 d1"] * 2,
                             mesh=(4, 4, 4), ntau=2, beta=8.0, nocc=4, h_shells=2, seed=13),
        "toy_wurtzite": dict(a=_hex(1.633), pos=wz_pos, species=[0, 0, 1, 1],
                             ao=["s1 p1"] * 4, aux=["s1 p1"] * 4,
                             mesh=(2, 2, 2), ntau=2, beta=6.0, nocc=8, h_shells=2, seed=14),
        "toy_rocksalt": dict(a=_FCC, pos=[[0, 0, 0], [0.5, 0.5, 0.5]], species=[0, 1],
                             ao=["s1 p1"] * 2, aux=["s1 p1 d1"] * 2,
                             mesh=(2, 2, 2), ntau=2, beta=6.0, nocc=4, h_shells=2, seed=15),
        # lattices only (IBZ-count pins against Table 2)
        "zincblende": dict(a=_FCC, pos=[[0, 0, 0], [0.25, 0.25, 0.25]], species=[0, 1],
                           ao=["s1"] * 2, aux=["s1"] * 2, mesh=(2, 2, 2), ntau=2, beta=1.0, nocc=1, seed=16),
        "hex_bn": dict(a=_hex(2.66), pos=[[1 / 3, 2 / 3, 0.25], [2 / 3, 1 / 3, 0.75], [2 / 3, 1 / 3, 0.25], [1 / 3, 2 / 3, 0.75]],
                       species=[0, 0, 1, 1], ao=["s1"] * 4, aux=["s1"] * 4, mesh=(2, 2, 2), ntau=2, beta=1.0,
                       nocc=2, seed=17),
    }
    if name not in table:
        raise KeyError(f"unknown crystal {name!r}")
    t = dict(table[name])
    t.update(over)
    return Crystal(name=name, a=t["a"], pos=t["pos"], species=t["species"],
                   ao_shells=[_shells(s) for s in t["ao"]], aux_shells=[_shells(s) for s in t["aux"]],
                   mesh=tuple(t["mesh"]), ntau=t["ntau"], beta=t["beta"], nocc=t["nocc"],
                   h_shells=t.get("h_shells", 2), seed=t["seed"])
