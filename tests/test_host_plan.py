"""Host logic of the C-ABI library, no GPU: the library loads and exports every declared symbol, the
plan (stars, pair list, layouts) is right, error conventions hold, and the grouped-GEMM descriptors --
executed by a numpy interpreter -- reproduce the oracle in all three modes."""
import ctypes
import os
import re

import numpy as np
import pytest

from gwsig_synth import make_inputs
from paper_2405_09494_b200 import build as gw_build

gw_build.build()
from paper_2405_09494_b200 import binding as B                                   # noqa: E402
from paper_2405_09494_b200.pack import Configured, configure_from_crystal        # noqa: E402
from tests.helpers import fold_to_orbital, oracle_sigma, rel_err, run_plan_numpy  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "gwsig.h")).read()
    declared = set(re.findall(r"\b(gwsig_[a-z0-9_]+)\s*\(", hdr))
    declared -= {"gwsig_ctx", "gwsig_status", "gwsig_mode", "gwsig_engine"}
    lib = ctypes.CDLL(B.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert declared == set(B.EXPORTS)


def test_struct_layouts_match_header():
    assert (B.IDX2.itemsize, B.SEG.itemsize, B.PROBLEM.itemsize) == (24, 120, 144)


def test_no_cpu_fallback_without_device():
    lib = B.Gwsig(device=-1)
    inp = make_inputs("cfg1", mesh=(2, 1, 1), nao=2, naux=2, ntau=2, nocc=1)
    cfg = Configured(lib, B.FULL_BZ, np.eye(3), (2, 1, 1), 2, 2, 2, 1.0, None, None, None)
    z = np.zeros(64, complex)
    with pytest.raises(B.GwsigError) as e:
        lib.sigma_eval(z, z, z, z)
    assert e.value.code == -4 and "no CPU fallback" in str(e.value)


def test_stars_and_pairs_match_setup():
    inp = make_inputs("toy_diamond4")
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ)
    st = cfg.setup
    assert np.array_equal(cfg.ir_list, st.ir_list) and np.array_equal(cfg.ir_of, st.ir_of) and np.array_equal(cfg.op_of, st.op_of)
    assert len(cfg.ir_list) == 8                       # Table 2, Si 4x4x4
    assert cfg.npairs == 64 * 8
    for p in (0, 7, 8, 100, 511):
        k1, k2, q, off, ne = lib.pair_info(p)
        assert q == p // 8 and k1 == cfg.ir_list[p % 8] and k2 == st.sub(k1, q)
        assert off == p * inp.naux * inp.nao ** 2 and ne == inp.naux * inp.nao ** 2
    full, ex = lib.flop_counts()
    unit = inp.ntau * 8 * (2 * inp.naux * inp.nao ** 3 + inp.naux ** 2 * inp.nao ** 2)
    assert full == 64 * 64 * unit and ex == 64 * 8 * unit


def test_error_conventions():
    inp = make_inputs("toy_sc")
    cr, sg = inp.cr, inp.cr.sg
    lib = B.Gwsig(device=-1)
    with pytest.raises(B.GwsigError) as e:
        lib.set_lattice(cr.a, (2, 2, 0), cr.nao, cr.naux, 2, 1.0)
    assert e.value.code == -1
    lib.set_lattice(cr.a, (2, 3, 2), cr.nao, cr.naux, 2, 1.0)
    lib.set_atoms(cr.pos, cr.ao_atom, cr.aux_atom)
    with pytest.raises(B.GwsigError) as e:              # cubic rotations do not map a 2x3x2 mesh onto itself
        lib.set_symmetry(sg.W, sg.w, cr.P_ao, cr.P_aux, sg.shift, B.IBZ)
    assert e.value.code == -2
    lib.set_lattice(cr.a, cr.mesh, cr.nao, cr.naux, 2, 1.0)
    lib.set_atoms(cr.pos, cr.ao_atom, cr.aux_atom)
    bad = cr.P_ao.copy(); bad[3, 0, 0] += 0.1
    with pytest.raises(B.GwsigError) as e:              # non-orthogonal representation matrix
        lib.set_symmetry(sg.W, sg.w, bad, cr.P_aux, sg.shift, B.IBZ)
    assert e.value.code == -2
    lib.set_symmetry(sg.W, sg.w, cr.P_ao, cr.P_aux, sg.shift, B.IBZ_BLOCK)
    nk = lib.nk
    with pytest.raises(B.GwsigError) as e:              # blocks that do not tile [0, nao)
        lib.set_blocks([np.array([0, cr.nao - 1])] * nk, [np.array([0, cr.naux])] * nk)
    assert e.value.code == -3
    with pytest.raises(B.GwsigError) as e:              # a star member whose blocks differ from its representative's
        offs = [np.array([0, cr.nao])] * nk
        offs[1] = np.array([0, 1, cr.nao])
        lib.set_blocks(offs, [np.array([0, cr.naux])] * nk)
    assert e.value.code == -3
    lib.set_blocks([np.array([0, cr.nao])] * nk, [np.array([0, cr.naux])] * nk)
    npairs, _ = lib.pair_count()
    with pytest.raises(B.GwsigError) as e:              # triple with a block index out of range
        lib.set_triples(np.arange(npairs + 1), np.tile([0, 1, 0], (npairs, 1)))
    assert e.value.code == -3


@pytest.mark.parametrize("name,mode,push,nt", [
    ("cfg1s", B.FULL_BZ, None, None), ("cfg1s", B.FULL_BZ, 8, 1),
    ("toy_diamond", B.IBZ, None, None), ("toy_diamond", B.IBZ, 6, 2),
    ("toy_diamond", B.IBZ_BLOCK, None, None), ("toy_diamond", B.IBZ_BLOCK, 3, 2),
    ("toy_wurtzite", B.IBZ_BLOCK, None, None), ("toy_rocksalt", B.IBZ_BLOCK, 9, None),
])
def test_descriptors_reproduce_oracle(name, mode, push, nt):
    lib = B.Gwsig(device=-1)
    if name == "cfg1s":
        inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=5, ntau=3, beta=4.0, nocc=1, seed=2)
        cfg = Configured(lib, mode, np.eye(3), (2, 2, 1), 3, 5, 3, 4.0, None, None, None)
        Gf, Wf = inp.G_full(), inp.W_full()
        G, W = cfg.pack_GW(lambda k: Gf[k], lambda q: Wf[q])
    else:
        inp = make_inputs(name)
        cfg = configure_from_crystal(lib, inp.cr, mode)
        G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    sig = run_plan_numpy(cfg, inp, G, W, V, push_pairs=push, nt=nt)
    got = fold_to_orbital(cfg, inp, cfg.unpack_sigma(sig))
    ref = oracle_sigma(inp, range(inp.nk))
    for k in range(inp.nk):
        for t in range(inp.ntau):
            assert rel_err(got[k][t], ref[k, t]) < 1e-12, (k, t)
    if mode == B.IBZ_BLOCK:
        full, ex = lib.flop_counts()
        assert 0 < ex < full * len(cfg.ir_list) / inp.nk


def test_output_points_subset_descriptors():
    """gwsig_set_output_points: Sigma at a listed subset of wedge points equals the same rows of the full plan."""
    inp = make_inputs("toy_diamond")
    cfgs = []
    for pick in (None, lambda wedge: [wedge[1]]):
        lib = B.Gwsig(device=-1)
        cfg = configure_from_crystal(lib, inp.cr, B.IBZ_BLOCK, out_points=pick)
        G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
        V = cfg.pack_V(inp.V2_rows)
        cfgs.append((cfg, cfg.unpack_sigma(run_plan_numpy(cfg, inp, G, W, V))))
    (full_cfg, full), (sub_cfg, sub) = cfgs
    assert sub_cfg.npairs == inp.nk and list(sub_cfg.out_list) == [full_cfg.ir_list[1]]
    assert np.abs(sub[0] - full[1]).max() <= 1e-13 * np.abs(full[1]).max()
    lib = B.Gwsig(device=-1)
    with pytest.raises(B.GwsigError) as e:             # not a wedge representative
        non_wedge = [k for k in range(inp.nk) if k not in set(full_cfg.ir_list)][0]
        configure_from_crystal(lib, inp.cr, B.IBZ, out_points=[non_wedge])
    assert e.value.code == -1


def test_stage3_split_k_parts_tile_the_segments():
    """stage 3 cuts long segment lists into parts (and segments along P') that add into one Sigma block: the parts of
    a block must cover every (pair, triple, P') exactly once -- checked through the interpreter on a config whose K is
    long enough to be cut (ntau small keeps it cheap)."""
    inp = make_inputs("toy_diamond4")
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ, out_points=lambda wedge: [wedge[0], wedge[3]])
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    pr, sg, _ = lib.plan_get(0, cfg.npairs, 1, 3)
    ksum = {}
    for P in pr:
        ksum[int(P["c_off"])] = ksum.get(int(P["c_off"]), 0) + sum(int(sg[s]["K"]) for s in range(P["seg_begin"], P["seg_begin"] + P["seg_count"]))
    assert len(pr) > len(ksum), "expected split-K parts"          # more problems than output blocks
    assert all(v == inp.nk * inp.naux * inp.nao for v in ksum.values())
    sig = run_plan_numpy(cfg, inp, G, W, V)
    got = cfg.unpack_sigma(sig)
    ref = oracle_sigma(inp, [int(k) for k in cfg.out_list])
    for a in range(len(cfg.out_list)):
        for t in range(inp.ntau):
            assert rel_err(got[a][t], ref[a, t]) < 1e-12


@pytest.mark.parametrize("name", ["toy_diamond", "toy_wurtzite"])
def test_general_gauge_eq28_host_plan(name):
    """explicit U in a scrambled gauge (a different random unitary inside every block at EVERY mesh point): the library
    forms O_block = U^{k'}^dagger O U^{k_I} (Eq. 28) and its unfold + contraction descriptors, run by the numpy
    interpreter, reproduce the oracle; a U that mixes blocks is refused."""
    inp = make_inputs(name)
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ_BLOCK, scramble_gauge=5)
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    sig = run_plan_numpy(cfg, inp, G, W, V, push_pairs=cfg.nk1 * 3)
    got = fold_to_orbital(cfg, inp, cfg.unpack_sigma(sig))
    ref = oracle_sigma(inp, range(inp.nk))
    assert max(rel_err(got[k][t], ref[k, t]) for k in range(inp.nk) for t in range(inp.ntau)) < 1e-11
    # a basis that mixes two blocks at a star member (not the representative, whose O_block is U^dagger U = 1) is refused
    k_bad = next(k for k in range(cfg.nk) if len(cfg.ao.off[k]) > 2 and cfg.ir_of[k] != k)
    Ubad = cfg.ao.U.copy()
    o = cfg.ao.off[k_bad]
    Ubad[k_bad][:, [o[0], o[1]]] = (Ubad[k_bad][:, [o[0], o[1]]] @ np.array([[1, 1], [1, -1]])) / np.sqrt(2)
    with pytest.raises(B.GwsigError) as e:
        lib.set_blocks(cfg.ao.off, cfg.aux.off, Ubad, cfg.aux.U)
    assert e.value.code == -3


def test_exchange_plan_skips_stage_two():
    """N2 (Eq. 21c): the exchange call runs stage 1 and feeds stage 3 directly; the same descriptors, interpreted in numpy with
    Y = X, reproduce oracle/exchange_oracle.py in block mode."""
    import copy
    from tests.helpers import oracle_exchange
    inp = make_inputs("toy_diamond")
    cr1 = copy.copy(inp.cr)
    cr1.ntau = 1
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, cr1, B.IBZ_BLOCK)
    gam = lambda k: -inp.G_k(int(k))[-1]
    G, _ = cfg.pack_GW(lambda k: gam(k)[None], lambda q: np.zeros((1, inp.naux, inp.naux), complex))
    V = cfg.pack_V(inp.V2_rows)
    K = run_plan_numpy(cfg, inp, G, None, V, exchange=True)
    got = fold_to_orbital(cfg, inp, cfg.unpack_sigma(K))
    ref = oracle_exchange(inp, gam, range(inp.nk))
    assert max(rel_err(got[k][0], ref[k]) for k in range(inp.nk)) < 1e-11


@pytest.mark.parametrize("name,mode", [("cfg1s", B.FULL_BZ), ("toy_diamond", B.IBZ), ("toy_wurtzite", B.IBZ)])
def test_p0_plan_matches_oracle(name, mode):
    """N1 (Eq. 20 / Algorithm 3): the three P0 stages of the plan, run by the numpy interpreter, against oracle/p0_oracle.py:
    every wedge q (every q in FULL_BZ), every tau, several pushes and tau chunks."""
    from tests.helpers import oracle_p0, pack_V_p0, run_p0_plan_numpy
    lib = B.Gwsig(device=-1)
    if name == "cfg1s":
        inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=5, ntau=4, beta=4.0, nocc=1, seed=2)
        cfg = Configured(lib, mode, np.eye(3), inp.kmesh.N, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
        Gf = inp.G_full()
        G, _ = cfg.pack_GW(lambda k: Gf[k], lambda q: np.zeros((inp.ntau, inp.naux, inp.naux), complex))
    else:
        inp = make_inputs(name)
        cfg = configure_from_crystal(lib, inp.cr, mode)
        G, _ = cfg.pack_GW(inp.G_k, lambda q: np.zeros((inp.ntau, inp.naux, inp.naux), complex))
    V = pack_V_p0(cfg, inp)
    got = run_p0_plan_numpy(cfg, inp, G, V, push_pairs=5, nt=max(1, inp.ntau - 1))
    ref = oracle_p0(inp, cfg.out_list)
    scale = np.abs(ref).max()
    assert np.abs(got - ref).max() < 1e-12 * scale


@pytest.mark.parametrize("name", ["toy_diamond4", "toy_wurtzite"])
def test_vtransform_plan_matches_oracle(name):
    """N4 (Eq. 27): the three launches of gwsig_block_transform_v, run by the numpy interpreter, give the packed
    block-basis V2 that oracle/block_oracle.py gives (packed by the documented layout); U handed over in the S5 gauge is
    recognised (no unfold is planned: O_block = 1)."""
    from tests.helpers import oracle_packed_V, run_vtransform_numpy
    inp = make_inputs(name)
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ_BLOCK, pass_U=True)
    cfg.pack_V(inp.V2_rows)                               # finds the allowed triples and calls set_triples
    p0, n = 5, 11
    got = run_vtransform_numpy(cfg, inp, p0, n)
    ref = oracle_packed_V(cfg, inp, range(p0, p0 + n))
    assert got.shape == ref.shape and np.abs(got - ref).max() < 1e-13 * np.abs(ref).max()
    with pytest.raises(B.GwsigError):                      # S5 gauge recognised: the Eq. 28 unfold stages are not available
        lib.plan_get(0, 4, inp.ntau, 11)


@pytest.mark.parametrize("name", ["toy_diamond4", "toy_wurtzite"])
def test_dense_vtransform_plan_detects_the_allowed_blocks(name):
    """N4: the launches of gwsig_block_maxabs (plan stages 41, 42, 44: the Eq. 27 transform for EVERY block), run
    by the numpy interpreter BEFORE any triples are set, give the oracle's dense block-basis tensor; thresholding its block
    maxima gives the triples the CPU pre-step (symsetup.block_V2) finds."""
    from oracle.block_oracle import block_transform_ref
    from tests.helpers import run_dense_vtransform_numpy
    inp = make_inputs(name)
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ_BLOCK, pass_U=True)
    p0, n = 3, 9
    got = run_dense_vtransform_numpy(cfg, inp, p0, n)
    with pytest.raises(B.GwsigError):                      # the packed step 3 needs the triples
        lib.plan_get(p0, n, 1, 43)
    for l in range(n):
        k1, k2, q = lib.pair_info(p0 + l, with_layout=False)[:3]
        V2 = inp.V2_rows(k1, [k2])[0]
        ref = block_transform_ref(V2, cfg.aux.U[q], cfg.ao.U[k2], cfg.ao.U[k1])
        assert np.abs(got[l] - ref).max() < 1e-13 * np.abs(ref).max()
        trip, _ = cfg.setup.block_V2(V2, k1, k2, cfg.ao, cfg.aux)
        op, o2, o1 = cfg.aux.off[q], cfg.ao.off[k2], cfg.ao.off[k1]
        mine = [(b, al, io) for b in range(len(op) - 1) for al in range(len(o2) - 1) for io in range(len(o1) - 1)
                if np.abs(got[l][op[b]:op[b + 1], o2[al]:o2[al + 1], o1[io]:o1[io + 1]]).max() > 1e-9 * np.abs(got[l]).max()]
        assert mine == [tuple(t) for t in trip]


def test_gridtransform_plan_matches_einsum():
    """N3 (Eq. 19): the tau <-> i Omega transform descriptors (plan stage 51), run by the numpy interpreter, are the einsum."""
    from tests.helpers import run_stage_numpy
    inp = make_inputs("toy_sc")
    lib = B.Gwsig(device=-1)
    cfg = configure_from_crystal(lib, inp.cr, B.IBZ)
    nq, n2, nin, nout = cfg.nk1, inp.naux ** 2, inp.ntau, 5
    rng = np.random.default_rng(1)
    src = rng.standard_normal(nq * nin * n2) + 1j * rng.standard_normal(nq * nin * n2)
    T = rng.standard_normal((nout, nin)) + 1j * rng.standard_normal((nout, nin))
    pr, sg, _ = lib.plan_get(0, nin, nout, 51)
    dst = np.zeros(nq * nout * n2, complex)
    run_stage_numpy(pr, sg, src, T.ravel(), dst, 0)
    want = np.einsum("oi,qim->qom", T, src.reshape(nq, nin, n2))
    assert np.abs(dst.reshape(nq, nout, n2) - want).max() < 1e-13
