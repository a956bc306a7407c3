"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element on the
same seeded inputs.  Bar (BASELINE.json north_star): max relative Frobenius error <= 1e-11 per (k, tau),
FP64, after folding the result back to the orbital basis."""
import numpy as np
import pytest

from tests.helpers import (fold_to_orbital, get_inputs, oracle_block_maxabs, oracle_exchange, oracle_p0, oracle_packed_V, oracle_sigma, pack_V_p0, rel_err,
                           triples_from_maxabs)

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _B():
    from paper_2405_09494_b200 import build as gw_build
    gw_build.build()
    from paper_2405_09494_b200 import binding
    return binding


def run_gpu(cfg, G, W, V, engine=0, pushes=None, scratch_mib=None, tau_chunk=None, hermitize=0, deterministic=0):
    torch = _torch()
    lib = cfg.lib
    lib.set_option("deterministic", deterministic)
    lib.set_option("engine", engine)
    lib.set_option("hermitize", hermitize)
    if scratch_mib:
        lib.set_option("scratch_mib", scratch_mib)
    lib.set_option("tau_chunk", tau_chunk or 0)
    dG, dW, dV = (torch.from_numpy(x).cuda() for x in (G, W, V))
    dS = torch.full((lib.buffer_sizes()[2],), float("nan"), dtype=torch.complex128, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    if pushes is None:
        lib.sigma_eval(dG, dV, dW, dS, stream)
    else:
        lib.sigma_begin(dG, dW, dS, stream)
        p0 = 0
        voff = [lib.pair_info(p)[3] for p in range(cfg.npairs)] + [V.size]
        while p0 < cfg.npairs:
            n = min(pushes, cfg.npairs - p0)
            lib.sigma_push_pairs(p0, n, dV[voff[p0]:])
            p0 += n
        lib.sigma_end()
    torch.cuda.synchronize()
    return dS.cpu().numpy()


def _check(cfg, inp, sig, ks=None, taus=None, tol=TOL):
    got = fold_to_orbital(cfg, inp, cfg.unpack_sigma(sig))
    ks = range(inp.nk) if ks is None else ks
    taus = np.arange(inp.ntau) if taus is None else np.asarray(taus)
    ref = oracle_sigma(inp, ks, taus)
    worst = 0.0
    for a, k in enumerate(ks):
        for b, t in enumerate(taus):
            worst = max(worst, rel_err(got[k][t], ref[a, b]))
    assert np.isfinite(sig).all()
    assert worst <= tol, worst
    return worst


def _setup(name, mode, **over):
    B = _B()
    from paper_2405_09494_b200.pack import Configured, configure_from_crystal
    lib = B.Gwsig(device=0)
    if name == "cfg1":
        inp = get_inputs("cfg1", **over)
        cfg = Configured(lib, mode, np.eye(3), inp.kmesh.N, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
        Gf, Wf = inp.G_full(), inp.W_full()
        G, W = cfg.pack_GW(lambda k: Gf[k], lambda q: Wf[q])
    else:
        inp = get_inputs(name, **over)
        cfg = configure_from_crystal(lib, inp.cr, mode)
        G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    return B, inp, cfg, G, W, V


@pytest.mark.parametrize("engine", [1, 0, 2, 3])
def test_cfg1_full_bz(engine):
    """BASELINE.json config 1, whole output."""
    B, inp, cfg, G, W, V = _setup("cfg1", 0)
    _check(cfg, inp, run_gpu(cfg, G, W, V, engine=engine))


def test_cfg1_ragged_and_chunked():
    """odd sizes (ragged tile tails in every stage), partial pushes, tau chunks, tiny scratch."""
    B, inp, cfg, G, W, V = _setup("cfg1", 0, mesh=(3, 2, 1), nao=7, naux=19, ntau=5, beta=4.0, nocc=3, seed=4)
    _check(cfg, inp, run_gpu(cfg, G, W, V, pushes=6, tau_chunk=2))
    _check(cfg, inp, run_gpu(cfg, G, W, V, pushes=12, scratch_mib=1))


@pytest.mark.parametrize("name", ["toy_diamond", "toy_wurtzite", "toy_rocksalt", "toy_sc"])
@pytest.mark.parametrize("mode", [1, 2])
def test_toys_ibz_and_block(name, mode):
    B, inp, cfg, G, W, V = _setup(name, mode)
    for engine in (1, 0, 2, 3):
        _check(cfg, inp, run_gpu(cfg, G, W, V, engine=engine))
    _check(cfg, inp, run_gpu(cfg, G, W, V, pushes=cfg.nk1 * 3, tau_chunk=1))


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_cfg2_all_modes(mode):
    """BASELINE.json config 2 (simple cubic, Oh), whole output, all three modes."""
    B, inp, cfg, G, W, V = _setup("cfg2", mode) if mode else _setup_full_from_crystal("cfg2")
    w = _check(cfg, inp, run_gpu(cfg, G, W, V))
    print("cfg2 mode", mode, "worst rel err", w)


def _setup_full_from_crystal(name):
    """FULL_BZ mode on a crystal: inputs given on the whole mesh, no symmetry passed."""
    B = _B()
    from paper_2405_09494_b200.pack import Configured
    inp = get_inputs(name)
    cr = inp.cr
    lib = B.Gwsig(device=0)
    cfg = Configured(lib, 0, cr.a, cr.mesh, cr.nao, cr.naux, cr.ntau, cr.beta, None, None, None)
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    return B, inp, cfg, G, W, V


def _pack_V_device(cfg, inp, batch=64):
    """block-mode packing of V for the large configs with the batched GPU pre-step (presetup_device.DeviceBlocker: Eq. 27
    transform, allowed-block detection, packing; checked against the per-pair numpy pre-step symsetup.block_V2 in
    tests/test_symsetup.py) -- the per-pair Python loop of cfg.pack_V costs minutes at config 5.  Dense V rows still come from
    the numpy generator."""
    torch = _torch()
    from paper_2405_09494_b200.presetup_device import DeviceBlocker
    lib, nk1 = cfg.lib, cfg.nk1
    blk = DeviceBlocker(cfg, torch, torch.device("cuda"))
    k2_of = lambda p: lib.pair_info(p, with_layout=False)[1]
    dense = {}
    for i1, k1 in enumerate(cfg.out_list):
        k2s = [k2_of(q * nk1 + i1) for q in range(cfg.nk)]
        dense[i1] = inp.V2_rows(int(k1), k2s)                    # [nk, naux, nao, nao], row q
    vmax = float(np.abs(dense[0]).max())
    pairs = list(range(cfg.npairs))
    info = [(p // nk1, k2_of(p), int(cfg.out_list[p % nk1])) for p in pairs]
    trip, Ts = [], []
    for b0 in range(0, cfg.npairs, batch):
        pb = pairs[b0:b0 + batch]
        qs, k2s, k1s = ([info[p][j] for p in pb] for j in range(3))
        V = torch.from_numpy(np.stack([dense[p % nk1][p // nk1] for p in pb])).cuda()
        T = blk.transform(V, qs, k2s, k1s)
        trip += blk.triples_from_maxabs(blk.block_maxabs(T, qs, k2s, k1s), qs, k2s, k1s, 1e-9, vmax)
        Ts.append((T.cpu(), qs, k2s, k1s))
    tptr = np.zeros(cfg.npairs + 1, np.int64)
    tptr[1:] = np.cumsum([len(t) for t in trip])
    lib.set_triples(tptr, np.concatenate(trip))
    cfg.triple_ptr, cfg.triples = tptr, trip
    total = lib.buffer_sizes()[3]
    out = torch.zeros(total, dtype=torch.complex128, device="cuda")
    base = 0
    for bi, (T, qs, k2s, k1s) in enumerate(Ts):
        tabs = blk.pack_tables(trip[bi * batch:bi * batch + len(qs)], qs, k2s, k1s)
        off = np.concatenate([[0], np.cumsum(tabs[3])])
        blk.pack(T.cuda(), qs, k2s, k1s, tabs, out, off[:-1] + base)
        base += int(off[-1])
    assert base == total
    return out.cpu().numpy()


def _sampled(name, mode, pick, taus, pushes_q=None):
    """BASELINE configs too large for a full oracle run: Sigma at a few wedge points (every output k1 is an
    independent sum over all q, gwsig_set_output_points), all tau on the GPU, oracle at the sampled tau."""
    B = _B()
    from paper_2405_09494_b200.pack import configure_from_crystal
    inp = get_inputs(name)
    lib = B.Gwsig(device=0)
    cfg = configure_from_crystal(lib, inp.cr, mode, out_points=pick)
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = _pack_V_device(cfg, inp) if (mode == 2 and name in ("cfg4", "cfg5")) else cfg.pack_V(inp.V2_rows)
    sig = run_gpu(cfg, G, W, V, pushes=None if pushes_q is None else pushes_q * cfg.nk1)
    w = _check(cfg, inp, sig, ks=[int(k) for k in cfg.out_list], taus=taus)
    print(name, "mode", mode, "points", list(cfg.out_list), "tau", list(taus), "worst rel err", w)


def _variants_hit(cfg):
    """(row groups, column groups) per MMA warp that the tiles of all three stages produce: the engine instantiates its
    main loop for each of the 16 combinations (zgemm_grouped.cu, ZG_VARIANTS).  Tiling rule of zgemm_grouped.cuh restated."""
    hit = set()
    for stage in (1, 2, 3):
        prob, _, _ = cfg.lib.plan_get(0, cfg.npairs, cfg.ntau, stage)
        for P in prob:
            M, N = int(P["M"]), int(P["N"])
            G = (N + 7) // 8
            tn = (G + 3) // 4
            ngs = {((j + 1) * G) // tn - (j * G) // tn for j in range(tn)}
            for m0 in range(0, M, 128):
                mg = (min(128, M - m0) + 7) // 8
                for wq in range(4):
                    if mg > wq:
                        hit |= {((mg - wq + 3) // 4, ng) for ng in ngs}
    return hit


_VARIANT_CASES = [(7, 5, 2), (10, 13, 3), (10, 21, 2), (12, 29, 3), (5, 27, 13), (3, 9, 37)]


def test_engine_variants_are_all_exercised():
    """every (row groups, column groups) variant of the tensor kernels' main loop, ragged M / N / K tails in all stages:
    small no-symmetry problems whose nao / naux / ntau are chosen so that the union of their tiles covers all 16."""
    hit = set()
    for nao, naux, ntau in _VARIANT_CASES:
        B, inp, cfg, G, W, V = _setup("cfg1", 0, mesh=(2, 1, 1), nao=nao, naux=naux, ntau=ntau, beta=3.0, nocc=max(1, nao // 2), seed=nao)
        cfg.lib.set_option("engine", 2)              # the 4-product kernel's 128-row tiling (its main loop has the 16 variants)
        hit |= _variants_hit(cfg)
        for engine in (0, 2, 3):
            _check(cfg, inp, run_gpu(cfg, G, W, V, engine=engine))
    assert hit == {(mi, ni) for mi in range(1, 5) for ni in range(1, 5)}, sorted(hit)


def test_cfg3_shaped_small_mesh_full_oracle():
    """BASELINE configs[2]'s real shell lists (nao 26, naux 116: cfg3's irrep block sizes, N not a multiple of 8, K not a
    multiple of 4, stage-3 segment lists cut along P') on a 2x2x2 mesh with 5 tau points, where the oracle can check EVERY
    (k, tau) of the zone: block mode with both tensor kernels, IBZ mode, several pushes and tau chunks."""
    B, inp, cfg, G, W, V = _setup("cfg3", 2, mesh=(2, 2, 2), ntau=5)
    for engine in (0, 2, 3):
        _check(cfg, inp, run_gpu(cfg, G, W, V, engine=engine))
    _check(cfg, inp, run_gpu(cfg, G, W, V, pushes=cfg.nk1 * 3, tau_chunk=2))
    B, inp, cfg, G, W, V = _setup("cfg3", 1, mesh=(2, 2, 2), ntau=5)
    _check(cfg, inp, run_gpu(cfg, G, W, V))


@pytest.mark.parametrize("name", ["toy_diamond4", "toy_wurtzite"])
def test_general_gauge_eq28(name):
    """explicit U in a scrambled gauge (independent random unitary inside every irrep block at EVERY mesh point): the
    library forms O_block = U^{k'}^dagger O U^{k_I} and unfolds the packed G and W blocks with it (Eq. 28)."""
    B = _B()
    from paper_2405_09494_b200.pack import configure_from_crystal
    inp = get_inputs(name)
    lib = B.Gwsig(device=0)
    cfg = configure_from_crystal(lib, inp.cr, 2, scramble_gauge=5)
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    V = cfg.pack_V(inp.V2_rows)
    _check(cfg, inp, run_gpu(cfg, G, W, V))
    _check(cfg, inp, run_gpu(cfg, G, W, V, pushes=cfg.nk1 * 3, tau_chunk=1, engine=2))


@pytest.mark.parametrize("name,mode", [("toy_diamond4", 2), ("toy_wurtzite", 1), ("cfg2", 2)])
def test_exchange_eq21c(name, mode):
    """N2: K^k = -(1/Nk) sum_{k'} V^{kk'} gamma^{k'} V^{k'k} (Eq. 21c) through gwsig_exchange_eval (stage 1 feeding
    stage 3, no W) against oracle/exchange_oracle.py, gamma^k = G^k(0^-) = -G^k(beta), one slice (ntau = 1)."""
    B = _B()
    torch = _torch()
    from paper_2405_09494_b200.pack import configure_from_crystal
    import copy
    inp = get_inputs(name)
    cr1 = copy.copy(inp.cr)
    cr1.ntau = 1                                                   # the context sees one "tau" slice: the density matrix
    lib = B.Gwsig(device=0)
    cfg = configure_from_crystal(lib, cr1, mode)
    gam = lambda k: -inp.G_k(int(k))[-1]
    G, _ = cfg.pack_GW(lambda k: gam(k)[None], lambda q: np.zeros((1, inp.naux, inp.naux), complex))
    V = cfg.pack_V(inp.V2_rows)
    dG, dV = torch.from_numpy(G).cuda(), torch.from_numpy(V).cuda()
    dK = torch.full((lib.buffer_sizes()[2],), float("nan"), dtype=torch.complex128, device="cuda")
    lib.exchange_eval(dG, dV, dK, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    got = fold_to_orbital(cfg, inp, cfg.unpack_sigma(dK.cpu().numpy()))
    ks = list(range(inp.nk)) if inp.nk <= 64 else list(range(0, inp.nk, 5))
    ref = oracle_exchange(inp, gam, ks)
    worst = max(rel_err(got[k][0], ref[a]) for a, k in enumerate(ks))
    assert worst <= TOL, worst


def test_deterministic_accumulation_is_bit_reproducible():
    """option "deterministic": the split-K parts of stage 3 go through private partial tiles and one ordered reduction instead
    of FP64 atomics in scheduler order: two runs give bit-identical Sigma, and the result still matches the oracle."""
    B, inp, cfg, G, W, V = _setup("cfg3", 2, mesh=(2, 2, 2), ntau=5)
    a = run_gpu(cfg, G, W, V, deterministic=1, tau_chunk=2)
    b = run_gpu(cfg, G, W, V, deterministic=1, tau_chunk=2)
    assert np.array_equal(a.view(np.float64), b.view(np.float64))
    _check(cfg, inp, a)
    c = run_gpu(cfg, G, W, V, deterministic=0, tau_chunk=2)
    assert np.abs(a - c).max() <= 1e-12 * np.abs(a).max()


@pytest.mark.parametrize("name,mode", [("cfg1", 0), ("toy_diamond4", 1), ("toy_wurtzite", 1), ("cfg2", 1)])
def test_p0_eq20(name, mode):
    """N1: bare bubble P0^q(tau) (Eq. 20, Algorithm 3) through gwsig_p0_eval / p0_push_pairs against
    oracle/p0_oracle.py: every output q (the wedge in IBZ mode), every tau; one call, and several pushes with tau chunks."""
    B = _B()
    torch = _torch()
    from paper_2405_09494_b200.pack import Configured, configure_from_crystal
    lib = B.Gwsig(device=0)
    if name == "cfg1":
        inp = get_inputs("cfg1")
        cfg = Configured(lib, mode, np.eye(3), inp.kmesh.N, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
        Gf = inp.G_full()
        G, _ = cfg.pack_GW(lambda k: Gf[k], lambda q: np.zeros((inp.ntau, inp.naux, inp.naux), complex))
    else:
        inp = get_inputs(name)
        cfg = configure_from_crystal(lib, inp.cr, mode)
        G, _ = cfg.pack_GW(inp.G_k, lambda q: np.zeros((inp.ntau, inp.naux, inp.naux), complex))
    V = pack_V_p0(cfg, inp)
    dG, dV = torch.from_numpy(G).cuda(), torch.from_numpy(V).cuda()
    nq = len(cfg.out_list)
    shape = (nq, inp.ntau, inp.naux, inp.naux)
    ref = oracle_p0(inp, cfg.out_list)
    stream = torch.cuda.current_stream().cuda_stream
    for variant in ("eval", "pushes"):
        dP = torch.full((int(np.prod(shape)),), float("nan"), dtype=torch.complex128, device="cuda")
        if variant == "eval":
            lib.set_option("tau_chunk", 0)
            lib.p0_eval(dG, dV, dP, stream)
        else:
            lib.set_option("tau_chunk", max(1, inp.ntau // 3))
            lib.p0_begin(dG, dP, stream)
            xs = inp.naux * inp.nao ** 2
            npairs, step = cfg.nk * nq, max(1, (cfg.nk * nq) // 3 + 1)
            for p0 in range(0, npairs, step):
                lib.p0_push_pairs(p0, min(step, npairs - p0), dV[p0 * xs:])
            lib.p0_end()
        torch.cuda.synchronize()
        got = dP.cpu().numpy().reshape(shape)
        worst = max(rel_err(got[i, t], ref[i, t]) for i in range(nq) for t in range(inp.ntau))
        assert worst <= TOL, (variant, worst)


@pytest.mark.parametrize("name", ["toy_diamond4", "toy_wurtzite", "cfg2"])
def test_block_transform_v_eq27(name):
    """N4: gwsig_block_transform_v (Eq. 27: dense orbital-basis V2 -> packed block-basis V2 on the device) against
    oracle/block_oracle.py, and the Sigma evaluated from that device-packed V against the Sigma oracle."""
    B = _B()
    torch = _torch()
    from paper_2405_09494_b200.pack import configure_from_crystal
    inp = get_inputs(name)
    lib = B.Gwsig(device=0)
    cfg = configure_from_crystal(lib, inp.cr, 2, pass_U=True)
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    Vnp = cfg.pack_V(inp.V2_rows)                           # numpy pre-step: finds the triples (set_triples); its V is NOT used below
    dense = np.concatenate([inp.V2_rows(lib.pair_info(p)[0], [lib.pair_info(p)[1]])[0].ravel() for p in range(cfg.npairs)])
    dD = torch.from_numpy(dense).cuda()
    dP = torch.full((Vnp.size,), float("nan"), dtype=torch.complex128, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    half = cfg.npairs // 2
    lib.block_transform_v(0, half, dD, dP, stream)                                         # two calls: offsets of a later range
    xs = inp.naux * inp.nao ** 2
    lib.block_transform_v(half, cfg.npairs - half, dD[half * xs:], dP[lib.pair_info(half)[3]:], stream)
    torch.cuda.synchronize()
    got = dP.cpu().numpy()
    sample = list(range(0, cfg.npairs, max(1, cfg.npairs // 25)))
    voff = [lib.pair_info(p)[3] for p in range(cfg.npairs)] + [Vnp.size]
    for p in sample:
        ref = oracle_packed_V(cfg, inp, [p])
        assert np.abs(got[voff[p]:voff[p + 1]] - ref).max() <= 1e-13 * np.abs(dense).max()
    _check(cfg, inp, run_gpu(cfg, G, W, got), ks=None if inp.nk <= 64 else list(range(0, inp.nk, 7)))


@pytest.mark.parametrize("name", ["toy_diamond4", "toy_wurtzite", "cfg2"])
def test_block_maxabs_device_prestep(name):
    """N4, detection: gwsig_block_maxabs (Eq. 27 for every block + block maxima on the device, no triples set yet) against the
    oracle's dense transform; its thresholded triples are the ones the CPU pre-step finds; the whole device pre-step
    (detection -> set_triples -> gwsig_block_transform_v) then feeds a Sigma evaluation that matches the Sigma oracle."""
    B = _B()
    torch = _torch()
    from paper_2405_09494_b200.pack import configure_from_crystal
    inp = get_inputs(name)
    lib = B.Gwsig(device=0)
    cfg = configure_from_crystal(lib, inp.cr, 2, pass_U=True)
    mb_aux = max(len(o) - 1 for o in cfg.aux.off) + 1                # one spare index each: unused candidates stay zero
    mb_ao = max(len(o) - 1 for o in cfg.ao.off)
    info = [lib.pair_info(p, with_layout=False) for p in range(cfg.npairs)]
    dense = np.concatenate([inp.V2_rows(i[0], [i[1]])[0].ravel() for i in info])
    dD = torch.from_numpy(dense).cuda()
    dM = torch.full((cfg.npairs * mb_aux * mb_ao * mb_ao,), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    xs = inp.naux * inp.nao ** 2
    third = cfg.npairs // 3
    lib.block_maxabs(0, third, dD, mb_aux, mb_ao, dM, stream)                                  # two calls: a later pair range
    lib.block_maxabs(third, cfg.npairs - third, dD[third * xs:], mb_aux, mb_ao, dM[third * mb_aux * mb_ao * mb_ao:], stream)
    torch.cuda.synchronize()
    got = dM.cpu().numpy().reshape(cfg.npairs, mb_aux, mb_ao, mb_ao)
    vmax = np.abs(dense).max()
    sample = list(range(0, cfg.npairs, max(1, cfg.npairs // 40)))
    ref = oracle_block_maxabs(cfg, inp, sample, mb_aux, mb_ao)
    assert np.abs(got[sample] - ref).max() <= 1e-12 * vmax
    assert got[:, mb_aux - 1].max() == 0.0                                                     # the spare index was never touched
    # forbidden blocks are zero to rounding, allowed ones are not: the threshold does not matter
    assert not ((got > 1e-12 * vmax) & (got < 1e-6 * vmax)).any()
    trip = triples_from_maxabs(got, 1e-9, vmax)
    Vnp = cfg.pack_V(inp.V2_rows)                                    # CPU pre-step (symsetup.block_V2): its triples are the reference
    assert all(np.array_equal(trip[p], cfg.triples[p]) for p in range(cfg.npairs))
    # device pre-step end to end: the triples found on the device, then the packed transform on the device, then Sigma
    tptr = np.zeros(cfg.npairs + 1, np.int64)
    tptr[1:] = np.cumsum([len(t) for t in trip])
    lib.set_triples(tptr, np.concatenate(trip))
    dP = torch.full((Vnp.size,), float("nan"), dtype=torch.complex128, device="cuda")
    lib.block_transform_v(0, cfg.npairs, dD, dP, stream)
    torch.cuda.synchronize()
    G, W = cfg.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    _check(cfg, inp, run_gpu(cfg, G, W, dP.cpu().numpy()), ks=None if inp.nk <= 64 else list(range(0, inp.nk, 7)))


@pytest.mark.parametrize("name,mode,nw", [("toy_wurtzite", 1, 3), ("cfg2", 1, 9), ("cfg1", 0, 7)])
def test_dyson_p_eq19(name, mode, nw):
    """N3: P = [1 - P0]^{-1} P0 per (q, Omega) with caller-supplied tau <-> i Omega transform matrices (Eq. 19)
    through gwsig_dyson_p against oracle/dyson_oracle.py; the input P0 is the oracle's own bare bubble, scaled to |P0| ~ 1 so that
    the solve is far from the perturbative regime; a singular 1 - P0 is reported."""
    B = _B()
    torch = _torch()
    from oracle.dyson_oracle import dyson_p_ref
    from paper_2405_09494_b200.pack import Configured, configure_from_crystal
    lib = B.Gwsig(device=0)
    if name == "cfg1":
        inp = get_inputs("cfg1")
        cfg = Configured(lib, mode, np.eye(3), inp.kmesh.N, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
    else:
        inp = get_inputs(name)
        cfg = configure_from_crystal(lib, inp.cr, mode)
    qs = list(cfg.out_list)[:6]
    lib.set_output_points(qs) if len(qs) < len(cfg.out_list) else None
    P0 = oracle_p0(inp, qs)
    P0 = P0 / np.abs(P0).max() * 0.9
    rng = np.random.default_rng(3)
    tau = np.arange(inp.ntau) * inp.beta / (inp.ntau - 1)
    om = 2 * np.pi * np.arange(nw) / inp.beta
    Tf = np.exp(1j * np.outer(om, tau)) * (inp.beta / inp.ntau) + 0.01 * rng.standard_normal((nw, inp.ntau))     # a quadrature-like matrix
    Tb = np.exp(-1j * np.outer(tau, om)) / inp.beta
    ref = dyson_p_ref(P0, Tf, Tb)
    dP0, dTf, dTb = (torch.from_numpy(np.ascontiguousarray(x, np.complex128)).cuda() for x in (P0, Tf, Tb))
    dP = torch.full((P0.size,), float("nan"), dtype=torch.complex128, device="cuda")
    lib.dyson_p(dP0, dTf, dTb, nw, dP, torch.cuda.current_stream().cuda_stream)
    got = dP.cpu().numpy().reshape(P0.shape)
    worst = max(rel_err(got[i, t], ref[i, t]) for i in range(len(qs)) for t in range(inp.ntau))
    cond = max(np.linalg.cond(np.eye(inp.naux) - np.einsum("wt,tab->wab", Tf, P0[i])).max() for i in range(len(qs)))
    assert worst <= max(TOL, 1e-15 * cond * 100), (worst, cond)
    # singular case: P0(i Omega) = 1 exactly for identity transforms
    if name == "cfg1":
        one = np.tile(np.eye(inp.naux, dtype=complex), (len(qs), inp.ntau, 1, 1))
        eye = torch.eye(inp.ntau, dtype=torch.complex128, device="cuda")
        with pytest.raises(B.GwsigError):
            lib.dyson_p(torch.from_numpy(one).cuda(), eye, eye, inp.ntau, dP, 0)


def test_output_point_subset_matches_full_run():
    B, inp, cfg, G, W, V = _setup("toy_diamond", 2)
    full = cfg.unpack_sigma(run_gpu(cfg, G, W, V))
    from paper_2405_09494_b200.pack import configure_from_crystal
    lib2 = B.Gwsig(device=0)
    cfg2 = configure_from_crystal(lib2, inp.cr, 2, out_points=lambda wedge: [wedge[2], wedge[0]])
    G2, W2 = cfg2.pack_GW(inp.G_k, lambda q: inp.W_full([q])[0])
    sub = cfg2.unpack_sigma(run_gpu(cfg2, G2, W2, cfg2.pack_V(inp.V2_rows)))
    for a, i in enumerate((2, 0)):
        assert np.abs(sub[a] - full[i]).max() <= 1e-13 * np.abs(full[i]).max()


def test_cfg3_sampled():
    """BASELINE configs[2] at full size: block mode at three wedge points of different little-group order (Gamma, a
    line point, a generic point), IBZ mode (unfold kernels, W ring, several pushes) at one of them."""
    _sampled("cfg3", 2, lambda wedge: [wedge[0], wedge[5], wedge[-1]], [0, 51, 103])
    _sampled("cfg3", 1, lambda wedge: [wedge[5]], [51], pushes_q=54)


def test_cfg4_sampled():
    """BASELINE configs[3] (wurtzite, 12 operations, nonsymmorphic), P9 sample: 2 wedge points x 2 tau in block mode,
    one of them again in IBZ mode with several pushes (the oracle run is shared)."""
    _sampled("cfg4", 2, lambda wedge: [wedge[0], wedge[9]], [0, 127])
    _sampled("cfg4", 1, lambda wedge: [wedge[9]], [127], pushes_q=24)


def test_cfg5_sampled():
    """BASELINE configs[4] (rock salt, 8x8x8): block mode at Gamma (full O_h little group: the most ragged block structure of
    the config), then IBZ mode (Nk * ntau = 69632 unfold targets: beyond a 65535 grid.y) at the same point in several pushes
    (the oracle run is shared).  One wedge point keeps the whole GPU suite near ten minutes; cfg4 samples a generic point."""
    _sampled("cfg5", 2, lambda wedge: [wedge[0]], [0, 135])
    _sampled("cfg5", 1, lambda wedge: [wedge[0]], [135], pushes_q=64)


@pytest.mark.parametrize("name", ["cfg1", "toy_diamond4", "toy_wurtzite", "cfg2"])
def test_hartree_eq21b(name):
    """J^k (Eq. 21b) through gwsig_hartree_eval against oracle/hartree_oracle.py at every mesh point; twice on the
    same inputs: the summation order is fixed, the results are bit-identical."""
    B = _B()
    torch = _torch()
    from oracle.hartree_oracle import hartree_ref
    from paper_2405_09494_b200.pack import Configured
    inp = get_inputs(name)
    lib = B.Gwsig(device=0)
    mesh = inp.kmesh.N
    Configured(lib, 0, np.eye(3), mesh, inp.nao, inp.naux, inp.ntau, inp.beta, None, None, None)
    nk = inp.nk
    G = np.stack([inp.G_k(k) for k in range(nk)]) if hasattr(inp, "G_k") else inp.G_full()
    gamma = np.ascontiguousarray(-G[:, -1])                          # gamma^k = G^k(0^-) = -G^k(beta)
    Vd = np.ascontiguousarray(inp.V_pairs(range(nk), range(nk)))     # V^{kk}_{Q,ij}
    ref = hartree_ref(nk, lambda k: gamma[k], lambda k: Vd[k], range(nk))
    dG, dV = torch.from_numpy(gamma).cuda(), torch.from_numpy(Vd).cuda()
    outs = []
    for _ in range(2):
        dJ = torch.full((nk * inp.nao * inp.nao,), float("nan"), dtype=torch.complex128, device="cuda")
        lib.hartree_eval(dG, dV, dJ, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        outs.append(dJ.cpu().numpy().reshape(nk, inp.nao, inp.nao))
    worst = max(rel_err(outs[0][k], ref[k]) for k in range(nk))
    assert worst <= TOL, worst
    assert np.array_equal(outs[0], outs[1])


def test_hermitize_option_and_observed_hermiticity():
    B, inp, cfg, G, W, V = _setup("toy_diamond", 1)
    s0 = run_gpu(cfg, G, W, V)
    s1 = run_gpu(cfg, G, W, V, hermitize=1)
    S0 = np.stack(cfg.unpack_sigma(s0))
    S1 = np.stack(cfg.unpack_sigma(s1))
    scale = np.abs(S0).max()
    assert np.abs(S0 - S0.conj().transpose(0, 1, 3, 2)).max() < 1e-12 * scale      # observed, not imposed
    assert np.abs(S1 - S1.conj().transpose(0, 1, 3, 2)).max() == 0                  # imposed
    assert np.abs(S1 - S0).max() < 1e-12 * scale


def test_push_order_is_enforced():
    B, inp, cfg, G, W, V = _setup("toy_sc", 1)
    torch = _torch()
    dG, dW, dV = (torch.from_numpy(x).cuda() for x in (G, W, V))
    dS = torch.zeros(cfg.lib.buffer_sizes()[2], dtype=torch.complex128, device="cuda")
    cfg.lib.sigma_begin(dG, dW, dS, 0)
    with pytest.raises(B.GwsigError) as e:
        cfg.lib.sigma_push_pairs(cfg.nk1, cfg.nk1, dV)
    assert e.value.code == -5
    with pytest.raises(B.GwsigError) as e:
        cfg.lib.sigma_end()
    assert e.value.code == -5


def test_fp64_probe_runs():
    B = _B()
    lib = B.Gwsig(device=0)
    t_dmma, _ = lib.probe_fp64(0, 8, 2, 4000)
    t_dfma, _ = lib.probe_fp64(1, 8, 2, 4000)
    print("FP64 probe TFLOP/s: DMMA", t_dmma, "DFMA", t_dfma)
    assert t_dmma > 1.0 and t_dfma > 1.0
