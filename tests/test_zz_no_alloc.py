"""gwsig_dyson_solve_noalloc (include/gwsig.h): the Eq. 19a solve with the library's fixed device scratch, for callers that
may not allocate, against the existing path (gwsig_dyson_p with identity grid transforms, which runs the same solve out of
context-owned buffers).  Collected last on purpose (file name): the suite runs with pytest -x.
Runs alone in a fresh process and after the other GPU tests (it shares no state with them but the library)."""
import numpy as np
import pytest

TOL = 1e-11          # the bar of tests/test_gpu_parity.py (relative Frobenius error per matrix)


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def _B():
    from paper_2405_09494_b200 import build as gw_build
    gw_build.build()
    from paper_2405_09494_b200 import binding
    return binding


def _existing_path(B, torch, P0):
    """P = [1 - P0]^{-1} P0 per (q, tau) through gwsig_dyson_p: identity tau <-> Omega matrices (nw = ntau)."""
    from paper_2405_09494_b200.pack import Configured
    nq, ntau, naux, _ = P0.shape
    lib = B.Gwsig(device=0)
    Configured(lib, 0, np.eye(3), (nq, 1, 1), 3, naux, ntau, 2.0, None, None, None)
    eye = torch.eye(ntau, dtype=torch.complex128, device="cuda")
    dP0 = torch.from_numpy(P0).cuda()
    dP = torch.full((P0.size,), float("nan"), dtype=torch.complex128, device="cuda")
    lib.dyson_p(dP0, eye, eye, ntau, dP, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return dP.cpu().numpy().reshape(P0.shape)


def _inputs(seed, nq, ntau, naux):
    rng = np.random.default_rng(seed)
    P0 = rng.standard_normal((nq, ntau, naux, naux)) + 1j * rng.standard_normal((nq, ntau, naux, naux))
    return np.ascontiguousarray(P0 * (0.9 / np.sqrt(2.0 * naux)), np.complex128)     # spectral radius ~ 0.9: far from perturbative


def _worst(got, ref):
    return max(np.linalg.norm(got[i, t] - ref[i, t]) / np.linalg.norm(ref[i, t]) for i in range(ref.shape[0]) for t in range(ref.shape[1]))


def test_noalloc_rejects_bad_sizes_before_touching_the_device():
    """no GPU needed: the size checks come first and say what the limit is."""
    B = _B()
    for nmat, n in ((1, B.NOALLOC_NMAX + 1), (1, 0), (-1, 4)):
        with pytest.raises(B.GwsigError) as e:
            B.dyson_solve_noalloc(None, None, nmat, n)
        assert e.value.code == -1 and "gwsig_dyson_solve_noalloc" in str(e.value)
    B.dyson_solve_noalloc(None, None, 0, 4)                            # nothing to do


@pytest.mark.gpu
def test_noalloc_matches_dyson_p_on_two_calls_in_a_row():
    B, torch = _B(), _torch()
    cases = [_inputs(11, 2, 5, 37), _inputs(12, 3, 4, 116)]          # second call: other n, more matrices, stale scratch of the first
    refs = [_existing_path(B, torch, P0) for P0 in cases]
    stream = torch.cuda.current_stream().cuda_stream
    outs, infos = [], []
    for P0 in cases:                                                  # two calls in a row on one stream, nothing in between
        nq, ntau, naux, _ = P0.shape
        dA = torch.from_numpy(P0).cuda()
        dX = torch.full((P0.size,), float("nan"), dtype=torch.complex128, device="cuda")
        info = torch.full((1,), 7, dtype=torch.int32, device="cuda")
        B.dyson_solve_noalloc(dA, dX, nq * ntau, naux, info, stream)
        outs.append((dA, dX)); infos.append(info)
    torch.cuda.synchronize()
    for P0, ref, (dA, dX), info in zip(cases, refs, outs, infos):
        got = dX.cpu().numpy().reshape(P0.shape)
        assert int(info.item()) == 0
        assert np.array_equal(dA.cpu().numpy(), P0)                   # input untouched
        cond = max(np.linalg.cond(np.eye(P0.shape[2]) - P0[i, t]) for i in range(P0.shape[0]) for t in range(P0.shape[1]))
        assert _worst(got, ref) <= max(TOL, 1e-13 * cond), (_worst(got, ref), cond)
        # and against the definition, so that a shared mistake cannot hide
        sol = np.linalg.solve(np.eye(P0.shape[2])[None, None] - P0, P0)
        assert _worst(got, sol) <= max(TOL, 1e-13 * cond)
    # the first problem again, in place, after the second call's contents: bit-identical to its first result
    P0 = cases[0]
    dA = torch.from_numpy(P0).cuda()
    B.dyson_solve_noalloc(dA, dA, P0.shape[0] * P0.shape[1], P0.shape[2], None, stream)
    torch.cuda.synchronize()
    assert np.array_equal(dA.cpu().numpy().reshape(P0.shape), outs[0][1].cpu().numpy().reshape(P0.shape))


@pytest.mark.gpu
def test_noalloc_allocates_nothing_and_rejects_oversize():
    B, torch = _B(), _torch()
    n = 24
    P0 = _inputs(5, 1, 3, n)
    dA = torch.from_numpy(P0).cuda()
    dX = torch.empty_like(dA)
    info = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.dyson_solve_noalloc(dA, dX, 3, n, info, 0)                      # first call on the device resolved the scratch address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        B.dyson_solve_noalloc(dA, dX, 3, n, info, 0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                      # device memory in use did not grow
    with pytest.raises(B.GwsigError) as e:
        B.dyson_solve_noalloc(dA, dX, 1, B.NOALLOC_NMAX + 1, info, 0)
    assert e.value.code == -1 and "GWSIG_NOALLOC_NMAX" in str(e.value)
    # largest size: one CTA's augmented matrix fills 2 MiB of the 16 MiB array
    big = _inputs(6, 1, 9, B.NOALLOC_NMAX)
    dB = torch.from_numpy(big).cuda()
    B.dyson_solve_noalloc(dB, dB, 9, B.NOALLOC_NMAX, info, 0)
    torch.cuda.synchronize()
    sol = np.linalg.solve(np.eye(B.NOALLOC_NMAX)[None, None] - big, big)
    assert int(info.item()) == 0 and _worst(dB.cpu().numpy().reshape(big.shape), sol) <= 1e-10
    # singular 1 - A is reported through d_info, without a synchronising call inside the library
    one = torch.eye(n, dtype=torch.complex128, device="cuda").reshape(1, n, n).contiguous()
    B.dyson_solve_noalloc(one, torch.empty_like(one), 1, n, info, 0)
    torch.cuda.synchronize()
    assert int(info.item()) == 1
