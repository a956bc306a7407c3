"""Pins for the CPU oracle: every test checks
``oracle.sigma_oracle`` against something other than itself -- explicit loops,
closed forms, or invariants that a dropped term / wrong sign / swapped index /
transposed operand would break."""
import numpy as np
import pytest

from gwsig_synth import make_inputs
from gwsig_synth.group import rep_at_k
from oracle.sigma_oracle import flops_per_output, sigma_brute, sigma_ref
from paper_2405_09494_b200.symsetup import SymSetup


def _c1(nao=3, naux=4, ntau=2, seed=5):
    return make_inputs("cfg1", mesh=(2, 2, 2), nao=nao, naux=naux, ntau=ntau, beta=3.0, nocc=1, seed=seed)


def _ref(inp, ks, G=None, W=None, V_pair=None):
    G = inp.G_full() if G is None else G
    W = inp.W_full() if W is None else W
    V_pair = inp.V_pair if V_pair is None else V_pair
    km = inp.kmesh
    return sigma_ref(inp.nk, km.sub, lambda k: G[k], lambda q: W[q], V_pair, ks)


# ---- P1: explicit seven-loop brute force ---------------------------------------

def test_ref_equals_brute_force():
    inp = _c1()
    G, W = inp.G_full(), inp.W_full()
    ks = [0, 3, 6]
    b = sigma_brute(inp.nk, inp.kmesh.sub, G, W, inp.V_pair, ks)
    r = _ref(inp, ks, G, W)
    assert np.abs(b - r).max() < 1e-14 * max(1.0, np.abs(b).max())
    assert np.abs(b).max() > 1e-3


def test_ref_equals_brute_force_with_independent_V_partners():
    """the oracle must not assume V^{k2,k1} = conj V^{k1,k2}: feed unrelated tensors."""
    inp = _c1(seed=9)
    rng = np.random.default_rng(3)
    Vfree = rng.standard_normal((8, 8, 4, 3, 3)) + 1j * rng.standard_normal((8, 8, 4, 3, 3))
    G = rng.standard_normal((8, 2, 3, 3)) + 1j * rng.standard_normal((8, 2, 3, 3))      # not Hermitian either
    W = rng.standard_normal((8, 2, 4, 4)) + 1j * rng.standard_normal((8, 2, 4, 4))
    vp = lambda a, b: Vfree[a, b]
    b = sigma_brute(8, inp.kmesh.sub, G, W, vp, [1, 4])
    r = sigma_ref(8, inp.kmesh.sub, lambda k: G[k], lambda q: W[q], vp, [1, 4])
    assert np.abs(b - r).max() < 1e-12 * np.abs(b).max()


# ---- P2: scalar closed forms ---------------------------------------------------------

def test_scalar_closed_form():
    """nao = naux = 1, k-independent v, g(tau), w(tau)  =>  Sigma = -|v|^2 g(tau) w(tau)."""
    from gwsig_synth.group import KMesh
    km = KMesh((2, 2, 2))
    v = 0.7 - 0.4j
    g = np.array([-0.9, -0.5, -0.2, -0.1])
    w = np.array([0.3, 0.2, 0.25, 0.4])
    G = np.broadcast_to(g[None, :, None, None], (8, 4, 1, 1))
    W = np.broadcast_to(w[None, :, None, None], (8, 4, 1, 1))
    vp = lambda k1, k2: np.full((1, 1, 1), v if k1 <= k2 else np.conj(v)) if k1 != k2 else np.full((1, 1, 1), abs(v))
    # use |v| on the diagonal pairs (they must be Hermitian in ij) and v / conj(v) off-diagonal
    out = sigma_ref(8, km.sub, lambda k: G[k], lambda q: W[q], vp, range(8))
    assert np.allclose(out[:, :, 0, 0], -(abs(v) ** 2) * g * w, atol=1e-15)


def test_exchange_like_closed_form():
    """W~ = delta_{QQ'} w, G = g 1  =>  Sigma_ij = -(g w / Nk) sum_{q,Q,a} V^{k,k-q}_{Q,ia} V^{k-q,k}_{Q,aj}
    (the shape of the exchange term Eq. 21c)."""
    inp = _c1(nao=3, naux=4, ntau=2)
    g, w = np.array([-0.6, -0.3]), np.array([0.5, 0.8])
    G = np.einsum("t,ab->tab", g, np.eye(3))[None].repeat(8, 0)
    W = np.einsum("t,ab->tab", w, np.eye(4))[None].repeat(8, 0)
    out = _ref(inp, range(8), G, W)
    for k in range(8):
        acc = np.zeros((3, 3), complex)
        for q in range(8):
            kq = inp.kmesh.sub(k, q)
            acc += np.einsum("Qia,Qaj->ij", inp.V_pair(k, kq), inp.V_pair(kq, k))
        for t in range(2):
            assert np.allclose(out[k, t], -(g[t] * w[t] / 8) * acc, atol=1e-13)


def test_only_the_right_q_enters():
    """G non-zero at one momentum p only, W~ non-zero at one q0 only: Sigma(k) is non-zero
    only at k = p + q0 and equals the single term (pins the k-q bookkeeping and its sign)."""
    inp = _c1()
    G0, W0 = inp.G_full(), inp.W_full()
    p, q0 = 5, 3
    G = np.zeros_like(G0); G[p] = G0[p]
    W = np.zeros_like(W0); W[q0] = W0[q0]
    out = _ref(inp, range(8), G, W)
    km = inp.kmesh
    ktarget = int(km.index(km.n[p] + km.n[q0]))
    for k in range(8):
        if k != ktarget:
            assert np.abs(out[k]).max() == 0
    single = -np.einsum("Qia,tab,tQP,Pbj->tij", inp.V_pair(ktarget, p), G0[p], W0[q0], inp.V_pair(p, ktarget),
                        optimize=True) / 8
    assert np.allclose(out[ktarget], single, atol=1e-14)


# ---- P3: bilinearity and gauge covariance ---------------------------------------------

def test_bilinear_in_G_and_W():
    inp = _c1()
    i2 = _c1(seed=77)
    G1, G2, W1, W2 = inp.G_full(), i2.G_full(), inp.W_full(), i2.W_full()
    a, b = 0.3 - 1.1j, 2.0 + 0.5j
    ks = [2, 7]
    lhs = _ref(inp, ks, a * G1 + b * G2, W1)
    assert np.allclose(lhs, a * _ref(inp, ks, G1, W1) + b * _ref(inp, ks, G2, W1), atol=1e-13)
    lhs = _ref(inp, ks, G1, a * W1 + b * W2)
    assert np.allclose(lhs, a * _ref(inp, ks, G1, W1) + b * _ref(inp, ks, G1, W2), atol=1e-13)


def _rand_unitary(rng, n):
    q, _ = np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))
    return q


def test_gauge_covariance_orbital_and_aux():
    """G -> T G T^dag, V^{k1k2} -> T^{k1} V T^{k2 dag}  =>  Sigma -> T Sigma T^dag; and in the aux space
    V^{k1k2}_Q -> sum_P S^{q}_{QP} V_P with q = k2 - k1, W~^q -> S^q W~ S^{q dag}, with
    S^{-q} = conj(S^q) (the relation J^{-q} = J^{q*} of PAPER.md:173 imposes on any aux basis change)
    =>  Sigma unchanged.  This is exactly what block-basis parity relies on (Eq. 26-27)."""
    inp = make_inputs("cfg1", mesh=(3, 2, 1), nao=3, naux=4, ntau=2, beta=3.0, nocc=1, seed=5)
    km, nk = inp.kmesh, inp.nk
    rng = np.random.default_rng(0)
    T = [_rand_unitary(rng, inp.nao) for _ in range(nk)]
    G, W = inp.G_full(), inp.W_full()
    base = _ref(inp, range(nk), G, W)
    Gt = np.stack([T[k] @ G[k] @ T[k].conj().T for k in range(nk)])
    vt = lambda k1, k2: np.einsum("Ii,Qij,Jj->QIJ", T[k1], inp.V_pair(k1, k2), T[k2].conj())
    out = _ref(inp, range(nk), Gt, W, vt)
    for k in range(nk):
        assert np.allclose(out[k], T[k] @ base[k] @ T[k].conj().T, atol=1e-13)

    S = [None] * nk
    for q in range(nk):
        mq = int(km.index(-km.n[q]))
        if S[q] is not None:
            continue
        if mq == q:
            S[q] = np.linalg.qr(rng.standard_normal((inp.naux, inp.naux)))[0].astype(complex)
        else:
            S[q] = _rand_unitary(rng, inp.naux)
            S[mq] = S[q].conj()
    assert any(int(km.index(-km.n[q])) != q for q in range(nk))

    def vs(k1, k2):
        q = int(km.index(km.n[k2] - km.n[k1]))
        return np.einsum("QP,Pij->Qij", S[q], inp.V_pair(k1, k2))

    Wt = np.stack([S[q] @ W[q] @ S[q].conj().T for q in range(nk)])
    out = _ref(inp, range(nk), G, Wt, vs)
    assert np.allclose(out, base, atol=1e-13)
    # and a wrong pairing (W~ transformed with the conjugate matrix) must NOT be invariant
    Wbad = np.stack([S[q].conj() @ W[q] @ S[q].T for q in range(nk)])
    assert np.abs(_ref(inp, range(nk), G, Wbad, vs) - base).max() > 1e-3 * np.abs(base).max()


# ---- P7: symmetry invariants on oracle output ------------------------------------------

@pytest.mark.parametrize("name", ["toy_diamond", "toy_wurtzite", "toy_sc"])
def test_sigma_covariance_hermiticity_and_block_zeros(name):
    inp = make_inputs(name)
    cr, sg, km = inp.cr, inp.cr.sg, inp.cr.kmesh
    S = _ref(inp, range(inp.nk))
    scale = np.abs(S).max()
    assert scale > 1e-4
    # Hermiticity of Sigma_ij(k, tau)
    assert np.abs(S - S.conj().transpose(0, 1, 3, 2)).max() < 1e-13 * scale
    # Sigma(g k) = O Sigma(k) O^dagger  (Eq. 22)
    _, _, _, rot = km.stars(sg)
    for g in range(sg.nops):
        for k in range(km.nk):
            kt = rot[g, k]
            O = rep_at_k(cr.P_ao[g], cr.ao_atom, sg.shift[g], km.frac[kt])
            assert np.abs(S[kt] - O @ S[k] @ O.conj().T).max() < 1e-12 * scale
    # exact zeros off the irrep blocks of U^dagger Sigma U  (Eq. 26)
    st = SymSetup(cr.mesh, sg.W, sg.w, sg.shift, cr.P_ao, cr.P_aux, cr.ao_atom, cr.aux_atom)
    ao = st.adapt("ao")
    nontrivial = 0
    for k in range(km.nk):
        Sb = ao.U[k].conj().T @ S[k] @ ao.U[k]
        mask = np.ones((cr.nao, cr.nao), bool)
        for b in range(ao.nblk(k)):
            mask[ao.off[k][b]:ao.off[k][b + 1], ao.off[k][b]:ao.off[k][b + 1]] = False
        nontrivial += ao.nblk(k) > 1
        if mask.any():
            assert np.abs(Sb[:, mask]).max() < 1e-12 * scale
    assert nontrivial > 0


def test_flop_model():
    assert flops_per_output(8, 8, 32) == 8 * 8 * (2 * 32 * 512 + 1024 * 64)


# ---- Hartree-Fock exchange, Eq. 21c --------------------------------------------------
def test_exchange_brute_vs_ref_and_scalar_closed_form():
    from oracle.exchange_oracle import exchange_brute, exchange_ref
    inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=4, ntau=2, beta=3.0, nocc=1, seed=8)
    rng = np.random.default_rng(3)
    gamma = rng.standard_normal((inp.nk, 3, 3)) + 1j * rng.standard_normal((inp.nk, 3, 3))
    # unrelated partners: the oracle must not assume V^{k'k} = conj-transpose of V^{kk'}
    Vb = {(a, b): rng.standard_normal((4, 3, 3)) + 1j * rng.standard_normal((4, 3, 3)) for a in range(inp.nk) for b in range(inp.nk)}
    Va = {(a, b): rng.standard_normal((4, 3, 3)) + 1j * rng.standard_normal((4, 3, 3)) for a in range(inp.nk) for b in range(inp.nk)}
    calls = {"n": 0}

    def V_pair(a, b):
        # exchange_* ask for V^{k k'} first, V^{k' k} second
        calls["n"] += 1
        return Va[(a, b)] if calls["n"] % 2 == 1 else Vb[(a, b)]
    ks = [0, 3]
    brute = exchange_brute(inp.nk, gamma, V_pair, ks)
    ref = exchange_ref(inp.nk, lambda k: gamma[k], V_pair, ks)
    assert np.abs(brute - ref).max() < 1e-13 * np.abs(ref).max()
    # independent einsum statement of Eq. 21c
    for a, k in enumerate(ks):
        want = -sum(np.einsum("Qia,ab,Qbj->ij", Va[(k, kp)], gamma[kp], Vb[(kp, k)]) for kp in range(inp.nk)) / inp.nk
        assert np.abs(ref[a] - want).max() < 1e-13 * np.abs(want).max()
    # scalar closed form: nao = naux = 1, k-independent v and gamma  =>  K = -|v|^2 gamma  (sign and 1/Nk)
    v, g = 0.7 - 0.4j, 0.3 + 0.1j
    K = exchange_ref(5, lambda k: np.array([[g]]), lambda a, b: np.array([[[v]]]) if a <= b else np.array([[[np.conj(v)]]]), [2])
    # pairs (k,k') with k<k' contribute v*conj(v), k>k' conj(v)*v, k=k' v*v: write the expected sum out
    want = -(2 * abs(v) ** 2 + 2 * abs(v) ** 2 + v * v) * g / 5
    assert abs(K[0, 0, 0] - want) < 1e-15


def test_exchange_is_eq16_with_delta_W_and_gamma():
    """the paper's own relation: K^k (Eq. 21c) is Sigma^k (Eq. 16) with W -> delta_{QQ'} and G(k - q, tau) -> gamma^{k - q};
    sigma_ref is pinned on its own above."""
    from oracle.exchange_oracle import exchange_ref
    from oracle.sigma_oracle import sigma_ref
    inp = make_inputs("cfg1", mesh=(3, 2, 1), nao=3, naux=4, ntau=2, beta=3.0, nocc=1, seed=5)
    rng = np.random.default_rng(11)
    gamma = rng.standard_normal((inp.nk, 3, 3)) + 1j * rng.standard_normal((inp.nk, 3, 3))
    ks = list(range(inp.nk))
    K = exchange_ref(inp.nk, lambda k: gamma[k], inp.V_pair, ks)
    S = sigma_ref(inp.nk, inp.kmesh.sub, lambda k: gamma[k][None], lambda q: np.eye(4, dtype=complex)[None], inp.V_pair, ks)
    assert np.abs(K - S[:, 0]).max() < 1e-13 * np.abs(K).max()


def test_exchange_gauge_covariance_and_hermiticity():
    from oracle.exchange_oracle import exchange_ref
    inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=4, ntau=2, beta=3.0, nocc=1, seed=6)
    G = inp.G_full()
    gamma = -G[:, -1]                                           # gamma^k = G^k(0^-) = -G^k(beta), Hermitian
    ks = list(range(inp.nk))
    K = exchange_ref(inp.nk, lambda k: gamma[k], inp.V_pair, ks)
    assert np.abs(K - K.conj().transpose(0, 2, 1)).max() < 1e-13 * np.abs(K).max()       # V^{k'k} = V^{kk'}^dagger, gamma Hermitian
    rng = np.random.default_rng(2)
    T = [np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))[0] for _ in range(inp.nk)]
    K2 = exchange_ref(inp.nk, lambda k: T[k] @ gamma[k] @ T[k].conj().T,
                      lambda a, b: np.einsum("ip,Qpq,jq->Qij", T[a], inp.V_pair(a, b), T[b].conj()), ks)
    for k in ks:
        assert np.abs(K2[k] - T[k] @ K[k] @ T[k].conj().T).max() < 1e-13 * np.abs(K).max()


# ---- bare bubble P0, Eq. 20 / Algorithm 3 --------------------------------
def _kadd(inp):
    return lambda k, q: int(inp.kmesh.index(inp.kmesh.n[k] + inp.kmesh.n[q]))


def test_p0_brute_vs_ref_and_einsum():
    from oracle.p0_oracle import p0_brute, p0_ref
    inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=2, naux=3, ntau=3, beta=3.0, nocc=1, seed=8)
    rng = np.random.default_rng(4)
    G = rng.standard_normal((inp.nk, 3, 2, 2)) + 1j * rng.standard_normal((inp.nk, 3, 2, 2))       # no structure assumed
    V = {(a, b): rng.standard_normal((3, 2, 2)) + 1j * rng.standard_normal((3, 2, 2)) for a in range(inp.nk) for b in range(inp.nk)}
    add = _kadd(inp)
    qs = [0, 3]
    brute = p0_brute(inp.nk, add, G, lambda a, b: V[(a, b)], qs)
    ref = p0_ref(inp.nk, add, lambda k: G[k], lambda a, b: V[(a, b)], qs)
    assert np.abs(brute - ref).max() < 1e-13 * np.abs(ref).max()
    for iq, q in enumerate(qs):
        for n in range(3):
            want = -sum(np.einsum("Qda,cd,ab,Pbc->QP", V[(k, add(k, q))], -G[k, 2 - n], G[add(k, q), n], V[(add(k, q), k)])
                        for k in range(inp.nk)) / inp.nk
            assert np.abs(ref[iq, n] - want).max() < 1e-13 * np.abs(want).max()
    sub = p0_ref(inp.nk, add, lambda k: G[k], lambda a, b: V[(a, b)], qs, tau_idx=[2, 0])
    assert np.abs(sub - ref[:, [2, 0]]).max() == 0


def test_p0_single_level_closed_form():
    """one orbital, one auxiliary function, a k-independent level eps and coupling v: P0 = |v|^2 n_F (1 - n_F) for every tau
    (G(tau) = -e^{-eps tau}/(1 + e^{-beta eps}); -G(-tau) G(tau) = G(beta - tau) G(tau) = e^{-beta eps}/(1 + e^{-beta eps})^2)."""
    from oracle.p0_oracle import p0_ref
    beta, eps, v, ntau, nk = 4.0, 0.37, 0.8 - 0.3j, 7, 4
    tau = np.arange(ntau) * beta / (ntau - 1)
    g = (-np.exp(-eps * tau) / (1 + np.exp(-beta * eps))).reshape(ntau, 1, 1).astype(complex)
    P0 = p0_ref(nk, lambda k, q: (k + q) % nk, lambda k: g, lambda a, b: np.array([[[v]]]) if a <= b else np.array([[[np.conj(v)]]]), [0, 1])
    nF = 1 / (1 + np.exp(beta * eps))
    # q = 0: V^{k,k} V^{k,k} = v v; q = 1: pairs (k, k+1): v conj(v) except the wrap-around pair (3, 0): conj(v) v
    assert np.abs(P0[0, :, 0, 0] - v * v * nF * (1 - nF)).max() < 1e-15
    assert np.abs(P0[1, :, 0, 0] - abs(v) ** 2 * nF * (1 - nF)).max() < 1e-15


def test_p0_gauge_and_hermiticity():
    from oracle.p0_oracle import p0_ref
    inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=4, ntau=4, beta=3.0, nocc=1, seed=6)
    G = inp.G_full()
    add = _kadd(inp)
    qs = list(range(inp.nk))
    P0 = p0_ref(inp.nk, add, lambda k: G[k], inp.V_pair, qs)
    assert np.abs(P0 - P0.conj().transpose(0, 1, 3, 2)).max() < 1e-13 * np.abs(P0).max()      # G Hermitian, V^{k'k} = V^{kk'}^dagger
    rng = np.random.default_rng(2)
    T = [np.linalg.qr(rng.standard_normal((3, 3)) + 1j * rng.standard_normal((3, 3)))[0] for _ in range(inp.nk)]
    P0g = p0_ref(inp.nk, add, lambda k: T[k] @ G[k] @ T[k].conj().T,
                 lambda a, b: np.einsum("ip,Ppq,jq->Pij", T[a], inp.V_pair(a, b), T[b].conj()), qs)
    assert np.abs(P0g - P0).max() < 1e-13 * np.abs(P0).max()                                  # orbital gauge: invariant
    # auxiliary gauge S at momentum q: V^{k,k+q}(Q) -> S V, its partner V^{k+q,k} = (V^{k,k+q})^dagger -> conj(S) V: P0 -> S P0 S^dagger
    S = np.linalg.qr(rng.standard_normal((4, 4)) + 1j * rng.standard_normal((4, 4)))[0]
    q = 3
    calls = {"n": 0}

    def Vaux(a, b):
        calls["n"] += 1                      # p0_ref asks for V^{k,k+q} first, V^{k+q,k} second
        return np.einsum("PQ,Qij->Pij", S if calls["n"] % 2 == 1 else S.conj(), inp.V_pair(a, b))
    P0s = p0_ref(inp.nk, add, lambda k: G[k], Vaux, [q])[0]
    want = np.einsum("PQ,tQR,SR->tPS", S, P0[q], S.conj())
    assert np.abs(P0s - want).max() < 1e-13 * np.abs(P0).max()


# ---- Eq. 27, block-basis transform of V ---------------------------------------------------
def test_block_transform_brute_inverse_norm():
    from oracle.block_oracle import block_transform_brute, block_transform_ref
    rng = np.random.default_rng(9)
    u = lambda n: np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))[0]
    V = rng.standard_normal((4, 3, 3)) + 1j * rng.standard_normal((4, 3, 3))
    Ux, U2, U1 = u(4), u(3), u(3)
    a, b = block_transform_brute(V, Ux, U2, U1), block_transform_ref(V, Ux, U2, U1)
    assert np.abs(a - b).max() < 1e-14
    assert abs(np.linalg.norm(b) - np.linalg.norm(V)) < 1e-13                         # unitary change of basis
    back = np.einsum("QP,ba,Pai,ji->Qbj", Ux, U2, b, U1.conj())                       # the inverse of Eq. 27 written out
    assert np.abs(back - V).max() < 1e-13


def test_block_transform_makes_sigma_covariant():
    """Sigma from block-basis inputs (Eq. 26 for G and W, Eq. 27 for BOTH V tensors) = U^dagger Sigma U: fixes which index of V
    carries which conjugation, against the independently pinned sigma_ref."""
    from oracle.block_oracle import block_transform_ref
    from oracle.sigma_oracle import sigma_ref
    inp = make_inputs("cfg1", mesh=(2, 2, 1), nao=3, naux=4, ntau=2, beta=3.0, nocc=1, seed=6)
    G, W = inp.G_full(), inp.W_full()
    rng = np.random.default_rng(5)
    u = lambda n: np.linalg.qr(rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n)))[0]
    U = [u(3) for _ in range(inp.nk)]
    Ux = [u(4) for _ in range(inp.nk)]
    sub = lambda a, b: int(inp.kmesh.sub(a, b))
    ks = list(range(inp.nk))
    S = sigma_ref(inp.nk, sub, lambda k: G[k], lambda q: W[q], inp.V_pair, ks)
    # V_pair(k1, k2) = V^{k1,k2}: first momentum k1, second k2, auxiliary momentum q = k2 - k1 -> Eq. 27 with (k2 -> k1, k1 -> k2)
    Vb = lambda k1, k2: block_transform_ref(inp.V_pair(k1, k2), Ux[sub(k2, k1)], U[k1], U[k2])
    # W^q_{QQ'}: Q contracts with the V of auxiliary momentum -q, Q' with the one of +q (reading A6); both carry conj(U_aux) from
    # Eq. 27, so the matching two-index object is W_blk[P,P'] = sum_{QQ'} Uaux^{-q}_{Q,P} W_{QQ'} Uaux^{q}_{Q',P'}
    def Wb(q):
        return np.einsum("QP,tQR,RS->tPS", Ux[sub(0, q)], W[q], Ux[q])
    Sb = sigma_ref(inp.nk, sub, lambda k: U[k].conj().T @ G[k] @ U[k], Wb, Vb, ks)
    for k in ks:
        want = U[k].conj().T @ S[k] @ U[k]
        assert np.abs(Sb[k] - want).max() < 1e-12 * np.abs(S).max()


# ---- Eq. 19: P = [1 - P0]^{-1} P0 per (q, Omega) with caller-supplied tau <-> i Omega transforms ------
def test_dyson_p_loops_scalar_series_resolvent():
    from oracle.dyson_oracle import dyson_p_loops, dyson_p_ref
    rng = np.random.default_rng(12)
    nq, ntau, nw, n = 2, 5, 4, 3
    P0 = 0.2 * (rng.standard_normal((nq, ntau, n, n)) + 1j * rng.standard_normal((nq, ntau, n, n)))
    Tf = rng.standard_normal((nw, ntau)) + 1j * rng.standard_normal((nw, ntau))
    Tb = rng.standard_normal((ntau, nw)) + 1j * rng.standard_normal((ntau, nw))
    a, b = dyson_p_loops(P0, Tf, Tb), dyson_p_ref(P0, Tf, Tb)
    assert np.abs(a - b).max() < 1e-12 * np.abs(b).max()
    # scalar closed form, identity transforms: P = p0 / (1 - p0)
    p0 = np.array([0.3 - 0.2j, -1.7 + 0.4j, 0.05j]).reshape(1, 3, 1, 1)
    P = dyson_p_ref(p0, np.eye(3), np.eye(3))
    assert np.abs(P - p0 / (1 - p0)).max() < 1e-15
    # geometric series (small norm) and the resolvent identity, one frequency, identity transforms
    A = 0.1 * (rng.standard_normal((4, 4)) + 1j * rng.standard_normal((4, 4)))
    P = dyson_p_ref(A.reshape(1, 1, 4, 4), np.eye(1), np.eye(1))[0, 0]
    series = sum(np.linalg.matrix_power(A, k) for k in range(1, 40))
    assert np.abs(P - series).max() < 1e-14
    assert np.abs(P - A - A @ P).max() < 1e-15 and np.abs(P - A - P @ A).max() < 1e-15
    # the transforms act linearly on either side of the solve: diagonal (commuting) P0 goes through entry by entry
    d = 0.3 * (rng.standard_normal((1, ntau, 2)) + 1j * rng.standard_normal((1, ntau, 2)))
    P0d = np.zeros((1, ntau, 2, 2), complex)
    P0d[..., 0, 0], P0d[..., 1, 1] = d[..., 0], d[..., 1]
    Pd = dyson_p_ref(P0d, Tf, Tb)
    for j in range(2):
        w = Tf @ d[0, :, j]
        assert np.abs(Pd[0, :, j, j] - Tb @ (w / (1 - w))).max() < 1e-13
    assert np.abs(Pd[..., 0, 1]).max() == 0


# ---- Hartree J, Eq. 21b ----------------------------------------------------------------
def test_hartree_brute_vs_ref_scalar_and_einsum():
    from oracle.hartree_oracle import aux_density, hartree_brute, hartree_ref
    rng = np.random.default_rng(12)
    nk, nao, naux = 3, 2, 3
    gamma = rng.standard_normal((nk, nao, nao)) + 1j * rng.standard_normal((nk, nao, nao))            # no structure assumed
    V = rng.standard_normal((nk, naux, nao, nao)) + 1j * rng.standard_normal((nk, naux, nao, nao))
    ks = [0, 2]
    brute = hartree_brute(nk, gamma, lambda k: V[k], ks)
    ref = hartree_ref(nk, lambda k: gamma[k], lambda k: V[k], ks)
    assert np.abs(brute - ref).max() < 1e-13 * np.abs(brute).max()
    # an independent statement of Eq. 21b: the index pattern typed out once more, as one einsum
    ein = np.einsum("kQij,pab,pQba->kij", V[ks], gamma, V) / nk
    assert np.abs(ein - ref).max() < 1e-13 * np.abs(ref).max()
    # a transposed gamma / V (gamma_ab V_ab instead of gamma_ab V_ba) is a different number
    wrong = np.einsum("kQij,pab,pQab->kij", V[ks], gamma, V) / nk
    assert np.abs(wrong - ref).max() > 1e-2 * np.abs(ref).max()
    # scalar closed form: nao = naux = 1  ->  J^k = v_k (1/Nk) sum_k' gamma_k' v_k'
    g1 = rng.standard_normal((nk, 1, 1)) + 1j * rng.standard_normal((nk, 1, 1))
    v1 = rng.standard_normal((nk, 1, 1, 1)) + 1j * rng.standard_normal((nk, 1, 1, 1))
    J1 = hartree_ref(nk, lambda k: g1[k], lambda k: v1[k], range(nk))
    want = v1[:, 0, 0, 0] * (g1[:, 0, 0] * v1[:, 0, 0, 0]).sum() / nk
    assert np.abs(J1[:, 0, 0] - want).max() < 1e-14 * np.abs(want).max()
    # Hartree energy identity: (1/Nk) sum_k tr[gamma^k J^k] = sum_Q rho_Q^2
    rho = aux_density(nk, lambda k: gamma[k], lambda k: V[k])
    Jall = hartree_ref(nk, lambda k: gamma[k], lambda k: V[k], range(nk))
    e = sum(np.trace(gamma[k] @ Jall[k]) for k in range(nk)) / nk
    assert abs(e - (rho * rho).sum()) < 1e-13 * abs(e)


def test_hartree_invariances():
    from oracle.hartree_oracle import hartree_ref
    rng = np.random.default_rng(13)
    nk, nao, naux = 4, 3, 5
    gamma = rng.standard_normal((nk, nao, nao)) + 1j * rng.standard_normal((nk, nao, nao))
    V = rng.standard_normal((nk, naux, nao, nao)) + 1j * rng.standard_normal((nk, naux, nao, nao))
    J = hartree_ref(nk, lambda k: gamma[k], lambda k: V[k], range(nk))
    # orbital unitaries T_k (independent per k): gamma -> T gamma T^dagger, V_Q -> T V_Q T^dagger  =>  rho unchanged, J -> T J T^dagger
    T = [np.linalg.qr(rng.standard_normal((nao, nao)) + 1j * rng.standard_normal((nao, nao)))[0] for _ in range(nk)]
    J2 = hartree_ref(nk, lambda k: T[k] @ gamma[k] @ T[k].conj().T, lambda k: np.einsum("ip,Qpq,jq->Qij", T[k], V[k], T[k].conj()), range(nk))
    for k in range(nk):
        assert np.abs(J2[k] - T[k] @ J[k] @ T[k].conj().T).max() < 1e-13 * np.abs(J).max()
    # a real orthogonal rotation of the auxiliary index (both V carry Q un-conjugated at q = 0) leaves J unchanged ...
    S = np.linalg.qr(rng.standard_normal((naux, naux)))[0]
    J3 = hartree_ref(nk, lambda k: gamma[k], lambda k: np.einsum("PQ,Qij->Pij", S, V[k]), range(nk))
    assert np.abs(J3 - J).max() < 1e-13 * np.abs(J).max()
    # ... a complex unitary one does not
    Sc = np.linalg.qr(rng.standard_normal((naux, naux)) + 1j * rng.standard_normal((naux, naux)))[0]
    J4 = hartree_ref(nk, lambda k: gamma[k], lambda k: np.einsum("PQ,Qij->Pij", Sc, V[k]), range(nk))
    assert np.abs(J4 - J).max() > 1e-3 * np.abs(J).max()
    # linear in gamma
    g2 = rng.standard_normal((nk, nao, nao)) + 1j * rng.standard_normal((nk, nao, nao))
    Jb = hartree_ref(nk, lambda k: g2[k], lambda k: V[k], range(nk))
    Jab = hartree_ref(nk, lambda k: gamma[k] + 2.0 * g2[k], lambda k: V[k], range(nk))
    assert np.abs(Jab - J - 2.0 * Jb).max() < 1e-13 * np.abs(Jab).max()


@pytest.mark.parametrize("name", ["toy_diamond", "toy_wurtzite"])
def test_hartree_on_a_symmetric_crystal(name):
    """Hermitian gamma and the generator's V^{kk}(Q)_{ij} = conj(V^{kk}(Q)_{ji}): rho is real and J Hermitian; J transforms like
    every one-body matrix, J(g k) = O J(k) O^dagger (Eq. 22)."""
    from oracle.hartree_oracle import aux_density, hartree_ref
    inp = make_inputs(name)
    cr, sg, km = inp.cr, inp.cr.sg, inp.cr.kmesh
    G = np.stack([inp.G_k(k) for k in range(inp.nk)])
    gamma = -G[:, -1]                                           # gamma^k = G^k(0^-) = -G^k(beta)
    Vd = inp.V_pairs(range(inp.nk), range(inp.nk))              # V^{kk}
    rho = aux_density(inp.nk, lambda k: gamma[k], lambda k: Vd[k])
    assert np.abs(rho.imag).max() < 1e-12 * np.abs(rho).max() and np.abs(rho).max() > 1e-6
    J = hartree_ref(inp.nk, lambda k: gamma[k], lambda k: Vd[k], range(inp.nk))
    scale = np.abs(J).max()
    assert np.abs(J - J.conj().transpose(0, 2, 1)).max() < 1e-12 * scale
    _, _, _, rot = km.stars(sg)
    for g in range(sg.nops):
        for k in range(km.nk):
            kt = rot[g, k]
            O = rep_at_k(cr.P_ao[g], cr.ao_atom, sg.shift[g], km.frac[kt])
            assert np.abs(J[kt] - O @ J[k] @ O.conj().T).max() < 1e-11 * scale
