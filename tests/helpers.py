"""Test-side helpers: fold Sigma back to the orbital basis on the full zone (Eq. 26, 22) and a
numpy interpreter of the library's grouped-GEMM descriptors (checks the HOST plan without a GPU).
Nothing here is used by the product path."""
import numpy as np

from gwsig_synth.group import rep_at_k
from paper_2405_09494_b200.binding import (FLAG_ACCUM, FLAG_CONJ_A, FLAG_CONJ_B, FULL_BZ, IBZ, IBZ_BLOCK, NODIV)


_INPUTS = {}
_ORACLE = {}


def get_inputs(name, **over):
    """seeded inputs of a config / toy, built once per test session (cfg3 costs ~20 s, cfg5 minutes)."""
    from gwsig_synth import make_inputs
    key = (name, tuple(sorted((k, str(v)) for k, v in over.items())))
    if key not in _INPUTS:
        _INPUTS[key] = make_inputs(name, **over)
        _INPUTS[key]._cache_key = key
    return _INPUTS[key]


def oracle_sigma(inp, ks, taus=None):
    """oracle/sigma_oracle.sigma_ref at the (k, tau) sample -> [len(ks), len(taus), nao, nao].

    The two V tensors of Eq. 16 are generated INDEPENDENTLY (V^{k,k2} by V1_rows, V^{k2,k} by V2_rows; the oracle does
    not assume the conjugation relation), one batched Bloch sum per sampled k instead of one dense sum per (k, q) call.
    One k at a time, so the V rows of a single k bound the memory (16 GB at cfg5).  Results are cached per
    (inputs, k, tau) for the session: tests of different modes on the same sample share one oracle run."""
    from oracle.sigma_oracle import sigma_ref
    taus = np.arange(inp.ntau) if taus is None else np.asarray(taus)
    nk = inp.nk
    ckey = getattr(inp, "_cache_key", None)
    need = [int(k) for k in ks if ckey is None or any((ckey, int(k), int(t)) not in _ORACLE for t in taus)]
    store = {}
    if need:
        Gs = {k: (inp.G_k(k) if hasattr(inp, "G_k") else inp.G_full()[k])[taus] for k in range(nk)}
        Ws = {q: inp.W_full([q])[0][taus] for q in range(nk)}
        for k in need:
            k2s = list(range(nk))
            rows2 = inp.V2_rows(k, k2s)                    # V^{k2,k}
            rows1 = inp.V1_rows(k, k2s)                    # V^{k,k2}

            diag = [0]

            def V_pair(a, b, k=k, rows1=rows1, rows2=rows2, diag=diag):
                if a == k and b == k:                      # q = 0: first call is V^{k,k-q}, second V^{k-q,k}
                    diag[0] ^= 1
                    return rows1[k] if diag[0] else rows2[k]
                return rows1[b] if a == k else rows2[a]
            res = sigma_ref(nk, inp.kmesh.sub, lambda kk: Gs[kk], lambda q: Ws[q], V_pair, [k])[0]
            del rows1, rows2
            for b, t in enumerate(taus):
                store[(k, int(t))] = res[b]
                if ckey is not None:
                    _ORACLE[(ckey, k, int(t))] = res[b]
    out = []
    for k in ks:
        out.append(np.stack([store[(int(k), int(t))] if (int(k), int(t)) in store else _ORACLE[(ckey, int(k), int(t))] for t in taus]))
    return np.stack(out)


def fold_to_orbital(cfg, inp, sigma_list):
    """list over cfg.out_list of [nt, nao, nao] (basis of the mode) -> dict k -> [nt, nao, nao] in the
    orbital basis for EVERY mesh point: Sigma_orb(k_I) = U Sigma_blk U^dagger (Eq. 26), then
    Sigma(k') = O Sigma(k_I) O^dagger (Eq. 22)."""
    out = {}
    for i, k in enumerate(cfg.out_list):
        S = sigma_list[i]
        if cfg.mode == IBZ_BLOCK:
            U = cfg.ao.U[k]
            S = U @ S @ U.conj().T
        out[int(k)] = S
    if cfg.mode == FULL_BZ:
        return out
    cr = inp.cr
    for k in range(cfg.nk):
        if k in out or int(cfg.ir_of[k]) not in out:     # (a restricted set of output points leaves stars out)
            continue
        g = int(cfg.op_of[k])
        O = rep_at_k(cr.P_ao[g], cr.ao_atom, cr.sg.shift[g], cr.kmesh.frac[k])
        out[k] = O @ out[int(cfg.ir_of[k])] @ O.conj().T
    return out


def rel_err(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def _idx(d, n):
    i = np.arange(n, dtype=np.int64)
    if d["div"] == NODIV:
        return i * d["lo"]
    return (i // d["div"]) * d["hi"] + (i % d["div"]) * d["lo"]


def run_stage_numpy(prob, seg, A, B, C, t0):
    """execute one stage's descriptors exactly as documented in include/gwsig_plan.h."""
    for P in prob:
        cm, cn = _idx(P["cm"], P["M"]), _idx(P["cn"], P["N"])
        for bt in range(P["nbatch"]):
            acc = np.zeros((P["M"], P["N"]), complex)
            for s in range(P["seg_begin"], P["seg_begin"] + P["seg_count"]):
                S = seg[s]
                a0 = S["a_off"] + bt * P["a_bstride"] + t0 * P["a_tstride"]
                b0 = S["b_off"] + bt * P["b_bstride"] + t0 * P["b_tstride"]
                Am = A[a0 + _idx(S["am"], P["M"])[:, None] + _idx(S["ak"], S["K"])[None, :]]
                Bm = B[b0 + _idx(S["bk"], S["K"])[:, None] + _idx(S["bn"], P["N"])[None, :]]
                if P["flags"] & FLAG_CONJ_A:
                    Am = Am.conj()
                if P["flags"] & FLAG_CONJ_B:
                    Bm = Bm.conj()
                acc += Am @ Bm
            ci = P["c_off"] + bt * P["c_bstride"] + t0 * P["c_tstride"] + cm[:, None] + cn[None, :]
            if P["flags"] & FLAG_ACCUM:
                C[ci] += acc
            else:
                C[ci] = acc


def oracle_exchange(inp, gamma_of, ks):
    """oracle/exchange_oracle.exchange_ref with independently generated V^{k k'} (V1_rows) and V^{k' k} (V2_rows)."""
    from oracle.exchange_oracle import exchange_ref
    out = []
    for k in ks:
        k = int(k)
        k2s = list(range(inp.nk))
        rows1, rows2 = inp.V1_rows(k, k2s), inp.V2_rows(k, k2s)
        diag = [0]

        def V_pair(a, b, k=k, rows1=rows1, rows2=rows2, diag=diag):
            if a == k and b == k:
                diag[0] ^= 1
                return rows1[k] if diag[0] else rows2[k]
            return rows1[b] if a == k else rows2[a]
        out.append(exchange_ref(inp.nk, gamma_of, V_pair, [k])[0])
    return np.stack(out)


def run_plan_numpy(cfg, inp, G_flat, W_flat, V_flat, push_pairs=None, nt=None, exchange=False):
    """emulate gwsig_sigma_eval's orchestration with the descriptors of gwsig_plan_get()."""
    lib = cfg.lib
    ntau, nao, naux, nk = cfg.ntau, cfg.nao, cfg.naux, cfg.nk
    nt = ntau if nt is None else nt
    push_pairs = cfg.npairs if push_pairs is None else push_pairs
    sig_elems = lib.buffer_sizes()[2]
    acc = np.zeros(sig_elems, complex)
    # G / W sources
    if cfg.mode == IBZ:
        cr = inp.cr
        Gi = G_flat.reshape(len(cfg.ir_list), ntau, nao, nao)
        Wi = None if exchange else W_flat.reshape(len(cfg.ir_list), ntau, naux, naux)
        ir_index = {int(k): i for i, k in enumerate(cfg.ir_list)}

        def unfold(X, P, atom, k):
            g = int(cfg.op_of[k])
            O = rep_at_k(P[g], atom, cr.sg.shift[g], cr.kmesh.frac[k])
            return O @ X[ir_index[int(cfg.ir_of[k])]] @ O.conj().T
        Gsrc = np.stack([unfold(Gi, cr.P_ao, cr.ao_atom, k) for k in range(nk)]).ravel()
    elif getattr(cfg, "general_gauge", False):
        # Eq. 28: packed blocks of every mesh point through the two unfold launches (plan stages 11, 12) with the library's O_block
        Oao, Oaux = block_O(cfg, inp, "ao"), block_O(cfg, inp, "aux")
        Gsrc = unfold_blocks_numpy(lib, 11, 0, nk, G_flat, Oao, ntau)
    else:
        Gsrc = G_flat
    voff = [lib.pair_info(p)[3] for p in range(cfg.npairs)] + [V_flat.size]
    p0 = 0
    while p0 < cfg.npairs:
        npp = min(push_pairs, cfg.npairs - p0)
        q_first, q_last = p0 // cfg.nk1, (p0 + npp - 1) // cfg.nk1
        if exchange:
            Wsrc = None
        elif cfg.mode == IBZ:
            Wsrc = np.stack([unfold(Wi, cr.P_aux, cr.aux_atom, q) for q in range(q_first, q_last + 1)]).ravel()
        elif getattr(cfg, "general_gauge", False):
            Wsrc = unfold_blocks_numpy(lib, 21, q_first, q_last - q_first + 1, W_flat, Oaux[q_first:q_last + 1], ntau)
        else:
            Wsrc = W_flat
        Vsub = V_flat[voff[p0]:voff[p0 + npp]]
        for t0 in range(0, ntau, nt):
            ntc = min(nt, ntau - t0)
            X = np.zeros(Vsub.size * ntc, complex)
            Y = np.zeros(Vsub.size * ntc, complex)
            pr, sg, _ = lib.plan_get(p0, npp, ntc, 1)
            run_stage_numpy(pr, sg, Gsrc, Vsub, X, t0)
            if exchange:                       # Eq. 21c: W -> delta, stage 2 skipped, stage 3 reads X
                Y = X
            else:
                pr, sg, _ = lib.plan_get(p0, npp, ntc, 2)
                run_stage_numpy(pr, sg, X, Wsrc, Y, t0)
            pr, sg, _ = lib.plan_get(p0, npp, ntc, 3)
            run_stage_numpy(pr, sg, Y, Vsub, acc, t0)
        p0 += npp
    return -acc / nk


def block_O(cfg, inp, kind):
    """test-side O_block = U^{k'}^dagger O^{k_I}(alpha^) U^{k_I} (Eq. 28), packed diagonal blocks per mesh point
    (list of flat arrays) -- what gwsig_set_blocks computes internally from U."""
    cr = inp.cr
    basis = cfg.ao if kind == "ao" else cfg.aux
    P, atom = (cr.P_ao, cr.ao_atom) if kind == "ao" else (cr.P_aux, cr.aux_atom)
    out = []
    for k in range(cfg.nk):
        g, kI = int(cfg.op_of[k]), int(cfg.ir_of[k])
        O = rep_at_k(P[g], atom, cr.sg.shift[g], cr.kmesh.frac[k])
        R = basis.U[k].conj().T @ O @ basis.U[kI]
        off = basis.off[k]
        out.append(np.concatenate([R[off[b]:off[b + 1], off[b]:off[b + 1]].ravel() for b in range(len(off) - 1)]))
    return out


def unfold_blocks_numpy(lib, stage0, k_first, k_count, X_flat, O_list, ntau):
    """run the two unfold launches (stage0 = 11 for G, 21 for W) with the numpy interpreter; O_list: packed O_block of the
    points k_first .. k_first + k_count - 1 (the library addresses O from mesh point 0: pad in front)."""
    pr1, sg1, _ = lib.plan_get(k_first, k_count, ntau, stage0)
    pr2, sg2, _ = lib.plan_get(k_first, k_count, ntau, stage0 + 1)
    Oall = np.concatenate(O_list)
    # b_off of the descriptors is relative to the whole-mesh O table: shift to this slice
    shift = int(min(S["b_off"] for S in sg1))
    Opad = np.concatenate([np.zeros(shift, complex), Oall])
    n_out = 0
    for P in pr1:
        n_out = max(n_out, int(P["c_off"] + _idx(P["cm"], P["M"])[-1] + _idx(P["cn"], P["N"])[-1] + 1))
    T = np.zeros(n_out, complex)
    run_stage_numpy(pr1, sg1, X_flat, Opad, T, 0)
    out = np.zeros(n_out, complex)
    run_stage_numpy(pr2, sg2, T, Opad, out, 0)
    return out


# ---- N1: bare bubble (Eq. 20) ---------------------------------------------------------------------------------
def p0_pairs(cfg, inp):
    """(k, q, k+q) of every P0 pair in the library's order: pair = k * nq + iq, q = out_list[iq]."""
    km = inp.kmesh
    return [(k, int(q), int(km.index(km.n[k] + km.n[int(q)]))) for k in range(cfg.nk) for q in cfg.out_list]


def pack_V_p0(cfg, inp):
    """T = V^{k,k+q}_{Q,da} [naux][nao][nao] for every P0 pair, flat."""
    return np.ascontiguousarray(np.concatenate([inp.V_pair(k, kq).ravel() for (k, q, kq) in p0_pairs(cfg, inp)]), np.complex128)


def oracle_p0(inp, qs, taus=None):
    """oracle/p0_oracle.p0_ref with independently generated V^{k,k+q} (V_pair(k, k+q)) and V^{k+q,k} (V_pair(k+q, k))."""
    from oracle.p0_oracle import p0_ref
    km = inp.kmesh
    Gc = {}

    def G_of(k):
        if k not in Gc:
            Gc[k] = inp.G_k(k) if hasattr(inp, "G_k") else inp.G_full()[k]
        return Gc[k]
    return p0_ref(inp.nk, lambda k, q: int(km.index(km.n[k] + km.n[q])), G_of, inp.V_pair, [int(q) for q in qs], taus)


def run_p0_plan_numpy(cfg, inp, G_flat, V_flat, push_pairs=None, nt=None):
    """emulate gwsig_p0_eval with the descriptors of plan stages 31, 32, 33 (Algorithm 3) -> [nq, ntau, naux, naux]."""
    lib = cfg.lib
    ntau, nao, naux, nk = cfg.ntau, cfg.nao, cfg.naux, cfg.nk
    nq = len(cfg.out_list)
    npairs = nk * nq
    nt = ntau if nt is None else nt
    push_pairs = npairs if push_pairs is None else push_pairs
    if cfg.mode == IBZ:
        cr = inp.cr
        Gi = G_flat.reshape(len(cfg.ir_list), ntau, nao, nao)
        ir_index = {int(k): i for i, k in enumerate(cfg.ir_list)}
        Gs = []
        for k in range(nk):
            g = int(cfg.op_of[k])
            O = rep_at_k(cr.P_ao[g], cr.ao_atom, cr.sg.shift[g], cr.kmesh.frac[k])
            Gs.append(O @ Gi[ir_index[int(cfg.ir_of[k])]] @ O.conj().T)
        Gsrc = np.stack(Gs)
    else:
        Gsrc = G_flat.reshape(nk, ntau, nao, nao)
    # the library's two transposed copies: G(beta - tau)^T (the sign of G(-tau) = -G(beta - tau) is in the scale) and G(tau)^T
    Grev = np.ascontiguousarray(Gsrc[:, ::-1].transpose(0, 1, 3, 2)).ravel()
    Gsrc = np.ascontiguousarray(Gsrc.transpose(0, 1, 3, 2)).ravel()
    acc = np.zeros(nq * ntau * naux * naux, complex)
    xs = naux * nao * nao
    p0 = 0
    while p0 < npairs:
        npp = min(push_pairs, npairs - p0)
        # the library's stage-1 / stage-2 descriptors address its aux-last copy T'[x][y][Q] = T[Q][x][y] of the pushed tensors
        Vsub = np.ascontiguousarray(V_flat[p0 * xs:(p0 + npp) * xs].reshape(npp, naux, nao * nao).transpose(0, 2, 1)).ravel()
        for t0 in range(0, ntau, nt):
            ntc = min(nt, ntau - t0)
            X1 = np.zeros(npp * xs * ntc, complex)
            X2 = np.zeros(npp * xs * ntc, complex)
            pr, sg, _ = lib.plan_get(p0, npp, ntc, 31)
            run_stage_numpy(pr, sg, Grev, Vsub, X1, t0)
            pr, sg, _ = lib.plan_get(p0, npp, ntc, 32)
            run_stage_numpy(pr, sg, Gsrc, Vsub, X2, t0)
            pr, sg, _ = lib.plan_get(p0, npp, ntc, 33)
            run_stage_numpy(pr, sg, X1, X2, acc, t0)
        p0 += npp
    return (acc / nk).reshape(nq, ntau, naux, naux)


# ---- N4: Eq. 27 on the device ----------------------------------------------------------------------------------
def oracle_packed_V(cfg, inp, pairs):
    """oracle/block_oracle.block_transform_ref of V2 = V^{k2,k1} for the given pairs, packed by the layout include/gwsig.h
    documents (aux block p major, [n_p][N_p], segments [a][i] in triple order) -- written out here, not taken from the package."""
    from oracle.block_oracle import block_transform_ref
    out = []
    for p in pairs:
        k1, k2, q, _, _ = cfg.lib.pair_info(p, with_layout=False)
        T = block_transform_ref(inp.V2_rows(k1, [k2])[0], cfg.aux.U[q], cfg.ao.U[k2], cfg.ao.U[k1])
        oq, o2, o1 = cfg.aux.off[q], cfg.ao.off[k2], cfg.ao.off[k1]
        trip = cfg.triples[p]
        for bp in range(len(oq) - 1):
            segs = [T[oq[bp]:oq[bp + 1], o2[a]:o2[a + 1], o1[i]:o1[i + 1]].reshape(oq[bp + 1] - oq[bp], -1) for (pp, a, i) in trip if pp == bp]
            if segs:
                out.append(np.concatenate(segs, axis=1).ravel())
    return np.concatenate(out)


def run_vtransform_numpy(cfg, inp, p0, npairs):
    """the three launches of gwsig_block_transform_v (plan stages 41, 42, 43) with the numpy interpreter."""
    lib = cfg.lib
    xs = cfg.naux * cfg.nao ** 2
    info = [lib.pair_info(p) for p in range(p0, p0 + npairs)]
    V = np.concatenate([inp.V2_rows(i[0], [i[1]])[0].ravel() for i in info])
    Uaux, Uao = np.ascontiguousarray(cfg.aux.U).ravel(), np.ascontiguousarray(cfg.ao.U).ravel()
    T1, T2 = np.zeros(npairs * xs, complex), np.zeros(npairs * xs, complex)
    out = np.zeros(sum(i[4] for i in info), complex)
    for step, (A, Bm, C) in enumerate(((V, Uaux, T1), (T1, Uao, T2), (T2, Uao, out)), 1):
        pr, sg, _ = lib.plan_get(p0, npairs, 1, 40 + step)
        run_stage_numpy(pr, sg, A, Bm, C, 0)
    return out


def oracle_block_maxabs(cfg, inp, pairs, mb_aux, mb_ao):
    """max |.| of every candidate block (p, alpha, iota) of the Eq. 27 transform (oracle/block_oracle.py, dense) of the listed
    pairs -> [len(pairs), mb_aux, mb_ao, mb_ao]; zero where a mesh point has fewer blocks."""
    from oracle.block_oracle import block_transform_ref
    lib = cfg.lib
    out = np.zeros((len(pairs), mb_aux, mb_ao, mb_ao))
    for n, p in enumerate(pairs):
        k1, k2, q = lib.pair_info(p, with_layout=False)[:3]
        T = block_transform_ref(inp.V2_rows(k1, [k2])[0], cfg.aux.U[q], cfg.ao.U[k2], cfg.ao.U[k1])
        op, o2, o1 = cfg.aux.off[q], cfg.ao.off[k2], cfg.ao.off[k1]
        for b in range(len(op) - 1):
            for al in range(len(o2) - 1):
                for io in range(len(o1) - 1):
                    out[n, b, al, io] = np.abs(T[op[b]:op[b + 1], o2[al]:o2[al + 1], o1[io]:o1[io + 1]]).max()
    return out


def triples_from_maxabs(mx, thresh, vmax):
    """allowed (p, alpha, iota) per pair from the block maxima, sorted by p, alpha, iota (the order symsetup.block_V2 uses)."""
    return [np.argwhere(m > thresh * vmax).astype(np.int32) for m in mx]


def run_dense_vtransform_numpy(cfg, inp, p0, npairs):
    """launches 41, 42, 44 of gwsig_block_maxabs (the Eq. 27 transform for EVERY block, dense) with the numpy interpreter."""
    lib = cfg.lib
    xs = cfg.naux * cfg.nao ** 2
    info = [lib.pair_info(p, with_layout=False) for p in range(p0, p0 + npairs)]
    V = np.concatenate([inp.V2_rows(i[0], [i[1]])[0].ravel() for i in info])
    Uaux, Uao = np.ascontiguousarray(cfg.aux.U).ravel(), np.ascontiguousarray(cfg.ao.U).ravel()
    T1, T2, T3 = (np.zeros(npairs * xs, complex) for _ in range(3))
    for step, (A, Bm, C) in zip((1, 2, 4), ((V, Uaux, T1), (T1, Uao, T2), (T2, Uao, T3))):
        pr, sg, _ = lib.plan_get(p0, npairs, 1, 40 + step)
        run_stage_numpy(pr, sg, A, Bm, C, 0)
    return T3.reshape(npairs, cfg.naux, cfg.nao, cfg.nao)
