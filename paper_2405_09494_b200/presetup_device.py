"""Device (torch) version of the host pre-step of ``symsetup`` for MANY pairs at once:
Eq. 27 block transform of V2 = V^{k2,k1}, detection of the allowed (p, alpha, iota)
blocks ("only non-zero blocks are considered") and packing into the ragged layout
``gwsig_sigma_push_pairs`` expects in IBZ_BLOCK mode (include/gwsig.h).

Like ``symsetup`` this is the paper's pre-step ("before starting the self-consistent GW calculation",
PAPER.md:261): it prepares INPUTS of the hot path, is never timed as part of it and evaluates no Sigma.
``symsetup.block_V2`` does the same per pair in numpy (one pair costs ~0.1 s at config 4); the large configs
have 4 032 / 14 848 pairs of 10 / 16 MB, so the transform runs as batched matrix products on the GPU and
the packing as one masked scatter per batch.  tests/test_symsetup.py checks it against ``symsetup.block_V2``.
"""
from __future__ import annotations

import numpy as np


class DeviceBlocker:
    """block bases of one configured crystal (``pack.Configured`` in IBZ_BLOCK mode) on a torch device."""

    def __init__(self, cfg, torch, dev):
        self.cfg, self.torch, self.dev = cfg, torch, dev
        ao, aux = cfg.ao, cfg.aux
        self.nk, self.nao, self.naux = cfg.nk, cfg.nao, cfg.naux
        self.U_ao = torch.from_numpy(np.ascontiguousarray(ao.U)).to(dev)          # [nk, nao, nao]
        self.U_aux = torch.from_numpy(np.ascontiguousarray(aux.U)).to(dev)        # [nk, naux, naux]
        # per mesh point: block id of every basis function, block offsets / sizes padded to the max block count
        self.nb_ao = np.array([len(o) - 1 for o in ao.off])
        self.nb_aux = np.array([len(o) - 1 for o in aux.off])
        self.mb_ao, self.mb_aux = int(self.nb_ao.max()), int(self.nb_aux.max())

        def tables(off_list, n, mb):
            lab = np.zeros((self.nk, n), np.int64)
            start = np.zeros((self.nk, mb), np.int64)
            size = np.zeros((self.nk, mb), np.int64)
            for k, off in enumerate(off_list):
                off = np.asarray(off)
                lab[k] = np.repeat(np.arange(len(off) - 1), np.diff(off))
                start[k, :len(off) - 1] = off[:-1]
                size[k, :len(off) - 1] = np.diff(off)
            return lab, start, size
        self.lab_ao, self.start_ao, self.size_ao = tables(ao.off, self.nao, self.mb_ao)
        self.lab_aux, self.start_aux, self.size_aux = tables(aux.off, self.naux, self.mb_aux)
        self.d_lab_ao = torch.from_numpy(self.lab_ao).to(dev)
        self.d_lab_aux = torch.from_numpy(self.lab_aux).to(dev)
        self.ncand = self.mb_aux * self.mb_ao * self.mb_ao          # candidate triples per pair (padded)

    # ---- Eq. 27 ------------------------------------------------------------------------------------
    def transform(self, V, qs, k2s, k1s):
        """V [n, naux, nao, nao] = V^{k2,k1}_{Q,bj} (orbital basis, device) ->
        V2blk_{P,a,i} = sum conj(Uaux^q_{Q,P}) conj(U^{k2}_{b,a}) V_{Q,bj} U^{k1}_{j,i}    (Eq. 27)"""
        t = self.torch
        n = V.shape[0]
        q, k2, k1 = (t.as_tensor(np.asarray(x), device=self.dev) for x in (qs, k2s, k1s))
        T = t.matmul(self.U_aux[q].conj().transpose(1, 2), V.reshape(n, self.naux, self.nao * self.nao))
        T = T.reshape(n, self.naux, self.nao, self.nao)
        T = t.matmul(self.U_ao[k2].conj().transpose(1, 2).unsqueeze(1), T)
        return t.matmul(T, self.U_ao[k1].unsqueeze(1))

    def _labels(self, qs, k2s, k1s):
        """candidate-triple id of every element (P, a, i) of every pair: (p * mb_ao + alpha) * mb_ao + iota."""
        t = self.torch
        q, k2, k1 = (t.as_tensor(np.asarray(x), device=self.dev) for x in (qs, k2s, k1s))
        lp = self.d_lab_aux[q][:, :, None, None]
        la = self.d_lab_ao[k2][:, None, :, None]
        li = self.d_lab_ao[k1][:, None, None, :]
        return (lp * self.mb_ao + la) * self.mb_ao + li

    def block_maxabs(self, T, qs, k2s, k1s):
        """max |.| of every candidate block of the transformed tensors -> [n, ncand] (host numpy)."""
        t = self.torch
        n = T.shape[0]
        L = self._labels(qs, k2s, k1s) + (t.arange(n, device=self.dev) * self.ncand)[:, None, None, None]
        out = t.zeros(n * self.ncand, dtype=t.float64, device=self.dev)
        out.scatter_reduce_(0, L.reshape(-1), T.abs().reshape(-1), "amax", include_self=True)
        return out.reshape(n, self.ncand).cpu().numpy()

    def triples_from_maxabs(self, mx, qs, k2s, k1s, thresh, vmax):
        """allowed (p, alpha, iota) per pair, sorted by p then alpha then iota (the order symsetup.block_V2 uses)."""
        out = []
        for r in range(mx.shape[0]):
            nbq, nb2, nb1 = self.nb_aux[qs[r]], self.nb_ao[k2s[r]], self.nb_ao[k1s[r]]
            m = mx[r].reshape(self.mb_aux, self.mb_ao, self.mb_ao)[:nbq, :nb2, :nb1]
            out.append(np.argwhere(m > thresh * vmax).astype(np.int32))
        return out

    # ---- packing -------------------------------------------------------------------------------------
    def pack_tables(self, triples, qs, k2s, k1s):
        """per pair: c0 of every candidate triple (-1 = not allowed), offset / row length of every aux block, total size."""
        n = len(triples)
        c0 = -np.ones((n, self.ncand), np.int64)
        poff = np.zeros((n, self.mb_aux), np.int64)
        Np = np.zeros((n, self.mb_aux), np.int64)
        size = np.zeros(n, np.int64)
        for r, T in enumerate(triples):
            q, k2, k1 = qs[r], k2s[r], k1s[r]
            if len(T):
                seg = self.size_ao[k2][T[:, 1]] * self.size_ao[k1][T[:, 2]]
                np.add.at(Np[r], T[:, 0], seg)
                # c0 = running sum of segment sizes inside each aux block (triples are sorted by p)
                cs = np.cumsum(seg) - seg
                first = np.zeros(self.mb_aux, np.int64)
                firstpos = np.searchsorted(T[:, 0], np.arange(self.mb_aux))
                ok = firstpos < len(T)
                first[ok] = cs[firstpos[ok]]
                c0[r, (T[:, 0] * self.mb_ao + T[:, 1]) * self.mb_ao + T[:, 2]] = cs - first[T[:, 0]]
            rows = self.size_aux[q] * Np[r]
            poff[r] = np.cumsum(rows) - rows
            size[r] = rows.sum()
        return c0, poff, Np, size

    def pack(self, T, qs, k2s, k1s, tables, dst, dst_off):
        """scatter the allowed blocks of T [n, naux, nao, nao] into the flat packed buffer ``dst`` (device complex128);
        pair r starts at element dst_off[r].  Layout: aux block p major, [n_p][N_p], segments [a][i] in triple order."""
        t = self.torch
        c0, poff, Np, _ = tables
        n = T.shape[0]
        dev = self.dev
        q, k2, k1 = (t.as_tensor(np.asarray(x), device=dev) for x in (qs, k2s, k1s))
        d = lambda a: t.as_tensor(a, device=dev)
        c0d, poffd, Npd = d(c0), d(poff), d(Np)
        lp = self.d_lab_aux[q]                                   # [n, naux]
        la, li = self.d_lab_ao[k2], self.d_lab_ao[k1]            # [n, nao]
        ar = t.arange(n, device=dev)[:, None]
        P_in = t.arange(self.naux, device=dev)[None, :] - d(self.start_aux)[q].gather(1, lp)      # row inside the aux block
        a_in = t.arange(self.nao, device=dev)[None, :] - d(self.start_ao)[k2].gather(1, la)
        i_in = t.arange(self.nao, device=dev)[None, :] - d(self.start_ao)[k1].gather(1, li)
        ni = d(self.size_ao)[k1].gather(1, li)                   # n_iota of the block each i belongs to
        rowbase = poffd.gather(1, lp) + P_in * Npd.gather(1, lp) + d(np.asarray(dst_off))[:, None]  # [n, naux]
        L = (lp[:, :, None, None] * self.mb_ao + la[:, None, :, None]) * self.mb_ao + li[:, None, None, :]
        c0e = c0d.gather(1, L.reshape(n, -1)).reshape(L.shape)
        idx = rowbase[:, :, None, None] + c0e + a_in[:, None, :, None] * ni[:, None, None, :] + i_in[:, None, None, :]
        mask = c0e >= 0
        dst[idx[mask]] = T[mask]
        del ar
