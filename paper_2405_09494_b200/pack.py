"""Host-side marshalling: configure a Gwsig context from plain group arrays and lay the
inputs out the way ``gwsig_sigma_eval`` expects them in each mode (include/gwsig.h).
No arithmetic of the hot path happens here; the block-basis transform of the inputs is the
paper's pre-step (Eq. 26-27) and lives in ``symsetup``.
"""
from __future__ import annotations

import numpy as np

from .binding import FULL_BZ, IBZ, IBZ_BLOCK, Gwsig
from .symsetup import SymSetup


class Configured:
    """a Gwsig context with lattice / symmetry (/ blocks) set, plus the host pre-step objects."""

    def __init__(self, lib: Gwsig, mode: int, a, mesh, nao, naux, ntau, beta, pos, ao_atom, aux_atom,
                 W=None, w=None, shift=None, P_ao=None, P_aux=None, seed: int = 7, out_points=None, scramble_gauge=None, pass_U=False):
        self.lib, self.mode = lib, mode
        self.general_gauge = scramble_gauge is not None and mode == IBZ_BLOCK
        self.nao, self.naux, self.ntau = nao, naux, ntau
        lib.set_lattice(a, mesh, nao, naux, ntau, beta)
        self.setup = None
        self.ao = self.aux = None
        if W is None:
            if mode != FULL_BZ:
                raise ValueError("IBZ modes need the space-group operations")
            lib.set_symmetry(None, None, None, None, None, mode)
        else:
            lib.set_atoms(pos, ao_atom, aux_atom)
            lib.set_symmetry(W, w, P_ao, P_aux, shift, mode)
            self.setup = SymSetup(mesh, W, w, shift, P_ao, P_aux, ao_atom, aux_atom, seed=seed)
        self.ir_list, self.ir_of, self.op_of = lib.get_ibz()
        if callable(out_points):                       # e.g. lambda wedge: wedge[:2]
            out_points = out_points(np.arange(lib.nk) if mode == FULL_BZ else self.ir_list)
        if out_points is not None:
            lib.set_output_points(out_points)
        self.npairs, self.nk1 = lib.pair_count()
        self.nk = lib.nk
        self.out_list = (np.arange(self.nk) if mode == FULL_BZ else self.ir_list) if out_points is None else np.asarray(out_points)
        if mode == IBZ_BLOCK:
            self.ao, self.aux = self.setup.adapt("ao"), self.setup.adapt("aux")
            if scramble_gauge is None and pass_U:
                lib.set_blocks(self.ao.off, self.aux.off, self.ao.U, self.aux.U)     # gauge S5 with U handed over (for Eq. 27 on the device)
            elif scramble_gauge is None:
                lib.set_blocks(self.ao.off, self.aux.off)                 # gauge S5: O_block = 1, no U needed
            else:                                                         # general gauge: the library forms O_block (Eq. 28)
                self.ao = self.setup.scramble(self.ao, scramble_gauge)
                self.aux = self.setup.scramble(self.aux, scramble_gauge + 1)
                lib.set_blocks(self.ao.off, self.aux.off, self.ao.U, self.aux.U)

    # ---- inputs -------------------------------------------------------------------------------
    def pack_GW(self, G_of, W_of):
        """G_of(k) -> [ntau,nao,nao], W_of(q) -> [ntau,naux,naux] in the orbital basis.
        Returns flat complex128 arrays in the layout of the current mode."""
        pts = np.arange(self.nk) if self.mode == FULL_BZ else self.ir_list
        if self.mode != IBZ_BLOCK:
            G = np.stack([G_of(int(k)) for k in pts]).ravel()
            W = np.stack([W_of(int(k)) for k in pts]).ravel()
            return np.ascontiguousarray(G, np.complex128), np.ascontiguousarray(W, np.complex128)
        st = self.setup
        G = np.concatenate([st.pack_diag_blocks(G_of(int(k)), self.ao.U[k], self.ao.off[k]).ravel() for k in pts])
        W = np.concatenate([st.pack_diag_blocks(W_of(int(k)), self.aux.U[k], self.aux.off[k]).ravel() for k in pts])
        return np.ascontiguousarray(G, np.complex128), np.ascontiguousarray(W, np.complex128)

    def pack_V(self, V2_rows, thresh: float = 1e-9):
        """V2_rows(k1, k2s) -> [len, naux, nao, nao] = V^{k2,k1}_{Q,bj}.  Returns the flat V buffer for ALL
        pairs in pair order; in IBZ_BLOCK mode also finds the allowed triples and calls set_triples."""
        lib = self.lib
        nk1 = self.nk1
        # pair = q * nk1 + i1, k2 = k1 - q: gather row-wise (one V2_rows call per k1), then order q-major
        per_pair = [None] * self.npairs
        trip = [None] * self.npairs
        vmax = None
        for i1, k1 in enumerate(self.out_list):
            k2s = [lib.pair_info(q * nk1 + i1, with_layout=False)[1] for q in range(self.nk)]
            rows = V2_rows(int(k1), k2s)
            if self.mode == IBZ_BLOCK and vmax is None:
                vmax = max(np.abs(rows).max(), 1e-300)
            for q in range(self.nk):
                p = q * nk1 + i1
                if self.mode == IBZ_BLOCK:
                    trip[p], per_pair[p] = self.setup.block_V2(rows[q], int(k1), int(k2s[q]), self.ao, self.aux,
                                                                thresh=thresh, vmax=vmax)
                else:
                    per_pair[p] = np.ascontiguousarray(rows[q]).ravel()
        if self.mode == IBZ_BLOCK:
            tptr = np.zeros(self.npairs + 1, np.int64)
            tptr[1:] = np.cumsum([len(t) for t in trip])
            lib.set_triples(tptr, np.concatenate(trip) if tptr[-1] else np.zeros((0, 3), np.int32))
            self.triple_ptr, self.triples = tptr, trip
        V = np.concatenate(per_pair)
        assert lib.buffer_sizes()[3] == V.size
        return np.ascontiguousarray(V, np.complex128)

    # ---- output ---------------------------------------------------------------------------------
    def unpack_sigma(self, sigma_flat: np.ndarray):
        """flat Sigma buffer -> list over out_list of [ntau, nao, nao] matrices in the basis of the mode
        (orbital basis, or block basis with zeros off the diagonal blocks)."""
        out = []
        if self.mode != IBZ_BLOCK:
            S = sigma_flat.reshape(len(self.out_list), self.ntau, self.nao, self.nao)
            return [S[i] for i in range(len(self.out_list))]
        o = 0
        for k in self.out_list:
            ss = self.ao.sumsq(k)
            out.append(SymSetup.unpack_diag_blocks(sigma_flat[o:o + self.ntau * ss].reshape(self.ntau, ss), self.ao.off[k]))
            o += self.ntau * ss
        return out


def configure_from_crystal(lib: Gwsig, cr, mode: int, seed: int = 7, out_points=None, scramble_gauge=None, pass_U=False) -> Configured:
    """convenience for the synthetic crystals of gwsig_synth (any object with the same fields)."""
    sg = cr.sg
    return Configured(lib, mode, cr.a, cr.mesh, cr.nao, cr.naux, cr.ntau, cr.beta, cr.pos, cr.ao_atom, cr.aux_atom,
                      W=sg.W, w=sg.w, shift=sg.shift, P_ao=cr.P_ao, P_aux=cr.P_aux, seed=seed, out_points=out_points,
                      scramble_gauge=scramble_gauge, pass_U=pass_U)
