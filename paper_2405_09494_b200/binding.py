"""Thin ctypes binding of libgwsig.so (include/gwsig.h).  Argument marshalling only:
every step of the hot path runs in the library's CUDA kernels.  Importing this module
fails loudly if the library has not been built (python -m paper_2405_09494_b200.build).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgwsig.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2405_09494_b200.build` "
                      "(there is no fallback implementation)")
_lib = C.CDLL(LIB_PATH)

FULL_BZ, IBZ, IBZ_BLOCK = 0, 1, 2
ENGINE_DMMA, ENGINE_REFERENCE, ENGINE_DMMA_4M, ENGINE_DMMA_3M = 0, 1, 2, 3
NODIV = 0x7FFFFFFF
FLAG_CONJ_A, FLAG_ACCUM, FLAG_A_KMAJOR, FLAG_CONJ_B = 1, 2, 4, 8

IDX2 = np.dtype([("hi", "<i8"), ("lo", "<i8"), ("div", "<i4"), ("pad_", "<i4")])
SEG = np.dtype([("a_off", "<i8"), ("b_off", "<i8"), ("am", IDX2), ("ak", IDX2), ("bk", IDX2), ("bn", IDX2),
                ("K", "<i4"), ("pad_", "<i4")])
PROBLEM = np.dtype([("c_off", "<i8"), ("a_bstride", "<i8"), ("b_bstride", "<i8"), ("c_bstride", "<i8"),
                    ("a_tstride", "<i8"), ("b_tstride", "<i8"), ("c_tstride", "<i8"), ("tile_begin", "<i8"),
                    ("cm", IDX2), ("cn", IDX2), ("M", "<i4"), ("N", "<i4"), ("seg_begin", "<i4"), ("seg_count", "<i4"),
                    ("nbatch", "<i4"), ("flags", "<i4"), ("tiles_m", "<i4"), ("tiles_n", "<i4")])
assert IDX2.itemsize == 24 and SEG.itemsize == 120 and PROBLEM.itemsize == 144

EXPORTS = ["gwsig_create", "gwsig_destroy", "gwsig_last_error", "gwsig_set_lattice", "gwsig_set_atoms",
           "gwsig_set_symmetry", "gwsig_set_blocks", "gwsig_set_triples", "gwsig_get_ibz", "gwsig_pair_count",
           "gwsig_pair_info", "gwsig_buffer_sizes", "gwsig_sigma_begin", "gwsig_sigma_push_pairs", "gwsig_sigma_end",
           "gwsig_sigma_eval", "gwsig_set_option", "gwsig_flop_counts", "gwsig_last_launch_count", "gwsig_plan_counts",
           "gwsig_plan_get", "gwsig_probe_fp64", "gwsig_kernel_times", "gwsig_sigma_abort", "gwsig_sigma_eval_host",
           "gwsig_set_output_points", "gwsig_exchange_begin", "gwsig_exchange_eval",
           "gwsig_p0_begin", "gwsig_p0_push_pairs", "gwsig_p0_end", "gwsig_p0_eval", "gwsig_block_transform_v", "gwsig_dyson_p",
           "gwsig_dyson_solve_noalloc", "gwsig_hartree_eval", "gwsig_block_maxabs"]

_vp, _i, _i64, _d = C.c_void_p, C.c_int, C.c_int64, C.c_double
_sig = {
    "gwsig_create": [C.POINTER(_vp), _i], "gwsig_destroy": [_vp],
    "gwsig_set_lattice": [_vp, _vp, _vp, _i, _i, _i, _d], "gwsig_set_atoms": [_vp, _i, _vp, _vp, _vp],
    "gwsig_set_symmetry": [_vp, _i, _vp, _vp, _vp, _vp, _vp, _i], "gwsig_set_blocks": [_vp, _vp, _vp, _vp, _vp, _vp, _vp],
    "gwsig_set_triples": [_vp, _i64, _vp, _vp], "gwsig_set_output_points": [_vp, _i, _vp], "gwsig_get_ibz": [_vp, _vp, _vp, _vp, _vp],
    "gwsig_pair_count": [_vp, _vp, _vp], "gwsig_pair_info": [_vp, _i64, _vp, _vp, _vp, _vp, _vp],
    "gwsig_buffer_sizes": [_vp, _vp, _vp, _vp, _vp], "gwsig_sigma_begin": [_vp, _vp, _vp, _vp, _vp],
    "gwsig_sigma_push_pairs": [_vp, _i64, _i64, _vp], "gwsig_sigma_end": [_vp],
    "gwsig_sigma_eval": [_vp, _vp, _vp, _vp, _vp, _vp], "gwsig_set_option": [_vp, C.c_char_p, _i64],
    "gwsig_flop_counts": [_vp, _vp, _vp], "gwsig_last_launch_count": [_vp, _vp],
    "gwsig_plan_counts": [_vp, _i64, _i64, _i, _i, _vp, _vp, _vp], "gwsig_plan_get": [_vp, _i64, _i64, _i, _i, _vp, _vp],
    "gwsig_probe_fp64": [_vp, _i, _i, _i, _i64, _vp, _vp], "gwsig_kernel_times": [_vp, _vp, _vp],
    "gwsig_sigma_abort": [_vp], "gwsig_sigma_eval_host": [_vp, _vp, _vp, _vp, _vp, _vp],
    "gwsig_exchange_begin": [_vp, _vp, _vp, _vp], "gwsig_exchange_eval": [_vp, _vp, _vp, _vp, _vp],
    "gwsig_p0_begin": [_vp, _vp, _vp, _vp], "gwsig_p0_push_pairs": [_vp, _i64, _i64, _vp], "gwsig_p0_end": [_vp],
    "gwsig_p0_eval": [_vp, _vp, _vp, _vp, _vp], "gwsig_block_transform_v": [_vp, _i64, _i64, _vp, _vp, _vp],
    "gwsig_dyson_p": [_vp, _vp, _vp, _vp, _i, _vp, _vp],
    "gwsig_dyson_solve_noalloc": [_vp, _vp, _i, _i, _vp, _vp, C.c_char_p, _i],
    "gwsig_hartree_eval": [_vp, _vp, _vp, _vp, _vp],
    "gwsig_block_maxabs": [_vp, _i64, _i64, _vp, _i, _i, _vp, _vp],
}
for _name, _args in _sig.items():
    getattr(_lib, _name).argtypes = _args
    getattr(_lib, _name).restype = _i
_lib.gwsig_last_error.argtypes = [_vp]
_lib.gwsig_last_error.restype = C.c_char_p


class GwsigError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"gwsig error {code}: {msg}")
        self.code = code


def _ptr(x):
    """device / host pointer of a torch tensor, numpy array, int or None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()          # torch tensor


def _np(x, dtype):
    return np.ascontiguousarray(x, dtype=dtype)


NOALLOC_NMAX, NOALLOC_SCRATCH_BYTES = 256, 16 << 20


def dyson_solve_noalloc(dA, dX, nmat, n, d_info=None, stream=0):
    """gwsig_dyson_solve_noalloc: X_m = [1 - A_m]^{-1} A_m (Eq. 19a) with the library's fixed device scratch; takes no
    context, allocates nothing, does not synchronise.  dA / dX: device complex128 [nmat][n][n]; d_info: device int32 or None."""
    err = C.create_string_buffer(256)
    rc = _lib.gwsig_dyson_solve_noalloc(_ptr(dA), _ptr(dX), int(nmat), int(n), _ptr(d_info), stream or None, err, len(err))
    if rc:
        raise GwsigError(rc, err.value.decode())


class Gwsig:
    """one gwsig context.  device < 0 gives a host-only context (plan calls work, sigma_* fail)."""

    def __init__(self, device: int = 0):
        self._h = _vp()
        rc = _lib.gwsig_create(C.byref(self._h), device)
        if rc:
            raise GwsigError(rc, "gwsig_create failed")

    def close(self):
        if self._h:
            _lib.gwsig_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc:
            raise GwsigError(rc, _lib.gwsig_last_error(self._h).decode())

    # ---- problem statement -----------------------------------------------------------------
    def set_lattice(self, a, mesh, nao, naux, ntau, beta):
        a, mesh = _np(a, np.float64), _np(mesh, np.int32)
        self._ck(_lib.gwsig_set_lattice(self._h, a.ctypes.data, mesh.ctypes.data, nao, naux, ntau, float(beta)))
        self.nao, self.naux, self.ntau, self.nk = nao, naux, ntau, int(np.prod(mesh))

    def set_atoms(self, pos, ao_atom, aux_atom):
        pos, ao, ax = _np(pos, np.float64), _np(ao_atom, np.int32), _np(aux_atom, np.int32)
        self._ck(_lib.gwsig_set_atoms(self._h, len(pos), pos.ctypes.data, ao.ctypes.data, ax.ctypes.data))

    def set_symmetry(self, rot, trans, D_ao, D_aux, shift, mode):
        if rot is None or len(rot) == 0:
            self._ck(_lib.gwsig_set_symmetry(self._h, 0, None, None, None, None, None, mode))
            return
        rot, trans = _np(rot, np.int32), _np(trans, np.float64)
        D_ao, D_aux, shift = _np(D_ao, np.float64), _np(D_aux, np.float64), _np(shift, np.int32)
        self._ck(_lib.gwsig_set_symmetry(self._h, len(rot), rot.ctypes.data, trans.ctypes.data, D_ao.ctypes.data,
                                         D_aux.ctypes.data, shift.ctypes.data, mode))

    def set_blocks(self, ao_off, aux_off, U_ao=None, U_aux=None):
        """ao_off / aux_off: per mesh point, the nblk+1 block offsets."""
        nb_ao = _np([len(o) - 1 for o in ao_off], np.int32)
        nb_ax = _np([len(o) - 1 for o in aux_off], np.int32)
        cat_ao = _np(np.concatenate([np.asarray(o) for o in ao_off]), np.int32)
        cat_ax = _np(np.concatenate([np.asarray(o) for o in aux_off]), np.int32)
        ua = None if U_ao is None else _np(U_ao, np.complex128)
        ux = None if U_aux is None else _np(U_aux, np.complex128)
        self._ck(_lib.gwsig_set_blocks(self._h, nb_ao.ctypes.data, cat_ao.ctypes.data, nb_ax.ctypes.data, cat_ax.ctypes.data,
                                       _ptr(ua), _ptr(ux)))

    def set_output_points(self, k_list):
        k = _np(k_list, np.int32)
        self._ck(_lib.gwsig_set_output_points(self._h, len(k), _ptr(k)))

    def set_triples(self, triple_ptr, triples):
        tp = _np(triple_ptr, np.int64)
        tr = _np(np.asarray(triples).reshape(-1, 3), np.int32)
        self._ck(_lib.gwsig_set_triples(self._h, len(tp) - 1, tp.ctypes.data, tr.ctypes.data))

    # ---- plan outputs ------------------------------------------------------------------------
    def get_ibz(self):
        nik = C.c_int()
        self._ck(_lib.gwsig_get_ibz(self._h, C.addressof(nik), None, None, None))
        ir_list = np.zeros(nik.value, np.int32)
        ir_of, op_of = np.zeros(self.nk, np.int32), np.zeros(self.nk, np.int32)
        self._ck(_lib.gwsig_get_ibz(self._h, None, ir_list.ctypes.data, ir_of.ctypes.data, op_of.ctypes.data))
        return ir_list, ir_of, op_of

    def pair_count(self):
        n, k = C.c_int64(), C.c_int()
        self._ck(_lib.gwsig_pair_count(self._h, C.addressof(n), C.addressof(k)))
        return n.value, k.value

    def pair_info(self, pair, with_layout=True):
        k1, k2, q = C.c_int(), C.c_int(), C.c_int()
        off, ne = C.c_int64(), C.c_int64()
        self._ck(_lib.gwsig_pair_info(self._h, pair, C.addressof(k1), C.addressof(k2), C.addressof(q),
                                      C.addressof(off) if with_layout else None, C.addressof(ne) if with_layout else None))
        return k1.value, k2.value, q.value, off.value, ne.value

    def buffer_sizes(self):
        v = [C.c_int64() for _ in range(4)]
        self._ck(_lib.gwsig_buffer_sizes(self._h, *[C.addressof(x) for x in v]))
        return tuple(x.value for x in v)       # g, w, sigma, v  (complex elements)

    def flop_counts(self):
        f, e = C.c_double(), C.c_double()
        self._ck(_lib.gwsig_flop_counts(self._h, C.addressof(f), C.addressof(e)))
        return f.value, e.value

    def last_launch_count(self):
        n = C.c_int64()
        self._ck(_lib.gwsig_last_launch_count(self._h, C.addressof(n)))
        return n.value

    KINDS = ("unfold_G", "unfold_W", "stage1_X=VG", "stage2_Y=WX", "stage3_S+=YV", "epilogue", "vtransform", "grid_transform", "dyson_solve", "hartree")

    def kernel_times(self):
        ms = np.zeros(len(self.KINDS), np.float64)
        n = np.zeros(len(self.KINDS), np.int64)
        self._ck(_lib.gwsig_kernel_times(self._h, ms.ctypes.data, n.ctypes.data))
        return {k: (float(m), int(c)) for k, m, c in zip(self.KINDS, ms, n)}

    def set_option(self, key, value):
        self._ck(_lib.gwsig_set_option(self._h, key.encode(), int(value)))

    def plan_get(self, p0, np_, nt, stage):
        npb, nsg, ntl = C.c_int64(), C.c_int64(), C.c_int64()
        self._ck(_lib.gwsig_plan_counts(self._h, p0, np_, nt, stage, C.addressof(npb), C.addressof(nsg), C.addressof(ntl)))
        prob = np.zeros(max(npb.value, 1), PROBLEM)
        seg = np.zeros(max(nsg.value, 1), SEG)
        self._ck(_lib.gwsig_plan_get(self._h, p0, np_, nt, stage, prob.ctypes.data, seg.ctypes.data))
        return prob[:npb.value], seg[:nsg.value], ntl.value

    # ---- evaluation (device pointers: torch tensors or raw ints) ------------------------------------
    def sigma_begin(self, dG, dW, dSigma, stream=0):
        self._ck(_lib.gwsig_sigma_begin(self._h, _ptr(dG), _ptr(dW), _ptr(dSigma), stream or None))

    def sigma_push_pairs(self, p0, np_, dV):
        self._ck(_lib.gwsig_sigma_push_pairs(self._h, p0, np_, _ptr(dV)))

    def sigma_end(self):
        self._ck(_lib.gwsig_sigma_end(self._h))

    def sigma_eval(self, dG, dV, dW, dSigma, stream=0):
        self._ck(_lib.gwsig_sigma_eval(self._h, _ptr(dG), _ptr(dV), _ptr(dW), _ptr(dSigma), stream or None))

    def exchange_begin(self, dGamma, dK, stream=0):
        self._ck(_lib.gwsig_exchange_begin(self._h, _ptr(dGamma), _ptr(dK), stream or None))

    def exchange_eval(self, dGamma, dV, dK, stream=0):
        self._ck(_lib.gwsig_exchange_eval(self._h, _ptr(dGamma), _ptr(dV), _ptr(dK), stream or None))

    def block_transform_v(self, p0, np_, dV_dense, dV_packed, stream=0):
        self._ck(_lib.gwsig_block_transform_v(self._h, p0, np_, _ptr(dV_dense), _ptr(dV_packed), stream or None))

    def block_maxabs(self, p0, np_, dV_dense, mb_aux, mb_ao, d_maxabs, stream=0):
        self._ck(_lib.gwsig_block_maxabs(self._h, int(p0), int(np_), _ptr(dV_dense), int(mb_aux), int(mb_ao), _ptr(d_maxabs), stream or None))

    def hartree_eval(self, dGamma, dVdiag, dJ, stream=0):
        self._ck(_lib.gwsig_hartree_eval(self._h, _ptr(dGamma), _ptr(dVdiag), _ptr(dJ), stream or None))

    def dyson_p(self, dP0, dTf, dTb, nw, dP, stream=0):
        self._ck(_lib.gwsig_dyson_p(self._h, _ptr(dP0), _ptr(dTf), _ptr(dTb), int(nw), _ptr(dP), stream or None))

    def p0_begin(self, dG, dP0, stream=0):
        self._ck(_lib.gwsig_p0_begin(self._h, _ptr(dG), _ptr(dP0), stream or None))

    def p0_push_pairs(self, p0, np_, dV):
        self._ck(_lib.gwsig_p0_push_pairs(self._h, p0, np_, _ptr(dV)))

    def p0_end(self):
        self._ck(_lib.gwsig_p0_end(self._h))

    def p0_eval(self, dG, dV, dP0, stream=0):
        self._ck(_lib.gwsig_p0_eval(self._h, _ptr(dG), _ptr(dV), _ptr(dP0), stream or None))

    def sigma_abort(self):
        self._ck(_lib.gwsig_sigma_abort(self._h))

    def sigma_eval_host(self, hG, hV, hW, hSigma, stream=0):
        """host buffers (numpy arrays or pinned CPU torch tensors); blocks until hSigma holds the result."""
        self._ck(_lib.gwsig_sigma_eval_host(self._h, _ptr(hG), _ptr(hV), _ptr(hW), _ptr(hSigma), stream or None))

    def probe_fp64(self, kind, warps_per_block=8, blocks_per_sm=2, iters=20000):
        t, ms = C.c_double(), C.c_double()
        self._ck(_lib.gwsig_probe_fp64(self._h, kind, warps_per_block, blocks_per_sm, iters, C.addressof(t), C.addressof(ms)))
        return t.value, ms.value
