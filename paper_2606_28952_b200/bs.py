"""Thin ctypes binding of libbs.so (include/bs.h): argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch is used here only for device memory
(complex128 tensors owned by the caller) and for the current CUDA stream.  There is no CPU
fallback: if libbs.so is missing or was not built, importing this module raises.
Function names mirror the C ABI one to one (bs_group_xmask, bs_sector_build, bs_apply, ...).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbs.so")

BS_OK = 0
BS_ERR_ARG, BS_ERR_ALLOC, BS_ERR_CUDA, BS_ERR_MISMATCH = -1, -2, -3, -4
BS_ERR_NOT_COMMUTING, BS_ERR_LEAVES_SECTOR = -5, -6
BS_MODE_CANONICAL, BS_MODE_SEQUENCE = 0, 1

# every symbol include/bs.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "bs_group_xmask", "bs_op_info", "bs_op_export", "bs_op_destroy",
    "bs_sector_build", "bs_sector_info", "bs_sector_export", "bs_sector_rank", "bs_sector_destroy",
    "bs_apply", "bs_apply_rows", "bs_apply_axpby", "bs_expect", "bs_vdot",
    "bs_apply_pauli_rotations", "bs_taylor_step", "bs_plan_describe", "bs_plan_info", "bs_plan_groups",
    "bs_symsector_build", "bs_symsector_info", "bs_symsector_destroy", "bs_sym_scatter", "bs_sym_gather", "bs_sym_apply",
    "bs_sym_expect", "bs_noalloc_setup", "bs_noalloc_max_dim", "bs_vdot_noalloc", "bs_jw_molecular", "bs_jw_hubbard", "bs_launch_count", "bs_last_error", "bs_version",
]


class BsError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libbs status {status}: {msg}")
        self.status = status


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_28952_b200.build` "
            "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
    L.bs_group_xmask.argtypes = [vp, vp, vp, i64, C.c_int, dbl, C.c_int, vp, i64, vp, C.POINTER(vp)]
    L.bs_op_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(C.c_int)]
    L.bs_op_export.argtypes = [vp] * 6
    L.bs_op_destroy.argtypes = [vp]
    L.bs_sector_build.argtypes = [C.c_int, C.c_int, C.c_int, vp, C.POINTER(vp)]
    L.bs_sector_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
    L.bs_sector_export.argtypes = [vp, vp, vp]
    L.bs_sector_rank.argtypes = [vp, vp, i64, vp]
    L.bs_sector_destroy.argtypes = [vp]
    L.bs_apply.argtypes = [vp, vp, vp, vp, vp]
    L.bs_apply_rows.argtypes = [vp, vp, vp, vp, i64, i64, vp]
    L.bs_apply_axpby.argtypes = [vp, vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), vp, vp]
    L.bs_expect.argtypes = [vp, vp, vp, C.POINTER(dbl), vp]
    L.bs_vdot.argtypes = [vp, vp, vp, C.POINTER(dbl), vp]
    L.bs_apply_pauli_rotations.argtypes = [vp, vp, vp, i64, vp, vp]
    L.bs_taylor_step.argtypes = [vp, vp, vp, vp, dbl, C.c_int, dbl, vp]
    L.bs_jw_molecular.argtypes = [C.c_int, vp, vp, dbl, vp, C.POINTER(vp)]
    L.bs_jw_hubbard.argtypes = [C.c_int, dbl, dbl, dbl, vp, C.POINTER(vp)]
    L.bs_plan_describe.argtypes = [vp, vp, C.c_char_p, i64, vp]
    L.bs_symsector_build.argtypes = [vp, vp, C.c_int, vp, C.POINTER(vp)]
    L.bs_symsector_info.argtypes = [vp, C.POINTER(i64), vp, vp]
    L.bs_symsector_destroy.argtypes = [vp]
    L.bs_sym_scatter.argtypes = [vp, vp, vp, vp]
    L.bs_sym_gather.argtypes = [vp, vp, vp, vp]
    L.bs_sym_apply.argtypes = [vp, vp, vp, vp, vp]
    L.bs_sym_expect.argtypes = [vp, vp, vp, C.POINTER(dbl), vp]
    L.bs_noalloc_setup.argtypes = []
    L.bs_noalloc_max_dim.restype = i64
    L.bs_vdot_noalloc.argtypes = [vp, vp, i64, vp, vp]
    L.bs_plan_info.argtypes = [vp, vp, C.POINTER(i64), vp]
    L.bs_plan_groups.argtypes = [vp, vp, vp, vp, i64, C.POINTER(i64), vp]
    L.bs_launch_count.restype = i64
    L.bs_last_error.restype = C.c_char_p
    L.bs_version.restype = C.c_char_p
    return L


_lib = _load()


def _check(rc: int):
    if rc != BS_OK:
        raise BsError(rc, _lib.bs_last_error().decode())


def _stream(stream=None):
    """cudaStream_t of `stream` (a torch.cuda.Stream) or of torch's current stream, as void*."""
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_ptr(t, dim: int, what: str):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.complex128 and t.is_contiguous()):
        raise TypeError(f"{what} must be a contiguous complex128 CUDA tensor")
    if t.numel() != dim:
        raise ValueError(f"{what} has {t.numel()} amplitudes, expected {dim}")
    return C.c_void_p(t.data_ptr())


def _np_ptr(a: np.ndarray):
    return C.c_void_p(a.ctypes.data)


def bs_version() -> str:
    return _lib.bs_version().decode()


def bs_launch_count() -> int:
    return int(_lib.bs_launch_count())


def bs_last_error() -> str:
    return _lib.bs_last_error().decode()


class Op:
    """bs_op_t handle: X-grouped Pauli sum resident on the device (a1 + a2)."""

    def __init__(self, handle):
        self._h = handle
        g, m, q = C.c_int64(), C.c_int64(), C.c_int()
        _check(_lib.bs_op_info(self._h, C.byref(g), C.byref(m), C.byref(q)))
        self.n_groups, self.n_terms, self.n_qubits = int(g.value), int(m.value), int(q.value)

    def export(self):
        """Host copies (xg, offs, z, c, w) of the device tables."""
        G, M = self.n_groups, self.n_terms
        xg = np.empty(G, np.uint64)
        offs = np.empty(G + 1, np.int64)
        z = np.empty(M, np.uint64)
        c = np.empty(M, np.complex128)
        w = np.empty(M, np.complex128)
        _check(_lib.bs_op_export(self._h, _np_ptr(xg), _np_ptr(offs), _np_ptr(z), _np_ptr(c), _np_ptr(w)))
        return xg, offs, z, c, w

    def destroy(self):
        if self._h:
            _lib.bs_op_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class Sector:
    """bs_sector_t handle: (N_alpha, N_beta) sector tables, or the full 2^n space (a3)."""

    def __init__(self, handle, n_orb, n_alpha, n_beta):
        self._h = handle
        self.n_orb, self.n_alpha, self.n_beta = n_orb, n_alpha, n_beta
        self.full = n_alpha < 0
        d, da, db = C.c_int64(), C.c_int64(), C.c_int64()
        _check(_lib.bs_sector_info(self._h, C.byref(d), C.byref(da), C.byref(db)))
        self.dim, self.dim_alpha, self.dim_beta = int(d.value), int(da.value), int(db.value)
        self.n_rows = self.dim if self.full else self.dim_alpha

    def export(self):
        a = np.empty(self.dim_alpha, np.uint64)
        b = np.empty(self.dim_beta, np.uint64)
        _check(_lib.bs_sector_export(self._h, _np_ptr(a), _np_ptr(b)))
        return a, b

    def rank(self, configs) -> np.ndarray:
        cfg = np.ascontiguousarray(configs, np.uint64)
        out = np.empty(len(cfg), np.int64)
        _check(_lib.bs_sector_rank(self._h, _np_ptr(cfg), len(cfg), _np_ptr(out)))
        return out

    def destroy(self):
        if self._h:
            _lib.bs_sector_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def bs_group_xmask(x, z, coeff, n_qubits: int, eps_drop: float = 1e-12, mode: int = BS_MODE_CANONICAL,
                   seq_offsets=None, stream=None) -> Op:
    """x, z: uint64[M]; coeff: complex128[M] true-Pauli coefficients (host arrays)."""
    x = np.ascontiguousarray(x, np.uint64)
    z = np.ascontiguousarray(z, np.uint64)
    c = np.ascontiguousarray(coeff, np.complex128)
    if not (len(x) == len(z) == len(c)):
        raise ValueError("x, z, coeff must have equal length")
    seq_p, n_seq = None, 0
    if seq_offsets is not None:
        seq = np.ascontiguousarray(seq_offsets, np.int64)
        seq_p, n_seq = _np_ptr(seq), len(seq) - 1
    h = C.c_void_p()
    _check(_lib.bs_group_xmask(_np_ptr(x), _np_ptr(z), _np_ptr(c), len(x), n_qubits, eps_drop, mode, seq_p,
                               n_seq, _stream(stream), C.byref(h)))
    return Op(h)


def bs_sector_build(n_orb: int, n_alpha: int = -1, n_beta: int = -1, stream=None) -> Sector:
    h = C.c_void_p()
    _check(_lib.bs_sector_build(n_orb, n_alpha, n_beta, _stream(stream), C.byref(h)))
    return Sector(h, n_orb, n_alpha, n_beta)


def bs_apply(op: Op, sector: Sector, psi_in, psi_out, stream=None):
    _check(_lib.bs_apply(op._h, sector._h, _dev_ptr(psi_in, sector.dim, "psi_in"),
                         _dev_ptr(psi_out, sector.dim, "psi_out"), _stream(stream)))
    return psi_out


def bs_apply_rows(op: Op, sector: Sector, psi_in, psi_out, row_lo: int, row_hi: int, stream=None):
    _check(_lib.bs_apply_rows(op._h, sector._h, _dev_ptr(psi_in, sector.dim, "psi_in"),
                              _dev_ptr(psi_out, sector.dim, "psi_out"), row_lo, row_hi, _stream(stream)))
    return psi_out


def bs_apply_axpby(op: Op, sector: Sector, psi_in, psi_out, alpha: complex, beta: complex, acc=None,
                   stream=None):
    a = (C.c_double * 2)(complex(alpha).real, complex(alpha).imag)
    b = (C.c_double * 2)(complex(beta).real, complex(beta).imag)
    acc_p = None if acc is None else _dev_ptr(acc, sector.dim, "acc")
    _check(_lib.bs_apply_axpby(op._h, sector._h, _dev_ptr(psi_in, sector.dim, "psi_in"),
                               _dev_ptr(psi_out, sector.dim, "psi_out"), a, b, acc_p, _stream(stream)))
    return psi_out


def bs_expect(op: Op, sector: Sector, psi, stream=None) -> complex:
    r = (C.c_double * 2)()
    _check(_lib.bs_expect(op._h, sector._h, _dev_ptr(psi, sector.dim, "psi"), r, _stream(stream)))
    return complex(r[0], r[1])


def bs_vdot(sector: Sector, a, b, stream=None) -> complex:
    r = (C.c_double * 2)()
    _check(_lib.bs_vdot(sector._h, _dev_ptr(a, sector.dim, "a"), _dev_ptr(b, sector.dim, "b"), r,
                        _stream(stream)))
    return complex(r[0], r[1])


def bs_noalloc_setup():
    _check(_lib.bs_noalloc_setup())


def bs_noalloc_max_dim() -> int:
    return int(_lib.bs_noalloc_max_dim())


def bs_vdot_noalloc(a, b, result, stream=None):
    """result (complex128 CUDA tensor of one element) <- <a|b>; allocates nothing, does not synchronise."""
    n = a.numel()
    _check(_lib.bs_vdot_noalloc(_dev_ptr(a, n, "a"), _dev_ptr(b, n, "b"), n, _dev_ptr(result, 1, "result"),
                                _stream(stream)))
    return result


def bs_apply_pauli_rotations(generators: Op, sector: Sector, thetas, psi, stream=None):
    th = np.ascontiguousarray(thetas, np.float64)
    _check(_lib.bs_apply_pauli_rotations(generators._h, sector._h, _np_ptr(th), len(th),
                                         _dev_ptr(psi, sector.dim, "psi"), _stream(stream)))
    return psi


def bs_taylor_step(op: Op, sector: Sector, psi, work, dt: float, order: int = 12, e_shift: float = 0.0,
                   stream=None):
    _check(_lib.bs_taylor_step(op._h, sector._h, _dev_ptr(psi, sector.dim, "psi"),
                               _dev_ptr(work, 2 * sector.dim, "work"), dt, order, e_shift, _stream(stream)))
    return psi


def bs_plan_describe(op: Op, sector: Sector, stream=None) -> str:
    buf = C.create_string_buffer(2048)
    _check(_lib.bs_plan_describe(op._h, sector._h, buf, 2048, _stream(stream)))
    return buf.value.decode()


class SymSector:
    """bs_symsector_t handle: one point-group block of a sector (Eq. 29-31)."""

    def __init__(self, sector: "Sector", orb_irrep, target_irrep: int, stream=None):
        lab = np.ascontiguousarray(orb_irrep, np.int32)
        if lab.shape != (sector.n_orb,):
            raise ValueError("orb_irrep must have one label per spatial orbital")
        h = C.c_void_p()
        _check(_lib.bs_symsector_build(sector._h, _np_ptr(lab), int(target_irrep), _stream(stream), C.byref(h)))
        self._h, self.parent = h, sector
        d = C.c_int64()
        da, db = np.zeros(8, np.int64), np.zeros(8, np.int64)
        _check(_lib.bs_symsector_info(self._h, C.byref(d), _np_ptr(da), _np_ptr(db)))
        self.dim, self.dim_alpha, self.dim_beta = int(d.value), da, db

    def __del__(self):
        if getattr(self, "_h", None):
            _lib.bs_symsector_destroy(self._h)
            self._h = None


def bs_symsector_build(sector, orb_irrep, target_irrep: int, stream=None) -> SymSector:
    return SymSector(sector, orb_irrep, target_irrep, stream)


def bs_sym_scatter(sym: SymSector, psi_blocked, psi_sector, stream=None):
    _check(_lib.bs_sym_scatter(sym._h, _dev_ptr(psi_blocked, sym.dim, "psi_blocked"),
                               _dev_ptr(psi_sector, sym.parent.dim, "psi_sector"), _stream(stream)))
    return psi_sector


def bs_sym_gather(sym: SymSector, psi_sector, psi_blocked, stream=None):
    _check(_lib.bs_sym_gather(sym._h, _dev_ptr(psi_sector, sym.parent.dim, "psi_sector"),
                              _dev_ptr(psi_blocked, sym.dim, "psi_blocked"), _stream(stream)))
    return psi_blocked


def bs_sym_apply(op: Op, sym: SymSector, psi_in, psi_out, stream=None):
    _check(_lib.bs_sym_apply(op._h, sym._h, _dev_ptr(psi_in, sym.dim, "psi_in"), _dev_ptr(psi_out, sym.dim, "psi_out"),
                             _stream(stream)))
    return psi_out


def bs_sym_expect(op: Op, sym: SymSector, psi, stream=None) -> complex:
    res = (C.c_double * 2)()
    _check(_lib.bs_sym_expect(op._h, sym._h, _dev_ptr(psi, sym.dim, "psi"), res, _stream(stream)))
    return complex(res[0], res[1])


PLAN_INFO_FIELDS = ("kernel_path", "fallback", "transposed", "kres", "vector_scratch_bytes", "kres_scratch_bytes",
                    "max_keys", "groups")


def bs_plan_info(op: Op, sector: Sector, stream=None) -> dict:
    """bs_plan_info as a dict (field names: PLAN_INFO_FIELDS)."""
    info = (C.c_int64 * 8)()
    _check(_lib.bs_plan_info(op._h, sector._h, info, _stream(stream)))
    return dict(zip(PLAN_INFO_FIELDS, (int(v) for v in info)))


def bs_plan_groups(op: Op, sector: Sector, stream=None):
    """(x masks u64[G], key counts i32[G]) of the plan's groups (bs_plan_groups)."""
    n = C.c_int64()
    _check(_lib.bs_plan_groups(op._h, sector._h, None, None, 0, C.byref(n), _stream(stream)))
    x = np.empty(n.value, np.uint64)
    nk = np.empty(n.value, np.int32)
    _check(_lib.bs_plan_groups(op._h, sector._h, _np_ptr(x), _np_ptr(nk), n.value, C.byref(n), _stream(stream)))
    return x, nk


def bs_jw_molecular(h, g, eps_drop: float = 1e-12, stream=None) -> Op:
    """Device-side JW construction + canonical reduction of a molecular Hamiltonian (chemist-notation g)."""
    h = np.ascontiguousarray(h, np.float64)
    g = np.ascontiguousarray(g, np.float64)
    n = h.shape[0]
    if h.shape != (n, n) or g.shape != (n, n, n, n):
        raise ValueError("h must be [n, n] and g [n, n, n, n]")
    out = C.c_void_p()
    _check(_lib.bs_jw_molecular(n, _np_ptr(h), _np_ptr(g), eps_drop, _stream(stream), C.byref(out)))
    return Op(out)


def bs_jw_hubbard(n_sites: int, t: float, U: float, eps_drop: float = 1e-12, stream=None) -> Op:
    out = C.c_void_p()
    _check(_lib.bs_jw_hubbard(n_sites, t, U, eps_drop, _stream(stream), C.byref(out)))
    return Op(out)
