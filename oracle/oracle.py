"""ctypes wrapper of the CPU oracle (oracle/bs_oracle.cpp) -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the product package and the product never imports it.
Argument marshalling only; all arithmetic is in bs_oracle.cpp.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# BS_ORACLE_SO: use an oracle library built elsewhere from the same source (e.g. with -O3 -march=native for the
# hours-long golden run of tests/golden/make_fullsize_golden.py); default: the portable in-tree -O2 build.
_SO = os.environ.get("BS_ORACLE_SO") or os.path.join(_HERE, "libbs_oracle.so")
_SRC = os.path.join(_HERE, "bs_oracle.cpp")
_lib = None

_u64p = np.ctypeslib.ndpointer(np.uint64, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(np.int64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (plain C++17 + OpenMP).  Building is not using."""
    if os.environ.get("BS_ORACLE_SO"):
        return _SO
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC]
        subprocess.check_call(cmd)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.orc_num_threads.restype = C.c_int
        L.orc_op_size.restype = C.c_int64
        L.orc_op_size.argtypes = [C.c_void_p]
        L.orc_op_free.argtypes = [C.c_void_p]
        L.orc_op_export.argtypes = [C.c_void_p, _u64p, _u64p, _f64p]
        L.orc_pauli_mul.argtypes = [C.c_uint64, C.c_uint64, _f64p, C.c_uint64, C.c_uint64, _f64p,
                                    C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), _f64p]
        L.orc_ladder_product.restype = C.c_void_p
        L.orc_ladder_product.argtypes = [_i32p, _i32p, C.c_int, _f64p, C.c_double]
        L.orc_excitation_generator.restype = C.c_void_p
        L.orc_excitation_generator.argtypes = [_i32p, C.c_int, _i32p, C.c_int, C.c_double]
        L.orc_molecular_h.restype = C.c_void_p
        L.orc_molecular_h.argtypes = [C.c_int, _f64p, _f64p, C.c_double]
        L.orc_hubbard_h.restype = C.c_void_p
        L.orc_hubbard_h.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double]
        L.orc_sector_new.restype = C.c_void_p
        L.orc_sector_new.argtypes = [C.c_int, C.c_int, C.c_int]
        L.orc_sector_free.argtypes = [C.c_void_p]
        L.orc_sector_dims.argtypes = [C.c_void_p] + [C.POINTER(C.c_int64)] * 3
        L.orc_sector_strings.argtypes = [C.c_void_p, _u64p, _u64p]
        L.orc_sector_index.argtypes = [C.c_void_p, _u64p, C.c_int64, _i64p]
        L.orc_apply_terms.argtypes = [C.c_void_p, _u64p, _u64p, _f64p, C.c_int64, _f64p, _f64p]
        L.orc_apply_sampled.argtypes = [C.c_void_p, _u64p, _u64p, _f64p, C.c_int64, _f64p, _i64p,
                                        C.c_int64, _f64p]
        L.orc_apply_grouped.argtypes = [C.c_void_p, _u64p, _u64p, _f64p, C.c_int64, _f64p, _f64p,
                                        C.c_int64, C.c_int64]
        L.orc_apply_grouped_slab.argtypes = [C.c_void_p, _u64p, _u64p, _f64p, C.c_int64, _f64p, _f64p,
                                             C.c_int64, C.c_int64]
        L.orc_vdot.argtypes = [_f64p, _f64p, C.c_int64, _f64p]
        L.orc_rot_fermionic.argtypes = [C.c_void_p, _i32p, C.c_int, _i32p, C.c_int, C.c_double, _f64p]
        L.orc_taylor_step.argtypes = [C.c_void_p, _u64p, _u64p, _f64p, C.c_int64, C.c_double,
                                      C.c_int, C.c_double, _f64p]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _reim(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a.view(np.float64)


class PauliOp:
    """Canonical Pauli sum: x, z (uint64) and true-Pauli coefficients c (complex128), sorted by (x, z)."""

    def __init__(self, x, z, c):
        self.x = np.ascontiguousarray(x, dtype=np.uint64)
        self.z = np.ascontiguousarray(z, dtype=np.uint64)
        self.c = np.ascontiguousarray(c, dtype=np.complex128)

    def __len__(self):
        return len(self.x)

    @property
    def n_groups(self) -> int:
        return int(len(np.unique(self.x)))


def _take(handle) -> PauliOp:
    L = lib()
    M = L.orc_op_size(handle)
    x = np.empty(M, np.uint64)
    z = np.empty(M, np.uint64)
    c = np.empty(M, np.complex128)
    L.orc_op_export(handle, x, z, c.view(np.float64))
    L.orc_op_free(handle)
    return PauliOp(x, z, c)


def pauli_mul(x1, z1, c1, x2, z2, c2):
    """(X,Z,C) product in XZ-ordered form, Eq. 19-21."""
    xo, zo = C.c_uint64(), C.c_uint64()
    co = np.zeros(2)
    lib().orc_pauli_mul(x1, z1, _reim(np.array([c1])), x2, z2, _reim(np.array([c2])),
                        C.byref(xo), C.byref(zo), co)
    return xo.value, zo.value, complex(co[0], co[1])


def ladder_product(idx, dag, scale=1.0, eps_drop=0.0) -> PauliOp:
    idx = np.ascontiguousarray(idx, np.int32)
    dag = np.ascontiguousarray(dag, np.int32)
    sc = _reim(np.array([scale]))
    return _take(lib().orc_ladder_product(idx, dag, len(idx), sc, eps_drop))


def molecular_h(h, g, eps_drop=1e-12) -> PauliOp:
    n = h.shape[0]
    return _take(lib().orc_molecular_h(n, np.ascontiguousarray(h, np.float64),
                                       np.ascontiguousarray(g, np.float64).reshape(-1), eps_drop))


def hubbard_h(L_sites, t, U, eps_drop=1e-12) -> PauliOp:
    return _take(lib().orc_hubbard_h(L_sites, t, U, eps_drop))


def excitation_generator(cre, ann, eps_drop=1e-14) -> PauliOp:
    """T - T^dag as a Pauli sum, T = prod a^dag_cre prod a_ann (Eq. 39 tau_k)."""
    cre = np.ascontiguousarray(cre, np.int32)
    ann = np.ascontiguousarray(ann, np.int32)
    return _take(lib().orc_excitation_generator(cre, len(cre), ann, len(ann), eps_drop))


class Sector:
    """(N_alpha, N_beta) sector of n_orb spatial orbitals, or the full 2^n space (n_alpha=-1)."""

    def __init__(self, n, n_alpha=-1, n_beta=-1):
        self.n, self.n_alpha, self.n_beta = n, n_alpha, n_beta
        self._h = lib().orc_sector_new(n, n_alpha, n_beta)
        d = [C.c_int64() for _ in range(3)]
        lib().orc_sector_dims(self._h, *[C.byref(v) for v in d])
        self.dim, self.dim_alpha, self.dim_beta = (int(v.value) for v in d)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_sector_free(self._h)
            self._h = None

    def strings(self):
        a = np.empty(self.dim_alpha, np.uint64)
        b = np.empty(self.dim_beta, np.uint64)
        lib().orc_sector_strings(self._h, a, b)
        return a, b

    def index(self, cfgs):
        cfgs = np.ascontiguousarray(cfgs, np.uint64)
        out = np.empty(len(cfgs), np.int64)
        lib().orc_sector_index(self._h, cfgs, len(cfgs), out)
        return out

    def apply(self, op: PauliOp, psi):
        psi = np.ascontiguousarray(psi, np.complex128)
        out = np.empty_like(psi)
        lib().orc_apply_terms(self._h, op.x, op.z, _reim(op.c), len(op), _reim(psi), _reim(out))
        return out

    def apply_sampled(self, op: PauliOp, psi, targets):
        psi = np.ascontiguousarray(psi, np.complex128)
        targets = np.ascontiguousarray(targets, np.int64)
        out = np.empty(len(targets), np.complex128)
        lib().orc_apply_sampled(self._h, op.x, op.z, _reim(op.c), len(op), _reim(psi), targets,
                                len(targets), _reim(out))
        return out

    def apply_grouped(self, op: PauliOp, psi, row_lo=0, row_hi=None, out=None):
        psi = np.ascontiguousarray(psi, np.complex128)
        if out is None:
            out = np.zeros_like(psi)
        if row_hi is None:
            row_hi = self.dim if self.n_alpha < 0 else self.dim_alpha
        lib().orc_apply_grouped(self._h, op.x, op.z, _reim(op.c), len(op), _reim(psi), _reim(out),
                                row_lo, row_hi)
        return out

    def apply_grouped_slab(self, op: PauliOp, psi, row_lo, row_hi):
        """Rows [row_lo, row_hi) of H psi as a (row_hi - row_lo, dim_beta) array (beta search hoisted)."""
        psi = np.ascontiguousarray(psi, np.complex128)
        out = np.empty((row_hi - row_lo, self.dim_beta), np.complex128)
        lib().orc_apply_grouped_slab(self._h, op.x, op.z, _reim(op.c), len(op), _reim(psi), _reim(out),
                                     row_lo, row_hi)
        return out

    def rot_fermionic(self, psi, cre, ann, theta):
        """In place: psi <- exp(theta (T - T^dag)) psi."""
        assert psi.dtype == np.complex128 and psi.flags.c_contiguous
        lib().orc_rot_fermionic(self._h, np.ascontiguousarray(cre, np.int32), len(cre),
                                np.ascontiguousarray(ann, np.int32), len(ann), float(theta), _reim(psi))

    def taylor_step(self, op: PauliOp, psi, dt, order, e_shift):
        """In place: one shifted Taylor step of exp(-i H dt)."""
        assert psi.dtype == np.complex128 and psi.flags.c_contiguous
        lib().orc_taylor_step(self._h, op.x, op.z, _reim(op.c), len(op), dt, order, e_shift, _reim(psi))


def vdot(a, b) -> complex:
    a = np.ascontiguousarray(a, np.complex128)
    b = np.ascontiguousarray(b, np.complex128)
    res = np.zeros(2)
    lib().orc_vdot(_reim(a), _reim(b), len(a), res)
    return complex(res[0], res[1])


def energy(sector: Sector, op: PauliOp, psi) -> complex:
    """<psi|H|psi> (Eq. 5)."""
    return vdot(psi, sector.apply(op, psi))
