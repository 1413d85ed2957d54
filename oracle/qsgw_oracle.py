"""ctypes binding of oracle/qsgw_oracle.c (plain C FP64 loops) -- TEST INFRASTRUCTURE.

The arithmetic lives in qsgw_oracle.c (each function cites the passage of
/root/reference/PAPER.md it follows: Eqs. (17)-(19), in RI form).
This file only compiles that C file with gcc, marshals numpy arrays, and returns numpy
arrays.  It imports nothing from the CUDA product package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qsgw_oracle.c")
_LIB = os.path.join(_HERE, "libqsgw_oracle.so")
_lock = threading.Lock()
_lib = None


def build_library(force: bool = False) -> str:
    """Compile qsgw_oracle.c -> libqsgw_oracle.so with gcc (-O2 -fopenmp); returns the path."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build_library())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        i64 = ctypes.c_int64
        lib.qsgw_oracle_num_threads.restype = ctypes.c_int
        lib.qsgw_oracle_set_num_threads.restype = None
        lib.qsgw_oracle_set_num_threads.argtypes = [ctypes.c_int]
        lib.qsgw_oracle_D.restype = ctypes.c_double
        lib.qsgw_oracle_D.argtypes = [ctypes.c_double] * 5
        lib.qsgw_oracle_pole_weights.restype = None
        lib.qsgw_oracle_pole_weights.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64, dp, dp, i64, dp, i64]
        lib.qsgw_oracle_residues.restype = None
        lib.qsgw_oracle_residues.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp, i64, i64, ctypes.c_int, ip, dp]
        lib.qsgw_oracle_sigma.restype = ctypes.c_int
        lib.qsgw_oracle_sigma.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64, dp, dp, dp, dp, dp, i64,
                                          ctypes.c_double, ctypes.c_int, ip, dp]
        lib.qsgw_oracle_sigma_diag.restype = ctypes.c_int
        lib.qsgw_oracle_sigma_diag.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, i64, dp, dp, dp, dp, dp, i64,
                                               ctypes.c_double, ctypes.c_int, dp, ctypes.c_int, ip, dp, dp]
        lib.qsgw_oracle_mp2_direct.restype = ctypes.c_int
        lib.qsgw_oracle_mp2_direct.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, ctypes.c_double, dp]
        lib.qsgw_oracle_mp2.restype = ctypes.c_int
        lib.qsgw_oracle_mp2.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int, dp]
        lib.qsgw_oracle_mp2_states.restype = ctypes.c_int
        lib.qsgw_oracle_mp2_states.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp, ctypes.c_double, ctypes.c_int,
                                               ctypes.c_int, ip, dp]
        lib.qsgw_oracle_casida_matrix.restype = ctypes.c_int
        lib.qsgw_oracle_casida_matrix.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp]
        lib.qsgw_oracle_casida_z.restype = ctypes.c_int
        lib.qsgw_oracle_casida_z.argtypes = [ctypes.c_int, ctypes.c_int, dp, i64, dp, dp, i64, dp, dp, i64]
        lib.qsgw_oracle_ao_to_mo.restype = ctypes.c_int
        lib.qsgw_oracle_ao_to_mo.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp, dp]
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {tuple(shape)}, got {a.shape}")
    return a


def num_threads() -> int:
    """OpenMP threads the oracle will use (its `cores` figure when timed as the CPU baseline)."""
    return int(_load().qsgw_oracle_num_threads())


def set_num_threads(n: int) -> None:
    """Use n OpenMP threads from now on (bench.py's one-core figure)."""
    _load().qsgw_oracle_set_num_threads(int(n))


def D(occ_m: float, eps_m: float, Omega_s: float, omega: float, eta: float) -> float:
    """D(m,s,omega) of SURVEY 8(c): real part of the two terms of Eq. (17)."""
    return float(_load().qsgw_oracle_D(occ_m, eps_m, Omega_s, omega, eta))


def pole_weights(B, Z, n_occ: int):
    """Step 1: V[P,s] = sum_ia B[P,i,a] Z[ia,s]  (first half of Eq. (18), RI form)."""
    B = _f64(B)
    naux, N, _ = B.shape
    Z = _f64(Z, (n_occ * (N - n_occ), np.shape(Z)[1]))
    n_pole = Z.shape[1]
    V = np.empty((naux, n_pole))
    _load().qsgw_oracle_pole_weights(N, n_occ, naux, n_pole, _dp(B), _dp(Z), n_pole, _dp(V), n_pole)
    return V


def residues(B, V, s: int, rows=None):
    """Step 2 for one pole s: w[r,m] = sqrt(2) sum_P B[P,p_r,m] V[P,s]  (Eq. (18))."""
    B = _f64(B)
    naux, N, _ = B.shape
    V = _f64(V)
    if rows is None:
        n_rows, rp, keep = N, None, None
    else:
        keep = np.ascontiguousarray(rows, dtype=np.int32)
        n_rows, rp = len(keep), keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
    w = np.empty((n_rows, N))
    _load().qsgw_oracle_residues(N, naux, _dp(B), _dp(V), V.shape[1], int(s), n_rows, rp, _dp(w))
    return w


def sigma(B, eps, occ, Omega, Z, eta: float, n_occ: int, states=None):
    """Steps 1-3: Sigma (Eqs. (17)-(19)) for the poles handed in.

    ``states`` (optional list of MO indices) restricts the OUTPUT to those rows/columns;
    all internal sums (ia, P, m, s) still run over their full ranges.
    """
    B = _f64(B)
    naux, N, N2 = B.shape
    if N != N2:
        raise ValueError("B must be [naux, N, N]")
    eps = _f64(eps, (N,))
    occ = _f64(occ, (N,))
    Omega = _f64(Omega)
    n_pole = Omega.shape[0]
    Z = _f64(Z, (n_occ * (N - n_occ), n_pole))
    if states is None:
        n_states, sp, keep = N, None, None
    else:
        keep = np.ascontiguousarray(states, dtype=np.int32)
        if keep.min() < 0 or keep.max() >= N:
            raise ValueError("states out of range")
        n_states, sp = len(keep), keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
    out = np.empty((n_states, n_states))
    rc = _load().qsgw_oracle_sigma(N, n_occ, naux, n_pole, _dp(B), _dp(eps), _dp(occ), _dp(Omega), _dp(Z),
                                   n_pole, float(eta), n_states, sp, _dp(out))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_sigma failed with {rc}")
    return out


def sigma_diag(B, eps, occ, Omega, Z, eta: float, n_occ: int, omega, states=None):
    """G0W0 diagonal Sigma_pp(omega_k): Eq. (17) with m = n = p on a real frequency grid.

    Returns (Re, Im), each [n_states, n_omega]; ``states`` (optional) lists the diagonal elements wanted.
    """
    B = _f64(B)
    naux, N, N2 = B.shape
    if N != N2:
        raise ValueError("B must be [naux, N, N]")
    eps = _f64(eps, (N,))
    occ = _f64(occ, (N,))
    Omega = _f64(Omega)
    n_pole = Omega.shape[0]
    Z = _f64(Z, (n_occ * (N - n_occ), n_pole))
    omega = _f64(omega)
    if omega.ndim != 1 or omega.shape[0] < 1:
        raise ValueError("omega must be a non-empty 1-D grid")
    if states is None:
        n_states, sp, keep = N, None, None
    else:
        keep = np.ascontiguousarray(states, dtype=np.int32)
        if keep.min() < 0 or keep.max() >= N:
            raise ValueError("states out of range")
        n_states, sp = len(keep), keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int))
    re = np.empty((n_states, omega.shape[0]))
    im = np.empty((n_states, omega.shape[0]))
    rc = _load().qsgw_oracle_sigma_diag(N, n_occ, naux, n_pole, _dp(B), _dp(eps), _dp(occ), _dp(Omega), _dp(Z),
                                        n_pole, float(eta), omega.shape[0], _dp(omega), n_states, sp, _dp(re), _dp(im))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_sigma_diag failed with {rc}")
    return re, im


def ao_to_mo(B_ao, C):
    """RI AO->MO transformation of the three-index factors: the RI analogue of Eq. (16)
    (RI remark PAPER.md:120), B^P_pq = sum_mu sum_nu C[mu][p] C[nu][q] B^P_mu,nu -- the defining double
    sum in plain C loops (qsgw_oracle_ao_to_mo), O(naux n_mo^2 nao^2): pass a sample of the auxiliary functions at
    large sizes (each P is independent).

    B_ao [naux, nao, nao], C [nao, n_mo] (AO coefficients of the MOs, column p = orbital p) -> [naux, n_mo, n_mo].
    Pinned in tests/test_oracle_aomo_pins.py (hand values, identity / permutation / selection, composition, trace).
    """
    B_ao = _f64(B_ao)
    C = _f64(C)
    if B_ao.ndim != 3 or B_ao.shape[1] != B_ao.shape[2] or C.ndim != 2 or C.shape[0] != B_ao.shape[1]:
        raise ValueError("need B_ao [naux, nao, nao] and C [nao, n_mo]")
    naux, nao, n_mo = B_ao.shape[0], B_ao.shape[1], C.shape[1]
    out = np.empty((naux, n_mo, n_mo))
    rc = _load().qsgw_oracle_ao_to_mo(naux, nao, n_mo, _dp(B_ao), _dp(C), _dp(out))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_ao_to_mo failed with {rc}")
    return out


def mp2_direct(B, eps, occ, eta: float, n_occ: int):
    """Second-order Coulomb (direct) term of the qsMP2 self-energy: first sum of Eq. (20) in Eq. (21), closed shell
    (PAPER.md:174-186).  The SOX term is not included.  Returns Sigma [N, N]."""
    B = _f64(B)
    naux, N, N2 = B.shape
    if N != N2:
        raise ValueError("B must be [naux, N, N]")
    eps = _f64(eps, (N,))
    occ = _f64(occ, (N,))
    out = np.empty((N, N))
    rc = _load().qsgw_oracle_mp2_direct(N, n_occ, naux, _dp(B), _dp(eps), _dp(occ), float(eta), _dp(out))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_mp2_direct failed with {rc}")
    return out


def mp2(B, eps, occ, eta: float, n_occ: int, sox_only: bool = False, states=None):
    """qsMP2 correlation self-energy: both sums of Eq. (20) (direct and second-order exchange) in Eq. (21), closed
    shell.  ``sox_only`` returns the exchange part alone.  Returns Sigma [N, N].

    ``states`` (optional list of MO indices) restricts the OUTPUT to those rows/columns (qsgw_oracle_mp2_states: all
    internal sums still run over their full ranges); returns [len(states), len(states)].
    """
    B = _f64(B)
    naux, N, N2 = B.shape
    if N != N2:
        raise ValueError("B must be [naux, N, N]")
    eps = _f64(eps, (N,))
    occ = _f64(occ, (N,))
    if states is not None:
        keep = np.ascontiguousarray(states, dtype=np.int32)
        if keep.ndim != 1 or len(keep) < 1 or keep.min() < 0 or keep.max() >= N:
            raise ValueError("states out of range")
        out = np.empty((len(keep), len(keep)))
        rc = _load().qsgw_oracle_mp2_states(N, n_occ, naux, _dp(B), _dp(eps), _dp(occ), float(eta), 1 if sox_only else 0,
                                            len(keep), keep.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _dp(out))
        if rc != 0:
            raise RuntimeError(f"qsgw_oracle_mp2_states failed with {rc}")
        return out
    out = np.empty((N, N))
    rc = _load().qsgw_oracle_mp2(N, n_occ, naux, _dp(B), _dp(eps), _dp(occ), float(eta), 1 if sox_only else 0, _dp(out))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_mp2 failed with {rc}")
    return out


def casida_matrix(B, eps, n_occ: int):
    """C = (A-B)^(1/2) (A+B) (A-B)^(1/2) of the closed-shell direct-RPA Casida problem, Eqs. (12)-(14)
    with RI integrals: C[ia,jb] = Delta_ia^2 delta + 4 sqrt(Delta_ia) (ia|jb) sqrt(Delta_jb).  Returns [n_ov, n_ov]."""
    B = _f64(B)
    naux, N, N2 = B.shape
    if N != N2:
        raise ValueError("B must be [naux, N, N]")
    eps = _f64(eps, (N,))
    nov = n_occ * (N - n_occ)
    C = np.empty((nov, nov))
    rc = _load().qsgw_oracle_casida_matrix(N, n_occ, naux, _dp(B), _dp(eps), _dp(C))
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_casida_matrix failed with {rc}")
    return C


def casida_z(eps, n_occ: int, lam, xi):
    """After the eigensolve: Omega = sqrt(lambda), Z[ia,s] = sqrt(Delta_ia) xi[ia,s] / sqrt(Omega_s)  (X + Y of Eq. (18))."""
    eps = _f64(eps)
    N = eps.shape[0]
    lam = _f64(lam)
    xi = _f64(xi)
    nov = n_occ * (N - n_occ)
    n_pole = lam.shape[0]
    if xi.shape != (nov, n_pole):
        raise ValueError(f"xi must be [{nov}, {n_pole}]")
    Omega = np.empty(n_pole)
    Z = np.empty((nov, n_pole))
    rc = _load().qsgw_oracle_casida_z(N, n_occ, _dp(eps), n_pole, _dp(lam), _dp(xi), n_pole, _dp(Omega), _dp(Z), n_pole)
    if rc != 0:
        raise RuntimeError(f"qsgw_oracle_casida_z failed with {rc} (non-positive eigenvalue?)")
    return Omega, Z


def casida(B, eps, n_occ: int):
    """The whole Casida / RPA step, Eqs. (12)-(14): (Omega [n_ov] ascending, Z = X + Y [n_ov, n_ov]).  Plain loops for C and
    for the back-transformation; the symmetric eigensolve between them is numpy.linalg.eigh (a library routine as a step)."""
    C = casida_matrix(B, eps, n_occ)
    lam, xi = np.linalg.eigh(C)
    return casida_z(eps, n_occ, lam, xi)
