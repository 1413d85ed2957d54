"""Thin ctypes binding of include/qsgw_sigma.h: argument marshalling only.

Every step of the path runs in the CUDA kernels of libqsgw_sigma.so; PyTorch is used for
device memory and streams.  There is no CPU fallback: if the shared library is missing or
there is no CUDA device the calls raise.  Function names are the C names.

Streams: a plan enqueues all its work on the stream it was created with.  Tensors handed to a
plan must have been produced on that stream (or the caller must have made the stream wait for
their producers), and must stay alive until the stream has passed the call -- the binding keeps
no references.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqsgw_sigma.so")

QSGW_SIGMA_OK = 0
QSGW_SIGMA_ERR_INVALID_ARG = -1
QSGW_SIGMA_ERR_ALLOC = -2
QSGW_SIGMA_ERR_CUDA = -3

EXPORTS = (
    "qsgw_sigma_create", "qsgw_sigma_build", "qsgw_sigma_begin", "qsgw_sigma_add_poles", "qsgw_sigma_finish",
    "qsgw_sigma_build_host", "qsgw_sigma_diag_build", "qsgw_mp2_direct_build", "qsgw_mp2_build", "qsgw_ri_ao_to_mo", "qsgw_ri_ao_to_mo_work_doubles", "qsgw_ri_ao_to_mo_static", "qsgw_ri_ao_to_mo_static_max_doubles", "qsgw_sigma_destroy", "qsgw_sigma_last_error", "qsgw_sigma_workspace_bytes",
    "qsgw_sigma_limit_pole_batch", "qsgw_sigma_set_profiling", "qsgw_sigma_get_stats", "qsgw_sigma_set_debug", "qsgw_sigma_version",
    "qsgw_sigma_pole_slice", "qsgw_casida_work_doubles", "qsgw_casida_matrix", "qsgw_casida_z",
)


class QsgwSigmaError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"qsgw_sigma error {code}: {message}")
        self.code = code


class qsgw_sigma_stats(ctypes.Structure):
    _fields_ = [
        ("ms_pack", ctypes.c_double), ("launches_pack", ctypes.c_int64),
        ("ms_stage1", ctypes.c_double), ("launches_stage1", ctypes.c_int64),
        ("ms_stage2", ctypes.c_double), ("launches_stage2", ctypes.c_int64),
        ("ms_stage3", ctypes.c_double), ("launches_stage3", ctypes.c_int64),
        ("ms_epilogue", ctypes.c_double), ("launches_epilogue", ctypes.c_int64),
        ("ms_diag", ctypes.c_double), ("launches_diag", ctypes.c_int64),
        ("kernel_launches", ctypes.c_int64), ("builds", ctypes.c_int64), ("poles", ctypes.c_int64),
    ]

    def as_dict(self):
        return {name: getattr(self, name) for name, _ in self._fields_}


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree libqsgw_sigma.so (built by paper_2210_17093_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} not found: build it with `python -m paper_2210_17093_b200.build` "
                "(there is no CPU fallback for the qsGW Sigma build)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, dp, i64, ci, cd = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        lib.qsgw_sigma_create.restype = ci
        lib.qsgw_sigma_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, i64, ci, vp]
        lib.qsgw_sigma_build.restype = ci
        lib.qsgw_sigma_build.argtypes = [vp, dp, dp, dp, dp, dp, i64, i64, cd, dp]
        lib.qsgw_sigma_begin.restype = ci
        lib.qsgw_sigma_begin.argtypes = [vp, dp, dp, dp, cd]
        lib.qsgw_sigma_add_poles.restype = ci
        lib.qsgw_sigma_add_poles.argtypes = [vp, dp, dp, i64, i64]
        lib.qsgw_sigma_finish.restype = ci
        lib.qsgw_sigma_finish.argtypes = [vp, dp]
        lib.qsgw_sigma_build_host.restype = ci
        lib.qsgw_sigma_build_host.argtypes = [vp, dp, dp, dp, dp, dp, i64, i64, cd, dp]
        lib.qsgw_sigma_diag_build.restype = ci
        lib.qsgw_sigma_diag_build.argtypes = [vp, dp, dp, dp, dp, dp, i64, i64, cd, dp, ci, dp, dp]
        lib.qsgw_mp2_direct_build.restype = ci
        lib.qsgw_mp2_direct_build.argtypes = [vp, dp, dp, dp, cd, dp]
        lib.qsgw_mp2_build.restype = ci
        lib.qsgw_mp2_build.argtypes = [vp, dp, dp, dp, cd, dp]
        lib.qsgw_ri_ao_to_mo.restype = ci
        lib.qsgw_ri_ao_to_mo.argtypes = [dp, dp, ci, ci, ci, dp, dp, vp]
        lib.qsgw_ri_ao_to_mo_work_doubles.restype = ctypes.c_size_t
        lib.qsgw_ri_ao_to_mo_work_doubles.argtypes = [ci, ci, ci]
        lib.qsgw_ri_ao_to_mo_static.restype = ci
        lib.qsgw_ri_ao_to_mo_static.argtypes = [dp, dp, ci, ci, ci, dp, vp]
        lib.qsgw_ri_ao_to_mo_static_max_doubles.restype = ctypes.c_size_t
        lib.qsgw_ri_ao_to_mo_static_max_doubles.argtypes = []
        lib.qsgw_sigma_destroy.restype = ci
        lib.qsgw_sigma_destroy.argtypes = [vp]
        lib.qsgw_sigma_last_error.restype = ctypes.c_char_p
        lib.qsgw_sigma_last_error.argtypes = [vp]
        lib.qsgw_sigma_workspace_bytes.restype = ctypes.c_size_t
        lib.qsgw_sigma_workspace_bytes.argtypes = [vp]
        lib.qsgw_sigma_limit_pole_batch.restype = ci
        lib.qsgw_sigma_limit_pole_batch.argtypes = [vp, i64]
        lib.qsgw_sigma_set_profiling.restype = ci
        lib.qsgw_sigma_set_profiling.argtypes = [vp, ci]
        lib.qsgw_sigma_get_stats.restype = ci
        lib.qsgw_sigma_get_stats.argtypes = [vp, ctypes.POINTER(qsgw_sigma_stats), ci]
        lib.qsgw_sigma_pole_slice.restype = ci
        lib.qsgw_sigma_pole_slice.argtypes = [i64, ci, ci, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        lib.qsgw_casida_work_doubles.restype = ctypes.c_size_t
        lib.qsgw_casida_work_doubles.argtypes = [ci, ci, ci]
        lib.qsgw_casida_matrix.restype = ci
        lib.qsgw_casida_matrix.argtypes = [dp, dp, ci, ci, ci, dp, dp, i64, vp]
        lib.qsgw_casida_z.restype = ci
        lib.qsgw_casida_z.argtypes = [dp, ci, ci, dp, dp, i64, i64, dp, dp, i64, vp]
        lib.qsgw_sigma_set_debug.restype = ci
        lib.qsgw_sigma_set_debug.argtypes = [vp, ci]
        lib.qsgw_sigma_version.restype = ci
        lib.qsgw_sigma_version.argtypes = []
        _lib = lib
    return _lib


def _check(rc: int, plan) -> None:
    if rc != QSGW_SIGMA_OK:
        msg = load_library().qsgw_sigma_last_error(plan)
        raise QsgwSigmaError(rc, msg.decode() if msg else "")


def _dev(t: torch.Tensor, name: str, shape=None) -> int:
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float64:
        raise TypeError(f"{name} must be a CUDA float64 tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


def _host(t: torch.Tensor, name: str, shape=None) -> int:
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise TypeError(f"{name} must be a contiguous host float64 tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t.data_ptr()


class Plan:
    """Handle returned by qsgw_sigma_create (holds the opaque qsgw_sigma_plan* and the sizes)."""

    def __init__(self, handle, n_mo, n_occ, n_aux, n_pole_max, s_block, stream, device):
        self.handle, self.n_mo, self.n_occ, self.n_aux = handle, n_mo, n_occ, n_aux
        self.n_pole_max, self.s_block, self.stream, self.device = n_pole_max, s_block, stream, device
        self.n_ov = n_occ * (n_mo - n_occ)

    def __del__(self):
        try:
            qsgw_sigma_destroy(self)
        except Exception:
            pass


def qsgw_sigma_create(n_mo: int, n_occ: int, n_aux: int, n_pole_max: int, s_block: int = 0,
                      stream: Optional[torch.cuda.Stream] = None) -> Plan:
    """The plan lives on the current CUDA device (the stream, if given, must belong to it)."""
    lib = load_library()
    device = None
    if torch.cuda.is_available():
        if stream is None:
            stream = torch.cuda.current_stream()
        device = torch.device("cuda", torch.cuda.current_device())
    sptr = ctypes.c_void_p(stream.cuda_stream if stream is not None else 0)
    h = ctypes.c_void_p()
    rc = lib.qsgw_sigma_create(ctypes.byref(h), int(n_mo), int(n_occ), int(n_aux), int(n_pole_max), int(s_block), sptr)
    _check(rc, None)
    return Plan(h, n_mo, n_occ, n_aux, n_pole_max, s_block, stream, device)


def _z_args(plan: Plan, Omega: torch.Tensor, Z: torch.Tensor, ptr):
    n_pole = Omega.shape[0]
    if Z.dim() != 2 or Z.shape != (plan.n_ov, n_pole) or Z.stride(1) != 1:
        raise ValueError(f"Z must be [{plan.n_ov}, {n_pole}] with unit column stride (a column slice of a larger Z is fine)")
    if not Omega.is_contiguous():
        raise ValueError("Omega must be contiguous")
    return ptr(Omega, "Omega"), ptr(Z, "Z"), int(Z.stride(0)) if Z.shape[0] > 1 else max(n_pole, int(Z.stride(0))), n_pole


def qsgw_sigma_build(plan: Plan, B, eps, occ, Omega, Z, eta: float, Sigma: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Sigma (Eq. 19) for the poles handed in; asynchronous on the plan's stream.  Z may be a column slice."""
    N = plan.n_mo
    if not B.is_contiguous() or not eps.is_contiguous() or not occ.is_contiguous():
        raise ValueError("B, eps, occ must be contiguous")
    if Sigma is None:
        Sigma = torch.empty((N, N), dtype=torch.float64, device=B.device)
    om, z, ldz, n_pole = _z_args(plan, Omega, Z, _dev)
    rc = load_library().qsgw_sigma_build(plan.handle, _dev(B, "B", (plan.n_aux, N, N)), _dev(eps, "eps", (N,)),
                                         _dev(occ, "occ", (N,)), om, z, ldz, n_pole, float(eta),
                                         _dev(Sigma, "Sigma", (N, N)))
    _check(rc, plan.handle)
    return Sigma


def qsgw_sigma_begin(plan: Plan, B, eps, occ, eta: float) -> None:
    N = plan.n_mo
    if not B.is_contiguous() or not eps.is_contiguous() or not occ.is_contiguous():
        raise ValueError("B, eps, occ must be contiguous")
    rc = load_library().qsgw_sigma_begin(plan.handle, _dev(B, "B", (plan.n_aux, N, N)), _dev(eps, "eps", (N,)),
                                         _dev(occ, "occ", (N,)), float(eta))
    _check(rc, plan.handle)


def qsgw_sigma_add_poles(plan: Plan, Omega, Z) -> None:
    om, z, ldz, n_pole = _z_args(plan, Omega, Z, _dev)
    _check(load_library().qsgw_sigma_add_poles(plan.handle, om, z, ldz, n_pole), plan.handle)


def qsgw_sigma_finish(plan: Plan, Sigma: Optional[torch.Tensor] = None) -> torch.Tensor:
    N = plan.n_mo
    if Sigma is None:
        Sigma = torch.empty((N, N), dtype=torch.float64, device=plan.device)
    _check(load_library().qsgw_sigma_finish(plan.handle, _dev(Sigma, "Sigma", (N, N))), plan.handle)
    return Sigma


def qsgw_sigma_build_host(plan: Plan, B, eps, occ, Omega, Z, eta: float, Sigma: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Same build from HOST tensors (pinned or pageable); uploads, builds, downloads, synchronises."""
    N = plan.n_mo
    if Sigma is None:
        Sigma = torch.empty((N, N), dtype=torch.float64)
    om, z, ldz, n_pole = _z_args(plan, Omega, Z, _host_strided)
    rc = load_library().qsgw_sigma_build_host(plan.handle, _host(B, "B", (plan.n_aux, N, N)), _host(eps, "eps", (N,)),
                                              _host(occ, "occ", (N,)), om, z, ldz, n_pole, float(eta),
                                              _host(Sigma, "Sigma", (N, N)))
    _check(rc, plan.handle)
    return Sigma


def qsgw_sigma_diag_build(plan: Plan, B, eps, occ, Omega, Z, eta: float, omega_grid, SigmaRe=None, SigmaIm=None):
    """G0W0 diagonal Sigma_pp(omega_k) (Eq. (17) with m = n) for all states p; returns (Re, Im), each [n_mo, n_omega]."""
    N = plan.n_mo
    if not B.is_contiguous() or not eps.is_contiguous() or not occ.is_contiguous() or not omega_grid.is_contiguous():
        raise ValueError("B, eps, occ, omega_grid must be contiguous")
    n_omega = int(omega_grid.shape[0])
    if SigmaRe is None:
        SigmaRe = torch.empty((N, n_omega), dtype=torch.float64, device=B.device)
    if SigmaIm is None:
        SigmaIm = torch.empty((N, n_omega), dtype=torch.float64, device=B.device)
    om, z, ldz, n_pole = _z_args(plan, Omega, Z, _dev)
    rc = load_library().qsgw_sigma_diag_build(plan.handle, _dev(B, "B", (plan.n_aux, N, N)), _dev(eps, "eps", (N,)),
                                              _dev(occ, "occ", (N,)), om, z, ldz, n_pole, float(eta),
                                              _dev(omega_grid, "omega_grid", (n_omega,)), n_omega,
                                              _dev(SigmaRe, "SigmaRe", (N, n_omega)), _dev(SigmaIm, "SigmaIm", (N, n_omega)))
    _check(rc, plan.handle)
    return SigmaRe, SigmaIm


def qsgw_mp2_direct_build(plan: Plan, B, eps, occ, eta: float, Sigma: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Direct (second-order Coulomb) term of the qsMP2 self-energy, Eq. (20) first sum in Eq. (21); SOX not included."""
    N = plan.n_mo
    if not B.is_contiguous() or not eps.is_contiguous() or not occ.is_contiguous():
        raise ValueError("B, eps, occ must be contiguous")
    if Sigma is None:
        Sigma = torch.empty((N, N), dtype=torch.float64, device=B.device)
    rc = load_library().qsgw_mp2_direct_build(plan.handle, _dev(B, "B", (plan.n_aux, N, N)), _dev(eps, "eps", (N,)),
                                              _dev(occ, "occ", (N,)), float(eta), _dev(Sigma, "Sigma", (N, N)))
    _check(rc, plan.handle)
    return Sigma


def qsgw_mp2_build(plan: Plan, B, eps, occ, eta: float, Sigma: Optional[torch.Tensor] = None) -> torch.Tensor:
    """qsMP2 correlation self-energy: direct + second-order exchange sums of Eq. (20) in Eq. (21)."""
    N = plan.n_mo
    if not B.is_contiguous() or not eps.is_contiguous() or not occ.is_contiguous():
        raise ValueError("B, eps, occ must be contiguous")
    if Sigma is None:
        Sigma = torch.empty((N, N), dtype=torch.float64, device=B.device)
    rc = load_library().qsgw_mp2_build(plan.handle, _dev(B, "B", (plan.n_aux, N, N)), _dev(eps, "eps", (N,)),
                                       _dev(occ, "occ", (N,)), float(eta), _dev(Sigma, "Sigma", (N, N)))
    _check(rc, plan.handle)
    return Sigma


def qsgw_ri_ao_to_mo_work_doubles(n_aux: int, n_ao: int, n_mo: int) -> int:
    return int(load_library().qsgw_ri_ao_to_mo_work_doubles(int(n_aux), int(n_ao), int(n_mo)))


def qsgw_ri_ao_to_mo_static_max_doubles() -> int:
    return int(load_library().qsgw_ri_ao_to_mo_static_max_doubles())


def qsgw_ri_ao_to_mo_static(B_ao: torch.Tensor, C: torch.Tensor, B_mo: torch.Tensor,
                            stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """qsgw_ri_ao_to_mo with the library's static scratch array: the call allocates nothing, so B_mo is the caller's.
    Calls that overlap on the GPU race on the shared scratch (include/qsgw_sigma.h)."""
    if B_ao.dim() != 3 or B_ao.shape[1] != B_ao.shape[2] or C.dim() != 2 or C.shape[0] != B_ao.shape[1]:
        raise ValueError("need B_ao [n_aux, n_ao, n_ao] and C [n_ao, n_mo]")
    if not B_ao.is_contiguous() or not C.is_contiguous():
        raise ValueError("B_ao and C must be contiguous")
    n_aux, n_ao, n_mo = int(B_ao.shape[0]), int(B_ao.shape[1]), int(C.shape[1])
    if stream is None:
        stream = torch.cuda.current_stream(B_ao.device)
    rc = load_library().qsgw_ri_ao_to_mo_static(_dev(B_ao, "B_ao"), _dev(C, "C"), n_aux, n_ao, n_mo,
                                                _dev(B_mo, "B_mo", (n_aux, n_mo, n_mo)), ctypes.c_void_p(stream.cuda_stream))
    _check(rc, None)
    return B_mo


def qsgw_ri_ao_to_mo(B_ao: torch.Tensor, C: torch.Tensor, B_mo: Optional[torch.Tensor] = None,
                     work: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """B_mo[P] = C^T B_ao[P] C for every auxiliary function P (RI AO->MO transformation); asynchronous on the stream."""
    if B_ao.dim() != 3 or B_ao.shape[1] != B_ao.shape[2] or C.dim() != 2 or C.shape[0] != B_ao.shape[1]:
        raise ValueError("need B_ao [n_aux, n_ao, n_ao] and C [n_ao, n_mo]")
    if not B_ao.is_contiguous() or not C.is_contiguous():
        raise ValueError("B_ao and C must be contiguous")
    n_aux, n_ao, n_mo = int(B_ao.shape[0]), int(B_ao.shape[1]), int(C.shape[1])
    if B_mo is None:
        B_mo = torch.empty((n_aux, n_mo, n_mo), dtype=torch.float64, device=B_ao.device)
    need = qsgw_ri_ao_to_mo_work_doubles(n_aux, n_ao, n_mo)
    if work is None:
        work = torch.empty(need, dtype=torch.float64, device=B_ao.device)
    if work.numel() < need or not work.is_contiguous():
        raise ValueError(f"work needs {need} contiguous doubles")
    if stream is None:
        stream = torch.cuda.current_stream(B_ao.device)
    for t in (B_ao, C, B_mo, work):       # the launch is asynchronous on `stream`: keep the allocator from reusing them early
        t.record_stream(stream)
    rc = load_library().qsgw_ri_ao_to_mo(_dev(B_ao, "B_ao"), _dev(C, "C"), n_aux, n_ao, n_mo, _dev(work, "work"),
                                         _dev(B_mo, "B_mo", (n_aux, n_mo, n_mo)), ctypes.c_void_p(stream.cuda_stream))
    _check(rc, None)
    return B_mo


def _host_strided(t: torch.Tensor, name: str) -> int:
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float64:
        raise TypeError(f"{name} must be a host float64 tensor")
    return t.data_ptr()


def qsgw_sigma_destroy(plan: Plan) -> None:
    if plan is not None and plan.handle is not None and plan.handle.value:
        h, plan.handle = plan.handle, ctypes.c_void_p()
        load_library().qsgw_sigma_destroy(h)


def qsgw_sigma_last_error(plan: Optional[Plan]) -> str:
    msg = load_library().qsgw_sigma_last_error(plan.handle if plan is not None else None)
    return msg.decode() if msg else ""


def qsgw_sigma_workspace_bytes(plan: Plan) -> int:
    return int(load_library().qsgw_sigma_workspace_bytes(plan.handle))


def qsgw_sigma_limit_pole_batch(plan: Plan, n: int) -> None:
    _check(load_library().qsgw_sigma_limit_pole_batch(plan.handle, int(n)), plan.handle)


def qsgw_sigma_set_profiling(plan: Plan, on: bool) -> None:
    _check(load_library().qsgw_sigma_set_profiling(plan.handle, 1 if on else 0), plan.handle)


def qsgw_sigma_get_stats(plan: Plan, reset: bool = False) -> dict:
    st = qsgw_sigma_stats()
    _check(load_library().qsgw_sigma_get_stats(plan.handle, ctypes.byref(st), 1 if reset else 0), plan.handle)
    return st.as_dict()


def qsgw_sigma_set_debug(plan: Plan, on: bool) -> None:
    """Device-side precondition checks (B symmetric and finite, occ in [0,1], Omega > 0) in begin / add_poles."""
    _check(load_library().qsgw_sigma_set_debug(plan.handle, 1 if on else 0), plan.handle)


def qsgw_sigma_pole_slice(n_pole: int, n_ranks: int, rank: int):
    """(s0, n): the contiguous slice of the pole index that rank `rank` of `n_ranks` builds (pure host arithmetic)."""
    s0, n = ctypes.c_int64(), ctypes.c_int64()
    _check(load_library().qsgw_sigma_pole_slice(int(n_pole), int(n_ranks), int(rank), ctypes.byref(s0), ctypes.byref(n)), None)
    return int(s0.value), int(n.value)


def qsgw_casida_work_doubles(n_mo: int, n_occ: int, n_aux: int) -> int:
    return int(load_library().qsgw_casida_work_doubles(int(n_mo), int(n_occ), int(n_aux)))


def qsgw_casida_matrix(B: torch.Tensor, eps: torch.Tensor, n_occ: int, C: Optional[torch.Tensor] = None,
                       work: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """C = (A-B)^(1/2) (A+B) (A-B)^(1/2) of the closed-shell RPA Casida problem (Eqs. (12)-(14)); [n_ov, n_ov], bit-symmetric."""
    if B.dim() != 3 or B.shape[1] != B.shape[2] or not B.is_contiguous() or not eps.is_contiguous():
        raise ValueError("need contiguous B [n_aux, n_mo, n_mo] and eps [n_mo]")
    n_aux, n_mo = int(B.shape[0]), int(B.shape[1])
    n_ov = n_occ * (n_mo - n_occ)
    if C is None:
        C = torch.empty((n_ov, n_ov), dtype=torch.float64, device=B.device)
    if C.dim() != 2 or tuple(C.shape) != (n_ov, n_ov) or C.stride(1) != 1:
        raise ValueError(f"C must be [{n_ov}, {n_ov}] with unit column stride")
    need = qsgw_casida_work_doubles(n_mo, n_occ, n_aux)
    if work is None:
        work = torch.empty(need, dtype=torch.float64, device=B.device)
    if work.numel() < need or not work.is_contiguous():
        raise ValueError(f"work needs {need} contiguous doubles")
    if stream is None:
        stream = torch.cuda.current_stream(B.device)
    for t in (B, eps, C, work):
        t.record_stream(stream)
    rc = load_library().qsgw_casida_matrix(_dev(B, "B"), _dev(eps, "eps", (n_mo,)), n_mo, int(n_occ), n_aux, _dev(work, "work"),
                                           _dev(C, "C"), int(C.stride(0)), ctypes.c_void_p(stream.cuda_stream))
    _check(rc, None)
    return C


def qsgw_casida_z(eps: torch.Tensor, n_occ: int, lam: torch.Tensor, xi: torch.Tensor, Omega: Optional[torch.Tensor] = None,
                  Z: Optional[torch.Tensor] = None, stream: Optional[torch.cuda.Stream] = None):
    """(Omega, Z): Omega = sqrt(lambda), Z[ia, s] = sqrt(Delta_ia) xi[ia, s] / sqrt(Omega_s) for the eigenpairs handed in."""
    n_mo = int(eps.shape[0])
    n_ov = n_occ * (n_mo - n_occ)
    n_pole = int(lam.shape[0])
    if xi.dim() != 2 or tuple(xi.shape) != (n_ov, n_pole) or xi.stride(1) != 1 or not lam.is_contiguous():
        raise ValueError(f"xi must be [{n_ov}, {n_pole}] with unit column stride (eigenvectors in the columns), lambda contiguous")
    if Omega is None:
        Omega = torch.empty(n_pole, dtype=torch.float64, device=xi.device)
    if Z is None:
        Z = torch.empty((n_ov, n_pole), dtype=torch.float64, device=xi.device)
    if stream is None:
        stream = torch.cuda.current_stream(xi.device)
    for t in (eps, lam, xi, Omega, Z):
        t.record_stream(stream)
    rc = load_library().qsgw_casida_z(_dev(eps, "eps"), n_mo, int(n_occ), _dev(lam, "lambda"), _dev(xi, "xi"), int(xi.stride(0)) if n_ov > 1 else n_pole,
                                      n_pole, _dev(Omega, "Omega", (n_pole,)), _dev(Z, "Z", (n_ov, n_pole)), int(Z.stride(0)) if n_ov > 1 else n_pole,
                                      ctypes.c_void_p(stream.cuda_stream))
    _check(rc, None)
    return Omega, Z


def qsgw_sigma_version() -> int:
    return int(load_library().qsgw_sigma_version())
