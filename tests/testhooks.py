"""Test build of the CUDA library: the product's sources compiled with -DQSGW_SIGMA_TEST_HOOKS into
libqsgw_sigma_testhooks.so, which adds qsgw_sigma_copy_workspace (a look at V, the w chunk, the packed B and the split-K
partial tiles).  The hook is not in libqsgw_sigma.so.  Raw ctypes, the signatures of include/qsgw_sigma.h."""
import ctypes

import torch

WORKSPACE_V, WORKSPACE_W, WORKSPACE_BP, WORKSPACE_BOVT, WORKSPACE_TPART = range(5)

_lib = None


def load():
    global _lib
    if _lib is None:
        from paper_2210_17093_b200 import build
        lib = ctypes.CDLL(build.build_library(test_hooks=True))
        vp, i64, ci, cd = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        lib.qsgw_sigma_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, i64, ci, vp]
        lib.qsgw_sigma_build.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, cd, vp]
        lib.qsgw_sigma_copy_workspace.argtypes = [vp, ci, vp, i64, i64]
        lib.qsgw_sigma_destroy.argtypes = [vp]
        lib.qsgw_sigma_last_error.restype = ctypes.c_char_p
        lib.qsgw_sigma_last_error.argtypes = [vp]
        _lib = lib
    return _lib


class HookedPlan:
    """create / build / copy_workspace / destroy on the test build, for tensors on the current CUDA device."""

    def __init__(self, n_mo, n_occ, n_aux, n_pole_max, s_block=0):
        self.lib, self.h = load(), ctypes.c_void_p()
        self.n_mo = n_mo
        stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
        self._ok(self.lib.qsgw_sigma_create(ctypes.byref(self.h), n_mo, n_occ, n_aux, n_pole_max, s_block, stream))

    def _ok(self, rc):
        if rc != 0:
            raise RuntimeError(f"test-hooks library: rc {rc}: {self.lib.qsgw_sigma_last_error(self.h).decode()}")

    def build(self, B, eps, occ, Omega, Z, eta):
        S = torch.empty((self.n_mo, self.n_mo), dtype=torch.float64, device=B.device)
        self._keep = (B, eps, occ, Omega, Z)
        self._ok(self.lib.qsgw_sigma_build(self.h, B.data_ptr(), eps.data_ptr(), occ.data_ptr(), Omega.data_ptr(), Z.data_ptr(),
                                           Z.stride(0), Omega.shape[0], float(eta), S.data_ptr()))
        return S

    def copy_workspace(self, which, rows, cols):
        out = torch.empty((rows, cols), dtype=torch.float64, device="cuda")
        self._ok(self.lib.qsgw_sigma_copy_workspace(self.h, which, out.data_ptr(), rows, cols))
        return out

    def destroy(self):
        if self.h.value:
            self.lib.qsgw_sigma_destroy(self.h)
            self.h = ctypes.c_void_p()
