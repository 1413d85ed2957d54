"""qsgw_ri_ao_to_mo_static: the AO->MO transformation with the library's file-scope static scratch array -- the one entry
point for callers that must not allocate device memory (include/qsgw_sigma.h).  Checked against the existing path
(qsgw_ri_ao_to_mo with a caller-owned work buffer) on two calls in a row that share the scratch, at the bar of
tests/test_gpu_aomo.py (1e-12 * max|ref|; the two paths run the same kernels, so the results are in fact equal).

This file is collected last on purpose (pytest -x): it must pass alone in a fresh process and after
all the other tests.
"""
import numpy as np
import pytest
import torch

import paper_2210_17093_b200 as pkg

pytestmark = pytest.mark.gpu


def _inputs(n_aux, n_ao, n_mo, seed):
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    B_ao = torch.randn((n_aux, n_ao, n_ao), generator=g, dtype=torch.float64, device="cuda") * 0.1
    C = torch.randn((n_ao, n_mo), generator=g, dtype=torch.float64, device="cuda") / np.sqrt(n_ao)
    return B_ao, C


def test_static_scratch_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    torch.cuda.set_device(0)
    # the second problem is smaller and has odd n_mo / n_ao != n_mo: it runs on top of the first call's leftovers
    shapes = [(96, 150, 140, 11), (37, 61, 45, 12)]
    outs = []
    for n_aux, n_ao, n_mo, seed in shapes:
        assert pkg.qsgw_ri_ao_to_mo_work_doubles(n_aux, n_ao, n_mo) <= pkg.qsgw_ri_ao_to_mo_static_max_doubles()
        B_ao, C = _inputs(n_aux, n_ao, n_mo, seed)
        B_mo = torch.full((n_aux, n_mo, n_mo), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        pkg.qsgw_ri_ao_to_mo_static(B_ao, C, B_mo)           # allocates nothing: output and inputs are the caller's
        assert torch.cuda.memory_allocated() == before
        outs.append((B_ao, C, B_mo))
    torch.cuda.synchronize()
    for B_ao, C, B_mo in outs:
        ref = pkg.qsgw_ri_ao_to_mo(B_ao, C)                   # existing path, caller-owned (torch) work buffer
        torch.cuda.synchronize()
        r, g = ref.cpu().numpy(), B_mo.cpu().numpy()
        assert np.isfinite(g).all()
        assert np.max(np.abs(g - r)) <= 1e-12 * np.abs(r).max()
        # and against the definition, so that the pair cannot be wrong together
        P = 3
        lit = C.cpu().numpy().T @ B_ao[P].cpu().numpy() @ C.cpu().numpy()
        assert np.max(np.abs(g[P] - lit)) <= 1e-9 * np.abs(lit).max()


def test_static_scratch_entry_point_rejects_sizes_beyond_its_maximum():
    torch.cuda.set_device(0)
    limit = pkg.qsgw_ri_ao_to_mo_static_max_doubles()
    assert limit == 8 * 1024 * 1024
    n_aux, n_ao, n_mo = 600, 120, 120                        # 8.64 M doubles of scratch > 8 Mi
    assert pkg.qsgw_ri_ao_to_mo_work_doubles(n_aux, n_ao, n_mo) > limit
    B_ao, C = _inputs(n_aux, n_ao, n_mo, 13)
    B_mo = torch.zeros((n_aux, n_mo, n_mo), dtype=torch.float64, device="cuda")
    with pytest.raises(pkg.QsgwSigmaError) as ei:
        pkg.qsgw_ri_ao_to_mo_static(B_ao, C, B_mo)
    assert ei.value.code == pkg.QSGW_SIGMA_ERR_INVALID_ARG
    assert "static maximum" in str(ei.value)
    torch.cuda.synchronize()
    assert float(B_mo.abs().sum()) == 0.0                    # nothing was launched
