"""Parity of qsgw_ri_ao_to_mo (row 8(f).2: B_mo[P] = C^T B_ao[P] C as two batched DMMA GEMMs) against
oracle.ao_to_mo, element by element on the same seeded inputs.  Bar: 1e-9 * max|ref| (measured ~1e-15)."""
import numpy as np
import pytest
import torch

import oracle

pytestmark = pytest.mark.gpu


def _pkg():
    import paper_2210_17093_b200 as pkg
    return pkg


def _case(seed, naux, nao, n_mo, sym=True):
    g = torch.Generator().manual_seed(seed)
    G = torch.randn((naux, nao, nao), generator=g, dtype=torch.float64)
    B = 0.5 * (G + G.transpose(1, 2)) if sym else G
    C = torch.randn((nao, n_mo), generator=g, dtype=torch.float64) / np.sqrt(nao)
    return B.contiguous(), C.contiguous()


@pytest.mark.parametrize("naux,nao,n_mo,sym", [
    (80, 24, 24, True),       # tiny config shapes
    (40, 120, 120, True),     # small config N (a tenth of its naux: the oracle is the O(N^4) double sum per P)
    (7, 37, 29, False),       # odd sizes, unsymmetric B, n_mo != n_ao: scalar loads and stores, ragged tiles
    (3, 130, 131, False),     # just over one tile in every dimension
    (5, 257, 64, True),       # K tail (257 = 8 * 32 + 1)
    (1, 1, 1, True),
])
def test_parity(naux, nao, n_mo, sym):
    pkg = _pkg()
    B, C = _case(100 + nao, naux, nao, n_mo, sym)
    got = pkg.qsgw_ri_ao_to_mo(B.cuda(), C.cuda())
    torch.cuda.synchronize()
    ref = oracle.ao_to_mo(B.numpy(), C.numpy())
    err = np.max(np.abs(got.cpu().numpy() - ref))
    assert err <= 1e-9 * np.abs(ref).max(), f"{err:.3e}"
    assert err <= 1e-12 * np.abs(ref).max()


def test_medium_config_shapes_and_misaligned_views():
    pkg = _pkg()
    B, C = _case(7, 1100, 300, 300)
    Bd, Cd = B.cuda(), C.cuda()
    got = pkg.qsgw_ri_ao_to_mo(Bd, Cd)
    sample = [0, 1, 15, 16, 547, 1098, 1099]           # the oracle is the O(N^4) double sum per auxiliary function
    ref = oracle.ao_to_mo(B[sample].numpy(), C.numpy())
    assert np.max(np.abs(got[sample].cpu().numpy() - ref)) <= 1e-12 * np.abs(ref).max()
    # operands and result at 8-byte (not 16-byte) aligned addresses
    flatB = torch.empty(Bd.numel() + 1, dtype=torch.float64, device="cuda")
    flatC = torch.empty(Cd.numel() + 1, dtype=torch.float64, device="cuda")
    flatO = torch.empty(1100 * 300 * 300 + 1, dtype=torch.float64, device="cuda")
    Bm = flatB[1:].view(1100, 300, 300); Bm.copy_(Bd)
    Cm = flatC[1:].view(300, 300); Cm.copy_(Cd)
    Om = flatO[1:].view(1100, 300, 300)
    pkg.qsgw_ri_ao_to_mo(Bm, Cm, B_mo=Om)
    torch.cuda.synchronize()
    assert torch.equal(Om, got)                      # same arithmetic order whatever the alignment
    with pytest.raises(ValueError):
        pkg.qsgw_ri_ao_to_mo(Bd, Cd, work=torch.empty(10, dtype=torch.float64, device="cuda"))


def test_transformed_b_feeds_the_sigma_build():
    """End of the chain: B_mo from the GPU transform goes straight into qsgw_sigma_build; the oracle does both steps."""
    import qsgw_inputs as qi
    pkg = _pkg()
    cfg = qi.custom_config(48, 9, 30, n_pole=120, seed=3)
    inp = qi.make_inputs(cfg)
    g = torch.Generator().manual_seed(5)
    Q, _ = torch.linalg.qr(torch.randn((48, 48), generator=g, dtype=torch.float64))
    B_ao = inp.B                                            # take the config's B as the AO-basis factors
    B_mo = pkg.qsgw_ri_ao_to_mo(B_ao.cuda(), Q.contiguous().cuda())
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, 0)
    S = pkg.qsgw_sigma_build(plan, B_mo, inp.eps.cuda(), inp.occ.cuda(), inp.Omega.cuda(), inp.Z.cuda(), cfg.eta)
    torch.cuda.synchronize()
    ref = oracle.sigma(oracle.ao_to_mo(B_ao.numpy(), Q.numpy()), inp.eps.numpy(), inp.occ.numpy(), inp.Omega.numpy(),
                       inp.Z.numpy(), cfg.eta, cfg.n_occ)
    assert np.max(np.abs(S.cpu().numpy() - ref)) <= 1e-9 * np.abs(ref).max()
    pkg.qsgw_sigma_destroy(plan)
