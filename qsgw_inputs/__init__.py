"""Seeded synthetic inputs for the qsGW Sigma^c build (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only draws the input tensors of
``BASELINE.json: configs`` -- B in the MO basis, eps, occupations, Omega, Z, eta -- with the
shapes and value distributions stated there.  Both the CPU oracle's tests and the CUDA
path's tests take their inputs from here, and parity is always checked on ONE set of
arrays (one side generates, the other receives a copy): host- and device-generated
tensors of the same (config, seed) are both deterministic but are NOT equal to each
other, because torch's CPU and CUDA generators differ.

The inputs stand in for the paper's workloads -- linear alkanes CH4..C7H16 in cc-pVTZ,
N = 86..434 basis functions (Table III), full RPA with n_s = o*v -- which
need molecules, basis sets and MOLGW itself and are not available here.

Recipe (BASELINE.json configs, readings #8, #11):
  eps   : occupied ~ U[-1.5,-0.2] Ha, virtual ~ U[0.05,5.0] Ha, each sorted ascending, occupied first
  occ   : 1 for m < o, else 0
  Omega : U[0.2,6.0] Ha, sorted ascending
  B[P]  : (G + G^T)/2 with G_pq ~ N(0, 0.1^2) i.i.d.           shape [naux, N, N]
  Z     : N(0,1)/sqrt(n_s)                                      shape [o*v, n_s], row i*v+(a-o)
  eta   : 1e-3 Ha
Every tensor is a function of (seed, tensor tag, block index): B is drawn in blocks of
``B_BLOCK`` auxiliary functions and Z in blocks of ``Z_BLOCK`` poles, so any pole range of Z
can be produced without the rest and does not depend on how the range is partitioned.
"""
from __future__ import annotations

import dataclasses
import hashlib
import math
from typing import Dict, Optional

import torch

B_BLOCK = 16      # auxiliary functions per generator block of B
Z_BLOCK = 256     # poles per generator block of Z


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    n_mo: int
    n_occ: int
    n_aux: int
    n_pole: int
    s_block: int
    eta: float
    seed: int

    @property
    def n_virt(self) -> int:
        return self.n_mo - self.n_occ

    @property
    def n_ov(self) -> int:
        return self.n_occ * self.n_virt


# BASELINE.json: configs, verbatim (s_block 0 = "library default" where the config names none).
CONFIGS: Dict[str, Config] = {
    "tiny":   Config("tiny",   24,   5,   80,   95,     0,    1e-3, 0),
    "small":  Config("small",  120,  20,  400,  2000,   0,    1e-3, 1),
    "medium": Config("medium", 300,  40,  1100, 10400,  2048, 1e-3, 2),
    "large":  Config("large",  600,  80,  2400, 41600,  4096, 1e-3, 3),
    "xl":     Config("xl",     1000, 150, 4000, 127500, 4096, 1e-3, 4),
}


def custom_config(n_mo: int, n_occ: int, n_aux: int, n_pole: Optional[int] = None, s_block: int = 0,
                  eta: float = 1e-3, seed: int = 0, name: str = "custom") -> Config:
    if n_pole is None:
        n_pole = n_occ * (n_mo - n_occ)
    return Config(name, n_mo, n_occ, n_aux, n_pole, s_block, eta, seed)


def _seed_for(seed: int, tag: str, block: int) -> int:
    h = hashlib.sha256(f"qsgw-inputs/{seed}/{tag}/{block}".encode()).digest()
    return int.from_bytes(h[:8], "little") & 0x7FFFFFFFFFFFFFFF


def _gen(device, seed: int, tag: str, block: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(_seed_for(seed, tag, block))
    return g


def make_eps(cfg: Config) -> torch.Tensor:
    """[n_mo] QP energies (Ha), always drawn on the host (identical for every device)."""
    g = _gen("cpu", cfg.seed, "eps", 0)
    lo = torch.rand(cfg.n_occ, generator=g, dtype=torch.float64) * (-0.2 - (-1.5)) + (-1.5)
    hi = torch.rand(cfg.n_virt, generator=g, dtype=torch.float64) * (5.0 - 0.05) + 0.05
    return torch.cat([torch.sort(lo).values, torch.sort(hi).values])


def make_occ(cfg: Config) -> torch.Tensor:
    f = torch.zeros(cfg.n_mo, dtype=torch.float64)
    f[: cfg.n_occ] = 1.0
    return f


def make_omega(cfg: Config) -> torch.Tensor:
    """[n_pole] RPA excitation energies (Ha), sorted; always drawn on the host."""
    g = _gen("cpu", cfg.seed, "Omega", 0)
    om = torch.rand(cfg.n_pole, generator=g, dtype=torch.float64) * (6.0 - 0.2) + 0.2
    return torch.sort(om).values


def make_B(cfg: Config, device="cpu", out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """[n_aux, n_mo, n_mo] RI factors, symmetric in the last two indices (reading #11)."""
    N = cfg.n_mo
    if out is None:
        out = torch.empty((cfg.n_aux, N, N), dtype=torch.float64, device=device)
    for b0 in range(0, cfg.n_aux, B_BLOCK):
        b1 = min(b0 + B_BLOCK, cfg.n_aux)
        g = _gen(device, cfg.seed, "B", b0 // B_BLOCK)
        G = torch.randn((B_BLOCK, N, N), generator=g, dtype=torch.float64, device=device)[: b1 - b0]
        G.mul_(0.1)
        out[b0:b1] = 0.5 * (G + G.transpose(1, 2))
    return out


def make_Z(cfg: Config, s0: int = 0, s1: Optional[int] = None, device="cpu",
           out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """[n_ov, s1-s0] columns s0..s1 of Z = X+Y (row i*v+(a-o)); independent of the partition used."""
    if s1 is None:
        s1 = cfg.n_pole
    assert 0 <= s0 <= s1 <= cfg.n_pole
    if out is None:
        out = torch.empty((cfg.n_ov, s1 - s0), dtype=torch.float64, device=device)
    scale = 1.0 / math.sqrt(cfg.n_pole)
    for blk in range(s0 // Z_BLOCK, (s1 + Z_BLOCK - 1) // Z_BLOCK if s1 > s0 else 0):
        c0, c1 = blk * Z_BLOCK, (blk + 1) * Z_BLOCK
        g = _gen(device, cfg.seed, "Z", blk)
        blkvals = torch.randn((cfg.n_ov, Z_BLOCK), generator=g, dtype=torch.float64, device=device)
        lo, hi = max(c0, s0), min(c1, s1)
        out[:, lo - s0: hi - s0] = blkvals[:, lo - c0: hi - c0] * scale
    return out


@dataclasses.dataclass
class Inputs:
    cfg: Config
    B: torch.Tensor
    eps: torch.Tensor
    occ: torch.Tensor
    Omega: torch.Tensor
    Z: Optional[torch.Tensor]   # None when Z is produced range by range (xl)
    eta: float


def make_inputs(cfg: Config, device="cpu", with_Z: bool = True) -> Inputs:
    """All inputs of one Sigma^c build on `device` (eps, occ, Omega are drawn on the host and moved)."""
    return Inputs(
        cfg=cfg,
        B=make_B(cfg, device),
        eps=make_eps(cfg).to(device),
        occ=make_occ(cfg).to(device),
        Omega=make_omega(cfg).to(device),
        Z=make_Z(cfg, device=device) if with_Z else None,
        eta=cfg.eta,
    )


def flop_model(cfg: Config, n_pole: Optional[int] = None) -> Dict[str, float]:
    """Algorithmic FP64 flop counts of SURVEY.md 8(a)/(d) (2 flops per multiply-add)."""
    N, naux = cfg.n_mo, cfg.n_aux
    ns = cfg.n_pole if n_pole is None else n_pole
    f1 = 2.0 * naux * cfg.n_ov * ns
    f2 = 2.0 * N * N * naux * ns
    f2sym = 2.0 * (N * (N + 1) // 2) * naux * ns
    f3 = 2.0 * N ** 3 * ns
    return {"F1": f1, "F2": f2, "F2sym": f2sym, "F3": f3, "F_min": f1 + f2sym + f3, "F_full": f1 + f2 + f3}
