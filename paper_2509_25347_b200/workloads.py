"""Seeded synthetic inputs shaped like the paper's runs (BASELINE.json `configs`; recipe in DESIGN.md §4).

This module holds NONE of the method's arithmetic: it only draws the per-cell input fields
(rho_g, rho_d, t_s, p_in, dt) that both the CUDA path and the CPU oracle consume.  It depends on torch only
(CPU or CUDA generator), and is imported by tests/, bench.py and __graft_entry__.py.

Layouts (include/dg.h): rho_g[ncells], rho_d[N][ncells], t_s[N][ncells], p_in[3][n][ncells], n = N+1,
cell index fastest, species 0 = gas.
"""
import math
from dataclasses import dataclass

import torch

CONFIG_CELLS = {1: 32 ** 3, 2: 128 ** 3, 3: 256 ** 3, 4: 256 ** 3, 5: 2 ** 22}
CONFIG_N = {1: 1, 2: 4, 3: 8, 4: 16}
SWEEP_N = (1, 2, 4, 8, 12, 16)


@dataclass
class Workload:
    name: str
    config: int
    N: int
    ncells: int
    dt: float
    rho_g: torch.Tensor
    rho_d: torch.Tensor
    t_s: torch.Tensor
    p_in: torch.Tensor

    @property
    def n(self):
        return self.N + 1

    def cells(self, idx):
        """Host float64 numpy copies of the selected cells (for the oracle)."""
        idx = torch.as_tensor(idx, device=self.rho_g.device, dtype=torch.long)
        return (self.rho_g[idx].cpu().numpy(), self.rho_d[:, idx].cpu().numpy(), self.t_s[:, idx].cpu().numpy(),
                self.p_in[:, :, idx].cpu().numpy())


def _uniform(shape, lo, hi, gen, device):
    return torch.rand(shape, generator=gen, device=device, dtype=torch.float64) * (hi - lo) + lo


def _loguniform(shape, lo, hi, gen, device):
    return torch.pow(10.0, _uniform(shape, math.log10(lo), math.log10(hi), gen, device))


def _normal(shape, std, gen, device):
    return torch.randn(shape, generator=gen, device=device, dtype=torch.float64) * std


def make_workload(config: int, ncells: int = None, N: int = None, device="cpu", seed: int = 0) -> Workload:
    """config 1..4 = BASELINE.json configs[0..3]; config 5 = the species sweep (give N; generator of config 4).

    `ncells` overrides the config's cell count (parity tests use reduced sizes of the same recipe).
    Generator seed = seed + config (reading R15).
    """
    if config not in CONFIG_CELLS:
        raise ValueError("config must be 1..5")
    if config == 5:
        if N is None:
            raise ValueError("config 5 (sweep) needs N")
    else:
        N = CONFIG_N[config] if N is None else N
    ncells = CONFIG_CELLS[config] if ncells is None else int(ncells)
    dev = torch.device(device)
    gen = torch.Generator(device=dev)
    gen.manual_seed(seed + config)
    n = N + 1
    if config == 1:
        dt = 0.1
        rho_g = torch.ones(ncells, dtype=torch.float64, device=dev)
        eps = _uniform((N, ncells), 0.01, 1.0, gen, dev)
        t_s = _uniform((N, ncells), 0.01, 1.0, gen, dev)
        p_in = _normal((3, n, ncells), 1.0, gen, dev)
    elif config == 2:
        dt = 1e-2
        rho_g = _loguniform((ncells,), 1e-2, 1e2, gen, dev)
        eps = _loguniform((N, ncells), 1e-3, 1.0, gen, dev)
        t_s = _loguniform((N, ncells), 1e-3, 10.0, gen, dev)
        p_in = _normal((3, n, ncells), 1.0, gen, dev)
    elif config == 3:
        dt = 1e-2
        rho_g = torch.ones(ncells, dtype=torch.float64, device=dev)
        # stopping times geometrically spaced over [1e-4, 1] with +-10 % per-cell jitter
        expo = torch.arange(N, dtype=torch.float64, device=dev) / max(N - 1, 1)
        t0 = 1e-4 * torch.pow(torch.tensor(1e4, dtype=torch.float64, device=dev), expo)
        t_s = t0[:, None] * (1.0 + 0.1 * _uniform((N, ncells), -1.0, 1.0, gen, dev))
        # MRN-like power-law weights w_i ~ sqrt(T_s,i) (Eq. 31), dust-to-gas ratios summing to 0.01
        w = torch.sqrt(t0)
        eps = (0.01 * w / w.sum())[:, None].expand(N, ncells).contiguous()
        # sinusoidal wave (wavenumber 2 pi) along x on component 0 + normal(0, 1e-3) noise on all components
        nx = round(ncells ** (1.0 / 3.0))
        if nx ** 3 != ncells:
            nx = ncells
        ix = torch.arange(ncells, device=dev) % nx
        wave = torch.sin(2.0 * math.pi * (ix.to(torch.float64) + 0.5) / nx)
        rho = torch.cat([rho_g[None, :], eps * rho_g[None, :]], dim=0)
        p_in = _normal((3, n, ncells), 1e-3, gen, dev)
        p_in[0] += rho * wave[None, :]
    else:  # 4 and the sweep
        dt = 1e-2
        rho_g = torch.ones(ncells, dtype=torch.float64, device=dev)
        eps = _loguniform((N, ncells), 1e-4, 10.0, gen, dev)
        t_s = _loguniform((N, ncells), 1e-6, 1e2, gen, dev)
        p_in = _normal((3, n, ncells), 1.0, gen, dev)
    rho_d = (eps * rho_g[None, :]).contiguous()
    name = f"config{config}_N{N}_{ncells}cells"
    return Workload(name=name, config=config, N=N, ncells=ncells, dt=dt, rho_g=rho_g.contiguous(), rho_d=rho_d,
                    t_s=t_s.contiguous(), p_in=p_in.contiguous())


def sample_cells(ncells: int, nsample: int, seed: int = 0):
    """Deterministic strided subsample of cell indices (sorted, unique), always containing cell 0 and the last cell."""
    if nsample >= ncells:
        return torch.arange(ncells)
    stride = ncells / nsample
    idx = (torch.arange(nsample, dtype=torch.float64) * stride).long()
    idx[-1] = ncells - 1
    return torch.unique(idx)
