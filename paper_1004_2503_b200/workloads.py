"""Seeded synthetic inputs for the ATON hot path (the five BASELINE.json configs).

This module is the ONLY code shared by the CUDA path and the CPU oracle's tests.  It holds no
radiative-transfer or chemistry arithmetic: it only builds input fields (gas density, initial
x/T/N/F, source lists) and the run parameters of each config.  It imports neither the CUDA binding
nor anything under ``oracle/``.

The paper's inputs are RAMSES snapshots (§2.1, L133 Table 1) that are not
available; the recipes below (restated in DESIGN.md "Input recipe") stand in for
them: log-normal density fields with a power-law spectrum spanning the paper's density range
(PAPER.md:L215-217), sources on density peaks projected NGP, one emitter per cell.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional

import torch

# Physical constants used only to define the workloads (box sizes, the Courant step).
C_CM_S = 2.99792458e10
KPC_CM = 3.0856775814913673e21
MPC_CM = 1.0e3 * KPC_CM
HUBBLE_h = 0.72  # WMAP-5-like; reading S14 in DESIGN.md
SEED_BASE = 10042503


@dataclasses.dataclass
class Workload:
    """One fully specified run: grid, physics switches, initial fields, sources, step plan."""
    name: str
    n: int                      # cells per side (cubic grid)
    box_cm: float               # physical side length
    params: Dict[str, float]    # keys mirror aton_params_t in include/aton.h
    nH: torch.Tensor            # [n,n,n] float32, cm^-3, C-order [z][y][x]
    x: torch.Tensor             # ionised fraction
    T: torch.Tensor             # K
    N: torch.Tensor             # photons cm^-3
    Fx: torch.Tensor            # photons cm^-2 s^-1
    Fy: torch.Tensor
    Fz: torch.Tensor
    src_pos: torch.Tensor       # [ns,3] float32, box units in [0,1), (x,y,z)
    src_rate: torch.Tensor      # [ns] float64, photons/s
    dt: float                   # s
    n_steps: int

    @property
    def dx(self) -> float:
        return self.box_cm / self.n

    def fields(self):
        return (self.nH, self.x, self.T, self.N, self.Fx, self.Fy, self.Fz)


def courant_dt(dx_cm: float, courant: float = 0.8, c: float = C_CM_S) -> float:
    """dt = courant * dx / (3c): reading S3 (unsplit 3-D LF is stable only for c dt/dx <= 1/3)."""
    return courant * dx_cm / (3.0 * c)


def default_params() -> Dict[str, float]:
    """PAPER.md:L89 single-group constants; every switch off except case-B recombination."""
    return dict(c_cm_s=C_CM_S, sigma_n=2.93e-18, sigma_e=2.49e-18, e_photon_eV=20.27,
                recomb_case=1, cooling=1, coll_ion=1, clump_model=0, clump_a=1.0, clump_b=2.0,
                redshift=-1.0, eps_sub=0.1, max_sub=1 << 14, clump_i_a=0.0, clump_i_b=0.0, flux=0)


# ----------------------------------------------------------------------------------------------
# Gaussian random field -> log-normal density
# ----------------------------------------------------------------------------------------------
def gaussian_field(n: int, slope: float, gen: torch.Generator, device="cpu") -> torch.Tensor:
    """Unit-variance, zero-mean periodic Gaussian field with P(k) ~ k^-slope on an n^3 grid.

    white noise -> rFFT -> multiply by k^(-slope/2), k=0 zeroed -> irFFT -> normalise.
    """
    w = torch.randn((n, n, n), generator=gen, device=device, dtype=torch.float32)
    wk = torch.fft.rfftn(w)
    del w
    kf = torch.fft.fftfreq(n, d=1.0 / n, device=device)
    kr = torch.fft.rfftfreq(n, d=1.0 / n, device=device)
    k2 = (kf[:, None, None] ** 2 + kf[None, :, None] ** 2 + kr[None, None, :] ** 2)
    k2[0, 0, 0] = 1.0
    amp = k2.pow(-0.25 * slope)
    amp[0, 0, 0] = 0.0
    del k2
    wk *= amp
    del amp
    g = torch.fft.irfftn(wk, s=(n, n, n))
    del wk
    g -= g.mean()
    g /= g.double().pow(2).mean().sqrt().float()
    return g


def lognormal_density(n: int, slope: float, sigma_ln: float, nbar: float,
                      gen: torch.Generator, device="cpu") -> torch.Tensor:
    """n_H = nbar * exp(sigma*g - sigma^2/2), then rescaled so the mean is exactly nbar."""
    g = gaussian_field(n, slope, gen, device)
    nH = torch.exp(sigma_ln * g - 0.5 * sigma_ln * sigma_ln)
    del g
    nH *= (1.0 / nH.double().mean()).float()
    nH *= nbar
    return nH.contiguous()


def _cell_centres(idx_flat: torch.Tensor, n: int) -> torch.Tensor:
    """flat index i + n*(j + n*k) -> positions ((i+.5)/n, (j+.5)/n, (k+.5)/n) in box units."""
    i = idx_flat % n
    j = (idx_flat // n) % n
    k = idx_flat // (n * n)
    pos = torch.stack([i, j, k], dim=1).to(torch.float32)
    return ((pos + 0.5) / n).contiguous()


def _local_maxima_top(nH: torch.Tensor, count: int) -> torch.Tensor:
    """Flat indices of the `count` densest strict 26-neighbour local maxima (periodic)."""
    n = nH.shape[0]
    ismax = torch.ones_like(nH, dtype=torch.bool)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                if dz == 0 and dy == 0 and dx == 0:
                    continue
                ismax &= nH > torch.roll(nH, shifts=(dz, dy, dx), dims=(0, 1, 2))
    idx = torch.nonzero(ismax.reshape(-1), as_tuple=False).reshape(-1)
    del ismax
    vals = nH.reshape(-1)[idx]
    if idx.numel() < count:
        raise ValueError(f"only {idx.numel()} local maxima, need {count}")
    top = torch.topk(vals, count, sorted=True).indices
    return idx[top]


def _rates_overdensity(nH: torch.Tensor, idx: torch.Tensor, nbar: float, dx: float,
                       total_time: float) -> torch.Tensor:
    """rate ~ overdensity^1.5, normalised to one photon per H atom over the run (reading S15)."""
    delta = (nH.reshape(-1)[idx].double() / nbar)
    wgt = delta.pow(1.5)
    n_atoms = float(nH.double().sum()) * dx ** 3
    return (wgt / wgt.sum() * (n_atoms / total_time)).cpu()


def _dark_start(nH: torch.Tensor, x0: float, T0: float):
    z = torch.zeros_like(nH)
    return (torch.full_like(nH, x0), torch.full_like(nH, T0), z, z.clone(), z.clone(), z.clone())


# ----------------------------------------------------------------------------------------------
# The five configs
# ----------------------------------------------------------------------------------------------
_CFG = {
    # id: (n, comoving Mpc/h, z, slope, sigma_ln, nbar, n_sources, n_steps)
    2: (128, 1.0, 9.0, 2.0, 1.5, 2.0e-4, 64, 1000),
    3: (256, 12.5, 9.0, 2.5, 2.0, 1.9e-7 * 10.0 ** 3, 2000, 2000),
    4: (512, 25.0, 8.0, 2.5, 2.2, 1.9e-7 * 9.0 ** 3, 20000, 1000),
    5: (1024, 100.0, 7.0, 2.5, 2.5, 1.9e-7 * 8.0 ** 3, 200000, 200),
}


def make_config(cfg: int, n: Optional[int] = None, device="cpu", seed: Optional[int] = None,
                n_steps: Optional[int] = None, norm_steps: Optional[int] = None) -> Workload:
    """Build BASELINE.json config `cfg` (1..5).

    `n` overrides the grid size to make a down-sized twin: same cell size dx, same density
    statistics, same number of sources per cell (at least 1), so a full run fits the CPU oracle.
    `norm_steps` (configs 3-5) is the number of steps over which the sources emit one photon per
    H atom (reading S15; default: the config's full step count) -- a short twin run can so reach
    the same half-reionised end state as the full run.
    """
    if cfg == 1:
        return _config1(n or 32, device, n_steps)
    if cfg not in _CFG:
        raise ValueError("cfg must be 1..5")
    n_full, lcom, z, slope, sigma_ln, nbar, ns_full, steps_full = _CFG[cfg]
    n = n or n_full
    dx = lcom * MPC_CM / HUBBLE_h / (1.0 + z) / n_full   # physical cell size of the full config
    box = dx * n
    gen = torch.Generator(device=device)
    gen.manual_seed(seed if seed is not None else SEED_BASE + cfg)
    nH = lognormal_density(n, slope, sigma_ln, nbar, gen, device)
    ns = max(1, int(round(ns_full * (n / n_full) ** 3)))
    steps = n_steps or steps_full
    dt = courant_dt(dx)
    p = default_params()
    flat = nH.reshape(-1)
    if cfg == 2:
        # 64 cells, probability ~ n_H, without replacement; rates log-uniform in [1e49, 1e51]
        idx = torch.multinomial(flat.double() / flat.double().sum(), ns, replacement=False,
                                generator=gen)
        u = torch.rand(ns, generator=gen, device=device, dtype=torch.float64)
        rate = (10.0 ** (49.0 + 2.0 * u)).cpu()
    elif cfg == 3:
        # uniform draw among cells above the 95th density percentile
        kth = int(0.95 * flat.numel())
        thr = torch.kthvalue(flat, kth).values
        cand = torch.nonzero(flat > thr, as_tuple=False).reshape(-1)
        perm = torch.randperm(cand.numel(), generator=gen, device=device)[:ns]
        idx = cand[perm]
        rate = _rates_overdensity(nH, idx, nbar, dx, (norm_steps or steps_full) * dt)
    else:
        idx = _local_maxima_top(nH, ns)
        rate = _rates_overdensity(nH, idx, nbar, dx, (norm_steps or steps_full) * dt)
        # case-A rates + recombination radiation, collisional ionisation, cooling, C_R = max(1, 1+2 delta)
        p.update(recomb_case=0, clump_model=1, clump_a=1.0, clump_b=2.0, redshift=z)
    if cfg in (2, 3):
        p.update(redshift=z)
    pos = _cell_centres(idx, n).cpu()
    x, T, N, Fx, Fy, Fz = _dark_start(nH, 1.0e-3, 100.0)
    return Workload(f"cfg{cfg}_{n}", n, box, p, nH, x, T, N, Fx, Fy, Fz, pos,
                    rate.to(torch.float64), dt, steps)


def _config1(n: int, device, n_steps) -> Workload:
    """32^3, 6.6 kpc box, uniform n_H = 1e-3, one 5e48 /s source in the corner cell (0,0,0)."""
    box = 6.6 * KPC_CM
    dx = box / 32.0
    nH = torch.full((n, n, n), 1.0e-3, dtype=torch.float32, device=device)
    p = default_params()
    p.update(sigma_n=1.63e-18, sigma_e=1.63e-18, e_photon_eV=29.6)
    x, T, N, Fx, Fy, Fz = _dark_start(nH, 1.2e-3, 100.0)
    pos = torch.tensor([[0.5 / n, 0.5 / n, 0.5 / n]], dtype=torch.float32)
    rate = torch.tensor([5.0e48], dtype=torch.float64)
    return Workload(f"cfg1_{n}", n, dx * n, p, nH, x, T, N, Fx, Fy, Fz, pos, rate,
                    courant_dt(dx), n_steps or 500)


def stromgren_twin(n: int = 32, device="cpu") -> Workload:
    """Scaled Stroemgren set-up: isothermal 1e4 K, case B, no collisional ionisation,
    n_H = 1, Q and dx chosen so that R_s = 10 cells and t_rec = 2000 steps; source at the centre."""
    alpha_B = 2.59e-13          # cm^3/s at 1e4 K (textbook value; the oracle's own fit is pinned to it)
    nH0 = 1.0
    t_rec = 1.0 / (alpha_B * nH0)
    dt = t_rec / 2000.0
    dx = dt * 3.0 * C_CM_S / 0.8
    Q = 4.0 / 3.0 * math.pi * (10.0 * dx) ** 3 * alpha_B * nH0 ** 2
    nH = torch.full((n, n, n), nH0, dtype=torch.float32, device=device)
    p = default_params()
    p.update(sigma_n=1.63e-18, sigma_e=1.63e-18, e_photon_eV=29.6, cooling=0, coll_ion=0)
    x, T, N, Fx, Fy, Fz = _dark_start(nH, 1.0e-6, 1.0e4)
    c0 = (n // 2 + 0.5) / n
    pos = torch.tensor([[c0, c0, c0]], dtype=torch.float32)
    return Workload(f"stromgren_{n}", n, dx * n, p, nH, x, T, N, Fx, Fy, Fz, pos,
                    torch.tensor([Q], dtype=torch.float64), dt, 8000)


# ----------------------------------------------------------------------------------------------
# Synthetic warm state: a plausible mid-reionisation state built directly (no RT arithmetic),
# so that large grids can be parity-checked on sub-cubes without running either code first.
# ----------------------------------------------------------------------------------------------
def synthetic_warm_state(w: Workload, seed: int = 7, device=None) -> Workload:
    """Replace the dark start of `w` by smooth random, realizable (|F| <= 0.9 cN) fields:
    ionised bubbles (x from a thresholded Gaussian field), hot where ionised, photons mostly inside
    bubbles, fluxes with random smooth directions and reduced flux in [0, 0.9)."""
    device = device or w.nH.device
    n = w.n
    gen = torch.Generator(device=device)
    gen.manual_seed(SEED_BASE * 3 + seed)
    g1 = gaussian_field(n, 3.0, gen, device)
    x = torch.sigmoid(4.0 * g1 + 0.5)
    x = (1.0e-3 + (0.99999 - 1.0e-3) * x).float()
    g2 = gaussian_field(n, 2.0, gen, device)
    T = (100.0 + 2.0e4 * x * torch.exp(0.3 * g2)).float()
    g3 = gaussian_field(n, 2.5, gen, device)
    nbar = float(w.nH.double().mean())
    N = (0.05 * nbar * (0.02 + x) * torch.exp(1.5 * g3)).float()
    del g2, g3
    f = 0.9 * torch.sigmoid(2.0 * gaussian_field(n, 2.0, gen, device))
    d = [gaussian_field(n, 3.0, gen, device) for _ in range(3)]
    norm = torch.sqrt(d[0] ** 2 + d[1] ** 2 + d[2] ** 2).clamp_min(1e-12)
    c = w.params["c_cm_s"]
    Fx, Fy, Fz = [(c * N * f * di / norm).float().contiguous() for di in d]
    return dataclasses.replace(w, name=w.name + "_warm", x=x.contiguous(), T=T.contiguous(),
                               N=N.contiguous(), Fx=Fx, Fy=Fy, Fz=Fz)


def cut_subcube(t: torch.Tensor, origin, size: int) -> torch.Tensor:
    """Periodic sub-cube t[z0:z0+size, y0:y0+size, x0:x0+size] (origin = (x0,y0,z0)), on CPU."""
    n = t.shape[0]
    x0, y0, z0 = origin
    iz = (torch.arange(size, device=t.device) + z0) % n
    iy = (torch.arange(size, device=t.device) + y0) % n
    ix = (torch.arange(size, device=t.device) + x0) % n
    return t[iz][:, iy][:, :, ix].contiguous().cpu()
