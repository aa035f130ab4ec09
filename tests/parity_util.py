"""Helpers shared by the GPU parity tests: run the CUDA path (through the C ABI binding) and the
fp64 oracle on the same seeded fp32 inputs and compare with BASELINE.json's metrics."""
from __future__ import annotations

import dataclasses

import numpy as np
import torch

from paper_1004_2503_b200 import workloads as wl

FIELDS = ("N", "Fx", "Fy", "Fz", "x", "T")


def gpu_run(w, n_steps, variant=None, tile=(0, 0), dt=None, chunks=None):
    """Run `n_steps` on the GPU; returns (dict of float32 numpy arrays, diag dict)."""
    from paper_1004_2503_b200 import aton
    a = aton.from_workload(w)
    if variant is not None:
        a.set_kernel(variant, *tile)
    if chunks:
        for c in chunks:
            a.step(dt or w.dt, c)
    else:
        a.step(dt or w.dt, n_steps)
    out = a.get_fields(device="cpu")
    diag = a.reduce()
    a.close()
    return {k: v.numpy() for k, v in out.items()}, diag


def oracle_run(orc, w, n_steps, dt=None, nH_mean=None):
    st, p = orc.from_workload(w, nH_mean)
    orc.step(st, p, dt or w.dt, n_steps, w.src_pos.numpy(), w.src_rate.numpy())
    return st, p


def state_to_workload(w, st):
    """Oracle state rounded to fp32 as a new workload (warm start handed to both codes, reading S17)."""
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32))
    return dataclasses.replace(w, x=t(st.x), T=t(st.T), N=t(st.N), Fx=t(st.Fx), Fy=t(st.Fy), Fz=t(st.Fz))


def max_rel_errors(g, st, c):
    """BASELINE.json 1-step metric: max relative error on N, x, T and |dF|/(cN) (reading S16),
    over cells with N > 1e-20 max N."""
    N = st.N
    m = N > 1e-20 * N.max()
    err = {}
    err["N"] = float(np.max(np.abs(g["N"][m] - N[m]) / N[m])) if m.any() else 0.0
    dF = np.sqrt((g["Fx"] - st.Fx) ** 2 + (g["Fy"] - st.Fy) ** 2 + (g["Fz"] - st.Fz) ** 2)
    err["F"] = float(np.max(dF[m] / (c * N[m]))) if m.any() else 0.0
    err["x"] = float(np.max(np.abs(g["x"] - st.x) / st.x))
    err["T"] = float(np.max(np.abs(g["T"] - st.T) / st.T))
    return err


def l1_errors(g, st, c):
    """BASELINE.json full-run metric: relative L1 error per field.  F is given twice: "F" against c*sum N (reading
    S16, the natural scale |F| <= cN) and "F_rel" against sum |F_ref| (the plain relative L1 of the flux itself)."""
    err = {}
    nsum = float(np.abs(st.N).sum())
    rel = lambda num: float(num / nsum) if nsum > 0 else (0.0 if num == 0 else float("inf"))   # dark region: exact zeros
    err["N"] = rel(np.abs(g["N"] - st.N).sum())
    dF = np.abs(g["Fx"] - st.Fx) + np.abs(g["Fy"] - st.Fy) + np.abs(g["Fz"] - st.Fz)
    err["F"] = rel(dF.sum() / c)
    fsum = float((np.abs(st.Fx) + np.abs(st.Fy) + np.abs(st.Fz)).sum())
    err["F_rel"] = float(dF.sum() / fsum) if fsum > 0 else (0.0 if dF.sum() == 0 else float("inf"))
    err["x"] = float(np.abs(g["x"] - st.x).sum() / np.abs(st.x).sum())
    err["T"] = float(np.abs(g["T"] - st.T).sum() / np.abs(st.T).sum())
    err["x_vol"] = float(abs(g["x"].astype(np.float64).mean() - st.x.mean()))
    return err


def twin(cfg, n, n_steps):
    """Down-sized twin of config `cfg` (same dx, density statistics and source density)."""
    return wl.make_config(cfg, n=n, n_steps=n_steps, norm_steps=n_steps)
