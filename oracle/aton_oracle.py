"""ctypes front end of the fp64 CPU oracle (oracle/aton_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "aton_oracle.c")
_LIB = os.path.join(_HERE, "libaton_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (+OpenMP over z-planes / cells)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [("c", C.c_double), ("dx", C.c_double), ("sigma_n", C.c_double),
                ("sigma_e", C.c_double), ("e_photon_eV", C.c_double), ("clump_a", C.c_double),
                ("clump_b", C.c_double), ("redshift", C.c_double), ("eps_sub", C.c_double),
                ("nH_mean", C.c_double), ("clump_i_a", C.c_double), ("clump_i_b", C.c_double),
                ("recomb_case", C.c_int), ("cooling", C.c_int),
                ("coll_ion", C.c_int), ("clump_model", C.c_int), ("max_sub", C.c_int), ("flux", C.c_int)]


class Rates(C.Structure):
    _fields_ = [(k, C.c_double) for k in
                ("alpha_A", "alpha_B", "beta", "z_recA", "z_recB", "z_ci", "z_exc", "z_ff",
                 "dl_recA", "dl_recB", "dl_ci", "dl_exc", "dl_ff")]


_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_chi.restype = C.c_double
        L.orc_chi.argtypes = [C.c_double]
        L.orc_closure.argtypes = [C.c_double, _dp, C.c_double, _dp]
        L.orc_transport.argtypes = [C.c_int] * 3 + [_dp] * 4 + [C.c_double] * 3 + [_dp] * 4
        L.orc_transport_hll.argtypes = [C.c_int] * 3 + [_dp] * 4 + [C.c_double] * 3 + [_dp] * 4
        L.orc_m1_wavespeeds.argtypes = [C.c_double, _dp, C.c_double, C.c_int, _dp, _dp]
        L.orc_flux_fn.argtypes = [C.c_int, C.c_double, _dp, C.c_double, _dp]
        L.orc_hll_flux.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, _dp]
        L.orc_inject.argtypes = [C.c_int] * 3 + [_dp, C.c_long, _dp, _dp, C.c_double, C.c_double]
        L.orc_rates.argtypes = [C.c_double, C.POINTER(Rates)]
        L.orc_clumping.restype = C.c_double
        L.orc_clumping.argtypes = [C.c_double, C.POINTER(Params)]
        L.orc_clumping_i.restype = C.c_double
        L.orc_clumping_i.argtypes = [C.c_double, C.POINTER(Params)]
        L.orc_chem_substep.restype = C.c_double
        L.orc_chem_substep.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, C.POINTER(Params)]
        L.orc_chem_cell.restype = C.c_int
        L.orc_chem_cell.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, C.POINTER(Params)]
        L.orc_chem_cell_trace.restype = C.c_int
        L.orc_chem_cell_trace.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, C.POINTER(Params), _dp, C.c_int]
        L.orc_cooling_probe.argtypes = [C.c_double] * 4 + [C.POINTER(Params), _dp]
        L.orc_chemistry.restype = C.c_longlong
        L.orc_chemistry.argtypes = [C.c_long] + [_dp] * 7 + [C.c_double, C.POINTER(Params),
                                                             C.POINTER(C.c_longlong)]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = ([C.c_int] * 3 + [_dp] * 7 + [C.c_long, _dp, _dp, C.c_double, C.c_int,
                                                            C.POINTER(Params), C.POINTER(C.c_longlong)])
        L.orc_reduce.argtypes = [C.c_long] + [_dp] * 7 + [C.POINTER(Params), _dp]
        L.orc_clumping_blocks.argtypes = [C.c_int] * 4 + [_dp] * 7
        L.orc_hist2d.argtypes = [C.c_long, _dp, _dp, C.c_int, C.c_int] + [C.c_double] * 4 + [C.c_int, C.c_int,
                                 C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
        L.orc_boost.restype = C.c_double
        L.orc_boost.argtypes = [C.c_double] * 3
        L.orc_star_rates.argtypes = [C.c_long, _dp, _dp, _dp] + [C.c_double] * 6 + [_dp]
        L.orc_thomson_tau.restype = C.c_double
        L.orc_thomson_tau.argtypes = [C.c_long, _dp, _dp, C.c_double, C.c_double, C.c_double]
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_get_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def make_params(params: Dict[str, float], dx: float, nH_mean: float = 1.0) -> Params:
    """params: dict with the keys of aton_params_t (include/aton.h); dx in cm."""
    c = params.get("c_cm_s", 0.0) or 2.99792458e10
    return Params(c=c, dx=dx, sigma_n=params["sigma_n"], sigma_e=params["sigma_e"],
                  e_photon_eV=params["e_photon_eV"], clump_a=params.get("clump_a", 1.0),
                  clump_b=params.get("clump_b", 2.0), redshift=params.get("redshift", -1.0),
                  eps_sub=params.get("eps_sub", 0.1) or 0.1, nH_mean=nH_mean,
                  clump_i_a=params.get("clump_i_a", 0.0), clump_i_b=params.get("clump_i_b", 0.0),
                  recomb_case=int(params.get("recomb_case", 1)), cooling=int(params.get("cooling", 1)),
                  coll_ion=int(params.get("coll_ion", 1)), clump_model=int(params.get("clump_model", 0)),
                  max_sub=int(params.get("max_sub", 1 << 14) or (1 << 14)), flux=int(params.get("flux", 0)))


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))


def get_threads() -> int:
    return int(lib().orc_get_threads())


def chi(f: float) -> float:
    return float(lib().orc_chi(float(f)))


def closure(N: float, F, c: float) -> np.ndarray:
    Fa = np.ascontiguousarray(F, dtype=np.float64)
    P = np.zeros(9)
    lib().orc_closure(float(N), _p(Fa), float(c), _p(P))
    return P.reshape(3, 3)


def transport(N, Fx, Fy, Fz, c: float, dx: float, dt: float):
    """One O2 step on [nz,ny,nx] float64 arrays; returns new (N,Fx,Fy,Fz)."""
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (N, Fx, Fy, Fz)]
    nz, ny, nx = a[0].shape
    o = [np.empty_like(a[0]) for _ in range(4)]
    lib().orc_transport(nx, ny, nz, *[_p(v) for v in a], c, dx, dt, *[_p(v) for v in o])
    return tuple(o)


def transport_hll(N, Fx, Fy, Fz, c: float, dx: float, dt: float):
    """One transport step with the HLL intercell flux on [nz,ny,nx] float64 arrays."""
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (N, Fx, Fy, Fz)]
    nz, ny, nx = a[0].shape
    o = [np.empty_like(a[0]) for _ in range(4)]
    lib().orc_transport_hll(nx, ny, nz, *[_p(v) for v in a], c, dx, dt, *[_p(v) for v in o])
    return tuple(o)


def m1_wavespeeds(N: float, F, c: float, d: int):
    """(lmin, lmax) of the M1 flux Jacobian in direction d (closed form)."""
    Fa = np.ascontiguousarray(F, dtype=np.float64)
    lo, hi = C.c_double(), C.c_double()
    lib().orc_m1_wavespeeds(float(N), _p(Fa), float(c), int(d), C.byref(lo), C.byref(hi))
    return lo.value, hi.value


def flux_fn(d: int, N: float, F, c: float) -> np.ndarray:
    """Physical flux (F_d, c^2 P_dx, c^2 P_dy, c^2 P_dz) of the 4 conserved variables through a face normal to d."""
    Fa = np.ascontiguousarray(F, dtype=np.float64)
    out = np.zeros(4)
    lib().orc_flux_fn(int(d), float(N), _p(Fa), float(c), _p(out))
    return out


def hll_flux(Ul, gl, Ur, gr, sm: float, sp: float) -> np.ndarray:
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (Ul, gl, Ur, gr)]
    out = np.zeros(4)
    lib().orc_hll_flux(*[_p(v) for v in a], float(sm), float(sp), _p(out))
    return out


def inject(N: np.ndarray, pos, rate, dt: float, dx: float) -> None:
    """In-place O3 on a [nz,ny,nx] float64 array."""
    nz, ny, nx = N.shape
    pos = np.ascontiguousarray(pos, dtype=np.float64).reshape(-1, 3)
    rate = np.ascontiguousarray(rate, dtype=np.float64)
    lib().orc_inject(nx, ny, nz, _p(N), len(rate), _p(pos), _p(rate), dt, dx)


def rates(T: float) -> Dict[str, float]:
    r = Rates()
    lib().orc_rates(float(T), C.byref(r))
    return {k: getattr(r, k) for k, _ in Rates._fields_}


def clumping(nH: float, p: Params) -> float:
    return float(lib().orc_clumping(float(nH), C.byref(p)))


def clumping_i(nH: float, p: Params) -> float:
    return float(lib().orc_clumping_i(float(nH), C.byref(p)))


def chem_substep(N: float, F, x: float, T: float, nH: float, dts: float, p: Params):
    """One backward-Euler sub-step; returns (N', F'[3], x', T', absorbed)."""
    n_, x_, t_ = C.c_double(N), C.c_double(x), C.c_double(T)
    Fa = np.array(F, dtype=np.float64)
    ab = lib().orc_chem_substep(C.byref(n_), _p(Fa), C.byref(x_), C.byref(t_), nH, dts, C.byref(p))
    return n_.value, Fa, x_.value, t_.value, float(ab)


def chem_cell(N: float, F, x: float, T: float, nH: float, dt: float, p: Params):
    """Sub-cycled operator Phi on one cell; returns (N', F'[3], x', T', n_sub)."""
    n_, x_, t_ = C.c_double(N), C.c_double(x), C.c_double(T)
    Fa = np.array(F, dtype=np.float64)
    ns = lib().orc_chem_cell(C.byref(n_), _p(Fa), C.byref(x_), C.byref(t_), nH, dt, C.byref(p))
    return n_.value, Fa, x_.value, t_.value, int(ns)


def chem_cell_trace(N: float, F, x: float, T: float, nH: float, dt: float, p: Params, cap: int = 4096):
    """chem_cell plus the (dts, N, x, T) at the start of every sub-step: returns (N', F', x', T', n_sub, trace[n,4])."""
    n_, x_, t_ = C.c_double(N), C.c_double(x), C.c_double(T)
    Fa = np.array(F, dtype=np.float64)
    tr = np.zeros((cap, 4))
    ns = lib().orc_chem_cell_trace(C.byref(n_), _p(Fa), C.byref(x_), C.byref(t_), nH, dt, C.byref(p), _p(tr), cap)
    return n_.value, Fa, x_.value, t_.value, int(ns), tr[:min(ns, cap)]


def cooling_probe(N: float, x: float, T: float, nH: float, p: Params) -> Dict[str, float]:
    """Lambda [erg cm^-3 s^-1], dLambda/dlnT and the net heating rate H - Lambda of the sub-step rule."""
    out = np.zeros(3)
    lib().orc_cooling_probe(float(N), float(x), float(T), float(nH), C.byref(p), _p(out))
    return {"Lambda": out[0], "Lambda_T": out[1], "edot": out[2]}


class State:
    """fp64 fields of one run, [nz,ny,nx] each."""

    def __init__(self, nH, x, T, N, Fx, Fy, Fz):
        self.nH, self.x, self.T, self.N, self.Fx, self.Fy, self.Fz = [
            np.array(v, dtype=np.float64, order="C", copy=True) for v in (nH, x, T, N, Fx, Fy, Fz)]
        self.sub_total = 0
        self.sub_max = 0

    @property
    def shape(self) -> Tuple[int, int, int]:
        return self.N.shape

    def copy(self) -> "State":
        return State(self.nH, self.x, self.T, self.N, self.Fx, self.Fy, self.Fz)


def chemistry(st: State, dt: float, p: Params) -> None:
    mx = C.c_longlong(0)
    tot = lib().orc_chemistry(st.N.size, _p(st.N), _p(st.Fx), _p(st.Fy), _p(st.Fz), _p(st.x),
                              _p(st.T), _p(st.nH), dt, C.byref(p), C.byref(mx))
    st.sub_total += int(tot)
    st.sub_max = max(st.sub_max, int(mx.value))


def step(st: State, p: Params, dt: float, n_steps: int, src_pos=None, src_rate=None) -> None:
    """O6: n_steps of transport -> inject -> chemistry, in place."""
    nz, ny, nx = st.shape
    if src_rate is None or len(src_rate) == 0:
        pos = np.zeros((1, 3)); rate = np.zeros(1); ns = 0
    else:
        pos = np.ascontiguousarray(src_pos, dtype=np.float64).reshape(-1, 3)
        rate = np.ascontiguousarray(src_rate, dtype=np.float64)
        ns = len(rate)
    stats = (C.c_longlong * 2)(0, 0)
    rc = lib().orc_step(nx, ny, nz, _p(st.N), _p(st.Fx), _p(st.Fy), _p(st.Fz), _p(st.x), _p(st.T),
                        _p(st.nH), ns, _p(pos), _p(rate), dt, n_steps, C.byref(p), stats)
    if rc != 0:
        raise MemoryError("orc_step: scratch allocation failed")
    st.sub_total += int(stats[0])
    st.sub_max = max(st.sub_max, int(stats[1]))


def reduce(st: State, p: Params) -> Dict[str, float]:
    out = np.zeros(10)
    lib().orc_reduce(st.N.size, _p(st.N), _p(st.Fx), _p(st.Fy), _p(st.Fz), _p(st.x), _p(st.T),
                     _p(st.nH), C.byref(p), _p(out))
    keys = ("x_vol", "x_mass", "gamma_vol", "gamma_mass", "photons_total", "T_vol", "f_max",
            "N_min", "n_nonfinite", "frac_x_half")
    return dict(zip(keys, out.tolist()))


def clumping_blocks(nH, x, N, b: int = 8) -> Dict[str, np.ndarray]:
    """Clumping-factor measurement over b^3 blocks: dict of [nz/b, ny/b, nx/b] arrays."""
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (nH, x, N)]
    nz, ny, nx = a[0].shape
    shape = (nz // b, ny // b, nx // b)
    out = [np.zeros(shape) for _ in range(4)]
    lib().orc_clumping_blocks(nx, ny, nz, b, *[_p(v) for v in a], *[_p(v) for v in out])
    return dict(zip(("nH", "x", "C_R", "C_I"), out))


def hist2d(a, b, log_a: bool, log_b: bool, a_range, b_range, na: int, nb: int):
    """2-D histogram counts[nb, na] and the number of values outside the ranges."""
    va = np.ascontiguousarray(a, dtype=np.float64).reshape(-1)
    vb = np.ascontiguousarray(b, dtype=np.float64).reshape(-1)
    counts = np.zeros((nb, na), dtype=np.int64)
    outside = C.c_longlong(0)
    lib().orc_hist2d(va.size, _p(va), _p(vb), int(log_a), int(log_b), float(a_range[0]), float(a_range[1]),
                     float(b_range[0]), float(b_range[1]), na, nb,
                     counts.ctypes.data_as(C.POINTER(C.c_longlong)), C.byref(outside))
    return counts, int(outside.value)


def boost(t: float, a_b: float, k_b: float) -> float:
    return float(lib().orc_boost(float(t), float(a_b), float(k_b)))


def star_rates(age1, life, nbaryons, photons_per_baryon, t_p, t_p1, f_esc, a_b, k_b) -> np.ndarray:
    """Effective emission rates of star particles over [t_p, t_p1] (section 2.3, Eq.8-9)."""
    a = [np.ascontiguousarray(v, dtype=np.float64) for v in (age1, life, nbaryons)]
    out = np.zeros(a[0].size)
    lib().orc_star_rates(a[0].size, *[_p(v) for v in a], float(photons_per_baryon), float(t_p), float(t_p1),
                         float(f_esc), float(a_b), float(k_b), _p(out))
    return out


def thomson_tau(z, x, nH0: float, H0: float, Om: float) -> float:
    zz, xx = [np.ascontiguousarray(v, dtype=np.float64) for v in (z, x)]
    return float(lib().orc_thomson_tau(zz.size, _p(zz), _p(xx), float(nH0), float(H0), float(Om)))


def from_workload(w, nH_mean: Optional[float] = None):
    """(State, Params) from a paper_1004_2503_b200.workloads.Workload (fp32 inputs up-cast)."""
    st = State(*[t.detach().cpu().numpy() for t in w.fields()])
    mean = float(st.nH.mean()) if nH_mean is None else nH_mean
    return st, make_params(w.params, w.dx, mean)
