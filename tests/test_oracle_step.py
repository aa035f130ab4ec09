"""Pins of the oracle's whole step (O3 injection, O5 diagnostics, O6 loop) against closed forms:
Stroemgren sphere growth (P7), first step from vacuum (P8), cube symmetry (P9), photon counting."""
import math

import numpy as np
import pytest

from paper_1004_2503_b200 import workloads as wl

C = wl.C_CM_S


def test_inject_ngp_semantics(orc):
    """S11: cell = floor(pos*n) mod n per axis; duplicates add; N += rate*dt/dx^3 (L103, L428)."""
    n = 4
    N = np.zeros((n, n, n))
    pos = np.array([[0.0, 0.0, 0.0], [0.25, 0.5, 0.75], [0.2499999, 0.5, 0.75],
                    [0.999999, 0.999999, 0.999999], [0.25, 0.5, 0.75], [1.0, 0.0, 0.0]])
    rate = np.array([1.0, 2.0, 4.0, 8.0, 16.0, 32.0])
    dt, dx = 3.0, 2.0
    orc.inject(N, pos, rate, dt, dx)
    k = dt / dx ** 3
    want = np.zeros_like(N)
    want[0, 0, 0] = (1.0 + 32.0) * k          # pos = 1.0 wraps to cell 0
    want[3, 2, 1] = (2.0 + 16.0) * k          # [z][y][x] = [3][2][1]
    want[3, 2, 0] = 4.0 * k
    want[3, 3, 3] = 8.0 * k
    assert np.array_equal(N, want)


def test_first_step_from_vacuum(orc):
    """P8 / S10: from a dark start only the source cell holds photons after one step, and its
    state is Phi applied to N = rate*dt/dx^3; every other cell just recombines."""
    w = wl.make_config(1, n=8)
    st, p = orc.from_workload(w)
    orc.step(st, p, w.dt, 1, w.src_pos.numpy(), w.src_rate.numpy())
    N0 = 5e48 * w.dt / w.dx ** 3
    x0, nH0 = float(w.x[0, 0, 0]), float(w.nH[0, 0, 0])          # fp32 inputs, up-cast
    Nn, Fn, xn, Tn, ns = orc.chem_cell(N0, [0, 0, 0], x0, 100.0, nH0, w.dt, p)
    assert st.N[0, 0, 0] == Nn and st.x[0, 0, 0] == xn and st.T[0, 0, 0] == Tn
    assert st.sub_max == ns and ns > 1
    mask = np.ones(st.N.shape, bool); mask[0, 0, 0] = False
    assert np.all(st.N[mask] == 0) and np.all(st.Fx == 0)
    _, _, xd, Td, _ = orc.chem_cell(0.0, [0, 0, 0], x0, 100.0, nH0, w.dt, p)
    assert np.all(st.x[mask] == xd) and np.all(st.T[mask] == Td) and xd < x0


def test_cube_symmetry(orc):
    """P9: a source at the centre cell of a uniform box gives fields invariant under the axis
    permutations and reflections of the cube (odd parity for the matching flux component)."""
    n = 9
    w = wl.make_config(1, n=n)
    c0 = (n // 2 + 0.5) / n
    st, p = orc.from_workload(w)
    orc.step(st, p, w.dt, 12, np.array([[c0, c0, c0]]), w.src_rate.numpy())
    N = st.N
    assert N.min() >= 0 and N[n // 2, n // 2, n // 2] == N.max()
    for perm in ((0, 2, 1), (1, 0, 2), (2, 1, 0), (1, 2, 0)):
        assert np.allclose(N.transpose(perm), N, rtol=1e-12, atol=0)
        assert np.allclose(st.x.transpose(perm), st.x, rtol=1e-12)
    assert np.allclose(N[::-1], N, rtol=1e-12) and np.allclose(N[:, :, ::-1], N, rtol=1e-12)
    assert np.allclose(st.Fx[:, :, ::-1], -st.Fx, rtol=1e-10, atol=1e-12 * C * N.max())
    assert np.allclose(st.Fz.transpose(2, 1, 0), st.Fx, rtol=1e-10, atol=1e-12 * C * N.max())
    # photons stream outwards
    assert st.Fx[n // 2, n // 2, n // 2 + 2] > 0 > st.Fx[n // 2, n // 2, n // 2 - 2]


def test_config1_early_photon_counting(orc):
    """P7 early-time law at config 1: 500 steps = 7e-4 t_rec, so (new ionised atoms + photons in the
    box) = Q t to within the small recombination/collisional corrections (0.99998 ->
    1.02), and the ionised volume matches R(t) = R_s (1-exp(-t/t_rec))^(1/3) ~ (3 Q t/(4 pi nH))^(1/3)."""
    w = wl.make_config(1)
    st, p = orc.from_workload(w)
    pos, rate = w.src_pos.numpy(), w.src_rate.numpy()
    x0 = 1.2e-3
    budget = []
    done = 0
    for upto in (1, 100, 500):
        orc.step(st, p, w.dt, upto - done, pos, rate)
        done = upto
        ion = ((st.x - x0) * st.nH).sum() * w.dx ** 3
        phot = st.N.sum() * w.dx ** 3
        budget.append((ion + phot) / (5e48 * upto * w.dt))
    assert budget[0] == pytest.approx(1.0, abs=2e-4)
    assert 0.99 < budget[1] < 1.03 and 0.99 < budget[2] < 1.05
    V_cells = (st.x - x0).sum() / (1 - x0)
    R_cells = (3 * V_cells / (4 * math.pi)) ** (1 / 3)
    alpha_B = 2.59e-13
    t = 500 * w.dt
    R_s = (3 * 5e48 / (4 * math.pi * alpha_B * 1e-6)) ** (1 / 3)
    R_t = R_s * (1 - math.exp(-t * alpha_B * 1e-3)) ** (1 / 3) / w.dx
    assert R_s / wl.KPC_CM == pytest.approx(5.4, rel=0.01)            # north_star's closed form
    assert R_cells == pytest.approx(R_t, rel=0.03)
    d = orc.reduce(st, p)
    assert d["n_nonfinite"] == 0 and d["f_max"] <= 1 + 1e-12 and d["N_min"] >= 0


@pytest.mark.slow
def test_stromgren_sphere_growth(orc):
    """P7: isothermal 1e4 K, case B, no collisional ionisation, uniform gas, one source:
    V_ion(t) = Q/(alpha_B nH^2) (1 - exp(-t/t_rec)).  Scaled twin: R_s = 10 cells, t_rec = 2000
    steps.  Tolerance 5 % on R (finite front width, as in the comparison-project literature)."""
    w = wl.stromgren_twin(32)
    st, p = orc.from_workload(w)
    alpha_B = orc.rates(1e4)["alpha_B"]
    assert alpha_B == pytest.approx(2.59e-13, rel=2e-3)
    Q = float(w.src_rate[0])
    t_rec = 1.0 / (alpha_B * 1.0)
    pos, rate = w.src_pos.numpy(), w.src_rate.numpy()
    done = 0
    for upto in (500, 1000, 2000, 4000, 8000):
        orc.step(st, p, w.dt, upto - done, pos, rate)
        done = upto
        t = upto * w.dt
        V = st.x.sum() * w.dx ** 3
        V_an = Q / alpha_B * (1 - math.exp(-t / t_rec))
        assert (V / V_an) ** (1 / 3) == pytest.approx(1.0, abs=0.05), (upto, V / V_an)
    R = (3 * st.x.sum() / (4 * math.pi)) ** (1 / 3)
    assert R == pytest.approx(10.0, rel=0.05)                           # R_s = 10 cells
    # sphericity: the front radius along an axis and along the diagonal agree within a cell
    c = 16
    prof_axis = st.x[c, c, c:]
    r_axis = np.interp(0.5, prof_axis[::-1], np.arange(len(prof_axis))[::-1])
    diag = np.array([st.x[c + i, c + i, c + i] for i in range(12)])
    r_diag = np.interp(0.5, diag[::-1], (np.arange(12) * math.sqrt(3))[::-1])
    assert abs(r_axis - r_diag) < 1.5


def test_reduce_definitions(orc):
    """O5: <x>_V = mean x (L149), <x>_M = sum nH x / sum nH (L303-305), Gamma = c sigma_n N (Eq.15)."""
    rng = np.random.default_rng(4)
    n = 5
    nH = 10 ** rng.uniform(-5, -2, (n, n, n)); x = rng.uniform(0, 1, (n, n, n))
    T = rng.uniform(10, 1e5, (n, n, n)); N = rng.uniform(0, 1e-5, (n, n, n))
    Fx = 0.5 * C * N; Fy = np.zeros_like(N); Fz = -0.5 * C * N
    st = orc.State(nH, x, T, N, Fx, Fy, Fz)
    p = orc.make_params(wl.default_params(), 2.0e20, 1.0)
    d = orc.reduce(st, p)
    assert d["x_vol"] == pytest.approx(x.mean()) and d["x_mass"] == pytest.approx((nH * x).sum() / nH.sum())
    g = C * 2.93e-18 * N
    assert d["gamma_vol"] == pytest.approx(g.mean()) and d["gamma_mass"] == pytest.approx((nH * g).sum() / nH.sum())
    assert d["photons_total"] == pytest.approx(N.sum() * 8e60)
    assert d["T_vol"] == pytest.approx(T.mean()) and d["f_max"] == pytest.approx(math.sqrt(0.5))
    assert d["N_min"] == N.min() and d["n_nonfinite"] == 0
    assert d["frac_x_half"] == pytest.approx((x >= 0.5).mean())
    st.T[0, 0, 0] = np.nan
    assert orc.reduce(st, p)["n_nonfinite"] == 1
