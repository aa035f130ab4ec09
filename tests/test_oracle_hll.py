"""Pins of the oracle's HLL intercell flux ("HLL or the simpler Lax-Friedrich scheme"; SURVEY NEXT-3;
DESIGN.md reading S20).  The paper prints neither the flux nor the wave speeds, so what is pinned is
(i) the closed-form wave speeds against the DEFINITION -- the extreme eigenvalues of the Jacobian of the oracle's own
M1 flux function, taken by finite differences and numpy's eigen-solver; (ii) the flux formula's limits (Lax-Friedrichs
at l = +-c, upwind on a beam); (iii) what any consistent conservative scheme must do (conservation, realizability,
the linearised amplification matrix with the signal speed c/sqrt3); (iv) that it is less diffusive than LF."""
import math

import numpy as np
import pytest

C = 2.99792458e10


def _jacobian_eigs(orc, d, N, F):
    """Eigenvalues of d FF_d / d U at U = (N, F) by central differences of orc.flux_fn, in units of c (F scaled by c)."""
    U = np.array([N, F[0] / C, F[1] / C, F[2] / C])                   # work with G = F/c so all entries are O(N)
    def ff(u):
        g = orc.flux_fn(d, u[0], u[1:] * C, C)
        return np.array([g[0] / C, g[1] / C ** 2, g[2] / C ** 2, g[3] / C ** 2])     # flux of (N, G) in units of c
    J = np.zeros((4, 4))
    for b in range(4):
        h = 1e-6 * N
        up, um = U.copy(), U.copy()
        up[b] += h; um[b] -= h
        J[:, b] = (ff(up) - ff(um)) / (2 * h)
    return np.linalg.eigvals(J)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_wavespeeds_are_the_extreme_eigenvalues_of_the_flux_jacobian(orc, d):
    rng = np.random.default_rng(40 + d)
    for f in (0.02, 0.1, 0.3, 0.5, 0.7, 0.9, 0.97):
        for _ in range(12):
            n = rng.normal(size=3); n /= np.linalg.norm(n)
            N = 10 ** rng.uniform(-6, 0)
            F = C * N * f * n
            ev = _jacobian_eigs(orc, d, N, F)
            assert np.abs(ev.imag).max() < 1e-5                      # hyperbolic: real eigenvalues
            lo, hi = orc.m1_wavespeeds(N, F, C, d)
            assert lo / C == pytest.approx(ev.real.min(), abs=2e-5)
            assert hi / C == pytest.approx(ev.real.max(), abs=2e-5)
            assert -1 - 1e-12 <= lo / C <= hi / C <= 1 + 1e-12         # never faster than light
            # the two middle eigenvalues are the transverse one, (2 - xi) mu / f, twice
            xi = math.sqrt(4 - 3 * f * f)
            mid = np.sort(ev.real)[1:3]
            assert np.allclose(mid, (2 - xi) * n[d] / f, atol=2e-5)


def test_wavespeed_limits(orc):
    """Diffusion limit: +-c/sqrt3 whatever the direction; free streaming: both speeds equal c cos(theta)."""
    lo, hi = orc.m1_wavespeeds(1.0, [0.0, 0.0, 0.0], C, 0)
    assert lo == pytest.approx(-C / math.sqrt(3), rel=1e-14) and hi == pytest.approx(C / math.sqrt(3), rel=1e-14)
    lo, hi = orc.m1_wavespeeds(0.0, [0.0, 0.0, 0.0], C, 1)            # vacuum cell (S2: f = 0)
    assert lo == pytest.approx(-C / math.sqrt(3)) and hi == pytest.approx(C / math.sqrt(3))
    for n in ([1, 0, 0], [0.6, 0.8, 0.0], [0, 0, -1], [2 / 7, -3 / 7, 6 / 7]):
        for d in range(3):
            lo, hi = orc.m1_wavespeeds(2.0, [C * 2.0 * v for v in n], C, d)
            assert lo == pytest.approx(C * n[d], abs=1e-7 * C) and hi == pytest.approx(C * n[d], abs=1e-7 * C)
    # f slightly above 1 (round-off) is clamped like in the closure
    lo, hi = orc.m1_wavespeeds(1.0, [C * 1.0000001, 0, 0], C, 0)
    assert hi == pytest.approx(C, rel=1e-12)


def test_hll_flux_formula_limits(orc):
    rng = np.random.default_rng(5)
    Ul, Ur, gl, gr = (rng.normal(size=4) for _ in range(4))
    # signal speeds +-c: the Lax-Friedrichs flux of orc_transport
    lf = 0.5 * (gl + gr) - 0.5 * C * (Ur - Ul)
    assert np.allclose(orc.hll_flux(Ul, gl, Ur, gr, -C, C), lf, rtol=1e-13)
    # everything moves right (l- = 0): the upwind (left) flux; everything moves left: the right flux
    assert np.allclose(orc.hll_flux(Ul, gl, Ur, gr, 0.0, 0.7 * C), gl, rtol=1e-14)
    assert np.allclose(orc.hll_flux(Ul, gl, Ur, gr, -0.3 * C, 0.0), gr, rtol=1e-14)
    # no signal crosses the face: the mean of two (then equal-normal-flux) states
    assert np.allclose(orc.hll_flux(Ul, gl, Ur, gr, 0.0, 0.0), 0.5 * (gl + gr), rtol=1e-14)
    # consistency: equal states give the physical flux whatever the speeds
    assert np.allclose(orc.hll_flux(Ul, gl, Ul, gl, -0.2 * C, 0.9 * C), gl, rtol=1e-13)


@pytest.mark.parametrize("axis,sign", [(0, 1), (0, -1), (1, 1), (2, -1)])
def test_hll_free_streaming_is_binomial_upwind(orc, axis, sign):
    """On an axis-aligned f = 1 beam l- = 0 (or l+ = 0): HLL is first-order upwind, like LF at speed c (P1)."""
    n, mu, p = 16, 0.25, 9
    prof = np.zeros(n); prof[3:6] = [1.0, 2.0, 0.5]
    shape = [1, 1, 1]; shape[2 - axis] = n
    N = np.broadcast_to(prof.reshape(shape), (n, n, n)).copy()
    F = [np.zeros_like(N) for _ in range(3)]
    F[axis] = sign * C * N
    dx = 1.0e21; dt = mu * dx / C
    for _ in range(p):
        N, F[0], F[1], F[2] = orc.transport_hll(N, F[0], F[1], F[2], C, dx, dt)
    want = np.zeros(n)
    for k in range(p + 1):
        want += math.comb(p, k) * mu ** k * (1 - mu) ** (p - k) * np.roll(prof, sign * k)
    line = np.moveaxis(N, 2 - axis, 0)[:, 0, 0]
    assert np.allclose(line, want, rtol=1e-12, atol=1e-15)
    assert np.allclose(F[axis], sign * C * N, rtol=1e-12, atol=1e-15 * C)


def _random_realizable(n, rng, fmax=0.99):
    N = 10 ** rng.uniform(-3, 0, size=(n, n, n))
    d = rng.normal(size=(3, n, n, n)); d /= np.linalg.norm(d, axis=0)
    f = rng.uniform(0, fmax, size=(n, n, n))
    return N, [C * N * f * d[a] for a in range(3)]


def test_hll_conservation_and_realizability(orc):
    """Telescoping face fluxes: sum N and sum F conserved; for c dt/dx <= 1/3 the update is a convex combination of
    realizable states (each HLL face state is one): N >= 0 and |F| <= cN are preserved; isotropic uniform gas is fixed."""
    rng = np.random.default_rng(9)
    n = 10
    N, F = _random_realizable(n, rng, 1.0)
    dx = 2.0e21; dt = dx / (3 * C)
    s0 = [N.sum()] + [f.sum() for f in F]
    for _ in range(25):
        N, F[0], F[1], F[2] = orc.transport_hll(N, F[0], F[1], F[2], C, dx, dt)
        assert N.min() >= 0
        fr = np.sqrt(F[0] ** 2 + F[1] ** 2 + F[2] ** 2) / (C * N)
        assert fr.max() <= 1 + 1e-12
    assert N.sum() == pytest.approx(s0[0], rel=1e-13)
    for a in range(3):
        assert F[a].sum() == pytest.approx(s0[1 + a], abs=1e-12 * C * s0[0])
    N = np.full((6, 6, 6), 0.37); Z = np.zeros_like(N)
    N1, a, b, c_ = orc.transport_hll(N, Z, Z, Z, C, dx, dt)
    assert np.array_equal(N1, N) and not a.any() and not b.any() and not c_.any()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_hll_diffusion_limit_amplification(orc, axis):
    """Linearised about an isotropic state the signal speeds are +-c/sqrt3, so a mode (N^, G^) is multiplied per step by
    M = (1 - (mu/sqrt3)(1 - cos th)) I - i mu sin th [[0, 1], [1/3, 0]] -- the P4 matrix of the LF scheme with its
    dissipation reduced by 1/sqrt3."""
    n, m, p, eps, mu = 32, 2, 40, 1e-6, 0.3
    th = 2 * math.pi * m / n
    shape = [1, 1, 1]; shape[2 - axis] = n
    cosx = np.cos(th * np.arange(n)).reshape(shape)
    N = np.broadcast_to(1.0 + eps * cosx, (n, n, n)).copy()
    F = [np.zeros_like(N) for _ in range(3)]
    dx = 1.0e21; dt = mu * dx / C
    for _ in range(p):
        N, F[0], F[1], F[2] = orc.transport_hll(N, F[0], F[1], F[2], C, dx, dt)
    M = (1 - mu / math.sqrt(3) * (1 - math.cos(th))) * np.eye(2) - 1j * mu * math.sin(th) * np.array([[0, 1], [1 / 3, 0]])
    v = np.linalg.matrix_power(M, p) @ np.array([eps, 0.0])
    line = np.moveaxis(N, 2 - axis, 0)[:, 0, 0]
    Nk = 2 * np.fft.fft(line - 1.0)[m] / n
    Gk = 2 * np.fft.fft(np.moveaxis(F[axis], 2 - axis, 0)[:, 0, 0])[m] / n / C
    assert Nk == pytest.approx(v[0], rel=1e-4, abs=1e-5 * eps)
    assert Gk == pytest.approx(v[1], rel=1e-4, abs=1e-5 * eps)
    # and the LF scheme damps the same mode harder
    Nl = np.broadcast_to(1.0 + eps * cosx, (n, n, n)).copy()
    Fl = [np.zeros_like(Nl) for _ in range(3)]
    for _ in range(p):
        Nl, Fl[0], Fl[1], Fl[2] = orc.transport(Nl, Fl[0], Fl[1], Fl[2], C, dx, dt)
    e_hll = abs(Nk) ** 2 + 3 * abs(Gk) ** 2
    Nlk = 2 * np.fft.fft(np.moveaxis(Nl, 2 - axis, 0)[:, 0, 0] - 1.0)[m] / n
    Glk = 2 * np.fft.fft(np.moveaxis(Fl[axis], 2 - axis, 0)[:, 0, 0])[m] / n / C
    assert e_hll > abs(Nlk) ** 2 + 3 * abs(Glk) ** 2


def test_hll_is_less_diffusive_than_lf_on_an_oblique_beam(orc):
    """A beam along (1,1,0)/sqrt2 with a Gaussian profile across it: after p steps the transverse spread (second moment
    about the centroid, perpendicular to the beam) has grown less with HLL than with LF, and both moved the centroid by
    p mu / sqrt2 cells along each axis."""
    n, mu, p = 32, 0.3, 30
    yy, xx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    prof = np.exp(-(((xx - 8) ** 2 + (yy - 8) ** 2) / (2 * 2.0 ** 2)))
    nd = np.array([1.0, 1.0, 0.0]) / math.sqrt(2)
    dx = 1.0e21; dt = mu * dx / C
    res = {}
    for name, fn in (("lf", orc.transport), ("hll", orc.transport_hll)):
        N = np.broadcast_to(prof[None], (4, n, n)).copy()
        F = [C * N * nd[a] for a in range(3)]
        for _ in range(p):
            N, F[0], F[1], F[2] = fn(N, F[0], F[1], F[2], C, dx, dt)
        w = N[0] / N[0].sum()
        cx, cy = (w * xx).sum(), (w * yy).sum()
        perp = ((xx - cx) - (yy - cy)) / math.sqrt(2)
        res[name] = (cx, cy, (w * perp ** 2).sum(), N[0].sum())
    for name in res:
        assert res[name][0] == pytest.approx(8 + p * mu / math.sqrt(2), abs=0.05)
        assert res[name][1] == pytest.approx(8 + p * mu / math.sqrt(2), abs=0.05)
        assert res[name][3] == pytest.approx(prof.sum(), rel=1e-12)
    assert res["hll"][2] < 0.8 * res["lf"][2]


def test_step_with_hll_flux_first_step_and_symmetry(orc):
    """orc_step honours params.flux: the first step from vacuum only touches the source cell (same as LF), later steps
    differ from LF, and a centred source in uniform gas stays symmetric under axis permutations."""
    from paper_1004_2503_b200 import workloads as wl
    w = wl.make_config(1, n=12)
    res = {}
    for flux in (0, 1):
        st, p = orc.from_workload(w)
        p.flux = flux
        orc.step(st, p, w.dt, 1, w.src_pos.numpy(), w.src_rate.numpy())
        first = st.N.copy()
        orc.step(st, p, w.dt, 5, w.src_pos.numpy(), w.src_rate.numpy())
        res[flux] = (first, st.N.copy(), st.x.copy())
    assert np.array_equal(res[0][0], res[1][0]) and np.count_nonzero(res[1][0]) == 1
    assert not np.allclose(res[0][1], res[1][1], rtol=1e-3)
    N = res[1][1]
    assert np.allclose(N, N.transpose(1, 0, 2), rtol=1e-12) and np.allclose(N, N.transpose(2, 1, 0), rtol=1e-12)
    assert res[1][1].sum() > 0 and res[1][2].max() <= 1.0
