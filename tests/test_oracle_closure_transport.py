"""Pins of the oracle's closure (O1) and transport (O2) against what the paper and mathematics fix.

Nothing here compares the oracle with itself: each test states a closed form, a limit the paper
prints, an invariant, or an exact solution of the difference scheme.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate

C = 2.99792458e10
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(name):
    out = {}
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


# ------------------------------------------------------------------ constants the paper prints
def test_paper_constants_are_blackbody_averages():
    """sigma_e (energy averaged), sigma_n (number averaged) and e=20.27 eV are the
    averages of the hydrogenic cross-section over a 50 000 K black body above 13.6 eV."""
    g = _golden("paper_constants.txt")
    x0 = 157807.0 / g["T_blackbody_K"]
    kT_eV = 8.617333e-5 * g["T_blackbody_K"]

    def sig(x):
        nu = x / x0
        eps = math.sqrt(max(nu - 1.0, 1e-12))
        return 6.30e-18 * nu ** -4 * math.exp(4 - 4 * math.atan(eps) / eps) / (1 - math.exp(-2 * math.pi / eps))

    num = integrate.quad(lambda x: x ** 3 / math.expm1(x), x0, 200)[0]
    den = integrate.quad(lambda x: x ** 2 / math.expm1(x), x0, 200)[0]
    sn = integrate.quad(lambda x: sig(x) * x ** 2 / math.expm1(x), x0 * (1 + 1e-9), 200)[0] / den
    se = integrate.quad(lambda x: sig(x) * x ** 3 / math.expm1(x), x0 * (1 + 1e-9), 200)[0] / num
    assert kT_eV * num / den == pytest.approx(g["e_photon_eV"], rel=1e-3)
    assert sn == pytest.approx(g["sigma_n_cm2"], rel=1e-2)
    assert se == pytest.approx(g["sigma_e_cm2"], rel=1e-2)
    from paper_1004_2503_b200.workloads import default_params
    p = default_params()
    assert p["sigma_n"] == g["sigma_n_cm2"] and p["sigma_e"] == g["sigma_e_cm2"]
    assert p["e_photon_eV"] == g["e_photon_eV"]


# ------------------------------------------------------------------ O1 closure
def test_chi_limits_and_shape(orc):
    g = _golden("paper_constants.txt")
    assert orc.chi(0.0) == pytest.approx(g["chi_diffusion"], abs=1e-15)
    assert orc.chi(1.0) == pytest.approx(g["chi_transport"], abs=1e-15)
    f = np.linspace(0, 1, 2001)
    ch = np.array([orc.chi(v) for v in f])
    assert np.all(np.diff(ch) > 0)                                  # monotone
    # M1 (Levermore) small-f expansion chi = 1/3 + f^2/2 + O(f^4) and slope 2 at f=1
    assert orc.chi(1e-3) - 1 / 3 == pytest.approx(0.5e-6, rel=1e-5)
    h = 1e-6
    assert (orc.chi(1.0) - orc.chi(1.0 - h)) / h == pytest.approx(2.0, rel=1e-4)
    # algebraically equivalent division-free form chi = (5 - 2 sqrt(4-3f^2))/3
    assert np.allclose(ch, (5 - 2 * np.sqrt(4 - 3 * f * f)) / 3, atol=1e-15)


def test_eddington_tensor_properties(orc):
    """Reading G1: D = (1-chi)/2 I + (3chi-1)/2 n(x)n.  Printed Eq.6 (L76) has trace 4chi-1."""
    rng = np.random.default_rng(0)
    for _ in range(200):
        N = 10 ** rng.uniform(-8, 2)
        n = rng.normal(size=3); n /= np.linalg.norm(n)
        f = rng.uniform(0, 1)
        P = orc.closure(N, C * N * f * n, C)
        D = P / N
        assert np.trace(D) == pytest.approx(1.0, abs=1e-13)              # tr D = 1
        assert np.allclose(D, D.T, atol=1e-15)
        # Eddington factor: n is an eigenvector with eigenvalue chi; the other two are (1-chi)/2
        assert np.allclose(D @ n, orc.chi(f) * n, atol=1e-13)
        ev = np.sort(np.linalg.eigvalsh(D))
        assert ev[0] == pytest.approx(0.5 * (1 - orc.chi(f)), abs=1e-12)
        assert ev[2] == pytest.approx(orc.chi(f), abs=1e-12)
    # limits the paper names (L78): pure diffusion D = I/3, pure transport D = n(x)n
    assert np.allclose(orc.closure(2.0, [0, 0, 0], C), 2.0 * np.eye(3) / 3, atol=1e-15)
    n = np.array([1.0, 2.0, -2.0]) / 3.0
    assert np.allclose(orc.closure(2.0, C * 2.0 * n, C), 2.0 * np.outer(n, n), atol=1e-14)


def test_closure_degenerate_inputs(orc):
    """Reading S2: f clamped to 1; N<=0 -> f=0; |F|=0 -> n=0."""
    n = np.array([0.0, 1.0, 0.0])
    assert np.allclose(orc.closure(1.0, 5 * C * n, C), np.outer(n, n), atol=1e-15)   # f>1 clamps
    assert np.allclose(orc.closure(0.0, [0, 0, 0], C), 0.0)
    P = orc.closure(-1.0, [0, 0, 0], C)
    assert np.allclose(P, -np.eye(3) / 3)


# ------------------------------------------------------------------ O2 transport
def _beam(n, axis, sign, prof):
    """N varying along `axis` only, F = sign*c*N along it (f = 1)."""
    shape = [1, 1, 1]; shape[2 - axis] = n           # arrays are [z][y][x]
    N = np.broadcast_to(prof.reshape(shape), (n, n, n)).copy()
    F = [np.zeros_like(N) for _ in range(3)]
    F[axis] = sign * C * N
    return N, F


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [1, -1])
def test_free_streaming_is_binomial_upwind(orc, axis, sign):
    """P1: for f=1 data the LF flux at speed c collapses to first-order upwind, so after p steps a
    spike is the binomial distribution C(p,k) mu^k (1-mu)^(p-k) displaced k cells down-stream."""
    n, p, mu = 16, 9, 0.3
    prof = np.zeros(n); prof[5] = 1.0
    N, F = _beam(n, axis, sign, prof)
    dx = 1.0e20; dt = mu * dx / C
    for _ in range(p):
        N, F[0], F[1], F[2] = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
    want = np.zeros(n)
    for k in range(p + 1):
        want[(5 + sign * k) % n] += math.comb(p, k) * mu ** k * (1 - mu) ** (p - k)
    line = np.moveaxis(N, 2 - axis, 0)[:, 3, 4]
    assert np.allclose(line, want, atol=1e-15)
    assert np.allclose(F[axis], sign * C * N, atol=1e-15 * C)            # f stays 1
    other = [a for a in range(3) if a != axis]
    assert np.all(F[other[0]] == 0) and np.all(F[other[1]] == 0)
    # centroid moved exactly p*mu cells (mod wrap not reached), variance p mu (1-mu)
    pos = (5 + sign * np.arange(p + 1))
    wts = np.array([math.comb(p, k) * mu ** k * (1 - mu) ** (p - k) for k in range(p + 1)])
    assert (pos * wts).sum() == pytest.approx(5 + sign * p * mu)


def test_oblique_beam_one_step(orc):
    """P1 (oblique): f=1 along (1,1,0)/sqrt2, N varying in x and y only:
    N' = (1-2mu)N + sum_d [ (mu/2)(1-n_d) N_{+d} + (mu/2)(1+n_d) N_{-d} ],  d in {x,y}."""
    n, mu = 12, 0.25
    rng = np.random.default_rng(3)
    prof = rng.uniform(0.5, 1.5, size=(n, n))                          # [y][x]
    N = np.broadcast_to(prof[None], (n, n, n)).copy()
    nd = np.array([1.0, 1.0, 0.0]) / math.sqrt(2)
    F = [C * N * nd[a] for a in range(3)]
    dx = 3.0e21; dt = mu * dx / C
    N1, Fx1, Fy1, Fz1 = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
    want = (1 - 2 * mu) * prof
    for ax, d in ((1, 0), (0, 1)):                                       # array axis, direction
        want = want + 0.5 * mu * (1 - nd[d]) * np.roll(prof, -1, axis=ax) \
                    + 0.5 * mu * (1 + nd[d]) * np.roll(prof, +1, axis=ax)
    assert np.allclose(N1[4], want, rtol=1e-13)
    # f = 1 data: P = n(x)n N, so every flux row of F is c n_j times the flux row of N and the scheme gives
    # F' = c n N' exactly -- this is where the OFF-DIAGONAL pressure P_xy enters (a dropped or transposed P_xy fails)
    assert np.allclose(Fx1, C * nd[0] * N1, rtol=1e-13) and np.allclose(Fy1, C * nd[1] * N1, rtol=1e-13)
    assert np.abs(Fz1).max() <= 1e-13 * C * N1.max()
    # a generic direction with all three components and all six off-diagonal terms live
    nd = np.array([2.0, -3.0, 6.0]) / 7.0
    N = rng.uniform(0.5, 1.5, size=(n, n, n))
    N1, Fx1, Fy1, Fz1 = orc.transport(N, C * N * nd[0], C * N * nd[1], C * N * nd[2], C, dx, dt)
    want = (1 - 3 * mu) * N
    for ax, d in ((2, 0), (1, 1), (0, 2)):
        want = want + 0.5 * mu * (1 - nd[d]) * np.roll(N, -1, axis=ax) + 0.5 * mu * (1 + nd[d]) * np.roll(N, +1, axis=ax)
    assert np.allclose(N1, want, rtol=1e-13)
    for Fj, nj in ((Fx1, nd[0]), (Fy1, nd[1]), (Fz1, nd[2])):
        assert np.allclose(Fj, C * nj * N1, rtol=1e-12)


def _random_realizable(n, rng, fmax=0.99):
    N = 10 ** rng.uniform(-3, 0, size=(n, n, n))
    d = rng.normal(size=(3, n, n, n)); d /= np.linalg.norm(d, axis=0)
    f = rng.uniform(0, fmax, size=(n, n, n))
    return N, [C * N * f * d[a] for a in range(3)]


def test_vacuum_conservation(orc):
    """P2: with no absorption and no sources sum N and each sum F_j are conserved (telescoping)."""
    rng = np.random.default_rng(1)
    N, F = _random_realizable(10, rng)
    s0 = [N.sum()] + [f.sum() for f in F]
    dx = 1e21; dt = 0.3 * dx / C
    for _ in range(5):
        N, F[0], F[1], F[2] = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
    s1 = [N.sum()] + [f.sum() for f in F]
    assert s1[0] == pytest.approx(s0[0], rel=1e-13)
    scale = C * s0[0]
    for a in range(3):
        assert abs(s1[1 + a] - s0[1 + a]) < 1e-13 * scale


def test_realizability_and_isotropic_fixed_point(orc):
    """P3: for mu <= 1/3, N >= 0 and |F| <= cN are preserved; a uniform isotropic field is fixed."""
    rng = np.random.default_rng(2)
    N, F = _random_realizable(10, rng, fmax=1.0)
    N[2:5, 2:5, 2:5] = 0.0
    for f in F:
        f[2:5, 2:5, 2:5] = 0.0
    dx = 1e21; dt = dx / (3 * C)
    for _ in range(6):
        N, F[0], F[1], F[2] = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
        assert N.min() >= 0.0
        Fn = np.sqrt(F[0] ** 2 + F[1] ** 2 + F[2] ** 2)
        assert np.all(Fn <= C * N * (1 + 1e-12))
    U = np.full((6, 6, 6), 0.7)
    Z = np.zeros_like(U)
    out = orc.transport(U, Z, Z, Z, C, dx, dt)
    assert np.array_equal(out[0], U) and all(np.all(o == 0) for o in out[1:])


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_diffusion_limit_amplification(orc, axis):
    """P4: a small mode N = N0(1 + eps cos(theta i)), F = 0 evolves with the linearised matrix
    M = (1 - mu(1-cos th)) I - i mu sin th [[0,1],[1/3,0]] acting on (N^, G^=F^/c): waves at
    c/sqrt3 because D -> I/3; error O(eps^2) since chi = 1/3 + f^2/2."""
    n, m, p, mu, eps = 32, 2, 40, 0.3, 1e-6
    th = 2 * math.pi * m / n
    i = np.arange(n)
    N, F = _beam(n, axis, 1, 1.0 + eps * np.cos(th * i))
    F[axis][:] = 0.0
    dx = 1e21; dt = mu * dx / C
    for _ in range(p):
        N, F[0], F[1], F[2] = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
    M = (1 - mu * (1 - math.cos(th))) * np.eye(2) - 1j * mu * math.sin(th) * np.array([[0, 1], [1 / 3, 0]])
    v = np.linalg.matrix_power(M, p) @ np.array([eps, 0.0])
    lineN = np.moveaxis(N, 2 - axis, 0)[:, 1, 2]
    lineG = np.moveaxis(F[axis], 2 - axis, 0)[:, 1, 2] / C
    # mode amplitude of exp(+i th i): fft coefficient m (numpy's sign convention -> conj)
    Nh = np.fft.fft(lineN - 1.0)[m] / n * 2
    Gh = np.fft.fft(lineG)[m] / n * 2
    assert abs(Nh - v[0]) < 1e-4 * eps
    assert abs(Gh - v[1]) < 1e-4 * eps


def test_checkerboard_mode_sets_the_stability_limit(orc):
    """Reading S3: the von Neumann factor of the unsplit 3-D LF scheme at theta=(pi,pi,pi) is
    1 - 6 mu, so mu = 1/3 is the stability limit (|1-6mu| = 1) and mu > 1/3 blows up."""
    n, eps = 8, 1e-7
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    N = 1.0 + eps * (-1.0) ** (i + j + k)
    Z = np.zeros_like(N)
    dx = 1e21
    for mu in (0.1, 1 / 3, 0.5):
        N1, *_ = orc.transport(N, Z, Z, Z, C, dx, mu * dx / C)
        amp = (N1[0, 0, 0] - 1.0) / eps
        assert amp == pytest.approx(1 - 6 * mu, abs=1e-6)


def test_axis_permutation_covariance(orc):
    """Relabelling the axes of the input (and the flux components) relabels the output: catches a
    transposed operand or a wrong stride in any one direction."""
    rng = np.random.default_rng(5)
    N, F = _random_realizable(6, rng)
    dx = 1e21; dt = 0.3 * dx / C
    ref = orc.transport(N, F[0], F[1], F[2], C, dx, dt)
    # swap x <-> z: arrays [z][y][x] -> transpose(2,1,0); flux components (Fx,Fy,Fz) -> (Fz,Fy,Fx)
    t = lambda a: np.ascontiguousarray(a.transpose(2, 1, 0))
    out = orc.transport(t(N), t(F[2]), t(F[1]), t(F[0]), C, dx, dt)
    assert np.allclose(t(out[0]), ref[0], rtol=1e-13)
    assert np.allclose(t(out[1]), ref[3], rtol=1e-12, atol=1e-13 * C)
    assert np.allclose(t(out[3]), ref[1], rtol=1e-12, atol=1e-13 * C)
    # reflection x -> -x flips the sign of Fx only
    r = lambda a: np.ascontiguousarray(a[:, :, ::-1])
    out = orc.transport(r(N), -r(F[0]), r(F[1]), r(F[2]), C, dx, dt)
    assert np.allclose(r(out[0]), ref[0], rtol=1e-13)
    assert np.allclose(-r(out[1]), ref[1], rtol=1e-12, atol=1e-13 * C)
    assert np.allclose(r(out[2]), ref[2], rtol=1e-12, atol=1e-13 * C)
