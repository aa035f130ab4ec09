"""Pins of the oracle's analysis / source front-end functions: clumping-factor measurement
over 8^3 blocks, 2-D distributions (Fig.5-19), star-particle emission rates (section 2.3, Eq.8-9) and
the Thomson optical depth (Eq.10)."""
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MYR = 3.15576e13


# ------------------------------------------------------------------ clumping blocks
def test_clumping_blocks_uniform_and_checkerboard(orc):
    b, n = 8, 16
    nH = np.full((n, n, n), 3e-4); x = np.full((n, n, n), 0.3); N = np.full((n, n, n), 2e-7)
    out = orc.clumping_blocks(nH, x, N, b)
    assert out["C_R"].shape == (2, 2, 2)
    for k, v in (("nH", 3e-4), ("x", 0.3), ("C_R", 1.0), ("C_I", 1.0)):
        assert np.allclose(out[k], v, rtol=1e-14)                       # a homogeneous block has no clumping
    # two-valued checkerboard in density (a, b), constant x: C_R = <n^2>/<n>^2 = 2 (a^2 + b^2)/(a + b)^2 by hand
    a_, b_ = 1e-4, 9e-4
    kk, jj, ii = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    chk = (kk + jj + ii) % 2
    nH = np.where(chk == 0, a_, b_)
    out = orc.clumping_blocks(nH, x, N, b)
    assert np.allclose(out["C_R"], 2 * (a_ ** 2 + b_ ** 2) / (a_ + b_) ** 2, rtol=1e-13)
    assert np.allclose(out["nH"], 0.5 * (a_ + b_), rtol=1e-14) and np.allclose(out["x"], 0.3, rtol=1e-14)
    # photons in phase with the neutral gas: the same number; in anti-phase: <ab>/(<a><b>) = 4ab/(a+b)^2 < 1
    out = orc.clumping_blocks(nH, x, np.where(chk == 0, a_, b_), b)
    assert np.allclose(out["C_I"], 2 * (a_ ** 2 + b_ ** 2) / (a_ + b_) ** 2, rtol=1e-13)
    out = orc.clumping_blocks(nH, x, np.where(chk == 0, b_, a_), b)
    assert np.allclose(out["C_I"], 4 * a_ * b_ / (a_ + b_) ** 2, rtol=1e-13)
    # x enters C_R as n_H x (<n_H^2 x^2>/<n_H x>^2): ionised where dense = more clumping
    xv = np.where(chk == 0, 0.1, 0.9)
    out = orc.clumping_blocks(nH, xv, N, b)
    u, v = a_ * 0.1, b_ * 0.9
    assert np.allclose(out["C_R"], 2 * (u * u + v * v) / (u + v) ** 2, rtol=1e-13)
    assert np.allclose(out["x"], (u + v) / (a_ + b_), rtol=1e-13)        # mass-weighted ionised fraction of the block


def test_clumping_blocks_invariants_and_degenerate_blocks(orc):
    rng = np.random.default_rng(2)
    n, b = 16, 8
    nH = 10 ** rng.uniform(-5, -2, (n, n, n)); x = rng.uniform(0, 1, (n, n, n)); N = 10 ** rng.uniform(-9, -5, (n, n, n))
    out = orc.clumping_blocks(nH, x, N, b)
    assert (out["C_R"] >= 1 - 1e-14).all()                             # Cauchy-Schwarz: <q^2> >= <q>^2
    out2 = orc.clumping_blocks(7.0 * nH, x, 0.01 * N, b)                # pure ratios: scale free
    assert np.allclose(out2["C_R"], out["C_R"], rtol=1e-12) and np.allclose(out2["C_I"], out["C_I"], rtol=1e-12)
    # brute force of one block with numpy
    s = (slice(8, 16), slice(0, 8), slice(8, 16))
    q = (nH * x)[s]
    assert out["C_R"][1, 0, 1] == pytest.approx((q ** 2).mean() / q.mean() ** 2, rel=1e-13)
    yn = ((1 - x) * nH)[s]
    assert out["C_I"][1, 0, 1] == pytest.approx((N[s] * yn).mean() / (N[s].mean() * yn.mean()), rel=1e-13)
    # block size 4 gives 4^3 blocks; a dark, fully neutral or fully ionised block reports 1 (reading S21)
    assert orc.clumping_blocks(nH, x, N, 4)["C_R"].shape == (4, 4, 4)
    out = orc.clumping_blocks(nH, np.zeros_like(x), np.zeros_like(N), b)
    assert (out["C_R"] == 1).all() and (out["C_I"] == 1).all() and (out["x"] == 0).all()
    out = orc.clumping_blocks(nH, np.ones_like(x), N, b)
    assert (out["C_I"] == 1).all()


# ------------------------------------------------------------------ 2-D histogram
def test_hist2d_against_numpy(orc):
    rng = np.random.default_rng(4)
    a = 10 ** rng.uniform(-6, -1, 20000); bq = rng.uniform(-0.2, 1.2, 20000)
    counts, outside = orc.hist2d(a, bq, True, False, (-5, -2), (0, 1), 12, 7)
    want, _, _ = np.histogram2d(bq, np.log10(a), bins=(7, 12), range=((0, 1), (-5, -2)))
    inside = (np.log10(a) >= -5) & (np.log10(a) < -2) & (bq >= 0) & (bq < 1)
    assert counts.sum() == inside.sum() and outside == (~inside).sum()
    # numpy closes the last bin on the right; no sample sits exactly there
    assert np.array_equal(counts, want.astype(np.int64))
    # edges: lo is inside, hi is outside; non-positive values on a log axis are outside
    c, o = orc.hist2d([1e-5, 1e-2, 0.0, -1.0, 1e-3], [0.0, 0.5, 0.5, 0.5, 1.0], True, False, (-5, -2), (0, 1), 3, 2)
    assert c.sum() == 1 and c[0, 0] == 1 and o == 4


# ------------------------------------------------------------------ star-particle sources (section 2.3)
def _table1():
    rows = [l.split() for l in open(os.path.join(GOLD, "paper_table1.txt")) if l.strip() and not l.startswith("#")]
    return {float(r[0]): (float(r[1]), float(r[2]) * MYR, float(r[3])) for r in rows}


def test_boost_factor_reading(orc):
    """Eq.9 with Table 1: B = SFR_converged/SFR_actual must be >= 1 and large for the under-resolved 100 Mpc/h box,
    about 1 for the 12.5 Mpc/h box that 'barely satisfies' the resolution criterion (L115); it decreases with time and
    tends to max(1, a_b)."""
    t1 = _table1()
    t = 700 * MYR
    B = {box: orc.boost(t, a, k) for box, (a, k, _) in t1.items()}
    assert B[12.5] == pytest.approx(max(1.0, 0.7 * math.exp(300 / 700)), rel=1e-12) and 1.0 <= B[12.5] < 1.1
    assert B[100.0] == pytest.approx(1.2 * math.exp(3000 / 700), rel=1e-12) and B[100.0] > 50
    assert B[12.5] <= B[25.0] < B[50.0] < B[100.0]
    for box, (a, k, _) in t1.items():
        assert orc.boost(400 * MYR, a, k) >= orc.boost(900 * MYR, a, k) >= 1.0
        assert orc.boost(1e30, a, k) == pytest.approx(max(1.0, a), rel=1e-9)


def test_star_rates_conserve_the_photons_of_each_star(orc):
    """Whatever the snapshot spacing, summing rate * (t_{p+1} - t_p) over the snapshots in which a star is seen gives
    photons_per_baryon * n_baryons (f_esc = B = 1): the three branches (born in the interval, alive throughout, dying in
    it) and the discard rule together account for every photon exactly once."""
    rng = np.random.default_rng(8)
    ns = 200
    t_birth = rng.uniform(100, 400, ns) * MYR
    life = rng.uniform(5, 20, ns) * MYR                                  # drawn between 5 and 20 Myr
    nbar = 10 ** rng.uniform(58, 61, ns)
    ppb = 5.0e4                                                           # between 24 000 and 98 000 (L97)
    snaps = np.sort(np.concatenate([[90 * MYR, 450 * MYR], rng.uniform(95, 445, 37) * MYR]))
    emitted = np.zeros(ns)
    for tp, tp1 in zip(snaps[:-1], snaps[1:]):
        seen = t_birth <= tp1                                             # stars of snapshot p+1
        age1 = tp1 - t_birth[seen]
        r = orc.star_rates(age1, life[seen], nbar[seen], ppb, tp, tp1, 1.0, 1e-30, 0.0)
        emitted[seen] += r * (tp1 - tp)
    assert np.allclose(emitted, ppb * nbar, rtol=1e-12)
    # single cases by hand: Ndot = ppb nbar / L
    L, nb, dtp = 10 * MYR, 1e60, 4 * MYR
    nd = ppb * nb / L
    one = lambda a1: orc.star_rates([a1], [L], [nb], ppb, 100 * MYR, 100 * MYR + dtp, 1.0, 1e-30, 0.0)[0]
    assert one(7 * MYR) == pytest.approx(nd, rel=1e-14)                  # alive throughout
    assert one(1 * MYR) == pytest.approx(nd * 0.25, rel=1e-14)           # born 1 Myr before the snapshot: diluted
    assert one(13 * MYR) == pytest.approx(nd * 0.25, rel=1e-14)          # a_p = 9 Myr: shines 1 more Myr of the 4
    assert one(14.5 * MYR) == 0.0                                        # a_p = 10.5 Myr > L: discarded
    # Eq.8: f_esc and the boost multiply
    r = orc.star_rates([7 * MYR], [L], [nb], ppb, 600 * MYR, 600 * MYR + dtp, 0.02, 1.2, 3000 * MYR)[0]
    assert r == pytest.approx(nd * 0.02 * 1.2 * math.exp(3000 / 602), rel=1e-12)


# ------------------------------------------------------------------ Thomson optical depth (Eq.10)
def test_thomson_tau_closed_form(orc):
    """Fully ionised hydrogen out to z_r in flat LCDM: tau = (2 c sigma_T nH0 / (3 H0 Om)) [sqrt(Om (1+z_r)^3 + 1 - Om) - 1]
    (the integral of (1+z)^2/E(z) is elementary); WMAP-5-like numbers give the textbook ~0.04 for z_r = 6.5."""
    H0 = 72e5 / 3.0856775814913673e24
    Om, nH0 = 0.26, 1.9e-7
    z = np.linspace(0, 6.5, 4001)
    tau = orc.thomson_tau(z, np.ones_like(z), nH0, H0, Om)
    want = 2 * 2.99792458e10 * 6.6524587e-25 * nH0 / (3 * H0 * Om) * (math.sqrt(Om * 7.5 ** 3 + 1 - Om) - 1)
    assert tau == pytest.approx(want, rel=1e-6)
    assert 0.03 < tau < 0.05
    # linear in x; a history that switches on at z = 6.5 adds nothing beyond it
    assert orc.thomson_tau(z, 0.5 * np.ones_like(z), nH0, H0, Om) == pytest.approx(0.5 * tau, rel=1e-12)
    z2 = np.concatenate([z, np.linspace(6.5, 12, 500)[1:]])
    x2 = np.concatenate([np.ones_like(z), np.zeros(499)])
    assert orc.thomson_tau(z2, x2, nH0, H0, Om) == pytest.approx(tau, rel=2e-3)
