"""GPU parity of the analysis / source front-end calls against the oracle: clumping-factor
measurement over 8^3 blocks, 2-D distributions (bit-exact counts), star-particle sources, Thomson optical depth."""
import math

import numpy as np
import pytest
import torch

from paper_1004_2503_b200 import workloads as wl
from parity_util import l1_errors, twin

pytestmark = pytest.mark.gpu
MYR = 3.15576e13


def _ctx(w):
    from paper_1004_2503_b200 import aton
    return aton.from_workload(w)


@pytest.mark.parametrize("n,block", [(64, 8), (32, 4), (48, 16), (40, 8)])
def test_clumping_blocks_against_oracle(orc, n, block):
    """A synthetic 'fine grid' (seeded log-normal density, bubbles, photons: workloads.synthetic_warm_state stands in for
    the paper's 12.5 Mpc/h run) measured over b^3 blocks: element by element against orc_clumping_blocks."""
    w = wl.synthetic_warm_state(twin(5, n, 10))
    a = _ctx(w)
    for device in ("cuda", "cpu"):
        g = a.clumping_blocks(block, device=device)
        ref = orc.clumping_blocks(w.nH.numpy(), w.x.numpy(), w.N.numpy(), block)
        for k in ("nH", "x", "C_R", "C_I"):
            assert g[k].shape == ref[k].shape
            assert np.allclose(g[k].cpu().numpy(), ref[k], rtol=2e-6, atol=0), k
        assert (g["C_R"] >= 1 - 1e-6).all() and float(g["C_R"].max()) > 1.5     # a log-normal field is clumpy
    # after a few steps the measurement follows the state (N is the current buffer)
    a.step(w.dt, 3)
    out = a.get_fields(device="cpu")
    g = a.clumping_blocks(block)
    ref = orc.clumping_blocks(out["nH"].numpy(), out["x"].numpy(), out["N"].numpy(), block)
    for k in ("nH", "x", "C_R", "C_I"):
        assert np.allclose(g[k].cpu().numpy(), ref[k], rtol=2e-6, atol=0), k
    from paper_1004_2503_b200 import aton
    with pytest.raises(aton.AtonError):
        a.clumping_blocks(7)                                           # must divide the grid
    a.close()


def test_clumping_blocks_uniform_and_dark(orc):
    from paper_1004_2503_b200 import aton
    w = wl.make_config(1)                                              # uniform gas, dark: C_R = 1, C_I = 1 (no photons)
    a = _ctx(w)
    g = a.clumping_blocks(8)
    assert torch.allclose(g["C_R"], torch.ones_like(g["C_R"]), rtol=1e-6) and bool((g["C_I"] == 1).all())
    assert torch.allclose(g["nH"], torch.full_like(g["nH"], 1e-3), rtol=1e-6)
    a.close()


def test_histogram2d_bit_exact(orc):
    """Counts are integers decided in fp64 on both sides: bit-exact, for every pair of quantities the paper plots."""
    from paper_1004_2503_b200 import aton
    w = wl.synthetic_warm_state(twin(4, 64, 10))
    a = _ctx(w)
    nH, x, T, N = (t.double().numpy() for t in (w.nH, w.x, w.T, w.N))
    cs = w.params["c_cm_s"] * w.params["sigma_n"]
    q = {aton.Q_NH: nH, aton.Q_X: x, aton.Q_NEUTRAL: 1.0 - x, aton.Q_T: T, aton.Q_N: N, aton.Q_GAMMA: cs * N}
    cases = [(aton.Q_NH, aton.Q_GAMMA, True, True, (-7, -1), (-16, -8), 48, 40),      # the J21(n_H) plane (Fig.5, 10)
             (aton.Q_NH, aton.Q_NEUTRAL, True, True, (-6, -2), (-6, 0), 32, 64),       # (1-x)(n_H) (Fig.11, 19)
             (aton.Q_NH, aton.Q_X, True, False, (-6, -2), (0, 1), 64, 64),
             (aton.Q_T, aton.Q_N, True, True, (1.5, 5.5), (-12, -4), 16, 16),
             (aton.Q_X, aton.Q_T, False, False, (0.2, 0.8), (0.0, 3e4), 7, 5)]
    for qa, qb, la, lb, ra, rb, na, nb in cases:
        counts, outside = a.histogram2d(qa, qb, la, lb, ra, rb, na, nb)
        ref, ref_out = orc.hist2d(q[qa], q[qb], la, lb, ra, rb, na, nb)
        assert np.array_equal(counts.numpy(), ref), (qa, qb)
        assert outside == ref_out and int(counts.sum()) + outside == w.n ** 3
    with pytest.raises(aton.AtonError):
        a.histogram2d(0, 1, True, False, (-6, -2), (0, 1), 128, 64)      # more than 4096 bins
    with pytest.raises(aton.AtonError):
        a.histogram2d(0, 9, True, False, (-6, -2), (0, 1), 8, 8)         # unknown quantity
    a.close()


def test_star_sources_against_oracle(orc):
    """aton_set_star_sources = the oracle's star rates handed to the ordinary source path: identical runs."""
    from paper_1004_2503_b200 import aton
    w = twin(3, 32, 40)
    rng = np.random.default_rng(21)
    ns = 300
    pos = torch.from_numpy(rng.uniform(0, 1, (ns, 3)).astype(np.float32))
    t_p, t_p1 = 600 * MYR, 600 * MYR + 40 * w.dt
    life = rng.uniform(5, 20, ns) * MYR
    age = rng.uniform(-0.2, 1.5, ns) * life + (t_p1 - t_p) * rng.uniform(0, 1, ns)     # born before / inside, alive / dead
    age = np.maximum(age, 1e-3 * MYR)
    nbar = 10 ** rng.uniform(61, 63, ns)
    ppb, f_esc, a_b, k_b = 6.0e4, 0.03, 1.2, 1500 * MYR
    rate = orc.star_rates(age, life, nbar, ppb, t_p, t_p1, f_esc, a_b, k_b)
    assert (rate == 0).any() and (rate > 0).sum() > 100
    a = aton.Aton(w.n, w.n, w.n, w.box_cm, w.params)
    a.set_fields(*[t.cuda() for t in (w.nH, w.x, w.T)])
    t64 = lambda v: torch.from_numpy(np.ascontiguousarray(v, dtype=np.float64))
    res = []
    for dev in ("cpu", "cuda"):
        a.set_fields(*[t.cuda() for t in (w.nH, w.x, w.T)])
        a.set_star_sources(pos.to(dev), t64(age).to(dev), t64(life).to(dev), t64(nbar).to(dev), ppb, t_p, t_p1, f_esc, a_b, k_b)
        a.step(w.dt, 40)
        res.append({k: v.numpy() for k, v in a.get_fields(device="cpu").items()})
    for k in res[0]:
        assert np.array_equal(res[0][k], res[1][k]), k
    # the same run with the oracle's rates through aton_set_sources: bit-identical (the rates agree to the last bit or
    # two; the merged per-cell densities round to the same fp32)
    a.set_fields(*[t.cuda() for t in (w.nH, w.x, w.T)])
    a.set_sources(pos, t64(rate))
    a.step(w.dt, 40)
    plain = {k: v.numpy() for k, v in a.get_fields(device="cpu").items()}
    for k in ("N", "x", "T"):
        assert np.allclose(plain[k], res[0][k], rtol=1e-6, atol=0), k
    a.close()
    # and against the oracle's own run with those sources
    st, p = orc.from_workload(w)
    orc.step(st, p, w.dt, 40, pos.double().numpy(), rate)
    err = l1_errors(res[0], st, p.c)
    assert max(err[k] for k in ("N", "F", "x", "T")) <= 1e-3 and err["x_vol"] <= 1e-3, err
    assert st.x.mean() > 2e-3                                          # the sources did ionise something


def test_thomson_tau_against_oracle(orc):
    from paper_1004_2503_b200 import aton
    a = aton.Aton(8, 8, 8, 8e21, wl.default_params())
    H0 = 72e5 / 3.0856775814913673e24
    rng = np.random.default_rng(3)
    z = np.sort(np.concatenate([[0.0], rng.uniform(0, 18, 400)]))
    x = 1 / (1 + np.exp((z - 7.0) / 0.6))                              # a reionisation history around z = 7
    tau = a.thomson_tau(torch.from_numpy(z), torch.from_numpy(x), 1.9e-7, H0, 0.26)
    assert tau == pytest.approx(orc.thomson_tau(z, x, 1.9e-7, H0, 0.26), rel=1e-12)
    assert 0.03 < tau < 0.06
    with pytest.raises(aton.AtonError):
        a.thomson_tau(torch.from_numpy(z[::-1].copy()), torch.from_numpy(x), 1.9e-7, H0, 0.26)
    a.close()
