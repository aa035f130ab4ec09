"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle on the same seeded inputs.

Tolerances are BASELINE.json's: after 1 step from a warm state max relative error <= 1e-4 on
N, F (as |dF|/(cN), reading S16), x, T where N > 1e-20 max N; after a full run relative L1 <= 1e-3
per field and |d<x>_V| <= 1e-3.
"""
import os

import numpy as np
import pytest
import torch

from paper_1004_2503_b200 import workloads as wl
from parity_util import (gpu_run, l1_errors, max_rel_errors, oracle_run, state_to_workload, twin)

pytestmark = pytest.mark.gpu

TOL_1STEP = float(os.environ.get("ATON_TOL_1STEP", "1e-4"))     # the north_star's bar; the override only ever tightens it (probing)
assert TOL_1STEP <= 1e-4
TOL_L1 = 1e-3
TOL_XVOL = 1e-3
# None = the library's default: the product kernel (variant 5, step_v5_kernel) on the 128-wide grids, its bit-identical
# predecessor (variant 4) on the 32- and 64-wide ones, the variant-2 fallback on the ragged 40^3 one; 0 and 2 are the
# cross-check kernels
VARIANTS = [None, 0, 2]
VIDS = ["default", "v0", "v2"]


_cache = {}


def _warm(orc, w, k):
    key = ("warm", w.name, k, tuple(sorted(w.params.items())))
    if key not in _cache:
        st, _ = oracle_run(orc, w, k)
        _cache[key] = state_to_workload(w, st)
    return _cache[key]


def _oracle_cached(orc, w, n_steps):
    key = ("run", w.name, n_steps, tuple(sorted(w.params.items())), float(w.N.double().sum()))
    if key not in _cache:
        _cache[key] = oracle_run(orc, w, n_steps)
    return _cache[key]


# workloads for the element-by-element checks: (builder, warm-up steps K, full-run steps)
def _cases():
    return {
        "cfg1_32": (lambda: wl.make_config(1), 60, 500),           # config 1 itself, its full 500 steps
        "cfg2_twin64": (lambda: twin(2, 64, 120), 60, 120),
        "cfg3_twin64": (lambda: twin(3, 64, 100), 50, 100),
        "cfg3_twin40": (lambda: twin(3, 40, 100), 50, 100),       # 40: tileable by neither 5 nor 4 -> variant-2 fallback, ragged tail
        "cfg4_twin64": (lambda: twin(4, 64, 100), 50, 100),       # case A + clumping + coll. ion.
        "cfg5_twin32": (lambda: twin(5, 32, 80), 40, 80),
        "cfg4_twin128": (lambda: twin(4, 128, 60), 30, 60),       # 128^3: the default is the product kernel, 16 rows per CTA
    }


@pytest.mark.parametrize("variant", VARIANTS, ids=VIDS)
@pytest.mark.parametrize("case", list(_cases().keys()))
def test_one_step_from_warm_state(orc, case, variant):
    """V2 / reading S17: both codes start from the oracle's state after K steps rounded to fp32."""
    build, k, _ = _cases()[case]
    w = build()
    ww = _warm(orc, w, k)
    st, p = _oracle_cached(orc, ww, 1)
    g, diag = gpu_run(ww, 1, variant)
    err = max_rel_errors(g, st, p.c)
    assert diag["n_nonfinite"] == 0
    for f, e in err.items():
        assert e <= TOL_1STEP, (case, variant, err)


@pytest.mark.parametrize("variant", VARIANTS, ids=VIDS)
@pytest.mark.parametrize("case", list(_cases().keys()))
def test_full_run(orc, case, variant):
    """V3: relative L1 per field <= 1e-3 and ionised volume fraction within 1e-3 after the run."""
    build, _, n_steps = _cases()[case]
    w = build()
    st, p = _oracle_cached(orc, w, n_steps)
    g, diag = gpu_run(w, n_steps, variant)
    err = l1_errors(g, st, p.c)
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == n_steps
    assert err["x_vol"] <= TOL_XVOL, (case, err)
    for f in ("N", "F", "F_rel", "x", "T"):
        assert err[f] <= TOL_L1, (case, variant, err)
    # diagnostics against the oracle's reduction of its own state
    d = orc.reduce(st, p)
    assert diag["x_vol"] == pytest.approx(d["x_vol"], abs=TOL_XVOL)
    assert diag["x_mass"] == pytest.approx(d["x_mass"], abs=2e-3)
    assert diag["photons_total"] == pytest.approx(d["photons_total"], rel=2e-3)
    assert diag["gamma_vol"] == pytest.approx(d["gamma_vol"], rel=2e-3)
    assert diag["f_max"] <= 1.0 + 1e-5 and diag["N_min"] >= 0.0
    # sub-cycle statistics are data dependent (H5) but of the same size
    assert diag["subcycles_total"] == pytest.approx(st.sub_total, rel=0.02)


@pytest.mark.parametrize("variant", VARIANTS, ids=VIDS)
def test_isothermal_and_no_collisions_switches(orc, variant):
    """The other physics-switch combinations (template instantiations) against the oracle."""
    for kw in (dict(cooling=0, coll_ion=0), dict(cooling=0, coll_ion=1, recomb_case=0),
               dict(cooling=1, coll_ion=0, recomb_case=0, clump_model=2, clump_a=3.0, clump_b=0.2),
               dict(cooling=1, coll_ion=0, redshift=9.0),
               # paper-form clumping (Eq.15): C_R = K nH^0.7 and C_I = K' nH^0.2
               dict(cooling=1, coll_ion=1, recomb_case=0, clump_model=2, clump_a=300.0, clump_b=0.7, clump_i_a=8.0, clump_i_b=0.2)):
        # 32^3 (default: variant 4) for every kernel; 128^3 (default: the product kernel, every FLAGS instantiation of it)
        for n, k in ((32, 40),) + (((128, 16),) if variant is None else ()):
            w = twin(3, n, 60)
            w.params.update(kw)
            ww = _warm(orc, w, k)
            st, p = oracle_run(orc, ww, 1)
            g, _ = gpu_run(ww, 1, variant)
            err = max_rel_errors(g, st, p.c)
            assert max(err.values()) <= TOL_1STEP, (n, kw, err)


@pytest.mark.parametrize("case", ["cfg1_32", "cfg3_twin64", "cfg4_twin64", "cfg3_twin40"])
def test_hll_flux_against_oracle(orc, case):
    """SURVEY NEXT-3 / PAPER.md:L85: the HLL intercell flux (aton_params_t.flux = 1) against the oracle's
    orc_transport_hll, same bars as the Lax-Friedrichs path: 1e-4 after one step from the oracle's warm HLL state,
    relative L1 1e-3 after the run; and the run differs from the LF run (it is another scheme, less diffusive)."""
    build, k, n_steps = _cases()[case]
    n_steps = min(n_steps, 150)
    w = build()
    w.params.update(flux=1)
    ww = _warm(orc, w, k)
    st, p = _oracle_cached(orc, ww, 1)
    assert p.flux == 1
    g, diag = gpu_run(ww, 1)
    err = max_rel_errors(g, st, p.c)
    assert diag["n_nonfinite"] == 0 and max(err.values()) <= TOL_1STEP, (case, err)
    st, p = _oracle_cached(orc, w, n_steps)
    g, diag = gpu_run(w, n_steps)
    err = l1_errors(g, st, p.c)
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == n_steps
    assert err["x_vol"] <= TOL_XVOL and max(err[f] for f in ("N", "F", "F_rel", "x", "T")) <= TOL_L1, (case, err)
    assert diag["f_max"] <= 1.0 + 1e-5 and diag["N_min"] >= 0.0
    w.params.update(flux=0)
    g0, _ = gpu_run(w, n_steps)
    assert np.abs(g0["N"] - g["N"]).sum() > 1e-2 * np.abs(g["N"]).sum()


@pytest.mark.parametrize("flux", [0, 1], ids=["lf", "hll"])
def test_switching_kernels_between_steps_changes_nothing_beyond_rounding(flux):
    """One context, the kernel changed between chunks of steps (5 -> 4 -> 2 -> 0 -> 5; with flux = 1: packed tiled ->
    one thread per cell -> tiled): no stale mask bit, queue entry, captured graph or argument block survives a switch.
    Compared with the same steps run by the default kernel alone (the variants agree to rounding)."""
    from paper_1004_2503_b200 import aton
    nx, ny, nz = 128, 16, 10
    nH, x, T, p, dx, pos, rate = _slab_case(nx, ny, nz, True, seed=77)
    p = dict(p, flux=flux)
    dt = wl.courant_dt(dx)
    f = [torch.from_numpy(np.ascontiguousarray(v, dtype=np.float32)).cuda() for v in (nH, x, T)]

    def run(plan):
        a = aton.Aton(nx, ny, nz, dx * nx, p)
        a.set_fields(*f)
        a.set_sources(torch.from_numpy(pos), torch.from_numpy(rate))
        for variant, n in plan:
            a.set_kernel(variant)
            a.step(dt, n)
        g = {k: v.numpy() for k, v in a.get_fields(device="cpu").items()}
        d = a.reduce()
        a.close()
        return g, d

    ref, dref = run([(5, 16)])
    mix, dmix = run([(5, 3), (4, 2), (2, 4), (0, 3), (5, 4)])
    assert dmix["steps_done"] == 16 and dmix["n_nonfinite"] == 0 and dref["cells_subcycled"] > 0
    for k in ("N", "Fx", "Fy", "Fz", "x", "T"):
        num = np.abs(ref[k].astype(np.float64) - mix[k]).sum()
        assert num <= 1e-5 * np.abs(ref[k].astype(np.float64)).sum(), (flux, k)
    for k in ("x", "T"):
        assert np.allclose(ref[k], mix[k], rtol=3e-4, atol=0), (flux, k)
    assert dmix["photons_total"] == pytest.approx(dref["photons_total"], rel=1e-5)
    assert dmix["subcycles_total"] == pytest.approx(dref["subcycles_total"], rel=1e-2)


def test_hll_tiled_kernel_agrees_with_the_one_thread_per_cell_kernel():
    """The tiled HLL kernel (default on grids with nx % 32 == 0 and ny % 8 == 0: every cell closed once per plane, records
    shared through shared memory, the product path's chemistry: fast sub-step + fix-up kernels) against step_hll_kernel
    (variant 0: one thread per cell, chemistry in place) -- on grids whose tiles wrap every periodic seam, ragged z chunks
    and nz = 1 included.  Same face formula in the same order: equal to rounding (both are held to the oracle separately,
    test_hll_flux_against_oracle)."""
    # 64-wide grids run the packed kernel (step_hll_pk_kernel), 32- and 96-wide ones the scalar tiled kernel
    for shape, steps in (((64, 16, 37), 20), ((32, 8, 1), 6), ((96, 24, 5), 12), ((64, 8, 1), 6), ((128, 8, 2), 8), ((192, 16, 33), 10)):
        nx, ny, nz = shape
        nH, x, T, p, dx, pos, rate = _slab_case(nx, ny, nz, True, seed=nx + nz)
        p = dict(p, flux=1)
        tiled, dt_ = _run_slab(5, (0, 0), nH, x, T, p, dx, pos, rate, steps)
        ref, dr = _run_slab(0, (0, 0), nH, x, T, p, dx, pos, rate, steps)
        assert dt_["n_nonfinite"] == 0 and dt_["photons_total"] > 0
        # F components against their natural scale c sum N (reading S16): with nz = 1 or 2 the z flux vanishes by symmetry
        # and what is left of it in either kernel is rounding noise
        cn = wl.C_CM_S * np.abs(ref["N"].astype(np.float64)).sum()
        for k in ("N", "Fx", "Fy", "Fz", "x", "T"):
            num = np.abs(ref[k].astype(np.float64) - tiled[k]).sum()
            den = cn if k[0] == "F" else np.abs(ref[k].astype(np.float64)).sum()
            assert num <= 1e-5 * den, (shape, k, num / den)
        for k in ("x", "T"):
            assert np.allclose(ref[k], tiled[k], rtol=3e-4, atol=0), (shape, k)
        assert dt_["subcycles_total"] == pytest.approx(dr["subcycles_total"], rel=1e-2)
        assert dt_["photons_total"] == pytest.approx(dr["photons_total"], rel=1e-5)


@pytest.mark.parametrize("variant", VARIANTS, ids=VIDS)
def test_reduce_matches_oracle(orc, variant):
    w = wl.synthetic_warm_state(twin(4, 32, 10))
    g, diag = gpu_run(w, 0, variant)
    st, p = orc.from_workload(w)
    d = orc.reduce(st, p)
    for k in ("x_vol", "x_mass", "gamma_vol", "gamma_mass", "photons_total", "T_vol", "N_min", "frac_x_half"):
        assert diag[k] == pytest.approx(d[k], rel=1e-6), k
    assert diag["f_max"] == pytest.approx(d["f_max"], rel=1e-5)
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == 0
    # upload -> download is the identity on n_H, x, T, N and within 2 ulp on F (stored as F/c)
    for k, src in (("nH", w.nH), ("x", w.x), ("T", w.T), ("N", w.N)):
        assert np.array_equal(g[k], src.numpy())
    assert np.allclose(g["Fx"], w.Fx.numpy(), rtol=3e-7, atol=0)


@pytest.mark.parametrize("variant", VARIANTS, ids=VIDS)
def test_determinism_and_checkpoint(variant):
    """V4: two runs are bit-identical, also when the steps are cut into several calls; and SURVEY 5's checkpoint:
    run 2k steps == run k, aton_get_fields, aton_set_fields into a NEW context, run k.  n_H, x, T, N round-trip
    bit-exactly; F does not (the device carries G = F/c: F -> fl(F/c) -> fl(c G) moves F by <= 2 ulp), so the resumed
    run agrees to rounding, not bitwise: stated tolerance 2e-5 relative per field after k more steps (2 ulp of F
    per restart, amplified by nothing: the scheme is a convex combination)."""
    from paper_1004_2503_b200 import aton
    w = wl.synthetic_warm_state(twin(4, 64, 10))
    a, da = gpu_run(w, 12, variant)
    b, _ = gpu_run(w, 12, variant)
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    c, _ = gpu_run(w, 12, variant, chunks=[5, 7])          # buffer parity across calls
    for k in a:
        assert np.array_equal(a[k], c[k]), k
    # checkpoint / resume through the public calls
    first = aton.from_workload(w)
    if variant is not None:
        first.set_kernel(variant)
    first.step(w.dt, 6)
    snap = first.get_fields(device="cpu")                  # the "snapshot every ~5000 steps" of PAPER.md:L411
    d6 = first.reduce()
    first.close()
    second = aton.Aton(w.n, w.n, w.n, w.box_cm, w.params)
    if variant is not None:
        second.set_kernel(variant)
    second.set_fields(*[snap[k].cuda() for k in ("nH", "x", "T", "N", "Fx", "Fy", "Fz")])
    second.set_sources(w.src_pos.contiguous(), w.src_rate.contiguous())
    again = second.get_fields(device="cpu")
    for k in ("nH", "x", "T", "N"):
        assert torch.equal(again[k], snap[k]), k           # exact round trip
    assert torch.allclose(again["Fx"], snap["Fx"], rtol=3e-7, atol=0)
    second.step(w.dt, 6)
    r = {k: v.numpy() for k, v in second.get_fields(device="cpu").items()}
    d12 = second.reduce()
    second.close()
    for k in ("N", "x", "T"):
        assert np.allclose(r[k], a[k], rtol=2e-5, atol=0), k
    for k in ("Fx", "Fy", "Fz"):
        assert np.abs(r[k] - a[k]).max() <= 2e-5 * wl.C_CM_S * a["N"].max(), k
    assert d12["steps_done"] == 6 and d6["steps_done"] == 6 and da["steps_done"] == 12
    assert d12["x_vol"] == pytest.approx(da["x_vol"], rel=1e-6)


def test_fixup_queue_is_race_free_under_load():
    """The fix-up kernel's shared-memory queue drains whenever it crosses its threshold: the decision must be the same
    for every thread of the block (a block-wide vote).  A state where ~10 % of the cells sub-cycle crosses the
    threshold thousands of times per step: repeated runs must be bit-identical (a racy drain redoes or skips cells)."""
    w = wl.synthetic_warm_state(twin(4, 128, 10))
    ref, dref = gpu_run(w, 3, None)
    assert dref["cells_subcycled"] > 0.02 * 3 * 128 ** 3
    for _ in range(8):
        g, d = gpu_run(w, 3, None)
        for k in ref:
            assert np.array_equal(ref[k], g[k]), k
        assert d["subcycles_total"] == dref["subcycles_total"] and d["cells_fp64"] == dref["cells_fp64"]


@pytest.mark.parametrize("variant", [None, 0, 2], ids=VIDS)
def test_cuda_graph_replay_equals_plain_launches(variant):
    """Small grids replay a captured pair of steps (aton_step with n_steps >= 4); stepping one step per
    call never captures.  Same bits, same counters, whatever the parity of the step counts and after a change of dt."""
    from paper_1004_2503_b200 import aton
    w = wl.make_config(1)
    runs = []
    for chunks in ([41], [1] * 41, [7, 1, 12, 21], [4, 37]):
        a = aton.from_workload(w)
        if variant is not None:
            a.set_kernel(variant)
        for c in chunks:
            a.step(w.dt, c)
        a.step(0.5 * w.dt, 9 if len(chunks) != 41 else 1)            # new dt: the captured graph must be rebuilt
        for _ in range(8 if len(chunks) == 41 else 0):
            a.step(0.5 * w.dt, 1)
        runs.append(({k: v.numpy() for k, v in a.get_fields(device="cpu").items()}, a.reduce(), a.launch_count()))
        a.close()
    for g, d, launches in runs[1:]:
        for k in g:
            assert np.array_equal(g[k], runs[0][0][k]), k
        for k in ("steps_done", "subcycles_total", "subcycles_max", "cells_subcycled", "cells_fp64"):
            assert d[k] == runs[0][1][k], k
        assert d["time_s"] == pytest.approx(runs[0][1]["time_s"], rel=1e-12)
        assert launches == runs[0][2]                                # gpu_launches counts replayed kernels too
    assert runs[0][1]["steps_done"] == 50


@pytest.mark.parametrize("variant,tiles", [(2, ((6, 0), (14, 0), (6, 5), (6, 40), (14, 1)))], ids=["v2"])
def test_tile_shape_independence(variant, tiles):
    """V4: the tiled kernels' result does not depend on the tile shape (bitwise)."""
    w = wl.synthetic_warm_state(twin(5, 40, 10))
    ref, dref = gpu_run(w, 6, variant, (0, 0))
    for tile in tiles:
        g, d = gpu_run(w, 6, variant, tile)
        for k in ref:
            assert np.array_equal(ref[k], g[k]), (tile, k)
        assert d["subcycles_total"] == dref["subcycles_total"] and d["cells_subcycled"] == dref["cells_subcycled"]


def test_tiled_vs_reference_kernel():
    """The three kernels differ only in rounding order (and in which cells take the sub-cycled path when the 10 %
    rule is decided within rounding: H5, continuous in the result)."""
    w = wl.synthetic_warm_state(twin(4, 64, 10))
    a, da = gpu_run(w, 3, 0)
    for variant in (2, 4):
        b, db = gpu_run(w, 3, variant)
        # each kernel is within 1e-4 of the oracle per step (the 1-step bar); two of them within 2e-4 of each other
        # per step, here over 3 steps from a state where half the cells sub-cycle
        for k in ("N", "x", "T"):
            assert np.allclose(a[k], b[k], rtol=3e-4, atol=0), (variant, k)
            assert np.mean(np.abs(a[k] - b[k]) > 2e-5 * np.abs(a[k])) < 1e-3, (variant, k)
        assert db["subcycles_total"] == pytest.approx(da["subcycles_total"], rel=1e-3)
        assert db["subcycles_max"] == da["subcycles_max"]


@pytest.mark.parametrize("variant", [2, 4], ids=["v2", "v4"])
def test_fixup_path_statistics(variant):
    """Cells that need sub-cycling are redone by the fix-up kernel, counted, and nothing is left queued (a second
    identical context gives the same counts); an isothermal run never sub-cycles (variant 4 still hands its one source
    cell per step to the fix-up kernel)."""
    w = wl.make_config(1)
    g, d = gpu_run(w, 40, variant)
    assert d["cells_subcycled"] > 0 and d["subcycles_max"] > 1
    assert d["subcycles_total"] > 40 * w.n ** 3
    assert 0 <= d["cells_fp64"] <= d["cells_subcycled"]
    g1, d1 = gpu_run(w, 40, variant)
    assert all(d1[k] == d[k] for k in ("cells_subcycled", "subcycles_total", "subcycles_max", "cells_fp64"))
    w2 = wl.make_config(1)
    w2.params.update(cooling=0)
    g2, d2 = gpu_run(w2, 10, variant)
    assert d2["cells_subcycled"] == (10 if variant == 4 else 0) and d2["cells_fp64"] == 0
    assert d2["subcycles_max"] == 1 and d2["subcycles_total"] == 10 * w.n ** 3


def test_non_cubic_grid_and_source_edges(orc):
    """nx != ny != nz, sources on cell edges / shared cells / the last cell, against the oracle."""
    from paper_1004_2503_b200 import aton
    nx, ny, nz = 24, 10, 7
    rng = np.random.default_rng(11)
    nH = (10 ** rng.uniform(-4, -2, (nz, ny, nx))).astype(np.float32)
    x = np.full((nz, ny, nx), 1e-3, np.float32)
    T = np.full((nz, ny, nx), 100.0, np.float32)
    p = wl.default_params()
    dx = 2.0e21
    pos = np.array([[0.0, 0.0, 0.0], [0.999999, 0.999999, 0.999999], [0.5, 0.5, 0.5], [0.5, 0.5, 0.5],
                    [1.0 / 24 * 3, 0.3, 0.2], [1.0, 0.0, 0.0]], np.float32)
    rate = np.array([1e50, 2e50, 3e50, 1e50, 5e49, 7e49])
    dt = wl.courant_dt(dx)
    for variant in (0, 2, 4):                 # 4 cannot tile 24 x 10: it runs the variant-2 kernel
        a = aton.Aton(nx, ny, nz, dx * nx, p)
        a.set_kernel(variant)
        a.set_fields(*[torch.from_numpy(v).cuda() for v in (nH, x, T)])
        a.set_sources(torch.from_numpy(pos), torch.from_numpy(rate))
        a.step(dt, 20)
        g = {k: v.numpy() for k, v in a.get_fields(device="cpu").items()}
        st = orc.State(nH, x, T, np.zeros_like(nH), np.zeros_like(nH), np.zeros_like(nH), np.zeros_like(nH))
        op = orc.make_params(p, dx, float(nH.astype(np.float64).mean()))
        orc.step(st, op, dt, 20, pos.astype(np.float64), rate)
        err = l1_errors(g, st, op.c)
        assert max(err.values()) <= TOL_L1, (variant, err)
        a.close()


def test_api_errors():
    from paper_1004_2503_b200 import aton
    p = wl.default_params()
    with pytest.raises(aton.AtonError) as e:
        aton.Aton(10, 8, 8, 1e21, p)                                  # nx % 4 != 0
    assert e.value.code == aton.EINVAL
    a = aton.Aton(8, 8, 8, 8e21, p)
    with pytest.raises(aton.AtonError) as e:
        a.step(1.0, 1)                                                # before set_fields
    assert e.value.code == aton.ESTATE
    one = torch.ones(8, 8, 8, device="cuda")
    with pytest.raises(aton.AtonError) as e:
        a.set_fields(0 * one, one, one)                               # n_H must be > 0
    assert e.value.code == aton.EINVAL
    a.set_fields(1e-3 * one, 1e-3 * one, 100 * one)
    with pytest.raises(aton.AtonError) as e:
        a.step(a.courant_dt(1.01), 1)                                 # c dt/dx > 1/3
    assert e.value.code == aton.EINVAL and "unstable" in str(e.value)
    assert a.courant_dt(0.8) == pytest.approx(0.8 * 1e21 / (3 * wl.C_CM_S))
    with pytest.raises(aton.AtonError):
        a.set_sources(torch.tensor([[1.5, 0.0, 0.0]]), torch.tensor([1e50], dtype=torch.float64))
    with pytest.raises(aton.AtonError):
        a.set_sources(torch.tensor([[0.5, 0.0, 0.0]]), torch.tensor([-1.0], dtype=torch.float64))
    a.step(0.0, 2)                                                    # dt <= 0 => Courant 0.8
    d = a.reduce()
    assert d["steps_done"] == 2 and d["time_s"] == pytest.approx(2 * a.courant_dt(0.8))
    assert a.launch_count() > 0
    for gone in (1, 3, 6, -1):
        with pytest.raises(aton.AtonError):
            a.set_kernel(gone)                                            # round 1's variants 1 and 3 no longer exist
    a.close()


def test_empty_sources_and_vacuum_conservation():
    """No sources, no absorption possible (x = 1 exactly): photons are conserved to fp32 rounding."""
    from paper_1004_2503_b200 import aton
    n = 32
    w = wl.synthetic_warm_state(twin(3, n, 10))
    p = dict(w.params); p.update(cooling=0, coll_ion=0)
    a = aton.Aton(n, n, n, w.box_cm, p)
    one = torch.ones(n, n, n, device="cuda")
    a.set_fields(1e-12 * one, one, 1e4 * one, w.N.cuda(), w.Fx.cuda(), w.Fy.cuda(), w.Fz.cuda())
    a.set_sources(None, None)
    before = a.reduce()["photons_total"]
    a.step(w.dt, 50)
    d = a.reduce()
    assert d["photons_total"] == pytest.approx(before, rel=2e-5)
    assert d["N_min"] >= 0 and d["f_max"] <= 1 + 1e-5
    a.close()


# ------------------------------------------------------------------------------------------------
# Non-cubic grids for the tiled kernels (variant 5: 128-cell row segments, 8 or 16 rows per CTA; variant 4: x extents of
# one to eight 32-cell warp tiles, ragged last CTA): several y tiles, ragged z chunks, sources on tile corners / edges and
# across every periodic seam.
# ------------------------------------------------------------------------------------------------
def _slab_case(nx, ny, nz, flags7, seed, paper_clumping=False):
    """Random log-normal-ish density on an (nz, ny, nx) grid, sources on tile corners / edges, physics of
    config 4 (flags7: case A + recombination radiation + clumping) or config 2 (case B)."""
    rng = np.random.default_rng(seed)
    nH = (2e-4 * np.exp(1.5 * rng.standard_normal((nz, ny, nx)) - 1.125)).astype(np.float32)
    x = np.full((nz, ny, nx), 1e-3, np.float32)
    T = np.full((nz, ny, nx), 100.0, np.float32)
    p = wl.default_params()
    p.update(redshift=8.0)
    if flags7:
        p.update(recomb_case=0, clump_model=1, clump_a=1.0, clump_b=2.0)
    if paper_clumping:      # Eq.15 with the fitted trends C_R ~ nH^0.7, C_I ~ nH^0.2 (L259, L269)
        p.update(clump_model=2, clump_a=300.0, clump_b=0.7, clump_i_a=8.0, clump_i_b=0.2)
    dx = 3.0e21
    cells = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (127 % nx, 7 % ny, 1 % nz), (128 % nx, 8 % ny, 2 % nz), (nx // 2, ny // 2, nz // 2),
             (3, ny - 1, 0), (nx - 4, 0, nz - 1)]
    pos = np.array([[(i + 0.5) / nx, (j + 0.5) / ny, (k + 0.5) / nz] for i, j, k in cells], np.float32)
    rate = 10 ** rng.uniform(49.5, 51, len(cells))
    return nH, x, T, p, dx, pos, rate


def _run_slab(variant, tile, nH, x, T, p, dx, pos, rate, n_steps, rad=None):
    from paper_1004_2503_b200 import aton
    nz, ny, nx = nH.shape
    a = aton.Aton(nx, ny, nz, dx * nx, p)
    a.set_kernel(variant, *tile)
    f = [torch.from_numpy(np.ascontiguousarray(v, dtype=np.float32)).cuda() for v in (nH, x, T) + tuple(rad or ())]
    a.set_fields(*f)
    a.set_sources(torch.from_numpy(pos), torch.from_numpy(rate))
    a.step(wl.courant_dt(dx), n_steps)
    g = {k: v.numpy() for k, v in a.get_fields(device="cpu").items()}
    d = a.reduce()
    a.close()
    return g, d


@pytest.mark.parametrize("variant,shape,flags7",
                         [(4, (128, 16, 11), True), (4, (256, 24, 9), False), (4, (32, 8, 5), True),
                          (4, (160, 12, 1), True), (4, (64, 4, 70), False), (4, (96, 8, 7), "paper"),
                          (5, (128, 16, 11), True), (5, (256, 24, 9), False), (5, (128, 8, 70), False),
                          (5, (384, 32, 1), True), (5, (128, 16, 7), "paper")],
                         ids=["v4_128x16x11_A", "v4_256x24x9_B",
                              "v4_32x8x5_A", "v4_160x12x1_A", "v4_64x4x70_B", "v4_96x8x7_paper_clumping",
                              "v5_128x16x11_A", "v5_256x24x9_B", "v5_128x8x70_B", "v5_384x32x1_A",
                              "v5_128x16x7_paper_clumping"])
def test_full_tile_kernels_against_oracle(orc, variant, shape, flags7):
    nx, ny, nz = shape
    nH, x, T, p, dx, pos, rate = _slab_case(nx, ny, nz, bool(flags7), seed=nx + ny + nz, paper_clumping=flags7 == "paper")
    dt = wl.courant_dt(dx)
    op = orc.make_params(p, dx, float(nH.astype(np.float64).mean()))
    zero = np.zeros_like(nH)
    # full run from the dark start (V3 metric)
    st = orc.State(nH, x, T, zero, zero, zero, zero)
    orc.step(st, op, dt, 40, pos.astype(np.float64), rate)
    g, d = _run_slab(variant, (0, 0), nH, x, T, p, dx, pos, rate, 40)
    err = l1_errors(g, st, op.c)
    assert d["n_nonfinite"] == 0 and max(err.values()) <= TOL_L1, err
    assert d["subcycles_total"] == pytest.approx(st.sub_total, rel=0.02)
    # one step from the oracle's warm state rounded to fp32 (V2 metric)
    warm = [np.ascontiguousarray(v, dtype=np.float32) for v in (st.x, st.T, st.N, st.Fx, st.Fy, st.Fz)]
    st1 = orc.State(nH, *warm)
    orc.step(st1, op, dt, 1, pos.astype(np.float64), rate)
    if variant == 5:    # rows per CTA (8 or 16) x planes per z chunk
        tiles = ((0, 0), (0, 1), (8, 3), (8, 64)) + (((16, 0), (16, 5)) if ny % 16 == 0 else ())
    else:
        tiles = ((0, 0), (0, 1), (4, 3), (4, 64)) + (((2, 0), (2, 5)) if nx % 64 == 0 else ())
    for tile in tiles:
        g1, d1 = _run_slab(variant, tile, nH, warm[0], warm[1], p, dx, pos, rate, 1, rad=warm[2:])
        e1 = max_rel_errors(g1, st1, op.c)
        assert max(e1.values()) <= TOL_1STEP, (tile, e1)


@pytest.mark.parametrize("variant,tiles", [(4, ((0, 0), (0, 1), (2, 2), (4, 0), (4, 5), (2, 13))),
                                           (5, ((0, 0), (0, 1), (8, 2), (16, 0), (16, 5), (8, 13)))], ids=["v4", "v5"])
def test_full_tile_kernels_tile_shape_independence_determinism_and_v2_agreement(variant, tiles):
    nH, x, T, p, dx, pos, rate = _slab_case(256, 32, 13, True, seed=5)
    ref, dref = _run_slab(variant, (0, 0), nH, x, T, p, dx, pos, rate, 25)
    assert dref["cells_subcycled"] > 0
    if variant == 5:    # variant 5 adds the neighbour terms in variant 4's order: the two agree bit for bit
        g4, d4 = _run_slab(4, (0, 0), nH, x, T, p, dx, pos, rate, 25)
        for k in ref:
            assert np.array_equal(ref[k], g4[k]), ("v4", k)
        assert d4["subcycles_total"] == dref["subcycles_total"]
    for tile in tiles:
        g, d = _run_slab(variant, tile, nH, x, T, p, dx, pos, rate, 25)
        for k in ref:
            assert np.array_equal(ref[k], g[k]), (tile, k)
        assert d["subcycles_total"] == dref["subcycles_total"] and d["cells_subcycled"] == dref["cells_subcycled"]
    # variant 2 sums the x and y neighbour terms in another order: equal to rounding
    g2, d2 = _run_slab(2, (0, 0), nH, x, T, p, dx, pos, rate, 25)
    for k in ("N", "x", "T"):
        assert np.allclose(ref[k], g2[k], rtol=5e-5, atol=0), k
    assert d2["subcycles_total"] == pytest.approx(dref["subcycles_total"], rel=1e-3)


# ------------------------------------------------------------------------------------------------
# BASELINE.json's full size (config 5, 1024^3) in the launch configuration bench.py times (default
# kernel variant and tile shape).  The oracle cannot run 2^30 cells, but the scheme's domain of
# dependence is one cell per step: a (m + 2p)^3 sub-cube of the INPUT state advanced p steps by the
# oracle (with whatever boundary) is exact in its inner m^3, which is compared with the same cells of
# the full-grid GPU run.  Both codes start from generator output only (dark start, or
# workloads.synthetic_warm_state): no oracle input comes from the CUDA path.
# ------------------------------------------------------------------------------------------------
def _subcube_sources(w, org, size):
    """Sources of the full grid that fall inside the periodic sub-cube at `org`, as (positions in sub-cube units, rates)."""
    n = w.n
    src_cell = torch.floor(w.src_pos.double() * n).long() % n           # (ns, 3) as (i, j, k)
    rel = (src_cell - torch.tensor(org)) % n
    inside = (rel < size).all(dim=1)
    return ((rel[inside].double() + 0.5) / size).numpy(), w.src_rate[inside].numpy()


def _subcube_check(orc, w, state_name, origins, m, p_steps, nH_mean):
    """p_steps of the full grid on the GPU against the oracle on (m + 2 p_steps)^3 sub-cubes: relative L1 of the inner
    m^3 (BASELINE.json's full-run metric; the per-cell 1-step bar is _onestep_check's job)."""
    from paper_1004_2503_b200 import aton
    n, size = w.n, m + 2 * p_steps
    a = aton.from_workload(w)
    a.step(w.dt, p_steps)
    out = a.get_fields(device="cuda", names=("x", "T", "N", "Fx", "Fy", "Fz"))
    diag = a.reduce()
    a.close()
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == p_steps
    worst = {}
    for org in origins:
        cut = {k: wl.cut_subcube(getattr(w, k), org, size).numpy() for k in ("nH", "x", "T", "N", "Fx", "Fy", "Fz")}
        st = orc.State(*[cut[k] for k in ("nH", "x", "T", "N", "Fx", "Fy", "Fz")])
        op = orc.make_params(w.params, w.dx, nH_mean)
        pos, rate = _subcube_sources(w, org, size)
        orc.step(st, op, w.dt, p_steps, pos, rate)
        sl = slice(p_steps, p_steps + m)
        inner_org = tuple(o + p_steps for o in org)
        g = {k: wl.cut_subcube(out[k], inner_org, m).numpy() for k in out}
        ref = type("S", (), {k: getattr(st, k)[sl, sl, sl] for k in ("N", "Fx", "Fy", "Fz", "x", "T")})
        err = l1_errors(g, ref, op.c)
        for k, e in err.items():
            worst[k] = max(worst.get(k, 0.0), e)
        assert max(err[k] for k in ("N", "F", "x", "T")) <= TOL_L1, (state_name, org, len(rate), err)
    return worst, diag


def _paste_subcube(dst, src, org):
    """dst[z0:z0+s, y0:y0+s, x0:x0+s] = src, periodic; dst on the GPU, src a numpy array."""
    n, s = dst.shape[0], src.shape[0]
    x0, y0, z0 = org
    iz = (torch.arange(s, device=dst.device) + z0) % n
    iy = (torch.arange(s, device=dst.device) + y0) % n
    ix = (torch.arange(s, device=dst.device) + x0) % n
    dst[iz[:, None, None], iy[None, :, None], ix[None, None, :]] = torch.from_numpy(np.ascontiguousarray(src, dtype=np.float32)).to(dst.device)


def _onestep_check(orc, w, origins, size, k_warm, nH_mean):
    """The north_star's 1-step bar at full size, in the bench's launch configuration: max relative error <= 1e-4 on
    N, F, x, T (where N > 1e-20 max N) after ONE step.  Two kinds of start, both made without the CUDA path:
      (a) oracle-evolved: each `size`^3 sub-cube of the dark full-size workload (its density, its sources) is evolved
          k_warm steps by the oracle as a small periodic box, rounded to fp32 and pasted into the full-size state;
      (b) the generator's synthetic warm state everywhere else (far from equilibrium: the heaviest sub-cycling).
    The GPU advances the WHOLE grid one step with the default kernel; the oracle advances each sub-cube one step;
    the cells whose stencil stays inside the sub-cube (the inner (size-2)^3) are compared one by one."""
    from paper_1004_2503_b200 import aton
    op = orc.make_params(w.params, w.dx, nH_mean)
    ww = wl.synthetic_warm_state(w)
    names = ("x", "T", "N", "Fx", "Fy", "Fz")
    for org in origins[0::2]:                                           # (a): evolve from the dark start, paste
        cut = {k: wl.cut_subcube(getattr(w, k), org, size).numpy() for k in ("nH",) + names}
        st = orc.State(*[cut[k] for k in ("nH",) + names])
        pos, rate = _subcube_sources(w, org, size)
        orc.step(st, op, w.dt, k_warm, pos, rate)
        for k in names:
            _paste_subcube(getattr(ww, k), getattr(st, k), org)
    refs = []
    for org in origins:                                                 # both kinds: one oracle step from what the GPU gets
        cut = {k: wl.cut_subcube(getattr(ww, k), org, size).numpy() for k in ("nH",) + names}
        st = orc.State(*[cut[k] for k in ("nH",) + names])
        pos, rate = _subcube_sources(w, org, size)
        orc.step(st, op, w.dt, 1, pos, rate)
        refs.append((org, st, cut, len(rate)))
    a = aton.from_workload(ww)
    del ww
    torch.cuda.empty_cache()
    a.step(w.dt, 1)
    out = a.get_fields(device="cuda", names=names)
    diag = a.reduce()
    a.close()
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == 1
    worst = {}
    sl = slice(1, size - 1)
    bad = []
    for org, st, cut, nsrc in refs:
        g = {k: wl.cut_subcube(out[k], tuple(o + 1 for o in org), size - 2).numpy() for k in names}
        ref = type("S", (), {k: getattr(st, k)[sl, sl, sl] for k in names})
        err = max_rel_errors(g, ref, op.c)
        for k, e in err.items():
            worst[k] = max(worst.get(k, 0.0), e)
        if max(err.values()) > TOL_1STEP:                              # name the worst cells: start state -> both results
            big = ref.N > 1e-20 * ref.N.max()
            for k in ("x", "T", "N"):
                e = np.abs(g[k] - getattr(ref, k)) / np.maximum(np.abs(getattr(ref, k)), 1e-300)
                if k == "N":
                    e = np.where(big, e, 0.0)
                for idx in np.argsort(e.ravel())[::-1][:3]:
                    kk, jj, ii = np.unravel_index(idx, e.shape)
                    if e[kk, jj, ii] > TOL_1STEP:
                        c0 = {f: float(cut[f][kk + 1, jj + 1, ii + 1]) for f in ("nH", "x", "T", "N")}
                        bad.append((org, nsrc, k, float(e[kk, jj, ii]), c0,
                                    {f: (float(g[f][kk, jj, ii]), float(getattr(ref, f)[kk, jj, ii])) for f in ("x", "T", "N")}))
            bad.append((org, nsrc, "max-rel", err, int(st.sub_max)))
    for b in bad:
        print("1-step bar violated:", b)
    print("1-step check:", {k: diag[k] for k in ("cells_subcycled", "cells_fp64", "subcycles_max")}, "worst", worst)
    assert not bad, bad[-1]
    return worst, diag


def _have_hbm(gb):
    return torch.cuda.is_available() and torch.cuda.get_device_properties(0).total_memory >= gb * 1e9


def _origins(w, size):
    """Sub-cubes: around the two brightest sources, across the periodic corner, across CTA / tile seams, a void."""
    n = w.n
    cells = (torch.floor(w.src_pos.double() * n).long() % n)
    top = torch.argsort(w.src_rate, descending=True)[:2]
    half = size // 2
    origins = [tuple(int(v) for v in ((cells[s] - half) % n)) for s in top]
    origins += [(n - 20, n - 20, n - 20), (128 - 20, 4 * 37 - 20, 64 - 20)]
    flat = int(torch.argmin(w.nH.reshape(-1)[: n * n * 64]))
    origins.append(tuple(int(v) for v in ((torch.tensor([flat % n, (flat // n) % n, flat // (n * n)]) - half) % n)))
    return origins


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_configs_on_subcubes_against_oracle(orc, cfg):
    """Configs 3 (256^3), 4 (512^3) and 5 (1024^3) at BASELINE.json's full grid sizes, default kernel and tile:
    8 steps from the dark start and from the synthetic warm state, relative L1 on sub-cubes."""
    n = {3: 256, 4: 512, 5: 1024}[cfg]
    if not _have_hbm(150 if cfg == 5 else 30):
        pytest.skip("needs the full working set in HBM (about 110 GB for 1024^3)")
    m, p_steps = 24, 8
    w = wl.make_config(cfg, device="cuda")
    assert w.n == n
    nH_mean = float(w.nH.double().mean())
    origins = _origins(w, m + 2 * p_steps)
    dark, _ = _subcube_check(orc, w, "dark", origins, m, p_steps, nH_mean)
    ww = wl.synthetic_warm_state(w)
    del w
    torch.cuda.empty_cache()
    warm, dw = _subcube_check(orc, ww, "warm", origins, m, p_steps, nH_mean)
    print(f"config {cfg}: worst relative L1 on sub-cubes: dark", dark, "warm", warm, "fp64 cells", dw["cells_fp64"])


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_one_step_bar(orc, cfg):
    """The 1-step bar (max relative error 1e-4, cell by cell) at the full grid sizes of configs 3-5."""
    n = {3: 256, 4: 512, 5: 1024}[cfg]
    if not _have_hbm(150 if cfg == 5 else 30):
        pytest.skip("needs the full working set in HBM (about 110 GB for 1024^3)")
    w = wl.make_config(cfg, device="cuda")
    assert w.n == n
    size = 40
    worst, diag = _onestep_check(orc, w, _origins(w, size), size, 16, float(w.nH.double().mean()))
    print(f"config {cfg}: worst 1-step max-rel errors on sub-cubes", worst, "cells redone", diag["cells_subcycled"],
          "in fp64", diag["cells_fp64"], "max sub-cycles", diag["subcycles_max"])


def _full_run(orc, w, steps):
    st, p = oracle_run(orc, w, steps)
    g, diag = gpu_run(w, steps)
    err = l1_errors(g, st, p.c)
    assert diag["n_nonfinite"] == 0 and diag["steps_done"] == steps
    assert err["x_vol"] <= TOL_XVOL and max(err[k] for k in ("N", "F", "F_rel", "x", "T")) <= TOL_L1, err
    d = orc.reduce(st, p)
    assert diag["x_mass"] == pytest.approx(d["x_mass"], abs=2e-3) and diag["photons_total"] == pytest.approx(d["photons_total"], rel=2e-3)
    assert diag["subcycles_total"] == pytest.approx(st.sub_total, rel=0.02)
    return err, diag


def test_config2_full_run_against_oracle(orc):
    """Config 2 in full: its 128^3 grid, all of its 1000 steps, default kernel (variant 5), against the oracle run on
    the whole grid (about 100 s of oracle on 16 cores) -- BASELINE.json's full-run metric."""
    w = wl.make_config(2)
    assert w.n == 128 and w.n_steps == 1000
    err, diag = _full_run(orc, w, w.n_steps)
    print("config 2, 1000 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


@pytest.mark.skipif(os.environ.get("ATON_SLOW", "") != "1", reason="config 3 in full is ~30 min of oracle: set ATON_SLOW=1")
def test_config3_full_run_against_oracle(orc):
    """Config 3 in full: 256^3, 2000 steps (opt-in; the result of the round's run is recorded in DESIGN.md)."""
    w = wl.make_config(3)
    assert w.n == 256 and w.n_steps == 2000
    err, diag = _full_run(orc, w, w.n_steps)
    print("config 3, 2000 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


@pytest.mark.skipif(os.environ.get("ATON_SLOW4", "") != "1", reason="512^3 on the whole grid is ~15 min of oracle: set ATON_SLOW4=1")
def test_config4_first_steps_on_the_whole_grid_against_oracle(orc):
    """Config 4 on its full 512^3 grid (case A + recombination radiation, collisional ionisation, cooling, C_R = max(1, 1 + 2 delta),
    2e4 sources), the first 120 of its 1000 steps, the WHOLE grid against the oracle (opt-in; the result of the round's run is
    recorded in DESIGN.md) -- the sub-cube tests see 5 x 24^3 cells of this grid, this one all 1.3e8."""
    w = wl.make_config(4)
    assert w.n == 512 and w.n_steps == 1000
    err, diag = _full_run(orc, w, 120)
    print("config 4, 120 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


@pytest.mark.skipif(os.environ.get("ATON_SLOW4", "") != "1", reason="512^3 on the whole grid is ~10 min of oracle: set ATON_SLOW4=1")
def test_config4_warm_state_on_the_whole_grid_against_oracle(orc):
    """The same grid from workloads.synthetic_warm_state (fronts everywhere: 47 % of the cells sub-cycle in the first step, the
    fix-up and fp64 kernels carry a large share of the work), 16 steps, the whole grid against the oracle (opt-in)."""
    w = wl.synthetic_warm_state(wl.make_config(4))
    err, diag = _full_run(orc, w, 16)
    print("config 4 warm, 16 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


def test_config3_warm_state_on_the_whole_grid_against_oracle(orc):
    """Config 3's full 256^3 grid from workloads.synthetic_warm_state (fronts everywhere, about half of the cells sub-cycle in
    the first step), 12 steps, every cell against the oracle: the fix-up / fp64 kernels under load at a config's real size,
    in the default suite (about half a minute of oracle)."""
    w = wl.synthetic_warm_state(wl.make_config(3))
    assert w.n == 256
    err, diag = _full_run(orc, w, 12)
    assert diag["cells_subcycled"] > 10 * 256 ** 3 // 100 and diag["cells_fp64"] > 0
    print("config 3 warm, 12 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


def test_config3_hll_flux_on_the_whole_grid_against_oracle(orc):
    """The HLL flux (the packed tiled kernel, step_hll_pk_kernel, with several z chunks per column tile) on config 3's full
    256^3 grid from the synthetic warm state, 8 steps, every cell against the oracle's orc_transport_hll."""
    w = wl.synthetic_warm_state(wl.make_config(3))
    w.params.update(flux=1)
    err, diag = _full_run(orc, w, 8)
    print("config 3 warm, HLL, 8 steps:", err, {k: diag[k] for k in ("x_vol", "cells_subcycled", "cells_fp64", "subcycles_max")})


@pytest.mark.parametrize("cfg", [3, 4])
def test_one_step_bar_on_a_whole_256_grid(orc, cfg):
    """The north_star's 1-step bar (max relative error <= 1e-4 on N, F, x, T, cell by cell) on EVERY cell of a 256^3 grid:
    config 3 itself, and a 256^3 twin of config 4 (case A, clumping, collisional ionisation).  Protocol of reading S17: both
    codes start from the oracle's own state -- here the synthetic warm state evolved 8 steps by the oracle -- rounded to
    fp32.  (Measured: 2.7e-5.  Straight from the synthetic state, which no scheme produces, a handful of cells reach
    1.0e-4 .. 1.7e-4: DESIGN.md 5.3.)"""
    w = wl.synthetic_warm_state(wl.make_config(cfg, n=256))
    st8, _ = oracle_run(orc, w, 8)
    ww = state_to_workload(w, st8)
    st1, p = oracle_run(orc, ww, 1)
    g, diag = gpu_run(ww, 1)
    err = max_rel_errors(g, st1, p.c)
    assert diag["n_nonfinite"] == 0 and diag["cells_subcycled"] > 10 ** 6
    assert max(err.values()) <= TOL_1STEP, (cfg, err)
