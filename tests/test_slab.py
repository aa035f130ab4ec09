"""z-slab decomposition: host-side plan and halo exchange on CPU with gloo (world sizes 2 and
3), and -- on one GPU -- slabs emulated as several contexts of one process whose halos are moved by the same plan:
a slab run must be bit-identical to the undivided run."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
from paper_1004_2503_b200 import slab  # noqa: E402
from paper_1004_2503_b200 import workloads as wl  # noqa: E402


def test_slab_plan():
    for nz, world in ((1024, 8), (13, 3), (7, 7), (10, 4)):
        spans = [slab.slab_range(nz, world, r) for r in range(world)]
        assert spans[0][0] == 0 and sum(n for _, n in spans) == nz
        for (b0, n0), (b1, _) in zip(spans, spans[1:]):
            assert b0 + n0 == b1                                   # contiguous, in rank order
        assert max(n for _, n in spans) - min(n for _, n in spans) <= 1
    assert slab.neighbours(4, 0) == (3, 1) and slab.neighbours(4, 3) == (2, 0) and slab.neighbours(1, 0) == (0, 0)
    with pytest.raises(ValueError):
        slab.slab_range(4, 5, 0)


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_1004_2503_b200 import slab
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
# every rank's first plane is filled with 10*rank + 1, its last plane with 10*rank + 2
mk = lambda v: torch.full((4, 3, 8), float(v))
send_lo, send_hi, recv_lo, recv_hi = mk(10 * rank + 1), mk(10 * rank + 2), mk(-1), mk(-1)
for _ in range(3):                                                 # repeated exchanges stay matched
    slab.exchange_halos(send_lo, send_hi, recv_lo, recv_hi, rank, world)
    below, above = slab.neighbours(world, rank)
    assert bool((recv_lo == 10 * below + 2).all()), (rank, recv_lo[0, 0, 0])      # last plane of the slab below
    assert bool((recv_hi == 10 * above + 1).all()), (rank, recv_hi[0, 0, 0])      # first plane of the slab above
sums = [10.0 + rank, 1.0 * rank, 2.0, 4.0, 0, 0, 0, 0, 0, 5, 1, 0.1 * (rank + 1), 3 + rank, -float(rank), 7.0]
d = slab.combine_sums(sums, None, world)
tot = sum(10.0 + r for r in range(world))
assert len(d) == 15 and abs(d[0] - tot) < 1e-12 and abs(d[1] - sum(range(world))) < 1e-12        # entries 0-10, 14 add
assert d[2] == 2.0 * world and d[3] == 4.0 * world and d[9] == 5 * world and d[10] == world and d[14] == 7.0 * world
assert abs(d[11] - 0.1 * world) < 1e-12 and d[12] == 2 + world and d[13] == -(world - 1)      # 11-12 max, 13 min
dist.destroy_process_group()
print("ok", rank)
"""


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_and_diagnostics_gloo(world):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    code = _WORKER.format(root=ROOT, port=port)
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1")
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for r, p in enumerate(procs):
        out, _ = p.communicate(timeout=240)
        assert p.returncode == 0 and f"ok {r}" in out, out


# ------------------------------------------------------------------------------------------------ GPU
def _case(nx, ny, nz, seed=2):
    rng = np.random.default_rng(seed)
    nH = torch.from_numpy((2e-4 * np.exp(1.5 * rng.standard_normal((nz, ny, nx)) - 1.125)).astype(np.float32)).cuda()
    p = wl.default_params()
    p.update(redshift=8.0, recomb_case=0, clump_model=1, clump_a=1.0, clump_b=2.0)     # needs the GLOBAL <n_H>
    dx = 3.0e21
    cells = [(0, 0, 0), (nx - 1, ny - 1, nz - 1), (5, 3, nz // 2), (7, 1, nz // 2 - 1), (nx // 2, ny // 2, 1 % nz)]
    pos = torch.tensor([[(i + 0.5) / nx, (j + 0.5) / ny, (k + 0.5) / nz] for i, j, k in cells], dtype=torch.float32)
    rate = torch.tensor(10 ** rng.uniform(49.5, 51, len(cells)), dtype=torch.float64)
    return nH, p, dx, pos, rate


@pytest.mark.gpu
# 128-wide grids run the product kernel (variant 5: 16 or 8 rows per CTA), the others the variant-4 fallback
@pytest.mark.parametrize("shape,world", [((64, 8, 12), 2), ((32, 12, 13), 3), ((64, 8, 5), 5), ((32, 8, 9), 1),
                                         ((128, 16, 12), 2), ((128, 8, 10), 3), ((256, 32, 7), 2),
                                         # the HLL flux on slabs: the packed tiled kernel (nx % 64 == 0) and the scalar one
                                         ((64, 8, 12, "hll"), 2), ((32, 16, 9, "hll"), 3), ((128, 16, 7, "hll"), 2)])
def test_slabs_on_one_gpu_equal_the_undivided_run(shape, world):
    from paper_1004_2503_b200 import aton
    nx, ny, nz = shape[:3]
    nH, p, dx, pos, rate = _case(nx, ny, nz)
    if len(shape) > 3:
        p = dict(p, flux=1)
    x0, T0 = torch.full_like(nH, 1e-3), torch.full_like(nH, 100.0)
    dt, steps = wl.courant_dt(dx), 14
    full = aton.Aton(nx, ny, nz, dx * nx, p)
    full.set_fields(nH, x0, T0)
    full.set_sources(pos, rate)
    full.step(dt, steps)
    ref = full.get_fields(device="cuda")
    dref = full.reduce()
    full.close()
    # the slabs: one SlabAton per emulated rank; halos moved by the module's own neighbour plan
    ranks = [slab.SlabAton(nx, ny, nz, dx * nx, p, rank=r, world=world) for r in range(world)]
    mean = float(nH.double().mean())
    for r, s in enumerate(ranks):
        sl = slice(s.z_begin, s.z_begin + s.nz_local)
        s.ctx.set_mean_density(mean)                      # what SlabAton.set_fields' all-reduce would give
        s.ctx.set_fields(nH[sl].contiguous(), x0[sl].contiguous(), T0[sl].contiguous())
        s.set_sources(pos, rate)
    for _ in range(steps):
        for s in ranks:
            s.ctx.halo_pack(s.buf["send_lo"], s.buf["send_hi"])
        for r, s in enumerate(ranks):
            below, above = slab.neighbours(world, r)
            s.buf["recv_lo"].copy_(ranks[below].buf["send_hi"])
            s.buf["recv_hi"].copy_(ranks[above].buf["send_lo"])
        for s in ranks:
            s.ctx.halo_unpack(s.buf["recv_lo"], s.buf["recv_hi"])
            s.ctx.step(dt, 1)
    sums = np.zeros(slab.aton.NSUMS)
    for s in ranks:
        out = s.get_fields(device="cuda")
        sl = slice(s.z_begin, s.z_begin + s.nz_local)
        for k in ("nH", "x", "T", "N", "Fx", "Fy", "Fz"):
            assert torch.equal(out[k], ref[k][sl]), (k, s.rank)
        v = np.array(s.ctx.reduce_sums())
        sums[:11] += v[:11]
        sums[11:13] = np.maximum(sums[11:13], v[11:13])
        sums[13] = v[13] if s.rank == 0 else min(sums[13], v[13])
        sums[14] += v[14]
        if s.rank > 0:
            s.close()
    d = ranks[0].ctx.diag_from_sums(list(sums))           # the library forms the means from the combined sums
    ranks[0].close()
    assert sums[0] == nx * ny * nz and d["n_nonfinite"] == 0
    assert d["gamma_vol"] == pytest.approx(dref["gamma_vol"], rel=1e-12) and d["photons_total"] == pytest.approx(dref["photons_total"], rel=1e-12)
    assert d["x_vol"] == pytest.approx(dref["x_vol"], rel=1e-12) and d["x_mass"] == pytest.approx(dref["x_mass"], rel=1e-12)
    assert d["T_vol"] == pytest.approx(dref["T_vol"], rel=1e-12) and d["f_max"] == pytest.approx(dref["f_max"], rel=1e-12)
    assert d["subcycles_total"] == dref["subcycles_total"] and d["cells_subcycled"] == dref["cells_subcycled"]
    assert d["subcycles_max"] == dref["subcycles_max"] and d["N_min"] == dref["N_min"]


@pytest.mark.gpu
def test_slab_class_world_size_1_and_errors():
    from paper_1004_2503_b200 import aton
    nx, ny, nz = 32, 8, 6
    nH, p, dx, pos, rate = _case(nx, ny, nz, seed=4)
    x0, T0 = torch.full_like(nH, 1e-3), torch.full_like(nH, 100.0)
    dt = wl.courant_dt(dx)
    full = aton.Aton(nx, ny, nz, dx * nx, p)
    full.set_fields(nH, x0, T0); full.set_sources(pos, rate); full.step(dt, 9)
    ref, dref = full.get_fields(device="cuda"), full.reduce()
    full.close()
    for native in (False, True):                           # world 1: a rank that is its own neighbour
        s = slab.SlabAton(nx, ny, nz, dx * nx, p, native=native)
        s.set_fields(nH, x0, T0); s.set_sources(pos, rate)
        if native:
            s.step(dt, 4); s.step(dt, 5)                   # aton_step_slab: runs of steps, ghost planes carried over
        else:
            s.step(dt, 9)
        out, d = s.get_fields(device="cuda"), s.reduce()
        for k in ref:
            assert torch.equal(out[k], ref[k]), (native, k)
        assert d["x_vol"] == pytest.approx(dref["x_vol"], rel=1e-12) and d["gamma_vol"] == pytest.approx(dref["gamma_vol"], rel=1e-6)
        assert d["steps_done"] == 9 and d["subcycles_total"] == dref["subcycles_total"]
        with pytest.raises(aton.AtonError):
            s.ctx.step(dt, 2)                              # aton_step: one step per halo exchange
        if not native:
            with pytest.raises(aton.AtonError):
                s.ctx.step_slab(dt, 1)                     # aton_step_slab needs aton_comm_init
        s.close()
    with pytest.raises(aton.AtonError):
        aton.Aton(24, 8, 6, dx * 24, p, slab=(0, 3))       # variant 4 needs nx % 32 == 0
    hp = dict(p); hp.update(flux=1)
    with pytest.raises(aton.AtonError):
        aton.Aton(32, 12, 6, dx * 32, hp, slab=(0, 3))     # the HLL flux on a slab needs the tiled kernels: ny % 8 == 0
    with pytest.raises(aton.AtonError):
        aton.Aton(32, 8, 6, dx * 32, p, slab=(4, 3))       # planes outside the grid
    a = aton.Aton(32, 8, 6, dx * 32, p)
    with pytest.raises(aton.AtonError):
        a.halo_pack(torch.zeros(4, 8, 32, device="cuda"), torch.zeros(4, 8, 32, device="cuda"))   # not a slab
    a.close()


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(64, 16, 10), (128, 16, 10)], ids=["v4_64x16x10", "v5_128x16x10"])
def test_native_slab_step_with_nccl_self_exchange_against_the_oracle(orc, shape):
    """aton_step_slab through a real NCCL communicator (one rank: every send pairs with the rank's own receive, the same
    code path as N ranks) on a grid with several z planes per launch range, against the ORACLE (not only the undivided
    CUDA run): relative L1 <= 1e-3 after 30 steps, and bit-identical to the undivided CUDA run."""
    from paper_1004_2503_b200 import aton
    from parity_util import l1_errors
    nx, ny, nz = shape
    nH, p, dx, pos, rate = _case(nx, ny, nz, seed=9)
    x0, T0 = torch.full_like(nH, 1e-3), torch.full_like(nH, 100.0)
    dt, steps = wl.courant_dt(dx), 30
    full = aton.Aton(nx, ny, nz, dx * nx, p)
    full.set_fields(nH, x0, T0); full.set_sources(pos, rate); full.step(dt, steps)
    ref = full.get_fields(device="cuda")
    full.close()
    s = slab.SlabAton(nx, ny, nz, dx * nx, p, native=False)
    s.ctx.comm_init(aton.comm_unique_id(), 0, 1)           # a 1-rank NCCL communicator instead of the copy shortcut
    s.native = True
    s.set_fields(nH, x0, T0); s.set_sources(pos, rate)
    s.step(dt, steps)
    out, d = s.get_fields(device="cpu"), s.reduce()
    s.close()
    for k in ref:
        assert torch.equal(out[k], ref[k].cpu()), k
    zero = np.zeros((nz, ny, nx), np.float32)
    st = orc.State(nH.cpu().numpy(), x0.cpu().numpy(), T0.cpu().numpy(), zero, zero, zero, zero)
    op = orc.make_params(p, dx, float(nH.double().mean()))
    orc.step(st, op, dt, steps, pos.double().numpy(), rate.numpy())
    err = l1_errors({k: v.numpy() for k, v in out.items()}, st, op.c)
    assert max(err[k] for k in ("N", "F", "x", "T")) <= 1e-3 and err["x_vol"] <= 1e-3, err
    assert d["x_vol"] == pytest.approx(st.x.mean(), abs=1e-3) and d["n_nonfinite"] == 0
