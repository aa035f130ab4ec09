"""z-slab decomposition of one ATON box over the ranks of a torch.distributed group.

The paper runs ATON on up to 128 GPUs by cutting the grid into cubes and staging the boundary faces of
(N, F) GPU -> host -> MPI -> host -> GPU every step (PAPER.md:L471-484, 10-15 % of the step).  Here the cut is
into z slabs -- a halo is then one contiguous nx*ny plane per field -- and the planes travel device to device:
`aton_halo_pack` gathers a slab's first / last plane of N, Gx, Gy, Gz into two buffers, `exchange_halos` moves
them to the neighbours (NCCL send/recv over NVLink; a copy when a rank is its own neighbour), and
`aton_halo_unpack` writes the received planes into the ghost planes the step kernel reads.  Chemistry is local;
the diagnostics need one all-reduce of 15 doubles.  Everything numerical runs in libaton.so (also the global mean
density and the means of the diagnostics: aton_set_mean_from_sums, aton_diag_from_sums): this module only decides who
sends which buffer to whom and which entries add, max or min.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Tuple

import torch
import torch.distributed as dist

from . import aton


def slab_range(nz: int, world: int, rank: int) -> Tuple[int, int]:
    """(z_begin, nz_local) of `rank`: nz planes dealt as evenly as possible, the first nz % world slabs one more."""
    if not 0 <= rank < world or world > nz:
        raise ValueError("need 0 <= rank < world <= nz")
    base, extra = divmod(nz, world)
    return rank * base + min(rank, extra), base + (1 if rank < extra else 0)


def neighbours(world: int, rank: int) -> Tuple[int, int]:
    """(rank of the slab below, rank of the slab above), periodic in z."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_halos(send_lo: torch.Tensor, send_hi: torch.Tensor, recv_lo: torch.Tensor, recv_hi: torch.Tensor,
                   rank: int, world: int, group=None) -> None:
    """My last plane (send_hi) becomes the ghost plane below the slab above (its recv_lo); my first plane
    (send_lo) the ghost plane above the slab below (its recv_hi).  Works on CPU (gloo) and CUDA (nccl) tensors."""
    below, above = neighbours(world, rank)
    if world == 1:
        recv_lo.copy_(send_hi)
        recv_hi.copy_(send_lo)
        return
    if world == 2:
        # both neighbours are the same rank: tag the two messages by order (sends and receives posted pairwise)
        ops = [dist.P2POp(dist.isend, send_hi, above, group=group), dist.P2POp(dist.irecv, recv_lo, below, group=group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        ops = [dist.P2POp(dist.isend, send_lo, below, group=group), dist.P2POp(dist.irecv, recv_hi, above, group=group)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        return
    ops = [dist.P2POp(dist.isend, send_hi, above, group=group), dist.P2POp(dist.irecv, recv_lo, below, group=group),
           dist.P2POp(dist.isend, send_lo, below, group=group), dist.P2POp(dist.irecv, recv_hi, above, group=group)]
    for r in dist.batch_isend_irecv(ops):
        r.wait()


def combine_sums(local: List[float], group=None, world: int = 1) -> List[float]:
    """All-reduce aton_reduce_sums across the slabs: entries 0-10 and 14 add, 11-12 take the max, 13 the min.  Returns the
    combined raw sums; the library forms the diagnostics from them (aton_diag_from_sums)."""
    t = torch.tensor(local, dtype=torch.float64)
    if world > 1:
        dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
        s, mx, mn = torch.cat([t[:11], t[14:15]]).to(dev), t[11:13].to(dev), t[13:14].to(dev)
        dist.all_reduce(s, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(mx, op=dist.ReduceOp.MAX, group=group)
        dist.all_reduce(mn, op=dist.ReduceOp.MIN, group=group)
        s = s.cpu()
        t = torch.cat([s[:11], mx.cpu(), mn.cpu(), s[11:12]])
    return t.tolist()


class SlabAton:
    """One rank's slab of a global nx x ny x nz box.  `fields` are this rank's planes (nz_local, ny, nx).

    Two ways to move the halos, same results:
      native=True   the library's own NCCL communicator (aton_comm_init; rank 0's unique id is broadcast through the
                    torch.distributed group) and aton_step_slab: the whole run of steps is one C call, the exchange runs
                    on a second stream beside the interior planes;
      native=False  aton_halo_pack -> exchange_halos (torch.distributed P2P: gloo on CPU tensors in the tests, NCCL on
                    GPUs) -> aton_halo_unpack -> aton_step(dt, 1), one step at a time."""

    def __init__(self, nx: int, ny: int, nz: int, lx_cm: float, params: Dict[str, float], rank: int = 0,
                 world: int = 1, group=None, stream: Optional[torch.cuda.Stream] = None, native: bool = False):
        self.rank, self.world, self.group, self.native = rank, world, group, native
        self.z_begin, self.nz_local = slab_range(nz, world, rank)
        self.params = dict(params)
        self.ctx = aton.Aton(nx, ny, nz, lx_cm, params, stream, slab=(self.z_begin, self.nz_local))
        self.buf = None
        if native:
            comm_id = None
            if world > 1:
                box = [aton.comm_unique_id() if rank == 0 else None]
                dist.broadcast_object_list(box, src=0, group=group)
                comm_id = box[0]
            self.ctx.comm_init(comm_id, rank, world)
        else:
            self.buf = {k: torch.empty((4, ny, nx), dtype=torch.float32, device="cuda")
                        for k in ("send_lo", "send_hi", "recv_lo", "recv_hi")}

    def set_fields(self, nH, x, T, N=None, Fx=None, Fy=None, Fz=None):
        self.ctx.set_fields(nH, x, T, N, Fx, Fy, Fz)
        # <n_H> of the linear clumping law is a GLOBAL mean
        if self.native:
            self.ctx.sync_mean_density()
        else:       # all-reduce the library's own sums, hand them back
            self.ctx.set_mean_from_sums(combine_sums(self.ctx.reduce_sums(), self.group, self.world))

    def set_sources(self, pos, rate):
        self.ctx.set_sources(pos, rate)          # global positions; the library keeps this slab's sources

    def step(self, dt: float, n_steps: int = 1):
        if self.native:
            self.ctx.step_slab(dt, n_steps)
            return
        b = self.buf
        for _ in range(n_steps):
            self.ctx.halo_pack(b["send_lo"], b["send_hi"])
            exchange_halos(b["send_lo"], b["send_hi"], b["recv_lo"], b["recv_hi"], self.rank, self.world, self.group)
            self.ctx.halo_unpack(b["recv_lo"], b["recv_hi"])
            self.ctx.step(dt, 1)

    def get_fields(self, **kw):
        return self.ctx.get_fields(**kw)

    def reduce(self) -> Dict[str, float]:
        """Global diagnostics: the slabs' raw sums combined, the means formed by the library."""
        if self.native:
            return self.ctx.reduce_global()
        return self.ctx.diag_from_sums(combine_sums(self.ctx.reduce_sums(), self.group, self.world))

    def close(self):
        self.ctx.close()
