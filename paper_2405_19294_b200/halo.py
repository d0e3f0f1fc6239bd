"""Slab decomposition along t: the plumbing around the C-ABI calls
hr_dphi_eo_halo_pack / hr_dphi_eo_interior / hr_dphi_eo_halo_apply (include/hr.h, third part).

Only torch.distributed plumbing lives here -- which rank is whose neighbour, which buffer goes where -- no
arithmetic of the method.  `exchange` works on whatever tensors it is given: CUDA tensors over NCCL on the GPUs,
CPU tensors over gloo in tests/test_multi_rank.py."""
from __future__ import annotations


def slab_plan(rank: int, world: int, T_global: int) -> dict:
    """Rank r owns global time-slices [r T_l, (r+1) T_l); neighbours are periodic; the global seam (bc[0]) lies
    below rank 0's first slice and above the last rank's last slice."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    if T_global % world or (T_global // world) % 2 or T_global // world < 2:
        raise ValueError(f"T={T_global} must split into {world} slabs of even extent >= 2 (site parity is global)")
    tl = T_global // world
    return {"T_local": tl, "t0": rank * tl, "prev": (rank - 1) % world, "next": (rank + 1) % world,
            "first_rank": rank == 0, "last_rank": rank == world - 1}


def exchange(send_up, send_dn, recv_prev, recv_next, plan: dict, group=None):
    """My send_up -> the next rank's recv_prev; my send_dn -> the previous rank's recv_next.  One rank: plain copies.
    Returns after the transfers have completed (torch.distributed semantics: on the current CUDA stream for NCCL)."""
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
    if world == 1:
        recv_prev.copy_(send_up)
        recv_next.copy_(send_dn)
        return
    ops = [dist.P2POp(dist.isend, send_up, plan["next"], group, tag=0),
           dist.P2POp(dist.irecv, recv_prev, plan["prev"], group, tag=0),
           dist.P2POp(dist.isend, send_dn, plan["prev"], group, tag=1),
           dist.P2POp(dist.irecv, recv_next, plan["next"], group, tag=1)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()


class SlabDphi:
    """Distributed Dphi_eo of one rank: owns the four face buffers and sequences pack -> exchange || interior -> apply."""

    def __init__(self, lat, prec: int, plan: dict, group=None):
        import torch
        from . import hr_halo_bytes
        self.lat, self.prec, self.plan, self.group = lat, prec, plan, group
        n = hr_halo_bytes(lat.ctx, prec)
        dev = f"cuda:{lat.device}"
        self.send_up, self.send_dn, self.recv_prev, self.recv_next = (torch.empty(n, dtype=torch.uint8, device=dev) for _ in range(4))

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_halo_apply, hr_dphi_eo_halo_pack, hr_dphi_eo_interior
        st = self.lat.stream()
        hr_dphi_eo_halo_pack(self.send_up, self.send_dn, inp, links, parity, st)
        hr_dphi_eo_interior(out, inp, links, parity, st)      # enqueued first: NCCL's transfer overlaps with it
        exchange(self.send_up, self.send_dn, self.recv_prev, self.recv_next, self.plan, self.group)
        hr_dphi_eo_halo_apply(out, self.recv_prev, self.recv_next, links, parity, self.plan["first_rank"], self.plan["last_rank"], st)
