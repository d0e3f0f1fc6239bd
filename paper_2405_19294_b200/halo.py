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


class PeerSlabDphi:
    """Distributed Dphi_eo of one rank with the messages written STRAIGHT INTO THE NEIGHBOURS' receive buffers by the pack
    kernel (peer memory mapped with CUDA IPC: over NVLink between GPUs, or inside one GPU between processes): projection
    and transfer are one kernel, there is no send/recv.  Receive buffers are double-buffered by call parity and one
    barrier per call orders the neighbours' stores before the own apply (fence()).  One rank: its own buffers."""

    def __init__(self, lat, prec: int, plan: dict, group=None):
        import torch.distributed as dist
        from . import hr_halo_buffers_alloc, hr_halo_bytes, hr_ipc_export, hr_ipc_open
        self.lat, self.prec, self.plan, self.group = lat, prec, plan, group
        self.nb = hr_halo_bytes(lat.ctx, prec)
        self.base = hr_halo_buffers_alloc(lat.ctx, prec)
        self.calls = 0
        self.world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
        self._opened = []
        if self.world == 1:
            self.prev_base = self.next_base = self.base
            return
        rank = dist.get_rank(group)
        handles = [None] * self.world
        dist.all_gather_object(handles, hr_ipc_export(lat.ctx, self.base), group=group)

        def peer(r):
            if r == rank:
                return self.base
            p = hr_ipc_open(lat.ctx, handles[r])
            self._opened.append(p)
            return p

        self.prev_base = peer(plan["prev"])
        self.next_base = self.prev_base if plan["next"] == plan["prev"] else peer(plan["next"])

    # offsets inside an allocation: [send_up | send_dn | recv_prev[0] | recv_next[0] | recv_prev[1] | recv_next[1]]
    def _recv_prev(self, base, k):
        return base + (2 + 2 * k) * self.nb

    def _recv_next(self, base, k):
        return base + (3 + 2 * k) * self.nb

    def fence(self):
        """Every rank's pack stores are complete and visible before anyone applies."""
        import torch
        import torch.distributed as dist
        if self.world == 1:
            return
        if dist.get_backend(self.group) == "nccl":
            if not hasattr(self, "_token"):
                self._token = torch.zeros(1, device=f"cuda:{self.lat.device}")
            dist.all_reduce(self._token, group=self.group)       # on the stream: ordered after the pack kernel, no host wait
        else:
            torch.cuda.synchronize(self.lat.device)
            dist.barrier(group=self.group)

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_halo_apply, hr_dphi_eo_halo_pack, hr_dphi_eo_interior
        st = self.lat.stream()
        k = self.calls & 1
        self.calls += 1
        # my "up" message is the NEXT rank's recv_prev, my "down" message the PREVIOUS rank's recv_next: peer stores
        hr_dphi_eo_halo_pack(self._recv_prev(self.next_base, k), self._recv_next(self.prev_base, k), inp, links, parity, st)
        hr_dphi_eo_interior(out, inp, links, parity, st)
        self.fence()
        hr_dphi_eo_halo_apply(out, self._recv_prev(self.base, k), self._recv_next(self.base, k), links, parity,
                              self.plan["first_rank"], self.plan["last_rank"], st)

    def close(self):
        from . import hr_halo_buffers_free, hr_ipc_close
        import torch
        torch.cuda.synchronize(self.lat.device)
        for p in self._opened:
            hr_ipc_close(self.lat.ctx, p)
        self._opened = []
        if self.base:
            hr_halo_buffers_free(self.lat.ctx, self.base)
            self.base = 0
