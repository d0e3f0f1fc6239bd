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


class AsyncExchange:
    """The NCCL exchange of a set of (send_up, send_dn, recv_prev, recv_next, prev, next) face buffers, started on a SIDE
    stream that waits only for the pack kernels, so that the transfer runs while the interior kernel (enqueued on the
    compute stream afterwards) computes -- PAPER.md:50: "compute the bulk while the messages are in flight".
    (torch's NCCL stream waits for the stream that is current when batch_isend_irecv is called: issued from the compute
    stream AFTER the interior launch the transfer would start only when the interior kernel has finished.)
    start(): after the pack launches; finish(): makes the compute stream wait for the transfers, before the applies.
    All directions go into ONE batch.  Matching between two ranks that are each other's previous AND next neighbour
    (two blocks in a direction) relies on both posting [send up, recv prev, send down, recv next] in this order."""

    def __init__(self, device, group=None):
        import torch
        self.torch, self.group = torch, group
        self.side = torch.cuda.Stream(device=device)
        self.packed = torch.cuda.Event()
        self.reqs = []

    def start(self, faces) -> None:
        import torch.distributed as dist
        torch = self.torch
        world = dist.get_world_size(self.group) if dist.is_available() and dist.is_initialized() else 1
        if world == 1:
            for su, sd, rp, rn, _, _ in faces:
                rp.copy_(su)
                rn.copy_(sd)
            self.reqs = []
            return
        ops = []
        for su, sd, rp, rn, prev, nxt in faces:
            ops += [dist.P2POp(dist.isend, su, nxt, self.group), dist.P2POp(dist.irecv, rp, prev, self.group),
                    dist.P2POp(dist.isend, sd, prev, self.group), dist.P2POp(dist.irecv, rn, nxt, self.group)]
        self.packed.record(torch.cuda.current_stream())
        with torch.cuda.stream(self.side):
            self.side.wait_event(self.packed)
            self.reqs = dist.batch_isend_irecv(ops)

    def finish(self) -> None:
        for req in self.reqs:
            req.wait()                       # the CURRENT (compute) stream waits for the transfer; no host wait
        self.reqs = []


class SlabDphi:
    """Distributed Dphi_eo of one rank: owns the four face buffers and sequences pack -> exchange || interior -> apply."""

    def __init__(self, lat, prec: int, plan: dict, group=None):
        import torch
        from . import hr_halo_bytes
        self.lat, self.prec, self.plan, self.group = lat, prec, plan, group
        n = hr_halo_bytes(lat.ctx, prec)
        dev = f"cuda:{lat.device}"
        self.send_up, self.send_dn, self.recv_prev, self.recv_next = (torch.empty(n, dtype=torch.uint8, device=dev) for _ in range(4))
        self.xch = AsyncExchange(dev, group)

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_halo_apply, hr_dphi_eo_halo_pack, hr_dphi_eo_interior
        st = self.lat.stream()
        hr_dphi_eo_halo_pack(self.send_up, self.send_dn, inp, links, parity, st)
        # pack -> [exchange on the side stream || interior on the compute stream] -> apply
        self.xch.start([(self.send_up, self.send_dn, self.recv_prev, self.recv_next, self.plan["prev"], self.plan["next"])])
        hr_dphi_eo_interior(out, inp, links, parity, st)
        self.xch.finish()
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


class SlabCG:
    """Dhat x = b on a lattice cut into slabs or blocks (one per rank): hr_cg_dhat_dist (include/hr.h) -- the CG of
    hr_cg_dhat, readings C20-C22, with every vector update AND every scalar recurrence inside libhr.  This class only
    supplies the two callbacks the library cannot know: the distributed Dphi_eo (`slab`: SlabDphi, PeerSlabDphi, BlockDphi
    or PeerBlockDphi) and the sum of a few doubles over the ranks (torch.distributed.all_reduce)."""

    def __init__(self, slab, links: int, m0: float, group=None):
        self.slab, self.links, self.m0, self.group = slab, links, float(m0), group
        self.lat, self.prec = slab.lat, slab.prec

    def allsum(self, vals):
        """Sum of a list of floats over the ranks (plumbing: one all-reduce)."""
        import torch
        import torch.distributed as dist
        if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(self.group) == 1:
            return list(vals)
        dev = f"cuda:{self.lat.device}" if dist.get_backend(self.group) == "nccl" else "cpu"
        t = torch.tensor(list(vals), dtype=torch.float64, device=dev)
        dist.all_reduce(t, group=self.group)
        return t.tolist()

    def solve(self, x, b, tol: float, maxiter: int):
        """x = Dhat^{-1} b (x0 = 0).  Returns (iterations, [|r_k|^2 / |rhs|^2])."""
        import torch
        from . import hr_cg_dhat_dist, hr_cg_dist_workspace_bytes
        lat = self.lat
        ws = torch.empty(hr_cg_dist_workspace_bytes(lat.ctx, self.prec), dtype=torch.uint8, device=f"cuda:{lat.device}")
        return hr_cg_dhat_dist(lat.ctx, self.prec, self.m0, x, b, tol, maxiter, ws,
                               lambda out, inp, parity: self.slab.dphi_eo(out, inp, self.links, parity),
                               self.allsum, lat.stream())


# ---- 4-D block decomposition ("4-D block partition, split t first, then z, y, x") ------------------
def block_plan(rank: int, grid, dims_global) -> dict:
    """Ranks form a grid (P_t, P_x, P_y, P_z), rank = ((c_t P_x + c_x) P_y + c_y) P_z + c_z; every rank owns a block of
    dims_global / grid sites with EVEN local extents (site parity is global).  Per direction mu: the neighbour ranks
    (periodic), whether this rank holds the first / last block (where the global seam bc[mu] sits) and whether the
    direction is split at all (P_mu > 1; an unsplit direction stays periodic inside the rank)."""
    grid = tuple(int(g) for g in grid)
    dims_global = tuple(int(v) for v in dims_global)
    world = grid[0] * grid[1] * grid[2] * grid[3]
    if len(grid) != 4 or min(grid) < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/grid")
    local = []
    for mu in range(4):
        if dims_global[mu] % grid[mu] or (dims_global[mu] // grid[mu]) % 2 or dims_global[mu] // grid[mu] < 2:
            raise ValueError(f"extent {dims_global[mu]} of direction {mu} must split into {grid[mu]} blocks of even extent >= 2")
        local.append(dims_global[mu] // grid[mu])
    if grid[3] > 1 and local[2] % 2:
        raise ValueError("a split in z needs an even local Y")
    c = [0, 0, 0, 0]
    r = rank
    for mu in (3, 2, 1, 0):
        c[mu] = r % grid[mu]
        r //= grid[mu]

    def rank_of(cc):
        return ((cc[0] * grid[1] + cc[1]) * grid[2] + cc[2]) * grid[3] + cc[3]

    prev, nxt = [], []
    for mu in range(4):
        a, b = list(c), list(c)
        a[mu] = (c[mu] - 1) % grid[mu]
        b[mu] = (c[mu] + 1) % grid[mu]
        prev.append(rank_of(a))
        nxt.append(rank_of(b))
    return {"grid": grid, "coords": tuple(c), "dims_local": tuple(local), "origin": tuple(c[mu] * local[mu] for mu in range(4)),
            "prev": prev, "next": nxt, "first": [c[mu] == 0 for mu in range(4)], "last": [c[mu] == grid[mu] - 1 for mu in range(4)],
            "split": [mu for mu in range(4) if grid[mu] > 1], "mask": sum(1 << mu for mu in range(4) if grid[mu] > 1)}


def _mask(flags) -> int:
    return sum(1 << mu for mu in range(4) if flags[mu])


class BlockDphi:
    """Distributed Dphi_eo of one rank of a 4-D block decomposition: for every split direction the four face buffers;
    pack (all directions, same input) -> [exchange of all faces in one NCCL batch on a side stream || interior launch with
    the split directions masked] -> apply (all directions, one launch).  Unmeasured on more than one GPU (none in this run)."""

    def __init__(self, lat, prec: int, plan: dict, group=None):
        import torch
        from . import hr_face_bytes
        self.lat, self.prec, self.plan, self.group = lat, prec, plan, group
        dev = f"cuda:{lat.device}"
        self.buf = {mu: [torch.empty(hr_face_bytes(lat.ctx, prec, mu), dtype=torch.uint8, device=dev) for _ in range(4)]
                    for mu in plan["split"]}                      # send_up, send_dn, recv_prev, recv_next
        self.xch = AsyncExchange(dev, group)

    def pack(self, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_faces_pack
        hr_dphi_eo_faces_pack(self.plan["mask"], {mu: b[0] for mu, b in self.buf.items()}, {mu: b[1] for mu, b in self.buf.items()},
                              inp, links, parity, self.lat.stream())         # all split directions in one launch

    def interior(self, out, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_interior_mask
        hr_dphi_eo_interior_mask(out, inp, links, parity, self.plan["mask"], self.lat.stream())

    def faces(self):
        return [(su, sd, rp, rn, self.plan["prev"][mu], self.plan["next"][mu]) for mu, (su, sd, rp, rn) in self.buf.items()]

    def apply(self, out, links: int, parity: int) -> None:
        from . import hr_dphi_eo_faces_apply
        hr_dphi_eo_faces_apply(self.plan["mask"], out, {mu: b[2] for mu, b in self.buf.items()}, {mu: b[3] for mu, b in self.buf.items()},
                               links, parity, _mask(self.plan["first"]), _mask(self.plan["last"]), self.lat.stream())   # one launch

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        self.pack(inp, links, parity)
        self.xch.start(self.faces())                 # one batch for all split directions, on the side stream
        self.interior(out, inp, links, parity)       # ... while the interior kernel runs on the compute stream
        self.xch.finish()
        self.apply(out, links, parity)


class PeerBlockDphi:
    """BlockDphi with the messages of every split direction written straight into the neighbours' receive buffers (CUDA IPC
    peer memory, as PeerSlabDphi): one allocation of six messages per direction, receive buffers double-buffered by call
    parity, ONE fence per call after all pack kernels."""

    def __init__(self, lat, prec: int, plan: dict, group=None):
        import torch.distributed as dist
        from . import hr_face_buffers_alloc, hr_face_bytes, hr_ipc_export, hr_ipc_open
        self.lat, self.prec, self.plan, self.group = lat, prec, plan, group
        self.world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
        self.calls = 0
        self.nb = {mu: hr_face_bytes(lat.ctx, prec, mu) for mu in plan["split"]}
        self.base = {mu: hr_face_buffers_alloc(lat.ctx, prec, mu) for mu in plan["split"]}
        self._opened = []
        self.prev_base, self.next_base = dict(self.base), dict(self.base)
        if self.world == 1:
            return
        rank = dist.get_rank(group)
        handles = [None] * self.world
        dist.all_gather_object(handles, {mu: hr_ipc_export(lat.ctx, b) for mu, b in self.base.items()}, group=group)
        mapped = {}

        def peer(r, mu):
            if r == rank:
                return self.base[mu]
            if (r, mu) not in mapped:
                mapped[(r, mu)] = hr_ipc_open(lat.ctx, handles[r][mu])
                self._opened.append(mapped[(r, mu)])
            return mapped[(r, mu)]

        for mu in plan["split"]:
            self.prev_base[mu] = peer(plan["prev"][mu], mu)
            self.next_base[mu] = peer(plan["next"][mu], mu)

    fence = PeerSlabDphi.fence

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        from . import hr_dphi_eo_faces_apply, hr_dphi_eo_faces_pack, hr_dphi_eo_interior_mask
        st = self.lat.stream()
        k = self.calls & 1
        self.calls += 1
        # my "up" message is the next rank's recv_prev[k], "down" the previous rank's recv_next[k]; all directions in one launch
        hr_dphi_eo_faces_pack(self.plan["mask"], {mu: self.next_base[mu] + (2 + 2 * k) * self.nb[mu] for mu in self.plan["split"]},
                              {mu: self.prev_base[mu] + (3 + 2 * k) * self.nb[mu] for mu in self.plan["split"]}, inp, links, parity, st)
        hr_dphi_eo_interior_mask(out, inp, links, parity, self.plan["mask"], st)
        self.fence()
        hr_dphi_eo_faces_apply(self.plan["mask"], out, {mu: self.base[mu] + (2 + 2 * k) * self.nb[mu] for mu in self.plan["split"]},
                               {mu: self.base[mu] + (3 + 2 * k) * self.nb[mu] for mu in self.plan["split"]}, links, parity,
                               _mask(self.plan["first"]), _mask(self.plan["last"]), st)

    def close(self):
        from . import hr_halo_buffers_free, hr_ipc_close
        import torch
        torch.cuda.synchronize(self.lat.device)
        for p in self._opened:
            hr_ipc_close(self.lat.ctx, p)
        self._opened = []
        for b in self.base.values():
            hr_halo_buffers_free(self.lat.ctx, b)
        self.base = {}
