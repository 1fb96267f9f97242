"""Slab decomposition of Algorithm 2.1 over several GPUs (section 6.5), one process per GPU.

The periodic box is cut into `world` equal slabs along x; rank r owns the grid planes [r Ml, (r + 1) Ml), Ml = M / world,
and the particles whose base grid index floor(x/h) lies in them.  The paper's communication steps and what does them here:

  MPI-SORT           `partition`: every rank sends each of its points to the owner of its slab (all-to-all, sizes first);
  MPI-GHOST-SOURCE   `ghost_sources`: the points within rc of a slab face go to that neighbour, which needs them as
                     P2P sources only (a slab plan spreads its first `Nown` sources, se.h se_plan_desc);
  MPI-GHOST-GRID     after P2G the P/2 - 1 planes below and the P/2 planes above the owned range are ADDED to the neighbours'
                     owned planes (`SlabEval.owned_planes`); between IFFT and G2P the same planes are filled with the
                     neighbours' values (`planes_back` / `gather_and_sum`);
  FFT / IFFT         slab-decomposed: 2-D R2C over (y, z) on the owned planes, all-to-all into ky-pencils, 1-D transform over
                     x, K4 on the pencil (se_scale_block), and the same way back (the paper uses cuFFTMp here; the local
                     transforms are cuFFT's, called through torch.fft).

All arithmetic of the method runs in the library's kernels through the C-ABI (K1, K2, K3, K5, K6 by the stage hooks of a slab
plan, K4 by se_scale_block); this module only moves data: torch for device memory, indexing and the cuFFT calls,
`torch.distributed` (NCCL between GPUs, gloo in the CPU tests of the host logic) for the exchanges.  `SlabLayout` is pure
index arithmetic and needs no GPU.
"""
from __future__ import annotations

import numpy as np


class SlabLayout:
    """Which planes and points belong to which rank; no GPU, no communication."""

    def __init__(self, L: float, M: int, P: int, rc: float, world: int):
        if world < 2 or M % world:
            raise ValueError("need at least two slabs and M a multiple of their number")
        self.L, self.M, self.P, self.rc, self.world = float(L), int(M), int(P), float(rc), int(world)
        self.h = self.L / self.M
        self.Ml = self.M // self.world
        self.Mx = self.Ml + self.P                 # local planes: P/2 - 1 below, Ml owned, P/2 above, one spare
        self.nlo, self.nhi = self.P // 2 - 1, self.P // 2
        if self.Ml < self.nhi or self.Mx > self.M or self.L / world < self.rc:
            raise ValueError("slabs too thin: need M/world >= P/2, M/world + P <= M and L/world >= rc")

    def px0(self, rank: int) -> int:
        """global index of local plane 0 of `rank`"""
        return (rank * self.Ml - self.nlo) % self.M

    @staticmethod
    def _quot(a, b):
        """a / b rounded as the IEEE quotient K1 takes (torch's CUDA kernels turn a division by a Python scalar into a
        multiplication by its reciprocal, which moves floor(x/h) by one for points within an ulp of a plane)"""
        import torch
        return torch.div(a, torch.full_like(a, b))

    def _wrap(self, x0):
        """x0 wrapped into [0, L) exactly as K1 does it (a result that is not in [0, L), e.g. L itself after rounding, is 0)"""
        if hasattr(x0, "floor"):                    # torch
            import torch
            xw = x0 - self.L * self._quot(x0, self.L).floor()
            return torch.where((xw >= 0) & (xw < self.L), xw, torch.zeros_like(xw))
        xw = x0 - self.L * np.floor(x0 / self.L)
        return np.where((xw >= 0) & (xw < self.L), xw, 0.0)

    def base_plane(self, x0):
        """floor(x_w / h) of first coordinates (numpy or torch, double), as the library takes it"""
        xw = self._wrap(x0)
        if hasattr(xw, "floor"):
            return self._quot(xw, self.h).floor().long().clamp(0, self.M) % self.M      # x/h may round up to M: plane 0
        return np.clip(np.floor(xw / self.h).astype(np.int64), 0, self.M) % self.M

    def owner(self, x0):
        """rank that owns each point (by the base grid plane of its first coordinate)"""
        return self.base_plane(x0) // self.Ml

    def ghost_masks(self, x0, rank: int):
        """(to_left, to_right): which of this rank's points lie within rc of its lower / upper face (periodic)"""
        lo, hi = rank * self.Ml * self.h, (rank + 1) * self.Ml * self.h
        xw = self._wrap(x0)
        if hasattr(xw, "floor"):                    # a point whose x/h rounds up to M lives in plane 0 (rank 0): it sits at 0-
            import torch
            xw = torch.where(self._quot(xw, self.h).floor() >= self.M, xw - self.L, xw)
        else:
            xw = np.where(np.floor(xw / self.h) >= self.M, xw - self.L, xw)
        to_left, to_right = (xw - lo) < self.rc, (hi - xw) <= self.rc
        if self.world == 2:                         # both neighbours are the same rank: a point goes there once
            to_left = to_left & ~to_right
        return to_left, to_right

    def local_planes(self, rank: int):
        """global plane index of every local plane of `rank` (numpy int64[Mx])"""
        return (self.px0(rank) + np.arange(self.Mx)) % self.M




class SlabEval:
    """One rank's share of a slab-decomposed evaluation.  The driver (`evaluate_distributed` below, or the single-process
    emulation of the tests) calls the phases in order and carries the messages between ranks."""

    def __init__(self, layout: SlabLayout, rank: int, xi: float, precision="fp64", window="gaussian"):
        self.lay, self.rank, self.xi, self.precision, self.window = layout, rank, float(xi), precision, window
        self.plan = None
        self.grid_plan = None
        self.side = None                            # side stream of the P2P stage

    # -- phase 1: ghost sources ------------------------------------------------------------------------------------
    def ghost_out(self, x, f):
        """own points (x, f: [n, 3] device tensors) -> messages (x, f) for the left and the right neighbour"""
        self.x, self.f = x.contiguous(), f.contiguous()
        ml, mr = self.lay.ghost_masks(x[:, 0].double(), self.rank)
        return (x[ml], f[ml]), (x[mr], f[mr])

    # -- phase 2: K1, K2, K3 on the slab plan ------------------------------------------------------------------------
    def near_and_spread(self, from_left, from_right, stream=None):
        """ghost points received -> sort, P2P (u^N of the owned points), P2G into the local slab grid.
        Returns the ghost planes for the left and the right neighbour ([3, nlo, M, M], [3, nhi, M, M])."""
        import torch
        from . import Plan, SE_BUF_GRID
        lay = self.lay
        n = self.x.shape[0]
        if n == 0:                                                     # a slab without points: nothing to evaluate or spread
            self.H = torch.zeros(3, lay.Mx, lay.M, lay.M, dtype=self.x.dtype, device=self.x.device)
            return self.H[:, :lay.nlo].contiguous(), self.H[:, lay.nlo + lay.Ml:lay.nlo + lay.Ml + lay.nhi].contiguous()
        xs = torch.cat([self.x, from_left[0], from_right[0]]).contiguous()
        fs = torch.cat([self.f, from_left[1], from_right[1]]).contiguous()
        key = (xs.shape[0], n)
        if self.plan is None or self._key != key:
            if self.plan is not None:
                self.plan.destroy()
            self.plan = Plan(xs.shape[0], lay.L, self.xi, lay.rc, lay.M, lay.P, self.precision, window=self.window,
                             Nt=n, Mx=lay.Mx, px0=lay.px0(self.rank), Nown=n)
            self._key = key
        p = self.plan
        p.set_targets(self.x)
        p.stage("sort", x=xs, f=fs, stream=stream)
        p.stage("p2g", stream=stream)
        self.H = p.read(SE_BUF_GRID, stream=stream)                    # [3, Mx, M, M]
        # P2P does not depend on the grid chain ("can be overlapped"): it runs on a side stream, next to the
        # exchanges and transforms that follow, and is joined before the sum
        main = stream if stream is not None else torch.cuda.current_stream()
        if self.side is None:
            self.side = torch.cuda.Stream()
        self.side.wait_stream(main)
        p.stage("p2p", stream=self.side)
        lo, hi = lay.nlo, lay.nhi
        return self.H[:, :lo].contiguous(), self.H[:, lo + lay.Ml:lo + lay.Ml + hi].contiguous()

    # -- phase 3: ghost-plane reduction ------------------------------------------------------------------------------
    def owned_planes(self, from_left, from_right):
        """ghost planes received (the left neighbour's upper ghosts, the right neighbour's lower ghosts) are added to the
        owned planes they overlap; returns the owned block [3, Ml, M, M]"""
        lay = self.lay
        own = self.H[:, lay.nlo:lay.nlo + lay.Ml].clone()
        own[:, :lay.nhi] += from_left                              # their planes above their range = my first P/2
        own[:, lay.Ml - lay.nlo:] += from_right                    # their planes below their range = my last P/2 - 1
        return own

    # -- phase 4: slab-decomposed 3-D transform with K4 in the middle -----------------------------------------------------
    # x-slabs --2-D R2C over (y, z)--> all-to-all --> ky-pencils --1-D C2C over x, K4, inverse 1-D--> all-to-all --> x-slabs
    # --2-D C2R--> owned planes.  The transforms are cuFFT's (through torch.fft; unnormalised in both directions, as in the
    # one-GPU plan), K4 is the library's kernel on the pencil block this rank holds (se_scale_block).
    def spectrum_out(self, own):
        """owned planes [3, Ml, M, M] -> one message per rank: the ky-block of the 2-D transforms that rank's pencil takes"""
        import torch
        lay = self.lay
        A = torch.fft.rfft2(own, dim=(2, 3))                            # [3, Ml, M, M/2+1]
        Ky = lay.M // lay.world
        return [A[:, :, d * Ky:(d + 1) * Ky].contiguous() for d in range(lay.world)]

    def pencil(self, blocks, stream=None):
        """the ky-blocks of all ranks' planes (rank order = plane order) -> scaled pencil -> one message per rank: the
        x-block of planes that rank owns"""
        import torch
        lay = self.lay
        Ky = lay.M // lay.world
        # the transform over x runs on a copy with x as the fastest index (cuFFT's strided 1-D transforms are several times
        # slower than two transposes), K4 on the x-slowest layout it is written for
        Bx = torch.cat(list(blocks), dim=1).permute(0, 2, 3, 1).contiguous()         # [3, Ky, M/2+1, M]
        S = torch.fft.fft(Bx, dim=3).permute(0, 3, 1, 2).contiguous()                # [3, M, Ky, M/2+1]
        self._tables().scale_block(S, self.rank * Ky, Ky, stream=stream)
        Bx = torch.fft.ifft(S.permute(0, 2, 3, 1).contiguous(), dim=3, norm="forward")   # unnormalised inverse
        B = Bx.permute(0, 3, 1, 2)
        return [B[:, d * lay.Ml:(d + 1) * lay.Ml].contiguous() for d in range(lay.world)]

    def planes_back(self, blocks):
        """the x-blocks of all pencils (rank order = ky order) -> H~ on the owned planes; returns the ghost planes the
        neighbours gather from: (my first P/2 planes for the left one, my last P/2 - 1 for the right one)"""
        import torch
        lay = self.lay
        A = torch.cat(list(blocks), dim=2)                              # [3, Ml, M, M/2+1]
        self.Ht = torch.fft.irfft2(A, s=(lay.M, lay.M), dim=(2, 3), norm="forward").contiguous()
        return self.Ht[:, :lay.nhi].contiguous(), self.Ht[:, lay.Ml - lay.nlo:].contiguous()

    # -- phase 5: K5, K6 -----------------------------------------------------------------------------------------------------
    def gather_and_sum(self, from_left, from_right, stream=None):
        """ghost planes received (the left neighbour's last P/2 - 1 planes, the right neighbour's first P/2) -> local grid ->
        G2P -> u = u^N + u^F - self term for the owned points ([n, 3])"""
        import torch
        from . import SE_BUF_GRID
        lay = self.lay
        if self.x.shape[0] == 0:
            return self.x.clone()
        spare = torch.zeros_like(self.Ht[:, :lay.Mx - lay.nlo - lay.Ml - lay.nhi])
        self.plan.write(SE_BUF_GRID, torch.cat([from_left, self.Ht, from_right, spare], dim=1).contiguous(), stream=stream)
        self.plan.stage("g2p", stream=stream)
        u = torch.empty_like(self.x)
        (stream if stream is not None else torch.cuda.current_stream()).wait_stream(self.side)     # u^N is ready
        self.plan.stage("sum", f=self.f, u=u, stream=stream)
        return u

    def _tables(self):
        """a plan whose multiplier tables K4 uses: this rank's slab plan, or a one-point one if the slab holds no points"""
        from . import Plan
        if self.plan is not None:
            return self.plan
        if self.grid_plan is None:
            lay = self.lay
            self.grid_plan = Plan(1, lay.L, self.xi, lay.rc, lay.M, lay.P, self.precision, window=self.window,
                                  Mx=lay.Mx, px0=lay.px0(self.rank))
        return self.grid_plan

    def destroy(self):
        for p in (self.plan, self.grid_plan):
            if p is not None:
                p.destroy()
        self.plan = self.grid_plan = None


def evaluate_emulated(lay: SlabLayout, xi, xs_per_rank, fs_per_rank, precision="fp64", window="gaussian"):
    """All ranks of a slab decomposition run one after the other in this process (one GPU): the exchanges are list
    shuffles.  For tests; returns the list of u per rank."""
    W = lay.world
    ranks = [SlabEval(lay, r, xi, precision, window) for r in range(W)]
    try:
        out = [ranks[r].ghost_out(xs_per_rank[r], fs_per_rank[r]) for r in range(W)]
        gp = [ranks[r].near_and_spread(out[(r - 1) % W][1], out[(r + 1) % W][0]) for r in range(W)]
        own = [ranks[r].owned_planes(gp[(r - 1) % W][1], gp[(r + 1) % W][0]) for r in range(W)]
        a = [ranks[r].spectrum_out(own[r]) for r in range(W)]                     # a[src][dst]
        b = [ranks[r].pencil([a[s][r] for s in range(W)]) for r in range(W)]
        g = [ranks[r].planes_back([b[s][r] for s in range(W)]) for r in range(W)]  # (for left, for right)
        return [ranks[r].gather_and_sum(g[(r - 1) % W][1], g[(r + 1) % W][0]) for r in range(W)]
    finally:
        for e in ranks:
            e.destroy()


# ---- torch.distributed driver ------------------------------------------------------------------------------------------

def _exchange(send_left, send_right, group=None):
    """send one tensor to the left and one to the right neighbour, receive theirs; shapes differ per rank: the leading
    sizes travel first.  Returns (from_left, from_right)."""
    import torch
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    left, right = (rank - 1) % world, (rank + 1) % world
    dev = send_left.device
    n_out = torch.tensor([send_left.shape[0], send_right.shape[0]], dtype=torch.int64, device=dev)
    sizes = [torch.zeros(2, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(sizes, n_out, group=group)
    n_from_left, n_from_right = int(sizes[left][1]), int(sizes[right][0])
    from_left = torch.empty((n_from_left,) + tuple(send_left.shape[1:]), dtype=send_left.dtype, device=dev)
    from_right = torch.empty((n_from_right,) + tuple(send_right.shape[1:]), dtype=send_right.dtype, device=dev)
    ops = [dist.P2POp(dist.isend, send_left.contiguous(), left, group), dist.P2POp(dist.isend, send_right.contiguous(), right, group),
           dist.P2POp(dist.irecv, from_left, left, group), dist.P2POp(dist.irecv, from_right, right, group)]
    if world == 2:                              # both neighbours are the same rank: keep the two messages apart by order
        ops = [dist.P2POp(dist.isend, send_left.contiguous(), left, group), dist.P2POp(dist.irecv, from_right, right, group),
               dist.P2POp(dist.isend, send_right.contiguous(), right, group), dist.P2POp(dist.irecv, from_left, left, group)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()
    return from_left, from_right


def partition(lay: SlabLayout, x, f, group=None):
    """MPI-SORT: every rank hands each of its points to the rank that owns its slab (all-to-all).  Returns this rank's
    points (x, f) and, for un-sorting, (source rank, index on the source rank) of each."""
    import torch
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    own = lay.owner(x[:, 0].double())
    order = torch.argsort(own, stable=True)
    counts = torch.bincount(own, minlength=world)
    recv_counts = torch.empty_like(counts)
    dist.all_to_all_single(recv_counts, counts, group=group)
    sc, rc_ = counts.tolist(), recv_counts.tolist()

    def a2a(t):
        out = torch.empty((sum(rc_),) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        dist.all_to_all_single(out, t[order].contiguous(), rc_, sc, group=group)
        return out

    src_rank = torch.repeat_interleave(torch.arange(world, device=x.device), recv_counts)
    idx = a2a(torch.arange(x.shape[0], device=x.device))
    return a2a(x), a2a(f), (src_rank, idx)


def _all_to_all(blocks, group=None):
    """blocks[d] goes to rank d; returns the list of blocks received, in rank order (all blocks have one shape).  Point to
    point operations: they exist on every backend (gloo has no all_to_all)."""
    import torch
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    out = [torch.empty_like(blocks[rank]) for _ in range(world)]
    out[rank].copy_(blocks[rank])
    ops = []
    for k in range(1, world):                   # same pairing order on both sides of every pair
        dst, src = (rank + k) % world, (rank - k) % world
        ops.append(dist.P2POp(dist.isend, blocks[dst].contiguous(), dst, group))
        ops.append(dist.P2POp(dist.irecv, out[src], src, group))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return out


def evaluate_distributed(ev: SlabEval, x, f, group=None, stream=None):
    """One slab-decomposed evaluation under torch.distributed (one process per GPU): x, f are the points this rank owns
    (see `partition`); returns u for them."""
    import torch
    (xl, fl), (xr, fr) = ev.ghost_out(x, f)
    gl, gr = _exchange(torch.cat([xl, fl], dim=1), torch.cat([xr, fr], dim=1), group)
    lo_planes, hi_planes = ev.near_and_spread((gl[:, :3].contiguous(), gl[:, 3:].contiguous()),
                                              (gr[:, :3].contiguous(), gr[:, 3:].contiguous()), stream=stream)
    # planes travel with the plane index first
    pl, pr = _exchange(lo_planes.transpose(0, 1).contiguous(), hi_planes.transpose(0, 1).contiguous(), group)
    own = ev.owned_planes(pl.transpose(0, 1), pr.transpose(0, 1))
    pencil_in = _all_to_all(ev.spectrum_out(own), group)
    planes_in = _all_to_all(ev.pencil(pencil_in, stream=stream), group)
    for_left, for_right = ev.planes_back(planes_in)
    gl, gr = _exchange(for_left.transpose(0, 1).contiguous(), for_right.transpose(0, 1).contiguous(), group)
    return ev.gather_and_sum(gl.transpose(0, 1).contiguous(), gr.transpose(0, 1).contiguous(), stream=stream)
