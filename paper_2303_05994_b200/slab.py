"""x1-slab decomposition with halo exchange (section 3.3, 323, 349 eq (9)).

The paper distributes f over MPI ranks and surrounds every sub-domain with halo cells; the
1-D interpolation along a distributed dim reads its neighbour's points from the halo, exchanged point-to-point
before the sweep.  On a B200 node the natural cut is along x1, the slowest dim of the C-order layout:
each rank owns one contiguous slab of L = n0/R planes, every sweep along x2..v3, the rotation and the density moment
rho(x) are local (no all-reduce: a rank owns whole v-blocks), and only the x1 sweep needs the neighbours'
w = q/2 + ceil(max |displacement in cells|) boundary planes -- contiguous blocks of w*n1*n2*n3*n4*n5 doubles, one
send and one receive per side on a periodic ring.

This module is plumbing: it plans the slab (sizes, neighbours, the four halo regions), moves halos with
torch.distributed point-to-point calls (NCCL on GPUs, gloo in the CPU tests) or, for one process holding several
slabs, with device copies, and sequences C-ABI calls.  Every arithmetic step runs in libbsl6d.so:
  * interior context: grid (L, n1..n5) on the interior view of the local array -- sweeps along dims 1-5, rotate, density;
  * x1 context: grid (L + 2w, n1..n5) with bsl6d_set_boundary(0, open) -- the x1 sweep over interior + halos.
The interior results are bit-identical to the same operation on the undivided grid (tests/test_gpu_slab.py).

Overlap (by eq (9) the x1 sweep is communication-bound, so the exchange "must be overlapped with the
interior"): the planes a neighbour needs -- the lowest and the highest w interior planes -- are brought up to date
FIRST (every operation between two x1 sweeps acts plane by plane, so it can run on the two boundary regions before the
middle), the exchange is posted, and the middle planes are computed while the halos travel
(Slab.strang_step_overlapped; exchange_start / exchange_finish).  Sub-slab contexts (grids of w or L-2w planes) do the
regional work; results stay bit-identical.  With halos as thick as half a slab (L = 2w) nothing is left to overlap.
Measured on hardware: single GPU only (this environment has one GPU per run); the N > 1 path is covered by the
world_size-2 gloo test of the exchange and by the single-GPU emulation with 2 and 4 slabs.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import List, Optional, Sequence

import torch

from . import api


@dataclass(frozen=True)
class SlabPlan:
    """Host-side geometry of one rank's slab (no device state)."""
    n_global: tuple
    world: int
    rank: int
    q: int
    L: int                 # interior planes of this rank
    w: int                 # halo planes per side
    plane: int             # doubles per x1 plane = n1*n2*n3*n4*n5
    left: int              # ring neighbours
    right: int

    @property
    def local_shape(self):
        return (self.L + 2 * self.w,) + tuple(self.n_global[1:])

    @property
    def x1_offset(self) -> int:
        """Global x1 index of the first interior plane."""
        return self.rank * self.L

    # plane ranges [lo, hi) inside the local array
    @property
    def interior(self):
        return (self.w, self.w + self.L)

    @property
    def send_lo(self):      # my lowest interior planes -> the LEFT neighbour's upper halo
        return (self.w, 2 * self.w)

    @property
    def send_hi(self):      # my highest interior planes -> the RIGHT neighbour's lower halo
        return (self.L, self.L + self.w)

    @property
    def recv_lo(self):      # lower halo <- the LEFT neighbour's send_hi
        return (0, self.w)

    @property
    def recv_hi(self):      # upper halo <- the RIGHT neighbour's send_lo
        return (self.w + self.L, 2 * self.w + self.L)

    @property
    def halo_bytes_per_side(self) -> int:
        return 8 * self.w * self.plane

    @property
    def regions(self):
        """Plane ranges of the local array for the overlapped step: (boundary low = send_lo, boundary high = send_hi,
        middle), or None when the two boundary regions overlap (L < 2w) -- then the whole interior is boundary."""
        if self.L < 2 * self.w:
            return None
        return (self.send_lo, self.send_hi, (2 * self.w, self.L))


def plan_slab(n_global: Sequence[int], degree: int, world: int, rank: int, max_shift_cells: float) -> SlabPlan:
    """Halo width: the stencil reaches q/2 nodes beyond the foot cell and the foot lies up to ceil(max|alpha|) cells
    away (k = floor(alpha) in [-ceil, ceil-1]).  The halo must come from the direct neighbours: w <= L."""
    n = tuple(int(v) for v in n_global)
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    if n[0] % world:
        raise ValueError(f"n0 = {n[0]} is not divisible by {world} ranks (PAPER.md:148: points per dim a multiple of "
                         f"the ranks per dim)")
    q = int(degree) + 1
    L = n[0] // world
    w = q // 2 + int(math.ceil(abs(float(max_shift_cells))))
    if w > L:
        raise ValueError(f"halo width {w} exceeds the slab thickness {L}: use fewer ranks or a smaller time step")
    plane = 1
    for v in n[1:]:
        plane *= v
    return SlabPlan(n, world, rank, q, L, w, plane, (rank - 1) % world, (rank + 1) % world)


def _planes(t: torch.Tensor, r):
    return t[r[0]:r[1]]


def exchange_local(plans: List[SlabPlan], locals_: List[torch.Tensor]) -> None:
    """One process holds every slab of the ring (tests; single-GPU emulation): halo exchange by device copies,
    one copy per halo (contiguous blocks)."""
    R = len(plans)
    for r in range(R):
        p = plans[r]
        _planes(locals_[r], p.recv_lo).copy_(_planes(locals_[p.left], plans[p.left].send_hi))
        _planes(locals_[r], p.recv_hi).copy_(_planes(locals_[p.right], plans[p.right].send_lo))


def exchange_start(plan: SlabPlan, f_local: torch.Tensor, group=None):
    """Post the periodic-ring halo exchange with the two neighbours over torch.distributed (one send and one receive
    per side, posted together) and return a handle for exchange_finish.  The boundary planes being sent must be final;
    work on other planes may be enqueued before exchange_finish (NCCL runs the transfers on its own stream)."""
    import torch.distributed as dist
    if plan.world == 1:
        _planes(f_local, plan.recv_lo).copy_(_planes(f_local, plan.send_hi))
        _planes(f_local, plan.recv_hi).copy_(_planes(f_local, plan.send_lo))
        return []
    ops = [
        dist.P2POp(dist.isend, _planes(f_local, plan.send_hi), plan.right, group, tag=1),
        dist.P2POp(dist.irecv, _planes(f_local, plan.recv_lo), plan.left, group, tag=1),
        dist.P2POp(dist.isend, _planes(f_local, plan.send_lo), plan.left, group, tag=2),
        dist.P2POp(dist.irecv, _planes(f_local, plan.recv_hi), plan.right, group, tag=2),
    ]
    # With two ranks both neighbours are the same peer.  Every rank posts the same order (hi out, lo in, lo out, hi in),
    # so NCCL's in-order matching per peer pairs my first send with the peer's first receive (gloo matches by tag).
    return dist.batch_isend_irecv(ops)


def exchange_finish(handle) -> None:
    """Wait for the transfers of exchange_start: the halos are filled when this returns (GPU: when the current stream
    gets past it)."""
    for r in handle or ():
        r.wait()


def exchange(plan: SlabPlan, f_local: torch.Tensor, group=None):
    """exchange_start + exchange_finish: returns after the halos of f_local are filled."""
    exchange_finish(exchange_start(plan, f_local, group))


class Slab:
    """One rank's slab: plan + the two library contexts (created on first use; needs a CUDA device)."""

    def __init__(self, n_global, lo, dx, degree: int, world: int, rank: int, max_shift_cells: float):
        self.plan = plan_slab(n_global, degree, world, rank, max_shift_cells)
        self.lo, self.dx, self.degree = tuple(lo), tuple(dx), int(degree)
        self._int: Optional[api.Context] = None
        self._x1: Optional[api.Context] = None
        self._sub = {}                                     # plane range -> context (overlapped step)

    # -- contexts ------------------------------------------------------------------------------------------
    @property
    def ctx_interior(self) -> api.Context:
        if self._int is None:
            p = self.plan
            lo = (self.lo[0] + p.x1_offset * self.dx[0],) + self.lo[1:]
            self._int = api.create((p.L,) + tuple(p.n_global[1:]), lo, self.dx, self.degree)
        return self._int

    @property
    def ctx_x1(self) -> api.Context:
        if self._x1 is None:
            p = self.plan
            lo = (self.lo[0] + (p.x1_offset - p.w) * self.dx[0],) + self.lo[1:]
            self._x1 = api.create(p.local_shape, lo, self.dx, self.degree)
            self._x1.set_boundary(0, True)
        return self._x1

    def ctx_planes(self, r) -> api.Context:
        """Context for planes [r[0], r[1]) of the local array (any operation that does not sweep x1)."""
        key = (int(r[0]), int(r[1]))
        if key == tuple(self.plan.interior):
            return self.ctx_interior
        if key not in self._sub:
            p = self.plan
            lo = (self.lo[0] + (p.x1_offset - p.w + key[0]) * self.dx[0],) + self.lo[1:]
            self._sub[key] = api.create((key[1] - key[0],) + tuple(p.n_global[1:]), lo, self.dx, self.degree)
        return self._sub[key]

    def launch_count(self) -> int:
        return sum(c.launch_count() for c in [self._int, self._x1] + list(self._sub.values()) if c is not None)

    def destroy(self):
        for c in [self._int, self._x1] + list(self._sub.values()):
            if c is not None:
                c.destroy()
        self._int = self._x1 = None
        self._sub = {}

    # -- storage -------------------------------------------------------------------------------------------
    def alloc(self, device="cuda") -> torch.Tensor:
        return torch.zeros(self.plan.local_shape, dtype=torch.float64, device=device)

    def interior(self, f_local: torch.Tensor) -> torch.Tensor:
        lo, hi = self.plan.interior
        return f_local[lo:hi]

    def scatter_from_global(self, f_global: torch.Tensor, f_local: torch.Tensor) -> torch.Tensor:
        p = self.plan
        self.interior(f_local).copy_(f_global[p.x1_offset:p.x1_offset + p.L])
        return f_local

    # -- operations (the halos of f_local must be current for advect_x1) ---------------------------------------
    def advect_x1(self, f_local: torch.Tensor, dt: float, max_check: bool = True):
        """x1 sweep over the whole local array, in place; interior results are exact, halo planes become stale."""
        if max_check:
            need = x1_planes_needed(self.lo, self.dx, self.plan.n_global, self.plan.q, dt)
            if need > self.plan.w:
                raise ValueError(f"a step of dt={dt:g} needs {need} halo planes, the slab has {self.plan.w}")
        self.ctx_x1.advect(f_local, f_local, 0, None, dt)

    def advect(self, f_local: torch.Tensor, dim: int, shift_source, dt: float):
        """Sweep along dim 1..5 on the interior, in place (E sources are over this rank's x points)."""
        assert 1 <= dim <= 5
        v = self.interior(f_local)
        self.ctx_interior.advect(v, v, dim, shift_source, dt)

    def rotate(self, f_local: torch.Tensor, B, dt: float):
        v = self.interior(f_local)
        self.ctx_interior.rotate(v, v, B, dt)

    def density(self, f_local: torch.Tensor, rho: torch.Tensor):
        return self.ctx_interior.density(self.interior(f_local), rho)

    def strang_step(self, f_local: torch.Tensor, E, B, dt: float, exchange_fn):
        """x1,x2,x3 (dt/2) -> v1,v2,v3 with E (dt) -> rotation -> x1,x2,x3 (dt/2); exchange_fn(f_local) refreshes the
        halos (it is called before each of the two x1 sweeps).  E: three tensors over THIS rank's (L, n1, n2) x points."""
        half = 0.5 * dt
        v = self.interior(f_local)
        ci = self.ctx_interior
        exchange_fn(f_local)
        self.advect_x1(f_local, half)
        seq = [(1, None, 0, half / self.dx[1]), (2, None, 0, half / self.dx[2])]
        if E is not None:
            seq += [(3 + d, E[d], 0x7, dt / self.dx[3 + d]) for d in range(3) if E[d] is not None]
        ci.advect_seq(v, v, seq)
        if B is not None:
            ci.rotate(v, v, B, dt)
        exchange_fn(f_local)
        self.advect_x1(f_local, half)
        ci.advect_seq(v, v, [(1, None, 0, half / self.dx[1]), (2, None, 0, half / self.dx[2])])

    # -- the same step with the exchanges overlapped ------------------------------------------------------------
    def local_ops(self, f_local: torch.Tensor, r, seq_x, E, B, dt_v: float, dt_rot: float):
        """On planes [r[0], r[1]) only: the x2/x3 sweeps of seq_x, then (if dt_v is not None) the E sweeps with the
        matching planes of E, then the rotation.  Everything here acts plane by plane."""
        lo, hi = int(r[0]), int(r[1])
        if hi <= lo:
            return
        v = f_local[lo:hi]
        c = self.ctx_planes((lo, hi))
        seq = list(seq_x)
        if dt_v is not None and E is not None:
            w = self.plan.w
            seq += [(3 + d, E[d][lo - w:hi - w], 0x7, dt_v / self.dx[3 + d]) for d in range(3) if E[d] is not None]
        if seq:
            c.advect_seq(v, v, seq)
        if dt_rot is not None and B is not None:
            c.rotate(v, v, B, dt_rot)

    def step_regions(self):
        """(regions computed before the exchange is posted, regions computed while it is in flight)."""
        reg = self.plan.regions
        if reg is None:
            return [self.plan.interior], []
        return [reg[0], reg[1]], [reg[2]]

    def strang_step_overlapped(self, f_local: torch.Tensor, E, B, dt: float, group=None, pending=None):
        """The Strang step of strang_step with both halo exchanges overlapped: the boundary regions are advanced first,
        the exchange is posted, the middle planes follow while the halos travel.  `pending`: the handle this method
        returned for the previous step (its trailing x2,x3 half-step already posted the exchange for this step's first
        x1 sweep); None = post it now.  Returns the handle for the next step; finish it with exchange_finish (or pass it
        on) before reading the halos.  Bit-identical to strang_step."""
        half = 0.5 * dt
        seq_x = [(1, None, 0, half / self.dx[1]), (2, None, 0, half / self.dx[2])]
        first, later = self.step_regions()
        if pending is None:
            pending = exchange_start(self.plan, f_local, group)
        exchange_finish(pending)
        self.advect_x1(f_local, half)
        for r in first:
            self.local_ops(f_local, r, seq_x, E, B, dt, dt)
        h = exchange_start(self.plan, f_local, group)
        for r in later:
            self.local_ops(f_local, r, seq_x, E, B, dt, dt)
        exchange_finish(h)
        self.advect_x1(f_local, half)
        for r in first:
            self.local_ops(f_local, r, seq_x, None, None, None, None)
        h = exchange_start(self.plan, f_local, group)
        for r in later:
            self.local_ops(f_local, r, seq_x, None, None, None, None)
        return h


def x1_planes_needed(lo, dx, n_global, q: int, dt: float) -> int:
    """Planes of a neighbour an x1 sweep of length dt can reach: half the stencil plus the largest displacement
    |v1| * |dt| / dx1 over the v1 nodes, rounded up (include/bsl6d.h, bsl6d_set_boundary / bsl6d_advect_x1_peer)."""
    vmax = max(abs(lo[3]), abs(lo[3] + (n_global[3] - 1) * dx[3]))
    return q // 2 + int(math.ceil(vmax * abs(dt) / dx[0]))


# ---- slabs WITHOUT halo planes: the x1 sweep reads the neighbours' planes through peer memory -------------------------
class PeerSlab:
    """One rank's slab as two plain arrays of L planes (ping-pong); the x1 sweep (bsl6d_advect_x1_peer) reads the w
    planes it needs from the neighbours' arrays where they are -- peer memory over NVLink when the neighbours are other
    GPUs, the same device in the single-process emulation -- so there are no halo planes, no exchange step and no
    halo traffic beyond the sweep's own loads: compute and communication are one kernel.  Everything else acts on the
    local array in place.  The ring must be synchronised before each x1 sweep (the neighbours' arrays must hold the
    state of the same step, and nobody may still be reading the buffer this sweep writes): `sync` does that --
    device synchronise + process-group barrier in a real run, nothing when one process steps all slabs in turn."""

    def __init__(self, n_global, lo, dx, degree: int, world: int, rank: int, max_shift_cells: float):
        self.plan = plan_slab(n_global, degree, world, rank, max_shift_cells)
        p = self.plan
        self.lo, self.dx, self.degree = tuple(lo), tuple(dx), int(degree)
        lo_loc = (self.lo[0] + p.x1_offset * self.dx[0],) + self.lo[1:]
        self.ctx = api.create((p.L,) + tuple(p.n_global[1:]), lo_loc, self.dx, self.degree)
        self.shape = (p.L,) + tuple(p.n_global[1:])
        self.buf = None            # [X, Y]
        self.cur = 0               # which buffer holds the state
        self.left = None           # [X, Y] of the ring neighbours (tensors this process can dereference)
        self.right = None

    def alloc(self, device="cuda"):
        self.buf = [torch.zeros(self.shape, dtype=torch.float64, device=device) for _ in range(2)]
        return self.buf

    def connect(self, left_bufs, right_bufs):
        """left_bufs / right_bufs: the neighbours' [X, Y] (same process), or what open_peer_buffers returned."""
        self.left, self.right = list(left_bufs), list(right_bufs)

    @property
    def f(self) -> torch.Tensor:
        return self.buf[self.cur]

    def destroy(self):
        self.ctx.destroy()

    def advect_x1(self, dt: float, max_check: bool = True):
        """The x1 sweep over peer memory.  The slab was planned for a largest displacement: a longer step would make the
        kernel read beyond the w neighbour planes it is promised (zeros, silently), so it is refused here."""
        if max_check:
            need = x1_planes_needed(self.lo, self.dx, self.plan.n_global, self.plan.q, dt)
            if need > self.plan.w or need > self.plan.L:
                raise ValueError(f"a step of dt={dt:g} needs {need} neighbour planes, the slab was planned for "
                                 f"{self.plan.w} (thickness {self.plan.L})")
        c = self.cur
        self.ctx.advect_x1_peer(self.buf[c], self.left[c], self.right[c], self.buf[1 - c], self.plan.w, None, dt)
        self.cur = 1 - c

    def local_part(self, E, B, dt_x: float, dt_v, dt_rot):
        f = self.f
        seq = [(1, None, 0, dt_x / self.dx[1]), (2, None, 0, dt_x / self.dx[2])]
        if dt_v is not None and E is not None:
            seq += [(3 + d, E[d], 0x7, dt_v / self.dx[3 + d]) for d in range(3) if E[d] is not None]
        self.ctx.advect_seq(f, f, seq)
        if dt_rot is not None and B is not None:
            self.ctx.rotate(f, f, B, dt_rot)

    def strang_step(self, E, B, dt: float, sync=lambda: None):
        half = 0.5 * dt
        sync()
        self.advect_x1(half)
        self.local_part(E, B, half, dt, dt)
        sync()
        self.advect_x1(half)
        self.local_part(None, None, half, None, None)


def ring_sync(group=None):
    """Barrier for PeerSlab.strang_step in a multi-process run: every rank's device work is complete, then all ranks
    meet.  (One per x1 sweep; a few tens of microseconds against sweeps of milliseconds.)"""
    import torch.distributed as dist
    torch.cuda.synchronize()
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.barrier(group)


def share_buffers(bufs):
    """Picklable CUDA-IPC descriptions of this rank's arrays, to be sent to the neighbours (all_gather_object)."""
    from torch.multiprocessing.reductions import reduce_tensor
    return [reduce_tensor(b)[1] for b in bufs]


def open_peer_buffers(descs):
    """Map a neighbour's arrays into this process (cudaIpcOpenMemHandle; peer access over NVLink is enabled by the
    runtime when the arrays live on another GPU).  The owner must keep them alive."""
    from torch.multiprocessing.reductions import rebuild_cuda_tensor
    bufs = [rebuild_cuda_tensor(*d) for d in descs]
    cur = torch.cuda.current_device()
    for b in bufs:
        if b.device.index != cur:
            # a kernel on THIS device will dereference the neighbour's pointers: make torch switch peer access on
            # (it does so on the first cross-device copy).  Not exercised on this one-GPU environment.
            if not torch.cuda.can_device_access_peer(cur, b.device.index):
                raise RuntimeError(f"cuda:{cur} cannot access cuda:{b.device.index} as a peer")
            torch.empty(1, dtype=b.dtype, device=f"cuda:{cur}").copy_(b.view(-1)[:1])
    return bufs
