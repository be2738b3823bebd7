"""Multi-GPU path: spatial domain decomposition on a 2-D (x, y) process grid with one
halo exchange per MD step -- what the paper gets from LAMMPS ("MD runs entirely on GPUs with zero CPU-GPU
data transfer except for I/O ... GPU-GPU communication"; weak scaling P:L239; "near-two-dimensional" P:L233).

One process per GPU.  This module is the HOST ORCHESTRATION only: it knows the geometry of the process grid (a few
scalars), decides which message goes to which rank, and moves message buffers with `torch.distributed`
point-to-point calls (NCCL over NVLink on GPUs; gloo in the CPU tests).  It does no arithmetic on atom data: selecting
the atoms of a face, packing and shifting them, compacting, appending ghosts, the per-step gather / scatter of
(x, v, F) and the rebuild decision all run in the library's CUDA kernels behind the C ABI (`flare_domain_*`,
csrc/domain.cu), with every count kept on the device.

Geometry.  The box is cut into px x py rectangles of widths w = L / p along the decomposed axes.  A rank evaluates
its owned atoms together with GHOST copies of every atom within the halo width h = 2 max r_cut + halo_skin of its
rectangle: with a halo two cutoffs wide the local energies of the ghosts that neighbour an owned atom are complete, so
F_k = sum_j (dE_k/dr_kj - dE_j/dr_jk) of an owned atom needs no reverse (force) exchange and the gather stays
atomics-free.  Local frame: a decomposed dimension is open, of length w + 2 h, with the owned rectangle at
[h, h + w); the frame of the lo (hi) neighbour is shifted by +w (-w), so periodic images need no special case.
Ghosts are exchanged in two phases (x, then y including the x ghosts: corners).

Time line.  REBUILD (all ranks together): migrate owned atoms that left the rectangle, select the atoms of the
four face strips (fixed send lists), exchange full rows at fixed message capacity with the count in the header (no
size round trip), append the ghosts after the owned atoms, one synchronisation to learn the new local count.
STEP (between rebuilds; nothing blocks the host): forward rows (x, v, F) of the fixed lists -> fixed ghost slots,
`flare_step(dt, 1)` on owned + ghosts (ghosts carry their owner's velocity and force, so the integrator moves them as
their owner does), rebuild signal.  Membership, order and counts are stable between rebuilds, so the context's
candidate neighbour list survives.  The signal -- "some atom has moved `trigger` since the rebuild", raised on the
device by the kernel that refreshes the candidate list -- is all-reduced (MAX) asynchronously and read `lag` steps
later, so every rank takes the same decision without a per-step host synchronisation; the halo skin covers
2 x trigger plus the motion of those `lag` steps (trigger = 0.35 halo_skin).  That last part is an assumption about
the run (time step, temperature, lag), so it is also CHECKED: the shell is complete as long as no atom has moved more
than halo_skin / 2 since the rebuild, and the engine raises FLARE_ERR_HALO_EXCEEDED (at the next check / rebuild /
gather) the moment one has -- the 0.15 halo_skin between trigger and limit is what the `lag` steps may use up.
"""
from __future__ import annotations

import collections

import numpy as np
import torch
import torch.distributed as dist

MSG_HEADER, MSG_FULL_ROW, MSG_FWD_ROW = 8, 11, 9  # include/flare_b200.h: message layout (doubles)


class PeerError(RuntimeError):
    """Another rank's engine reported an error; this rank stops with it instead of blocking in the next exchange."""


class Engine:
    """What the decomposition needs from a force engine: the device data plane of include/flare_b200.h."""

    device = torch.device("cpu")

    def begin(self, pos, vel, types, tags, box, pbc, trigger): raise NotImplementedError
    def set_limit(self, max_displacement): pass            # optional guard: displacement that invalidates the ghost shell
    def migrate_pack(self, axis, lo_bound, hi_bound, shift_lo, shift_hi, msg_lo, msg_hi, cap): raise NotImplementedError
    def migrate_unpack(self, msg_lo_in, msg_hi_in, cap): raise NotImplementedError
    def border_pack(self, phase, axis, lo_a, lo_b, hi_a, hi_b, shift_lo, shift_hi, msg_lo, msg_hi, cap): raise NotImplementedError
    def border_unpack(self, phase, msg_lo_in, msg_hi_in, cap): raise NotImplementedError
    def commit(self): raise NotImplementedError            # -> dict(n_local, n_owned, send[4], recv[4], recv_off[4])
    def forward_pack(self, phase, msg_lo, msg_hi): raise NotImplementedError
    def forward_unpack(self, phase, msg_lo_in, msg_hi_in): raise NotImplementedError
    def step(self, dt, n_steps, variances): raise NotImplementedError   # n_steps = 0: forces of the current positions
    def signal(self, flag): raise NotImplementedError      # flag: int32[2] tensor on `device`: [0] rebuild wanted, [1] error bits
    def check(self): raise NotImplementedError             # raise this rank's pending engine error, if any
    def owned(self, variances): raise NotImplementedError  # -> host dict(tags, pos (local frame), vel, E, F, V)


class CudaEngine(Engine):
    """The product engine: libflare_b200 through its binding.  The workspace is bound once, for `capacity` atoms."""

    def __init__(self, flare_ctx, capacity: int):
        self.ctx = flare_ctx
        self.device = flare_ctx.device
        self.capacity = int(capacity)
        self.ctx.bind(self.capacity)
        self.n_owned = 0

    def begin(self, pos, vel, types, tags, box, pbc, trigger):
        dev = self.device
        n = len(tags)
        if n > self.capacity:
            raise ValueError(f"{n} owned atoms exceed the engine capacity {self.capacity}")
        self.ctx.domain_begin(n, torch.as_tensor(pos, dtype=torch.float64).reshape(n, 3).to(dev),
                              torch.as_tensor(vel, dtype=torch.float64).reshape(n, 3).to(dev),
                              torch.as_tensor(types, dtype=torch.int32).to(dev), torch.as_tensor(tags, dtype=torch.int64).to(dev),
                              box, pbc, trigger)
        self.n_owned = n

    def set_limit(self, max_displacement): self.ctx.domain_set_limit(max_displacement)

    def migrate_pack(self, *a): self.ctx.domain_migrate_pack(*a)
    def migrate_unpack(self, *a): self.ctx.domain_migrate_unpack(*a)
    def border_pack(self, *a): self.ctx.domain_border_pack(*a)
    def border_unpack(self, *a): self.ctx.domain_border_unpack(*a)

    def commit(self):
        c = self.ctx.domain_commit()
        self.n_owned = c["n_owned"]
        return c

    def forward_pack(self, *a): self.ctx.domain_forward_pack(*a)
    def forward_unpack(self, *a): self.ctx.domain_forward_unpack(*a)

    def step(self, dt, n_steps, variances):
        self.ctx.step(dt, n_steps, want_variance=variances)

    def signal(self, flag):
        self.ctx.domain_signal(flag[0:1])
        self.ctx.domain_status(flag[1:2])

    def check(self): self.ctx.check()

    def owned(self, variances):
        n = self.n_owned
        st = self.ctx.get_state(variances=variances)
        out = {k: (st[k][:n].cpu().numpy() if st[k] is not None else None) for k in ("pos", "vel", "E", "F", "V")}
        out["tags"] = self.ctx.domain_tags()[:n].cpu().numpy()
        return out


class DomainDecomposition:
    """One rank of a px x py process grid over two axes of an orthorhombic box (rank = cx * py + cy)."""

    def __init__(self, engine: Engine, box, pbc, r_cut_max: float, grid=None, axes=(0, 1), halo_skin: float = 1.2,
                 lag: int = 2, border_capacity: int | None = None, migrate_capacity: int = 8192, self_halo: bool = False,
                 group=None, rank: int | None = None, world: int | None = None, trigger_fraction: float = 0.35):
        self.engine = engine
        self.group = group
        # rank / world default to the process group's; given explicitly they describe a rank's geometry without one (tests)
        self.world = world if world is not None else (dist.get_world_size(group) if dist.is_initialized() else 1)
        self.rank = rank if rank is not None else (dist.get_rank(group) if dist.is_initialized() else 0)
        if grid is None:
            grid = (self.world, 1)
        if grid[0] * grid[1] != self.world:
            raise ValueError(f"process grid {grid} does not match the world size {self.world}")
        b = np.asarray(box, dtype=np.float64).reshape(-1)
        self.L = (np.diag(b.reshape(3, 3)) if b.size == 9 else b.reshape(3)).copy()
        self.pbc = np.asarray(pbc, dtype=np.int32).reshape(3).copy()
        self.h = 2.0 * float(r_cut_max) + float(halo_skin)
        if not halo_skin > 0.0:
            raise ValueError("halo_skin must be > 0")
        if not 1 <= int(lag) <= 16:
            # the flag posted after step k is read before step k + lag: with more than a few steps in between, the margin
            # between trigger and limit (0.15 halo_skin per atom) is used up at any temperature worth simulating
            raise ValueError(f"lag must be between 1 and 16 steps, not {lag}")
        if not 0.0 < trigger_fraction < 0.5:
            raise ValueError("trigger_fraction must lie in (0, 0.5): the shell is complete up to halo_skin / 2 per atom")
        # a fast system (hot, light atoms, long time step) wants a lower fraction: (0.5 - fraction) halo_skin is what an
        # atom may still move between raising the signal and the rebuild, `lag` steps later
        self.trigger = float(trigger_fraction) * float(halo_skin)
        self.limit = 0.5 * float(halo_skin)   # beyond this the ghost shell may miss a neighbour of an owned atom: an error
        self.lag = int(lag)
        coords = (self.rank // grid[1], self.rank % grid[1])
        # decomposed axes = exchange phases, in order
        self.phases = []
        self.local_L = self.L.copy()
        self.local_pbc = self.pbc.copy()
        self.lo = np.zeros(3)
        for axis, p, c in zip(axes, grid, coords):
            # an axis with one rank keeps its periodic boundary inside the engine -- unless self_halo asks for the
            # full data path on it too (the rank is then its own neighbour on both sides: its ghosts are its own
            # periodic images; used to exercise and time the data plane on one GPU)
            if p == 1 and not (self_halo and self.pbc[axis]):
                continue
            if not self.pbc[axis]:
                raise ValueError("a decomposed axis must be periodic")
            w = self.L[axis] / p
            if w < self.h:
                raise ValueError(f"domain width {w:.3f} along axis {axis} is smaller than the halo {self.h:.3f}")
            step = grid[1] if axis == axes[0] else 1
            base = self.rank - c * step
            self.phases.append(dict(axis=axis, p=p, c=c, w=w, lo_rank=base + ((c - 1) % p) * step,
                                    hi_rank=base + ((c + 1) % p) * step))
            self.local_L[axis] = w + 2.0 * self.h
            self.local_pbc[axis] = 0
            self.lo[axis] = c * w - self.h  # global coordinate of the local origin
        self.local_box = np.diag(self.local_L).reshape(9)
        self.border_capacity = border_capacity
        self.migrate_capacity = int(migrate_capacity)
        self.counts = None
        self.built = False
        self.rebuilds = 0
        self.bytes_sent = 0
        self._flags = collections.deque()
        self._ring, self._ring_pos = None, 0  # lag + 1 signal slots (device flag, pinned copy, event), allocated once
        self._fwd = None
        self._rb = None

    # ------------------------------------------------------------------ initial distribution and collection (I/O)
    def scatter(self, pos, vel, types):
        """Every rank passes the same full system (host arrays); each keeps the atoms of its rectangle, in its frame."""
        pos = np.array(pos, dtype=np.float64).reshape(-1, 3)
        n_all = len(pos)
        vel = np.zeros((n_all, 3)) if vel is None else np.asarray(vel, dtype=np.float64).reshape(-1, 3)
        types = np.asarray(types, dtype=np.int32).reshape(-1)
        mine = np.ones(n_all, dtype=bool)
        for ph in self.phases:
            a, Lx = ph["axis"], self.L[ph["axis"]]
            x = pos[:, a] - Lx * np.floor(pos[:, a] / Lx)
            x[x >= Lx] = 0.0
            pos[:, a] = x
            mine &= np.clip(np.floor(x / ph["w"]).astype(np.int64), 0, ph["p"] - 1) == ph["c"]
        idx = np.nonzero(mine)[0]
        local = pos[idx] - self.lo[None, :]
        if self.border_capacity is None and self.phases:
            # the same on every rank (both ends of a message must agree on its size): a face strip of a rectangle of
            # uniform density, widened by the ghosts of the first phase, with 50 % to spare
            q = max(self.h / ph["w"] for ph in self.phases)
            self.border_capacity = int(1.5 * (n_all / self.world) * q * (1.0 + 2.0 * q)) + 4096
        self.engine.begin(local, vel[idx], types[idx], idx.astype(np.int64), self.local_box, self.local_pbc, self.trigger)
        if self.phases:
            self.engine.set_limit(self.limit)
        self.built = False
        self._flags.clear()
        return self

    def gather(self, variances: bool = True):
        """Rank 0 gets dict(pos, vel, F, E, V, types-free) of the whole system in the original atom order; others None."""
        o = self.engine.owned(variances)
        pos = o["pos"] + self.lo[None, :]
        for ph in self.phases:
            a, Lx = ph["axis"], self.L[ph["axis"]]
            pos[:, a] -= Lx * np.floor(pos[:, a] / Lx)
        mine = dict(tags=o["tags"], pos=pos, vel=o["vel"], E=o["E"], F=o["F"],
                    V=o["V"] if o["V"] is not None else np.zeros(len(pos)))
        if self.world == 1:
            parts = [mine]
        else:
            parts = [None] * self.world
            dist.all_gather_object(parts, mine, group=self.group)
        if self.rank != 0:
            return None
        tags = np.concatenate([p["tags"] for p in parts])
        order = np.argsort(tags, kind="stable")
        assert np.array_equal(tags[order], np.arange(len(tags))), "atoms lost or duplicated"
        return {k: np.concatenate([p[k] for p in parts])[order] for k in ("pos", "vel", "E", "F", "V")}

    # ------------------------------------------------------------------ messages
    def _new_msg(self, rows, width):
        return torch.zeros(MSG_HEADER + rows * width, dtype=torch.float64, device=self.engine.device)

    def _exchange(self, ph, out_lo, out_hi, in_lo, in_hi):
        """Send out_lo to the lo neighbour and out_hi to the hi neighbour; receive in_lo from lo, in_hi from hi.
        Sizes are known on both sides.  gloo (CPU tests) stages through host memory."""
        lo, hi = ph["lo_rank"], ph["hi_rank"]
        if ph["p"] == 1:  # self-exchange: what I send towards hi arrives from my lo side
            in_lo.copy_(out_hi)
            in_hi.copy_(out_lo)
            self.bytes_sent += 8 * (out_lo.numel() + out_hi.numel())
            return
        host = dist.get_backend(self.group) == "gloo" and self.engine.device.type != "cpu"
        so, si = ([t.cpu() for t in (out_lo, out_hi)], [torch.empty_like(t, device="cpu") for t in (in_lo, in_hi)]) if host \
            else ([out_lo, out_hi], [in_lo, in_hi])
        # receives in the peer's send order (with two ranks along the axis both messages come from the same peer, its
        # to-lo first: that one arrives "from hi"): NCCL matches by order, not by tag
        ops = [dist.P2POp(dist.isend, so[0], lo, self.group, tag=1), dist.P2POp(dist.isend, so[1], hi, self.group, tag=2),
               dist.P2POp(dist.irecv, si[1], hi, self.group, tag=1), dist.P2POp(dist.irecv, si[0], lo, self.group, tag=2)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        if host:
            in_lo.copy_(si[0])
            in_hi.copy_(si[1])
        self.bytes_sent += 8 * (out_lo.numel() + out_hi.numel())

    # ------------------------------------------------------------------ rebuild
    def rebuild(self):
        """Migration, new send lists, new ghost shell; one synchronisation at the end (the new local atom count)."""
        e = self.engine
        mcap, bcap = self.migrate_capacity, self.border_capacity
        if self._rb is None and self.phases:  # the fixed-capacity rebuild messages are allocated once
            self._rb = {k: [self._new_msg(cap, MSG_FULL_ROW) for _ in range(4)] for k, cap in (("m", mcap), ("b", bcap))}
        for ph in self.phases:
            out_lo, out_hi, in_lo, in_hi = self._rb["m"]
            e.migrate_pack(ph["axis"], self.h, self.h + ph["w"], ph["w"], -ph["w"], out_lo, out_hi, mcap)
            self._exchange(ph, out_lo, out_hi, in_lo, in_hi)
            e.migrate_unpack(in_lo, in_hi, mcap)
        inf = float("inf")
        for k, ph in enumerate(self.phases):
            out_lo, out_hi, in_lo, in_hi = self._rb["b"]
            e.border_pack(k, ph["axis"], -inf, 2.0 * self.h, ph["w"], inf, ph["w"], -ph["w"], out_lo, out_hi, bcap)
            self._exchange(ph, out_lo, out_hi, in_lo, in_hi)
            e.border_unpack(k, in_lo, in_hi, bcap)
        # an overflow (message, send list, capacity) shows on the rank it happened on only: agree on the outcome before
        # anybody walks into the next exchange alone
        try:
            counts, failure = e.commit(), None
        except Exception as ex:  # noqa: BLE001 -- whatever the engine raises, the peers must hear of it
            counts, failure = None, ex
        self._raise_together(1 if failure is not None else 0, failure, "the domain rebuild")
        self.counts = counts
        c = self.counts
        self._fwd = [dict(out_lo=self._new_msg(c["send"][2 * k], MSG_FWD_ROW), out_hi=self._new_msg(c["send"][2 * k + 1], MSG_FWD_ROW),
                          in_lo=self._new_msg(c["recv"][2 * k], MSG_FWD_ROW), in_hi=self._new_msg(c["recv"][2 * k + 1], MSG_FWD_ROW))
                     for k in range(len(self.phases))]
        self.built = True
        self.rebuilds += 1
        self._flags.clear()  # signals raised before this rebuild are stale

    def _forward(self):
        for k, ph in enumerate(self.phases):
            m = self._fwd[k]
            self.engine.forward_pack(k, m["out_lo"], m["out_hi"])
            self._exchange(ph, m["out_lo"], m["out_hi"], m["in_lo"], m["in_hi"])
            self.engine.forward_unpack(k, m["in_lo"], m["in_hi"])

    def _raise_together(self, status: int, failure, where: str):
        """All ranks call this at the same point with their own status (0 = fine): if any is non-zero, every rank raises
        -- its own error where it has one, PeerError elsewhere."""
        worst = status
        if self.world > 1:
            on_host = dist.get_backend(self.group) == "gloo"
            t = torch.tensor([status], dtype=torch.int32, device="cpu" if on_host else self.engine.device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
            worst = int(t.item())
        if failure is not None:
            raise failure
        if worst != 0:
            raise PeerError(f"rank {self.rank}: another rank reported an engine error during {where} (status {worst:#x})")

    # ------------------------------------------------------------------ rebuild signal (asynchronous, lagged)
    def _post_signal(self):
        dev = self.engine.device
        if self._ring is None:
            # at most `lag` signals are in flight (one is read before the next is posted): lag + 1 slots never collide
            cuda = dev.type == "cuda"
            self._ring = [(torch.zeros(2, dtype=torch.int32, device=dev),
                           torch.empty(2, dtype=torch.int32, pin_memory=True) if cuda else None,
                           torch.cuda.Event() if cuda else None) for _ in range(self.lag + 1)]
        flag, pinned, ev = self._ring[self._ring_pos % len(self._ring)]
        self._ring_pos += 1
        flag.zero_()  # [0] rebuild wanted, [1] this rank's error bits so far
        self.engine.signal(flag)
        if self.world > 1:
            if dist.get_backend(self.group) == "gloo" and dev.type != "cpu":
                f = flag.cpu()
                dist.all_reduce(f, op=dist.ReduceOp.MAX, group=self.group)
                flag = f
            else:
                dist.all_reduce(flag, op=dist.ReduceOp.MAX, group=self.group)
        if flag.is_cuda:
            pinned.copy_(flag, non_blocking=True)
            ev.record()
            self._flags.append((pinned, ev))
        else:
            self._flags.append((flag.clone(), None))  # the slot is reused lag + 1 steps from now

    def _signal_due(self) -> bool:
        """The flag posted `lag` steps ago (identical on all ranks); waiting on it does not stall the GPU.  It carries
        the ranks' error bits too: an engine error anywhere stops every rank here, in the same step."""
        if len(self._flags) < self.lag:
            return False
        host, ev = self._flags.popleft()
        if ev is not None:
            ev.synchronize()
        if int(host[1]) != 0:
            self.engine.check()  # the rank(s) the error belongs to raise it with its own message
            raise PeerError(f"rank {self.rank}: another rank reported an engine error (bits {int(host[1]):#x})")
        return bool(int(host[0]) != 0)

    # ------------------------------------------------------------------ the two entry points
    def compute(self, variances: bool = False):
        """Forces, energies (and variances) of the current positions on every rank's owned atoms."""
        if not self.built:
            self.rebuild()
        self._forward()
        self.engine.step(0.0, 0, variances)
        return self

    def step(self, dt: float, n_steps: int = 1, variances: bool = False):
        """n_steps of velocity Verlet on the decomposed system."""
        if not self.built:
            self.compute(variances)
        for _ in range(n_steps):
            if self.phases and self._signal_due():
                self.rebuild()
            self._forward()
            self.engine.step(dt, 1, variances)
            if self.phases:
                self._post_signal()
        return self
