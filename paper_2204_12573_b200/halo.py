"""Multi-GPU path: spatial domain decomposition with one halo exchange per
evaluation -- what the paper gets from LAMMPS ("All ... GPU-GPU communication is handled by LAMMPS";
weak scaling P:L239).  One process per GPU; `torch.distributed` point-to-point messages between neighbouring
slabs (NCCL over NVLink on GPUs, gloo in the CPU tests).  Everything the force field computes still runs in
the CUDA kernels behind the C ABI: this module only decides which atoms go where (argument marshalling).

Decomposition: the box is cut along one periodic axis into `world` slabs of width w = L / world; rank r owns
the atoms with coordinate in [r w, (r+1) w).  Each rank evaluates its owned atoms together with GHOST copies
of every atom within g = 2 max r_cut of its slab: with a halo two cutoffs wide the local energies of the ghosts
that neighbour an owned atom are themselves complete, so the forces on owned atoms,
F_k = sum_j (dE_k/dr_kj - dE_j/dr_jk), need no reverse (force) exchange and the gather stays atomics-free.
Inside a rank the slab is an OPEN dimension of length w + 2 g (local coordinate = offset from the slab centre,
nearest image); the other two dimensions keep their boundary conditions.

Per MD step: (1) halo exchange of (x, v, F, type) of the atoms near the two faces -- ghosts carry their owner's
velocity and force so that the library's integrator moves them exactly as their owner does; (2) one
`Engine.md_step` on owned + ghosts; (3) migration of owned atoms that left the slab (with v, F, global id).
Requirements: w >= g (only adjacent slabs talk), w >= 2 g when world == 2 (no atom is a ghost twice), and
atoms move less than w per step.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


class Engine:
    """What the decomposition needs from a force engine.  Tensors live on `device`."""

    device = torch.device("cpu")

    def evaluate(self, pos, types, box, pbc, variances):  # -> E [n], F [n,3], V [n] or None
        raise NotImplementedError

    def md_step(self, pos, vel, frc, types, box, pbc, dt, variances):  # -> pos, vel, E, F, V
        raise NotImplementedError


class CudaEngine(Engine):
    """The product engine: libflare_b200 through its binding.  The workspace is sized once for `capacity` atoms."""

    def __init__(self, flare_ctx, capacity: int):
        self.ctx = flare_ctx
        self.device = flare_ctx.device
        self.capacity = int(capacity)
        self._ws = None

    def _bind(self, n):
        if n > self.capacity:
            raise ValueError(f"{n} local atoms exceed the engine capacity {self.capacity}")
        if self._ws is None:
            self.ctx.bind(self.capacity)  # allocates the workspace for the capacity
            self._ws = self.ctx._workspace
        if self.ctx.n_atoms != n:  # re-binding drops the candidate neighbour list: only when the size changed
            self.ctx.bind(n, workspace=self._ws)

    def evaluate(self, pos, types, box, pbc, variances):
        self._bind(pos.shape[0])
        e, f, v = self.ctx.compute(pos.contiguous(), types.contiguous(), box, pbc, variances=variances)
        return e, f, v

    def md_step(self, pos, vel, frc, types, box, pbc, dt, variances):
        self._bind(pos.shape[0])
        self.ctx.set_state(pos.contiguous(), vel.contiguous(), types.contiguous(), box, pbc)
        self.ctx.set_forces(frc.contiguous())
        self.ctx.step(dt, 1, want_variance=variances)
        st = self.ctx.get_state(variances=variances)
        return st["pos"], st["vel"], st["E"], st["F"], st["V"]


class SlabDecomposition:
    """State of one rank: its owned atoms (global coordinates) and the geometry of its slab."""

    def __init__(self, engine: Engine, box, pbc, r_cut_max: float, axis: int = 0, group=None):
        self.engine = engine
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.axis = int(axis)
        b = np.asarray(box, dtype=np.float64).reshape(-1)
        self.L = (np.diag(b.reshape(3, 3)) if b.size == 9 else b.reshape(3)).copy()
        self.pbc = np.asarray(pbc, dtype=np.int32).reshape(3).copy()
        self.g = 2.0 * float(r_cut_max)
        self.w = self.L[self.axis] / self.world
        if self.world > 1:
            if not self.pbc[self.axis]:
                raise ValueError("the decomposed axis must be periodic")
            if self.w < self.g or (self.world == 2 and self.w < 2.0 * self.g):
                raise ValueError(f"slab width {self.w:.3f} too small for a halo of {self.g:.3f} on {self.world} ranks")
        self.lo = self.rank * self.w
        self.centre = self.lo + 0.5 * self.w
        # local box: the slab plus its halo, open along the axis
        self.local_L = self.L.copy()
        self.local_pbc = self.pbc.copy()
        if self.world > 1:
            self.local_L[self.axis] = self.w + 2.0 * self.g
            self.local_pbc[self.axis] = 0
        self.local_box = np.diag(self.local_L).reshape(9)
        self.pos = self.vel = self.frc = self.types = self.gid = None
        self.E = self.V = None
        self.bytes_sent = 0

    # ------------------------------------------------------------------ geometry
    def owner_of(self, x_axis):
        """Rank owning a (wrapped) coordinate along the axis."""
        r = torch.floor(x_axis / self.w).to(torch.int64)
        return torch.clamp(r, 0, self.world - 1)

    def _wrap_axis(self, pos):
        if self.world > 1 or self.pbc[self.axis]:
            L = self.L[self.axis]
            x = pos[:, self.axis]
            x = x - L * torch.floor(x / L)
            x = torch.where(x >= L, torch.zeros_like(x), x)
            pos = pos.clone()
            pos[:, self.axis] = x
        return pos

    def _to_local(self, pos):
        """Global -> local coordinates (nearest image to the slab centre, shifted so that the slab starts at g)."""
        if self.world == 1:
            return pos
        L = self.L[self.axis]
        d = pos[:, self.axis] - self.centre
        d = d - L * torch.round(d / L)
        out = pos.clone()
        out[:, self.axis] = d + 0.5 * self.w + self.g
        return out

    def _to_global(self, pos_local):
        if self.world == 1:
            return pos_local
        out = pos_local.clone()
        out[:, self.axis] = pos_local[:, self.axis] - self.g + self.lo
        return self._wrap_axis(out)

    # ------------------------------------------------------------------ scatter the initial system
    def scatter(self, pos, vel, types):
        """Every rank passes the same full system (host arrays); each keeps the atoms of its slab."""
        dev = self.engine.device
        pos = torch.as_tensor(np.asarray(pos, dtype=np.float64).reshape(-1, 3))
        pos = self._wrap_axis(pos)
        mine = self.owner_of(pos[:, self.axis]) == self.rank if self.world > 1 else torch.ones(len(pos), dtype=torch.bool)
        idx = torch.nonzero(mine).reshape(-1)
        self.gid = idx.to(dev)
        self.pos = pos[idx].to(dev)
        v = np.zeros((len(pos), 3)) if vel is None else np.asarray(vel, dtype=np.float64).reshape(-1, 3)
        self.vel = torch.as_tensor(v)[idx].to(dev)
        self.types = torch.as_tensor(np.asarray(types, dtype=np.int32))[idx].to(dev)
        self.frc = None
        return self

    # ------------------------------------------------------------------ messages
    def _exchange(self, to_left, to_right):
        """Send one payload [n, c] (float64) to each neighbour, receive theirs.  Returns (from_left, from_right)."""
        left, right = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        host = dist.get_backend(self.group) == "gloo"
        dev = self.engine.device
        c = to_left.shape[1]
        send = [t.cpu() if host else t.contiguous() for t in (to_left, to_right)]
        cdev = torch.device("cpu") if host else dev
        n_out = torch.tensor([send[0].shape[0], send[1].shape[0]], dtype=torch.int64, device=cdev)
        n_in = torch.zeros(2, dtype=torch.int64, device=cdev)
        # sizes first: my "to_left" count goes to the left neighbour, who stores it as its "from_right" count
        ops = [dist.P2POp(dist.isend, n_out[0:1], left, self.group, tag=1), dist.P2POp(dist.isend, n_out[1:2], right, self.group, tag=2),
               # receives in the peer's send order (its to_left arrives "from right"): NCCL matches by order, not tag
               dist.P2POp(dist.irecv, n_in[1:2], right, self.group, tag=1), dist.P2POp(dist.irecv, n_in[0:1], left, self.group, tag=2)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        n_l, n_r = int(n_in[0]), int(n_in[1])
        recv = [torch.empty((n_l, c), dtype=torch.float64, device=cdev), torch.empty((n_r, c), dtype=torch.float64, device=cdev)]
        ops = []
        if send[0].shape[0]:
            ops.append(dist.P2POp(dist.isend, send[0], left, self.group, tag=3))
        if send[1].shape[0]:
            ops.append(dist.P2POp(dist.isend, send[1], right, self.group, tag=4))
        if n_r:
            ops.append(dist.P2POp(dist.irecv, recv[1], right, self.group, tag=3))
        if n_l:
            ops.append(dist.P2POp(dist.irecv, recv[0], left, self.group, tag=4))
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()
        self.bytes_sent += 8 * c * (send[0].shape[0] + send[1].shape[0])
        return recv[0].to(dev), recv[1].to(dev)

    def _halo(self, with_dynamics: bool):
        """Ghost copies (global coordinates) of the neighbours' atoms within g of my slab."""
        dev = self.engine.device
        n = self.pos.shape[0]
        if self.world == 1:
            z = torch.zeros((0, 3), dtype=torch.float64, device=dev)
            return z, z, z, torch.zeros(0, dtype=torch.int32, device=dev)
        x = self.pos[:, self.axis] - self.lo
        cols = [self.pos, self.types.to(torch.float64).reshape(n, 1)]
        if with_dynamics:
            cols += [self.vel, self.frc]
        payload = torch.cat(cols, dim=1)
        got_l, got_r = self._exchange(payload[x < self.g], payload[x >= self.w - self.g])
        got = torch.cat([got_l, got_r], dim=0)
        gpos, gtyp = got[:, 0:3], got[:, 3].to(torch.int32)
        if with_dynamics:
            return gpos, got[:, 4:7], got[:, 7:10], gtyp
        z = torch.zeros_like(gpos)
        return gpos, z, z, gtyp

    def _migrate(self):
        """Hand owned atoms that left the slab to the neighbour that now owns them."""
        if self.world == 1:
            return
        n = self.pos.shape[0]
        owner = self.owner_of(self.pos[:, self.axis])
        left, right = (self.rank - 1) % self.world, (self.rank + 1) % self.world
        stay = owner == self.rank
        go_l = (owner == left) & ~stay
        go_r = (owner == right) & ~stay & ~go_l
        if bool((~(stay | go_l | go_r)).any()):
            raise RuntimeError("an atom moved further than one slab in one step")
        payload = torch.cat([self.pos, self.vel, self.frc, self.types.to(torch.float64).reshape(n, 1),
                             self.gid.to(torch.float64).reshape(n, 1), self.E.reshape(n, 1),
                             (self.V if self.V is not None else torch.zeros_like(self.E)).reshape(n, 1)], dim=1)
        got_l, got_r = self._exchange(payload[go_l], payload[go_r])
        allp = torch.cat([payload[stay], got_l, got_r], dim=0)
        self.pos, self.vel, self.frc = allp[:, 0:3].contiguous(), allp[:, 3:6].contiguous(), allp[:, 6:9].contiguous()
        self.types, self.gid = allp[:, 9].to(torch.int32), allp[:, 10].to(torch.int64)
        self.E = allp[:, 11].contiguous()
        self.V = allp[:, 12].contiguous() if self.V is not None else None

    # ------------------------------------------------------------------ the two entry points
    def compute(self, variances: bool = False):
        """One distributed force-field evaluation: E, F, V of the owned atoms (also kept as the MD forces)."""
        gpos, _, _, gtyp = self._halo(False)
        n = self.pos.shape[0]
        lpos = self._to_local(torch.cat([self.pos, gpos], dim=0))
        ltyp = torch.cat([self.types, gtyp], dim=0)
        e, f, v = self.engine.evaluate(lpos, ltyp, self.local_box, self.local_pbc, variances)
        self.E, self.frc = e[:n].clone(), f[:n].clone()
        self.V = v[:n].clone() if v is not None else None
        return self.E, self.frc, self.V

    def step(self, dt: float, n_steps: int = 1, variances: bool = False):
        """n_steps of velocity Verlet on the decomposed system."""
        if self.frc is None:
            self.compute(variances)
        for _ in range(n_steps):
            gpos, gvel, gfrc, gtyp = self._halo(True)
            n = self.pos.shape[0]
            lpos = self._to_local(torch.cat([self.pos, gpos], dim=0))
            lvel = torch.cat([self.vel, gvel], dim=0)
            lfrc = torch.cat([self.frc, gfrc], dim=0)
            ltyp = torch.cat([self.types, gtyp], dim=0)
            p, v, e, f, var = self.engine.md_step(lpos, lvel, lfrc, ltyp, self.local_box, self.local_pbc, dt, variances)
            self.pos = self._to_global(p[:n]) if self.world > 1 else p[:n].clone()
            self.vel, self.frc, self.E = v[:n].clone(), f[:n].clone(), e[:n].clone()
            self.V = var[:n].clone() if var is not None else None
            self._migrate()
        return self

    # ------------------------------------------------------------------ collect (tests, output)
    def gather(self):
        """Rank 0 gets dict(pos, vel, F, E, V, types) of the whole system in the original atom order; others None."""
        n = self.pos.shape[0]
        V = self.V if self.V is not None else torch.zeros(n, dtype=torch.float64, device=self.pos.device)
        E = self.E if self.E is not None else torch.zeros(n, dtype=torch.float64, device=self.pos.device)
        F = self.frc if self.frc is not None else torch.zeros_like(self.pos)
        mine = torch.cat([self.gid.to(torch.float64).reshape(n, 1), self.pos, self.vel, F, E.reshape(n, 1), V.reshape(n, 1),
                          self.types.to(torch.float64).reshape(n, 1)], dim=1).cpu()
        if self.world == 1:
            parts = [mine]
        else:
            parts = [None] * self.world
            dist.all_gather_object(parts, mine.numpy(), group=self.group)
            parts = [torch.as_tensor(p) for p in parts]
        if self.rank != 0:
            return None
        allp = torch.cat(parts, dim=0).numpy()
        order = np.argsort(allp[:, 0].astype(np.int64), kind="stable")
        a = allp[order]
        assert np.array_equal(a[:, 0].astype(np.int64), np.arange(a.shape[0])), "atoms lost or duplicated"
        return dict(pos=a[:, 1:4], vel=a[:, 4:7], F=a[:, 7:10], E=a[:, 10], V=a[:, 11], types=a[:, 12].astype(np.int32))
