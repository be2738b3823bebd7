"""Test infrastructure: a numpy restatement of the domain data plane (include/flare_b200.h, flare_domain_*) with the
CPU oracle as the force field, behind the `halo.Engine` interface.  It lets the world_size > 1 orchestration of
`paper_2204_12573_b200.halo.DomainDecomposition` run on CPU over gloo, and it is the reference the CUDA data plane is
compared with on the GPU (same calls, same messages).  Written from the header's description, not from domain.cu."""
import numpy as np
import torch

KAPPA = 9.648533212331e-3
H, FULL, FWD = 8, 11, 9


class HaloExceeded(RuntimeError):
    """The reference's FLARE_ERR_HALO_EXCEEDED."""


class NumpyOracleEngine:
    device = torch.device("cpu")

    def __init__(self, oracle, mass, n_max, l_max, r_cut, beta, sigma, capacity=1 << 30):
        self.o, self.mass, self.n_max, self.l_max, self.rc, self.beta, self.sigma = oracle, np.asarray(mass), n_max, l_max, r_cut, beta, sigma
        self.capacity = capacity
        self.max_local = 0
        self.evaluations = 0

    # ---- state
    def begin(self, pos, vel, types, tags, box, pbc, trigger):
        n = len(tags)
        self.x = np.array(pos, dtype=np.float64).reshape(n, 3)
        self.v = np.array(vel, dtype=np.float64).reshape(n, 3)
        self.f = np.zeros((n, 3))
        self.t = np.array(types, dtype=np.int32).reshape(n)
        self.tag = np.array(tags, dtype=np.int64).reshape(n)
        self.E = np.zeros(n)
        self.V = np.zeros(n)
        self.box = np.asarray(box, dtype=np.float64).reshape(9)
        self.pbc = np.asarray(pbc, dtype=np.int32).reshape(3)
        self.trigger = trigger
        self.n_owned = n
        self.forces_valid = False
        self.lists = [np.zeros(0, np.int64)] * 4
        self.shift = np.zeros((4, 3))
        self.recv_off, self.recv_cnt = [0] * 4, [0] * 4
        self.ref = None
        self.need = 0
        self.limit = 0.0
        self.error = 0

    def set_limit(self, max_displacement):
        """flare_domain_set_limit: a displacement of that size since the last rebuild is an error, not a signal."""
        assert max_displacement == 0.0 or max_displacement > self.trigger
        self.limit = float(max_displacement)

    def _truncate(self, n):
        self.x, self.v, self.f, self.t, self.tag = self.x[:n], self.v[:n], self.f[:n], self.t[:n], self.tag[:n]

    def _rows(self, idx, shift, with_force=True):
        r = np.zeros((len(idx), FULL))
        r[:, 0:3] = self.x[idx] + shift
        r[:, 3:6] = self.v[idx]
        if with_force:
            r[:, 6:9] = self.f[idx]
        r[:, 9] = self.t[idx]
        r[:, 10] = self.tag[idx]
        return r

    @staticmethod
    def _put(msg, rows, width, cap):
        assert len(rows) <= cap, "message capacity exceeded"
        msg[0] = float(len(rows))
        msg[H:H + rows.size] = torch.as_tensor(rows.reshape(-1))

    @staticmethod
    def _get(msg, width):
        n = int(msg[0])
        return msg[H:H + n * width].numpy().reshape(n, width)

    def _append(self, rows):
        self.x = np.concatenate([self.x, rows[:, 0:3]])
        self.v = np.concatenate([self.v, rows[:, 3:6]])
        self.f = np.concatenate([self.f, rows[:, 6:9]])
        self.t = np.concatenate([self.t, rows[:, 9].astype(np.int32)])
        self.tag = np.concatenate([self.tag, rows[:, 10].astype(np.int64)])
        assert len(self.x) <= self.capacity

    # ---- migration
    def migrate_pack(self, axis, lo_bound, hi_bound, shift_lo, shift_hi, msg_lo, msg_hi, cap):
        self._truncate(self.n_owned)
        c = self.x[:, axis]
        go_lo, go_hi = c < lo_bound, c >= hi_bound
        for sel, sh, msg in ((go_lo, shift_lo, msg_lo), (go_hi, shift_hi, msg_hi)):
            s3 = np.zeros(3)
            s3[axis] = sh
            self._put(msg, self._rows(np.nonzero(sel)[0], s3), FULL, cap)
        stay = ~(go_lo | go_hi)
        self.x, self.v, self.f, self.t, self.tag = self.x[stay], self.v[stay], self.f[stay], self.t[stay], self.tag[stay]
        self.n_owned = len(self.x)

    def migrate_unpack(self, msg_lo_in, msg_hi_in, cap):
        for msg in (msg_lo_in, msg_hi_in):
            if msg is not None:
                self._append(self._get(msg, FULL))
        self.n_owned = len(self.x)

    # ---- borders
    def border_pack(self, phase, axis, lo_a, lo_b, hi_a, hi_b, shift_lo, shift_hi, msg_lo, msg_hi, cap):
        if phase == 0:
            self._truncate(self.n_owned)
        c = self.x[:, axis]
        for side, (a, b, sh, msg) in enumerate(((lo_a, lo_b, shift_lo, msg_lo), (hi_a, hi_b, shift_hi, msg_hi))):
            idx = np.nonzero((c >= a) & (c < b))[0]
            q = 2 * phase + side
            self.lists[q] = idx
            self.shift[q] = 0.0
            self.shift[q, axis] = sh
            self._put(msg, self._rows(idx, self.shift[q], self.forces_valid), FULL, cap)

    def border_unpack(self, phase, msg_lo_in, msg_hi_in, cap):
        for side, msg in enumerate((msg_lo_in, msg_hi_in)):
            rows = self._get(msg, FULL) if msg is not None else np.zeros((0, FULL))
            q = 2 * phase + side
            self.recv_off[q], self.recv_cnt[q] = len(self.x), len(rows)
            self._append(rows)

    def check(self):
        if self.error:
            self.error = 0
            raise HaloExceeded("an atom has moved further since the last rebuild than the ghost shell covers")

    def commit(self):
        self.check()
        n = len(self.x)
        self.E, self.V = np.zeros(n), np.zeros(n)
        self.ref = self.x.copy()
        self.need = 0
        self.max_local = max(self.max_local, n)
        return dict(n_local=n, n_owned=self.n_owned, send=[len(l) for l in self.lists], recv=list(self.recv_cnt),
                    recv_off=list(self.recv_off))

    # ---- per step
    def forward_pack(self, phase, msg_lo, msg_hi):
        for side, msg in enumerate((msg_lo, msg_hi)):
            q = 2 * phase + side
            idx = self.lists[q]
            rows = np.concatenate([self.x[idx] + self.shift[q], self.v[idx], self.f[idx]], axis=1) if len(idx) else np.zeros((0, FWD))
            self._put(msg, rows, FWD, 1 << 30)

    def forward_unpack(self, phase, msg_lo_in, msg_hi_in):
        for side, msg in enumerate((msg_lo_in, msg_hi_in)):
            q = 2 * phase + side
            rows = self._get(msg, FWD)
            assert len(rows) == self.recv_cnt[q]
            sl = slice(self.recv_off[q], self.recv_off[q] + len(rows))
            self.x[sl], self.v[sl], self.f[sl] = rows[:, 0:3], rows[:, 3:6], rows[:, 6:9]

    def _evaluate(self):
        self.evaluations += 1
        E, F, V = self.o.compute(self.x, self.t, self.box, self.pbc, self.n_max, self.l_max, self.rc, self.beta, self.sigma,
                                 nbr_method=0)
        self.E, self.f, self.V = E, F, V
        self.forces_valid = True
        if self.ref is not None and len(self.ref) == len(self.x):
            d = self.x - self.ref
            L = self.box.reshape(3, 3).diagonal()
            for k in range(3):
                if self.pbc[k]:
                    d[:, k] -= L[k] * np.round(d[:, k] / L[k])
            if len(d) and np.sqrt((d * d).sum(1)).max() >= self.trigger:
                self.need = 1
            if self.limit > 0.0 and len(d) and np.sqrt((d * d).sum(1)).max() >= self.limit:
                self.error |= 32  # reported like the device's flag: by signal (bits), check and commit (exception)

    def step(self, dt, n_steps, variances):
        if not self.forces_valid:
            self._evaluate()
        for _ in range(n_steps):
            acc = (0.5 * dt * KAPPA / self.mass[self.t])[:, None]
            self.v = self.v + acc * self.f
            self.x = self.x + dt * self.v
            L = self.box.reshape(3, 3).diagonal()
            for k in range(3):
                if self.pbc[k]:
                    self.x[:, k] -= L[k] * np.floor(self.x[:, k] / L[k])
            self._evaluate()
            self.v = self.v + acc * self.f

    def signal(self, flag):
        flag[0] = 1 if (self.need or self.trigger <= 0.0) else 0
        flag[1] = self.error

    def owned(self, variances):
        n = self.n_owned
        return dict(tags=self.tag[:n].copy(), pos=self.x[:n].copy(), vel=self.v[:n].copy(), E=self.E[:n].copy(),
                    F=self.f[:n].copy(), V=self.V[:n].copy() if variances else None)
