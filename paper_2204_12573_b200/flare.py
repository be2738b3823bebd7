"""Thin Python binding over libflare_b200.so (include/flare_b200.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels; PyTorch is used here for
device memory (the workspace and the result tensors) and the CUDA stream.  There is no CPU
fallback: loading fails loudly if the shared library is missing, and flare_create fails
without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libflare_b200.so")

OK = 0
ERRORS = {
    -1: "FLARE_ERR_INVALID_ARG", -2: "FLARE_ERR_BOX_TOO_SMALL", -3: "FLARE_ERR_UNSUPPORTED_BOX",
    -4: "FLARE_ERR_WORKSPACE_TOO_SMALL", -5: "FLARE_ERR_NEIGHBOR_OVERFLOW", -6: "FLARE_ERR_CUDA",
    -7: "FLARE_ERR_NONFINITE", -8: "FLARE_ERR_UNSUPPORTED", -9: "FLARE_ERR_NOT_BOUND",
    -10: "FLARE_ERR_HALO_EXCEEDED",
}
OPT_MAX_NEIGHBORS, OPT_CHUNK_ATOMS, OPT_TIMING, OPT_SPECIES_SPARSE, OPT_SKIN, OPT_SKIN_REBUILDS = 1, 2, 3, 4, 5, 6
OPT_GRAPH, OPT_GRAPH_REPLAYS = 7, 8
PHASES = ("neighbor", "descriptor", "qform", "backprop", "gather", "integrate")

# every symbol include/flare_b200.h declares (checked by the CPU test-suite)
EXPORTS = (
    "flare_create", "flare_destroy", "flare_num_descriptors", "flare_set_option", "flare_get_option",
    "flare_workspace_bytes", "flare_bind", "flare_compute", "flare_compute_host", "flare_check",
    "flare_set_state", "flare_set_state_host", "flare_set_forces", "flare_set_forces_host", "flare_step", "flare_get_state", "flare_get_state_host",
    "flare_get_neighbors", "flare_get_descriptors", "flare_get_groups", "flare_get_rows", "flare_get_timings", "flare_kernel_launches",
    "flare_last_error",
    "flare_step_nvt", "flare_get_thermostat", "flare_set_thermostat", "flare_get_virial", "flare_virial_static", "flare_analyze",
    "flare_domain_begin", "flare_domain_migrate_pack", "flare_domain_migrate_unpack", "flare_domain_border_pack",
    "flare_domain_border_unpack", "flare_domain_commit", "flare_domain_forward_pack", "flare_domain_forward_unpack",
    "flare_domain_signal", "flare_domain_get_tags", "flare_domain_set_limit", "flare_domain_status",
)
VIRIAL_STATIC_MAX_ATOMS = 4194304  # FLARE_VIRIAL_STATIC_MAX_ATOMS
MSG_HEADER, MSG_FULL_ROW, MSG_FWD_ROW = 8, 11, 9  # message layout of the domain data plane (doubles)


class FlareError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"{ERRORS.get(code, code)}: {message}")
        self.code = code


_lib = None


def load_library():
    """dlopen libflare_b200.so (built by `python -m paper_2204_12573_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2204_12573_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_double
    lib.flare_create.argtypes = [C.POINTER(vp), i32, vp, i32, i32, vp, vp, vp, i32]
    lib.flare_destroy.argtypes = [vp]
    lib.flare_destroy.restype = None
    lib.flare_num_descriptors.argtypes = [vp]
    lib.flare_set_option.argtypes = [vp, i32, i64]
    lib.flare_get_option.argtypes = [vp, i32, C.POINTER(i64)]
    lib.flare_workspace_bytes.argtypes = [vp, i64]
    lib.flare_workspace_bytes.restype = C.c_size_t
    lib.flare_bind.argtypes = [vp, i64, vp, C.c_size_t, vp]
    lib.flare_compute.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.flare_compute_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.flare_check.argtypes = [vp]
    lib.flare_set_state.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.flare_set_state_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.flare_set_forces.argtypes = [vp, vp]
    lib.flare_set_forces_host.argtypes = [vp, vp]
    lib.flare_step.argtypes = [vp, dbl, i32, i32]
    lib.flare_get_state.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.flare_get_state_host.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.flare_get_neighbors.argtypes = [vp, vp, vp, C.c_int32]
    lib.flare_get_descriptors.argtypes = [vp, vp, vp]
    lib.flare_get_groups.argtypes = [vp, vp, vp, vp]
    lib.flare_get_rows.argtypes = [vp, vp]
    lib.flare_get_timings.argtypes = [vp, vp, vp]
    lib.flare_kernel_launches.argtypes = [vp]
    lib.flare_kernel_launches.restype = i64
    lib.flare_last_error.argtypes = [vp]
    lib.flare_last_error.restype = C.c_char_p
    lib.flare_step_nvt.argtypes = [vp, dbl, i32, i32, dbl, dbl]
    lib.flare_get_thermostat.argtypes = [vp, C.POINTER(dbl), C.POINTER(dbl)]
    lib.flare_set_thermostat.argtypes = [vp, dbl, dbl]
    lib.flare_get_virial.argtypes = [vp, vp]
    lib.flare_virial_static.argtypes = [vp, vp]
    lib.flare_analyze.argtypes = [vp, dbl, i32, i32, dbl, C.POINTER(dbl), C.POINTER(i64), vp, vp]
    lib.flare_domain_begin.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, dbl]
    lib.flare_domain_migrate_pack.argtypes = [vp, i32, dbl, dbl, dbl, dbl, vp, vp, i64]
    lib.flare_domain_migrate_unpack.argtypes = [vp, vp, vp, i64]
    lib.flare_domain_border_pack.argtypes = [vp, i32, i32, dbl, dbl, dbl, dbl, dbl, dbl, vp, vp, i64]
    lib.flare_domain_border_unpack.argtypes = [vp, i32, vp, vp, i64]
    lib.flare_domain_commit.argtypes = [vp, vp]
    lib.flare_domain_forward_pack.argtypes = [vp, i32, vp, vp]
    lib.flare_domain_forward_unpack.argtypes = [vp, i32, vp, vp]
    lib.flare_domain_signal.argtypes = [vp, vp]
    lib.flare_domain_get_tags.argtypes = [vp, vp]
    lib.flare_domain_set_limit.argtypes = [vp, dbl]
    lib.flare_domain_status.argtypes = [vp, vp]
    _lib = lib
    return lib


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _box9(box):
    b = np.asarray(box, dtype=np.float64)
    if b.size == 3:
        b = np.diag(b.reshape(3))
    return np.ascontiguousarray(b.reshape(9))


class Flare:
    """One model context bound to one CUDA device (flare_create ... flare_destroy)."""

    def __init__(self, mass, n_max: int, l_max: int, r_cut, beta, sigma=None, device: int = 0,
                 max_neighbors: int | None = None, chunk_atoms: int | None = None, timing: bool = False,
                 species_sparse: bool | None = None, skin: float | None = None, graph: int | None = None):
        import torch  # device memory + stream only

        self._torch = torch
        self._lib = load_library()
        self._ctx = C.c_void_p()
        mass = _np(mass, np.float64)
        r_cut = _np(r_cut, np.float64)
        S = mass.size
        assert r_cut.size == S * S
        nv = S * n_max
        P = nv * (nv + 1) // 2 * (l_max + 1)
        beta = _np(beta, np.float64)
        assert beta.size == S * P * P, "beta must be [S][P][P]"
        if sigma is not None:
            sigma = _np(sigma, np.float64)
            assert sigma.size == S * P * P
        rc = self._lib.flare_create(C.byref(self._ctx), S, _hp(mass), n_max, l_max, _hp(r_cut), _hp(beta), _hp(sigma),
                                    int(device))
        if rc != OK:
            raise FlareError(rc, "flare_create failed")
        self.device = torch.device("cuda", int(device))
        self.n_species, self.n_max, self.l_max, self.P = S, n_max, l_max, P
        self.has_sigma = sigma is not None
        self.n_atoms = None
        self._workspace = None
        self._stream = None
        if max_neighbors is not None:
            self.set_option(OPT_MAX_NEIGHBORS, max_neighbors)
        if chunk_atoms is not None:
            self.set_option(OPT_CHUNK_ATOMS, chunk_atoms)
        if timing:
            self.set_option(OPT_TIMING, 1)
        if species_sparse is not None:
            self.set_option(OPT_SPECIES_SPARSE, 1 if species_sparse else 0)
        if skin is not None:
            self.set_option(OPT_SKIN, int(round(1e3 * skin)))  # Angstrom -> 1e-3 Angstrom
        if graph is not None:
            self.set_option(OPT_GRAPH, int(graph))  # -1 automatic, 0 never, 1 always

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc: int):
        if rc != OK:
            msg = self._lib.flare_last_error(self._ctx)
            raise FlareError(rc, msg.decode() if msg else "")

    def close(self):
        if getattr(self, "_ctx", None) and self._ctx.value:
            self._lib.flare_destroy(self._ctx)
            self._ctx = C.c_void_p()
            self._workspace = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, option: int, value: int):
        self._check(self._lib.flare_set_option(self._ctx, option, int(value)))

    def get_option(self, option: int) -> int:
        v = C.c_int64(0)
        self._check(self._lib.flare_get_option(self._ctx, option, C.byref(v)))
        return int(v.value)

    def workspace_bytes(self, n_atoms: int) -> int:
        return int(self._lib.flare_workspace_bytes(self._ctx, int(n_atoms)))

    def bind(self, n_atoms: int, stream=None, workspace=None):
        """Attach the workspace for n_atoms on `stream` (default: current).  The workspace is a torch uint8 tensor:
        allocated here, or an earlier (large enough) one passed as `workspace` to avoid re-allocation."""
        torch = self._torch
        nbytes = self.workspace_bytes(n_atoms)
        if nbytes == 0:
            raise FlareError(-1, "flare_workspace_bytes returned 0")
        if workspace is not None and workspace.numel() >= nbytes:
            self._workspace = workspace
        else:
            self._workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._check(self._lib.flare_bind(self._ctx, int(n_atoms), C.c_void_p(self._workspace.data_ptr()),
                                         self._workspace.numel(), C.c_void_p(self._stream.cuda_stream)))
        self.n_atoms = int(n_atoms)
        return self

    def _dev(self, t, dtype, shape):
        torch = self._torch
        assert t.is_cuda and t.dtype == dtype and t.is_contiguous() and tuple(t.shape) == shape, (t.dtype, t.shape)
        return C.c_void_p(t.data_ptr())

    # ------------------------------------------------------------------ evaluation
    def compute(self, pos, types, box, pbc, energies=True, forces=True, variances=False, out=None, check=True):
        """Device tensors in, device tensors out: (E [N], F [N,3], V [N]); entries not asked for are None."""
        torch = self._torch
        n = self.n_atoms
        p_pos = self._dev(pos, torch.float64, (n, 3))
        p_typ = self._dev(types, torch.int32, (n,))
        if out is None:
            e = torch.empty(n, dtype=torch.float64, device=self.device) if energies else None
            f = torch.empty((n, 3), dtype=torch.float64, device=self.device) if forces else None
            v = torch.empty(n, dtype=torch.float64, device=self.device) if variances else None
        else:
            e, f, v = out
        boxh, pbch = _box9(box), _np(pbc, np.int32)
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._check(self._lib.flare_compute(self._ctx, p_pos, p_typ, _hp(boxh), _hp(pbch), ptr(e), ptr(f), ptr(v)))
        if check:
            self.check()
        return e, f, v

    def compute_host(self, pos, types, box, pbc, energies=True, forces=True, variances=False, out=None):
        """Host (numpy) arrays in and out through flare_compute_host (copies inside the call)."""
        n = self.n_atoms
        pos = _np(pos, np.float64).reshape(n, 3)
        types = _np(types, np.int32).reshape(n)
        if out is None:
            e = np.empty(n) if energies else None
            f = np.empty((n, 3)) if forces else None
            v = np.empty(n) if variances else None
        else:
            e, f, v = out
        boxh, pbch = _box9(box), _np(pbc, np.int32)
        self._check(self._lib.flare_compute_host(self._ctx, _hp(pos), _hp(types), _hp(boxh), _hp(pbch), _hp(e), _hp(f),
                                                 _hp(v)))
        return e, f, v

    def check(self):
        self._check(self._lib.flare_check(self._ctx))

    # ------------------------------------------------------------------ molecular dynamics
    def set_state(self, pos, vel, types, box, pbc):
        torch = self._torch
        n = self.n_atoms
        boxh, pbch = _box9(box), _np(pbc, np.int32)
        if isinstance(pos, np.ndarray):
            pos = _np(pos, np.float64).reshape(n, 3)
            vel = None if vel is None else _np(vel, np.float64).reshape(n, 3)
            types = _np(types, np.int32).reshape(n)
            self._check(self._lib.flare_set_state_host(self._ctx, _hp(pos), _hp(vel), _hp(types), _hp(boxh), _hp(pbch)))
        else:
            pv = None if vel is None else self._dev(vel, torch.float64, (n, 3))
            self._check(self._lib.flare_set_state(self._ctx, self._dev(pos, torch.float64, (n, 3)), pv,
                                                  self._dev(types, torch.int32, (n,)), _hp(boxh), _hp(pbch)))

    def set_forces(self, f):
        """Forces belonging to the state just set (skips the initial evaluation of step())."""
        n = self.n_atoms
        if isinstance(f, np.ndarray):
            f = _np(f, np.float64).reshape(n, 3)
            self._check(self._lib.flare_set_forces_host(self._ctx, _hp(f)))
        else:
            self._check(self._lib.flare_set_forces(self._ctx, self._dev(f, self._torch.float64, (n, 3))))

    def step(self, dt_fs: float, n_steps: int = 1, want_variance: bool = False):
        self._check(self._lib.flare_step(self._ctx, float(dt_fs), int(n_steps), 1 if want_variance else 0))

    def step_nvt(self, dt_fs: float, n_steps: int, T_kelvin: float, tau_fs: float, want_variance: bool = False):
        self._check(self._lib.flare_step_nvt(self._ctx, float(dt_fs), int(n_steps), 1 if want_variance else 0,
                                             float(T_kelvin), float(tau_fs)))

    def thermostat(self):
        xi, eta = C.c_double(0.0), C.c_double(0.0)
        self._check(self._lib.flare_get_thermostat(self._ctx, C.byref(xi), C.byref(eta)))
        return xi.value, eta.value

    def set_thermostat(self, xi: float, eta: float):
        self._check(self._lib.flare_set_thermostat(self._ctx, float(xi), float(eta)))

    def virial(self):
        """[3,3] virial dE/d eps (eV) of the last evaluation."""
        w = np.zeros(9)
        self._check(self._lib.flare_get_virial(self._ctx, _hp(w)))
        return w.reshape(3, 3)

    def virial_static(self, out):
        """Enqueue the virial of the last evaluation into `out`, a caller-owned float64 CUDA tensor of 9 elements, and
        return it (valid after the bound stream is synchronised).  For callers that may not allocate device memory:
        the reduction scratch is a static array inside the library (flare_virial_static in include/flare_b200.h:
        at most VIRIAL_STATIC_MAX_ATOMS atoms, one shared array per GPU, so overlapping calls race)."""
        if out.dtype != self._torch.float64 or out.numel() != 9 or not out.is_cuda or not out.is_contiguous():
            raise ValueError("out must be a contiguous float64 CUDA tensor with 9 elements")
        self._check(self._lib.flare_virial_static(self._ctx, C.c_void_p(out.data_ptr())))
        return out

    def analyze(self, threshold: float = 0.0, species_a: int = 0, species_b: int = 0, r_coord: float = 1.0,
                uncertainty: bool = True, coordination: bool = True):
        """dict(max_unc, n_above, coord (device int32 tensor), hist[16]) of the last evaluation."""
        mx, na = C.c_double(0.0), C.c_int64(0)
        hist = np.zeros(16, np.int64)
        coord = self._torch.zeros(self.n_atoms, dtype=self._torch.int32, device=self.device) if coordination else None
        self._check(self._lib.flare_analyze(
            self._ctx, float(threshold), int(species_a), int(species_b), float(r_coord),
            C.byref(mx) if uncertainty else None, C.byref(na) if uncertainty else None,
            C.c_void_p(coord.data_ptr()) if coordination else None, _hp(hist) if coordination else None))
        return dict(max_unc=mx.value if uncertainty else None, n_above=na.value if uncertainty else None,
                    coord=coord, hist=hist if coordination else None)

    def get_state(self, variances: bool = False, results: bool = True):
        """Device tensors dict(pos, vel, E, F[, V]); results=False: positions and velocities only (no evaluation needed)."""
        torch = self._torch
        n = self.n_atoms
        mk = lambda *s: torch.empty(s, dtype=torch.float64, device=self.device)
        pos, vel = mk(n, 3), mk(n, 3)
        e, f = (mk(n), mk(n, 3)) if results else (None, None)
        v = mk(n) if (variances and results) else None
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._check(self._lib.flare_get_state(self._ctx, ptr(pos), ptr(vel), ptr(e), ptr(f), ptr(v)))
        self.check()
        return dict(pos=pos, vel=vel, E=e, F=f, V=v)

    def get_state_host(self, variances: bool = False, out=None):
        n = self.n_atoms
        if out is None:
            out = dict(pos=np.empty((n, 3)), vel=np.empty((n, 3)), E=np.empty(n), F=np.empty((n, 3)),
                       V=np.empty(n) if variances else None)
        self._check(self._lib.flare_get_state_host(self._ctx, _hp(out["pos"]), _hp(out["vel"]), _hp(out["E"]),
                                                   _hp(out["F"]), _hp(out.get("V"))))
        return out

    # ------------------------------------------------------------------ domain decomposition (device data plane)
    def _msg(self, t):
        return None if t is None else self._dev(t, self._torch.float64, tuple(t.shape))

    def domain_begin(self, n_owned, pos, vel, types, tags, box, pbc, trigger: float):
        torch = self._torch
        n = int(n_owned)
        boxh, pbch = _box9(box), _np(pbc, np.int32)
        self._check(self._lib.flare_domain_begin(
            self._ctx, n, self._dev(pos, torch.float64, (n, 3)), None if vel is None else self._dev(vel, torch.float64, (n, 3)),
            self._dev(types, torch.int32, (n,)), self._dev(tags, torch.int64, (n,)), _hp(boxh), _hp(pbch), float(trigger)))
        self.n_atoms = n

    def domain_migrate_pack(self, axis, lo_bound, hi_bound, shift_lo, shift_hi, msg_lo, msg_hi, cap_rows):
        self._check(self._lib.flare_domain_migrate_pack(self._ctx, int(axis), float(lo_bound), float(hi_bound), float(shift_lo),
                                                        float(shift_hi), self._msg(msg_lo), self._msg(msg_hi), int(cap_rows)))

    def domain_migrate_unpack(self, msg_lo_in, msg_hi_in, cap_rows):
        self._check(self._lib.flare_domain_migrate_unpack(self._ctx, self._msg(msg_lo_in), self._msg(msg_hi_in), int(cap_rows)))

    def domain_border_pack(self, phase, axis, lo_a, lo_b, hi_a, hi_b, shift_lo, shift_hi, msg_lo, msg_hi, cap_rows):
        self._check(self._lib.flare_domain_border_pack(self._ctx, int(phase), int(axis), float(lo_a), float(lo_b), float(hi_a),
                                                       float(hi_b), float(shift_lo), float(shift_hi), self._msg(msg_lo),
                                                       self._msg(msg_hi), int(cap_rows)))

    def domain_border_unpack(self, phase, msg_lo_in, msg_hi_in, cap_rows):
        self._check(self._lib.flare_domain_border_unpack(self._ctx, int(phase), self._msg(msg_lo_in), self._msg(msg_hi_in),
                                                         int(cap_rows)))

    def domain_commit(self):
        """-> dict(n_local, n_owned, send[4], recv[4], recv_off[4]); n_atoms becomes n_local."""
        c = np.zeros(14, np.int64)
        self._check(self._lib.flare_domain_commit(self._ctx, _hp(c)))
        self.n_atoms = int(c[0])
        return dict(n_local=int(c[0]), n_owned=int(c[1]), send=[int(v) for v in c[2:6]], recv=[int(v) for v in c[6:10]],
                    recv_off=[int(v) for v in c[10:14]])

    def domain_forward_pack(self, phase, msg_lo, msg_hi):
        self._check(self._lib.flare_domain_forward_pack(self._ctx, int(phase), self._msg(msg_lo), self._msg(msg_hi)))

    def domain_forward_unpack(self, phase, msg_lo_in, msg_hi_in):
        self._check(self._lib.flare_domain_forward_unpack(self._ctx, int(phase), self._msg(msg_lo_in), self._msg(msg_hi_in)))

    def domain_set_limit(self, max_displacement: float):
        """Displacement since the last domain rebuild beyond which the ghost shell is no longer trusted (an error)."""
        self._check(self._lib.flare_domain_set_limit(self._ctx, float(max_displacement)))

    def domain_status(self, status):
        """Device-side error bits so far -> int32[1] device tensor (asynchronous, not cleared)."""
        self._check(self._lib.flare_domain_status(self._ctx, self._dev(status, self._torch.int32, (1,))))

    def domain_signal(self, flag):
        self._check(self._lib.flare_domain_signal(self._ctx, self._dev(flag, self._torch.int32, (1,))))

    def domain_tags(self):
        t = self._torch.empty(self.n_atoms, dtype=self._torch.int64, device=self.device)
        self._check(self._lib.flare_domain_get_tags(self._ctx, C.c_void_p(t.data_ptr())))
        return t

    # ------------------------------------------------------------------ hooks
    def neighbors(self, stride: int | None = None):
        n = self.n_atoms
        stride = stride or self.get_option(OPT_MAX_NEIGHBORS)
        cnt = np.zeros(n, np.int32)
        idx = np.full((n, stride), -1, np.int32)
        self._check(self._lib.flare_get_neighbors(self._ctx, _hp(cnt), _hp(idx), stride))
        return cnt, idx

    def descriptors(self):
        n = self.n_atoms
        bh = np.zeros((n, self.P))
        nrm = np.zeros(n)
        self._check(self._lib.flare_get_descriptors(self._ctx, _hp(bh), _hp(nrm)))
        return bh, nrm

    def groups(self):
        """[(rows, components)] of the quadratic-form groups of the last evaluation."""
        n = C.c_int32(0)
        rows = np.zeros(64, np.int64)
        comps = np.zeros(64, np.int32)
        self._check(self._lib.flare_get_groups(self._ctx, C.cast(C.byref(n), C.c_void_p), _hp(rows), _hp(comps)))
        return [(int(rows[g]), int(comps[g])) for g in range(n.value)]

    def rows(self):
        """Quadratic-form row of every atom (caller's order) in the last evaluation."""
        row = np.zeros(self.n_atoms, np.int32)
        self._check(self._lib.flare_get_rows(self._ctx, _hp(row)))
        return row

    def qform_flops(self, variance: bool, symmetric: bool = False) -> float:
        """Flops of steps a4 (+ a5) per evaluation.  Default: SURVEY.md 8(d)'s algorithmic count, 2 P_g^2 per atom and
        per form.  symmetric=True: what the kernel needs since the variance tiles use the symmetry of Sigma -- all of
        W = beta d (it feeds the forces) but only the 16 x 16 blocks of Sigma on and above the diagonal (512 flops each)."""
        tot = 0.0
        for r, p in self.groups():
            tot += r * 2.0 * p * p
            if variance and symmetric:
                nsb = (p + 15) // 16
                tot += r * 512.0 * (nsb * (nsb + 1) // 2)
            elif variance:
                tot += r * 2.0 * p * p
        return float(tot)

    def timings(self):
        ms = np.zeros(len(PHASES))
        launches = np.zeros(len(PHASES), np.int64)
        self._check(self._lib.flare_get_timings(self._ctx, _hp(ms), _hp(launches)))
        return {p: (float(ms[i]), int(launches[i])) for i, p in enumerate(PHASES)}

    def kernel_launches(self) -> int:
        return int(self._lib.flare_kernel_launches(self._ctx))


def from_system(system, device: int = 0, variance: bool = True, **kw) -> Flare:
    """Context for a workloads.System (model matrices must be present)."""
    return Flare(system.mass, system.n_max, system.l_max, system.r_cut, system.beta,
                 system.sigma if variance else None, device=device, **kw)
