"""ctypes loader for the CPU oracle (oracle/flare_oracle.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It does not import the product package
and shares nothing with the CUDA path.  Every function is a 1:1 marshalling of a C entry
point; the arithmetic (cited to the paper there) lives in flare_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "flare_oracle.c")
_LIB = os.path.join(_HERE, "libflare_oracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-D_GNU_SOURCE"]

_lib = None


def build(force: bool = False) -> str:
    """gcc-compile the oracle next to its source (no-op when up to date)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.oracle_cutoff.restype = C.c_double
        _lib.oracle_cutoff.argtypes = [C.c_double, C.c_double, C.c_void_p]
        _lib.oracle_chebyshev.argtypes = [C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        _lib.oracle_radial.argtypes = [C.c_int, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _box9(box):
    b = _f64(box)
    if b.size == 3:
        b = np.diag(b.reshape(3))
    return _f64(b.reshape(9))


def _pbc3(pbc):
    return np.ascontiguousarray(pbc, dtype=np.int32).reshape(3)


class OracleError(RuntimeError):
    pass


def _check(rc, what):
    if rc != 0:
        raise OracleError(f"{what} failed with code {rc}")


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(C.c_int(int(n)))


def num_descriptors(S: int, n_max: int, l_max: int) -> int:
    return int(lib().oracle_num_descriptors(S, n_max, l_max))


def b2_index(S, n_max, l_max, v1, v2, l) -> int:
    return int(lib().oracle_b2_index(S, n_max, l_max, v1, v2, l))


def chebyshev(n_max: int, x: float):
    T = np.zeros(n_max)
    dT = np.zeros(n_max)
    lib().oracle_chebyshev(n_max, float(x), _p(T), _p(dT))
    return T, dT


def cutoff(r: float, rc: float):
    d = C.c_double(0.0)
    f = lib().oracle_cutoff(float(r), float(rc), C.cast(C.byref(d), C.c_void_p))
    return float(f), float(d.value)


def radial(n_max: int, r: float, rc: float):
    g = np.zeros(n_max)
    dg = np.zeros(n_max)
    lib().oracle_radial(n_max, float(r), float(rc), _p(g), _p(dg))
    return g, dg


def ylm(l_max: int, u):
    """Real orthonormal Y_lm at unit vector u and the (unprojected) gradient of the
    polynomial extension, shape [(l_max+1)^2] and [(l_max+1)^2, 3]."""
    u = _f64(u).reshape(3)
    L2 = (l_max + 1) ** 2
    Y = np.zeros(L2)
    dY = np.zeros((L2, 3))
    lib().oracle_ylm(C.c_int(l_max), _p(u), _p(Y), _p(dY))
    return Y, dY


def wrap(pos, box, pbc):
    pos = _f64(pos).reshape(-1, 3)
    out = np.empty_like(pos)
    lib().oracle_wrap(C.c_int64(pos.shape[0]), _p(pos), _p(_box9(box)), _p(_pbc3(pbc)), _p(out))
    return out


def neighbors(pos, types, box, pbc, r_cut, method: int = 1, cap: int = 96):
    """Neighbour sets (caller's order), rows sorted by j.  Returns (cnt[N], idx[N,cap])."""
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    N = pos.shape[0]
    r_cut = _f64(r_cut)
    S = int(round(np.sqrt(r_cut.size)))
    cnt = np.zeros(N, dtype=np.int32)
    idx = np.full((N, cap), -1, dtype=np.int32)
    rc = lib().oracle_neighbors(C.c_int64(N), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)), C.c_int(S),
                                _p(r_cut), C.c_int(method), _p(cnt), _p(idx), C.c_int32(cap))
    _check(rc, "oracle_neighbors")
    return cnt, idx


def descriptor_env(S, n_max, l_max, r_cut, si, rij, sj):
    """A, B, B^, nrm of one explicit environment (displacements rij[M,3], species sj[M])."""
    rij = _f64(rij).reshape(-1, 3)
    sj = _i32(sj)
    r_cut = _f64(r_cut)
    P = num_descriptors(S, n_max, l_max)
    L2 = (l_max + 1) ** 2
    A = np.zeros((S * n_max, L2))
    B = np.zeros(P)
    Bh = np.zeros(P)
    nrm = C.c_double(0.0)
    rc = lib().oracle_descriptor_env(C.c_int(S), C.c_int(n_max), C.c_int(l_max), _p(r_cut), C.c_int(si),
                                     C.c_int(rij.shape[0]), _p(rij), _p(sj), _p(A), _p(B), _p(Bh), C.byref(nrm))
    _check(rc, "oracle_descriptor_env")
    return A, B, Bh, float(nrm.value)


def descriptor(pos, types, box, pbc, n_max, l_max, r_cut, i):
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    r_cut = _f64(r_cut)
    S = int(round(np.sqrt(r_cut.size)))
    P = num_descriptors(S, n_max, l_max)
    L2 = (l_max + 1) ** 2
    A = np.zeros((S * n_max, L2))
    B = np.zeros(P)
    Bh = np.zeros(P)
    nrm = C.c_double(0.0)
    rc = lib().oracle_descriptor(C.c_int64(pos.shape[0]), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)),
                                 C.c_int(S), C.c_int(n_max), C.c_int(l_max), _p(r_cut), C.c_int64(i), _p(A), _p(B),
                                 _p(Bh), C.byref(nrm))
    _check(rc, "oracle_descriptor")
    return A, B, Bh, float(nrm.value)


def _model_args(n_max, l_max, r_cut, beta, sigma):
    r_cut = _f64(r_cut)
    S = int(round(np.sqrt(r_cut.size)))
    P = num_descriptors(S, n_max, l_max)
    beta = _f64(beta)
    assert beta.size == S * P * P, (beta.shape, S, P)
    if sigma is not None:
        sigma = _f64(sigma)
        assert sigma.size == S * P * P
    return S, r_cut, beta, sigma


def compute(pos, types, box, pbc, n_max, l_max, r_cut, beta, sigma=None, nbr_method: int = 1, forces: bool = True):
    """Per-atom E [N], F [N,3], V [N] (V zeros when sigma is None)."""
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    N = pos.shape[0]
    S, r_cut, beta, sigma = _model_args(n_max, l_max, r_cut, beta, sigma)
    E = np.zeros(N)
    F = np.zeros((N, 3)) if forces else None
    V = np.zeros(N)
    rc = lib().oracle_compute(C.c_int64(N), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)), C.c_int(S),
                              C.c_int(n_max), C.c_int(l_max), _p(r_cut), _p(beta), _p(sigma), C.c_int(nbr_method),
                              _p(E), _p(F), _p(V))
    _check(rc, "oracle_compute")
    return E, F, V


def compute_selected(pos, types, box, pbc, n_max, l_max, r_cut, beta, sigma, sel, forces: bool = True):
    """E, F, V of the atoms in `sel` only (each needs its neighbours' environments too)."""
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    N = pos.shape[0]
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    S, r_cut, beta, sigma = _model_args(n_max, l_max, r_cut, beta, sigma)
    E = np.zeros(sel.size)
    F = np.zeros((sel.size, 3))
    V = np.zeros(sel.size)
    rc = lib().oracle_compute_selected(C.c_int64(N), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)), C.c_int(S),
                                       C.c_int(n_max), C.c_int(l_max), _p(r_cut), _p(beta), _p(sigma),
                                       C.c_int64(sel.size), _p(sel), C.c_int(1 if forces else 0), _p(E), _p(F), _p(V))
    _check(rc, "oracle_compute_selected")
    return E, F, V


def step(pos, vel, types, mass, box, pbc, n_max, l_max, r_cut, beta, sigma, dt, n_steps, nbr_method: int = 1):
    """Velocity-Verlet NVE.  Returns dict(pos, vel, E, F, V, pe[n_steps+1], ke[n_steps+1])."""
    pos = _f64(pos).reshape(-1, 3).copy()
    vel = _f64(vel).reshape(-1, 3).copy()
    types = _i32(types)
    mass = _f64(mass)
    N = pos.shape[0]
    S, r_cut, beta, sigma = _model_args(n_max, l_max, r_cut, beta, sigma)
    E = np.zeros(N)
    F = np.zeros((N, 3))
    V = np.zeros(N)
    pe = np.zeros(n_steps + 1)
    ke = np.zeros(n_steps + 1)
    rc = lib().oracle_step(C.c_int64(N), _p(pos), _p(vel), _p(types), _p(mass), _p(_box9(box)), _p(_pbc3(pbc)),
                           C.c_int(S), C.c_int(n_max), C.c_int(l_max), _p(r_cut), _p(beta), _p(sigma),
                           C.c_int(nbr_method), C.c_double(dt), C.c_int(n_steps), _p(E), _p(F), _p(V), _p(pe), _p(ke))
    _check(rc, "oracle_step")
    return dict(pos=pos, vel=vel, E=E, F=F, V=V, pe=pe, ke=ke)


def compute_virial(pos, types, box, pbc, n_max, l_max, r_cut, beta, sigma=None, nbr_method: int = 1):
    """E [N], F [N,3], V [N] and the virial Xi [3,3] = dE/d eps (eV); potential stress = Xi / volume."""
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    N = pos.shape[0]
    S, r_cut, beta, sigma = _model_args(n_max, l_max, r_cut, beta, sigma)
    E, F, V, W = np.zeros(N), np.zeros((N, 3)), np.zeros(N), np.zeros(9)
    rc = lib().oracle_compute_virial(C.c_int64(N), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)), C.c_int(S),
                                     C.c_int(n_max), C.c_int(l_max), _p(r_cut), _p(beta), _p(sigma),
                                     C.c_int(nbr_method), _p(E), _p(F), _p(V), _p(W))
    _check(rc, "oracle_compute_virial")
    return E, F, V, W.reshape(3, 3)


def analyze(pos, types, box, pbc, var, threshold, species_a, species_b, r_coord):
    """(max sqrt(V), #atoms with sqrt(V) > threshold, coordination numbers [N]) by brute force."""
    pos = _f64(pos).reshape(-1, 3)
    types = _i32(types)
    N = pos.shape[0]
    var = None if var is None else _f64(var)
    mx = C.c_double(0.0)
    na = C.c_int64(0)
    coord = np.zeros(N, dtype=np.int32)
    rc = lib().oracle_analyze(C.c_int64(N), _p(pos), _p(types), _p(_box9(box)), _p(_pbc3(pbc)), _p(var),
                              C.c_double(threshold), C.c_int(species_a), C.c_int(species_b), C.c_double(r_coord),
                              C.byref(mx), C.byref(na), _p(coord))
    _check(rc, "oracle_analyze")
    return mx.value, na.value, coord


def step_nvt(pos, vel, types, mass, box, pbc, n_max, l_max, r_cut, beta, dt, n_steps, T_target, tau, xi_eta=(0.0, 0.0),
             nbr_method: int = 1):
    """Nose-Hoover NVT.  Returns dict(pos, vel, E, F, xi, eta, cons[n_steps+1], temp[n_steps+1])."""
    pos = _f64(pos).reshape(-1, 3).copy()
    vel = _f64(vel).reshape(-1, 3).copy()
    types = _i32(types)
    mass = _f64(mass)
    N = pos.shape[0]
    S, r_cut, beta, _ = _model_args(n_max, l_max, r_cut, beta, None)
    E, F = np.zeros(N), np.zeros((N, 3))
    xe = _f64(np.array(xi_eta, dtype=np.float64))
    cons, temp = np.zeros(n_steps + 1), np.zeros(n_steps + 1)
    rc = lib().oracle_step_nvt(C.c_int64(N), _p(pos), _p(vel), _p(types), _p(mass), _p(_box9(box)), _p(_pbc3(pbc)),
                               C.c_int(S), C.c_int(n_max), C.c_int(l_max), _p(r_cut), _p(beta), None,
                               C.c_int(nbr_method), C.c_double(dt), C.c_int(n_steps), C.c_double(T_target),
                               C.c_double(tau), _p(xe), _p(E), _p(F), _p(cons), _p(temp))
    _check(rc, "oracle_step_nvt")
    return dict(pos=pos, vel=vel, E=E, F=F, xi=float(xe[0]), eta=float(xe[1]), cons=cons, temp=temp)
