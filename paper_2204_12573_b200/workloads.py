"""Seeded synthetic inputs shaped like the paper's workloads.

This module holds NO arithmetic of the method (no basis functions, no descriptors, no
forces): only geometry, random draws and unit constants.  It serves both the CUDA path
(tests, bench.py) and the oracle's tests, and imports neither.

The paper's workload is H2 gas over a Pt(111) slab; its structure files and
trained beta/gamma are not available, so these generators stand in for them: a thin
fcc(111) metal slab, a sparse diatomic gas above it, two species with very different
neighbour counts, and seeded random symmetric beta / PSD Sigma.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

ROOT_SEED = 220412573
KAPPA = 9.648533212331e-3  # (eV/amu) in Angstrom^2/fs^2
KB = 8.617333262e-5  # eV/K
MASS_PT = 195.084
MASS_H = 1.008
A_PT = 3.92  # Angstrom, fcc lattice constant of BASELINE.json's configs

STREAMS = ("jitter", "h2", "velocities", "beta", "sigma")


def streams(config_index: int) -> dict:
    """Child generators [jitter, h2, velocities, beta, sigma] of config c (1-based)."""
    root = np.random.SeedSequence(ROOT_SEED)
    child = root.spawn(5)[config_index - 1].spawn(5)
    return {name: np.random.Generator(np.random.PCG64(s)) for name, s in zip(STREAMS, child)}


def num_descriptors(S: int, n_max: int, l_max: int) -> int:
    nv = S * n_max
    return nv * (nv + 1) // 2 * (l_max + 1)


@dataclass
class System:
    name: str
    pos: np.ndarray  # [N,3] f64 Angstrom
    types: np.ndarray  # [N] i32
    box: np.ndarray  # [9] f64 row-major cell vectors (orthorhombic)
    pbc: np.ndarray  # [3] i32
    mass: np.ndarray  # [S] amu
    r_cut: np.ndarray  # [S,S]
    n_max: int
    l_max: int
    vel: np.ndarray | None = None  # [N,3] Angstrom/fs
    beta: np.ndarray | None = None  # [S,P,P]
    sigma: np.ndarray | None = None  # [S,P,P]
    meta: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_species(self) -> int:
        return int(self.mass.shape[0])

    @property
    def P(self) -> int:
        return num_descriptors(self.n_species, self.n_max, self.l_max)


# ----------------------------------------------------------------------------- model matrices


def random_beta(rng, S: int, P: int, e0: float = 1.0) -> np.ndarray:
    """beta^(s) = e0 (G+G^T)/(2 sqrt(2P)), G_ij ~ N(0,1): symmetric, spectral norm ~ e0."""
    out = np.empty((S, P, P))
    for s in range(S):
        g = rng.standard_normal((P, P))
        out[s] = e0 * (g + g.T) / (2.0 * np.sqrt(2.0 * P))
    return out


def random_sigma(rng, S: int, P: int, scale: float = 1e-3) -> np.ndarray:
    """Sigma^(s) = scale G G^T / P: symmetric positive semi-definite."""
    out = np.empty((S, P, P))
    for s in range(S):
        g = rng.standard_normal((P, P))
        out[s] = scale * (g @ g.T) / P
    return out


def maxwell_velocities(rng, types, mass, temperature: float) -> np.ndarray:
    """N(0, kB T kappa / m) per component, COM velocity removed, rescaled to exactly T (3N-3 dof)."""
    m = np.asarray(mass)[np.asarray(types)]
    n = m.shape[0]
    v = rng.standard_normal((n, 3)) * np.sqrt(KB * temperature * KAPPA / m)[:, None]
    if n > 1:
        v -= (m[:, None] * v).sum(0) / m.sum()
        ke = 0.5 * (m[:, None] * v * v).sum() / KAPPA
        t_now = 2.0 * ke / ((3 * n - 3) * KB)
        if t_now > 0:
            v *= np.sqrt(temperature / t_now)
    return v


def kinetic_energy(vel, types, mass) -> float:
    m = np.asarray(mass)[np.asarray(types)]
    return float(0.5 * (m[:, None] * vel * vel).sum() / KAPPA)


# ----------------------------------------------------------------------------- geometry


def fcc_bulk(n_cells: int = 4, a: float = A_PT, jitter: float = 0.05, rng=None):
    """fcc conventional cells, periodic; optional seeded Gaussian jitter; wrapped into the box."""
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    g = np.arange(n_cells)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    pos = (cells[:, None, :] + basis[None, :, :]).reshape(-1, 3) * a
    L = n_cells * a
    if jitter and rng is not None:
        pos = pos + rng.normal(0.0, jitter, pos.shape)
    pos = pos - L * np.floor(pos / L)
    pos[pos >= L] = 0.0
    box = np.diag([L, L, L]).reshape(9)
    return pos, np.zeros(pos.shape[0], np.int32), box, np.ones(3, np.int32)


def pt111_slab(nx: int, ny: int, n_layers: int = 6, a: float = A_PT, gap: float = 20.0):
    """Pt(111) slab in an orthorhombic cell: ax = a/sqrt2, ay = sqrt3 ax, layer spacing a/sqrt3,
    two atoms per rectangular cell per layer, layer k shifted by (0, k ay/3) (ABC stacking),
    bottom layer at z = 0, `gap` Angstrom of vacuum above the top layer."""
    ax = a / np.sqrt(2.0)
    ay = np.sqrt(3.0) * ax
    dz = a / np.sqrt(3.0)
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")
    base = np.stack([ix.ravel() * ax, iy.ravel() * ay], -1)
    xy = np.concatenate([base, base + np.array([0.5 * ax, 0.5 * ay])], 0)
    layers = []
    for k in range(n_layers):
        p = np.empty((xy.shape[0], 3))
        p[:, 0] = xy[:, 0]
        p[:, 1] = np.mod(xy[:, 1] + k * ay / 3.0, ny * ay)
        p[:, 2] = k * dz
        layers.append(p)
    pos = np.concatenate(layers, 0)
    L = np.array([nx * ax, ny * ay, (n_layers - 1) * dz + gap])
    return pos, L, (n_layers - 1) * dz


def place_h2(rng, n_mol: int, L, z_lo: float, z_hi: float, bond: float = 0.74, min_sep: float = 1.0):
    """n_mol H2 molecules: centre uniform in x,y and z in [z_lo,z_hi], axis uniform on the sphere,
    atoms at centre +- bond/2.  Molecules with an H closer than min_sep to an H of a LOWER-index
    molecule are redrawn (all at once, repeated until none remain)."""
    from scipy.spatial import cKDTree

    def draw(k):
        c = np.empty((k, 3))
        c[:, 0] = rng.uniform(0.0, L[0], k)
        c[:, 1] = rng.uniform(0.0, L[1], k)
        c[:, 2] = rng.uniform(z_lo, z_hi, k)
        ax = rng.standard_normal((k, 3))
        ax /= np.linalg.norm(ax, axis=1)[:, None]
        return c, ax

    centre, axis = draw(n_mol)
    for _ in range(200):
        h = np.concatenate([centre + 0.5 * bond * axis, centre - 0.5 * bond * axis], 0)
        hw = np.mod(h, L)
        hw[hw >= L] = 0.0
        tree = cKDTree(hw, boxsize=L)
        pairs = tree.query_pairs(min_sep, output_type="ndarray")
        if pairs.size == 0:
            break
        mol = pairs % n_mol
        other = mol[:, 0] != mol[:, 1]
        bad = np.unique(np.max(mol[other], axis=1)) if other.any() else np.empty(0, int)
        if bad.size == 0:
            break
        c2, a2 = draw(bad.size)
        centre[bad] = c2
        axis[bad] = a2
    else:  # pragma: no cover
        raise RuntimeError("H2 placement did not converge")
    # interleave so that the two atoms of molecule k are adjacent: 2k, 2k+1
    h = np.empty((2 * n_mol, 3))
    h[0::2] = centre + 0.5 * bond * axis
    h[1::2] = centre - 0.5 * bond * axis
    return h


def h2_pt111(nx: int, ny: int, n_h2: int, rng_jitter=None, rng_h2=None, jitter: float = 0.05, n_layers: int = 6):
    """The H2/Pt(111)-shaped system: species 0 = Pt, 1 = H; periodic in x, y, z."""
    slab, L, z_top = pt111_slab(nx, ny, n_layers)
    if rng_jitter is not None and jitter:
        slab = slab + rng_jitter.normal(0.0, jitter, slab.shape)
    h = place_h2(rng_h2, n_h2, L, z_top + 2.0, z_top + 18.0) if n_h2 > 0 else np.empty((0, 3))
    pos = np.concatenate([slab, h], 0)
    pos = pos - L * np.floor(pos / L)
    pos[pos >= L] = 0.0
    types = np.concatenate([np.zeros(slab.shape[0], np.int32), np.ones(h.shape[0], np.int32)])
    return pos, types, np.diag(L).reshape(9), np.ones(3, np.int32)


# ----------------------------------------------------------------------------- BASELINE.json configs

R_CUT_1 = np.array([[4.25]])
R_CUT_2 = np.array([[4.25, 3.0], [3.0, 3.0]])  # "4.25 (Pt-Pt) and 3.0 (H pairs)": every pair with an H


def _finish(name, c, pos, types, box, pbc, mass, r_cut, n_max, l_max, temperature, with_model, meta):
    st = streams(c)
    S = mass.shape[0]
    sysm = System(name, pos, types, box, pbc, mass, r_cut, n_max, l_max, meta=meta)
    sysm.vel = maxwell_velocities(st["velocities"], types, mass, temperature)
    if with_model:
        P = num_descriptors(S, n_max, l_max)
        sysm.beta = random_beta(st["beta"], S, P)
        sysm.sigma = random_sigma(st["sigma"], S, P)
    return sysm


def config1(with_model: bool = True) -> System:
    """C1: fcc Pt 4x4x4 (256 atoms), jitter 0.05 A, n_max 8, l_max 3, r_cut 4.25, P=144; 300 K, dt 1 fs."""
    st = streams(1)
    pos, types, box, pbc = fcc_bulk(4, A_PT, 0.05, st["jitter"])
    return _finish("C1_fcc_Pt_256", 1, pos, types, box, pbc, np.array([MASS_PT]), R_CUT_1, 8, 3, 300.0, with_model,
                   dict(dt_fs=1.0, n_steps=10, temperature=300.0))


def h2_pt111_config(c: int, nx: int, ny: int, n_h2: int, n_max: int = 8, l_max: int = 3, temperature: float = 500.0,
                    with_model: bool = True, name: str | None = None) -> System:
    st = streams(c)
    pos, types, box, pbc = h2_pt111(nx, ny, n_h2, st["jitter"], st["h2"])
    return _finish(name or f"C{c}_H2_Pt111_{pos.shape[0]}", c, pos, types, box, pbc, np.array([MASS_PT, MASS_H]),
                   R_CUT_2, n_max, l_max, temperature, with_model,
                   dict(dt_fs=0.5, temperature=temperature, nx=nx, ny=ny, n_h2=n_h2))


def config2(with_model: bool = True) -> System:
    """C2: 12x6 rectangular (= 12x12 primitive) cells x 6 layers = 864 Pt + 200 H2 = 1264 atoms; P=544."""
    s = h2_pt111_config(2, 12, 6, 200, with_model=with_model)
    s.meta["n_steps"] = 100
    return s


def config3(with_model: bool = True, n_max: int = 8, l_max: int = 3) -> System:
    """C3: 408x204 rectangular cells x 6 layers = 998 784 Pt + 41 616 H2 = 1 082 016 atoms."""
    s = h2_pt111_config(3, 408, 204, 41616, n_max, l_max, with_model=with_model)
    s.meta["n_steps"] = 100
    return s


def config4(with_model: bool = True) -> System:
    """C4: 1240x620 rectangular cells, 384 400 H2: 9 994 400 atoms."""
    s = h2_pt111_config(4, 1240, 620, 384400, with_model=with_model)
    s.meta["n_steps"] = 50
    return s


def config5(n_max: int, l_max: int, with_model: bool = True) -> System:
    """C5: C3's geometry (same streams as config 5) with (n_max,l_max) in {(8,3),(10,4),(12,6)}."""
    s = h2_pt111_config(5, 408, 204, 41616, n_max, l_max, with_model=with_model,
                        name=f"C5_H2_Pt111_n{n_max}_l{l_max}")
    s.meta["n_steps"] = 50
    return s


def tile_like_c3(nx: int, ny: int, c: int = 3, n_max: int = 8, l_max: int = 3, with_model: bool = True) -> System:
    """A smaller tile of the C3 construction (0.25 H2 per surface Pt) for parity tests."""
    n_h2 = (2 * nx * ny) // 4
    return h2_pt111_config(c, nx, ny, n_h2, n_max, l_max, with_model=with_model, name=f"tile_{nx}x{ny}")
