"""Pins for the oracle's quadratic forms, forces, neighbour sets and integrator
(SURVEY.md 8(c)).  Expected values: numpy library routines, closed forms, finite differences
of the oracle's OWN energy (a different code path from its analytic gradient), symmetry
arguments and brute force.
"""
import numpy as np
import pytest

from paper_2204_12573_b200 import workloads as w


def small_fcc(rng, n_cells=3, jitter=0.08):
    pos, types, box, pbc = w.fcc_bulk(n_cells, w.A_PT, jitter, rng)
    return pos, types, box, pbc


def two_species_cluster(rng, n=40, L=60.0):
    """A compact random two-species cluster in a big NON-periodic box (isolated)."""
    pos = rng.uniform(-3.2, 3.2, (n, 3))
    # thin out pairs that are too close
    keep = []
    for i in range(n):
        if all(np.linalg.norm(pos[i] - pos[j]) > 0.9 for j in keep):
            keep.append(i)
    pos = pos[keep] + L / 2
    types = rng.integers(0, 2, len(keep)).astype(np.int32)
    return pos, types, np.diag([L, L, L]).reshape(9), np.zeros(3, np.int32)


R2 = np.array([[4.25, 3.0], [3.0, 3.0]])


# ----------------------------------------------------------------------------- E and V


def test_energy_and_variance_vs_numpy(oracle):
    rng = np.random.default_rng(0)
    pos, types, box, pbc = two_species_cluster(rng)
    n_max, l_max, S = 3, 2, 2
    P = oracle.num_descriptors(S, n_max, l_max)
    beta = rng.standard_normal((S, P, P))  # deliberately NOT symmetric: x^T beta x only sees the symmetric part
    sigma = w.random_sigma(rng, S, P)
    E, F, V = oracle.compute(pos, types, box, pbc, n_max, l_max, R2, beta, sigma, nbr_method=0)
    for i in range(len(types)):
        _, _, Bh, nrm = oracle.descriptor(pos, types, box, pbc, n_max, l_max, R2, i)
        if nrm == 0:
            assert E[i] == 0 and V[i] == 0
            continue
        assert abs(E[i] - Bh @ beta[types[i]] @ Bh) < 1e-13 * max(1, abs(E[i]))
        assert abs(V[i] - Bh @ sigma[types[i]] @ Bh) < 1e-15
    # symmetrising beta changes neither energies nor forces (R10)
    bs = 0.5 * (beta + beta.transpose(0, 2, 1))
    E2, F2, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, R2, bs, sigma, nbr_method=0)
    np.testing.assert_allclose(E2, E, atol=1e-13)
    np.testing.assert_allclose(F2, F, atol=1e-12)


def test_special_matrices(oracle):
    rng = np.random.default_rng(1)
    pos, types, box, pbc = small_fcc(rng)
    n_max, l_max = 4, 3
    P = oracle.num_descriptors(1, n_max, l_max)
    eye = np.eye(P)[None]
    E, F, V = oracle.compute(pos, types, box, pbc, n_max, l_max, w.R_CUT_1, eye, 0.37 * eye)
    np.testing.assert_allclose(E, 1.0, atol=1e-14)  # beta = I  => E_i = |B^|^2 = 1
    np.testing.assert_allclose(V, 0.37, atol=1e-14)  # Sigma = cI => V_i = c
    np.testing.assert_allclose(F, 0.0, atol=1e-12)  # constant energy => no force: tests d nrm/dr (R11)
    u = rng.standard_normal(P)
    E, _, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, w.R_CUT_1, np.outer(u, u)[None], None)
    for i in (0, 5, 50):
        _, _, Bh, _ = oracle.descriptor(pos, types, box, pbc, n_max, l_max, w.R_CUT_1, i)
        assert abs(E[i] - (u @ Bh) ** 2) < 1e-12


def test_species_subblock_energy(oracle):
    """An atom with same-species neighbours only: E from the full S=2 beta equals E from its
    single-species sub-block on the compacted descriptor (correctness statement of P:L155)."""
    rng = np.random.default_rng(2)
    pos, types, box, pbc = small_fcc(rng)  # all species 0
    n_max, l_max = 4, 2
    P2, P1 = oracle.num_descriptors(2, n_max, l_max), oracle.num_descriptors(1, n_max, l_max)
    beta2 = w.random_beta(rng, 2, P2)
    keep = [oracle.b2_index(2, n_max, l_max, v1, v2, l) for v1 in range(n_max) for v2 in range(v1, n_max)
            for l in range(l_max + 1)]
    assert len(keep) == P1
    beta1 = beta2[0][np.ix_(keep, keep)][None]
    E2, F2, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, np.array([[4.25, 3.0], [3.0, 3.0]]), beta2)
    E1, F1, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, w.R_CUT_1, beta1)
    np.testing.assert_allclose(E2, E1, atol=1e-14)
    np.testing.assert_allclose(F2, F1, atol=1e-13)


def test_isolated_atom_and_empty_system(oracle):
    P = oracle.num_descriptors(1, 3, 2)
    beta = np.eye(P)[None]
    box = np.diag([30.0, 30, 30]).reshape(9)
    pos = np.array([[5.0, 5, 5], [20.0, 20, 20], [21.0, 20, 20]])
    E, F, V = oracle.compute(pos, np.zeros(3, np.int32), box, [1, 1, 1], 3, 2, w.R_CUT_1, beta, beta)
    assert E[0] == 0 and V[0] == 0 and np.all(F[0] == 0)  # R8
    assert E[1] == pytest.approx(1.0) and E[2] == pytest.approx(1.0)
    E, F, V = oracle.compute(np.zeros((0, 3)), np.zeros(0, np.int32), box, [1, 1, 1], 3, 2, w.R_CUT_1, beta, beta)
    assert E.size == 0 and F.size == 0


# ----------------------------------------------------------------------------- forces


def _fd_force(oracle, pos, types, box, pbc, n_max, l_max, r_cut, beta, k, d, h):
    def etot(x):
        E, _, _ = oracle.compute(x, types, box, pbc, n_max, l_max, r_cut, beta, None, nbr_method=0, forces=False)
        return E.sum()

    def diff(hh):
        xp, xm = pos.copy(), pos.copy()
        xp[k, d] += hh
        xm[k, d] -= hh
        return -(etot(xp) - etot(xm)) / (2 * hh)

    return (4 * diff(h / 2) - diff(h)) / 3  # Richardson


@pytest.mark.parametrize("case", ["fcc_1sp", "cluster_2sp", "slab_2sp"])
def test_forces_vs_finite_differences(oracle, case):
    rng = np.random.default_rng(3)
    if case == "fcc_1sp":
        pos, types, box, pbc = small_fcc(rng)
        n_max, l_max, r_cut, S = 5, 3, w.R_CUT_1, 1
    elif case == "cluster_2sp":
        pos, types, box, pbc = two_species_cluster(rng)
        n_max, l_max, r_cut, S = 3, 4, R2, 2
    else:
        pos, types, box, pbc = w.h2_pt111(4, 2, 6, rng, rng, n_layers=3)
        n_max, l_max, r_cut, S = 3, 2, R2, 2
    P = oracle.num_descriptors(S, n_max, l_max)
    beta = w.random_beta(rng, S, P)
    _, F, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, r_cut, beta, None, nbr_method=0)
    scale = np.abs(F).max()
    assert scale > 1e-3
    atoms = rng.choice(len(types), 4, replace=False)
    if case == "slab_2sp":
        atoms = np.concatenate([atoms[:2], [len(types) - 1, len(types) - 4]])  # make sure H atoms are probed
    for k in atoms:
        for d in range(3):
            fd = _fd_force(oracle, pos, types, box, pbc, n_max, l_max, r_cut, beta, k, d, 2e-3)
            assert abs(F[k, d] - fd) < 2e-8 * scale, (case, k, d, F[k, d], fd)


def test_zero_net_force_and_torque(oracle):
    rng = np.random.default_rng(4)
    pos, types, box, pbc = two_species_cluster(rng)
    n_max, l_max = 4, 3
    beta = w.random_beta(rng, 2, oracle.num_descriptors(2, n_max, l_max))
    _, F, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, R2, beta, None, nbr_method=0)
    scale = np.abs(F).max()
    assert np.abs(F.sum(0)).max() < 1e-13 * max(1, scale) * len(types)  # translation invariance
    torque = np.cross(pos - pos.mean(0), F).sum(0)  # rotation invariance (isolated cluster)
    assert np.abs(torque).max() < 1e-11 * max(1, scale) * len(types)
    # periodic slab: net force still vanishes
    s = w.tile_like_c3(6, 3, n_max=3, l_max=2)
    _, F, _ = oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta)
    assert np.abs(F.sum(0)).max() < 1e-12 * len(s.types)


def test_perfect_fcc_has_zero_force_and_identical_descriptors(oracle):
    """Inversion symmetry of every site of an un-jittered fcc lattice => F = 0 for ANY beta."""
    pos, types, box, pbc = w.fcc_bulk(3, w.A_PT, 0.0, None)
    n_max, l_max = 6, 3
    rng = np.random.default_rng(5)
    beta = w.random_beta(rng, 1, oracle.num_descriptors(1, n_max, l_max))
    E, F, _ = oracle.compute(pos, types, box, pbc, n_max, l_max, w.R_CUT_1, beta)
    assert np.abs(F).max() < 1e-12
    assert np.ptp(E) < 1e-13
    cnt, _ = oracle.neighbors(pos, types, box, pbc, w.R_CUT_1, 0)
    assert np.all(cnt == 18)  # shells at a/sqrt2 (12) and a (6); next shell 4.80 A is outside 4.25


def test_compute_selected_matches_full(oracle):
    s = w.tile_like_c3(6, 3, n_max=3, l_max=2)
    E, F, V = oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
    sel = np.array([0, 7, 100, s.n_atoms - 1, s.n_atoms - 2, 55])
    Es, Fs, Vs = oracle.compute_selected(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, sel)
    np.testing.assert_allclose(Es, E[sel], atol=1e-15)
    np.testing.assert_allclose(Vs, V[sel], atol=1e-17)
    np.testing.assert_allclose(Fs, F[sel], atol=1e-13)


# ----------------------------------------------------------------------------- neighbour sets


def _brute_numpy(pos, types, box, pbc, r_cut):
    """Independent O(N^2) brute force in numpy with the canonical arithmetic of R6."""
    L = np.asarray(box).reshape(3, 3).diagonal()
    x = pos.copy()
    for d in range(3):
        if pbc[d]:
            x[:, d] = x[:, d] - L[d] * np.floor(x[:, d] / L[d])
            x[x[:, d] >= L[d], d] = 0.0
    out = []
    for i in range(len(x)):
        dx = x - x[i]
        for d in range(3):
            if pbc[d]:
                col = dx[:, d]
                col = np.where(col > 0.5 * L[d], col - L[d], np.where(col < -0.5 * L[d], col + L[d], col))
                dx[:, d] = col
        d2 = (dx[:, 0] * dx[:, 0] + dx[:, 1] * dx[:, 1]) + dx[:, 2] * dx[:, 2]
        rc = np.asarray(r_cut)[types[i], types]
        m = d2 < rc * rc
        m[i] = False
        out.append(np.nonzero(m)[0])
    return out


@pytest.mark.parametrize("case", ["C1", "C2", "gas_open"])
def test_neighbour_sets_vs_brute_force(oracle, case):
    if case == "C1":
        s = w.config1(with_model=False)
        pos, types, box, pbc, r_cut = s.pos, s.types, s.box, s.pbc, s.r_cut
    elif case == "C2":
        s = w.config2(with_model=False)
        pos, types, box, pbc, r_cut = s.pos, s.types, s.box, s.pbc, s.r_cut
    else:
        rng = np.random.default_rng(6)
        pos = rng.uniform(0, 25, (400, 3))
        types = rng.integers(0, 2, 400).astype(np.int32)
        box, pbc, r_cut = np.diag([25.0, 25, 25]).reshape(9), np.array([1, 0, 1], np.int32), R2
    want = _brute_numpy(pos, types, box, pbc, r_cut)
    for method in (0, 1):
        cnt, idx = oracle.neighbors(pos, types, box, pbc, r_cut, method)
        assert [len(r) for r in want] == cnt.tolist()
        for i, r in enumerate(want):
            assert np.array_equal(idx[i, : cnt[i]], r)
    # symmetric: i in N(j) <=> j in N(i)
    pairs = {(i, j) for i in range(len(want)) for j in want[i]}
    assert all((j, i) in pairs for (i, j) in pairs)


def test_box_checks(oracle):
    pos = np.zeros((2, 3))
    t = np.zeros(2, np.int32)
    with pytest.raises(oracle.OracleError):  # periodic length < 2 r_cut (R7)
        oracle.neighbors(pos, t, np.diag([8.0, 20, 20]).reshape(9), [1, 1, 1], w.R_CUT_1)
    tri = np.diag([20.0, 20, 20])
    tri[1, 0] = 1.0
    with pytest.raises(oracle.OracleError):  # triclinic unsupported (R7)
        oracle.neighbors(pos, t, tri.reshape(9), [1, 1, 1], w.R_CUT_1)
    with pytest.raises(oracle.OracleError):  # asymmetric cutoffs (R5)
        oracle.neighbors(pos, t, np.diag([20.0, 20, 20]).reshape(9), [1, 1, 1], [[4.0, 3.0], [2.0, 3.0]])


# ----------------------------------------------------------------------------- integrator


def _md_case(oracle):
    rng = np.random.default_rng(7)
    pos, types, box, pbc = small_fcc(rng, 3, 0.05)
    n_max, l_max = 3, 2
    beta = w.random_beta(rng, 1, oracle.num_descriptors(1, n_max, l_max), e0=2.0)
    mass = np.array([w.MASS_PT])
    vel = w.maxwell_velocities(rng, types, mass, 300.0)
    return pos, vel, types, mass, box, pbc, n_max, l_max, beta


def test_nve_energy_drift_scales_as_dt_squared(oracle):
    pos, vel, types, mass, box, pbc, n_max, l_max, beta = _md_case(oracle)
    fl = []
    for dt, n in ((4.0, 20), (2.0, 40)):
        r = oracle.step(pos, vel, types, mass, box, pbc, n_max, l_max, w.R_CUT_1, beta, None, dt, n)
        h = r["pe"] + r["ke"]
        fl.append(np.abs(h - h[0]).max())
        assert abs(r["ke"][0] - w.kinetic_energy(vel, types, mass)) < 1e-12
    assert fl[0] < 5e-3 * abs(r["ke"][0])  # conserved to a small fraction of KE
    assert 2.5 < fl[0] / fl[1] < 6.0  # halve dt => fluctuation / ~4


def test_time_reversal_and_momentum(oracle):
    pos, vel, types, mass, box, pbc, n_max, l_max, beta = _md_case(oracle)
    r = oracle.step(pos, vel, types, mass, box, pbc, n_max, l_max, w.R_CUT_1, beta, None, 1.0, 15)
    m = mass[types][:, None]
    assert np.abs((m * r["vel"]).sum(0) - (m * vel).sum(0)).max() < 1e-13
    back = oracle.step(r["pos"], -r["vel"], types, mass, box, pbc, n_max, l_max, w.R_CUT_1, beta, None, 1.0, 15)
    L = np.asarray(box).reshape(3, 3).diagonal()
    d = back["pos"] - oracle.wrap(pos, box, pbc)
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    np.testing.assert_allclose(-back["vel"], vel, atol=1e-12)
