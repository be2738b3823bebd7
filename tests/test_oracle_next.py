"""Pins for the oracle's NEXT-row functions: virial / stress, on-the-fly
analysis (maximum uncertainty, H coordination numbers) and the Nose-Hoover thermostat.
Expected values come from finite differences of the oracle's own total energy under strain,
symmetry arguments, the construction of the synthetic H2 gas, numpy, and the NVE integrator."""
import numpy as np

from paper_2204_12573_b200 import workloads as w

R2 = np.array([[4.25, 3.0], [3.0, 3.0]])


def _model(rng, S, n_max, l_max, oracle):
    P = oracle.num_descriptors(S, n_max, l_max)
    return w.random_beta(rng, S, P), w.random_sigma(rng, S, P)


# ----------------------------------------------------------------------------- virial


def test_virial_diagonal_vs_strain_finite_differences(oracle):
    """Xi_aa = dE/d eps_aa: scale box length and coordinates along a by (1 + eps) and difference the energy."""
    rng = np.random.default_rng(11)
    pos, types, box, pbc = w.fcc_bulk(3, w.A_PT, 0.08, rng)
    n_max, l_max = 4, 2
    beta, _ = _model(rng, 1, n_max, l_max, oracle)
    rc = np.array([[4.25]])
    _, _, _, Xi = oracle.compute_virial(pos, types, box, pbc, n_max, l_max, rc, beta)
    B = np.asarray(box, float).reshape(3, 3)

    def energy(a, eps):
        sc = np.ones(3)
        sc[a] += eps
        E, _, _ = oracle.compute(pos * sc, types, (B * sc).reshape(9), pbc, n_max, l_max, rc, beta, forces=False)
        return E.sum()

    for a in range(3):
        h = 1e-4
        d1 = (energy(a, h) - energy(a, -h)) / (2 * h)
        d2 = (energy(a, h / 2) - energy(a, -h / 2)) / h
        fd = (4 * d2 - d1) / 3  # Richardson
        assert abs(Xi[a, a] - fd) < 1e-7 * max(1.0, abs(fd))


def test_virial_symmetric_and_rotation_covariant(oracle):
    rng = np.random.default_rng(12)
    n = 30
    x = rng.uniform(-3.0, 3.0, (n, 3))
    types = rng.integers(0, 2, n).astype(np.int32)
    L = 60.0
    box, pbc = np.diag([L, L, L]).reshape(9), np.zeros(3, np.int32)
    n_max, l_max = 3, 3
    beta, _ = _model(rng, 2, n_max, l_max, oracle)
    _, _, _, Xi = oracle.compute_virial(x + L / 2, types, box, pbc, n_max, l_max, R2, beta)
    assert np.abs(Xi).max() > 1e-3
    np.testing.assert_allclose(Xi, Xi.T, atol=1e-11)  # E is rotation invariant => no torque => symmetric
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    _, _, _, Xr = oracle.compute_virial(x @ q.T + L / 2, types, box, pbc, n_max, l_max, R2, beta)
    np.testing.assert_allclose(Xr, q @ Xi @ q.T, atol=1e-10)


def test_virial_vanishes_for_identity_beta_and_matches_pair_sum(oracle):
    rng = np.random.default_rng(13)
    pos, types, box, pbc = w.fcc_bulk(3, w.A_PT, 0.08, rng)
    n_max, l_max = 3, 2
    P = oracle.num_descriptors(1, n_max, l_max)
    rc = np.array([[4.25]])
    # beta = I => E_i = 1 whatever the geometry => every derivative vanishes
    _, _, _, Xi = oracle.compute_virial(pos, types, box, pbc, n_max, l_max, rc, np.eye(P)[None])
    assert np.abs(Xi).max() < 1e-12
    # trace = dE/d lambda under uniform scaling
    beta = w.random_beta(rng, 1, P)
    _, _, _, Xi = oracle.compute_virial(pos, types, box, pbc, n_max, l_max, rc, beta)
    B = np.asarray(box, float).reshape(3, 3)
    h = 1e-5
    e = [oracle.compute(pos * (1 + s), types, (B * (1 + s)).reshape(9), pbc, n_max, l_max, rc, beta,
                        forces=False)[0].sum() for s in (h, -h)]
    assert abs(np.trace(Xi) - (e[0] - e[1]) / (2 * h)) < 1e-6 * max(1.0, abs(np.trace(Xi)))


# ----------------------------------------------------------------------------- analysis


def test_h_coordination_of_the_synthetic_gas(oracle):
    """Every H of config 2 has exactly one H within 1 A: its bond partner at 0.74 A (the generator keeps H atoms
    of different molecules at least 1.0 A apart); Pt atoms get 0."""
    s = w.config2()
    var = np.linspace(-1e-4, 4e-4, s.n_atoms)
    mx, na, coord = oracle.analyze(s.pos, s.types, s.box, s.pbc, var, 0.015, 1, 1, 1.0)
    assert np.all(coord[s.types == 1] == 1) and np.all(coord[s.types == 0] == 0)
    assert mx == np.sqrt(var.max())
    assert na == int(np.sum(np.sqrt(np.maximum(var, 0)) > 0.015))
    # a shorter radius than the bond finds nothing
    _, _, c0 = oracle.analyze(s.pos, s.types, s.box, s.pbc, None, 0.0, 1, 1, 0.7)
    assert not c0.any()


def test_coordination_across_the_periodic_boundary(oracle):
    L = 12.0
    pos = np.array([[0.1, 5.0, 5.0], [L - 0.3, 5.0, 5.0], [6.0, 5.0, 5.0], [6.0, 5.9, 5.0], [6.0, 5.0, 5.95]])
    types = np.array([1, 1, 1, 1, 0], np.int32)
    box = np.diag([L, L, L]).reshape(9)
    _, _, c = oracle.analyze(pos, types, box, np.ones(3, np.int32), None, 0.0, 1, 1, 1.0)
    assert c.tolist() == [1, 1, 1, 1, 0]
    _, _, c = oracle.analyze(pos, types, box, np.zeros(3, np.int32), None, 0.0, 1, 1, 1.0)
    assert c.tolist() == [0, 0, 1, 1, 0]  # open boundaries: no image
    _, _, c = oracle.analyze(pos, types, box, np.ones(3, np.int32), None, 0.0, 1, 0, 1.0)
    assert c.tolist() == [0, 0, 1, 0, 0]  # H -> Pt coordination: only atom 2 has the Pt within 1 A


# ----------------------------------------------------------------------------- Nose-Hoover


def _c1_small(oracle):
    rng = np.random.default_rng(21)
    pos, types, box, pbc = w.fcc_bulk(2, w.A_PT, 0.05, rng)  # 32 atoms, L = 7.84 < 2 r_cut: use r_cut 3.5
    n_max, l_max = 3, 2
    P = oracle.num_descriptors(1, n_max, l_max)
    beta = w.random_beta(rng, 1, P)
    mass = np.array([w.MASS_PT])
    vel = w.maxwell_velocities(rng, types, mass, 300.0)
    return pos, vel, types, mass, box, pbc, n_max, l_max, np.array([[3.5]]), beta


def test_nvt_reduces_to_nve_for_infinite_thermostat_mass(oracle):
    a = _c1_small(oracle)
    pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta = a
    nve = oracle.step(pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta, None, 1.0, 8)
    nvt = oracle.step_nvt(pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta, 1.0, 8, 300.0, 1e9)
    np.testing.assert_allclose(nvt["pos"], nve["pos"], atol=1e-12)
    np.testing.assert_allclose(nvt["vel"], nve["vel"], atol=1e-13)
    assert abs(nvt["xi"]) < 1e-12


def test_nvt_conserved_quantity_scales_as_dt_squared(oracle):
    pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta = _c1_small(oracle)
    spread = []
    for dt, n in ((2.0, 20), (1.0, 40)):
        r = oracle.step_nvt(pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta, dt, n, 450.0, 25.0)
        c = r["cons"]
        assert np.abs(c - c[0]).max() < 1e-3 * abs(r["temp"][0] * 8.617333262e-5 * 3 * len(types) / 2)
        spread.append(np.abs(c - c[0]).max())
        assert abs(r["xi"]) > 1e-6  # the thermostat is really acting
    assert spread[1] < 0.45 * spread[0]


def test_nvt_is_time_reversible_and_heats_towards_the_target(oracle):
    pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta = _c1_small(oracle)
    f = oracle.step_nvt(pos, vel, types, mass, box, pbc, n_max, l_max, rc, beta, 1.0, 12, 900.0, 15.0)
    b = oracle.step_nvt(f["pos"], -f["vel"], types, mass, box, pbc, n_max, l_max, rc, beta, 1.0, 12, 900.0, 15.0,
                        xi_eta=(-f["xi"], f["eta"]))
    d = b["pos"] - oracle.wrap(pos, box, pbc)
    L = np.asarray(box, float).reshape(3, 3).diagonal()
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    np.testing.assert_allclose(-b["vel"], vel, atol=1e-10)
    # target 900 K from 300 K with a short time constant: xi < 0 pumps kinetic energy in
    assert f["xi"] < 0 and f["temp"][-1] > f["temp"][0]
    # zero total momentum is preserved by the uniform scaling
    p = (f["vel"] * mass[types][:, None]).sum(0)
    assert np.abs(p).max() < 1e-10
