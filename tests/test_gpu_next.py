"""GPU parity of the NEXT rows against the oracle, through the C ABI:
virial, on-the-fly analysis (maximum uncertainty, coordination numbers) and the Nose-Hoover thermostat."""
import numpy as np
import pytest

from paper_2204_12573_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch

    return torch


@pytest.fixture(scope="module")
def flare():
    from paper_2204_12573_b200 import flare as fl

    fl.load_library()
    return fl


def evaluated(torch, flare, s, **kw):
    ctx = flare.from_system(s, **kw).bind(s.n_atoms)
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    e, f, v = ctx.compute(pos, types, s.box, s.pbc, variances=True)
    torch.cuda.synchronize()
    return ctx, e.cpu().numpy(), f.cpu().numpy(), v.cpu().numpy()


@pytest.mark.parametrize("name", ["c1", "c2", "tile"])
def test_virial_matches_oracle(oracle, torch, flare, name):
    s = {"c1": w.config1, "c2": w.config2, "tile": lambda: w.tile_like_c3(10, 5, n_max=5, l_max=4)}[name]()
    ctx, _, _, _ = evaluated(torch, flare, s)
    Xi = ctx.virial()
    _, _, _, ref = oracle.compute_virial(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
    scale = np.abs(ref).max()
    assert scale > 1e-3
    # a sum over ~20 N pair terms: absolute tolerance relative to the largest component
    assert np.abs(Xi - ref).max() <= 1e-10 * scale
    assert np.abs(Xi - Xi.T).max() <= 1e-10 * scale
    # fixed summation order: bit-reproducible
    assert np.array_equal(Xi, ctx.virial())
    # dense and species-sparse evaluation give the same virial
    ctx_d, _, _, _ = evaluated(torch, flare, s, species_sparse=False)
    assert np.abs(ctx_d.virial() - ref).max() <= 1e-10 * scale


def test_analysis_matches_oracle(oracle, torch, flare):
    s = w.config2()
    ctx, _, _, v = evaluated(torch, flare, s)
    thr = float(np.sqrt(np.median(np.maximum(v, 0))))
    a = ctx.analyze(threshold=thr, species_a=1, species_b=1, r_coord=1.0)
    V_or = oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, forces=False)[2]
    mx, na, coord = oracle.analyze(s.pos, s.types, s.box, s.pbc, V_or, thr, 1, 1, 1.0)
    assert abs(a["max_unc"] - mx) <= 1e-10 * mx
    # the count is an integer decided in floating point: atoms within rounding of the threshold may differ
    near = int(np.sum(np.abs(np.sqrt(np.maximum(V_or, 0)) - thr) < 1e-10 * thr))
    assert abs(a["n_above"] - na) <= near
    assert np.array_equal(a["coord"].cpu().numpy(), coord)  # integer result: exact
    assert a["hist"][1] == 400 and a["hist"].sum() == 400   # every H of the synthetic gas has one H within 1 A
    # max over the GPU's own variances is exact
    assert a["max_unc"] == np.sqrt(max(v.max(), 0.0))
    # other species pairs and radii
    for sa, sb, r in ((1, 0, 2.9), (0, 0, 3.0), (0, 1, 3.0), (1, 1, 0.5)):
        g = ctx.analyze(species_a=sa, species_b=sb, r_coord=r, uncertainty=False)
        _, _, c = oracle.analyze(s.pos, s.types, s.box, s.pbc, None, 0.0, sa, sb, r)
        assert np.array_equal(g["coord"].cpu().numpy(), c)
        assert g["hist"].sum() == int(np.sum(s.types == sa))


def test_analysis_argument_errors(torch, flare):
    s = w.config2()
    ctx = flare.from_system(s).bind(s.n_atoms)
    with pytest.raises(flare.FlareError):
        ctx.analyze()  # nothing evaluated yet
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    ctx.compute(pos, types, s.box, s.pbc, variances=False)
    with pytest.raises(flare.FlareError):
        ctx.analyze(uncertainty=True, coordination=False)  # no variances in the last evaluation
    with pytest.raises(flare.FlareError):
        ctx.analyze(species_a=1, species_b=1, r_coord=3.5, uncertainty=False)  # beyond r_cut[H][H] = 3.0
    with pytest.raises(flare.FlareError):
        ctx.analyze(species_a=2, species_b=0, r_coord=1.0, uncertainty=False)
    assert ctx.analyze(species_a=1, species_b=1, r_coord=1.0, uncertainty=False)["hist"][1] == 400


def test_nvt_matches_oracle_trajectory(oracle, torch, flare):
    s = w.config1()
    ctx = flare.from_system(s).bind(s.n_atoms)
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    ctx.step_nvt(1.0, 8, 450.0, 20.0)
    st = ctx.get_state_host()
    xi, eta = ctx.thermostat()
    ref = oracle.step_nvt(s.pos, s.vel, s.types, s.mass, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, 1.0, 8,
                          450.0, 20.0)
    assert np.abs(st["pos"] - ref["pos"]).max() < 1e-10
    assert np.abs(st["vel"] - ref["vel"]).max() < 1e-12
    assert abs(xi - ref["xi"]) < 1e-12 * max(1.0, abs(ref["xi"])) and abs(xi) > 1e-6
    assert abs(eta - ref["eta"]) < 1e-12
    # continuing in two calls equals one call (the thermostat state persists on the device)
    ctx2 = flare.from_system(s).bind(s.n_atoms)
    ctx2.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    ctx2.step_nvt(1.0, 3, 450.0, 20.0)
    ctx2.step_nvt(1.0, 5, 450.0, 20.0)
    st2 = ctx2.get_state_host()
    assert np.array_equal(st2["pos"], st["pos"]) and np.array_equal(st2["vel"], st["vel"])
    assert ctx2.thermostat() == (xi, eta)


def test_nvt_conserved_quantity_and_set_thermostat(oracle, torch, flare):
    s = w.config2()
    ctx = flare.from_system(s).bind(s.n_atoms)
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    T, tau, dt = 450.0, 25.0, 0.5
    g = 3 * s.n_atoms - 3
    gkT = g * 8.617333262e-5 * T
    Q = gkT * tau * tau
    cons = []
    ctx.step(dt, 0)
    for _ in range(6):
        st = ctx.get_state_host()
        xi, eta = ctx.thermostat()
        cons.append(w.kinetic_energy(st["vel"], s.types, s.mass) + st["E"].sum() + 0.5 * Q * xi * xi + gkT * eta)
        ctx.step_nvt(dt, 10, T, tau)
    cons = np.array(cons)
    ke0 = w.kinetic_energy(s.vel, s.types, s.mass)
    assert np.abs(cons - cons[0]).max() < 2e-3 * ke0
    # time reversal through set_thermostat: flip v and xi, integrate back
    st = ctx.get_state_host()
    xi, eta = ctx.thermostat()
    ctx.set_state(st["pos"], -st["vel"], s.types, s.box, s.pbc)
    ctx.set_thermostat(-xi, eta)
    ctx.step_nvt(dt, 60, T, tau)  # the loop above made 6 x 10 steps
    back = ctx.get_state_host()
    L = np.asarray(s.box, float).reshape(3, 3).diagonal()
    d = back["pos"] - oracle.wrap(s.pos, s.box, s.pbc)
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-7
    with pytest.raises(flare.FlareError):
        ctx.step_nvt(dt, 1, -1.0, tau)
