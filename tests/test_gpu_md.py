"""GPU molecular dynamics (step a9) against the oracle: trajectories are chaotic, so parity is by
RE-SYNC (feed the GPU's positions to the oracle and compare E, F, V there) plus short-run agreement,
conserved-quantity traces and time reversal."""
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


def start(torch, flare, s, **kw):
    ctx = flare.from_system(s, **kw).bind(s.n_atoms)
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)  # host arrays -> flare_set_state_host
    return ctx


def total_energy(st, s):
    ke = w.kinetic_energy(st["vel"], s.types, s.mass)
    return ke + st["E"].sum(), ke


def test_config1_ten_steps_match_oracle_trajectory(oracle, torch, flare):
    s = w.config1()
    ctx = start(torch, flare, s)
    ctx.step(1.0, 10, want_variance=True)
    st = ctx.get_state_host(variances=True)
    ref = oracle.step(s.pos, s.vel, s.types, s.mass, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, 1.0, 10)
    # 10 steps: round-off has not been amplified yet
    assert np.abs(st["pos"] - ref["pos"]).max() < 1e-10
    assert np.abs(st["vel"] - ref["vel"]).max() < 1e-12
    assert np.abs(st["F"] - ref["F"]).max() < 1e-9
    assert np.abs(st["E"] - ref["E"]).max() < 1e-10
    assert np.abs(st["V"] - ref["V"]).max() < 1e-13
    h_gpu, _ = total_energy(st, s)
    assert abs(h_gpu - (ref["pe"][-1] + ref["ke"][-1])) < 1e-9


def test_config2_resync_parity_during_md(oracle, torch, flare):
    s = w.config2()
    ctx = start(torch, flare, s)
    h = []
    for block in range(4):
        ctx.step(0.5, 25, want_variance=True)
        st = ctx.get_state_host(variances=True)
        E, F, V = oracle.compute(st["pos"], s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
        assert np.all(np.abs(st["E"] - E) <= 1e-12 + 1e-10 * np.abs(E))
        assert np.all(np.abs(st["F"] - F) <= 1e-12 + 1e-10 * np.abs(F))
        assert np.all(np.abs(st["V"] - V) <= 1e-15 + 1e-10 * np.abs(V))
        h.append(total_energy(st, s))
    h0 = w.kinetic_energy(s.vel, s.types, s.mass)
    drift = max(abs(x[0] - h[0][0]) for x in h)
    assert drift < 2e-3 * h0, (drift, h0)  # NVE: conserved to a small fraction of the kinetic energy
    # positions stay wrapped
    L = np.asarray(s.box).reshape(3, 3).diagonal()
    assert np.all(st["pos"] >= 0) and np.all(st["pos"] < L)


def test_drift_scales_with_dt_squared_and_time_reversal(torch, flare):
    s = w.config1()
    fl = []
    for dt, n in ((4.0, 20), (2.0, 40)):
        ctx = start(torch, flare, s, variance=False)
        ctx.step(dt, 0)
        h0, _ = total_energy(ctx.get_state_host(), s)
        worst = 0.0
        for _ in range(n // 5):
            ctx.step(dt, 5)
            hh, _ = total_energy(ctx.get_state_host(), s)
            worst = max(worst, abs(hh - h0))
        fl.append(worst)
    assert 2.0 < fl[0] / fl[1] < 8.0, fl
    # time reversal
    ctx = start(torch, flare, s, variance=False)
    ctx.step(1.0, 20)
    st = ctx.get_state_host()
    ctx.set_state(st["pos"], -st["vel"], s.types, s.box, s.pbc)
    ctx.step(1.0, 20)
    back = ctx.get_state_host()
    L = np.asarray(s.box).reshape(3, 3).diagonal()
    d = back["pos"] - s.pos
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-9
    assert np.abs(-back["vel"] - s.vel).max() < 1e-11
    # momentum conservation
    m = s.mass[s.types][:, None]
    assert np.abs((m * back["vel"]).sum(0) + (m * s.vel).sum(0)).max() < 1e-11


def test_supplied_forces_skip_the_initial_evaluation(torch, flare):
    s = w.config1()
    ctx = start(torch, flare, s, variance=False)
    ctx.step(1.0, 3)
    a = ctx.get_state_host()
    ctx2 = start(torch, flare, s, variance=False)
    ctx2.step(1.0, 1)
    mid = ctx2.get_state_host()
    n0 = ctx2.kernel_launches()
    ctx2.set_state(mid["pos"], mid["vel"], s.types, s.box, s.pbc)
    ctx2.set_forces(mid["F"])
    ctx2.step(1.0, 2)
    per_eval = (ctx2.kernel_launches() - n0)
    b = ctx2.get_state_host()
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["vel"], b["vel"])
    ctx3 = start(torch, flare, s, variance=False)
    n1 = ctx3.kernel_launches()
    ctx3.step(1.0, 2)
    assert ctx3.kernel_launches() - n1 > per_eval  # that one evaluated the initial forces as well


def test_skin_list_reuse_is_exact(oracle, torch, flare):
    """The candidate list with a skin (R12) is reused across steps and rebuilt on the device when an atom has moved
    skin/2: trajectories agree with the rebuild-every-step path to rounding, the neighbour sets at the end are the
    oracle's bit for bit, and the run really did both reuse and rebuild the list."""
    s = w.config2()
    out = {}
    for skin in (0.0, 0.4):
        ctx = start(torch, flare, s, skin=skin)
        ctx.step(0.5, 60, want_variance=True)
        st = ctx.get_state_host(variances=True)
        out[skin] = (ctx, st)
    (c0, a), (c1, b) = out[0.0], out[0.4]
    assert c0.get_option(flare.OPT_SKIN) == 0 and c1.get_option(flare.OPT_SKIN) == 400
    rebuilds = c1.get_option(flare.OPT_SKIN_REBUILDS)
    assert 1 < rebuilds < 61, rebuilds          # 61 evaluations: some rebuilt, most reused
    assert c0.get_option(flare.OPT_SKIN_REBUILDS) == 0
    assert np.abs(a["pos"] - b["pos"]).max() < 1e-9
    assert np.abs(a["F"] - b["F"]).max() < 1e-7
    cnt_g, idx_g = c1.neighbors()
    cnt_o, idx_o = oracle.neighbors(b["pos"], s.types, s.box, s.pbc, s.r_cut, 0, cap=idx_g.shape[1])
    assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)
    E, F, V = oracle.compute(b["pos"], s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, nbr_method=0)
    assert np.all(np.abs(b["E"] - E) <= 1e-12 + 1e-10 * np.abs(E))
    assert np.all(np.abs(b["F"] - F) <= 1e-12 + 1e-10 * np.abs(F))
    assert np.all(np.abs(b["V"] - V) <= 1e-15 + 1e-10 * np.abs(V))
    # a jump of one atom far beyond the skin (new positions through set_state) forces a rebuild and stays exact
    pos2 = b["pos"].copy()
    pos2[900] += np.array([3.0, -2.0, 1.5])
    c1.set_state(pos2, b["vel"], s.types, s.box, s.pbc)
    c1.step(0.5, 0, want_variance=False)
    assert c1.get_option(flare.OPT_SKIN_REBUILDS) == rebuilds + 1
    cnt_g, idx_g = c1.neighbors()
    cnt_o, idx_o = oracle.neighbors(pos2, s.types, s.box, s.pbc, s.r_cut, 0, cap=idx_g.shape[1])
    assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)


@pytest.mark.parametrize("case", ["open_z", "two_cells", "hot_gas"])
def test_skin_list_edge_geometries(oracle, torch, flare, case):
    """The reused candidate list in the geometries where its bookkeeping could go wrong: an open dimension with atoms
    leaving the box, a periodic box only two cells wide (every cell is its own neighbour several times over), and a hot
    two-species gas whose atoms cross cell and box boundaries every few steps.  After the run the neighbour sets must be
    the oracle's bit for bit and E, F, V must agree at the final positions."""
    rng = np.random.default_rng(77)
    if case == "open_z":
        s = w.tile_like_c3(10, 5, n_max=3, l_max=2)
        s.pbc = np.array([1, 1, 0], np.int32)
        s.vel = w.maxwell_velocities(rng, s.types, s.mass, 3000.0)
        dt, steps = 1.0, 40
    elif case == "two_cells":
        pos, types, box, pbc = w.fcc_bulk(2, w.A_PT, 0.05, rng)  # L = 7.84 A: two cells of 3.9 A per dimension
        s = w.System("two_cells", pos, types, box, pbc, np.array([w.MASS_PT]), np.array([[3.5]]), 3, 2)
        P = w.num_descriptors(1, 3, 2)
        s.beta, s.sigma = w.random_beta(rng, 1, P), w.random_sigma(rng, 1, P)
        s.vel = w.maxwell_velocities(rng, s.types, s.mass, 20000.0)
        dt, steps = 2.0, 60
    else:
        n = 300
        L = 24.0
        pos = rng.uniform(0, L, (n, 3))
        keep = [0]
        for i in range(1, n):
            d = pos[keep] - pos[i]
            d -= L * np.round(d / L)
            if np.min(np.linalg.norm(d, axis=1)) > 1.3:
                keep.append(i)
        pos = pos[keep]
        types = rng.integers(0, 2, len(keep)).astype(np.int32)
        s = w.System("hot_gas", pos, types, np.diag([L, L, L]).reshape(9), np.ones(3, np.int32),
                     np.array([w.MASS_PT, w.MASS_H]), w.R_CUT_2, 3, 2)
        P = w.num_descriptors(2, 3, 2)
        s.beta, s.sigma = w.random_beta(rng, 2, P), w.random_sigma(rng, 2, P)
        s.vel = w.maxwell_velocities(rng, s.types, s.mass, 4000.0)
        dt, steps = 1.0, 60
    ctx = start(torch, flare, s)
    assert ctx.get_option(flare.OPT_SKIN) == 400
    ctx.step(dt, steps, want_variance=True)
    st = ctx.get_state_host(variances=True)
    rebuilds = ctx.get_option(flare.OPT_SKIN_REBUILDS)
    assert 1 <= rebuilds <= steps + 1
    cnt_g, idx_g = ctx.neighbors()
    cnt_o, idx_o = oracle.neighbors(st["pos"], s.types, s.box, s.pbc, s.r_cut, 0, cap=idx_g.shape[1])
    assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)
    E, F, V = oracle.compute(st["pos"], s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, nbr_method=0)
    assert np.all(np.abs(st["E"] - E) <= 1e-12 + 1e-10 * np.abs(E))
    assert np.all(np.abs(st["F"] - F) <= 1e-12 + 1e-10 * np.abs(F))
    assert np.all(np.abs(st["V"] - V) <= 1e-15 + 1e-10 * np.abs(V))
    # the same run with the list rebuilt at every evaluation ends in the same place (to rounding)
    ref = start(torch, flare, s, skin=0.0)
    ref.step(dt, steps, want_variance=True)
    rp = ref.get_state_host()["pos"]
    d = st["pos"] - rp
    L3 = np.asarray(s.box, float).reshape(3, 3).diagonal()
    for a in range(3):
        if s.pbc[a]:
            d[:, a] -= L3[a] * np.round(d[:, a] / L3[a])
    assert np.abs(d).max() < 1e-7


# ----------------------------------------------------------------------------- CUDA-graph replay of the step (small systems)


@pytest.mark.parametrize("name", ["c1", "c2_hot", "c2_nvt", "c2_noskin"])
def test_graph_replay_is_bit_identical_to_plain_launches(torch, flare, name):
    """FLARE_OPT_GRAPH: a run replayed from the captured step (with the candidate-list rebuild chain as a conditional
    IF node) gives bit for bit the trajectory of plain launches, across list rebuilds, for NVE and NVT, with and
    without a candidate list; the graph is really used (replay counter) and dropped when dt changes."""
    if name == "c1":
        s, dt, steps = w.config1(), 1.0, 40
    else:
        s, dt, steps = w.config2(), 0.5, 60
        if name == "c2_hot":  # hot gas: several rebuilds of the candidate list inside the run
            s.vel = w.maxwell_velocities(np.random.default_rng(5), s.types, s.mass, 6000.0)
    kw = dict(skin=0.0) if name == "c2_noskin" else {}
    runs = {}
    for graph in (0, 1):
        ctx = start(torch, flare, s, graph=graph, **kw)
        if name == "c2_nvt":
            ctx.step_nvt(dt, steps, 500.0, 50.0, want_variance=True)
            ctx.step_nvt(dt, 5, 500.0, 50.0, want_variance=True)
        else:
            ctx.step(dt, steps, want_variance=True)
            ctx.step(dt, 5, want_variance=True)       # a second call keeps replaying
            ctx.step(0.5 * dt, 4, want_variance=True)  # new dt: one plain step, a new capture, replays
        st = ctx.get_state_host(variances=True)
        runs[graph] = (st, ctx.get_option(flare.OPT_SKIN_REBUILDS), ctx.get_option(flare.OPT_GRAPH_REPLAYS),
                       ctx.thermostat() if name == "c2_nvt" else None, ctx.kernel_launches())
    (a, ra, pa, ta, la), (b, rb, pb, tb, lb) = runs[0], runs[1]
    assert pa == 0 and pb >= steps + 5 - 1 - 1
    for k in ("pos", "vel", "E", "F", "V"):
        assert np.array_equal(a[k], b[k]), k
    assert ra == rb and ta == tb
    if name == "c2_hot":
        assert rb >= 3, rb  # the IF body ran inside replayed steps
    if name == "c2_noskin":
        assert rb == 0
    # a replayed step on a kept list launches fewer kernels than a plain one (the rebuild chain is skipped, not emptied)
    if name in ("c1", "c2_nvt"):
        assert lb < la


def test_graph_option_automatic_threshold_and_off(torch, flare):
    s = w.config1()
    ctx = start(torch, flare, s)  # automatic: 256 atoms are far below the threshold
    assert ctx.get_option(flare.OPT_GRAPH) == -1
    ctx.step(1.0, 6)
    assert ctx.get_option(flare.OPT_GRAPH_REPLAYS) == 5  # step 1 plain, step 2 captured + replayed, ...
    ctx.set_option(flare.OPT_GRAPH, 0)
    ctx.step(1.0, 3)
    assert ctx.get_option(flare.OPT_GRAPH_REPLAYS) == 5
    # an error inside a replayed run is still reported, and the run recovers on plain launches
    bad = s.pos.copy()
    bad[3] = np.nan
    ctx.set_option(flare.OPT_GRAPH, 1)
    ctx.step(1.0, 3)
    ctx.set_state(bad, s.vel, s.types, s.box, s.pbc)
    with pytest.raises(flare.FlareError) as ei:
        ctx.step(1.0, 2)
        ctx.check()
    assert ei.value.code == -7
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    ctx.step(1.0, 3)
    ctx.check()
