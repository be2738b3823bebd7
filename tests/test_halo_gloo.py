"""The N > 1 path on CPU: `paper_2204_12573_b200.halo.DomainDecomposition` with world_size 2, 3 and 4 (a 2 x 2 grid)
over gloo.  The engine here is tests/domain_reference.py (a numpy restatement of the device data plane with the ORACLE
as the force field; the product engine is CudaEngine), so what is tested is the orchestration: process-grid geometry,
message routing (incl. two ranks along an axis, where both messages go to the same peer), the two-phase ghost
exchange with corners, fixed send lists between rebuilds, migration, the lagged rebuild signal.
Reference: the same oracle on the undivided system."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2204_12573_b200 import workloads as w

RC = np.array([[3.4, 3.0], [3.0, 3.0]])
N_MAX, L_MAX = 3, 2
MASS = np.array([12.0, 1.5])
HALO_SKIN = 2.0


def make_system(nx=8, ny=8, nz=2):
    rng = np.random.default_rng(77)
    a = w.A_PT
    base = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    cells = np.array([[i, j, k] for i in range(nx) for j in range(ny) for k in range(nz)])
    pos = ((cells[:, None, :] + base[None]) * a).reshape(-1, 3) + rng.normal(0, 0.06, (nx * ny * nz * 4, 3))
    types = (rng.random(len(pos)) < 0.3).astype(np.int32)
    box = np.diag([nx * a, ny * a, nz * a]).reshape(9)
    pbc = np.ones(3, np.int32)
    vel = w.maxwell_velocities(rng, types, MASS, 2500.0)
    P = w.num_descriptors(2, N_MAX, L_MAX)
    return pos, vel, types, box, pbc, w.random_beta(rng, 2, P), w.random_sigma(rng, 2, P)


def _worker(rank, world, grid, port, n_steps, dt, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from domain_reference import NumpyOracleEngine
        from oracle import flare_oracle
        from paper_2204_12573_b200.halo import DomainDecomposition

        flare_oracle.set_num_threads(2)
        pos, vel, types, box, pbc, beta, sigma = make_system()
        eng = NumpyOracleEngine(flare_oracle, MASS, N_MAX, L_MAX, RC, beta, sigma)
        # 2500 K, 1.5 amu, dt = 1 fs: the fastest atoms do 0.2 A per step, so the signal is raised early enough
        # (0.25 of the skin) for the two steps of lag to stay inside the shell's guarantee (checked by the engine)
        dd = DomainDecomposition(eng, box, pbc, RC.max(), grid=grid, halo_skin=HALO_SKIN,
                                 trigger_fraction=0.25).scatter(pos, vel, types)
        own0 = set(eng.tag[:eng.n_owned].tolist())
        dd.compute(variances=True)
        first = dd.gather()
        dd.step(dt, n_steps, variances=True)
        last = dd.gather()
        moved = len(own0.symmetric_difference(set(eng.tag[:eng.n_owned].tolist())))
        stats = torch.tensor([moved, eng.max_local, dd.bytes_sent, dd.rebuilds, eng.evaluations], dtype=torch.int64)
        dist.all_reduce(stats, op=dist.ReduceOp.SUM)
        if rank == 0:
            q.put((first, last, stats.tolist(), len(pos)))
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world,grid", [(2, (2, 1)), (3, (3, 1)), (4, (2, 2)), (2, (1, 2))])
def test_domain_decomposition_matches_the_undivided_system(oracle, world, grid):
    n_steps, dt = 12, 1.0
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, grid, port, n_steps, dt, q)) for r in range(world)]
    for p in procs:
        p.start()
    first, last, stats, n = q.get(timeout=400)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pos, vel, types, box, pbc, beta, sigma = make_system()
    E, F, V = oracle.compute(pos, types, box, pbc, N_MAX, L_MAX, RC, beta, sigma, nbr_method=0)
    np.testing.assert_allclose(first["E"], E, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(first["F"], F, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(first["V"], V, rtol=1e-12, atol=1e-16)
    ref = oracle.step(pos, vel, types, MASS, box, pbc, N_MAX, L_MAX, RC, beta, sigma, dt, n_steps, nbr_method=0)
    Lb = np.asarray(box).reshape(3, 3).diagonal()
    d = last["pos"] - ref["pos"]
    d -= Lb * np.round(d / Lb)
    assert np.abs(d).max() < 1e-10
    assert np.abs(last["vel"] - ref["vel"]).max() < 1e-11
    assert np.abs(last["F"] - ref["F"]).max() < 1e-8
    assert np.abs(last["E"] - ref["E"]).max() < 1e-9
    moved, max_local_sum, sent, rebuilds, evaluations = stats
    assert rebuilds >= 2 * world, "the run should contain a rebuild after the first one"
    assert rebuilds < world * n_steps // 2, "between rebuilds the send lists and ghost slots are reused"
    assert moved > 0, "the test system should make at least one atom change domains"
    assert sent > 0
    assert evaluations == world * (n_steps + 1)


def _failing_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from domain_reference import HaloExceeded, NumpyOracleEngine
        from oracle import flare_oracle
        from paper_2204_12573_b200.halo import DomainDecomposition, PeerError

        flare_oracle.set_num_threads(2)
        pos, vel, types, box, pbc, beta, sigma = make_system()
        if rank != 0:
            vel = vel * np.where(pos[:, :1] < 0.5 * box[0], 1.0, 0.05)  # the atoms of the other ranks' half barely move
        eng = NumpyOracleEngine(flare_oracle, MASS, N_MAX, L_MAX, RC, beta, sigma)
        # a thin skin read six steps late: the fast atoms leave the shell's guarantee long before the rebuild arrives
        dd = DomainDecomposition(eng, box, pbc, RC.max(), grid=(world, 1), halo_skin=0.8, lag=6).scatter(pos, vel, types)
        steps = 0
        try:
            for _ in range(14):
                dd.step(1.0, 1)
                steps += 1
            q.put((rank, "no error", steps))
        except (HaloExceeded, PeerError) as ex:
            q.put((rank, type(ex).__name__, steps))
    finally:
        dist.destroy_process_group()


def test_an_engine_error_on_one_rank_stops_every_rank_in_the_same_step():
    """an error used to surface on the rank it happened on only, leaving its peers blocked in the next
    exchange until the backend's timeout.  The ranks' error bits now ride with the lagged rebuild signal (all-reduce
    MAX), so all of them stop in the same step -- the owner with its own error, the others with PeerError -- and the
    ghost-shell guard (an atom moved more than halo_skin / 2 since the rebuild) is what raises it here."""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_failing_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    kinds = [g[1] for g in got]
    assert "no error" not in kinds, got
    assert "HaloExceeded" in kinds, got
    assert got[0][2] == got[1][2], f"the ranks stopped in different steps: {got}"
    assert 6 <= got[0][2] < 14


def test_geometry_checks():
    from paper_2204_12573_b200.halo import DomainDecomposition, Engine

    # world 1 (no process group): the whole box, periodic flags untouched, no exchange phases
    dd = DomainDecomposition(Engine(), np.diag([20.0, 10.0, 10.0]).reshape(9), [1, 1, 0], 3.0)
    assert dd.world == 1 and dd.local_pbc.tolist() == [1, 1, 0] and dd.local_L.tolist() == [20.0, 10.0, 10.0]
    assert dd.phases == [] and dd.h == pytest.approx(7.2) and dd.trigger == pytest.approx(0.42)
    assert dd.limit == pytest.approx(0.6)  # the shell is complete up to half the skin per atom
    with pytest.raises(ValueError):
        DomainDecomposition(Engine(), np.diag([20.0, 10.0, 10.0]).reshape(9), [1, 1, 0], 3.0, grid=(2, 1))
    for bad in (dict(lag=0), dict(lag=17), dict(trigger_fraction=0.5), dict(trigger_fraction=0.0), dict(halo_skin=0.0)):
        with pytest.raises(ValueError):
            DomainDecomposition(Engine(), np.diag([20.0, 10.0, 10.0]).reshape(9), [1, 1, 0], 3.0, **bad)


def test_process_grid_geometry_4x2():
    """Rank <-> (cx, cy) mapping, mutual neighbours along both axes (periodic wrap), local frames that tile the box."""
    from paper_2204_12573_b200.halo import DomainDecomposition, Engine

    box, pbc, rc = np.diag([120.0, 60.0, 30.0]).reshape(9), [1, 1, 0], 3.0
    dds = [DomainDecomposition(Engine(), box, pbc, rc, grid=(4, 2), halo_skin=1.0, rank=r, world=8) for r in range(8)]
    for r, dd in enumerate(dds):
        cx, cy = r // 2, r % 2
        phx, phy = dd.phases
        assert (phx["axis"], phx["p"], phx["c"], phy["axis"], phy["p"], phy["c"]) == (0, 4, cx, 1, 2, cy)
        assert phx["lo_rank"] == ((cx - 1) % 4) * 2 + cy and phx["hi_rank"] == ((cx + 1) % 4) * 2 + cy
        assert phy["lo_rank"] == cx * 2 + (cy - 1) % 2 and phy["hi_rank"] == cx * 2 + (cy + 1) % 2
        # neighbours are mutual
        assert dds[phx["hi_rank"]].phases[0]["lo_rank"] == r and dds[phy["hi_rank"]].phases[1]["lo_rank"] == r
        # local frame: open along x and y with the owned rectangle at [h, h + w); z untouched
        assert dd.local_pbc.tolist() == [0, 0, 0] and dd.h == pytest.approx(7.0)
        assert dd.local_L.tolist() == pytest.approx([30.0 + 14.0, 30.0 + 14.0, 30.0])
        assert dd.lo.tolist() == pytest.approx([cx * 30.0 - 7.0, cy * 30.0 - 7.0, 0.0])
    with pytest.raises(ValueError):  # a domain narrower than the halo
        DomainDecomposition(Engine(), box, pbc, rc, grid=(4, 2), halo_skin=30.0, rank=0, world=8)
