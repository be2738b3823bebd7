"""The N > 1 path on CPU: `paper_2204_12573_b200.halo.SlabDecomposition` with world_size 2 and 3 over gloo.
The force engine here is the ORACLE (tests may use it; the product engine is CudaEngine), so what is tested is
the decomposition itself: halo selection two cutoffs wide, local open-boundary frames, ghost dynamics, migration,
message plumbing.  Reference: the same oracle on the undivided system."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2204_12573_b200 import workloads as w

KAPPA = 9.648533212331e-3
RC = np.array([[3.4, 3.0], [3.0, 3.0]])
N_MAX, L_MAX = 3, 2
MASS = np.array([12.0, 1.5])


def make_system():
    rng = np.random.default_rng(77)
    a = w.A_PT
    nx, ny, nz = 8, 2, 2
    base = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]])
    cells = np.array([[i, j, k] for i in range(nx) for j in range(ny) for k in range(nz)])
    pos = ((cells[:, None, :] + base[None]) * a).reshape(-1, 3) + rng.normal(0, 0.06, (nx * ny * nz * 4, 3))
    types = (rng.random(len(pos)) < 0.3).astype(np.int32)
    box = np.diag([nx * a, ny * a, nz * a]).reshape(9)
    pbc = np.ones(3, np.int32)
    vel = w.maxwell_velocities(rng, types, MASS, 2500.0)
    P = w.num_descriptors(2, N_MAX, L_MAX)
    return pos, vel, types, box, pbc, w.random_beta(rng, 2, P), w.random_sigma(rng, 2, P)


class OracleEngine:
    device = torch.device("cpu")

    def __init__(self, oracle, beta, sigma):
        self.o, self.beta, self.sigma = oracle, beta, sigma
        self.max_local = 0

    def evaluate(self, pos, types, box, pbc, variances):
        self.max_local = max(self.max_local, pos.shape[0])
        E, F, V = self.o.compute(pos.numpy(), types.numpy(), box, pbc, N_MAX, L_MAX, RC, self.beta, self.sigma, nbr_method=0)
        return torch.as_tensor(E), torch.as_tensor(F), torch.as_tensor(V) if variances else None

    def md_step(self, pos, vel, frc, types, box, pbc, dt, variances):
        x, v, f, t = pos.numpy().copy(), vel.numpy().copy(), frc.numpy(), types.numpy()
        acc = (0.5 * dt * KAPPA / MASS[t])[:, None]
        v += acc * f
        x += dt * v
        L = np.asarray(box).reshape(3, 3).diagonal()
        for d in range(3):
            if pbc[d]:
                x[:, d] -= L[d] * np.floor(x[:, d] / L[d])
        E, F, V = self.evaluate(torch.as_tensor(x), types, box, pbc, variances)
        v += acc * F.numpy()
        return torch.as_tensor(x), torch.as_tensor(v), E, F, V


def _worker(rank, world, port, n_steps, dt, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import flare_oracle
        from paper_2204_12573_b200.halo import SlabDecomposition

        flare_oracle.set_num_threads(2)
        pos, vel, types, box, pbc, beta, sigma = make_system()
        eng = OracleEngine(flare_oracle, beta, sigma)
        dd = SlabDecomposition(eng, box, pbc, RC.max(), axis=0).scatter(pos, vel, types)
        own0 = set(dd.gid.tolist())
        dd.compute(variances=True)
        first = dd.gather()
        dd.step(dt, n_steps, variances=True)
        last = dd.gather()
        moved = len(own0.symmetric_difference(set(dd.gid.tolist())))
        stats = torch.tensor([moved, eng.max_local, dd.bytes_sent], dtype=torch.int64)
        dist.all_reduce(stats, op=dist.ReduceOp.SUM)
        if rank == 0:
            q.put((first, last, stats.tolist(), len(pos)))
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_slab_decomposition_matches_the_undivided_system(oracle, world):
    n_steps, dt = 6, 2.0
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_steps, dt, q))
             for r in range(world)]
    for p in procs:
        p.start()
    first, last, stats, n = q.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    pos, vel, types, box, pbc, beta, sigma = make_system()
    E, F, V = oracle.compute(pos, types, box, pbc, N_MAX, L_MAX, RC, beta, sigma, nbr_method=0)
    np.testing.assert_allclose(first["E"], E, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(first["F"], F, rtol=1e-11, atol=1e-12)
    np.testing.assert_allclose(first["V"], V, rtol=1e-12, atol=1e-16)
    assert np.array_equal(first["types"], types)
    ref = oracle.step(pos, vel, types, MASS, box, pbc, N_MAX, L_MAX, RC, beta, sigma, dt, n_steps, nbr_method=0)
    Lb = np.asarray(box).reshape(3, 3).diagonal()
    d = last["pos"] - ref["pos"]
    d -= Lb * np.round(d / Lb)
    assert np.abs(d).max() < 1e-10
    assert np.abs(last["vel"] - ref["vel"]).max() < 1e-11
    assert np.abs(last["F"] - ref["F"]).max() < 1e-8
    assert np.abs(last["E"] - ref["E"]).max() < 1e-9
    moved, max_local_sum, sent = stats
    assert moved > 0, "the test system should make at least one atom change slabs"
    assert sent > 0
    # every rank evaluates its slab plus a halo, not the whole system
    assert max_local_sum < world * n



def test_geometry_checks():
    from paper_2204_12573_b200.halo import Engine, SlabDecomposition

    # world 1 (no process group): the whole box, periodic flags untouched
    dd = SlabDecomposition(Engine(), np.diag([20.0, 10.0, 10.0]).reshape(9), [1, 1, 0], 3.0)
    assert dd.world == 1 and dd.local_pbc.tolist() == [1, 1, 0] and dd.local_L.tolist() == [20.0, 10.0, 10.0]
    x = torch.tensor([[-0.5, 1.0, 1.0], [20.0, 2.0, 2.0], [7.0, 3.0, 3.0]], dtype=torch.float64)
    assert torch.allclose(dd._wrap_axis(x)[:, 0], torch.tensor([19.5, 0.0, 7.0], dtype=torch.float64))
