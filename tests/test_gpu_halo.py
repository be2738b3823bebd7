"""The decomposed path with the PRODUCT engine (CudaEngine -> libflare_b200): two ranks share the one GPU of the
test box and exchange halos over gloo (host-side waits only: no kernel waits on another rank).  Reference: the
undivided system evaluated by one context on the same GPU."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2204_12573_b200 import workloads as w

pytestmark = pytest.mark.gpu


def _system():
    return w.tile_like_c3(26, 6, n_max=4, l_max=3)


def _worker(rank, world, port, n_steps, dt, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2204_12573_b200 import flare
        from paper_2204_12573_b200.halo import CudaEngine, SlabDecomposition

        s = _system()
        eng = CudaEngine(flare.from_system(s, device=0), capacity=s.n_atoms)
        dd = SlabDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), axis=0).scatter(s.pos, s.vel, s.types)
        dd.compute(variances=True)
        first = dd.gather()
        dd.step(dt, n_steps, variances=True)
        last = dd.gather()
        launches = torch.tensor([eng.ctx.kernel_launches()], dtype=torch.int64)
        dist.all_reduce(launches)
        if rank == 0:
            q.put((first, last, int(launches)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_on_one_gpu_match_the_undivided_system():
    from paper_2204_12573_b200 import flare

    n_steps, dt, world = 5, 0.5, 2
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_steps, dt, q)) for r in range(world)]
    for p in procs:
        p.start()
    first, last, launches = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert launches > 0
    s = _system()
    one = flare.from_system(s).bind(s.n_atoms)
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    e, f, v = one.compute(pos, types, s.box, s.pbc, variances=True)
    e, f, v = e.cpu().numpy(), f.cpu().numpy(), v.cpu().numpy()
    assert np.all(np.abs(first["E"] - e) <= 1e-12 + 1e-10 * np.abs(e))
    assert np.all(np.abs(first["F"] - f) <= 1e-12 + 1e-10 * np.abs(f))
    assert np.all(np.abs(first["V"] - v) <= 1e-15 + 1e-10 * np.abs(v))
    one.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    one.step(dt, n_steps, want_variance=True)
    ref = one.get_state_host(variances=True)
    L = np.asarray(s.box, float).reshape(3, 3).diagonal()
    d = last["pos"] - ref["pos"]
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-10
    assert np.abs(last["vel"] - ref["vel"]).max() < 1e-11
    assert np.abs(last["F"] - ref["F"]).max() < 1e-8
