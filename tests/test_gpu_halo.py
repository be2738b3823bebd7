"""The decomposed path with the PRODUCT engine (CudaEngine -> libflare_b200, device data plane of csrc/domain.cu).
 * one process, one GPU, the rank as its own neighbour along x and y (self-halo): every data-plane kernel and the
   step loop, against the undivided periodic context and, call by call, against tests/domain_reference.py;
 * 2 and 4 (2 x 2) ranks sharing the one GPU of the test box, messages over gloo (host-side waits only: no kernel
   waits on another rank), against the undivided system; the candidate neighbour list must survive the steps between
   two rebuilds."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2204_12573_b200 import workloads as w

pytestmark = pytest.mark.gpu
OPT_SKIN_REBUILDS = 6


def _system():
    return w.tile_like_c3(26, 6, n_max=4, l_max=3)


def _capacity(s, world):
    return int(3.5 * s.n_atoms / world) + 4096  # owned + the ghost shell of a small tile (mostly halo)


def _reference_run(s, dt, n_steps):
    from paper_2204_12573_b200 import flare

    one = flare.from_system(s).bind(s.n_atoms)
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    e, f, v = one.compute(pos, types, s.box, s.pbc, variances=True)
    first = dict(E=e.cpu().numpy(), F=f.cpu().numpy(), V=v.cpu().numpy())
    one.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    one.step(dt, n_steps, want_variance=True)
    return first, one.get_state_host(variances=True)


def _compare(s, first, last, ref_first, ref_last):
    e, f, v = ref_first["E"], ref_first["F"], ref_first["V"]
    assert np.all(np.abs(first["E"] - e) <= 1e-12 + 1e-10 * np.abs(e))
    assert np.all(np.abs(first["F"] - f) <= 1e-12 + 1e-10 * np.abs(f))
    assert np.all(np.abs(first["V"] - v) <= 1e-15 + 1e-10 * np.abs(v))
    L = np.asarray(s.box, float).reshape(3, 3).diagonal()
    d = last["pos"] - ref_last["pos"]
    d -= L * np.round(d / L)
    assert np.abs(d).max() < 1e-10
    assert np.abs(last["vel"] - ref_last["vel"]).max() < 1e-11
    assert np.abs(last["F"] - ref_last["F"]).max() < 1e-8
    assert np.abs(last["E"] - ref_last["E"]).max() < 1e-9


def test_self_halo_on_one_gpu_matches_the_periodic_context(oracle):
    """World size 1, but x and y go through the whole data path (the rank's ghosts are its own periodic images).
    The first evaluation is compared with the ORACLE on the undivided system directly (not only through the
    undivided CUDA context), at the parity tolerances."""
    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import CudaEngine, DomainDecomposition

    s = _system()
    n_steps, dt = 40, 0.5
    eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
    dd = DomainDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), grid=(1, 1), self_halo=True, halo_skin=1.0)
    assert len(dd.phases) == 2
    dd.scatter(s.pos, s.vel, s.types)
    dd.compute(variances=True)
    first = dd.gather()
    assert dd.counts["n_owned"] == s.n_atoms and dd.counts["n_local"] > 2 * s.n_atoms
    dd.step(dt, n_steps, variances=True)
    last = dd.gather()
    eng.ctx.check()
    ref_first, ref_last = _reference_run(s, dt, n_steps)
    _compare(s, first, last, ref_first, ref_last)
    E, F, V = oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
    assert np.all(np.abs(first["E"] - E) <= 1e-12 + 1e-10 * np.abs(E))
    assert np.all(np.abs(first["F"] - F) <= 1e-12 + 1e-10 * np.abs(F))
    assert np.all(np.abs(first["V"] - V) <= 1e-15 + 1e-10 * np.abs(V))
    assert 2 <= dd.rebuilds < n_steps // 3, dd.rebuilds
    # the candidate list is rebuilt with the ghost shell, not every step
    assert eng.ctx.get_option(OPT_SKIN_REBUILDS) <= dd.rebuilds + 2


def test_self_halo_long_hot_run_keeps_every_atom_and_the_energy():
    """300 steps at 1500 K through dozens of rebuilds and migrations: no atom lost or duplicated (gather checks the tags),
    zero net force, and the same total energy as the undivided run (trajectories are chaotic, the energy is not)."""
    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import CudaEngine, DomainDecomposition

    s = w.tile_like_c3(48, 24)
    s.vel = w.maxwell_velocities(np.random.default_rng(11), s.types, s.mass, 1500.0)
    n_steps, dt = 300, 0.5
    one = flare.from_system(s).bind(s.n_atoms)
    one.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    one.step(dt, n_steps, want_variance=True)
    ref = one.get_state_host(variances=True)
    e_ref = ref["E"].sum() + w.kinetic_energy(ref["vel"], s.types, s.mass)
    eng = CudaEngine(flare.from_system(s, device=0), capacity=3 * s.n_atoms + 4096)
    # hot atoms in a random potential are fast: raise the rebuild signal early (0.2 of the skin) so that the two steps of
    # lag stay inside the ghost shell's guarantee, which the engine checks (FLARE_ERR_HALO_EXCEEDED otherwise)
    dd = DomainDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), grid=(1, 1), self_halo=True, halo_skin=1.5,
                             trigger_fraction=0.2)
    dd.scatter(s.pos, s.vel, s.types)
    dd.step(dt, n_steps, variances=True)
    got = dd.gather()
    eng.ctx.check()
    e_got = got["E"].sum() + w.kinetic_energy(got["vel"], s.types, s.mass)
    assert dd.rebuilds > 20 and dd.counts["n_owned"] == s.n_atoms
    assert np.abs(got["F"].sum(0)).max() < 1e-9
    assert abs(e_got - e_ref) < 1e-3 * max(1.0, abs(e_ref) * 1e-3), (e_got, e_ref)


def test_data_plane_matches_the_numpy_reference_call_by_call():
    """Same calls, same messages: migration (atoms pushed over both faces), two border phases, commit, a forward round."""
    from domain_reference import NumpyOracleEngine
    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import MSG_FULL_ROW, MSG_FWD_ROW, MSG_HEADER, CudaEngine

    s = _system()
    rng = np.random.default_rng(3)
    n = s.n_atoms
    L = np.asarray(s.box, float).reshape(3, 3).diagonal()
    h = 9.0
    pos = s.pos + np.array([h, h, 0.0])  # local frame of a 1 x 1 "grid": owned rectangle [h, h + L)
    leave = rng.choice(n, 40, replace=False)
    pos[leave[:20], 0] = h - rng.random(20)          # left through the x-lo face
    pos[leave[20:], 0] = h + L[0] + rng.random(20)   # ... x-hi face
    box = np.diag([L[0] + 2 * h, L[1] + 2 * h, L[2]]).reshape(9)
    pbc = [0, 0, 1]
    tags = np.arange(n, dtype=np.int64)
    cuda = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
    ref = NumpyOracleEngine(None, s.mass, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma)
    mcap, bcap = 64, 4 * n
    for e in (cuda, ref):
        e.begin(pos, s.vel, s.types, tags, box, pbc, 0.3)

    def msgs(e, rows, width):
        return [torch.zeros(MSG_HEADER + rows * width, dtype=torch.float64, device=e.device) for _ in range(2)]

    def same(a, b, width):
        a, b = a.cpu(), b.cpu()
        cnt = int(b[0])
        assert int(a[0]) == cnt
        assert torch.equal(a[MSG_HEADER:MSG_HEADER + cnt * width], b[MSG_HEADER:MSG_HEADER + cnt * width])
        return cnt

    out = {}
    for e in (cuda, ref):
        lo, hi = msgs(e, mcap, MSG_FULL_ROW)
        e.migrate_pack(0, h, h + L[0], L[0], -L[0], lo, hi, mcap)
        e.migrate_unpack(hi, lo, mcap)  # self-exchange: what goes out through hi comes back in from lo
        out[e] = [lo, hi]
    assert same(out[cuda][0], out[ref][0], MSG_FULL_ROW) == 20 and same(out[cuda][1], out[ref][1], MSG_FULL_ROW) == 20
    inf = float("inf")
    for phase, axis in ((0, 0), (1, 1)):
        for e in (cuda, ref):
            lo, hi = msgs(e, bcap, MSG_FULL_ROW)
            e.border_pack(phase, axis, -inf, 2 * h, L[axis], inf, L[axis], -L[axis], lo, hi, bcap)
            e.border_unpack(phase, hi, lo, bcap)
            out[e] = [lo, hi]
        assert same(out[cuda][0], out[ref][0], MSG_FULL_ROW) > 0 and same(out[cuda][1], out[ref][1], MSG_FULL_ROW) > 0
    cc, cr = cuda.commit(), ref.commit()
    assert cc == cr and cc["n_owned"] == n
    for phase in (0, 1):
        for e, c in ((cuda, cc), (ref, cr)):
            lo = torch.zeros(MSG_HEADER + c["send"][2 * phase] * MSG_FWD_ROW, dtype=torch.float64, device=e.device)
            hi = torch.zeros(MSG_HEADER + c["send"][2 * phase + 1] * MSG_FWD_ROW, dtype=torch.float64, device=e.device)
            e.forward_pack(phase, lo, hi)
            e.forward_unpack(phase, hi, lo)
            out[e] = [lo, hi]
        same(out[cuda][0], out[ref][0], MSG_FWD_ROW)
        same(out[cuda][1], out[ref][1], MSG_FWD_ROW)
    # the whole local state (owned in their compacted order, then the four ghost blocks) is identical
    st = cuda.ctx.get_state(results=False)
    assert np.array_equal(st["pos"].cpu().numpy(), ref.x) and np.array_equal(st["vel"].cpu().numpy(), ref.v)
    assert np.array_equal(cuda.ctx.domain_tags().cpu().numpy(), ref.tag)
    # capacity errors are reported, not silent
    lo, hi = msgs(cuda, 4, MSG_FULL_ROW)
    cuda.border_pack(0, 0, -inf, 2 * h, L[0], inf, L[0], -L[0], lo, hi, 4)
    with pytest.raises(flare.FlareError) as ei:
        cuda.ctx.check()
    assert ei.value.code == -4


def test_a_bad_message_header_is_clamped_and_reported():
    """The row count in a message header comes from a peer.  One that is above the capacity both sides agreed on,
    negative or not a number (a peer built with another capacity, a stale buffer) must not make the unpack kernels
    read past the message: rows are clamped to the capacity and the error surfaces at the next check / commit."""
    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import MSG_FULL_ROW, MSG_HEADER, CudaEngine

    s = _system()
    n, cap = s.n_atoms, 8
    L = np.asarray(s.box, float).reshape(3, 3).diagonal()
    box = np.diag([L[0] + 18.0, L[1] + 18.0, L[2]]).reshape(9)
    for header, rows_kept in ((1.0e9, cap), (float(cap + 1), cap), (-3.0, 0), (float("nan"), 0)):
        eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
        eng.begin(s.pos + np.array([9.0, 9.0, 0.0]), s.vel, s.types, np.arange(n, dtype=np.int64), box, [0, 0, 1], 0.3)
        bad = torch.zeros(MSG_HEADER + cap * MSG_FULL_ROW, dtype=torch.float64, device="cuda")
        bad[0] = header
        good = torch.zeros_like(bad)
        eng.border_unpack(0, bad, good, cap)
        with pytest.raises(flare.FlareError) as ei:
            eng.commit()
        assert ei.value.code == -4
        assert eng.commit()["n_local"] == n + rows_kept   # the flag is cleared; the clamped count stands
    # an in-range header raises nothing
    eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
    eng.begin(s.pos + np.array([9.0, 9.0, 0.0]), s.vel, s.types, np.arange(n, dtype=np.int64), box, [0, 0, 1], 0.3)
    ok = torch.zeros(MSG_HEADER + cap * MSG_FULL_ROW, dtype=torch.float64, device="cuda")
    ok[0] = float(cap)
    eng.border_unpack(0, ok, torch.zeros_like(ok), cap)
    assert eng.commit()["n_local"] == n + cap


def test_an_outrun_ghost_shell_is_an_error_not_a_wrong_force():
    """A thin halo skin whose rebuild signal is read eight steps late: hot H atoms move more than half the skin before
    the rebuild arrives, so the shell's guarantee (every ghost an owned atom's force needs is present) no longer holds.
    The displacement kernel flags it and the run stops with FLARE_ERR_HALO_EXCEEDED instead of integrating on."""
    from paper_2204_12573_b200 import flare
    from paper_2204_12573_b200.halo import CudaEngine, DomainDecomposition

    s = _system()
    s.vel = w.maxwell_velocities(np.random.default_rng(5), s.types, s.mass, 1500.0)
    eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
    dd = DomainDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), grid=(1, 1), self_halo=True, halo_skin=0.3, lag=8)
    dd.scatter(s.pos, s.vel, s.types)
    with pytest.raises(flare.FlareError) as ei:
        dd.step(1.0, 30)
        eng.ctx.check()
    assert ei.value.code == -10 and "ghost shell" in str(ei.value)
    # the same run with the default skin and lag stays inside the guarantee
    eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, 1))
    dd = DomainDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), grid=(1, 1), self_halo=True)
    dd.scatter(s.pos, s.vel, s.types)
    dd.step(0.5, 30)
    eng.ctx.check()
    # the limit must lie above the trigger; 0 switches the guard off
    with pytest.raises(flare.FlareError) as ei:
        eng.ctx.domain_set_limit(0.5 * dd.trigger)
    assert ei.value.code == -1
    eng.ctx.domain_set_limit(0.0)


def test_plain_calls_are_refused_in_domain_mode_until_rebind():
    """In domain mode the context works on its local atoms (fewer than the bound capacity): whole-system calls are
    refused instead of silently evaluating a truncated system; flare_bind returns the context to plain use.  A
    flare_domain_begin that fails (bad box) leaves the context as it was."""
    from paper_2204_12573_b200 import flare

    s = _system()
    n = s.n_atoms
    ctx = flare.from_system(s).bind(n)
    pos = torch.as_tensor(s.pos, dtype=torch.float64, device="cuda")
    types = torch.as_tensor(s.types, dtype=torch.int32, device="cuda")
    e0, f0, _ = ctx.compute(pos, types, s.box, s.pbc)
    half = n // 2
    tags = torch.arange(half, dtype=torch.int64, device="cuda")
    tri = np.array(s.box, dtype=np.float64).reshape(3, 3).copy()
    tri[0, 1] = 1.0
    with pytest.raises(flare.FlareError) as ei:   # non-orthorhombic: refused, and the context stays plain
        ctx.domain_begin(half, pos[:half].contiguous(), None, types[:half].contiguous(), tags, tri.reshape(9), s.pbc, 0.3)
    assert ei.value.code == -3
    ctx.n_atoms = n
    e1, f1, _ = ctx.compute(pos, types, s.box, s.pbc)
    assert torch.equal(e0, e1) and torch.equal(f0, f1)
    ctx.domain_begin(half, pos[:half].contiguous(), None, types[:half].contiguous(), tags, s.box, s.pbc, 0.3)
    ctx.domain_commit()
    ctx.n_atoms = n
    for call in (lambda: ctx.compute(pos, types, s.box, s.pbc),
                 lambda: ctx.compute_host(s.pos, s.types, s.box, s.pbc),
                 lambda: ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc),
                 lambda: ctx.set_state(pos, None, types, s.box, s.pbc)):
        with pytest.raises(flare.FlareError) as ei:
            call()
        assert ei.value.code == -1 and "domain mode" in str(ei.value)
    ctx.bind(n)
    e2, f2, _ = ctx.compute(pos, types, s.box, s.pbc)
    assert torch.equal(e0, e2) and torch.equal(f0, f2)


def _worker(rank, world, grid, port, n_steps, dt, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2204_12573_b200 import flare
        from paper_2204_12573_b200.halo import CudaEngine, DomainDecomposition

        s = _system()
        eng = CudaEngine(flare.from_system(s, device=0), capacity=_capacity(s, world))
        dd = DomainDecomposition(eng, s.box, s.pbc, float(np.max(s.r_cut)), grid=grid, halo_skin=1.0)
        dd.scatter(s.pos, s.vel, s.types)
        dd.compute(variances=True)
        first = dd.gather()
        dd.step(dt, n_steps, variances=True)
        last = dd.gather()
        eng.ctx.check()
        stats = torch.tensor([eng.ctx.kernel_launches(), dd.rebuilds, eng.ctx.get_option(OPT_SKIN_REBUILDS)], dtype=torch.int64)
        dist.all_reduce(stats, op=dist.ReduceOp.MAX)
        if rank == 0:
            q.put((first, last, stats.tolist()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,grid", [(2, (2, 1)), (4, (2, 2))])
def test_ranks_sharing_one_gpu_match_the_undivided_system(world, grid):
    n_steps, dt = 30, 0.5
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, grid, port, n_steps, dt, q)) for r in range(world)]
    for p in procs:
        p.start()
    first, last, (launches, rebuilds, list_rebuilds) = q.get(timeout=400)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert launches > 0
    s = _system()
    ref_first, ref_last = _reference_run(s, dt, n_steps)
    _compare(s, first, last, ref_first, ref_last)
    assert 2 <= rebuilds < n_steps // 3, rebuilds
    assert list_rebuilds <= rebuilds + 2, (list_rebuilds, rebuilds)  # the candidate list survives the steps in between
