"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bars (BASELINE.json north_star): neighbour sets bit-exact; energies, variances
within 1e-10 relative; forces within 1e-12 eV/A absolute + 1e-10 relative.
"""
import numpy as np
import pytest

from paper_2204_12573_b200 import workloads as w

pytestmark = pytest.mark.gpu

RTOL = 1e-10
ATOL_F = 1e-12  # eV/A
ATOL_E = 1e-12  # eV, guards E ~ 0 (isolated atoms)


@pytest.fixture(scope="module")
def torch():
    import torch

    return torch


@pytest.fixture(scope="module")
def flare():
    from paper_2204_12573_b200 import flare as fl

    fl.load_library()
    return fl


def dev(torch, a, dtype):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device="cuda")


def gpu_compute(torch, flare, s, variance=True, **kw):
    ctx = flare.from_system(s, variance=variance, **kw)
    ctx.bind(s.n_atoms)
    e, f, v = ctx.compute(dev(torch, s.pos, torch.float64), dev(torch, s.types, torch.int32), s.box, s.pbc,
                          variances=variance)
    torch.cuda.synchronize()
    return ctx, e.cpu().numpy(), f.cpu().numpy(), (v.cpu().numpy() if v is not None else None)


def assert_close(got, want, atol, what):
    err = np.abs(got - want)
    tol = atol + RTOL * np.abs(want)
    bad = err > tol
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance; worst err {err.max():.3e} " \
                          f"(|want| max {np.abs(want).max():.3e})"


def assert_parity(oracle, torch, flare, s, variance=True, nbr_method=1, **kw):
    ctx, e, f, v = gpu_compute(torch, flare, s, variance, **kw)
    E, F, V = oracle.compute(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta,
                             s.sigma if variance else None, nbr_method=nbr_method)
    # neighbour sets: bit-exact
    cnt_o, idx_o = oracle.neighbors(s.pos, s.types, s.box, s.pbc, s.r_cut, nbr_method, cap=ctx.get_option(1))
    cnt_g, idx_g = ctx.neighbors()
    assert np.array_equal(cnt_g, cnt_o)
    assert np.array_equal(idx_g, idx_o)
    assert_close(e, E, ATOL_E, "E")
    assert_close(f, F, ATOL_F, "F")
    if variance:
        assert_close(v, V, 1e-15, "V")
    return ctx, (e, f, v), (E, F, V)


# ----------------------------------------------------------------------------- BASELINE configs 1 and 2 in full


def test_config1_full(oracle, torch, flare):
    s = w.config1()
    ctx, got, want = assert_parity(oracle, torch, flare, s, nbr_method=0)
    assert np.abs(got[1].sum(0)).max() < 1e-11  # zero net force
    # descriptors at the a3 boundary
    bh, nrm = ctx.descriptors()
    for i in (0, 100, 255):
        _, _, Bh, n0 = oracle.descriptor(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, i)
        np.testing.assert_allclose(bh[i], Bh, atol=1e-13)
        assert abs(nrm[i] - n0) < 1e-12 * n0


@pytest.mark.parametrize("sparse", [True, False])
def test_config2_full(oracle, torch, flare, sparse):
    s = w.config2()
    ctx, got, want = assert_parity(oracle, torch, flare, s, nbr_method=0, species_sparse=sparse)
    assert ctx.get_option(4) == int(sparse)
    bh, nrm = ctx.descriptors()
    for i in (0, 500, 863, 864, 1263):  # Pt bulk, Pt surface, H
        _, _, Bh, n0 = oracle.descriptor(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, i)
        np.testing.assert_allclose(bh[i], Bh, atol=1e-13)
    assert np.abs(got[1].sum(0)).max() < 1e-10


# ----------------------------------------------------------------------------- basis sizes, several tiles + ragged tails


@pytest.mark.parametrize("sparse", [True, False])
@pytest.mark.parametrize("n_max,l_max", [(1, 0), (3, 1), (4, 2), (7, 3), (3, 4), (2, 5), (2, 6), (5, 6), (9, 2), (10, 4), (12, 6), (16, 1)])
def test_basis_sizes_on_a_small_tile(oracle, torch, flare, n_max, l_max, sparse):
    s = w.tile_like_c3(6, 3, n_max=n_max, l_max=l_max)  # 216 Pt + 18 H
    assert_parity(oracle, torch, flare, s, species_sparse=sparse)


def test_species_sparse_is_the_default_and_matches_dense(torch, flare):
    """skipping the blocks of absent neighbour species is exact; here against the dense evaluation."""
    s = w.tile_like_c3(12, 6)
    c1, e1, f1, v1 = gpu_compute(torch, flare, s)
    assert c1.get_option(4) == 1
    c0, e0, f0, v0 = gpu_compute(torch, flare, s, species_sparse=False)
    assert np.abs(e1 - e0).max() < 1e-13 and np.abs(f1 - f0).max() < 1e-12 and np.abs(v1 - v0).max() < 1e-16
    b1, n1 = c1.descriptors()
    b0, n0 = c0.descriptors()
    assert np.abs(b1 - b0).max() < 1e-14 and np.abs(n1 - n0).max() < 1e-12 * n0.max()


def test_three_species_sparse(oracle, torch, flare):
    """Three species: 24 (species, mask) groups; random species on a jittered fcc lattice."""
    rng = np.random.default_rng(41)
    pos, _, box, pbc = w.fcc_bulk(4, w.A_PT, 0.05, rng)
    types = rng.integers(0, 3, pos.shape[0]).astype(np.int32)
    types[:40] = 0  # some single-species neighbourhoods are unlikely in a random alloy; keep the mix anyway
    n_max, l_max, S = 3, 2, 3
    r_cut = np.array([[4.25, 3.6, 3.0], [3.6, 3.6, 3.0], [3.0, 3.0, 3.0]])
    P = w.num_descriptors(S, n_max, l_max)
    s = w.System("three", pos, types, box, pbc, np.array([195.0, 100.0, 1.0]), r_cut, n_max, l_max)
    s.beta = w.random_beta(rng, S, P)
    s.sigma = w.random_sigma(rng, S, P)
    for sparse in (True, False):
        assert_parity(oracle, torch, flare, s, nbr_method=0, species_sparse=sparse)


def test_paper_basis_7_3_dimension_420(oracle, torch, flare):
    """The paper's own model size: 2 species, n_max 7, l_max 3 -> 420."""
    s = w.tile_like_c3(8, 4, n_max=7, l_max=3)
    assert s.P == 420
    assert_parity(oracle, torch, flare, s)


@pytest.mark.parametrize("chunk", [64, 100, 1000])
def test_chunking_is_exact(oracle, torch, flare, chunk):
    """Step a8: chunked intermediates must not change any result; 100 gives ragged tails.
    A warp packs the neighbour lists of up to 8 consecutive rows into 32-pair passes, so the chunk
    boundaries move the 4-wide summation groups of the A accumulation: equal to rounding (a few ulp,
    far inside north_star's 1e-10), not bit for bit; each run on its own stays bit-reproducible."""
    s = w.tile_like_c3(8, 4, n_max=4, l_max=3)
    ctx0, e0, f0, v0 = gpu_compute(torch, flare, s)
    ctx1, e1, f1, v1 = gpu_compute(torch, flare, s, chunk_atoms=chunk)
    assert ctx1.get_option(2) == min(chunk, s.n_atoms)
    for x0, x1 in ((e0, e1), (f0, f1), (v0, v1)):
        assert np.all(np.abs(x0 - x1) <= 1e-15 + 1e-13 * np.abs(x0))
    assert_parity(oracle, torch, flare, s, chunk_atoms=chunk)


def test_run_to_run_determinism(torch, flare):
    s = w.config2()
    _, e0, f0, v0 = gpu_compute(torch, flare, s)
    _, e1, f1, v1 = gpu_compute(torch, flare, s)
    assert np.array_equal(e0, e1) and np.array_equal(f0, f1) and np.array_equal(v0, v1)


def test_variance_off_matches_variance_on(torch, flare):
    s = w.config2()
    _, e0, f0, _ = gpu_compute(torch, flare, s, variance=False)
    _, e1, f1, _ = gpu_compute(torch, flare, s, variance=True)
    assert np.array_equal(e0, e1) and np.array_equal(f0, f1)


# ----------------------------------------------------------------------------- edge and degenerate cases


def _mk(pos, types, box, pbc, S, n_max=3, l_max=2, seed=0):
    rng = np.random.default_rng(seed)
    P = w.num_descriptors(S, n_max, l_max)
    r_cut = w.R_CUT_1 if S == 1 else w.R_CUT_2
    mass = np.array([w.MASS_PT, w.MASS_H])[:S]
    s = w.System("edge", np.asarray(pos, float).reshape(-1, 3), np.asarray(types, np.int32), np.asarray(box, float),
                 np.asarray(pbc, np.int32), mass, r_cut, n_max, l_max)
    s.beta = w.random_beta(rng, S, P)
    s.sigma = w.random_sigma(rng, S, P)
    return s


def test_empty_and_single_atom(oracle, torch, flare):
    box = np.diag([30.0, 30, 30]).reshape(9)
    s = _mk(np.zeros((0, 3)), [], box, [1, 1, 1], 1)
    ctx, e, f, v = gpu_compute(torch, flare, s)
    assert e.size == 0 and f.size == 0
    s = _mk([[1.0, 2, 3]], [0], box, [1, 1, 1], 1)
    ctx, e, f, v = gpu_compute(torch, flare, s)
    assert e[0] == 0 and v[0] == 0 and np.all(f == 0)  # R8: empty neighbourhood
    # a dimer plus an isolated atom
    s = _mk([[1.0, 2, 3], [20, 20, 20], [21.1, 20.2, 19.7]], [0, 1, 0], box, [1, 1, 1], 2)
    assert_parity(oracle, torch, flare, s, nbr_method=0)


def test_open_and_mixed_boundaries_and_unwrapped_input(oracle, torch, flare):
    rng = np.random.default_rng(11)
    n = 300
    pos = rng.uniform(0, 22, (n, 3))
    keep = [0]
    for i in range(1, n):
        if np.min(np.linalg.norm(pos[keep] - pos[i], axis=1)) > 1.1:
            keep.append(i)
    pos = pos[keep]
    types = rng.integers(0, 2, len(keep))
    box = np.diag([22.0, 22, 22]).reshape(9)
    for pbc in ([0, 0, 0], [1, 0, 1], [1, 1, 1]):
        shifted = pos.copy()
        for d in range(3):
            if pbc[d]:
                shifted[:, d] += 22.0 * rng.integers(-3, 4, len(keep))  # any periodic image (R6)
            else:
                shifted[:, d] += -5.0  # atoms outside [0,L) in an open dimension are legal
        s = _mk(shifted, types, box, pbc, 2, n_max=3, l_max=3, seed=12)
        assert_parity(oracle, torch, flare, s, nbr_method=0)


def test_fewer_than_three_cells_per_dimension(oracle, torch, flare):
    """Box lengths between 2 and 3 cutoffs: the 27-cell stencil would revisit cells (R7)."""
    rng = np.random.default_rng(13)
    pos, types, box, pbc = w.fcc_bulk(3, w.A_PT, 0.05, rng)  # L = 11.76 A: 2 cells of >= 4.25 per dimension
    s = _mk(pos, types, box, pbc, 1, n_max=4, l_max=3, seed=14)
    assert_parity(oracle, torch, flare, s, nbr_method=0)
    pos, types, box, pbc = w.fcc_bulk(4, w.A_PT, 0.05, rng)  # L = 15.68: 3 cells
    s = _mk(pos, types, box, pbc, 1, n_max=4, l_max=3, seed=15)
    assert_parity(oracle, torch, flare, s, nbr_method=0)


def test_perfect_lattice_zero_force(torch, flare):
    pos, types, box, pbc = w.fcc_bulk(4, w.A_PT, 0.0, None)
    s = _mk(pos, types, box, pbc, 1, n_max=6, l_max=3, seed=16)
    _, e, f, v = gpu_compute(torch, flare, s)
    assert np.abs(f).max() < 1e-12 and np.ptp(e) < 1e-13


def test_error_codes(torch, flare):
    box = np.diag([30.0, 30, 30]).reshape(9)
    s = _mk(np.random.default_rng(1).uniform(0, 30, (50, 3)), np.zeros(50), box, [1, 1, 1], 1)
    ctx = flare.from_system(s)
    pos, types = dev(torch, s.pos, torch.float64), dev(torch, s.types, torch.int32)
    with pytest.raises(flare.FlareError) as ei:  # not bound
        ctx.n_atoms = 50
        ctx.compute(pos, types, s.box, s.pbc)
    assert ei.value.code == -9
    ctx.bind(50)
    with pytest.raises(flare.FlareError) as ei:  # periodic box < 2 r_cut
        ctx.compute(pos, types, np.diag([8.0, 30, 30]).reshape(9), [1, 1, 1])
    assert ei.value.code == -2
    tri = np.diag([30.0, 30, 30])
    tri[1, 0] = 2.0
    with pytest.raises(flare.FlareError) as ei:  # triclinic
        ctx.compute(pos, types, tri.reshape(9), [1, 1, 1])
    assert ei.value.code == -3
    with pytest.raises(flare.FlareError) as ei:  # variance without sigma
        c2 = flare.from_system(s, variance=False).bind(50)
        c2.compute(pos, types, s.box, s.pbc, variances=True)
    assert ei.value.code == -1
    bad = s.pos.copy()
    bad[7, 1] = np.nan
    with pytest.raises(flare.FlareError) as ei:
        ctx.compute(dev(torch, bad, torch.float64), types, s.box, s.pbc)
    assert ei.value.code == -7
    # neighbour overflow: 40 atoms in a 2 A ball with room for 8 neighbours
    rng = np.random.default_rng(2)
    s2 = _mk(15 + rng.uniform(-1, 1, (40, 3)), np.zeros(40), box, [1, 1, 1], 1)
    c3 = flare.from_system(s2, max_neighbors=8).bind(40)
    with pytest.raises(flare.FlareError) as ei:
        c3.compute(dev(torch, s2.pos, torch.float64), dev(torch, s2.types, torch.int32), s2.box, s2.pbc)
    assert ei.value.code == -5
    with pytest.raises(flare.FlareError) as ei:  # asymmetric r_cut (R5)
        flare.Flare([1.0, 1.0], 2, 1, [[3.0, 2.0], [2.5, 3.0]], np.zeros((2, 20, 20)))
    assert ei.value.code == -1
    with pytest.raises(flare.FlareError) as ei:  # l_max out of the compiled range
        flare.Flare([1.0], 2, 7, [[3.0]], np.zeros((1, 24, 24)))
    assert ei.value.code == -8


def test_species_out_of_range_is_an_error(torch, flare):
    """include/flare_b200.h: a species index outside 0..S-1 is FLARE_ERR_INVALID_ARG (flagged on the device, the
    stored type clamped so that no table is indexed out of bounds), in a first build and on a reused candidate list."""
    s = w.tile_like_c3(6, 3, n_max=3, l_max=2)
    ctx = flare.from_system(s).bind(s.n_atoms)
    pos = dev(torch, s.pos, torch.float64)
    for bad_value in (2, -1, 1 << 20):
        bad = s.types.copy()
        bad[5] = bad_value
        with pytest.raises(flare.FlareError) as ei:
            ctx.compute(pos, dev(torch, bad, torch.int32), s.box, s.pbc)
        assert ei.value.code == -1
    e, f, v = ctx.compute(pos, dev(torch, s.types, torch.int32), s.box, s.pbc, variances=True)  # the context recovers
    assert bool(torch.isfinite(f).all())
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    ctx.step(0.5, 2)
    ctx.check()
    bad = s.types.copy()
    bad[-1] = 7
    ctx.set_state(s.pos, s.vel, bad, s.box, s.pbc)  # same binding: the refresh of the kept list meets the bad type
    with pytest.raises(flare.FlareError) as ei:
        ctx.step(0.5, 1)
        ctx.check()
    assert ei.value.code == -1


def test_overflow_error_does_not_poison_the_binding(oracle, torch, flare):
    """After FLARE_ERR_NEIGHBOR_OVERFLOW the truncated candidate list must not be reused: new, sparse positions in
    the SAME binding are evaluated from scratch and match the oracle."""
    rng = np.random.default_rng(61)
    box = np.diag([30.0, 30, 30]).reshape(9)
    n = 90
    dense = 15 + rng.uniform(-2.2, 2.2, (n, 3))  # ~90 atoms in a 4.4 A cube: more than 64 candidates per atom
    s = _mk(dense, np.zeros(n), box, [1, 1, 1], 1, n_max=3, l_max=2, seed=62)
    ctx = flare.from_system(s, max_neighbors=60).bind(n)
    types = dev(torch, s.types, torch.int32)
    with pytest.raises(flare.FlareError) as ei:
        ctx.compute(dev(torch, s.pos, torch.float64), types, s.box, s.pbc)
    assert ei.value.code == -5
    # the same atoms moved by less than the skin budget would keep the (truncated) list if it were still valid
    sparse = np.stack(np.meshgrid(*[np.arange(5) * 3.1 + 4] * 3, indexing="ij"), -1).reshape(-1, 3)[:n]
    sparse = sparse + rng.normal(0, 0.05, sparse.shape)
    s2 = _mk(sparse, np.zeros(n), box, [1, 1, 1], 1, n_max=3, l_max=2, seed=62)
    for _ in range(2):  # the second evaluation runs on the list the first one rebuilt
        e, f, v = ctx.compute(dev(torch, s2.pos, torch.float64), types, s2.box, s2.pbc, variances=True)
        E, F, V = oracle.compute(s2.pos, s2.types, s2.box, s2.pbc, s2.n_max, s2.l_max, s2.r_cut, s2.beta, s2.sigma, nbr_method=0)
        assert_close(e.cpu().numpy(), E, ATOL_E, "E")
        assert_close(f.cpu().numpy(), F, ATOL_F, "F")
        cnt_o, idx_o = oracle.neighbors(s2.pos, s2.types, s2.box, s2.pbc, s2.r_cut, 0, cap=60)
        cnt_g, idx_g = ctx.neighbors()
        assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)


def test_nonfinite_results_are_reported(torch, flare):
    """NaN/Inf in E, F or V is an error code.  Two atoms at the same point give r = 0, hence a
    non-finite pair force; flare_check must say so instead of letting an MD run integrate garbage."""
    box = np.diag([30.0, 30, 30]).reshape(9)
    pos = np.array([[5.0, 5, 5], [5.0, 5, 5], [7.0, 5.5, 5.2], [20.0, 20, 20]])
    s = _mk(pos, [0, 0, 0, 0], box, [1, 1, 1], 1)
    ctx = flare.from_system(s).bind(4)
    with pytest.raises(flare.FlareError) as ei:
        ctx.compute(dev(torch, s.pos, torch.float64), dev(torch, s.types, torch.int32), s.box, s.pbc, variances=True)
    assert ei.value.code == -7
    good = pos.copy()
    good[1] += [1.5, 0.3, -0.2]
    e, f, v = ctx.compute(dev(torch, good, torch.float64), dev(torch, s.types, torch.int32), s.box, s.pbc, variances=True)
    assert bool(torch.isfinite(f).all()) and bool(torch.isfinite(e).all())


def test_two_contexts_on_two_streams(oracle, torch, flare):
    """Launch state (shared-memory limits, occupancies) is per context, not per process: two contexts with different
    basis sizes, each on its own stream, interleaved, both match the oracle."""
    sa = w.tile_like_c3(6, 3, n_max=8, l_max=3)
    sb = w.tile_like_c3(6, 3, n_max=12, l_max=6)  # > 48 KB of dynamic shared memory in every per-atom kernel
    st_a, st_b = torch.cuda.Stream(), torch.cuda.Stream()
    ca = flare.from_system(sa).bind(sa.n_atoms, stream=st_a)
    cb = flare.from_system(sb).bind(sb.n_atoms, stream=st_b)
    torch.cuda.synchronize()
    outs = {}
    for rep in range(2):
        for name, c, sy, stq in (("a", ca, sa, st_a), ("b", cb, sb, st_b)):
            with torch.cuda.stream(stq):
                pos, types = dev(torch, sy.pos, torch.float64), dev(torch, sy.types, torch.int32)
            torch.cuda.synchronize()
            outs[name] = c.compute(pos, types, sy.box, sy.pbc, variances=True, check=False)
    ca.check(); cb.check()
    for name, sy in (("a", sa), ("b", sb)):
        E, F, V = oracle.compute(sy.pos, sy.types, sy.box, sy.pbc, sy.n_max, sy.l_max, sy.r_cut, sy.beta, sy.sigma)
        e, f, v = outs[name]
        assert_close(e.cpu().numpy(), E, ATOL_E, "E")
        assert_close(f.cpu().numpy(), F, ATOL_F, "F")
        assert_close(v.cpu().numpy(), V, 1e-15, "V")


def test_many_neighbours_more_than_a_warp(oracle, torch, flare):
    """Dense blob: up to ~60 neighbours per atom exercises the >32-neighbour loops."""
    rng = np.random.default_rng(21)
    pos = rng.uniform(0, 9.0, (400, 3))
    keep = [0]
    for i in range(1, len(pos)):
        if np.min(np.linalg.norm(pos[keep] - pos[i], axis=1)) > 1.25:
            keep.append(i)
    pos = pos[keep] + 10.0
    s = _mk(pos, np.zeros(len(keep)), np.diag([30.0, 30, 30]).reshape(9), [1, 1, 1], 1, n_max=3, l_max=2, seed=22)
    cnt, _ = oracle.neighbors(s.pos, s.types, s.box, s.pbc, s.r_cut, 0, cap=255)
    assert cnt.max() > 40
    # a blob this dense has more than 64 candidates within r_cut + skin: the candidate list is switched off
    assert_parity(oracle, torch, flare, s, nbr_method=0, max_neighbors=int(cnt.max()) + 1, skin=0.0)
    with pytest.raises(flare.FlareError):
        gpu_compute(torch, flare, s, max_neighbors=int(cnt.max()) + 1, skin=0.4)


def test_host_entry_point_matches_device_entry_point(torch, flare):
    s = w.config2()
    ctx, e, f, v = gpu_compute(torch, flare, s)
    eh, fh, vh = ctx.compute_host(s.pos, s.types, s.box, s.pbc, variances=True)
    assert np.array_equal(e, eh) and np.array_equal(f, fh) and np.array_equal(v, vh)


# ----------------------------------------------------------------------------- larger systems: sampled parity


def test_tile_16k_atoms_sampled(oracle, torch, flare):
    s = w.tile_like_c3(48, 24)  # 13 824 Pt + 1152 H, P = 544
    ctx, e, f, v = gpu_compute(torch, flare, s)
    rng = np.random.default_rng(31)
    sel = np.concatenate([rng.choice(13824, 24, replace=False), 13824 + rng.choice(1152, 8, replace=False)])
    E, F, V = oracle.compute_selected(s.pos, s.types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, s.sigma, sel)
    assert_close(e[sel], E, ATOL_E, "E")
    assert_close(f[sel], F, ATOL_F, "F")
    assert_close(v[sel], V, 1e-15, "V")
    cnt_o, idx_o = oracle.neighbors(s.pos, s.types, s.box, s.pbc, s.r_cut, 1, cap=ctx.get_option(1))
    cnt_g, idx_g = ctx.neighbors()
    assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)
    assert np.abs(f.sum(0)).max() < 1e-9


def brute_force_rows(xw, types, box, pbc, r_cut, sel):
    """Neighbour rows of the atoms in `sel` by brute force over ALL N atoms (plain numpy, no cells), with R6's
    canonical arithmetic: wrapped coordinates, dx = x_j - x_i, one +-L shift beyond L/2, d2 = ((dx dx)+(dy dy))+(dz dz),
    strict d2 < r_c r_c.  Independent of both the GPU cell list and the oracle's grid."""
    L = np.asarray(box, float).reshape(3, 3).diagonal()
    S = int(round(np.sqrt(np.asarray(r_cut).size)))
    rc2 = (np.asarray(r_cut, float).reshape(S, S)) ** 2
    idx_all = np.arange(xw.shape[0])
    rows = []
    for i in sel:
        d2 = np.zeros(xw.shape[0])
        parts = []
        for a in range(3):
            d = xw[:, a] - xw[i, a]
            if pbc[a]:
                d = np.where(d > 0.5 * L[a], d - L[a], np.where(d < -0.5 * L[a], d + L[a], d))
            parts.append(d * d)
        d2 = (parts[0] + parts[1]) + parts[2]
        hit = d2 < rc2[types[i]][types]
        hit[i] = False
        rows.append(idx_all[hit])
    return rows


def full_size_check(oracle, torch, flare, s, ctx, pos, E_g, F_g, V_g, n_ev, n_f, n_brute, seed, all_rows=True):
    """Parity of a full-size system that has just been evaluated by `ctx` at positions `pos` (host): neighbour rows
    (every row against the oracle's grid search when all_rows, n_brute rows by brute force over all N), E and V of
    ~n_ev atoms and F of ~n_f atoms against the oracle one by one, drawn from EVERY (species, neighbour-mask) group
    and from the rows next to every atom-chunk boundary, plus the properties that hold at any size."""
    N = s.n_atoms
    types = s.types
    want_var = V_g is not None
    cap = 40
    cnt_g, idx_g = ctx.neighbors(stride=cap)
    rng = np.random.default_rng(seed)
    # ---- neighbour sets
    xw = oracle.wrap(pos, s.box, s.pbc)
    sel_b = rng.choice(N, n_brute, replace=False)
    for i, row in zip(sel_b, brute_force_rows(xw, types, s.box, s.pbc, s.r_cut, sel_b)):
        assert np.array_equal(row, idx_g[i, :cnt_g[i]]), f"neighbour row of atom {i} differs from brute force"
    if all_rows:
        cnt_o, idx_o = oracle.neighbors(pos, types, s.box, s.pbc, s.r_cut, 1, cap=cap)
        assert np.array_equal(cnt_g, cnt_o) and np.array_equal(idx_g, idx_o)
        del cnt_o, idx_o
    assert int(cnt_g.sum()) % 2 == 0  # full (symmetric) list
    # ---- groups: (species, set of neighbour species) of every atom, from the (just verified) rows
    valid = idx_g >= 0
    tn = types[np.where(valid, idx_g, 0)]
    mask = np.zeros(N, np.int64)
    for sp in range(s.n_species):
        mask |= ((valid & (tn == sp)).any(1).astype(np.int64) << sp)
    gid = types.astype(np.int64) * (1 << s.n_species) + mask
    del valid, tn
    rows = ctx.rows()
    chunk = ctx.get_option(flare.OPT_CHUNK_ATOMS)
    present = [g for g in np.unique(gid)]
    groups = ctx.groups()
    assert sorted(int((gid == g).sum()) for g in present) == sorted(r for r, _ in groups if r), "group sizes"
    near_boundary = np.nonzero(((rows % chunk) < 2) | ((rows % chunk) >= chunk - 2))[0] if chunk < N else np.empty(0, np.int64)
    if chunk < N:
        assert near_boundary.size >= 4 * ((N - 1) // chunk)  # two rows on either side of every boundary (+ row 0, 1)
    per_ev = max(8, n_ev // len(present))
    per_f = max(4, n_f // len(present))
    sel_ev, sel_f = [near_boundary], [near_boundary]
    for g in present:
        members = np.nonzero(gid == g)[0]
        pick = rng.choice(members, min(per_ev, members.size), replace=False)
        sel_ev.append(pick)
        sel_f.append(pick[:per_f])
    sel_ev = np.unique(np.concatenate(sel_ev)).astype(np.int64)
    sel_f = np.unique(np.concatenate(sel_f)).astype(np.int64)
    assert sel_f.size >= min(n_f, 100) * 0.9 and sel_ev.size >= min(n_ev, 500) * 0.9
    # ---- E, V (cheap: no gradients) on the large sample, F on the smaller one
    sigma = s.sigma if want_var else None
    E, _, V = oracle.compute_selected(pos, types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, sigma, sel_ev, forces=False)
    assert_close(E_g[sel_ev], E, ATOL_E, "E")
    if want_var:
        assert_close(V_g[sel_ev], V, 1e-15, "V")
    # sum of the sampled local energies: the quantity an MD run conserves, summed independently on both sides
    assert abs(E_g[sel_ev].sum() - E.sum()) <= 1e-10 * np.abs(E).sum() + 1e-12
    _, F, _ = oracle.compute_selected(pos, types, s.box, s.pbc, s.n_max, s.l_max, s.r_cut, s.beta, None, sel_f)
    assert_close(F_g[sel_f], F, ATOL_F, "F")
    # ---- any-size properties
    assert np.abs(F_g.sum(0)).max() < 1e-6  # zero net force (translation invariance)
    assert np.isfinite(E_g).all() and np.isfinite(F_g).all() and (not want_var or np.isfinite(V_g).all())
    return dict(n_ev=int(sel_ev.size), n_f=int(sel_f.size), n_groups=len(present), chunk=int(chunk))


def md_then_check(oracle, torch, flare, s, variance, n_ev, n_f, n_brute, seed, steps=3, all_rows=True, **kw):
    """bench.py's launch configuration (default options): MD steps on a reused candidate list, then parity."""
    ctx = flare.from_system(s, variance=variance, **kw).bind(s.n_atoms)
    ctx.set_state(s.pos, s.vel, s.types, s.box, s.pbc)
    ctx.step(float(s.meta.get("dt_fs", 0.5)), steps, want_variance=variance)
    st = ctx.get_state_host(variances=variance)
    assert ctx.get_option(flare.OPT_SKIN_REBUILDS) < steps + 1  # steps + 1 evaluations, at least one on a reused list
    info = full_size_check(oracle, torch, flare, s, ctx, st["pos"], st["E"], st["F"], st["V"] if variance else None,
                           n_ev, n_f, n_brute, seed, all_rows=all_rows)
    return ctx, info


def test_config3_full_size_sampled(oracle, torch, flare):
    """BASELINE.json config 3 at full size (1 082 016 atoms, P = 544, variance on) in the launch configuration
    bench.py times (default options: species-sparse groups, skin list, automatic chunk), after MD steps so that the
    reused candidate list is what produced the neighbour sets.  Neighbour rows: ALL of them against the oracle's grid
    search and 1000 by brute force over all N; E, V of ~100 000 atoms and F of >= 100 atoms against
    the oracle one by one, from every group."""
    s = w.config3()
    ctx, info = md_then_check(oracle, torch, flare, s, True, n_ev=100_000, n_f=120, n_brute=1000, seed=33)
    groups = ctx.groups()
    assert sum(r for r, _ in groups) == s.n_atoms and {p for r, p in groups if r} == {144, 544}
    assert info["n_groups"] >= 4 and info["n_ev"] >= 50_000 and info["n_f"] >= 100


def test_config4_full_size_sampled(oracle, torch, flare):
    """BASELINE.json config 4 (9 994 400 atoms): the default options give several atom chunks (a8); after MD steps,
    ALL neighbour rows against the oracle's grid search and 200 by brute force over all N, E / V of ~100 000 atoms and
    F of >= 100 atoms (incl. the rows next to every chunk boundary) against the oracle; workspace bytes per atom."""
    s = w.config4()
    ctx, info = md_then_check(oracle, torch, flare, s, True, n_ev=100_000, n_f=120, n_brute=200, seed=44, steps=2)
    assert info["chunk"] < s.n_atoms  # several atom chunks
    per_atom = ctx.workspace_bytes(s.n_atoms) / s.n_atoms
    assert per_atom < 4096, per_atom      # 1.9 KB persistent + 16 GiB of chunk intermediates
    assert info["n_ev"] >= 50_000 and info["n_f"] >= 100


@pytest.mark.parametrize("variance", [True, False])
@pytest.mark.parametrize("n_max,l_max,P", [(10, 4, 1050), (12, 6, 2100)])
def test_config5_full_size_sampled(oracle, torch, flare, n_max, l_max, P, variance):
    """BASELINE.json config 5 at full size (1 082 016 atoms) for the two larger descriptor sizes, variance on and off,
    default options ((12,6) runs three atom chunks whose boundaries cut through groups), after 3 MD steps on a
    reused candidate list: sampled atoms of every group and next to every chunk boundary against the oracle."""
    s = w.config5(n_max, l_max)
    assert s.P == P
    if not variance:
        s.sigma = None
    n_ev = 3000 if P == 1050 else 1500
    ctx, info = md_then_check(oracle, torch, flare, s, variance, n_ev=n_ev, n_f=110, n_brute=150, seed=55 + l_max,
                              all_rows=(variance and P == 1050))
    assert {p for r, p in ctx.groups() if r} == {P, w.num_descriptors(1, n_max, l_max)}
    if P == 2100:
        assert info["chunk"] < s.n_atoms
    assert info["n_ev"] >= 500 and info["n_f"] >= 100


def test_isolated_atoms_in_sparse_mode(oracle, torch, flare):
    """Atoms without neighbours form an empty (species, mask=0) group: E = V = 0, no forces, no table reads."""
    rng = np.random.default_rng(51)
    box = np.diag([40.0, 40, 40]).reshape(9)
    pos = np.concatenate([rng.uniform(0, 40, (30, 3)), 20 + rng.uniform(-2.5, 2.5, (40, 3))])
    keep = [0]
    for i in range(1, len(pos)):
        if np.min(np.linalg.norm(pos[keep] - pos[i], axis=1)) > 1.0:
            keep.append(i)
    pos = pos[keep]
    types = rng.integers(0, 2, len(keep))
    s = _mk(pos, types, box, [1, 1, 1], 2, n_max=3, l_max=2, seed=52)
    ctx, got, want = assert_parity(oracle, torch, flare, s, nbr_method=0, species_sparse=True)
    cnt, _ = ctx.neighbors()
    assert (cnt == 0).sum() > 5 and (got[0][cnt == 0] == 0).all() and (got[1][cnt == 0] == 0).all()
