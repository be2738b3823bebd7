"""CPU-side checks of the product (no GPU): the C-ABI library loads and exports every symbol the
header declares, the binding fails loudly without a device, the workload generators follow their
recipe, and the product path never touches the oracle."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built_lib():
    from paper_2204_12573_b200 import build

    return build.build()


def test_library_exports_every_declared_symbol(built_lib):
    from paper_2204_12573_b200 import flare

    header = open(os.path.join(ROOT, "include", "flare_b200.h")).read()
    declared = set(re.findall(r"\b(flare_[a-z0-9_]+)\s*\(", header))
    declared.discard("flare_ctx")
    assert declared == set(flare.EXPORTS), declared ^ set(flare.EXPORTS)
    lib = ctypes.CDLL(built_lib)
    for name in declared:
        assert hasattr(lib, name), name


def test_probe_library_exports_every_declared_symbol(built_lib):
    """The bench hooks (include/flare_probes.h) live in a library of their own, outside the product ABI."""
    from paper_2204_12573_b200 import build, probes

    header = open(os.path.join(ROOT, "include", "flare_probes.h")).read()
    declared = set(re.findall(r"\b(flare_probe_[a-z0-9_]+)\s*\(", header))
    assert declared == set(probes.EXPORTS), declared ^ set(probes.EXPORTS)
    lib = ctypes.CDLL(build.PROBES_LIB)
    for name in declared:
        assert hasattr(lib, name), name
    product = ctypes.CDLL(built_lib)
    for name in declared:
        assert not hasattr(product, name), f"{name} leaked into the product ABI"


def test_binding_loads_and_create_fails_loudly_without_gpu(built_lib):
    import torch

    from paper_2204_12573_b200 import flare

    flare.load_library()
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(flare.FlareError) as ei:
        flare.Flare([195.0], 2, 1, [[4.0]], np.zeros((1, 6, 6)))
    assert ei.value.code == -6  # FLARE_ERR_CUDA: there is no CPU fallback


def test_create_validates_arguments_before_touching_cuda(built_lib):
    from paper_2204_12573_b200 import flare

    lib = flare.load_library()
    ctx = ctypes.c_void_p()
    m = np.array([1.0])
    rc_ = np.array([3.0])
    beta = np.zeros(36)
    p = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    assert lib.flare_create(ctypes.byref(ctx), 0, p(m), 2, 1, p(rc_), p(beta), None, 0) == -1
    assert lib.flare_create(ctypes.byref(ctx), 1, p(m), 2, 9, p(rc_), p(beta), None, 0) == -8
    assert lib.flare_create(ctypes.byref(ctx), 1, p(m), 99, 1, p(rc_), p(beta), None, 0) == -8
    assert lib.flare_create(ctypes.byref(ctx), 1, None, 2, 1, p(rc_), p(beta), None, 0) == -1
    assert lib.flare_workspace_bytes(None, 10) == 0
    assert lib.flare_bind(None, 10, None, 0, None) == -1


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2204_12573_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "flare_oracle" not in text and "import oracle" not in text and "from oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2204_12573_b200" not in text.replace("paper_2204_12573_b200/csrc", ""), f


def test_workload_recipes():
    from paper_2204_12573_b200 import workloads as w

    s1 = w.config1()
    assert s1.n_atoms == 256 and s1.P == 144 and s1.beta.shape == (1, 144, 144)
    assert abs(s1.box[0] - 15.68) < 1e-12
    s2 = w.config2()
    assert s2.n_atoms == 1264 and (s2.types == 0).sum() == 864 and s2.P == 544
    np.testing.assert_allclose(np.asarray(s2.box).reshape(3, 3).diagonal(), [33.2623, 28.8060, 31.3161], atol=1e-3)
    # seeded: same call, same arrays
    assert np.array_equal(w.config2().pos, s2.pos) and np.array_equal(w.config2().beta, s2.beta)
    # beta symmetric with spectral norm ~ 1 eV; sigma PSD ~ 1e-3
    assert np.allclose(s2.beta[0], s2.beta[0].T)
    assert 0.5 < np.abs(np.linalg.eigvalsh(s2.beta[1])).max() < 2.0
    ev = np.linalg.eigvalsh(s2.sigma[0])
    assert ev.min() > -1e-12 and 1e-3 < ev.max() < 1e-2
    # H2 bond length and separation rule
    h = s2.pos[864:]
    L = np.asarray(s2.box).reshape(3, 3).diagonal()
    d = h[0::2] - h[1::2]
    d -= L * np.round(d / L)
    np.testing.assert_allclose(np.linalg.norm(d, axis=1), 0.74, atol=1e-12)
    # temperature exactly 500 K with 3N-3 degrees of freedom, zero total momentum
    ke = w.kinetic_energy(s2.vel, s2.types, s2.mass)
    assert abs(2 * ke / ((3 * 1264 - 3) * w.KB) - 500.0) < 1e-9
    assert np.abs((s2.mass[s2.types][:, None] * s2.vel).sum(0)).max() < 1e-12
    # size bookkeeping of the big configs (not generated here)
    assert 2 * 408 * 204 * 6 + 2 * 41616 == 1082016
    assert 2 * 1240 * 620 * 6 + 2 * 384400 == 9994400
    assert [w.num_descriptors(2, a, b) for a, b in ((8, 3), (10, 4), (12, 6))] == [544, 1050, 2100]


def test_slab_geometry_is_fcc111():
    from paper_2204_12573_b200 import workloads as w

    pos, L, z_top = w.pt111_slab(6, 4, 6)
    from scipy.spatial import cKDTree

    tree = cKDTree(np.mod(pos, L), boxsize=L)
    d, _ = tree.query(np.mod(pos, L), k=13)
    nn = w.A_PT / np.sqrt(2)
    # every atom's nearest neighbours sit at a/sqrt2: 12 in the bulk layers, 9 on the two surfaces
    bulk = (pos[:, 2] > 1.0) & (pos[:, 2] < z_top - 1.0)
    assert np.allclose(d[bulk, 1:13], nn, atol=1e-9)
    assert np.allclose(d[~bulk, 1:10], nn, atol=1e-9) and np.all(d[~bulk, 10] > nn + 0.5)


def test_static_scratch_entry_point_constants_and_no_allocation_calls():
    """flare_virial_static (for callers that may not allocate): the limit in the header, in the binding and in the kernel
    file agree, and neither its translation unit nor its entry point names an allocating CUDA call."""
    from paper_2204_12573_b200 import flare

    header = open(os.path.join(ROOT, "include", "flare_b200.h")).read()
    limit = int(re.search(r"#define\s+FLARE_VIRIAL_STATIC_MAX_ATOMS\s+(\d+)", header).group(1))
    assert limit == flare.VIRIAL_STATIC_MAX_ATOMS == 2048 * 2048
    csrc = os.path.join(ROOT, "paper_2204_12573_b200", "csrc")
    unit = open(os.path.join(csrc, "virial_static.cu")).read()
    code = "\n".join(line.split("//")[0] for line in unit.splitlines())  # comments may name the calls it avoids
    assert re.search(r"static\s+__device__\s+__align__\(256\)\s+double\s+g_virial_rows\[", code)
    assert "cudaGetSymbolAddress" in code
    api = open(os.path.join(csrc, "flare_api.cu")).read()
    body = api[api.index("int flare_virial_static("):]
    body = body[:body.index("\n}\n")]
    for text in (code, body):
        for call in ("cudaMalloc", "cudaFree", "cudaMallocAsync", "cudaHostAlloc", "cub::", "thrust::"):
            assert call not in text, call
