"""Pins for the oracle's basis functions and descriptor (SURVEY.md 8(c) "What pins each part").

Every expected value here comes from the paper, a closed form, or an independent library
routine (scipy / numpy) -- never from the oracle itself or from the CUDA path.
"""
import os

import numpy as np
import pytest
from scipy.spatial.transform import Rotation
from scipy.special import eval_legendre, sph_harm_y

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- P and index structure


def test_descriptor_dimension_paper(oracle):
    """420 components with two species, 112 with one."""
    for line in open(os.path.join(GOLDEN, "paper_dims.txt")):
        if line.startswith("#") or not line.strip():
            continue
        S, n_max, l_max, P = map(int, line.split())
        assert oracle.num_descriptors(S, n_max, l_max) == P


@pytest.mark.parametrize("S,n_max,l_max,P", [(1, 8, 3, 144), (2, 8, 3, 544), (2, 10, 4, 1050), (2, 12, 6, 2100)])
def test_descriptor_dimension_configs(oracle, S, n_max, l_max, P):
    """BASELINE.json configs state P=144 and P=544; SURVEY 8 derives 1050 and 2100."""
    assert oracle.num_descriptors(S, n_max, l_max) == P


def test_b2_index_is_a_bijection_in_order(oracle):
    S, n_max, l_max = 2, 3, 2
    Nv, L = S * n_max, l_max + 1
    seen = []
    for v1 in range(Nv):
        for v2 in range(v1, Nv):
            for l in range(L):
                seen.append(oracle.b2_index(S, n_max, l_max, v1, v2, l))
    assert seen == list(range(oracle.num_descriptors(S, n_max, l_max)))


# ----------------------------------------------------------------------------- radial basis


def test_chebyshev_closed_forms(oracle):
    n_max = 12
    n = np.arange(n_max)
    for theta in np.linspace(0.05, 3.1, 17):
        T, dT = oracle.chebyshev(n_max, np.cos(theta))
        np.testing.assert_allclose(T, np.cos(n * theta), atol=2e-13)
        # d/dx cos(n acos x) = n sin(n theta)/sin(theta)
        np.testing.assert_allclose(dT, n * np.sin(n * theta) / np.sin(theta), atol=2e-11)
    T, dT = oracle.chebyshev(n_max, 1.0)
    np.testing.assert_allclose(T, 1.0)
    np.testing.assert_allclose(dT, n.astype(float) ** 2)
    T, _ = oracle.chebyshev(n_max, -1.0)
    np.testing.assert_allclose(T, (-1.0) ** n)


def test_chebyshev_vs_numpy_polynomial(oracle):
    from numpy.polynomial import chebyshev as cheb

    n_max = 10
    for x in [-0.93, -0.2, 0.0, 0.41, 0.999]:
        T, dT = oracle.chebyshev(n_max, x)
        for k in range(n_max):
            c = np.zeros(k + 1)
            c[k] = 1.0
            assert abs(T[k] - cheb.chebval(x, c)) < 1e-13
            assert abs(dT[k] - cheb.chebval(x, cheb.chebder(c))) < 1e-11


def test_cutoff_closed_forms(oracle):
    rc = 4.25
    f0, d0 = oracle.cutoff(0.0, rc)
    fh, dh = oracle.cutoff(rc / 2, rc)
    f1, d1 = oracle.cutoff(rc, rc)
    assert f0 == 1.0 and abs(d0) < 1e-16
    assert abs(fh - 0.5) < 1e-16 and abs(dh + np.pi / (2 * rc)) < 1e-15
    assert abs(f1) < 1e-16 and abs(d1) < 1e-15
    fq, _ = oracle.cutoff(rc / 3, rc)
    assert abs(fq - 0.75) < 1e-15  # 1/2 (1 + cos(pi/3))


def test_radial_is_chebyshev_times_cutoff_and_derivative(oracle):
    rc, n_max = 3.0, 8
    for r in [0.4, 0.74, 1.7, 2.95]:
        g, dg = oracle.radial(n_max, r, rc)
        x = 2 * r / rc - 1
        np.testing.assert_allclose(g, np.cos(np.arange(n_max) * np.arccos(x)) * 0.5 * (1 + np.cos(np.pi * r / rc)),
                                   atol=1e-13)
        h = 1e-5
        gp, _ = oracle.radial(n_max, r + h, rc)
        gm, _ = oracle.radial(n_max, r - h, rc)
        gp2, _ = oracle.radial(n_max, r + h / 2, rc)
        gm2, _ = oracle.radial(n_max, r - h / 2, rc)
        fd = (4 * (gp2 - gm2) / h - (gp - gm) / (2 * h)) / 3
        np.testing.assert_allclose(dg, fd, atol=2e-9)
    # x = 2r/rc - 1 reaches +1 at the cutoff where every g~_n vanishes with zero slope in f_c
    g, dg = oracle.radial(n_max, rc, rc)
    np.testing.assert_allclose(g, 0.0, atol=1e-15)


# ----------------------------------------------------------------------------- spherical harmonics


def _unit(rng, k):
    v = rng.standard_normal((k, 3))
    return v / np.linalg.norm(v, axis=1)[:, None]


def _real_from_scipy(l_max, u):
    """Real orthonormal Y_lm built from scipy's complex (Condon-Shortley) Y_l^m:
    Y_l,+m = sqrt2 (-1)^m Re Y_l^m, Y_l,-m = sqrt2 (-1)^m Im Y_l^m (index l*l + l + m)."""
    theta = np.arccos(np.clip(u[2], -1, 1))
    phi = np.arctan2(u[1], u[0])
    out = np.zeros((l_max + 1) ** 2)
    for l in range(l_max + 1):
        out[l * l + l] = sph_harm_y(l, 0, theta, phi).real
        for m in range(1, l + 1):
            y = sph_harm_y(l, m, theta, phi)
            out[l * l + l + m] = np.sqrt(2) * (-1) ** m * y.real
            out[l * l + l - m] = np.sqrt(2) * (-1) ** m * y.imag
    return out


def test_ylm_vs_scipy(oracle):
    rng = np.random.default_rng(1)
    l_max = 6
    for u in _unit(rng, 25):
        Y, _ = oracle.ylm(l_max, u)
        np.testing.assert_allclose(Y, _real_from_scipy(l_max, u), atol=5e-14)


def test_ylm_y00_and_poles(oracle):
    for u in ([0, 0, 1.0], [0, 0, -1.0], [1.0, 0, 0]):
        Y, dY = oracle.ylm(6, u)
        assert abs(Y[0] - 1 / np.sqrt(4 * np.pi)) < 1e-16
        assert np.all(np.isfinite(Y)) and np.all(np.isfinite(dY))
    # on +z only m = 0 survives and Y_l0 = sqrt((2l+1)/4pi)
    Y, _ = oracle.ylm(6, [0, 0, 1.0])
    for l in range(7):
        for m in range(-l, l + 1):
            want = np.sqrt((2 * l + 1) / (4 * np.pi)) if m == 0 else 0.0
            assert abs(Y[l * l + l + m] - want) < 1e-14


def test_ylm_orthonormal_by_quadrature(oracle):
    l_max = 6
    L2 = (l_max + 1) ** 2
    t, w = np.polynomial.legendre.leggauss(l_max + 2)
    nphi = 2 * l_max + 3
    G = np.zeros((L2, L2))
    for ti, wi in zip(t, w):
        s = np.sqrt(1 - ti * ti)
        for k in range(nphi):
            phi = 2 * np.pi * k / nphi
            Y, _ = oracle.ylm(l_max, [s * np.cos(phi), s * np.sin(phi), ti])
            G += wi * (2 * np.pi / nphi) * np.outer(Y, Y)
    np.testing.assert_allclose(G, np.eye(L2), atol=2e-13)


def test_ylm_addition_theorem_and_unsold(oracle):
    rng = np.random.default_rng(2)
    l_max = 6
    a, b = _unit(rng, 12), _unit(rng, 12)
    for ua, ub in zip(a, b):
        Ya, _ = oracle.ylm(l_max, ua)
        Yb, _ = oracle.ylm(l_max, ub)
        for l in range(l_max + 1):
            sl = slice(l * l, (l + 1) ** 2)
            want = (2 * l + 1) / (4 * np.pi) * eval_legendre(l, float(ua @ ub))
            assert abs(Ya[sl] @ Yb[sl] - want) < 1e-13
            assert abs(Ya[sl] @ Ya[sl] - (2 * l + 1) / (4 * np.pi)) < 1e-13


def test_ylm_gradient_projected_matches_finite_difference(oracle):
    """grad Y_lm(r) = (1/r)(I - u u^T) grad_u Y~: compare with central differences of Y(r/|r|)."""
    rng = np.random.default_rng(3)
    l_max = 6
    pts = list(_unit(rng, 6) * rng.uniform(0.7, 3.0, (6, 1))) + [np.array([0.0, 0.0, 1.3]), np.array([0, 0, -2.0])]
    for r in pts:
        rn = np.linalg.norm(r)
        u = r / rn
        _, dY = oracle.ylm(l_max, u)
        grad = (dY - np.outer(dY @ u, u)) / rn
        h = 1e-5
        for d in range(3):
            e = np.zeros(3)
            e[d] = h
            Yp, _ = oracle.ylm(l_max, (r + e) / np.linalg.norm(r + e))
            Ym, _ = oracle.ylm(l_max, (r - e) / np.linalg.norm(r - e))
            np.testing.assert_allclose(grad[:, d], (Yp - Ym) / (2 * h), atol=5e-9)


# ----------------------------------------------------------------------------- A and B2


def _random_env(rng, M, S, rmin=0.8, rmax=2.9):
    rij = _unit(rng, M) * rng.uniform(rmin, rmax, (M, 1))
    sj = rng.integers(0, S, M).astype(np.int32)
    return rij, sj


def test_A_single_neighbour_on_z(oracle):
    n_max, l_max, rc = 8, 3, 4.25
    r = 2.77
    A, B, Bh, nrm = oracle.descriptor_env(1, n_max, l_max, [[rc]], 0, [[0, 0, r]], [0])
    g = np.cos(np.arange(n_max) * np.arccos(2 * r / rc - 1)) * 0.5 * (1 + np.cos(np.pi * r / rc))
    for n in range(n_max):
        for l in range(l_max + 1):
            for m in range(-l, l + 1):
                want = g[n] * np.sqrt((2 * l + 1) / (4 * np.pi)) if m == 0 else 0.0
                assert abs(A[n, l * l + l + m] - want) < 1e-14
    # single neighbour => B[n1,n2,l] = g_n1 g_n2 (2l+1)/4pi  (true for most gas-phase H)
    p = 0
    for n1 in range(n_max):
        for n2 in range(n1, n_max):
            for l in range(l_max + 1):
                assert abs(B[p] - g[n1] * g[n2] * (2 * l + 1) / (4 * np.pi)) < 1e-14
                p += 1
    assert abs(np.linalg.norm(Bh) - 1) < 1e-14 and abs(nrm - np.linalg.norm(B)) < 1e-14


def _b2_legendre_pair_sum(S, n_max, l_max, r_cut, si, rij, sj):
    """B[nu1,nu2,l] = (2l+1)/(4pi) sum_{j in s1} sum_{k in s2} g~_n1(r_j) g~_n2(r_k) P_l(u_j.u_k):
    an O(M^2) route that never forms Y_lm or A (addition theorem)."""
    r_cut = np.asarray(r_cut, float).reshape(S, S)
    M = len(sj)
    r = np.linalg.norm(rij, axis=1)
    u = rij / r[:, None]
    g = np.zeros((M, n_max))
    for j in range(M):
        rc = r_cut[si, sj[j]]
        g[j] = np.cos(np.arange(n_max) * np.arccos(np.clip(2 * r[j] / rc - 1, -1, 1))) * 0.5 * (1 + np.cos(np.pi * r[j] / rc))
    cosg = np.clip(u @ u.T, -1, 1)
    Nv = S * n_max
    out = []
    for v1 in range(Nv):
        s1, n1 = divmod(v1, n_max)
        for v2 in range(v1, Nv):
            s2, n2 = divmod(v2, n_max)
            for l in range(l_max + 1):
                w = np.outer(g[:, n1] * (sj == s1), g[:, n2] * (sj == s2))
                out.append((2 * l + 1) / (4 * np.pi) * np.sum(w * eval_legendre(l, cosg)))
    return np.array(out)


@pytest.mark.parametrize("S,n_max,l_max,M", [(1, 8, 3, 18), (2, 8, 3, 14), (2, 4, 6, 9), (3, 2, 2, 7)])
def test_B2_vs_legendre_pair_sum(oracle, S, n_max, l_max, M):
    rng = np.random.default_rng(10 + S + l_max)
    r_cut = np.full((S, S), 3.0)
    r_cut[0, 0] = 4.25
    rij, sj = _random_env(rng, M, S)
    for si in range(S):
        A, B, Bh, nrm = oracle.descriptor_env(S, n_max, l_max, r_cut, si, rij, sj)
        want = _b2_legendre_pair_sum(S, n_max, l_max, r_cut, si, rij, sj)
        np.testing.assert_allclose(B, want, atol=2e-13 * max(1.0, np.abs(want).max()))
        np.testing.assert_allclose(Bh, want / np.linalg.norm(want), atol=1e-13)


def test_B2_l0_closed_form(oracle):
    rng = np.random.default_rng(5)
    n_max, l_max = 5, 2
    rij, sj = _random_env(rng, 11, 1)
    A, B, _, _ = oracle.descriptor_env(1, n_max, l_max, [[3.0]], 0, rij, sj)
    r = np.linalg.norm(rij, axis=1)
    g = np.cos(np.outer(np.arccos(2 * r / 3.0 - 1), np.arange(n_max))) * (0.5 * (1 + np.cos(np.pi * r / 3.0)))[:, None]
    sg = g.sum(0)
    for n1 in range(n_max):
        for n2 in range(n1, n_max):
            p = oracle.b2_index(1, n_max, l_max, n1, n2, 0)
            assert abs(B[p] - sg[n1] * sg[n2] / (4 * np.pi)) < 1e-13


def test_B2_invariances(oracle):
    rng = np.random.default_rng(6)
    S, n_max, l_max = 2, 6, 4
    r_cut = [[4.25, 3.0], [3.0, 3.0]]
    rij, sj = _random_env(rng, 13, S)
    _, B0, _, _ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, rij, sj)
    scale = np.abs(B0).max()
    for R in Rotation.random(4, random_state=7):
        _, B1, _, _ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, R.apply(rij), sj)
        np.testing.assert_allclose(B1, B0, atol=2e-13 * scale)
    _, B2, _, _ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, -rij, sj)  # inversion
    np.testing.assert_allclose(B2, B0, atol=2e-13 * scale)
    perm = rng.permutation(len(sj))
    _, B3, _, _ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, rij[perm], sj[perm])
    np.testing.assert_allclose(B3, B0, atol=2e-13 * scale)
    # A itself is NOT invariant (equivariant basis): a rotation must change it
    A0, *_ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, rij, sj)
    A1, *_ = oracle.descriptor_env(S, n_max, l_max, r_cut, 0, Rotation.random(random_state=9).apply(rij), sj)
    assert np.abs(A0 - A1).max() > 1e-3


def test_descriptor_translation_invariance_in_a_system(oracle):
    from paper_2204_12573_b200 import workloads as w

    s = w.config1(with_model=False)
    i = 17
    _, B0, _, _ = oracle.descriptor(s.pos, s.types, s.box, s.pbc, 4, 3, s.r_cut, i)
    shift = np.array([3.3, -7.9, 21.0])
    _, B1, _, _ = oracle.descriptor(s.pos + shift, s.types, s.box, s.pbc, 4, 3, s.r_cut, i)
    np.testing.assert_allclose(B1, B0, atol=1e-11 * np.abs(B0).max())


def test_species_blocks_are_zero_for_absent_species(oracle):
    """with neighbours of one species only, every component touching the other
    species' radial channels vanishes (the 420 -> 112 statement)."""
    rng = np.random.default_rng(8)
    S, n_max, l_max = 2, 7, 3
    rij, _ = _random_env(rng, 12, 1)
    sj = np.zeros(12, np.int32)
    _, B, _, _ = oracle.descriptor_env(S, n_max, l_max, [[4.25, 3.0], [3.0, 3.0]], 0, rij, sj)
    nz = 0
    for v1 in range(S * n_max):
        for v2 in range(v1, S * n_max):
            for l in range(l_max + 1):
                p = oracle.b2_index(S, n_max, l_max, v1, v2, l)
                if v1 < n_max and v2 < n_max:
                    nz += 1
                else:
                    assert B[p] == 0.0
    assert nz == 112 and B.size == 420
