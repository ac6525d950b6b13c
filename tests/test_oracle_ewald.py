"""Pins for the oracle's periodic-boundary functions (NEXT-3; App. A, Eq. A.1-A.3; DESIGN.md
readings P1-P5).  CPU only.  What the mathematics fixes about the Ewald sum of 1/r in a cubic box with a
neutralising background, none of it taken from the oracle's own formula:
  * psi does not depend on the splitting parameter alpha (checked over a decade of alpha);
  * differences psi(u1) - psi(u2) equal a brute-force lattice sum over spherical shells of images plus the
    background's (2 pi/3)(|u1|^2 - |u2|^2);
  * psi(u) - 1/|u| -> -2.8372974795 at u = 0, the Madelung-type constant of the simple cubic lattice
    (tests/golden/ewald_sc_constant.txt);
  * the mean of psi over the box is zero: the mean of corr1 = psi - 1/r equals minus the mean of 1/r over the
    unit cube, -2.3800774 (tests/golden/cube_self_potential.txt, already pinned by a brute-force quadrature);
  * the Laplacian of corr1 is 4 pi (the uniform background) everywhere inside the box;
  * cubic symmetry and periodicity;
  * a uniform grid of equal masses under periodic boundaries is a finer simple cubic lattice: Phi_i =
    +2.8372974795 G m N / L at every cell -- through the table, the interpolation, the wrap and the own-cell term.
"""
import os

import numpy as np
import pytest

import bh_workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden(fname, key):
    for line in open(os.path.join(GOLD, fname)):
        if not line.startswith("#") and line.strip():
            k, v = line.split()
            if k == key:
                return float(v)
    raise KeyError(key)


XI = _golden("ewald_sc_constant.txt", "xi_sc")             # 2.8372974795
CUBE = _golden("cube_self_potential.txt", "cube_self")     # 2.3800774

POINTS = [(0.31, 0.12, -0.07), (0.5, 0.5, 0.5), (0.05, 0.0, 0.0), (0.49, -0.2, 0.33), (0.25, 0.25, 0.0)]


def test_psi_is_independent_of_alpha(oracle):
    # a decade of the splitting parameter; enough terms for both sums at either end
    for u in POINTS:
        vals = [oracle.ewald_psi(u, a=a, nser=14) for a in (0.8, 1.3, 2.0, 3.1, 5.0, 8.0)]
        assert np.ptp(vals) <= 2e-11 * max(1.0, abs(vals[0])), (u, vals)


def test_psi_differences_equal_shell_summed_lattice_sum(oracle):
    # S(u) = sum over images |n| <= R of 1/|u - n| is conditionally convergent, but for cubic symmetry the
    # difference S(u1) - S(u2) + (2 pi/3)(|u1|^2 - |u2|^2) converges like 1/R^2 to psi(u1) - psi(u2)
    R = 60
    g = np.arange(-R, R + 1)
    n = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3).astype(np.float64)
    n = n[(n * n).sum(1) <= R * R]
    def S(u):
        return (1.0 / np.sqrt(((np.asarray(u) - n) ** 2).sum(1))).sum()
    for u1, u2 in ((POINTS[0], POINTS[3]), (POINTS[1], POINTS[2]), (POINTS[4], POINTS[0])):
        brute = S(u1) - S(u2) + 2 * np.pi / 3 * (np.dot(u1, u1) - np.dot(u2, u2))
        ewald = oracle.ewald_psi(u1) - oracle.ewald_psi(u2)
        assert abs(brute - ewald) <= 2e-3 * max(1.0, abs(ewald)), (u1, u2, brute, ewald)


def test_madelung_constant_zero_mean_and_laplacian(oracle):
    assert abs(oracle.ewald_corr((0.0, 0.0, 0.0)) + XI) <= 1e-9
    assert abs(oracle.ewald_corr((1e-4, 0.0, 0.0)) + XI) <= 1e-6          # continuous at the origin
    # mean over the box by the midpoint rule on the octant (corr1 is even): -mean(1/r over the unit cube)
    m = 24
    c = (np.arange(m) + 0.5) / (2 * m)
    mean = np.mean([oracle.ewald_corr((x, y, z), nser=4) for x in c for y in c for z in c])
    # the midpoint rule's leading error is -(h^2/24) mean(laplacian) = -(h^2/24) 4 pi (the Laplacian is pinned below)
    h = 1.0 / (2 * m)
    assert abs(mean + h * h / 24 * 4 * np.pi + CUBE) <= 3e-6, mean
    # Laplacian by central differences: the background's 4 pi, also right at a face of the box
    h = 1e-3
    for u in (POINTS[0], (0.5, 0.1, 0.2), (0.02, 0.03, 0.01)):
        lap = sum(oracle.ewald_corr(np.add(u, e)) + oracle.ewald_corr(np.subtract(u, e)) for e in np.eye(3) * h)
        lap = (lap - 6 * oracle.ewald_corr(u)) / h ** 2
        assert abs(lap - 4 * np.pi) <= 1e-3 * 4 * np.pi, (u, lap)


def test_symmetry_and_periodicity(oracle):
    u = np.array(POINTS[0])
    ref = oracle.ewald_psi(u)
    for perm in ((1, 0, 2), (2, 1, 0), (1, 2, 0)):
        for sgn in ((1, 1, -1), (-1, 1, 1), (-1, -1, -1)):
            assert abs(oracle.ewald_psi(u[list(perm)] * sgn) - ref) <= 1e-12
    for shift in ((1, 0, 0), (0, -1, 0), (1, 1, -1)):
        assert abs(oracle.ewald_psi(u + shift, nser=7) - oracle.ewald_psi(u, nser=7)) <= 1e-10
    assert abs(oracle.ewald_psi(u) - (oracle.ewald_corr(u) + 1 / np.linalg.norm(u))) <= 1e-13


@pytest.fixture(scope="module")
def table(oracle):
    return oracle.EwaldTable(N=34, nref=3)


def test_table_layout_and_interpolation_error(oracle, table):
    N = table.N
    for lev in range(table.nref):
        h = 0.5 / (N - 2) / 2 ** lev
        g = table.grid(lev)
        assert np.array_equal(g, g.transpose(1, 0, 2)) and np.array_equal(g, g.transpose(2, 1, 0))
        top = N - 2                               # a grid serves points whose nearest grid point is <= N - 2
        for (i, j, k) in ((0, 0, 0), (3, 1, 7), (N - 1, N - 1, N - 1), (N - 1, 0, 5)):
            assert abs(g[k, j, i] - oracle.ewald_corr((i * h, j * h, k * h))) <= 1e-12
            i, j, k = min(i, top), min(j, top), min(k, top)
            assert abs(table.interp((i * h, -j * h, k * h)) - g[k, j, i]) <= 1e-12       # exact at the grid points
    rng = np.random.default_rng(5)
    # a quadratic is reproduced to h^3: N = 34 (h = 1/64) gives ~1e-5 of psi's O(1) scale on the coarse grid, and the nested
    # grids are 8 and 64 times better near the origin
    for scale, tol in ((0.5, 6e-5), (0.25, 8e-6), (0.125, 1e-6)):
        u = rng.uniform(-scale, scale, (300, 3))
        err = max(abs(table.interp(p) - oracle.ewald_corr(p, nser=4)) for p in u)
        assert err <= tol, (scale, err)
    one = oracle.EwaldTable(N=34, nref=1)
    u = rng.uniform(-0.1, 0.1, (100, 3))
    assert max(abs(one.interp(p) - oracle.ewald_corr(p, nser=4)) for p in u) > \
        5 * max(abs(table.interp(p) - oracle.ewald_corr(p, nser=4)) for p in u)          # the nesting does refine


def test_uniform_periodic_grid_is_a_finer_cubic_lattice(oracle, table):
    # 8^3 equal masses in a periodic unit box: together with their images a simple cubic lattice of spacing 1/8
    ng = 8
    x, y, z = W._grid_centres(ng)
    m = np.full(x.size, 0.37)
    t = oracle.OracleTree(x, y, z, m, [0, 0, 0, 1.0])
    exact = XI * 0.37 * ng
    # (the net potential of a uniform periodic medium is what is left of a large cancellation -- the gross sum of
    #  |m psi| is ~50 times larger -- so the tree code's 1e-3 monopole errors show as per cent here)
    for theta, tol in ((0.0, 2e-4), (0.5, 5e-2)):
        phi = t.potential_periodic(theta, table, G=1.0)
        assert np.ptp(phi) <= 1e-9 * exact if theta == 0.0 else True     # every cell sees the same lattice
        assert np.max(np.abs(phi - exact)) <= tol * exact, (theta, phi[:3], exact)


@pytest.mark.parametrize("w", [W.random_points(300, seed=61), W.clustered_points(400, seed=62)], ids=lambda w: w.name)
def test_periodic_walk_against_the_exact_ewald_sum(oracle, table, w):
    """theta = 0 is the direct periodic sum through the table (interpolation error only); the tree code converges
    to it with theta; translating every point by the same vector (mod L) changes nothing."""
    L = float(w.cube[3])
    pos = np.stack([w.x, w.y, w.z], 1)
    exact = np.zeros(w.n)
    for i in range(0, w.n, 7):                                        # every 7th target: the exact sum is slow
        d = (pos[i] - pos) / L
        d -= np.rint(d)
        s = w.m[i] * oracle.ewald_corr((0, 0, 0), nser=4) / L
        for j in range(w.n):
            if j != i:
                s += w.m[j] * oracle.ewald_psi(d[j], nser=4) / L
        exact[i] = -w.G * s
    sel = np.arange(0, w.n, 7)
    # a periodic potential has zero mean: its values are what is left of a cancellation, so errors are measured
    # against the gross scale G M / L, not against the values themselves
    scale = w.G * w.m.sum() / L
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    phi0 = t.potential_periodic(0.0, table, G=w.G)
    assert np.max(np.abs(phi0[sel] - exact[sel])) <= 2e-5 * scale
    errs = [np.max(np.abs(t.potential_periodic(th, table, G=w.G, group=1)[sel] - exact[sel])) / scale for th in (1.0, 0.6, 0.3)]
    assert errs[0] > errs[1] > errs[2] and errs[2] <= 5e-3, errs   # large nodes near half the box converge slowly
    shift = np.array([0.37, 0.81, 0.12]) * L
    p2 = np.mod(pos - w.cube[:3] + shift, L) + w.cube[:3]
    t2 = oracle.OracleTree(p2[:, 0], p2[:, 1], p2[:, 2], w.m, w.cube)
    phi_shift = t2.potential_periodic(0.0, table, G=w.G)
    assert np.max(np.abs(phi_shift - phi0)) <= 2e-5 * scale
    # the isolated potential differs: the images and the background matter
    assert np.max(np.abs(t.potential(0.0, w.G) - phi0)) > 1e-1 * scale
