"""Pins for the oracle's walk and direct sum (W-rules; Eq. 2, 47 Eq. 3, 52 Eq. 4, 176).  CPU only."""
import numpy as np
import pytest

import bh_workloads as W
from tests import analytic as A


def numpy_direct(x, y, z, m, G=1.0):
    """Independent all-pairs sum (dense matrix), Eq. 2 without the printed 1/2."""
    d = np.sqrt((x[:, None] - x[None, :]) ** 2 + (y[:, None] - y[None, :]) ** 2 + (z[:, None] - z[None, :]) ** 2)
    with np.errstate(divide="ignore"):
        inv = np.where(d > 0, 1.0 / d, 0.0)
    return -G * (inv * m[None, :]).sum(axis=1)


def test_direct_hand_example(oracle):
    # three masses on a right triangle with legs 0.5: every distance is 0.5 or sqrt(0.5)
    x = np.array([0.25, 0.75, 0.25]); y = np.array([0.25, 0.25, 0.75]); z = np.array([0.25, 0.25, 0.25])
    m = np.array([1.0, 2.0, 3.0])
    phi = oracle.direct(x, y, z, m, G=2.0)
    r = np.sqrt(0.5)
    assert np.allclose(phi, [-2 * (2 / 0.5 + 3 / 0.5), -2 * (1 / 0.5 + 3 / r), -2 * (1 / 0.5 + 2 / r)], rtol=1e-15)
    # target subset, original indices
    assert np.array_equal(oracle.direct(x, y, z, m, G=2.0, targets=[2, 0]), phi[[2, 0]])


@pytest.mark.parametrize("w", [W.random_points(300, seed=11), W.clustered_points(257, seed=12),
                               W.with_duplicates(W.random_points(100, seed=13), 17)], ids=lambda w: w.name)
def test_direct_vs_numpy_and_theta0(oracle, w):
    ref = numpy_direct(w.x, w.y, w.z, w.m)
    phi_d = oracle.direct(w.x, w.y, w.z, w.m)
    assert np.allclose(phi_d, ref, rtol=1e-13, atol=0)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _, perm = t.sorted_keys_perm()
    for group in (1, 32):
        phi0, cnt = t.potential(0.0, group=group, want_counts=True)
        # theta = 0 opens everything: interaction set = all j != i, every cell reached as a leaf
        assert np.all(cnt[:, 0] == 0) and np.all(cnt[:, 1] == w.n)
        # the DFS visits sources in sorted order -> bit-equal to a sequential sum in that order
        xs, ys, zs, ms = w.x[perm], w.y[perm], w.z[perm], w.m[perm]
        for s in (0, 1, w.n // 2, w.n - 1):
            d2 = (xs[s] - xs) ** 2 + (ys[s] - ys) ** 2 + (zs[s] - zs) ** 2
            keep = d2 > 0
            keep[s] = False
            seq = np.cumsum(ms[keep] / np.sqrt(d2[keep]))[-1]
            assert phi0[perm[s]] == -seq
        assert np.allclose(phi0, ref, rtol=1e-13)


def test_accept_uses_centre_of_mass_and_counts(oracle):
    # a tight pair far from a lone target; theta = 1: the node holding the pair is accepted,
    # and the result is exactly -(m1+m2)/|r - com|  (com, not the geometric centre)
    x = np.array([0.0625, 0.1875, 0.9375]); y = np.array([0.0625, 0.0625, 0.9375]); z = np.array([0.0625, 0.0625, 0.9375])
    m = np.array([1.0, 3.0, 5.0])
    t = oracle.OracleTree(x, y, z, m, [0, 0, 0, 1.0])
    phi, cnt = t.potential(1.0, group=1, want_counts=True)
    com = np.array([(0.0625 + 3 * 0.1875) / 4, 0.0625, 0.0625])
    d = np.linalg.norm(np.array([0.9375] * 3) - com)
    _, perm = t.sorted_keys_perm()
    tgt = int(np.where(perm == 2)[0][0])
    assert phi[2] == -(4.0 / d)
    # root opened; the level-1 node (octant 0) holding the pair: l = 1/2, r_c = 1/2 < d -> accepted
    assert cnt[tgt].tolist() == [1, 1, 1]  # accepted level-1..2 node, own leaf cell, opened root
    # for the pair members the far cell is a leaf under the root: exact 1/r terms
    assert phi[0] == -(3.0 / 0.125 + 5.0 / np.linalg.norm([0.875, 0.875, 0.875]))


def test_strict_inequality_opens_on_tie(oracle):
    # node of size 1/2 with com (0.25,0.125,0.125); target at distance exactly 1/2; theta = 1 -> r_c = 1/2
    x = np.array([0.125, 0.375, 0.75]); y = np.array([0.125, 0.125, 0.125]); z = np.array([0.125, 0.125, 0.125])
    m = np.array([1.0, 1.0, 1.0])
    t = oracle.OracleTree(x, y, z, m, [0, 0, 0, 1.0])
    phi = t.potential(1.0, group=1)
    assert phi[2] == -(1 / 0.625 + 1 / 0.375)      # opened (d > r_c is false on a tie), not -(2/0.5)
    phi = t.potential(1.0001, group=1)
    assert phi[2] == -(2 / 0.5)                     # slightly larger theta: accepted


def test_eq4_opens_where_eq3_accepts(oracle):
    # com near the corner of a level-2 node: Eq. 3 accepts, Eq. 4 (extra delta) opens
    x = np.array([0.24, 0.12, 0.585]); y = np.array([0.24, 0.22, 0.24]); z = np.array([0.24, 0.24, 0.24])
    m = np.array([1.0, 1.0, 1e-3])
    t = oracle.OracleTree(x, y, z, m, [0, 0, 0, 1.0])
    nd = t.nodes()
    k = np.where(nd["level"] == 2)[0][0]
    d = np.linalg.norm([0.585 - nd["Rx"][k], 0.24 - nd["Ry"][k], 0.24 - nd["Rz"][k]])
    theta = 1.0
    assert 0.25 / theta < d < 0.25 / theta + nd["delta"][k] and d < 0.5
    _, perm = t.sorted_keys_perm()
    tgt = int(np.where(perm == 2)[0][0])
    p3, c3 = t.potential(theta, mac=oracle.MAC_BH86, group=1, want_counts=True)
    p4, c4 = t.potential(theta, mac=oracle.MAC_BARNES94, group=1, want_counts=True)
    assert c3[tgt].tolist() == [1, 1, 2] and p3[2] == -(2.0 / d)   # root + level-1 opened, level-2 accepted
    assert c4[tgt].tolist() == [0, 3, 3]
    assert p4[2] == oracle.direct(x, y, z, m)[2]


@pytest.mark.parametrize("w", [W.random_points(2000, seed=21), W.clustered_points(1500, seed=22)], ids=lambda w: w.name)
def test_convergence_with_theta(oracle, w):
    ref = oracle.direct(w.x, w.y, w.z, w.m)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    for mac in (oracle.MAC_BH86, oracle.MAC_BARNES94):
        errs1, errs32, rms1, ints1, ints32 = [], [], [], [], []
        for theta in (1.0, 0.7, 0.5, 0.3, 0.1):
            p1, c1 = t.potential(theta, mac=mac, group=1, want_counts=True)
            p32, c32 = t.potential(theta, mac=mac, group=32, want_counts=True)
            errs1.append(np.max(np.abs(p1 / ref - 1)))
            errs32.append(np.sqrt(np.mean((p32 / ref - 1) ** 2)))
            rms1.append(np.sqrt(np.mean((p1 / ref - 1) ** 2)))
            ints1.append((c1[:, 0] + c1[:, 1]).mean())
            ints32.append((c32[:, 0] + c32[:, 1]).mean())
        assert all(a > b for a, b in zip(errs1, errs1[1:])), errs1      # error falls monotonically with theta
        assert errs1[0] < 0.05 and errs1[2] < 5e-3 and errs1[-1] < 1e-4
        # group lists refine every member's own list: statistically (rms) the group error is not larger
        assert all(a <= b * 1.02 for a, b in zip(errs32, rms1)), (errs32, rms1)
        assert all(a < b for a, b in zip(ints1, ints1[1:]))                # work grows as theta falls
        assert all(a >= b for a, b in zip(ints32, ints1))


def test_group_partial_last_group_and_restricted_walk(oracle):
    w = W.random_points(70, seed=31)  # 3 groups of 32: 32 + 32 + 6
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    full, cnt = t.potential(0.6, want_counts=True)
    assert cnt.shape == (3, 3)
    part, c1 = t.potential(0.6, groups=(1, 3), want_counts=True)
    _, perm = t.sorted_keys_perm()
    assert np.all(np.isnan(part[perm[:32]])) and np.array_equal(part[perm[32:]], full[perm[32:]])
    assert np.array_equal(c1, cnt[1:])
    # n = 1: a lone leaf, Phi = 0
    t1 = oracle.OracleTree([0.3], [0.3], [0.3], [2.0], [0, 0, 0, 1.0])
    assert t1.n_nodes == 0 and t1.potential(0.5).tolist() == [0.0]


def test_mac_fp32_decisions_match_on_dyadic_grid(oracle):
    # lattice positions and centred coms are exact in fp32 and ties cannot occur: same lists
    x, y, z = W._grid_centres(16)
    t = oracle.OracleTree(x, y, z, np.full(x.size, 1.0 / x.size), [0, 0, 0, 1.0])
    for theta in (0.5, 1.0):
        p64, c64 = t.potential(theta, want_counts=True)
        p32, c32 = t.potential(theta, mac_fp32=True, want_counts=True)
        assert np.array_equal(c64, c32) and np.array_equal(p64, p32)
    w = W.turbulent_medium(16)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    c64 = t.potential(0.5, want_counts=True)[1]
    c32 = t.potential(0.5, mac_fp32=True, want_counts=True)[1]
    assert (c64 != c32).any(axis=1).mean() < 0.05  # flips are rare


# ---- pin of the oracle's mac_fp32 branch (W8) against tests/fp32_decision.py --------------------
@pytest.mark.parametrize("w", [W.random_points(1500, seed=41), W.clustered_points(1200, seed=42, ),
                               W.with_duplicates(W.random_points(300, seed=43), 25, near=2e-3)], ids=lambda w: w.name)
@pytest.mark.parametrize("theta,mac,group", [(0.7, 0, 32), (0.3, 1, 32), (0.45, 1, 1), (0.9, 0, 32)])
def test_mac_fp32_branch_equals_numpy_float32_restatement(oracle, w, theta, mac, group):
    """Non-dyadic inputs, 1/theta inexact in fp32: the per-group (accepted, leaf, opened) counters of the oracle's
    fp32-decision mode equal those of an independent numpy-float32 walk written from reading W8."""
    from tests import fp32_decision as F
    if group == 1 and w.n > 400:
        w = W.Workload(w.name + "_head", w.x[:400], w.y[:400], w.z[:400], w.m[:400], cube=w.cube)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _, perm = t.sorted_keys_perm()
    _, c32 = t.potential(theta, mac=mac, group=group, mac_fp32=True, want_counts=True)
    ref = F.walk_counts_fp32(w.x[perm], w.y[perm], w.z[perm], t.nodes(), float(w.cube[3]), theta, mac, group)
    assert np.array_equal(c32, ref)


def _threshold_scan(oracle, theta, mac, yz, accept_fn, level=2, steps=160):
    """A tight pair (a chain of nodes with one centre of mass R) and a lone target whose x runs through
    consecutive fp32 values across the distance at which the level-`level` node of the chain switches from
    opened to accepted.  Returns (oracle decisions, decisions of `accept_fn`) per step, True = accepted."""
    px = np.array([0.13, 0.17]); py = np.array([0.11, 0.12]); pz = np.array([0.09, 0.10]); pm = np.array([1.0, 2.3])
    R = np.array([(px * pm).sum(), (py * pm).sum(), (pz * pm).sum()]) / pm.sum()
    size = 2.0 ** -level
    rc = size / theta + (np.linalg.norm(R - (np.floor(R / size) + 0.5) * size) if mac == 1 else 0.0)
    ty, tz = yz
    x0 = np.float32(R[0] + np.sqrt(rc * rc - (ty - R[1]) ** 2 - (tz - R[2]) ** 2))
    xs = [x0]
    for _ in range(steps // 2):
        xs.insert(0, np.nextafter(xs[0], np.float32(-1))); xs.append(np.nextafter(xs[-1], np.float32(2)))
    got, ref = [], []
    for xt in xs:
        x = np.append(px, float(xt)); y = np.append(py, ty); z = np.append(pz, tz); m = np.append(pm, 0.7)
        t = oracle.OracleTree(x, y, z, m, [0, 0, 0, 1.0])
        _, perm = t.sorted_keys_perm()
        s = int(np.where(perm == 2)[0][0])
        _, c = t.potential(theta, mac=mac, group=1, mac_fp32=True, want_counts=True)
        nd = t.nodes()
        k = int(np.where(nd["level"] == level)[0][0])
        # root .. level-1 are opened for this target (d < their r_c); the chain node at `level` decides
        assert c[s, 2] in (level, level + 1) and c[s, 0] == 1
        got.append(c[s, 2] == level)
        ref.append(accept_fn(np.float32(xt), np.float32(ty), np.float32(tz), (nd["Rx"][k], nd["Ry"][k], nd["Rz"][k]),
                             size, nd["delta"][k], theta, mac))
    return np.array(got), np.array(ref)


def test_mac_fp32_branch_at_the_threshold(oracle):
    """One-ulp steps of a target across r_c: the oracle's fp32 decision equals the restatement at EVERY step, and
    the plausible mistakes -- l/theta instead of l*(1/theta), the fma chain nested the other way round, unfused
    multiply-adds, the decision taken in fp64 -- each disagree with the oracle at some step, so this pin would
    catch them."""
    from tests import fp32_decision as F
    f32 = np.float32

    def w8(tx, ty, tz, R, size, delta, theta, mac):
        return F.group_accepts_fp32([tx], [ty], [tz], R, size, delta, theta, mac)

    def div_theta(tx, ty, tz, R, size, delta, theta, mac):
        rc = f32(f32(size) / f32(theta))
        rc = f32(rc + f32(delta)) if mac == 1 else rc
        return bool(F.d2_fp32([tx], [ty], [tz], R)[0] > f32(rc * rc))

    def nest_x_last(tx, ty, tz, R, size, delta, theta, mac):
        dx, dy, dz = (f32(f32(a) - f32(b)) for a, b in zip((tx, ty, tz), R))
        d2 = F.fma32(dx, dx, F.fma32(dy, dy, f32(dz * dz)))
        return bool(d2 > F.rc2_fp32(size, delta, theta, mac))

    def unfused(tx, ty, tz, R, size, delta, theta, mac):
        dx, dy, dz = (f32(f32(a) - f32(b)) for a, b in zip((tx, ty, tz), R))
        d2 = f32(f32(f32(dx * dx) + f32(dy * dy)) + f32(dz * dz))
        return bool(d2 > F.rc2_fp32(size, delta, theta, mac))

    def in_fp64(tx, ty, tz, R, size, delta, theta, mac):
        rc = size / theta + (delta if mac == 1 else 0.0)
        d2 = sum((float(a) - float(b)) ** 2 for a, b in zip((tx, ty, tz), R))
        return d2 > rc * rc

    variants = {"div_theta": div_theta, "nest_x_last": nest_x_last, "unfused": unfused, "in_fp64": in_fp64}
    caught = {k: 0 for k in variants}
    for theta, mac, yz in ((0.7, 0, (0.3141, 0.2718)), (0.3, 1, (0.4567, 0.3789)), (0.9, 1, (0.2222, 0.3333)),
                           (0.55, 0, (0.19, 0.41)), (0.35, 0, (0.6180339, 0.5772156)), (0.77, 1, (0.33, 0.07)),
                           (0.62, 0, (0.2468, 0.1357)), (0.41, 1, (0.52, 0.23)), (0.83, 0, (0.05, 0.31)),
                           (0.48, 0, (0.3775, 0.4425)), (0.66, 1, (0.1414, 0.1732)), (0.37, 1, (0.29, 0.61))):
        got, ref = _threshold_scan(oracle, theta, mac, yz, w8)
        assert got[0] != got[-1]                               # the scan does cross the threshold
        assert np.array_equal(got, ref), (theta, mac)
        for name, fn in variants.items():
            _, alt = _threshold_scan(oracle, theta, mac, yz, fn)
            caught[name] += int(np.sum(alt != got))
    assert all(v > 0 for v in caught.values()), caught


def test_uniform_sphere_closed_form(oracle):
    # configs[0] at 32^3: direct sum vs -2 pi G rho (R^2 - r^2/3) inside, -GM/r outside
    w = W.uniform_sphere(32)
    rng = np.random.default_rng(0)
    r = np.sqrt((w.x - .5) ** 2 + (w.y - .5) ** 2 + (w.z - .5) ** 2)
    inside = np.where(r < 0.3)[0]
    outside = np.where(r > 0.55)[0]
    tg = np.concatenate([rng.choice(inside, 150, replace=False), rng.choice(outside, 150, replace=False)])
    phi = oracle.direct(w.x, w.y, w.z, w.m, targets=tg)
    phi = phi - A.CUBE_SELF * w.m[tg] / w.meta["dx"]  # the cell's own uniform-cube self term (test side only)
    M_disc = w.m.sum()
    ana = A.sphere_potential(r[tg], 0.4)
    err = np.abs(phi / ana - 1)
    assert err[:150].max() < 1.5e-2 and err[150:].max() < 1.0e-2  # binary-filled sphere: 1e-2 level
    # outside, with the discrete mass instead of the continuum mass, Newton's shell theorem holds to 1e-4
    assert np.abs(phi[150:] / (-M_disc / r[tg][150:]) - 1).max() < 2e-4
    # and the sign/factor: a BH walk at theta=0.5 stays within 1 % of direct
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    bh = t.potential(0.5)[tg] - A.CUBE_SELF * w.m[tg] / w.meta["dx"]
    assert np.abs(bh / phi - 1).max() < 1e-2


def test_maclaurin_closed_forms_selfconsistent():
    e, a1 = 0.9, 0.4
    A1, A3 = A.maclaurin_A(e)
    a3 = a1 * np.sqrt(1 - e * e)
    assert abs(2 * A1 + A3 - 2) < 1e-14                       # Chandrasekhar's identity
    assert abs(a3 - 0.174355958) < 1e-9 and abs(A1 - 0.434974233) < 1e-9 and abs(A3 - 1.130051535) < 1e-9
    assert abs(A.maclaurin_interior(0, 0, 0, a1, e) + 0.5452087) < 1e-7
    # continuity interior/exterior on the surface, and far field -> -GM/r
    for th in np.linspace(0, np.pi / 2, 7):
        xs, zs = a1 * np.sin(th), a3 * np.cos(th)
        assert abs(A.maclaurin_interior(xs, 0, zs, a1, e) - A.maclaurin_exterior(xs, 0, zs, a1, e)) < 1e-12
    M = 4 / 3 * np.pi * a1 * a1 * a3
    for p in ((30.0, 0, 0), (0, 0, 30.0), (20.0, 10.0, 15.0)):
        r = np.linalg.norm(p)
        assert abs(A.maclaurin_exterior(*p, a1, e) / (-M / r) - 1) < 1e-4
    # e -> 0 limit is the sphere
    assert abs(A.maclaurin_interior(0.1, 0.2, 0.05, 0.4, 1e-4) - A.sphere_potential(np.sqrt(0.0525), 0.4)) < 1e-8


def test_maclaurin_spheroid_direct_sum(oracle):
    # configs[1] shape at 64^3 (the oracle's direct sum on 400 sampled targets): interior and exterior
    w = W.maclaurin_spheroid(64)
    e, a1, a3 = w.meta["ecc"], w.meta["a1"], w.meta["a3"]
    X, Y, Z = w.x - .5, w.y - .5, w.z - .5
    s = (X * X + Y * Y) / a1 ** 2 + Z * Z / a3 ** 2
    rng = np.random.default_rng(3)
    tin = rng.choice(np.where(s < 0.6)[0], 200, replace=False)
    tout = rng.choice(np.where(s > 1.6)[0], 200, replace=False)
    tg = np.concatenate([tin, tout])
    phi = oracle.direct(w.x, w.y, w.z, w.m, targets=tg) - A.CUBE_SELF * w.m[tg] / w.meta["dx"]
    ana = np.concatenate([A.maclaurin_interior(X[tin], Y[tin], Z[tin], a1, e), A.maclaurin_exterior(X[tout], Y[tout], Z[tout], a1, e)])
    err = np.abs(phi / ana - 1)  # Eq. 13
    assert err.max() < 1e-3, err.max()   # paper's own direct sum: 2.17e-4 on a finer mesh
    # the printed (uncorrected) Eq. 6 would be off by tens of per cent: make sure this pin can tell
    A1, A3 = A.maclaurin_A(e)
    printed = -np.pi * (2 * A1 * a1 ** 2 - A1 * (X[tin] ** 2 + Y[tin] ** 2) - A3 * (a3 ** 2 - Z[tin] ** 2))
    assert np.abs(phi[:200] / printed - 1).min() > 0.05


def test_golden_constants_rederived():
    import os
    g = {}
    for f in ("maclaurin_e0.9.txt", "cube_self_potential.txt"):
        for line in open(os.path.join(os.path.dirname(__file__), "golden", f)):
            if not line.startswith("#") and line.strip():
                k, v = line.split()
                g[k] = float(v)
    A1, A3 = A.maclaurin_A(0.9)
    a3 = 0.4 * np.sqrt(1 - 0.81)
    assert abs(g["a3"] - a3) < 1e-9 and abs(g["A1"] - A1) < 1e-9 and abs(g["A3"] - A3) < 1e-9
    assert abs(g["abs_phi_centre"] - np.pi * (2 * A1 * 0.16 + A3 * a3 ** 2)) < 1e-7
    assert abs(g["cube_self"] - A.CUBE_SELF) < 1e-7
    # brute-force check of the cube constant: midpoint rule on a fine sub-grid (excluding nothing: integrable)
    n = 60
    c = (np.arange(n) + 0.5) / n - 0.5
    X, Y, Z = np.meshgrid(c, c, c, indexing="ij")
    assert abs((1 / np.sqrt(X * X + Y * Y + Z * Z)).mean() - A.CUBE_SELF) < 2e-3
