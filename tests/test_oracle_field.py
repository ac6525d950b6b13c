"""Pins for the oracle's accelerations (NEXT-4: g = -grad Phi alongside Phi in the same
walk).  CPU only.  Pinned by: a numpy brute force, the numerical gradient of the
direct-sum potential, Newton's third law, the theta = 0 identity with the direct sum, convergence with
theta, the two-body closed form and the uniform-sphere field g(r) = -(4/3) pi G rho r."""
import numpy as np
import pytest

import bh_workloads as W


def _brute_acc(x, y, z, m, G=1.0):
    p = np.stack([x, y, z], axis=1)
    d = p[:, None, :] - p[None, :, :]                      # r_i - r_j
    r2 = (d ** 2).sum(-1)
    np.fill_diagonal(r2, np.inf)
    w = np.where(r2 > 0, m[None, :] / (r2 * np.sqrt(r2)), 0.0)
    return -G * (w[:, :, None] * d).sum(1)


def test_direct_acc_equals_numpy_bruteforce_and_two_body(oracle):
    w = W.random_points(300, seed=3)
    got = oracle.direct_acc(w.x, w.y, w.z, w.m, G=2.5)
    ref = _brute_acc(w.x, w.y, w.z, w.m, G=2.5)
    assert np.allclose(got, ref, rtol=1e-12, atol=1e-15)
    # two bodies on the x axis: g_0 = +G m_1/d^2 x^, g_1 = -G m_0/d^2 x^
    x = np.array([0.25, 0.75]); o = np.array([0.5, 0.5]); m = np.array([2.0, 3.0])
    g = oracle.direct_acc(x, o, o, m, G=1.0)
    assert np.allclose(g, [[3.0 / 0.25, 0, 0], [-2.0 / 0.25, 0, 0]], rtol=1e-15)
    # subset of targets
    sub = np.array([5, 17, 200], dtype=np.int64)
    assert np.array_equal(oracle.direct_acc(w.x, w.y, w.z, w.m, G=2.5, targets=sub), got[sub])


def test_direct_acc_is_minus_numerical_gradient_of_direct_phi(oracle):
    """Move one cell by +-h with all others fixed: (Phi(x+h) - Phi(x-h))/2h = -g_x to O(h^2)."""
    w = W.clustered_points(200, seed=8)
    g = oracle.direct_acc(w.x, w.y, w.z, w.m)
    h = 1e-6
    for i in (0, 57, 133):
        t = np.array([i], dtype=np.int64)
        for k, name in enumerate("xyz"):
            c = {n: getattr(w, n).copy() for n in "xyz"}
            c[name][i] += h
            up = oracle.direct(c["x"], c["y"], c["z"], w.m, targets=t)[0]
            c[name][i] -= 2 * h
            dn = oracle.direct(c["x"], c["y"], c["z"], w.m, targets=t)[0]
            assert -(up - dn) / (2 * h) == pytest.approx(g[i, k], rel=2e-5, abs=1e-7 * np.abs(g[i]).max())


def test_third_law_total_force_vanishes(oracle):
    w = W.clustered_points(500, seed=9)
    g = oracle.direct_acc(w.x, w.y, w.z, w.m)
    f = (w.m[:, None] * g).sum(0)
    assert np.abs(f).max() <= 1e-12 * np.abs(w.m[:, None] * g).sum()


@pytest.mark.parametrize("group", [1, 32])
def test_theta_zero_field_is_direct_sum(oracle, group):
    w = W.with_duplicates(W.clustered_points(400, seed=4), 20)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    phi, acc = t.field(0.0, w.G, group=group)
    assert np.allclose(phi, oracle.direct(w.x, w.y, w.z, w.m, w.G), rtol=1e-13)
    ref = oracle.direct_acc(w.x, w.y, w.z, w.m, w.G)
    assert np.allclose(acc, ref, rtol=1e-11, atol=1e-13 * np.abs(ref).max())
    # and Phi is the unchanged potential walk
    assert np.array_equal(phi, t.potential(0.0, w.G, group=group))


def test_field_converges_with_theta_and_phi_unchanged(oracle):
    w = W.clustered_points(3000, seed=5)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    ref = oracle.direct_acc(w.x, w.y, w.z, w.m, w.G)
    norm = np.linalg.norm(ref, axis=1)
    med, mx = [], []
    for theta in (1.0, 0.7, 0.5, 0.3, 0.1):
        phi, acc = t.field(theta, w.G, mac=1, group=1)
        assert np.array_equal(phi, t.potential(theta, w.G, mac=1, group=1))
        e = np.linalg.norm(acc - ref, axis=1) / norm
        med.append(np.median(e))
        mx.append(e.max())
    # monopole forces: ~theta^2 relative error; the maximum sits on cells where the field nearly cancels
    assert all(med[i + 1] < med[i] for i in range(4)) and all(mx[i + 1] < mx[i] for i in range(4)), (med, mx)
    assert med[0] < 5e-2 and med[2] < 1e-2 and med[-1] < 1e-4 and mx[-1] < 2e-3, (med, mx)
    # the group vote only refines every member's list
    _, a32 = t.field(0.5, w.G, mac=1, group=32)
    e32 = np.linalg.norm(a32 - ref, axis=1) / norm
    assert np.median(e32) <= med[2] and e32.max() <= mx[2]


def test_uniform_sphere_field_closed_form(oracle):
    """Inside a uniform sphere g = -(4/3) pi G rho (r - c); outside -G M (r - c)/|r - c|^3.  The 32^3
    point-mass sphere has a stair-cased surface, so the bar is a few per cent well inside / outside."""
    w = W.uniform_sphere(32)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _, acc = t.field(0.5, w.G, mac=1)
    p = np.stack([w.x, w.y, w.z], axis=1) - 0.5
    r = np.linalg.norm(p, axis=1)
    rho, R = 1.0, 0.4
    M = w.m.sum()
    inside = (r > 0.1) & (r < 0.3)
    g_in = -(4.0 / 3.0) * np.pi * w.G * rho * p[inside]
    err_in = np.linalg.norm(acc[inside] - g_in, axis=1) / np.linalg.norm(g_in, axis=1)
    assert np.median(err_in) < 1e-2 and err_in.max() < 8e-2, (np.median(err_in), err_in.max())
    outside = r > 0.5
    g_out = -w.G * M * p[outside] / r[outside, None] ** 3
    err_out = np.linalg.norm(acc[outside] - g_out, axis=1) / np.linalg.norm(g_out, axis=1)
    assert err_out.max() < 1e-2, err_out.max()
