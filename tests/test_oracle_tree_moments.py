"""Pins for the oracle's octree and monopoles (T-rules, M-rules).  CPU only."""
import math

import numpy as np
import pytest

import bh_workloads as W


def brute_tree(x, y, z, cube):
    """Recursive partition on quantised integer coordinates (no Morton keys): returns
    {(level, (px,py,pz)): frozenset(original indices)} for every sub-cube holding >= 2 points,
    levels 0..20, plus level-21 entries for >= 2 points in the same finest cell."""
    s = 2097152.0 / cube[3]
    q = np.stack([np.clip(np.floor((np.asarray(v) - c0) * s), 0, 2097151).astype(np.int64)
                  for v, c0 in zip((x, y, z), cube[:3])], axis=1)
    out = {}

    def rec(level, idx):
        if len(idx) < 2:
            return
        sh = 21 - level
        out[(level, tuple((q[idx[0]] >> sh).tolist()))] = frozenset(idx.tolist())
        if level == 21:
            return
        sub = q[idx] >> (sh - 1)
        code = (sub[:, 0] & 1) + 2 * (sub[:, 1] & 1) + 4 * (sub[:, 2] & 1)
        for o in range(8):
            rec(level + 1, idx[code == o])

    rec(0, np.arange(len(x)))
    return out


def deinterleave(prefix, level):
    p = [0, 0, 0]
    for k in range(level):
        for a in range(3):
            p[a] |= ((int(prefix) >> (3 * k + a)) & 1) << k
    return tuple(p)


def tiny_inputs():
    ws = [W.random_points(200, seed=1), W.clustered_points(300, seed=2),
          W.with_duplicates(W.random_points(64, seed=3), 20), W.with_duplicates(W.clustered_points(100, seed=4), 30, near=1e-9),
          W.random_points(2, seed=5), W.random_points(3, seed=6, cube=(-2.0, 1.0, 5.0, 4.0))]
    return ws


@pytest.mark.parametrize("w", tiny_inputs(), ids=lambda w: w.name)
def test_tree_equals_bruteforce_partition(oracle, w):
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    keys, perm = t.sorted_keys_perm()
    nd = t.nodes()
    ref = brute_tree(w.x, w.y, w.z, w.cube)
    got = {}
    for i in range(t.n_nodes):
        lev = int(nd["level"][i])
        got[(lev, deinterleave(nd["prefix"][i], lev))] = frozenset(perm[nd["lo"][i]:nd["hi"][i]].tolist())
    assert got == ref
    # canonical order is strictly increasing in (level, prefix)
    order = list(zip(nd["level"].tolist(), nd["prefix"].tolist()))
    assert order == sorted(order) and len(set(order)) == len(order)
    # sorted keys ascending, ties by index
    assert np.all(np.diff(keys.astype(np.int64)) >= 0)
    tie = np.diff(keys.astype(np.int64)) == 0
    assert np.all(np.diff(perm.astype(np.int64))[tie] > 0)
    # the deepest internal level reported
    assert t.depth == max(l for (l, _) in ref if l < 21)


def test_chain_and_bucket_shapes(oracle):
    # two points 3e-7 apart in x only: a single-child chain from the root down to where they separate
    x = np.array([0.3, 0.3 + 3e-7]); y = np.array([0.3, 0.3]); z = np.array([0.3, 0.3])
    t = oracle.OracleTree(x, y, z, np.ones(2), [0, 0, 0, 1.0])
    nd = t.nodes()
    q0, q1 = int(math.floor(0.3 * 2097152)), int(math.floor((0.3 + 3e-7) * 2097152))
    sep = 21 - (q0 ^ q1).bit_length()  # deepest level at which both share the cell
    assert nd["level"].tolist() == list(range(sep + 1)) and np.all(nd["nchild"][:-1] == 1) and nd["nchild"][-1] == 2
    # three coincident points + one other: bucket leaf at level 21 under a chain of 21 internal nodes
    x = np.array([0.7, 0.7, 0.7, 0.1]); y = x.copy(); z = x.copy()
    t = oracle.OracleTree(x, y, z, np.ones(4), [0, 0, 0, 1.0])
    nd = t.nodes()
    assert nd["level"].tolist() == list(range(22)) and nd["nchild"][-1] == 3 and nd["hi"][-1] - nd["lo"][-1] == 3
    assert nd["nchild"][0] == 2 and t.depth == 20


@pytest.mark.parametrize("kk", [1, 2, 3, 4, 5])
def test_grid_counts_depth_and_centred_moments(oracle, kk):
    ng = 1 << kk
    x, y, z = W._grid_centres(ng)
    n = ng ** 3
    t = oracle.OracleTree(x, y, z, np.full(n, 1.0 / n), [0, 0, 0, 1.0])
    assert t.n_nodes == (n - 1) // 7 and t.depth == kk - 1  # T-rule 6
    nd = t.nodes()
    assert np.all(nd["nchild"] == 8)
    size = 0.5 ** nd["level"]
    for a, R in enumerate(("Rx", "Ry", "Rz")):
        pa = np.array([deinterleave(p, l)[a] for p, l in zip(nd["prefix"], nd["level"])])
        assert np.allclose(nd[R], (pa + 0.5) * size, rtol=0, atol=1e-15)
    assert np.all(nd["delta"] < 1e-15)
    assert np.allclose(nd["M"], (nd["hi"] - nd["lo"]) / n, rtol=1e-14)


@pytest.mark.parametrize("w", tiny_inputs()[:4] + [W.uniform_sphere(8)], ids=lambda w: w.name)
def test_moments_eq5_from_flat_ranges(oracle, w):
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _, perm = t.sorted_keys_perm()
    nd = t.nodes()
    # root invariants (BASELINE.json): total mass and mass-weighted mean position
    assert nd["level"][0] == 0 and nd["lo"][0] == 0 and nd["hi"][0] == w.n
    Mtot = math.fsum(w.m)
    assert abs(nd["M"][0] - Mtot) <= 1e-13 * Mtot
    for R, v in (("Rx", w.x), ("Ry", w.y), ("Rz", w.z)):
        assert abs(nd[R][0] - math.fsum(w.m * v) / Mtot) <= 1e-13 * w.cube[3]
    L = w.cube[3]
    for i in range(t.n_nodes):
        idx = perm[nd["lo"][i]:nd["hi"][i]]
        M = math.fsum(w.m[idx])
        lev = int(nd["level"][i])
        size = L / 2 ** lev
        p = deinterleave(nd["prefix"][i], lev)
        centre = [w.cube[a] + (p[a] + 0.5) * size for a in range(3)]
        if M == 0.0:  # M-rule 2
            assert nd["M"][i] == 0.0 and nd["delta"][i] == 0.0
            assert [nd["Rx"][i], nd["Ry"][i], nd["Rz"][i]] == centre
            continue
        assert abs(nd["M"][i] - M) <= 1e-13 * M
        R = [math.fsum(w.m[idx] * v[idx]) / M for v in (w.x, w.y, w.z)]  # Eq. 5
        got = [nd["Rx"][i], nd["Ry"][i], nd["Rz"][i]]
        assert max(abs(a - b) for a, b in zip(R, got)) <= 1e-13 * L
        delta = math.sqrt(sum((a - b) ** 2 for a, b in zip(R, centre)))
        assert abs(nd["delta"][i] - delta) <= 1e-12 * L
        if lev < 21:
            assert nd["delta"][i] <= math.sqrt(3) / 2 * size * (1 + 1e-12)  # com inside the node's cube


def test_sphere_workload_has_zero_mass_nodes(oracle):
    w = W.uniform_sphere(32)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    nd = t.nodes()
    assert t.n_nodes == 4681 and t.depth == 4
    zero = nd["M"] == 0.0
    assert zero.sum() > 100 and np.all(nd["delta"][zero] == 0.0)
