"""Pins for the oracle's keys and sort (K-rules, S-rule).  CPU only."""
import numpy as np
import pytest

import bh_workloads as W


def part1by2(q):
    """Independent bit-spread (magic-number method, not the oracle's per-bit loop)."""
    q = q.astype(np.uint64) & np.uint64(0x1FFFFF)
    q = (q | (q << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
    q = (q | (q << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
    q = (q | (q << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
    q = (q | (q << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
    q = (q | (q << np.uint64(2))) & np.uint64(0x1249249249249249)
    return q


def morton(qx, qy, qz):
    return part1by2(qx) | (part1by2(qy) << np.uint64(1)) | (part1by2(qz) << np.uint64(2))


def test_hand_values(oracle):
    # q = (1,0,0) -> 1 ; (0,1,0) -> 2 ; (0,0,1) -> 4 ; (2,0,0) -> 8 ; all-ones -> 2^63-1 ; bit 63 = 0
    s = 1.0 / 2097152.0
    pts = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [0, 0, 1], [2, 0, 0], [3, 5, 6], [2097151, 2097151, 2097151]], float)
    c = (pts + 0.5) * s
    k, nc = oracle.keys(c[:, 0], c[:, 1], c[:, 2], [0, 0, 0, 1.0])
    assert nc == 0
    # (3,5,6): x=011 y=101 z=110 -> bit triplets (z y x) per level k: k0: x1 y1 z0 -> 0b011=3 ; k1: x1 y0 z1 -> 0b101=5 ; k2: x0 y1 z1 -> 0b110=6
    assert k.tolist() == [0, 1, 2, 4, 8, 3 | (5 << 3) | (6 << 6), (1 << 63) - 1]


@pytest.mark.parametrize("kk", [1, 3, 5, 7])
def test_grid_closed_form(oracle, kk):
    ng = 1 << kk
    w = W.uniform_sphere(ng)
    k, nc = oracle.keys(w.x, w.y, w.z, w.cube)
    i = np.arange(ng, dtype=np.uint64)
    q = i * np.uint64(1 << (21 - kk)) + np.uint64(1 << (20 - kk))  # K-rule 3
    QX, QY, QZ = np.meshgrid(q, q, q, indexing="ij")
    assert nc == 0
    assert np.array_equal(k, morton(QX.ravel(), QY.ravel(), QZ.ravel()))
    # octant of the level-(l+1) child = x + 2y + 4z of the (l+1)-th coordinate bits from the top
    for lev in range(kk):
        octant = (k >> np.uint64(3 * (20 - lev))) & np.uint64(7)
        bx = (QX.ravel() >> np.uint64(20 - lev)) & np.uint64(1)
        by = (QY.ravel() >> np.uint64(20 - lev)) & np.uint64(1)
        bz = (QZ.ravel() >> np.uint64(20 - lev)) & np.uint64(1)
        assert np.array_equal(octant, bx + np.uint64(2) * by + np.uint64(4) * bz)


def test_random_vs_independent_interleave(oracle):
    rng = np.random.default_rng(5)
    cube = np.array([-1.5, 2.0, 0.25, 3.0])
    p = cube[:3] + cube[3] * rng.random((5000, 3))
    k, nc = oracle.keys(p[:, 0], p[:, 1], p[:, 2], cube)
    s = 2097152.0 / cube[3]
    q = [np.floor((p[:, a] - cube[a]) * s).astype(np.uint64) for a in range(3)]
    assert nc == 0 and np.array_equal(k, morton(*q))
    assert (k >> np.uint64(63)).max() == 0


def test_clamp_and_nan(oracle):
    x = np.array([-0.1, 1.0, 1.5, 0.5, np.nan, 0.999999999999])
    y = np.full(6, 0.5); z = np.full(6, 0.5)
    k, nc = oracle.keys(x, y, z, [0, 0, 0, 1.0])
    qx = np.array([0, 2097151, 2097151, 1048576, 0, 2097151], dtype=np.uint64)
    qh = np.full(6, 1048576, dtype=np.uint64)
    assert np.array_equal(k, morton(qx, qh, qh))
    assert nc == 4  # -0.1, 1.0 (t = 2^21 exactly), 1.5, NaN


def test_sort_is_stable_key_index_order(oracle):
    rng = np.random.default_rng(1)
    k = rng.integers(0, 50, 4000).astype(np.uint64) << np.uint64(40)  # many ties
    perm = oracle.sort_perm(k)
    ref = np.lexsort((np.arange(k.size), k))  # ascending key, ties by ascending index
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(np.sort(perm), np.arange(k.size))
