"""Pins for the oracle's Find-Essential-Nodes step (§3.2.4, Fig. 7; E1-E4).
CPU only.  The selection is pinned by (i) an independent recursive partition in numpy that works on
quantised integer coordinates and flat sums (no Morton keys, no tree), (ii) the limits the paper
states -- between 1 entry (the root) and n entries (all cells), PAPER.md:106 --, (iii) mass and
centre-of-mass conservation of the emitted set, and (iv) the physics: the essential set reproduces
the donor's potential inside the receiver's box to Barnes-Hut accuracy, converging with theta."""
import numpy as np
import pytest

import bh_workloads as W


def brute_essential(x, y, z, m, cube, blo, bhi, theta, mac):
    """Recursive partition on integer coordinates; node moments from FLAT sums over its points.
    Returns a list of (level, frozenset(original indices)) for every emitted entry."""
    x, y, z, m = (np.asarray(a, dtype=np.float64) for a in (x, y, z, m))
    s = 2097152.0 / cube[3]
    q = np.stack([np.clip(np.floor((v - c0) * s), 0, 2097151).astype(np.int64)
                  for v, c0 in zip((x, y, z), cube[:3])], axis=1)
    blo, bhi = np.asarray(blo, float), np.asarray(bhi, float)
    out = []

    def rec(level, idx):
        if len(idx) == 1:
            out.append((level, frozenset(idx.tolist())))
            return
        if level == 21:                       # bucket: every cell on its own
            for i in idx:
                out.append((22, frozenset([int(i)])))
            return
        size = cube[3] / 2.0 ** level
        M = m[idx].sum()
        if M != 0.0:
            R = np.array([(m[idx] * v[idx]).sum() / M for v in (x, y, z)])
        else:
            R = np.array([c0 + ((q[idx[0], a] >> (21 - level)) + 0.5) * size for a, c0 in enumerate(cube[:3])])
        centre = np.array([c0 + ((q[idx[0], a] >> (21 - level)) + 0.5) * size for a, c0 in enumerate(cube[:3])])
        rc = np.inf if theta == 0 else size / theta + (np.linalg.norm(R - centre) if mac == 1 else 0.0)
        d = np.maximum(np.maximum(blo - R, R - bhi), 0.0)
        if theta > 0 and float(d @ d) > rc * rc:
            out.append((level, frozenset(idx.tolist())))
            return
        sub = q[idx] >> (20 - level)
        code = (sub[:, 0] & 1) + 2 * (sub[:, 1] & 1) + 4 * (sub[:, 2] & 1)
        for o in range(8):
            if np.any(code == o):
                rec(level + 1, idx[code == o])

    n = len(x)
    if n == 1:
        return [(1, frozenset([0]))]
    rec(0, np.arange(n))
    return out


BOXES = [((1.5, 0.2, 0.2), (2.0, 0.8, 0.8)),       # beside the cube
         ((0.6, 0.6, 0.6), (0.9, 0.9, 0.9)),       # inside it (overlapping domains)
         ((-3.0, -3.0, -3.0), (-2.5, -2.5, -2.5)),  # far away
         ((1.0, 0.0, 0.0), (1.5, 1.0, 1.0))]       # touching face


def _inputs():
    return [W.random_points(300, seed=11), W.clustered_points(400, seed=12),
            W.with_duplicates(W.random_points(100, seed=13), 20),
            W.with_duplicates(W.clustered_points(150, seed=14), 30, near=1e-3), W.uniform_sphere(8)]


@pytest.mark.parametrize("mac", [0, 1], ids=["eq3", "eq4"])
@pytest.mark.parametrize("theta", [0.3, 0.7, 1.0])
@pytest.mark.parametrize("w", _inputs(), ids=lambda w: w.name)
def test_essential_set_equals_bruteforce(oracle, w, theta, mac):
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _, perm = t.sorted_keys_perm()
    for blo, bhi in BOXES:
        rec, lev, lo, hi = t.essential_nodes(blo, bhi, theta, mac=mac, want_ranges=True)
        got = sorted((int(l), tuple(sorted(perm[a:b].tolist()))) for l, a, b in zip(lev, lo, hi))
        ref = sorted((l, tuple(sorted(s))) for l, s in brute_essential(w.x, w.y, w.z, w.m, w.cube, blo, bhi, theta, mac))
        assert got == ref
        # canonical order: ascending (level, first sorted cell)
        order = np.lexsort((lo, lev))
        assert np.array_equal(order, np.arange(len(lev)))
        # every entry is the monopole of its range (flat sums)
        for k in range(len(lev)):
            idx = perm[lo[k]:hi[k]]
            M = w.m[idx].sum()
            assert rec[k, 3] == pytest.approx(M, rel=1e-13, abs=1e-300)
            if M != 0 and len(idx) > 1:
                for a, v in enumerate((w.x, w.y, w.z)):
                    assert rec[k, a] == pytest.approx((w.m[idx] * v[idx]).sum() / M, rel=1e-12, abs=1e-13)


def test_limits_root_only_and_all_cells(oracle):
    """'the number of Essential Nodes may vary between 1 (the process just sends its
    root node) and n (the process sends all data cells)'."""
    w = W.random_points(500, seed=21)
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    far = t.essential_nodes((50.0, 50.0, 50.0), (51.0, 51.0, 51.0), 1.0)
    assert far.shape == (1, 4)
    assert far[0, 3] == pytest.approx(w.m.sum(), rel=1e-13)
    for a, v in enumerate((w.x, w.y, w.z)):
        assert far[0, a] == pytest.approx((w.m * v).sum() / w.m.sum(), rel=1e-12)
    # theta = 0 opens everything; a box covering the whole cube opens everything for theta <= 1 with Eq. 4
    for rec in (t.essential_nodes((2.0, 2.0, 2.0), (3.0, 3.0, 3.0), 0.0),
                t.essential_nodes((0.0, 0.0, 0.0), (1.0, 1.0, 1.0), 1.0, mac=1)):
        assert rec.shape == (w.n, 4)
        got = rec[np.lexsort(rec.T[::-1])]
        ref = np.stack([w.x, w.y, w.z, w.m], axis=1)
        ref = ref[np.lexsort(ref.T[::-1])]
        assert np.array_equal(got, ref)


@pytest.mark.parametrize("w", [W.clustered_points(2000, seed=31), W.amr_collapsing_core(nroot=2, max_level=3)],
                         ids=lambda w: w.name)
def test_mass_conserved_and_potential_in_box(oracle, w):
    """The emitted ranges partition the cells (mass and first moment conserved), and for points inside
    the receiver's box the essential set gives the donor's potential to Barnes-Hut accuracy: the
    error against the direct sum falls with theta and vanishes at theta = 0."""
    t = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    blo, bhi = np.array([1.1, 0.1, 0.3]), np.array([1.6, 0.7, 0.9])
    rng = np.random.default_rng(5)
    pts = blo + (bhi - blo) * rng.random((64, 3))
    src = np.stack([w.x, w.y, w.z], axis=1)
    exact = -np.array([(w.m / np.linalg.norm(src - p, axis=1)).sum() for p in pts])
    errs = []
    for theta in (1.0, 0.7, 0.5, 0.3, 0.0):
        rec, lev, lo, hi = t.essential_nodes(blo, bhi, theta, want_ranges=True)
        cover = np.zeros(w.n + 1, dtype=np.int64)
        np.add.at(cover, lo, 1)
        np.add.at(cover, hi, -1)
        assert np.all(np.cumsum(cover)[:-1] == 1)              # disjoint ranges covering [0, n)
        assert rec[:, 3].sum() == pytest.approx(w.m.sum(), rel=1e-12)
        for a, v in enumerate((w.x, w.y, w.z)):
            assert (rec[:, 3] * rec[:, a]).sum() == pytest.approx((w.m * v).sum(), rel=1e-11)
        approx = -np.array([(rec[:, 3] / np.linalg.norm(rec[:, :3] - p, axis=1)).sum() for p in pts])
        errs.append(np.max(np.abs(approx - exact) / np.abs(exact)))
    assert errs[-1] < 1e-13                                    # theta = 0: all cells, exact
    assert errs[0] < 2e-2 and errs[2] < 5e-3                   # theta = 1 ~ 1 %, 0.5 well below
    assert all(errs[i + 1] <= errs[i] * 1.05 + 1e-15 for i in range(len(errs) - 1))
    assert len(t.essential_nodes(blo, bhi, 0.3)) > len(t.essential_nodes(blo, bhi, 1.0))
