"""GPU parity for NEXT-1: Find Essential Nodes and the locally
essential tree built from them, through the C ABI, against the fp64 oracle.

Bars: the essential set is selected in fp64 on bit-identical moments, so entries, order and values are
compared for EQUALITY; Phi of a LET walk within max 1e-4 / median 1e-6 relative of the oracle run through
the same procedure (decisions in fp32 on both sides, W8), and at Barnes-Hut accuracy against
the fp64 direct sum over ALL cells of all domains."""
import numpy as np
import pytest

import bh_workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def bh():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_1509_07370_b200 as pkg
    return pkg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()


BOXES = [((1.5, 0.2, 0.2), (2.0, 0.8, 0.8)), ((0.6, 0.6, 0.6), (0.9, 0.9, 0.9)),
         ((-3.0, -3.0, -3.0), (-2.5, -2.5, -2.5)), ((1.0, 0.0, 0.0), (1.5, 1.0, 1.0)),
         ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0))]

CASES = [wl.uniform_sphere(16), wl.random_points(4099, seed=2), wl.clustered_points(3000, seed=3),
         wl.with_duplicates(wl.random_points(500, seed=4), 40, seed=4),
         wl.with_duplicates(wl.random_points(500, seed=5), 40, seed=5, near=2e-3),
         wl.amr_collapsing_core(nroot=2, max_level=3),
         wl.random_points(2, seed=5), wl.random_points(3, seed=6), wl.random_points(17, seed=7)]   # fewer slots than a tile


@pytest.mark.parametrize("mac", [0, 1], ids=["eq3", "eq4"])
@pytest.mark.parametrize("theta", [0.5, 1.0, 0.0])
@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_essential_nodes_equal_oracle(bh, oracle, w, theta, mac):
    ctx = bh.Context(0)
    ctx.set_mac(mac)
    ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    for blo, bhi in BOXES:
        got = ctx.essential_nodes(blo, bhi, theta).cpu().numpy()
        ref = ot.essential_nodes(blo, bhi, theta, mac=mac)
        assert got.shape == ref.shape, (blo, got.shape, ref.shape)
        assert np.array_equal(got, ref), blo
        # a first guess of the capacity that is too small is grown, one that is large enough is used
        assert np.array_equal(ctx.essential_nodes(blo, bhi, theta, cap=3).cpu().numpy(), ref)
        assert np.array_equal(ctx.essential_nodes(blo, bhi, theta, cap=w.n).cpu().numpy(), ref)


def test_essential_nodes_edge_cases(bh, oracle):
    import ctypes as C
    ctx = bh.Context(0)
    L = bh.lib()
    lo, hi = (C.c_double * 3)(2, 2, 2), (C.c_double * 3)(3, 3, 3)
    cnt = C.c_int64(-7)
    assert L.bh_essential_nodes(ctx._h, lo, hi, 0.5, None, 0, C.byref(cnt)) == -2          # not built
    one = wl.random_points(1, seed=9)
    ctx.build(_dev(one.x), _dev(one.y), _dev(one.z), _dev(one.m), one.cube)
    got = ctx.essential_nodes((2, 2, 2), (3, 3, 3), 0.5).cpu().numpy()
    assert np.array_equal(got, np.array([[one.x[0], one.y[0], one.z[0], one.m[0]]]))
    w = wl.random_points(1000, seed=1)
    ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
    assert L.bh_essential_nodes(ctx._h, lo, hi, 0.5, None, 0, C.byref(cnt)) == -5 and cnt.value >= 1   # size query
    assert L.bh_essential_nodes(ctx._h, hi, lo, 0.5, None, 0, C.byref(cnt)) == -1          # inverted box
    assert L.bh_essential_nodes(ctx._h, lo, hi, -1.0, None, 0, C.byref(cnt)) == -1
    assert L.bh_essential_nodes(ctx._h, lo, hi, 0.5, None, 0, None) == -1
    far = ctx.essential_nodes((50, 50, 50), (51, 51, 51), 1.0).cpu().numpy()
    assert far.shape == (1, 4) and far[0, 3] == pytest.approx(w.m.sum(), rel=1e-13)       # just the root


def _slabs(w, P):
    """P domains of (nearly) equal cell count, cut along x (the host code's decomposition is not part of
    the path; any spatial split exercises it)."""
    order = np.argsort(w.x, kind="stable")
    return [np.sort(c) for c in np.array_split(order, P)]


def _oracle_let(oracle, w, parts, theta, mac):
    """The procedure of paper_1509_07370_b200/let.py written with the oracle: local trees, essential
    nodes per remote box, union in the common cube, walk with the own cells as targets."""
    boxes = [((w.x[i].min(), w.y[i].min(), w.z[i].min()), (w.x[i].max(), w.y[i].max(), w.z[i].max())) for i in parts]
    inbox = [[] for _ in parts]
    sent = [[0] * len(parts) for _ in parts]
    for d, i in enumerate(parts):
        t = oracle.OracleTree(w.x[i], w.y[i], w.z[i], w.m[i], w.cube)
        for e in range(len(parts)):
            if e != d:
                rec = t.essential_nodes(boxes[e][0], boxes[e][1], theta, mac=mac)
                sent[d][e] = len(rec)
                inbox[e].append(rec)
    phis = []
    for e, i in enumerate(parts):
        ext = np.concatenate(inbox[e]) if inbox[e] else np.zeros((0, 4))
        u = [np.concatenate([a[i], ext[:, k]]) for k, a in enumerate((w.x, w.y, w.z, w.m))]
        t = oracle.OracleTree(*u, w.cube)
        phis.append(t.potential(theta, w.G, mac=mac, mac_fp32=True)[: len(i)])
    return phis, sent


@pytest.mark.parametrize("P", [2, 4])
@pytest.mark.parametrize("w", [wl.clustered_points(6000, seed=41), wl.amr_collapsing_core(nroot=2, max_level=3),
                               wl.uniform_sphere(16)], ids=lambda w: w.name)
def test_let_equals_oracle_procedure_and_direct_sum(bh, oracle, w, P):
    from paper_1509_07370_b200 import let
    theta, mac = 0.5, 1
    parts = _slabs(w, P)
    dparts = [tuple(_dev(a[i]) for a in (w.x, w.y, w.z, w.m)) for i in parts]
    phis, sent = let.let_potential_serial(dparts, w.cube, theta, w.G, mac=mac)
    ophis, osent = _oracle_let(oracle, w, parts, theta, mac)
    assert sent == osent
    rng = np.random.default_rng(7)
    for i, p, op in zip(parts, phis, ophis):
        p = p.cpu().numpy()
        assert p.shape == op.shape
        nz = op != 0
        rel = np.abs(p[nz] - op[nz]) / np.abs(op[nz])
        assert rel.max() <= 1e-4 and np.median(rel) <= 1e-6, (rel.max(), np.median(rel))
        sub = rng.choice(len(i), size=min(256, len(i)), replace=False)     # direct sum on a sample of the domain's cells
        ex = oracle.direct(w.x, w.y, w.z, w.m, w.G, targets=i[sub].astype(np.int64))
        nz = ex != 0
        err = np.abs(p[sub][nz] - ex[nz]) / np.abs(ex[nz])
        assert err.max() < 1e-2 and np.median(err) < 2e-3, (err.max(), np.median(err))    # theta = 0.5
    # far fewer entries travel than cells exist (the point of the LET)
    assert sum(map(sum, sent)) < (P - 1) * w.n


def test_num_targets_leaves_results_unchanged(bh, oracle):
    """Source-only cells still vote and are still summed (W-rules unchanged): Phi of the targets is
    bit-equal to the full walk's, groups without a target report zero counters."""
    w = wl.clustered_points(5000, seed=43)
    ctx = bh.Context(0)
    ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
    full = ctx.potential(0.5, w.G).cpu().numpy()
    cnt_full = ctx.last_group_counts().cpu().numpy()
    nt = 1234
    ctx.set_num_targets(nt)
    part = ctx.potential(0.5, w.G)
    assert part.shape[0] == nt
    assert np.array_equal(part.cpu().numpy(), full[:nt])
    cnt = ctx.last_group_counts().cpu().numpy()
    perm = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube).sorted_keys_perm()[1]
    ng = cnt.shape[0]
    has = np.array([np.any(perm[32 * g: 32 * g + 32] < nt) for g in range(ng)])
    pair_has = has.copy()
    pair_has[0::2] |= np.pad(has[1::2], (0, len(has[0::2]) - len(has[1::2])))
    pair_has[1::2] |= has[0::2][: len(has[1::2])]
    assert np.array_equal(cnt[pair_has], cnt_full[pair_has])      # a warp walks two adjacent groups together
    assert np.all(cnt[~pair_has] == 0)
    for g1 in (1,):
        ctx.set_group(g1)
        p1 = ctx.potential(0.5, w.G)
        ctx.set_num_targets(-1)
        f1 = ctx.potential(0.5, w.G)
        assert np.array_equal(p1.cpu().numpy(), f1.cpu().numpy()[:nt])
