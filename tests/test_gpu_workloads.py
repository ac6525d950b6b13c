"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot walk 16.8 M targets in seconds, so per workload: Morton keys, permutation and tree
topology are compared in full (the oracle's build takes seconds), node moments in full, and Phi plus
the per-group interaction counters on sampled runs of groups the oracle walks one by one (groups are
independent given the tree, so parity on a sample is exact for that sample).  Configs 0 and 1 are
also held against the closed forms the paper uses (§4.1), config 4 is the
opening-angle sweep with the direct-sum-on-subsample error.
"""
import numpy as np
import pytest

import bh_workloads as wl
from tests import analytic, parity

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


def _build(bh, w):
    ctx = bh.Context(0)
    ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
    return ctx


def _check_sampled(ctx, ot, w, theta, mac=0, nruns=12, per=24):
    """Phi and the per-group counters of sampled runs of groups under the protocol of tests/parity.py (fp64
    oracle with flips counted and reported; fp32-decision oracle flip-free)."""
    ngroups = (w.n + 31) // 32
    rep = parity.check_walk(ctx, ot, w, theta, mac=mac, runs=parity.sample_runs(ngroups, nruns, per))
    return rep["phi"], rep["counts"]


def _check_essential(ctx, ot, w, theta=0.5):
    """NEXT-1 at full size: the essential set for a face-neighbour domain and for a distant one equals the
    oracle's entry for entry (selection in fp64 on bit-identical moments)."""
    x0, y0, z0, L = w.cube
    for mac in (1, 0):
        ctx.set_mac(mac)
        for lo, hi in (((x0 + L, y0, z0), (x0 + 2 * L, y0 + L, z0 + L)),
                       ((x0 - 9 * L, y0 + 3 * L, z0), (x0 - 8 * L, y0 + 4 * L, z0 + L))):
            got = ctx.essential_nodes(lo, hi, theta).cpu().numpy()
            ref = ot.essential_nodes(lo, hi, theta, mac=mac)
            assert got.shape == ref.shape and np.array_equal(got, ref), (mac, lo, got.shape, ref.shape)
    ctx.set_mac(0)


def _check_tree(ctx, ot, w):
    t = {k: v.cpu().numpy() for k, v in ctx.export_tree().items()}
    ok, op = ot.sorted_keys_perm()
    assert np.array_equal(t["keys"].view(np.uint64), ok), "Morton keys differ"
    assert np.array_equal(t["perm"].view(np.uint32), op), "permutation differs"
    on = ot.nodes()
    n, nn, ns = ctx.tree_sizes()
    assert (n, nn, ns) == (w.n, ot.n_nodes, w.n + ot.n_nodes)
    for k in ("level", "lo", "hi", "nchild"):
        assert np.array_equal(t[k].astype(np.int64), on[k].astype(np.int64)), k
    assert np.array_equal(t["prefix"].view(np.uint64), on["prefix"].astype(np.uint64))
    scale = np.maximum(np.abs(on["M"]), 1e-300)
    assert np.max(np.abs(t["M"] - on["M"]) / scale) <= 1e-6
    for k in ("Rx", "Ry", "Rz", "delta"):
        assert np.max(np.abs(t[k] - on[k])) / w.cube[3] <= 1e-6, k


def test_config0_uniform_sphere(bh, oracle):
    """32^3 sphere: full oracle parity, full direct sum, closed form 2 pi G rho (R^2 - r^2/3) inside."""
    w = wl.by_name("sphere32")
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _check_tree(ctx, ot, w)
    phi, _ = _check_sampled(ctx, ot, w, 0.5, nruns=1, per=1 << 20)       # all 1024 groups
    direct = ctx.potential_direct(w.G).cpu().numpy()
    ref = oracle.direct(w.x, w.y, w.z, w.m, w.G)
    assert np.max(np.abs(direct - ref) / np.abs(ref)) <= 1e-12
    assert np.max(np.abs(phi - direct) / np.abs(direct)) <= 5e-3          # the tree code's own error at theta 0.5
    r = np.sqrt((w.x - 0.5) ** 2 + (w.y - 0.5) ** 2 + (w.z - 0.5) ** 2)
    inside = r < 0.3
    exact = analytic.sphere_potential(r[inside], 0.4, 1.0, w.G)
    assert np.max(np.abs(phi[inside] - exact) / np.abs(exact)) <= 2e-2    # 32^3 staircase of the sphere's surface


def test_config1_maclaurin(bh, oracle):
    """128^3 MacLaurin spheroid (e = 0.9): sampled oracle parity, analytic interior potential (Eq. 6, R12)."""
    w = wl.by_name("maclaurin128")
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _check_tree(ctx, ot, w)
    phi, _ = _check_sampled(ctx, ot, w, 0.5, nruns=32, per=32)
    a1, e = 0.4, 0.9
    a3 = a1 * np.sqrt(1 - e * e)
    X, Y, Z = w.x - 0.5, w.y - 0.5, w.z - 0.5
    deep = (X * X + Y * Y) / (0.8 * a1) ** 2 + Z * Z / (0.8 * a3) ** 2 < 1.0
    exact = analytic.maclaurin_interior(X[deep], Y[deep], Z[deep], a1, e, 1.0, w.G)
    assert np.max(np.abs(phi[deep] - exact) / np.abs(exact)) <= 1e-2


def test_config2_amr_core_and_config4_theta_sweep(bh, oracle):
    """~3.9 M-cell AMR collapsing core: tree in full, then theta in {0.3, 0.5, 0.7, 1.0}: sampled oracle
    parity, interactions per target, and the error against the fp64 direct sum on 4096 sampled targets."""
    w = wl.by_name("amr_core")
    assert 2_000_000 <= w.n <= 5_000_000
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _check_tree(ctx, ot, w)
    _check_essential(ctx, ot, w)
    rng = np.random.Generator(np.random.PCG64(4096))
    tg = np.sort(rng.choice(w.n, 4096, replace=False)).astype(np.int64)
    direct = ctx.potential_direct(w.G, targets=torch.from_numpy(tg).cuda()).cpu().numpy()
    sub = rng.choice(4096, 64, replace=False)                              # the oracle's direct sum on a few of them
    ref = oracle.direct(w.x, w.y, w.z, w.m, w.G, targets=tg[sub])
    assert np.max(np.abs(direct[sub] - ref) / np.abs(ref)) <= 1e-12
    errs, inter = [], []
    for theta in (0.3, 0.5, 0.7, 1.0):
        phi, cnt = _check_sampled(ctx, ot, w, theta, nruns=32, per=32)      # 1024 of ~122 k groups per theta
        errs.append(np.max(np.abs(phi[tg] - direct) / np.abs(direct)))
        inter.append(ctx.get_stats().interactions / w.n)
    assert all(a < b for a, b in zip(errs, errs[1:])), errs               # error grows with theta
    assert all(a > b for a, b in zip(inter, inter[1:])), inter            # work shrinks with theta
    assert errs[0] <= 2e-3 and errs[1] <= 1e-2


def test_config3_turb256_bench_configuration(bh, oracle):
    """The workload bench.py times (16.8 M cells, theta 0.5): keys / topology / moments in full, Phi sampled."""
    w = wl.by_name("turb256")
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    _check_tree(ctx, ot, w)
    st = ctx.get_stats()
    assert st.n_nodes == (w.n - 1) // 7 and st.depth == 7 and st.sort_passes == 3
    _check_essential(ctx, ot, w)
    _check_sampled(ctx, ot, w, 0.5, nruns=64, per=64)           # 4096 of 524,288 groups, like bench.py's parity key
    _check_sampled(ctx, ot, w, 0.5, mac=1, nruns=16, per=16)
    # properties that hold at any size: every potential is finite and negative (all masses are positive)
    phi = ctx.potential(0.5, w.G).cpu().numpy()
    assert np.all(np.isfinite(phi)) and np.all(phi < 0)


def test_large_grid_512_properties(bh):
    """134 M cells (512^3 uniform grid, equal masses): well past BASELINE's largest config.  The oracle cannot
    build this in seconds, so the checks are properties that hold at any size: node count (n-1)/7, depth 8,
    3 sort passes, root moments, the mirror symmetry of Phi, and sampled targets against the fp64 direct sum."""
    ng = 512
    n = ng ** 3
    free, _ = torch.cuda.mem_get_info()
    if free < 40 * (1 << 30):
        pytest.skip("needs 40 GB of free device memory")
    ax = (torch.arange(ng, dtype=torch.float64, device="cuda") + 0.5) / ng
    x = ax.view(ng, 1, 1).expand(ng, ng, ng).reshape(-1).contiguous()
    y = ax.view(1, ng, 1).expand(ng, ng, ng).reshape(-1).contiguous()
    z = ax.view(1, 1, ng).expand(ng, ng, ng).reshape(-1).contiguous()
    m = torch.full((n,), 1.0 / n, dtype=torch.float64, device="cuda")
    ctx = bh.Context(0)
    ctx.build(x, y, z, m, (0.0, 0.0, 0.0, 1.0))
    st = ctx.get_stats()
    assert st.n_nodes == (n - 1) // 7 and st.depth == 8 and st.sort_passes == 4 and st.n_clamped == 0
    t = ctx.export_tree()
    assert abs(float(t["M"][0]) - 1.0) <= 1e-12
    for k in ("Rx", "Ry", "Rz"):
        assert abs(float(t[k][0]) - 0.5) <= 1e-12
    keys = t["keys"].view(torch.int64)
    assert bool((keys[1:] > keys[:-1]).all())                     # strictly ascending: all keys distinct
    del t, keys
    phi = ctx.potential(0.5, 1.0)
    st = ctx.get_stats()
    assert 1000 < st.interactions / n < 2600
    p3 = phi.view(ng, ng, ng)
    for dim in (0, 1, 2):                                         # the cube of equal masses is mirror symmetric
        assert float((p3 - p3.flip(dim)).abs().max()) <= 2e-5 * float(phi.abs().max())
    rng = np.random.Generator(np.random.PCG64(512))
    tg = torch.from_numpy(np.sort(rng.choice(n, 64, replace=False)).astype(np.int64)).cuda()
    direct = ctx.potential_direct(1.0, targets=tg)
    rel = ((phi[tg] - direct) / direct).abs()
    assert float(rel.max()) <= 5e-3                               # the tree code's own error at theta = 0.5
    centre = float(phi.view(ng, ng, ng)[ng // 2, ng // 2, ng // 2])
    assert abs(centre + analytic.CUBE_SELF) <= 2e-3 * analytic.CUBE_SELF   # -Phi at the centre of a unit cube of unit mass


def test_size_limits(bh):
    """n >= 2^30 is refused before anything is touched (30-bit tile counters of the sort); n >= 2^31 is invalid."""
    ctx = bh.Context(0)
    one = torch.zeros(1, dtype=torch.float64, device="cuda")
    L = bh.lib()
    import ctypes
    cube = (ctypes.c_double * 4)(0.0, 0.0, 0.0, 1.0)
    p = one.data_ptr()
    assert L.bh_build(ctx._h, p, p, p, p, 1 << 30, cube) == -5    # BH_ERR_TOO_LARGE
    assert L.bh_build(ctx._h, p, p, p, p, 1 << 31, cube) == -1    # BH_ERR_INVALID_ARG
    assert L.bh_build(ctx._h, p, p, p, p, 0, cube) == -1
