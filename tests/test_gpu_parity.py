"""GPU parity: libbh (CUDA, through the C ABI) against the fp64 CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): Morton keys, permutation and tree topology bit-exact; node mass and
centre of mass within 1e-6 relative; Phi within max relative error 1e-4 and median 1e-6 of the fp64 oracle
(criterion evaluated in fp64 as the paper writes it), accounting for fp32-vs-fp64 opening flips, whose
count is reported -- the protocol is tests/parity.py (primary: fp64 oracle with flips counted; secondary:
the CPU-pinned fp32-decision mode, flip-free, every group's counters and the Phi kernel's own entry counts).
"""
import numpy as np
import pytest

import bh_workloads as wl
from tests import parity

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


def _small_cases():
    cases = [
        wl.uniform_sphere(16),
        wl.random_points(1000, seed=1),
        wl.random_points(4099, seed=2, cube=(-1.0, 2.0, 0.5, 3.0)),
        wl.clustered_points(3000, seed=3),
        wl.with_duplicates(wl.random_points(500, seed=4), 40, seed=4),              # bucket leaves
        wl.with_duplicates(wl.random_points(500, seed=5), 40, seed=5, near=2e-3),   # single-child chains
        wl.amr_collapsing_core(nroot=2, max_level=3),
    ]
    return cases


CASES = _small_cases()
# Pairs 3e-7 apart: chains down to level ~21.  Topology and moments must still be bit-exact; Phi is
# not compared there because the walk holds positions in fp32 (W9: a pair at distance d
# carries a relative distance error up to ~2^-23 L/d, which exceeds 1e-4 below d ~ 1e-3 L; AMR cell
# centres are dyadic and never that close).
DEEP_CHAINS = wl.with_duplicates(wl.random_points(500, seed=5), 40, seed=5, near=3e-7)
TOPO_CASES = CASES + [DEEP_CHAINS]


def _tree_np(ctx):
    t = {k: v.cpu().numpy() for k, v in ctx.export_tree().items()}
    t["keys"] = t["keys"].view(np.uint64)
    t["perm"] = t["perm"].view(np.uint32)
    t["prefix"] = t["prefix"].view(np.uint64)
    return t


@pytest.mark.parametrize("w", TOPO_CASES, ids=lambda w: w.name)
def test_keys_perm_topology_bit_exact(bh, oracle, w):
    ctx = _build(bh, w)
    t = _tree_np(ctx)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    ok, op = ot.sorted_keys_perm()
    assert np.array_equal(t["keys"], ok)
    assert np.array_equal(t["perm"], op)
    on = ot.nodes()
    n, nn, ns = ctx.tree_sizes()
    assert nn == ot.n_nodes and n == w.n and ns == n + nn
    for k in ("level", "prefix", "lo", "hi", "nchild"):
        assert np.array_equal(t[k].astype(np.int64), on[k].astype(np.int64)), k
    st = ctx.get_stats()
    assert st.depth == ot.depth and st.n_clamped == ot.n_clamped


@pytest.mark.parametrize("w", TOPO_CASES, ids=lambda w: w.name)
def test_moments(bh, oracle, w):
    ctx = _build(bh, w)
    t = _tree_np(ctx)
    on = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube).nodes()
    L = w.cube[3]
    scale = np.maximum(np.abs(on["M"]), 1e-300)
    assert np.max(np.abs(t["M"] - on["M"]) / scale) <= 1e-6
    for k in ("Rx", "Ry", "Rz"):
        assert np.max(np.abs(t[k] - on[k])) / L <= 1e-6
    assert np.max(np.abs(t["delta"] - on["delta"])) / L <= 1e-6
    # the reduction mirrors the oracle's operation order, so in practice it is bit-identical
    assert np.array_equal(t["M"], on["M"])


def _phi_check(phi, ref, max_tol=1e-4, med_tol=1e-6):
    scale = np.abs(ref)
    ok = scale > 0
    rel = np.abs(phi[ok] - ref[ok]) / scale[ok]
    assert np.all(phi[~ok] == 0.0)
    assert np.max(rel) <= max_tol, f"max rel {np.max(rel):.3e}"
    assert np.median(rel) <= med_tol, f"median rel {np.median(rel):.3e}"
    return rel


@pytest.mark.parametrize("mac", [0, 1], ids=["eq3", "eq4"])
@pytest.mark.parametrize("theta", [0.5, 1.0, 0.3])
@pytest.mark.parametrize("w", CASES, ids=lambda w: w.name)
def test_phi_vs_oracle(bh, oracle, w, theta, mac):
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    rep = parity.check_walk(ctx, ot, w, theta, mac=mac)
    inter = ctx.last_interactions().cpu().numpy().view(np.uint32)
    perm = ot.sorted_keys_perm()[1]
    cnt = rep["counts"]
    assert np.array_equal(inter[perm], np.repeat(cnt[:, 0] + cnt[:, 1], 32)[: w.n])
    st = ctx.get_stats()
    assert st.interactions == st.interactions_counted == float(inter.astype(np.int64).sum())
    assert st.walk_group == 32


@pytest.mark.parametrize("theta", [0.5, 1.0])
@pytest.mark.parametrize("w", [CASES[1], CASES[3], CASES[4], CASES[6]], ids=lambda w: w.name)
def test_group1_walk(bh, oracle, w, theta):
    """BH_OPT_GROUP = 1 (W5): every target walks alone -- the textbook per-particle BH."""
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    parity.check_walk(ctx, ot, w, theta, group=1)
    assert ctx.get_stats().walk_group == 1
    parity.check_walk(ctx, ot, w, theta, group=32)      # and back: the pair walk on the same tree


def test_group_outputs_follow_the_group_of_the_last_walk(bh, oracle):
    """The per-group outputs are sized by the group of the LAST WALK (bh_last_walk_group), whatever the option
    says now; asking for the statistics of a per-target walk re-runs nothing that writes through a null Phi."""
    w = CASES[1]
    ctx = _build(bh, w)
    ctx.set_group(1)
    phi1 = ctx.potential(0.5, w.G).cpu().numpy()
    ctx.set_group(32)                                    # option changed, no walk yet
    assert ctx.last_walk_group() == 1
    assert ctx.last_group_counts().shape == (w.n, 3) and ctx.last_group_evaluated().shape == (w.n,)
    st = ctx.get_stats()
    assert st.walk_group == 1 and st.interactions == st.interactions_counted > 0
    ctx.set_num_targets(w.n // 2)                        # invalidates the counters; the next walk refills them
    ctx.set_group(1)
    ctx.potential(0.5, w.G)
    assert ctx.get_stats().interactions > 0
    ctx.set_num_targets(-1)
    ctx.set_group(32)
    assert np.all(np.isfinite(phi1))
    torch.cuda.synchronize()


@pytest.mark.parametrize("w", [CASES[1], CASES[4]], ids=lambda w: w.name)
def test_theta_zero_is_direct_sum(bh, oracle, w):
    ctx = _build(bh, w)
    phi0 = ctx.potential(0.0, w.G).cpu().numpy()
    ref = oracle.direct(w.x, w.y, w.z, w.m, w.G)
    _phi_check(phi0, ref, max_tol=2e-5, med_tol=1e-6)
    st = ctx.get_stats()
    assert st.n_accepted == 0
    ngroups = (w.n + 31) // 32
    assert st.n_leaf == ngroups * w.n          # every group sums every cell


@pytest.mark.parametrize("w", [CASES[1], CASES[4], CASES[0]], ids=lambda w: w.name)
def test_direct_fp64(bh, oracle, w):
    ctx = _build(bh, w)
    ref = oracle.direct(w.x, w.y, w.z, w.m, w.G)
    phi = ctx.potential_direct(w.G).cpu().numpy()
    nz = ref != 0
    assert np.max(np.abs(phi[nz] - ref[nz]) / np.abs(ref[nz])) <= 1e-12
    rng = np.random.Generator(np.random.PCG64(4096))
    tg = rng.integers(0, w.n, 97)
    sub = ctx.potential_direct(w.G, targets=torch.from_numpy(tg).cuda()).cpu().numpy()
    assert np.max(np.abs(sub - ref[tg]) / np.maximum(np.abs(ref[tg]), 1e-300)) <= 1e-12


def test_deep_chains_walk_counts(bh, oracle):
    """Near-coincident pairs: the interaction lists still agree group by group and Phi is finite (Phi itself is
    not compared here: W9)."""
    w = DEEP_CHAINS
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    rep = parity.check_walk(ctx, ot, w, 0.5, check_phi=False)
    assert np.all(np.isfinite(rep["phi"])) and np.all(rep["phi"] < 0)


def test_edge_cases(bh, oracle):
    # n = 1: no tree, Phi = 0
    ctx = bh.Context(0)
    one = _dev([0.3])
    ctx.build(one, one, one, _dev([2.0]), (0, 0, 0, 1))
    assert ctx.tree_sizes() == (1, 0, 0)
    assert ctx.potential(0.5).cpu().numpy()[0] == 0.0
    # n = 2, 33 (ragged last group), all points coincident, points outside the cube (clamped)
    for w in (wl.random_points(2, seed=7), wl.random_points(33, seed=8), wl.random_points(65, seed=9)):
        ctx = _build(bh, w)
        parity.check_walk(ctx, oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube), w, 0.5)
    n = 50
    same = wl.Workload("coincident", np.full(n, 0.25), np.full(n, 0.5), np.full(n, 0.75), np.ones(n))
    ctx = _build(bh, same)
    assert np.all(ctx.potential(0.5).cpu().numpy() == 0.0)          # zero-distance pairs are skipped
    st = ctx.get_stats()
    assert st.max_bucket == n and st.n_nodes == 22 and st.sort_passes == 0
    w = wl.random_points(300, seed=10, cube=(-0.2, -0.2, -0.2, 1.4))
    w.cube = np.array([0.0, 0.0, 0.0, 1.0])                          # many points now fall outside
    ctx = _build(bh, w)
    ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
    assert ctx.get_stats().n_clamped == ot.n_clamped > 0
    t = _tree_np(ctx)
    assert np.array_equal(t["keys"], ot.sorted_keys_perm()[0])
    parity.check_walk(ctx, ot, w, 0.7)


def test_argument_errors(bh):
    ctx = bh.Context(0)
    x = _dev(np.linspace(0.1, 0.9, 10))
    with pytest.raises(bh.BHError):
        ctx.potential(0.5)                                           # not built
    with pytest.raises(bh.BHError):
        ctx.build(x, x, x, x, (0, 0, 0, 0.0))                        # L <= 0
    ctx.build(x, x, x, x, (0, 0, 0, 1.0))
    with pytest.raises(bh.BHError):
        ctx.potential(-1.0)
    with pytest.raises(bh.BHError):
        ctx.potential(float("nan"))
    with pytest.raises(bh.BHError):
        ctx.set_option(99, 0)


def test_solve_host_matches_device_path(bh):
    w = wl.random_points(5000, seed=11)
    ctx = _build(bh, w)
    phi_d = ctx.potential(0.5).cpu().numpy()
    phi_h = bh.Context(0).solve_host(w.x, w.y, w.z, w.m, w.cube, 0.5)
    assert np.array_equal(phi_d, phi_h)


@pytest.mark.parametrize("w", [CASES[1], CASES[4], CASES[6]], ids=lambda w: w.name)
def test_update_masses_equals_rebuild(bh, oracle, w):
    """bh_update_masses (NEXT-2): new masses on the same cells reuse keys / sort / topology
    and give what a fresh build with those masses gives, bit for bit; and both match the oracle."""
    rng = np.random.Generator(np.random.PCG64(84))
    m2 = w.m * rng.uniform(0.25, 4.0, w.n)
    m2[rng.integers(0, w.n, 5)] = 0.0                                  # a few massless cells
    ctx = _build(bh, w)
    ctx.potential(0.5, w.G)                                            # the tree has been used before
    ctx.update_masses(_dev(m2))
    phi_u = ctx.potential(0.5, w.G).cpu().numpy()
    t_u = _tree_np(ctx)
    w2 = wl.Workload(w.name + "_m2", w.x, w.y, w.z, m2, cube=w.cube)
    ctx2 = _build(bh, w2)
    phi_r = ctx2.potential(0.5, w.G).cpu().numpy()
    t_r = _tree_np(ctx2)
    assert np.array_equal(phi_u, phi_r)
    for k in ("keys", "perm", "level", "lo", "hi", "M", "Rx", "Ry", "Rz", "delta"):
        assert np.array_equal(t_u[k], t_r[k]), k
    ot = oracle.OracleTree(w.x, w.y, w.z, m2, w.cube)
    rep = parity.check_walk(ctx, ot, w2, 0.5)
    assert np.array_equal(rep["phi"], phi_u)
    tg = rng.integers(0, w.n, 64)                                      # the direct sum sees the new masses too
    sub = ctx.potential_direct(w.G, targets=torch.from_numpy(tg).cuda()).cpu().numpy()
    dref = oracle.direct(w.x, w.y, w.z, m2, w.G, targets=tg)
    nz = dref != 0
    assert np.max(np.abs(sub[nz] - dref[nz]) / np.abs(dref[nz])) <= 1e-12


def test_context_reuse_across_inputs(bh, oracle):
    """One context, many builds: the sort plan speculated from the previous build (hit when the same
    input comes again, miss and redo when another one comes) and the aux records kept zero between
    builds must leave every build identical to one made in a fresh context."""
    ctx = bh.Context(0)
    seq = [CASES[0], CASES[0], CASES[1], CASES[4], CASES[6], CASES[6], CASES[2], CASES[0], DEEP_CHAINS, CASES[3]]
    for w in seq:
        ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
        t = _tree_np(ctx)
        ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
        ok, op = ot.sorted_keys_perm()
        assert np.array_equal(t["keys"], ok), w.name
        assert np.array_equal(t["perm"], op), w.name
        on = ot.nodes()
        for k in ("level", "prefix", "lo", "hi", "nchild"):
            assert np.array_equal(t[k].astype(np.int64), on[k].astype(np.int64)), (w.name, k)
        if w is DEEP_CHAINS:
            continue
        parity.check_walk(ctx, ot, w, w.theta)


def test_speculated_level_totals_hit_and_miss(bh, oracle):
    """Same n, same varying key bits, another topology: the second build starts its sort on the first one's plan
    (a hit) and enqueues assign + moments on the first one's level totals (a miss: the device-side gate stays
    closed, the kernels return, the host repeats them on the true totals); a third build of the same cells hits
    both.  Every build must equal the oracle's tree, moments and Phi, and the repeated build the one before it
    bit for bit."""
    a, b = wl.random_points(20000, seed=11), wl.random_points(20000, seed=12)
    ka = np.bitwise_or.reduce(oracle.OracleTree(a.x, a.y, a.z, a.m, a.cube).sorted_keys_perm()[0])
    kb = np.bitwise_or.reduce(oracle.OracleTree(b.x, b.y, b.z, b.m, b.cube).sorted_keys_perm()[0])
    assert ka == kb                                   # the premise: the sort plan of one serves the other
    ctx = bh.Context(0)
    prev = None
    for w in (a, b, b, a, a):
        ctx.build(_dev(w.x), _dev(w.y), _dev(w.z), _dev(w.m), w.cube)
        t = _tree_np(ctx)
        ot = oracle.OracleTree(w.x, w.y, w.z, w.m, w.cube)
        ok, op = ot.sorted_keys_perm()
        assert np.array_equal(t["keys"], ok) and np.array_equal(t["perm"], op)
        on = ot.nodes()
        for k in ("level", "prefix", "lo", "hi", "nchild"):
            assert np.array_equal(t[k].astype(np.int64), on[k].astype(np.int64)), k
        assert np.array_equal(t["M"], on["M"])
        phi = ctx.potential(0.5, w.G).cpu().numpy()
        parity.check_walk(ctx, ot, w, 0.5, phi=phi)
        if prev is not None and prev[0] is w:
            assert np.array_equal(phi, prev[1])
        prev = (w, phi)


def test_measured_fma_peak_is_near_nominal(bh):
    """The measured denominator of the walk's roofline (bench.py's aid, its own small library -- not libbh):
    register-resident FMA chains reach most of SMs x 128 lanes x 2 x clock and never exceed it."""
    from paper_1509_07370_b200 import fma_peak
    packed, scalar = fma_peak.measure(0)
    props = torch.cuda.get_device_properties(0)
    nominal = props.multi_processor_count * 128 * 2 * 1.965e9 / 1e12       # at the B200's maximum SM clock
    assert 0.5 * nominal <= scalar <= 1.05 * nominal and 0.5 * nominal <= packed <= 1.05 * nominal, (packed, scalar)
