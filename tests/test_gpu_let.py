"""GPU parity for NEXT-1: Find Essential Nodes and the locally
essential tree built from them, through the C ABI, against the fp64 oracle.

Bars: the essential set is selected in fp64 on bit-identical moments, so entries, order and values are
compared for EQUALITY; Phi of a LET walk within max 1e-4 / median 1e-6 relative of the oracle run through
the same procedure with the criterion in fp64 (targets of groups whose list flipped between fp32 and fp64
decisions are counted, reported and held to the tree code's own error; tests/parity.py), the same bars against
the CPU-pinned fp32-decision mode on every target, and Barnes-Hut accuracy against the fp64 direct sum over
ALL cells of all domains."""
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
        p64, c64 = t.potential(theta, w.G, mac=mac, want_counts=True)
        p32, c32 = t.potential(theta, w.G, mac=mac, mac_fp32=True, want_counts=True)
        flipped_group = np.any(c64 != c32, axis=1)
        inv = np.empty(len(u[0]), dtype=np.int64)
        inv[t.sorted_keys_perm()[1].astype(np.int64)] = np.arange(len(u[0]))       # sorted slot of every cell
        phis.append((p64[: len(i)], p32[: len(i)], flipped_group[inv[: len(i)] // 32]))
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
    for i, p, (op64, op32, flipped) in zip(parts, phis, ophis):
        p = p.cpu().numpy()
        assert p.shape == op64.shape
        rel32 = parity._rel(p, op32)                                        # flip-free: fp32 decisions on both sides
        assert rel32.max() <= 1e-4 and np.median(rel32) <= 1e-6, (rel32.max(), np.median(rel32))
        nz = op64 != 0
        rel = np.abs(p - op64)[nz] / np.abs(op64[nz])
        keep = ~flipped[nz]
        assert rel[keep].max() <= 1e-4 and np.median(rel[keep]) <= 1e-6, (rel[keep].max(), np.median(rel[keep]))
        assert flipped.mean() <= parity.FLIP_CEILING and (keep.all() or rel[~keep].max() <= parity.tree_tol(theta))
        print(f"LET {w.name} P={P}: {int(flipped.sum())} of {len(i)} targets sit in groups whose list flipped fp32-vs-fp64")
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


# ---- the multi-process product path: let.let_potential with libbh's own select / solve ----
def _free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _let_worker(rank, world, port, q, empty_rank, name):
    """One rank of a gloo group; all ranks share cuda:0 (the kernels of different ranks never wait on each
    other: the only cross-rank steps are host-side gloo calls).  Default select / solve = libbh."""
    import torch.distributed as dist
    import bh_workloads as wl_
    from paper_1509_07370_b200 import let
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = _LET_INPUTS[name]()
    owners = world - (1 if empty_rank is not None else 0)
    parts = _slabs(w, owners)
    if empty_rank is not None:
        parts.insert(empty_rank, np.zeros(0, dtype=np.int64))       # a rank without cells
    i = parts[rank]
    t = [torch.from_numpy(np.ascontiguousarray(a[i])).cuda() for a in (w.x, w.y, w.z, w.m)]
    phi, info = let.let_potential(*t, w.cube, 0.5, w.G, mac=1)        # the product path: no select / solve injected
    q.put((rank, phi.cpu().numpy(), info))
    dist.barrier()
    dist.destroy_process_group()


_LET_INPUTS = {"clustered": lambda: wl.clustered_points(6000, seed=41),
               "amr": lambda: wl.amr_collapsing_core(nroot=2, max_level=3)}


@pytest.mark.parametrize("world,empty_rank,name", [(2, None, "clustered"), (3, None, "amr"), (3, 1, "clustered")])
def test_let_across_processes_with_product_kernels(bh, oracle, world, empty_rank, name):
    """let.let_potential under a real process group (gloo; the records are staged through host tensors), every
    rank running bh_build / bh_essential_nodes / bh_potential of libbh on the GPU: entry counts equal to the
    oracle procedure's, Phi within the bars of tests/parity.py, Barnes-Hut accuracy against the direct sum."""
    import torch.multiprocessing as mp
    theta, mac = 0.5, 1
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_let_worker, args=(r, world, port, q, empty_rank, name)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=600) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = _LET_INPUTS[name]()
    owners = world - (1 if empty_rank is not None else 0)
    own_parts = _slabs(w, owners)
    ophis, osent = _oracle_let(oracle, w, own_parts, theta, mac)
    ranks_with_cells = [r for r in range(world) if r != empty_rank]
    exact = None
    for k, r in enumerate(ranks_with_cells):
        rank, phi, info = got[r]
        assert info["sent"] == [0 if e == empty_rank or e == r else osent[k][ranks_with_cells.index(e)] for e in range(world)]
        assert info["received"] == [0 if e == empty_rank or e == r else osent[ranks_with_cells.index(e)][k] for e in range(world)]
        op64, op32, flipped = ophis[k]
        assert phi.shape == op64.shape
        rel32 = parity._rel(phi, op32)
        assert rel32.max() <= 1e-4 and np.median(rel32) <= 1e-6, (rel32.max(), np.median(rel32))
        rel = np.abs(phi - op64) / np.abs(op64)
        assert rel[~flipped].max() <= 1e-4 and np.median(rel[~flipped]) <= 1e-6
        assert flipped.mean() <= parity.FLIP_CEILING and (not flipped.any() or rel[flipped].max() <= parity.tree_tol(theta))
        i = own_parts[k]
        sub = np.random.default_rng(11 + k).choice(len(i), size=min(128, len(i)), replace=False)
        ex = oracle.direct(w.x, w.y, w.z, w.m, w.G, targets=i[sub].astype(np.int64))
        assert (np.abs(phi[sub] - ex) / np.abs(ex)).max() < 1e-2
    if empty_rank is not None:
        assert got[empty_rank][1].shape == (0,) and sum(got[empty_rank][2]["sent"]) == 0


# ---- the fused selection + exchange: bh_essential_nodes gathers straight into the RECEIVER's memory ----------------
def _peer_worker(rank, world, port, q, mail, name):
    """Every rank allocates one inbox per sender and hands it to that sender through a torch.multiprocessing queue
    (CUDA IPC: the buffer is mapped into the sender's process); senders then select with the mapped buffer as `out`."""
    import torch.distributed as dist
    from paper_1509_07370_b200 import let, binding
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    w = _LET_INPUTS[name]()
    parts = _slabs(w, world)
    i = parts[rank]
    t = [torch.from_numpy(np.ascontiguousarray(a[i])).cuda() for a in (w.x, w.y, w.z, w.m)]
    cap = w.n                                                        # an essential set never exceeds the sender's cells
    inbox = [None if s == rank else torch.zeros((cap, 4), dtype=torch.float64, device="cuda") for s in range(world)]
    for s in range(world):
        if s != rank:
            mail[s].put((rank, inbox[s]))                            # rank s will write its records for us in here
    peer_out = [None] * world
    for _ in range(world - 1):
        r, buf = mail[rank].get(timeout=300)
        peer_out[r] = buf
    ctx = binding.Context(0)
    ctx.set_mac(1)
    phi, info = let.let_potential(*t, w.cube, 0.5, w.G, mac=1, ctx=ctx, peer_out=peer_out, inbox=inbox)
    phi2, info2 = let.let_potential(*t, w.cube, 0.5, w.G, mac=1, ctx=ctx, peer_out=peer_out, inbox=inbox)   # buffers reused
    assert torch.equal(phi, phi2) and info2["received"] == info["received"]
    q.put((rank, phi.cpu().numpy(), info))
    dist.barrier()
    del peer_out
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,name", [(2, "clustered"), (3, "amr")])
def test_let_with_peer_mapped_inboxes(bh, oracle, world, name):
    """The essential-node records go from the selecting kernel straight into the receiving process's device buffer
    (mapped through CUDA IPC; over NVLink the same pointer arithmetic is a P2P store): no send / receive calls, one
    all-gather of counts.  Same results as the oracle procedure."""
    import torch.multiprocessing as mp
    theta, mac = 0.5, 1
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    mail = [ctx.Queue() for _ in range(world)]
    port = _free_port()
    procs = [ctx.Process(target=_peer_worker, args=(r, world, port, q, mail, name)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=600) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = _LET_INPUTS[name]()
    parts = _slabs(w, world)
    ophis, osent = _oracle_let(oracle, w, parts, theta, mac)
    for r, (rank, phi, info) in enumerate(got):
        assert info["sent"] == osent[r] and info["received"] == [osent[s][r] for s in range(world)]
        op64, op32, flipped = ophis[r]
        rel32 = parity._rel(phi, op32)
        assert rel32.max() <= 1e-4 and np.median(rel32) <= 1e-6, (rel32.max(), np.median(rel32))
        rel = np.abs(phi - op64) / np.abs(op64)
        assert rel[~flipped].max() <= 1e-4 and np.median(rel[~flipped]) <= 1e-6
