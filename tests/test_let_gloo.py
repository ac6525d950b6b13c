"""N > 1 host logic of the locally-essential-tree solve on CPU (gloo, world_size 2 and 3): the box
all-gather, the count exchange and the point-to-point record exchange of paper_1509_07370_b200/let.py.
libbh cannot run here (no GPU, no CPU fallback), so the two device steps are injected: `select` and
`solve` call the ORACLE (tests may).  The distributed result must equal the same procedure done in one
process, and sit at Barnes-Hut accuracy against the direct sum over all ranks' cells."""
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _split(w, world):
    order = np.argsort(w.x, kind="stable")
    return [np.sort(c) for c in np.array_split(order, world)]


def _oracle_select(x, y, z, m, cube, boxes, theta, mac):
    import oracle
    t = oracle.OracleTree(x.numpy(), y.numpy(), z.numpy(), m.numpy(), cube)
    return [None if b is None else torch.from_numpy(t.essential_nodes(b[0], b[1], theta, mac=mac)) for b in boxes]


def _oracle_solve(x, y, z, m, cube, n_targets, theta, G, mac):
    import oracle
    t = oracle.OracleTree(x.numpy(), y.numpy(), z.numpy(), m.numpy(), cube)
    return torch.from_numpy(t.potential(theta, G, mac=mac)[:n_targets].copy())


def _worker(rank, world, port, q, empty_rank):
    import torch.distributed as dist
    import bh_workloads as wl
    import oracle
    from paper_1509_07370_b200 import let
    oracle.build_library()
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    w = wl.clustered_points(1500, seed=77)
    owners = world - (1 if empty_rank is not None else 0)
    parts = _split(w, owners)
    if empty_rank is not None:
        parts.insert(empty_rank, np.zeros(0, dtype=np.int64))       # a rank without cells
    i = parts[rank]
    t = [torch.from_numpy(np.ascontiguousarray(a[i])) for a in (w.x, w.y, w.z, w.m)]
    phi, info = let.let_potential(*t, w.cube, 0.5, w.G, mac=1, select=_oracle_select, solve=_oracle_solve)
    q.put((rank, phi.numpy(), info))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,empty_rank", [(2, None), (3, None), (3, 1)])
def test_let_over_gloo_ranks_equals_one_process(oracle, world, empty_rank):
    import torch.multiprocessing as mp
    import bh_workloads as wl
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q, empty_rank)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # the same procedure in this process
    w = wl.clustered_points(1500, seed=77)
    owners = world - (1 if empty_rank is not None else 0)
    parts = _split(w, owners)
    if empty_rank is not None:
        parts.insert(empty_rank, np.zeros(0, dtype=np.int64))
    boxes = [None if len(i) == 0 else ((w.x[i].min(), w.y[i].min(), w.z[i].min()), (w.x[i].max(), w.y[i].max(), w.z[i].max()))
             for i in parts]
    inbox = [[] for _ in parts]
    sent = [[0] * world for _ in parts]
    for d, i in enumerate(parts):
        if len(i) == 0:
            continue
        t = oracle.OracleTree(w.x[i], w.y[i], w.z[i], w.m[i], w.cube)
        for e in range(world):
            if e != d and boxes[e] is not None:
                rec = t.essential_nodes(boxes[e][0], boxes[e][1], 0.5, mac=1)
                sent[d][e] = len(rec)
                inbox[e].append(rec)
    exact = oracle.direct(w.x, w.y, w.z, w.m, w.G)
    for (rank, phi, info), i in zip(got, parts):
        assert info["sent"] == sent[rank]
        assert info["received"] == [sent[d][rank] for d in range(world)]
        if len(i) == 0:
            assert phi.shape == (0,)
            continue
        ext = np.concatenate(inbox[rank]) if inbox[rank] else np.zeros((0, 4))
        u = [np.concatenate([a[i], ext[:, k]]) for k, a in enumerate((w.x, w.y, w.z, w.m))]
        ref = oracle.OracleTree(*u, w.cube).potential(0.5, w.G, mac=1)[: len(i)]
        assert np.array_equal(phi, ref)
        err = np.abs(phi - exact[i]) / np.abs(exact[i])
        assert err.max() < 1e-2


def test_single_process_let_is_plain_solve():
    """Without a process group the LET solve is the plain solve over the own cells."""
    from paper_1509_07370_b200 import let
    x = torch.tensor([0.1, 0.6, 0.7], dtype=torch.float64)
    calls = []

    def solve(x, y, z, m, cube, n_targets, theta, G, mac):
        calls.append((int(x.shape[0]), n_targets))
        return torch.zeros(n_targets, dtype=torch.float64)

    phi, info = let.let_potential(x, x, x, x, (0, 0, 0, 1), 0.5, select=lambda *a: [], solve=solve)
    assert calls == [(3, 3)] and phi.shape == (3,) and info["world"] == 1
    lo, hi = let.domain_box(x, x, x)
    assert lo == (0.1, 0.1, 0.1) and hi == (0.7, 0.7, 0.7)
