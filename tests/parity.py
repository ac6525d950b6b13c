"""The parity protocol of the GPU tests (BASELINE.json north_star; W8).

PRIMARY: the CUDA path against the oracle as the paper states the criterion -- d > l/theta (Eq. 3,
PAPER.md:47) or d > l/theta + delta (Eq. 4) evaluated in fp64.  The kernel takes the same
decision in fp32, so a node whose d^2 is within ~1e-7 of r_c^2 for the deciding member can fall on the other
side ("flip"): the group then sums the node's children instead of the node or the reverse.  Groups whose
(accepted, leaf, opened) counters differ from the fp64 oracle's are COUNTED and reported; Phi must agree within
1e-4 max / 1e-6 median relative on the groups that did not flip, within the tree code's own error on those
that did, and the flipped fraction must stay under a stated ceiling.

SECONDARY (flip-free): against the oracle's fp32-decision mode, which is pinned on the CPU by an independent
numpy-float32 restatement (tests/test_oracle_walk.py): counters equal for EVERY group, the number of list
entries the timed Phi kernel itself evaluated (bh_last_group_evaluated) equal to accepted + leaf, Phi within
1e-4 / 1e-6 everywhere.
"""
import numpy as np

MAX_TOL = 1e-4       # north_star: max relative error of Phi
MED_TOL = 1e-6       # north_star: median relative error of Phi
FLIP_CEILING = 0.05  # stated ceiling on the fraction of groups whose list differs from the fp64 oracle's


def tree_tol(theta):
    """Bound on |dPhi|/|Phi| of a group whose list differs by flipped nodes: far below the Barnes-Hut error
    itself (max 5e-3 at theta 0.5, 5e-2 at theta 1 on the oracle's own pins, tests/test_oracle_walk.py)."""
    return max(2e-4, 0.02 * theta * theta)


def _rel(phi, ref):
    ok = ref != 0
    assert np.all(phi[~ok] == 0.0)
    return np.abs(phi[ok] - ref[ok]) / np.abs(ref[ok])


def check_walk(ctx, ot, w, theta, mac=0, group=32, runs=None, phi=None, max_tol=MAX_TOL, med_tol=MED_TOL,
               flip_ceiling=FLIP_CEILING, check_phi=True, label=""):
    """Runs bh_potential (unless `phi` is given: a numpy array of the last walk's result) and applies both
    comparisons on the groups in `runs` (list of (g0, g1); None = all groups).  Returns a report dict."""
    ctx.set_mac(mac)
    ctx.set_group(group)
    if phi is None:
        phi = ctx.potential(theta, w.G).cpu().numpy()
    cnt = ctx.last_group_counts().cpu().numpy()
    ev = ctx.last_group_evaluated().cpu().numpy().astype(np.int64)
    perm = ot.sorted_keys_perm()[1].astype(np.int64)
    n = w.n
    ngroups = (n + group - 1) // group
    assert cnt.shape == (ngroups, 3) and ev.shape == (ngroups,)
    if runs is None:
        runs = [(0, ngroups)]
    b64, b32 = np.full(n, np.nan), np.full(n, np.nan)
    rel_keep, rel_flip, rel32 = [], [], []
    flips = ng = 0
    for g0, g1 in runs:
        _, c64 = ot.potential(theta, w.G, mac=mac, group=group, mac_fp32=False, groups=(g0, g1), want_counts=True, out=b64)
        _, c32 = ot.potential(theta, w.G, mac=mac, group=group, mac_fp32=True, groups=(g0, g1), want_counts=True, out=b32)
        # secondary, flip-free: the same decisions in the same precision give the same lists
        bad = np.any(cnt[g0:g1] != c32, axis=1)
        assert not bad.any(), f"{label}: {int(bad.sum())} of {g1 - g0} groups differ from the fp32-decision oracle"
        assert np.array_equal(ev[g0:g1], c32[:, 0] + c32[:, 1]), f"{label}: the Phi kernel's own entry counts differ"
        flipped = np.any(cnt[g0:g1] != c64, axis=1)
        flips += int(flipped.sum())
        ng += g1 - g0
        if not check_phi:
            continue
        for g in range(g0, g1):
            tg = perm[group * g:min(group * (g + 1), n)]
            (rel_flip if flipped[g - g0] else rel_keep).append(_rel(phi[tg], b64[tg]))
            rel32.append(_rel(phi[tg], b32[tg]))
    rep = {"groups": ng, "flips_fp32_vs_fp64": flips, "theta": theta, "mac": mac, "group": group}
    assert flips <= flip_ceiling * ng + 1, f"{label}: {flips} of {ng} groups flipped"
    if check_phi:
        keep = np.concatenate(rel_keep) if rel_keep else np.zeros(0)
        flp = np.concatenate(rel_flip) if rel_flip else np.zeros(0)
        r32 = np.concatenate(rel32) if rel32 else np.zeros(0)
        if keep.size:
            rep["max_rel"], rep["median_rel"] = float(keep.max()), float(np.median(keep))
            assert keep.max() <= max_tol, f"{label}: max rel {keep.max():.3e} vs the fp64 oracle"
            assert np.median(keep) <= med_tol, f"{label}: median rel {np.median(keep):.3e} vs the fp64 oracle"
        if flp.size:
            rep["max_rel_flipped"] = float(flp.max())
            assert flp.max() <= tree_tol(theta), f"{label}: flipped groups off by {flp.max():.3e}"
        if r32.size:
            assert r32.max() <= max_tol and np.median(r32) <= med_tol, (label, r32.max(), np.median(r32))
    print(f"parity {label or w.name} theta={theta} mac={mac} group={group}: {ng} groups, "
          f"{flips} flips fp32-vs-fp64, max rel {rep.get('max_rel', 0):.2e}, median {rep.get('median_rel', 0):.2e}"
          + (f", flipped groups max {rep['max_rel_flipped']:.2e}" if "max_rel_flipped" in rep else ""))
    rep["phi"] = phi
    rep["counts"] = cnt
    return rep


def sample_runs(ngroups, nruns, per):
    """`nruns` evenly spaced runs of `per` consecutive groups, first and last group included."""
    per = min(per, ngroups)
    starts = np.unique(np.linspace(0, ngroups - per, nruns).astype(np.int64))
    return [(int(s), int(s) + per) for s in starts]


def check_field(ctx, ot, w, theta, acc, mac=0, group=32, runs=None, max_tol=MAX_TOL, med_tol=MED_TOL,
                flip_ceiling=FLIP_CEILING, label=""):
    """g = -grad Phi of the LAST bh_field call (`acc`: numpy [n, 3]) under the same protocol: against the oracle's
    field with fp64 decisions on the groups whose lists agree (flipped groups counted, held to 10 x the tree
    tolerance -- a gradient feels a swapped node more than a potential), and against the fp32-decision mode on
    every group.  `max_tol` / `med_tol`: the bars DESIGN.md §9c derives for g."""
    cnt = ctx.last_group_counts().cpu().numpy()
    perm = ot.sorted_keys_perm()[1].astype(np.int64)
    n = w.n
    ngroups = (n + group - 1) // group
    if runs is None:
        runs = [(0, ngroups)]
    keep, flp, r32 = [], [], []
    flips = ng = 0
    pbuf = np.full(n, np.nan)
    o64, o32 = (pbuf, np.full((n, 3), np.nan)), (pbuf, np.full((n, 3), np.nan))

    def rel(a, ref):
        nr = np.linalg.norm(ref, axis=1)
        ok = nr > 0
        return np.linalg.norm(a - ref, axis=1)[ok] / nr[ok]

    for g0, g1 in runs:
        _, c64 = ot.potential(theta, w.G, mac=mac, group=group, mac_fp32=False, groups=(g0, g1), want_counts=True,
                              out=pbuf)
        _, a64 = ot.field(theta, w.G, mac=mac, group=group, mac_fp32=False, groups=(g0, g1), out=o64)
        _, a32 = ot.field(theta, w.G, mac=mac, group=group, mac_fp32=True, groups=(g0, g1), out=o32)
        flipped = np.any(cnt[g0:g1] != c64, axis=1)
        flips += int(flipped.sum())
        ng += g1 - g0
        for g in range(g0, g1):
            tg = perm[group * g:min(group * (g + 1), n)]
            (flp if flipped[g - g0] else keep).append(rel(acc[tg], a64[tg]))
            r32.append(rel(acc[tg], a32[tg]))
    assert flips <= flip_ceiling * ng + 1, f"{label}: {flips} of {ng} groups flipped"
    keep = np.concatenate(keep) if keep else np.zeros(0)
    flp = np.concatenate(flp) if flp else np.zeros(0)
    r32 = np.concatenate(r32)
    if keep.size:
        assert keep.max() <= max_tol and np.median(keep) <= med_tol, (label, keep.max(), np.median(keep))
    if flp.size:
        assert flp.max() <= max(10 * tree_tol(theta), max_tol), (label, flp.max())
    if r32.size:
        assert r32.max() <= max_tol and np.median(r32) <= med_tol, (label, r32.max(), np.median(r32))
    print(f"field parity {label or w.name} theta={theta} mac={mac} group={group}: {ng} groups, {flips} flips, "
          f"max rel {keep.max() if keep.size else 0:.2e}, median {np.median(keep) if keep.size else 0:.2e}")
    return {"groups": ng, "flips_fp32_vs_fp64": flips}
