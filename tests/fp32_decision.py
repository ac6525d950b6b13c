"""An independent numpy-float32 restatement of DESIGN.md reading W8 (the opening decision in the kernel's
arithmetic type), used to PIN the oracle's `mac_fp32` branch (oracle/bh_oracle.c, group_accepts) on the CPU.

W8: operands rounded to fp32 -- (float) of the fp64 sorted position, of R, of l, of delta, of 1/theta;
r_c = l * (1/theta) [+ delta]; r_c^2 = r_c * r_c; d^2 = fma(dz, dz, fma(dy, dy, dx * dx)) with
dx = x_t - R_x etc.; accept iff d^2 > r_c^2 for EVERY member of the group.

Nothing here is shared with oracle/ or with the CUDA path: the fused multiply-add is built from exact
float64 products and an error-free sum, the walk is a plain Python depth-first search over the node list
the oracle exports (level, lo, hi, M, R, delta), and only the per-group counters are compared.
"""
import numpy as np

F32 = np.float32


def fma32(a, b, c):
    """Correctly rounded float32 fma(a, b, c) for float32 arrays: the product of two float32 is exact in
    float64; the sum with c is made error-free (TwoSum: s + err == a*b + c exactly) and rounded ONCE to
    float32 -- when the float64 sum s sits exactly on the midpoint of two float32 neighbours, the residual
    err decides the direction, so there is no double rounding."""
    a, b, c = (np.asarray(v, dtype=F32).astype(np.float64) for v in (a, b, c))
    p = a * b                                   # exact: 24 x 24 bits
    s = p + c
    bb = s - p
    err = (p - (s - bb)) + (c - bb)             # TwoSum residual
    rd = s.astype(F32)                          # round-to-nearest-even of s
    rd64 = rd.astype(np.float64)
    lo = np.where(rd64 > s, np.nextafter(rd, F32(-np.inf)), rd).astype(F32)
    hi = np.where(rd64 < s, np.nextafter(rd, F32(np.inf)), rd).astype(F32)
    mid = 0.5 * (lo.astype(np.float64) + hi.astype(np.float64))
    on_mid = (lo != hi) & (s == mid) & (err != 0)
    return np.where(on_mid, np.where(err > 0, hi, lo), rd).astype(F32)


def d2_fp32(tx, ty, tz, R):
    """fp32 squared distance of fp32-rounded targets to the fp32-rounded point R, nesting of W8."""
    dx = (np.asarray(tx, F32) - F32(R[0])).astype(F32)
    dy = (np.asarray(ty, F32) - F32(R[1])).astype(F32)
    dz = (np.asarray(tz, F32) - F32(R[2])).astype(F32)
    return fma32(dz, dz, fma32(dy, dy, (dx * dx).astype(F32)))


def rc2_fp32(size, delta, theta, mac):
    """r_c^2 of W8: r_c = l * (1/theta) (+ delta with Eq. 4), every operand and result fp32."""
    rc = F32(F32(size) * F32(1.0 / theta))
    if mac == 1:
        rc = F32(rc + F32(delta))
    return F32(rc * rc)


def group_accepts_fp32(tx, ty, tz, R, size, delta, theta, mac):
    if theta == 0.0:
        return False
    return bool(np.all(d2_fp32(tx, ty, tz, R) > rc2_fp32(size, delta, theta, mac)))


def children_of(nodes):
    """child lists from the canonical node list: per node a list of ('n', node index) / ('c', sorted cell),
    ascending cell order (= ascending octant order).  A level-21 node (bucket) has only cells."""
    start = {(int(l), int(lo)): i for i, (l, lo) in enumerate(zip(nodes["level"], nodes["lo"]))}
    out = []
    for i in range(len(nodes["level"])):
        lev, lo, hi = int(nodes["level"][i]), int(nodes["lo"][i]), int(nodes["hi"][i])
        ch, s = [], lo
        while s < hi:
            j = start.get((lev + 1, s)) if lev < 21 else None
            if j is None:
                ch.append(("c", s)); s += 1
            else:
                ch.append(("n", j)); s = int(nodes["hi"][j])
        out.append(ch)
    return out


def walk_counts_fp32(xs, ys, zs, nodes, L, theta, mac=0, group=32):
    """(accepted, leaf, opened) per group of `group` consecutive sorted cells (W1-W6) with the opening
    decision of W8.  xs, ys, zs: fp64 positions in SORTED order; nodes: the oracle's canonical node list."""
    n = len(xs)
    kids = children_of(nodes)
    root = {(int(l), int(lo)): i for i, (l, lo) in enumerate(zip(nodes["level"], nodes["lo"]))}.get((0, 0))
    ng = (n + group - 1) // group
    counts = np.zeros((ng, 3), dtype=np.int64)
    x32, y32, z32 = xs.astype(F32), ys.astype(F32), zs.astype(F32)
    for g in range(ng):
        t0, t1 = g * group, min(n, (g + 1) * group)
        tx, ty, tz = x32[t0:t1], y32[t0:t1], z32[t0:t1]
        stack = [("n", root)] if n >= 2 else []
        acc = leaf = opened = 0
        while stack:
            kind, i = stack.pop()
            if kind == "c":
                leaf += 1
                continue
            if int(nodes["level"][i]) == 21:                       # bucket: all its cells, neither accepted nor opened
                leaf += len(kids[i])
                continue
            R = (nodes["Rx"][i], nodes["Ry"][i], nodes["Rz"][i])
            size = np.ldexp(L, -int(nodes["level"][i]))
            if group_accepts_fp32(tx, ty, tz, R, size, nodes["delta"][i], theta, mac):
                acc += 1
            else:
                opened += 1
                stack.extend(reversed(kids[i]))
        counts[g] = (acc, leaf, opened)
    return counts
