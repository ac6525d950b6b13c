"""ctypes wrapper of oracle/bh_oracle.c (test infrastructure; see the C file's header).

Argument marshalling only -- every number comes from the C code.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bh_oracle.c")
_LIB = os.path.join(_HERE, "libbh_oracle.so")

MAC_BH86 = 0      # Eq. 3
MAC_BARNES94 = 1  # Eq. 4


def build_library(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off (K-rule 1: no FMA contraction in the key expression)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-Wall", "-fPIC", "-shared",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_library())
        dp, u64p, u32p, i64p, i32p = (C.POINTER(C.c_double), C.POINTER(C.c_uint64), C.POINTER(C.c_uint32),
                                      C.POINTER(C.c_int64), C.POINTER(C.c_int32))
        lib.orc_keys.argtypes = [dp, dp, dp, C.c_int64, dp, u64p, i64p]
        lib.orc_sort.argtypes = [u64p, C.c_int64, u32p]
        lib.orc_build.argtypes = [dp, dp, dp, dp, C.c_int64, dp]
        lib.orc_build.restype = C.c_void_p
        lib.orc_free.argtypes = [C.c_void_p]
        lib.orc_free.restype = None
        for f in ("orc_num_cells", "orc_num_nodes", "orc_num_clamped"):
            getattr(lib, f).argtypes = [C.c_void_p]
            getattr(lib, f).restype = C.c_int64
        lib.orc_depth.argtypes = [C.c_void_p]
        lib.orc_depth.restype = C.c_int32
        lib.orc_get_sorted.argtypes = [C.c_void_p, u64p, u32p]
        lib.orc_export_nodes.argtypes = [C.c_void_p, i32p, u64p, i64p, i64p, dp, dp, dp, dp, dp, i32p]
        lib.orc_potential.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                                      C.c_int64, C.c_int64, dp, i64p]
        lib.orc_direct.argtypes = [dp, dp, dp, dp, C.c_int64, C.c_double, i64p, C.c_int64, dp]
        lib.orc_field.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int,
                                  C.c_int64, C.c_int64, dp, dp, i64p]
        lib.orc_direct_acc.argtypes = [dp, dp, dp, dp, C.c_int64, C.c_double, i64p, C.c_int64, dp]
        lib.orc_essential_nodes.argtypes = [C.c_void_p, dp, dp, C.c_double, C.c_int, dp, i32p, i64p, i64p]
        lib.orc_essential_nodes.restype = C.c_int64
        lib.orc_ewald_psi.argtypes = [dp, C.c_double, C.c_int]
        lib.orc_ewald_psi.restype = C.c_double
        lib.orc_ewald_corr.argtypes = [dp, C.c_double, C.c_int]
        lib.orc_ewald_corr.restype = C.c_double
        lib.orc_ewald_table.argtypes = [C.c_int, C.c_int, C.c_double, C.c_int, dp]
        lib.orc_ewald_interp.argtypes = [dp, C.c_int, C.c_int, dp]
        lib.orc_ewald_interp.restype = C.c_double
        lib.orc_potential_periodic.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int, C.c_int, dp, C.c_int, C.c_int,
                                               C.c_int64, C.c_int64, dp, i64p]
        _lib = lib
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def keys(x, y, z, cube):
    """63-bit Morton keys in the caller's order; returns (keys uint64[n], n_clamped)."""
    x, y, z, cube = _f64(x), _f64(y), _f64(z), _f64(cube)
    out = np.empty(x.shape[0], dtype=np.uint64)
    nc = C.c_int64(0)
    rc = _L().orc_keys(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), x.shape[0],
                       _p(cube, C.c_double), _p(out, C.c_uint64), C.byref(nc))
    if rc != 0:
        raise ValueError("orc_keys: invalid argument")
    return out, int(nc.value)


def sort_perm(k):
    """Stable ascending (key, index) order: perm[s] = original index of sorted slot s."""
    k = np.ascontiguousarray(k, dtype=np.uint64)
    perm = np.empty(k.shape[0], dtype=np.uint32)
    if _L().orc_sort(_p(k, C.c_uint64), k.shape[0], _p(perm, C.c_uint32)) != 0:
        raise ValueError("orc_sort failed")
    return perm


def direct(x, y, z, m, G=1.0, targets=None):
    """Eq. 2: Phi_i = -G sum_{j!=i} m_j/|r_i-r_j| for all i or the listed targets."""
    x, y, z, m = _f64(x), _f64(y), _f64(z), _f64(m)
    n = x.shape[0]
    if targets is None:
        phi = np.empty(n, dtype=np.float64)
        rc = _L().orc_direct(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(m, C.c_double), n,
                             G, None, 0, _p(phi, C.c_double))
    else:
        t = np.ascontiguousarray(targets, dtype=np.int64)
        phi = np.empty(t.shape[0], dtype=np.float64)
        rc = _L().orc_direct(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(m, C.c_double), n,
                             G, _p(t, C.c_int64), t.shape[0], _p(phi, C.c_double))
    if rc != 0:
        raise ValueError("orc_direct: invalid argument")
    return phi


def direct_acc(x, y, z, m, G=1.0, targets=None):
    """g_i = -grad Phi_i of Eq. 2 written out: -G sum_{j!=i} m_j (r_i-r_j)/|r_i-r_j|^3; returns [count, 3]."""
    x, y, z, m = _f64(x), _f64(y), _f64(z), _f64(m)
    n = x.shape[0]
    t = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    cnt = n if t is None else t.shape[0]
    acc = np.empty((cnt, 3), dtype=np.float64)
    rc = _L().orc_direct_acc(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(m, C.c_double), n, G,
                             None if t is None else _p(t, C.c_int64), cnt, _p(acc, C.c_double))
    if rc != 0:
        raise ValueError("orc_direct_acc: invalid argument")
    return acc


def ewald_psi(u, a=2.0, nser=5):
    """psi1(u): the Ewald sum of 1/r in the unit cube with neutralising background (Eq. A.1-A.3;
    DESIGN.md reading P1), u = r/L; a = alpha L; sums over |n_i|, |h_i| <= nser."""
    u = _f64(u)
    return float(_L().orc_ewald_psi(_p(u, C.c_double), float(a), int(nser)))


def ewald_corr(u, a=2.0, nser=5):
    """corr1(u) = psi1(u) - 1/|u| (its finite limit at u = 0): what the field array tabulates (reading P2)."""
    u = _f64(u)
    return float(_L().orc_ewald_corr(_p(u, C.c_double), float(a), int(nser)))


class EwaldTable:
    """The nested-grid Ewald field array (readings P3, P4): `nref` grids of N^3 points of corr1
    on the octant u_a >= 0, spacing (1/2)/(N-2)/2^k (u = 1/2^(k+1) is point N-2 of grid k); quadratic interpolation."""

    def __init__(self, N=32, nref=1, a=2.0, nser=5):
        self.N, self.nref, self.a, self.nser = int(N), int(nref), float(a), int(nser)
        self.data = np.empty(self.nref * self.N ** 3, dtype=np.float64)
        if _L().orc_ewald_table(self.N, self.nref, self.a, self.nser, _p(self.data, C.c_double)) != 0:
            raise ValueError("orc_ewald_table: invalid argument")

    def grid(self, lev=0):
        return self.data[lev * self.N ** 3:(lev + 1) * self.N ** 3].reshape(self.N, self.N, self.N)   # [k][j][i]

    def interp(self, u):
        u = _f64(u)
        return float(_L().orc_ewald_interp(_p(self.data, C.c_double), self.N, self.nref, _p(u, C.c_double)))


class OracleTree:
    """keys -> sort -> octree -> monopoles for one set of cells (orc_build)."""

    def __init__(self, x, y, z, m, cube):
        x, y, z, m, cube = _f64(x), _f64(y), _f64(z), _f64(m), _f64(cube)
        self._h = _L().orc_build(_p(x, C.c_double), _p(y, C.c_double), _p(z, C.c_double), _p(m, C.c_double),
                                 x.shape[0], _p(cube, C.c_double))
        if not self._h:
            raise ValueError("orc_build: invalid argument or out of memory")
        self.n = int(_L().orc_num_cells(self._h))
        self.n_nodes = int(_L().orc_num_nodes(self._h))      # internal nodes + level-21 buckets
        self.n_clamped = int(_L().orc_num_clamped(self._h))
        self.depth = int(_L().orc_depth(self._h))

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            _L().orc_free(h)
            self._h = None

    def sorted_keys_perm(self):
        k = np.empty(self.n, dtype=np.uint64)
        p = np.empty(self.n, dtype=np.uint32)
        _L().orc_get_sorted(self._h, _p(k, C.c_uint64), _p(p, C.c_uint32))
        return k, p

    def nodes(self):
        """Canonical node list (sorted by (level, prefix)) as a dict of arrays."""
        nn = self.n_nodes
        out = dict(level=np.empty(nn, np.int32), prefix=np.empty(nn, np.uint64), lo=np.empty(nn, np.int64),
                   hi=np.empty(nn, np.int64), M=np.empty(nn), Rx=np.empty(nn), Ry=np.empty(nn), Rz=np.empty(nn),
                   delta=np.empty(nn), nchild=np.empty(nn, np.int32))
        _L().orc_export_nodes(self._h, _p(out["level"], C.c_int32), _p(out["prefix"], C.c_uint64),
                              _p(out["lo"], C.c_int64), _p(out["hi"], C.c_int64), _p(out["M"], C.c_double),
                              _p(out["Rx"], C.c_double), _p(out["Ry"], C.c_double), _p(out["Rz"], C.c_double),
                              _p(out["delta"], C.c_double), _p(out["nchild"], C.c_int32))
        return out

    def potential(self, theta, G=1.0, mac=MAC_BH86, group=32, mac_fp32=False, groups=None, want_counts=False,
                  out=None):
        """Group walk (W-rules).  Returns phi in ORIGINAL order (NaN where not walked when `groups`
        = (begin, end) restricts the walk) and, if asked, counts[ngroups_walked, 3] =
        (accepted nodes, leaf cells, opened nodes).  `out`: reuse a float64[n] buffer (marshalling only)."""
        ng = (self.n + group - 1) // group
        gb, ge = (0, ng) if groups is None else groups
        phi = np.full(self.n, np.nan) if out is None else out
        counts = np.zeros((max(ge - gb, 0), 3), dtype=np.int64)
        rc = _L().orc_potential(self._h, float(theta), float(G), int(mac), int(group), int(bool(mac_fp32)),
                                gb, ge, _p(phi, C.c_double), _p(counts, C.c_int64))
        if rc != 0:
            raise ValueError("orc_potential: invalid argument")
        return (phi, counts) if want_counts else phi

    def potential_periodic(self, theta, table, G=1.0, mac=MAC_BH86, group=32, groups=None, want_counts=False, out=None):
        """The group walk under periodic boundaries (App. A; reading P5): minimum-image displacements in the opening
        test and the sums, every entry contributing M (1/d + corr1(d/L)/L) with corr1 interpolated in `table`
        (an EwaldTable); the tree's cube is the periodic box.  Decisions in fp64."""
        ng = (self.n + group - 1) // group
        gb, ge = (0, ng) if groups is None else groups
        phi = np.full(self.n, np.nan) if out is None else out
        counts = np.zeros((max(ge - gb, 0), 3), dtype=np.int64)
        rc = _L().orc_potential_periodic(self._h, float(theta), float(G), int(mac), int(group),
                                         _p(table.data, C.c_double), table.N, table.nref, gb, ge,
                                         _p(phi, C.c_double), _p(counts, C.c_int64))
        if rc != 0:
            raise ValueError("orc_potential_periodic: invalid argument")
        return (phi, counts) if want_counts else phi

    def essential_nodes(self, box_lo, box_hi, theta, mac=MAC_BARNES94, want_ranges=False):
        """Find Essential Nodes: this tree pruned against the remote domain box
        [box_lo, box_hi] with the minimum-distance criterion.  Returns rec[k, 4] = (x, y, z, m) in
        ascending (level, first sorted cell) order and, if asked, (level, lo, hi) per entry."""
        blo, bhi = _f64(box_lo), _f64(box_hi)
        rec = np.empty((max(self.n, 1), 4), dtype=np.float64)
        lev = np.empty(max(self.n, 1), dtype=np.int32)
        lo = np.empty(max(self.n, 1), dtype=np.int64)
        hi = np.empty(max(self.n, 1), dtype=np.int64)
        k = _L().orc_essential_nodes(self._h, _p(blo, C.c_double), _p(bhi, C.c_double), float(theta), int(mac),
                                     _p(rec, C.c_double), _p(lev, C.c_int32), _p(lo, C.c_int64), _p(hi, C.c_int64))
        if k < 0:
            raise ValueError("orc_essential_nodes: invalid argument")
        rec = rec[:k].copy()
        return (rec, lev[:k].copy(), lo[:k].copy(), hi[:k].copy()) if want_ranges else rec

    def field(self, theta, G=1.0, mac=MAC_BH86, group=32, mac_fp32=False, groups=None, out=None):
        """NEXT-4: the group walk returning (phi[n], acc[n, 3]) in ORIGINAL order; acc = -grad phi evaluated
        on the same interaction lists (monopole gradient of every accepted node and leaf cell).
        `groups` = (begin, end) restricts the walk; cells not walked stay NaN.
        `out`: reuse a (float64[n], float64[n, 3]) pair of buffers (marshalling only)."""
        ng = (self.n + group - 1) // group
        gb, ge = (0, ng) if groups is None else groups
        phi, acc = (np.full(self.n, np.nan), np.full((self.n, 3), np.nan)) if out is None else out
        rc = _L().orc_field(self._h, float(theta), float(G), int(mac), int(group), int(bool(mac_fp32)),
                            gb, ge, _p(phi, C.c_double), _p(acc, C.c_double), None)
        if rc != 0:
            raise ValueError("orc_field: invalid argument")
        return phi, acc
