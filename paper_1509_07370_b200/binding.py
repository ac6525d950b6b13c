"""ctypes binding of libbh (include/bh.h).  Same names as the C ABI; marshalling only."""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

BH_MAC_BH86 = 0       # Eq. 3
BH_MAC_BARNES94 = 1   # Eq. 4
BH_OPT_MAC = 1
BH_OPT_GROUP = 2
BH_OPT_PASS_TIMING = 3
BH_OPT_PERIODIC = 4
BH_OPT_EWALD_N = 5
BH_OPT_EWALD_NREF = 6
BH_DIRECT_ALL_MAX = 1 << 18

EXPORTED_SYMBOLS = (
    "bh_create", "bh_destroy", "bh_strerror", "bh_last_cuda_error", "bh_set_option", "bh_build", "bh_potential",
    "bh_potential_direct", "bh_solve_host", "bh_tree_sizes", "bh_export_tree", "bh_last_group_counts",
    "bh_last_interactions", "bh_get_stats", "bh_update_masses", "bh_essential_nodes", "bh_set_num_targets", "bh_field",
    "bh_last_group_evaluated", "bh_last_walk_group", "bh_get_build_passes", "bh_host_breakdown", "bh_ewald_table",
    "bh_direct_noalloc", "bh_noalloc_last_error",
)


class Stats(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_nodes", C.c_int64), ("n_slots", C.c_int64), ("depth", C.c_int32),
                ("sort_passes", C.c_int32), ("n_clamped", C.c_int64), ("max_bucket", C.c_int64),
                ("n_accepted", C.c_int64), ("n_leaf", C.c_int64), ("n_opened", C.c_int64),
                ("n_exact_tests", C.c_int64), ("interactions", C.c_double),
                ("ms_keys", C.c_float), ("ms_sort", C.c_float), ("ms_count", C.c_float),
                ("ms_assign", C.c_float), ("ms_moments", C.c_float), ("ms_build_total", C.c_float),
                ("ms_walk", C.c_float), ("launches_build", C.c_int32), ("launches_walk", C.c_int32),
                ("walk_group", C.c_int32), ("interactions_counted", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Pass(C.Structure):
    _fields_ = [("name", C.c_char * 24), ("ms", C.c_float), ("alg_bytes", C.c_double)]


class BHError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libbh error {code}: {msg}")
        self.code = code


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Loads (building first if needed) libbh.so.  Raises if it cannot be built: no fallback."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, i64, i32 = C.c_void_p, C.c_void_p, C.c_int64, C.c_int
        L.bh_create.argtypes = [C.POINTER(vp), i32, vp]
        L.bh_destroy.argtypes = [vp]
        L.bh_strerror.argtypes = [i32]
        L.bh_strerror.restype = C.c_char_p
        L.bh_last_cuda_error.argtypes = [vp]
        L.bh_last_cuda_error.restype = C.c_char_p
        L.bh_set_option.argtypes = [vp, i32, i32]
        L.bh_build.argtypes = [vp, dp, dp, dp, dp, i64, C.POINTER(C.c_double)]
        L.bh_update_masses.argtypes = [vp, dp]
        L.bh_essential_nodes.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double, dp, i64,
                                         C.POINTER(i64)]
        L.bh_set_num_targets.argtypes = [vp, i64]
        L.bh_potential.argtypes = [vp, C.c_double, C.c_double, dp]
        L.bh_field.argtypes = [vp, C.c_double, C.c_double, dp, dp]
        L.bh_potential_direct.argtypes = [vp, C.c_double, dp, i64, dp]
        L.bh_solve_host.argtypes = [vp, dp, dp, dp, dp, i64, C.POINTER(C.c_double), C.c_double, C.c_double, dp]
        L.bh_tree_sizes.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
        L.bh_export_tree.argtypes = [vp] + [dp] * 12
        L.bh_last_group_counts.argtypes = [vp, dp]
        L.bh_last_interactions.argtypes = [vp, dp]
        L.bh_last_group_evaluated.argtypes = [vp, dp]
        L.bh_last_walk_group.argtypes = [vp]
        L.bh_get_build_passes.argtypes = [vp, C.POINTER(Pass), i32, C.POINTER(i32)]
        L.bh_host_breakdown.argtypes = [vp, C.POINTER(C.c_float)]
        L.bh_ewald_table.argtypes = [vp, dp, i64, C.POINTER(i32), C.POINTER(i32)]
        L.bh_get_stats.argtypes = [vp, C.POINTER(Stats)]
        L.bh_direct_noalloc.argtypes = [i32, vp, dp, dp, dp, dp, i64, C.c_double, dp]
        L.bh_noalloc_last_error.argtypes = []
        L.bh_noalloc_last_error.restype = C.c_char_p
        for name in EXPORTED_SYMBOLS:
            if name not in ("bh_strerror", "bh_last_cuda_error", "bh_noalloc_last_error"):
                getattr(L, name).restype = i32
        _lib = L
    return _lib


NOALLOC_MAX_N = 32768      # BH_NOALLOC_MAX_N of include/bh.h


def direct_noalloc(x, y, z, m, G: float = 1.0, out=None, stream=None):
    """bh_direct_noalloc: the fp64 direct sum of n <= NOALLOC_MAX_N cells with its scratch in a static device array
    of libbh -- no context, no allocation inside the library.  x, y, z, m: contiguous float64 CUDA tensors; `out`:
    float64 CUDA tensor [n] (allocated by torch here when None -- pass it to keep the whole call allocation-free);
    `stream`: a torch.cuda.Stream (default: the current stream of the tensors' device).  Asynchronous."""
    import torch
    n = x.numel()
    dev = x.device
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device=dev)
    ptrs = []
    for t in (x, y, z, m, out):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
                and t.numel() == n and t.device == dev):
            raise TypeError("expected contiguous float64 CUDA tensors of one length on one device")
        ptrs.append(C.c_void_p(t.data_ptr()))
    st = stream if stream is not None else torch.cuda.current_stream(dev)
    L = lib()
    rc = L.bh_direct_noalloc(dev.index if dev.index is not None else torch.cuda.current_device(),
                             C.c_void_p(st.cuda_stream), ptrs[0], ptrs[1], ptrs[2], ptrs[3], n, float(G), ptrs[4])
    if rc != 0:
        raise BHError(rc, (L.bh_noalloc_last_error() or L.bh_strerror(rc)).decode())
    return out


def _cube(c):
    return (C.c_double * 4)(*[float(v) for v in c])


class Context:
    """One tree on one CUDA stream (bh_create ... bh_destroy).  Tensors are torch CUDA tensors.

    Stream contract: every call enqueues its kernels on the stream given here (default: the torch stream
    current at construction).  Tensors handed to a call while ANOTHER torch stream is current are marked
    with `record_stream`, so the caching allocator does not reuse them while libbh kernels are in flight;
    ordering between the two streams stays the caller's business (wait_stream / events)."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        self._torch = torch
        self._L = lib()
        self._h = C.c_void_p()
        self.device = int(device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        self._check(self._L.bh_create(C.byref(self._h), self.device, C.c_void_p(stream.cuda_stream)))
        self.n = 0

    # -- helpers ------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != 0:
            msg = self._L.bh_strerror(rc).decode()
            if self._h:
                extra = self._L.bh_last_cuda_error(self._h).decode()
                if extra:
                    msg += " [" + extra + "]"
            raise BHError(rc, msg)

    def _dev(self, t, dtype):
        torch = self._torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
            raise TypeError(f"expected a contiguous CUDA tensor of dtype {dtype}")
        if torch.cuda.current_stream(self.device) != self.stream:
            t.record_stream(self.stream)        # the tensor is used on the context's stream, not the current one
        return C.c_void_p(t.data_ptr())

    def close(self):
        if getattr(self, "_h", None):
            self._L.bh_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, same names ----------------------------------------------------------------------
    def set_option(self, key: int, value: int):
        self._check(self._L.bh_set_option(self._h, int(key), int(value)))

    def set_mac(self, mac: int):
        self.set_option(BH_OPT_MAC, mac)

    def set_group(self, group: int):
        self.set_option(BH_OPT_GROUP, group)

    def set_periodic(self, on: bool, N: int = None, nref: int = None):
        """BH_OPT_PERIODIC (+ the size of the Ewald field array): the cube of the build is a periodic box."""
        if N is not None:
            self.set_option(BH_OPT_EWALD_N, int(N))
        if nref is not None:
            self.set_option(BH_OPT_EWALD_NREF, int(nref))
        self.set_option(BH_OPT_PERIODIC, 1 if on else 0)

    def ewald_table(self):
        """bh_ewald_table: CUDA float64 tensor [nref, N, N, N] (k, j, i order) of corr1 on the nested grids."""
        torch = self._torch
        N, nref = C.c_int(0), C.c_int(0)
        self._L.bh_ewald_table(self._h, None, 0, C.byref(N), C.byref(nref))
        out = torch.empty((nref.value, N.value, N.value, N.value), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._L.bh_ewald_table(self._h, self._dev(out, torch.float64), out.numel(), C.byref(N), C.byref(nref)))
        return out

    def build(self, x, y, z, m, cube):
        f64 = self._torch.float64
        n = x.numel()
        for t in (y, z, m):
            if t.numel() != n:
                raise ValueError("x, y, z, m must have the same length")
        self._check(self._L.bh_build(self._h, self._dev(x, f64), self._dev(y, f64), self._dev(z, f64),
                                     self._dev(m, f64), n, _cube(cube)))
        self.n = n

    def update_masses(self, m):
        """New masses for the cells of the last build (positions unchanged): leaf records and moments only."""
        if m.numel() != self.n:
            raise ValueError("m must have the length of the last build")
        self._check(self._L.bh_update_masses(self._h, self._dev(m, self._torch.float64)))

    def essential_nodes(self, box_lo, box_hi, theta: float, cap: int = 0):
        """bh_essential_nodes: the last build's tree pruned against the remote box; returns a CUDA tensor
        [count, 4] = (x, y, z, m) per essential entry.  `cap`: first guess of the count (0: a guess from this
        context's previous selections, so that a repeated exchange does not run the selection twice)."""
        torch = self._torch
        lo = (C.c_double * 3)(*[float(v) for v in box_lo])
        hi = (C.c_double * 3)(*[float(v) for v in box_hi])
        cnt = C.c_int64(0)
        TOO_LARGE = -5
        if cap <= 0:
            n = getattr(self, "n", 0)
            cap = getattr(self, "_ess_cap", 0) or min(n, max(4096, n // 8))
        while True:
            out = torch.empty((max(cap, 1), 4), dtype=torch.float64, device=f"cuda:{self.device}")
            rc = self._L.bh_essential_nodes(self._h, lo, hi, float(theta), self._dev(out, torch.float64) if cap else None,
                                            cap, C.byref(cnt))
            if rc == TOO_LARGE and cnt.value > cap:
                cap = int(cnt.value)
                continue
            self._check(rc)
            self._ess_cap = max(getattr(self, "_ess_cap", 0), int(cnt.value * 1.25) + 64)
            res = out[: cnt.value]
            return res.clone() if cap > cnt.value + (cnt.value >> 2) + 4096 else res     # do not pin a much larger buffer

    def essential_nodes_into(self, box_lo, box_hi, theta: float, out) -> int:
        """bh_essential_nodes with a caller-owned destination: `out` is a [cap, 4] float64 CUDA tensor -- of this
        process, or device memory of ANOTHER rank mapped into this one (CUDA IPC / symmetric memory over NVLink): the
        gather kernel's 32-byte record stores then ARE the transfer.  Returns the number of entries; raises
        BH_ERR_TOO_LARGE if they do not fit (the first cap entries are written)."""
        lo = (C.c_double * 3)(*[float(v) for v in box_lo])
        hi = (C.c_double * 3)(*[float(v) for v in box_hi])
        cnt = C.c_int64(0)
        self._check(self._L.bh_essential_nodes(self._h, lo, hi, float(theta), self._dev(out, self._torch.float64),
                                               int(out.shape[0]), C.byref(cnt)))
        return int(cnt.value)

    def set_num_targets(self, ntargets: int):
        """bh_set_num_targets: cells with original index < ntargets are targets, the rest sources only (-1: all)."""
        self._check(self._L.bh_set_num_targets(self._h, int(ntargets)))
        self._ntargets = int(ntargets)

    def potential(self, theta: float, G: float = 1.0, out=None):
        torch = self._torch
        if out is None:
            nt = getattr(self, "_ntargets", -1)
            out = torch.empty(self.n if nt < 0 else min(nt, self.n), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._L.bh_potential(self._h, float(theta), float(G), self._dev(out, torch.float64)))
        return out

    def field(self, theta: float, G: float = 1.0):
        """bh_field: (phi[n], acc[n, 3]) -- the potential and g = -grad phi from the same walk."""
        torch = self._torch
        nt = getattr(self, "_ntargets", -1)
        cnt = self.n if nt < 0 else min(nt, self.n)
        phi = torch.empty(cnt, dtype=torch.float64, device=f"cuda:{self.device}")
        acc = torch.empty((cnt, 3), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._L.bh_field(self._h, float(theta), float(G), self._dev(phi, torch.float64),
                                     self._dev(acc, torch.float64)))
        return phi, acc

    def potential_direct(self, G: float = 1.0, targets=None, out=None):
        torch = self._torch
        nt = self.n if targets is None else targets.numel()
        if out is None:
            out = torch.empty(nt, dtype=torch.float64, device=f"cuda:{self.device}")
        tp = C.c_void_p(0) if targets is None else self._dev(targets, torch.int64)
        self._check(self._L.bh_potential_direct(self._h, float(G), tp, nt, self._dev(out, torch.float64)))
        return out

    def solve_host(self, x, y, z, m, cube, theta: float, G: float = 1.0, out=None):
        """numpy / CPU-tensor float64 inputs; returns (or fills) a host float64 array."""
        import numpy as np
        arrs = []
        for a in (x, y, z, m):
            if hasattr(a, "numpy"):
                a = a.numpy()
            a = np.ascontiguousarray(a, dtype=np.float64)
            arrs.append(a)
        n = arrs[0].shape[0]
        if out is None:
            out = np.empty(n, dtype=np.float64)
        o = out.numpy() if hasattr(out, "numpy") else out
        self._check(self._L.bh_solve_host(self._h, *[C.c_void_p(a.ctypes.data) for a in arrs], n, _cube(cube),
                                          float(theta), float(G), C.c_void_p(o.ctypes.data)))
        self.n = n
        return out

    def host_breakdown(self):
        """bh_host_breakdown: dict of the last solve_host's device-side time split in ms."""
        ms = (C.c_float * 4)()
        self._check(self._L.bh_host_breakdown(self._h, ms))
        return {"h2d_ms": ms[0], "device_ms": ms[1], "d2h_ms": ms[2], "total_ms": ms[3],
                "overlap_ms": ms[0] + ms[1] + ms[2] - ms[3]}

    def build_passes(self):
        """bh_get_build_passes: [(name, ms, algorithmic bytes)] of the last build (BH_OPT_PASS_TIMING on)."""
        cap = 96
        arr = (Pass * cap)()
        cnt = C.c_int(0)
        self._check(self._L.bh_get_build_passes(self._h, arr, cap, C.byref(cnt)))
        return [(arr[k].name.decode(), float(arr[k].ms), float(arr[k].alg_bytes)) for k in range(cnt.value)]

    def tree_sizes(self):
        n, nn, ns = C.c_int64(), C.c_int64(), C.c_int64()
        self._check(self._L.bh_tree_sizes(self._h, C.byref(n), C.byref(nn), C.byref(ns)))
        return n.value, nn.value, ns.value

    def export_tree(self):
        """Returns dict of CUDA tensors: keys, perm and the canonical node list."""
        torch = self._torch
        n, nn, _ = self.tree_sizes()
        dev = f"cuda:{self.device}"
        out = dict(
            keys=torch.empty(n, dtype=torch.int64, device=dev), perm=torch.empty(n, dtype=torch.int32, device=dev),
            level=torch.empty(nn, dtype=torch.int32, device=dev), prefix=torch.empty(nn, dtype=torch.int64, device=dev),
            lo=torch.empty(nn, dtype=torch.int64, device=dev), hi=torch.empty(nn, dtype=torch.int64, device=dev),
            nchild=torch.empty(nn, dtype=torch.int32, device=dev), M=torch.empty(nn, dtype=torch.float64, device=dev),
            Rx=torch.empty(nn, dtype=torch.float64, device=dev), Ry=torch.empty(nn, dtype=torch.float64, device=dev),
            Rz=torch.empty(nn, dtype=torch.float64, device=dev), delta=torch.empty(nn, dtype=torch.float64, device=dev))
        order = ("keys", "perm", "level", "prefix", "lo", "hi", "nchild", "M", "Rx", "Ry", "Rz", "delta")
        self._check(self._L.bh_export_tree(self._h, *[self._dev(out[k], out[k].dtype) for k in order]))
        return out

    def last_walk_group(self) -> int:
        """BH_OPT_GROUP of the last walk (32 or 1)."""
        g = self._L.bh_last_walk_group(self._h)
        if g < 0:
            self._check(g)
        return g

    def last_group_counts(self):
        """[ngroups, 3] int64 = (accepted, leaf, opened) per group of the last walk; ngroups follows the
        group size of that walk (bh_last_walk_group), not an argument of this call."""
        torch = self._torch
        group = self.last_walk_group()
        ng = (self.n + group - 1) // group
        out = torch.empty((ng, 3), dtype=torch.int64, device=f"cuda:{self.device}")
        self._check(self._L.bh_last_group_counts(self._h, self._dev(out, torch.int64)))
        return out

    def last_group_evaluated(self):
        """[ngroups] int32: list entries the Phi kernel itself evaluated for each group of the last walk."""
        torch = self._torch
        group = self.last_walk_group()
        ng = (self.n + group - 1) // group
        out = torch.empty(ng, dtype=torch.int32, device=f"cuda:{self.device}")
        self._check(self._L.bh_last_group_evaluated(self._h, self._dev(out, torch.int32)))
        return out

    def last_interactions(self):
        torch = self._torch
        out = torch.empty(self.n, dtype=torch.int32, device=f"cuda:{self.device}")
        self._check(self._L.bh_last_interactions(self._h, self._dev(out, torch.int32)))
        return out

    def get_stats(self) -> Stats:
        s = Stats()
        self._check(self._L.bh_get_stats(self._h, C.byref(s)))
        return s
