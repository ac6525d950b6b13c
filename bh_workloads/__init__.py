"""Seeded synthetic input generators shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no keys, no tree, no potential): it only
produces point masses -- fp64 cell centres x, y, z, masses m -- inside a bounding cube, with the
shapes, sizes and structure of the workloads named in BASELINE.json `configs` / SURVEY.md §8(d).
They stand in for the paper's FLASH/PARAMESH meshes (§4.1 MacLaurin spheroid,
PAPER.md:244-299 §4.2.1 centrally condensed AMR cores), which are not available.

Every generator returns a `Workload` (plain container).  Randomness is
`numpy.random.Generator(PCG64(seed))` or, for the AMR field, a counter-based integer hash so that a
cell's perturbation depends only on (seed, level, i, j, k).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "Workload", "uniform_sphere", "maclaurin_spheroid", "amr_collapsing_core", "turbulent_medium",
    "random_points", "clustered_points", "with_duplicates", "by_name", "CONFIG_NAMES",
]


@dataclass
class Workload:
    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    m: np.ndarray
    cube: np.ndarray = field(default_factory=lambda: np.array([0.0, 0.0, 0.0, 1.0]))
    theta: float = 0.5
    G: float = 1.0
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.x.shape[0])


def _grid_centres(ng: int):
    """Cell centres (i+1/2)/ng of an ng^3 grid in the unit cube, raster order (i slowest)."""
    c = (np.arange(ng, dtype=np.float64) + 0.5) / ng
    X, Y, Z = np.meshgrid(c, c, c, indexing="ij")
    return X.ravel(), Y.ravel(), Z.ravel()


def uniform_sphere(ng: int = 32, radius: float = 0.4, rho: float = 1.0) -> Workload:
    """configs[0]: rho=1 sphere of radius 0.4 about (1/2,1/2,1/2) sampled on an ng^3 grid.

    m = rho*dV for centres inside the sphere, 0 outside; zero-mass cells are kept as cells and
    as targets.
    """
    x, y, z = _grid_centres(ng)
    r2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
    m = np.where(r2 <= radius * radius, rho / ng ** 3, 0.0)
    return Workload(f"sphere{ng}", x, y, z, m, meta=dict(ng=ng, radius=radius, rho=rho, dx=1.0 / ng))


def maclaurin_spheroid(ng: int = 128, a1: float = 0.4, ecc: float = 0.9, rho: float = 1.0, sub: int = 4) -> Workload:
    """configs[1]: uniform oblate spheroid, a1=a2=0.4, a3=a1*sqrt(1-e^2), axis z, centred.

    Fill fraction = (# of the sub^3 sub-cell centres inside)/sub^3; m = rho*f*dV.
    Shape after PAPER.md:228 (§4.1: uniform density inside, eccentricity 0.9, unit box).
    """
    a3 = a1 * np.sqrt(1.0 - ecc * ecc)
    c = (np.arange(ng, dtype=np.float64) + 0.5) / ng
    off = ((np.arange(sub, dtype=np.float64) + 0.5) / sub - 0.5) / ng
    # separable: (x-.5)^2/a1^2 for all sub-samples along each axis
    sx = ((c[:, None] + off[None, :] - 0.5) / a1) ** 2          # (ng, sub)
    sz = ((c[:, None] + off[None, :] - 0.5) / a3) ** 2
    fill = np.zeros((ng, ng, ng), dtype=np.float64)
    for a in range(sub):
        for b in range(sub):
            sxy = sx[:, a][:, None] + sx[:, b][None, :]          # (ng, ng)
            for cc in range(sub):
                fill += (sxy[:, :, None] + sz[:, cc][None, None, :]) <= 1.0
    fill /= sub ** 3
    x, y, z = _grid_centres(ng)
    m = rho * fill.ravel() / ng ** 3
    return Workload(f"maclaurin{ng}", x, y, z, m,
                    meta=dict(ng=ng, a1=a1, a3=float(a3), ecc=ecc, rho=rho, dx=1.0 / ng, sub=sub))


# ---- counter-based hash -> standard normal (for the AMR workload) ---------------------------------
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix64(v: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        v = (v + np.uint64(0x9E3779B97F4A7C15)) & _M64
        v = ((v ^ (v >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        v = ((v ^ (v >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return v ^ (v >> np.uint64(31))


def _cell_normal(seed: int, level: int, i: np.ndarray, j: np.ndarray, k: np.ndarray) -> np.ndarray:
    """Standard normal deviate that depends only on (seed, level, i, j, k)."""
    with np.errstate(over="ignore"):
        h = _mix64(np.uint64(seed) * np.uint64(0x2545F4914F6CDD1D) + np.uint64(level))
        h = _mix64(h ^ i.astype(np.uint64))
        h = _mix64(h ^ (j.astype(np.uint64) << np.uint64(21)))
        h = _mix64(h ^ (k.astype(np.uint64) << np.uint64(42)))
        h2 = _mix64(h ^ np.uint64(0xD6E8FEB86659FD93))
    u1 = ((h >> np.uint64(11)).astype(np.float64) + 0.5) / 9007199254740992.0
    u2 = ((h2 >> np.uint64(11)).astype(np.float64) + 0.5) / 9007199254740992.0
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def amr_collapsing_core(nroot: int = 4, max_level: int = 6, seed: int = 1509, rho_c: float = 1.0e3,
                        r_c: float = 0.05, sigma: float = 0.1, nb: int = 8) -> Workload:
    """configs[2]: collapsing cloud core on a FLASH/PARAMESH-style block-structured AMR grid.

    Blocks of nb^3 cells; `nroot`^3 root blocks at level 1; a level-l block (l < max_level) is
    refined into 8 children if max(rho) over its cells > 4^l (background = 1).
    rho(r) = rho_c/(1+(r/r_c)^2) about the cube centre times exp(sigma*g - sigma^2/2), g ~ N(0,1)
    per cell from a counter hash.  Leaf cells: centre, m = rho*dx^3.  `nroot=4` is the reading that
    gives "about 4M cells".
    """
    o = np.arange(nb, dtype=np.int64)
    OI, OJ, OK = [a.ravel() for a in np.meshgrid(o, o, o, indexing="ij")]
    r = np.arange(nroot, dtype=np.int64)
    blocks = np.stack([a.ravel() for a in np.meshgrid(r, r, r, indexing="ij")], axis=1)
    xs, ys, zs, ms, dxs = [], [], [], [], []
    per_level = {}
    for level in range(1, max_level + 1):
        if blocks.shape[0] == 0:
            break
        ncell_dim = nroot * nb * (1 << (level - 1))
        dx = 1.0 / ncell_dim
        keep_x, keep_y, keep_z, keep_m = [], [], [], []
        refine = np.zeros(blocks.shape[0], dtype=bool)
        for s in range(0, blocks.shape[0], 4096):                 # bounded temporaries
            b = blocks[s:s + 4096]
            ci = (b[:, 0:1] * nb + OI[None, :])
            cj = (b[:, 1:2] * nb + OJ[None, :])
            ck = (b[:, 2:3] * nb + OK[None, :])
            cx = (ci + 0.5) * dx
            cy = (cj + 0.5) * dx
            cz = (ck + 0.5) * dx
            rr2 = (cx - 0.5) ** 2 + (cy - 0.5) ** 2 + (cz - 0.5) ** 2
            rho = rho_c / (1.0 + rr2 / (r_c * r_c)) + 0.0
            rho = np.maximum(rho, 1.0)                              # background density 1
            g = _cell_normal(seed, level, ci, cj, ck)
            rho = rho * np.exp(sigma * g - 0.5 * sigma * sigma)
            ref = (rho.max(axis=1) > 4.0 ** level) if level < max_level else np.zeros(b.shape[0], bool)
            refine[s:s + 4096] = ref
            leaf = ~ref
            keep_x.append(cx[leaf].ravel()); keep_y.append(cy[leaf].ravel()); keep_z.append(cz[leaf].ravel())
            keep_m.append((rho[leaf] * dx ** 3).ravel())
        nleaf = sum(a.size for a in keep_x)
        per_level[level] = nleaf
        if nleaf:
            xs += keep_x; ys += keep_y; zs += keep_z; ms += keep_m
            dxs.append(np.full(nleaf, dx))
        par = blocks[refine]
        ch = np.stack([a.ravel() for a in np.meshgrid([0, 1], [0, 1], [0, 1], indexing="ij")], axis=1)
        blocks = (par[:, None, :] * 2 + ch[None, :, :]).reshape(-1, 3)
    x = np.concatenate(xs); y = np.concatenate(ys); z = np.concatenate(zs); m = np.concatenate(ms)
    return Workload(f"amr_core_r{nroot}_l{max_level}", x, y, z, m,
                    meta=dict(nroot=nroot, max_level=max_level, seed=seed, cells_per_level=per_level,
                              dx=np.concatenate(dxs), finest_dx=1.0 / (nroot * nb * (1 << (max_level - 1)))))


def turbulent_medium(ng: int = 256, seed: int = 7370, sigma_ln: float = 1.0, slope: float = -4.0) -> Workload:
    """configs[3]: lognormal density from a seeded Gaussian random field with P(k) ~ k^slope.

    White noise -> FFT -> multiply by k^(slope/2) (k=0 zeroed) -> inverse FFT -> unit variance g;
    rho = exp(sigma*g - sigma^2/2); m = rho/ng^3.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    w = rng.standard_normal((ng, ng, ng))
    wk = np.fft.rfftn(w, axes=(0, 1, 2))
    del w
    kx = np.fft.fftfreq(ng) * ng
    kz = np.fft.rfftfreq(ng) * ng
    k2 = kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    amp = k2 ** (slope / 4.0)
    amp[0, 0, 0] = 0.0
    wk *= amp
    del amp, k2
    g = np.fft.irfftn(wk, s=(ng, ng, ng), axes=(0, 1, 2))
    del wk
    g -= g.mean()
    g /= g.std()
    rho = np.exp(sigma_ln * g - 0.5 * sigma_ln ** 2)
    x, y, z = _grid_centres(ng)
    m = rho.ravel() / ng ** 3
    return Workload(f"turb{ng}", x, y, z, m, meta=dict(ng=ng, seed=seed, sigma_ln=sigma_ln, dx=1.0 / ng))


# ---- small irregular inputs for the tests (chains, buckets, clamping) -----------------------------
def random_points(n: int, seed: int = 0, cube=(0.0, 0.0, 0.0, 1.0), mass="uniform") -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    x0, y0, z0, L = cube
    x = x0 + L * rng.random(n); y = y0 + L * rng.random(n); z = z0 + L * rng.random(n)
    m = rng.random(n) + 0.1 if mass == "uniform" else np.exp(rng.standard_normal(n))
    return Workload(f"rand{n}_s{seed}", x, y, z, m / m.sum(), cube=np.array(cube, dtype=np.float64))


def clustered_points(n: int, seed: int = 0, nclump: int = 6, scale: float = 0.01) -> Workload:
    """Strongly clustered points (deep, ragged trees with single-child chains)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    cen = 0.15 + 0.7 * rng.random((nclump, 3))
    which = rng.integers(0, nclump, n)
    s = scale * np.exp(rng.standard_normal(nclump))[which]
    p = cen[which] + s[:, None] * rng.standard_normal((n, 3))
    p = np.clip(p, 1e-9, 1.0 - 1e-9)
    m = np.exp(0.5 * rng.standard_normal(n))
    return Workload(f"clump{n}_s{seed}", p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy(), m / m.sum())


def with_duplicates(w: Workload, ndup: int, seed: int = 0, near: float = 0.0) -> Workload:
    """Append `ndup` copies of randomly chosen points (exact duplicates -> bucket leaves;
    `near` > 0 displaces the copy by that amount along x -> deep single-child chains)."""
    rng = np.random.Generator(np.random.PCG64(seed + 99))
    pick = rng.integers(0, w.n, ndup)
    x = np.concatenate([w.x, w.x[pick] + near]); y = np.concatenate([w.y, w.y[pick]])
    z = np.concatenate([w.z, w.z[pick]]); m = np.concatenate([w.m, 0.5 * w.m[pick]])
    return Workload(w.name + f"_dup{ndup}", x, y, z, m, cube=w.cube.copy(), theta=w.theta, G=w.G)


CONFIG_NAMES = ("sphere32", "maclaurin128", "amr_core", "turb256")


def by_name(name: str) -> Workload:
    """The BASELINE.json configs by short name (configs[4] is a theta sweep over 'amr_core')."""
    if name == "sphere32":
        return uniform_sphere(32)
    if name == "maclaurin128":
        return maclaurin_spheroid(128)
    if name == "amr_core":
        return amr_collapsing_core()
    if name == "turb256":
        return turbulent_medium(256)
    if name.startswith("turb"):
        return turbulent_medium(int(name[4:]))
    if name.startswith("sphere"):
        return uniform_sphere(int(name[6:]))
    if name.startswith("maclaurin"):
        return maclaurin_spheroid(int(name[9:]))
    if name.startswith("amr_small"):
        return amr_collapsing_core(nroot=2, max_level=4)
    raise ValueError(name)
