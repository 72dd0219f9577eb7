"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side callers.

This module holds NO arithmetic of the method (no stencil, no CPML recursion, no
coefficient tables): only the workloads of BASELINE.json's five configs — grid
sizes, source positions, source wavelets, the heterogeneous medium — generated
once on the host and handed as the same fp32 arrays to both sides (DESIGN.md
"Input recipe").  The paper uses no dataset (homogeneous cubes with CPML,
PAPER.md P:290-303); these configs stand in for its workloads at B200 scale.
"""
import functools
import math

import numpy as np

F0 = 0.04                     # Ricker peak frequency of every BASELINE config
COURANT = 0.4                 # c_max dt / dx (BASELINE config 1; reading R15)
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(x):
    """Counter-based generator: splitmix64 finaliser on a uint64 array (wraps mod 2^64)."""
    x = np.asarray(x, np.uint64)
    with np.errstate(over="ignore"):
        x = x + np.uint64(0x9E3779B97F4A7C15)
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return x ^ (x >> np.uint64(31))


def hash_unit(seed, idx):
    """float32 in [-1, 1): top 24 bits of splitmix64(seed + idx).  The oracle and the CUDA
    library each carry their own copy of this generator for device-/window-side fills."""
    with np.errstate(over="ignore"):
        h = splitmix64(np.uint64(seed) + np.asarray(idx, np.uint64))
    return ((h >> np.uint64(40)).astype(np.float32) * np.float32(1.0 / 8388608.0) - np.float32(1.0)).astype(np.float32)


def hash_field(seed, which, gdim, off=(0, 0, 0), shape=None, scale=1.0):
    """Window [off, off+shape) of the counter-based field `which` of a gdim=(NX,NY,NZ) grid; (Nz,Ny,Nx) fp32."""
    nx, ny, nz = shape if shape is not None else gdim
    i = np.arange(nx, dtype=np.uint64) + np.uint64(off[0])
    j = np.arange(ny, dtype=np.uint64) + np.uint64(off[1])
    k = np.arange(nz, dtype=np.uint64) + np.uint64(off[2])
    with np.errstate(over="ignore"):
        g = i[None, None, :] + np.uint64(gdim[0]) * (j[None, :, None] + np.uint64(gdim[1]) * k[:, None, None])
        s = np.uint64(seed) + (np.uint64(which) << np.uint64(56))
    return (np.float32(scale) * hash_unit(s, g)).astype(np.float32)


def ricker(nsteps, dt, f0=F0, t0=None):
    """Source table w[n] = fp32(dt * s(n dt - t0)), s(t) = (1 - 2a^2) exp(-a^2), a = pi f0 t
    (Ricker form of PAPER.md P:193; t0 = 1/f0 and unit amplitude are reading R14)."""
    t0 = 1.0 / f0 if t0 is None else t0
    t = np.arange(nsteps, dtype=np.float64) * dt - t0
    a2 = (math.pi * f0 * t) ** 2
    return (dt * (1.0 - 2.0 * a2) * np.exp(-a2)).astype(np.float32)


def normals(seed, count, start=0):
    """Standard normals from the counter-based generator by Box-Muller (two counters per sample)."""
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        u1 = (splitmix64(np.uint64(seed) + np.uint64(2) * idx) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
        u2 = (splitmix64(np.uint64(seed) + np.uint64(2) * idx + np.uint64(1)) >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)


@functools.lru_cache(maxsize=2)
def smooth_medium(shape_xyz, seed=20260691, sigma=8.0, amp=0.3, lo=0.7, hi=1.3):
    """Heterogeneous wave speed of BASELINE config 3 (reading R22): seeded N(0,1) field, separable
    Gaussian filter (sigma cells, truncated at 4 sigma, periodic wrap), re-normalised to zero mean /
    unit std, c = clip(1 + amp g, lo, hi).  Returns fp32 (Nz,Ny,Nx), read-only (cached: half a minute at 552^3)."""
    from scipy.ndimage import gaussian_filter1d

    nx, ny, nz = shape_xyz
    g = np.empty((nz, ny, nx), np.float32)
    plane = nx * ny
    for k in range(nz):
        g[k] = normals(seed, plane, start=k * plane).reshape(ny, nx).astype(np.float32)
    for ax in range(3):
        g = gaussian_filter1d(g, sigma, axis=ax, mode="wrap", truncate=4.0, output=np.float32)
    m = float(g.mean(dtype=np.float64))
    s = float(g.std(dtype=np.float64))
    g -= np.float32(m)
    g *= np.float32(1.0 / s)
    c = np.float32(1.0) + np.float32(amp) * g
    np.clip(c, lo, hi, out=c)
    c.setflags(write=False)
    return c


def seeded_sources(n, total_xyz, margin=32, seed=20260692):
    """n source positions drawn uniformly from the total grid shrunk by `margin` cells per side."""
    out = np.zeros((n, 3), np.int32)
    for s in range(n):
        for a in range(3):
            span = total_xyz[a] - 2 * margin
            u = int(splitmix64(np.uint64(seed + 3 * s + a))) % span
            out[s, a] = margin + u
    return out


class Workload:
    """Plain description of one run: everything both sides need, nothing computed by the method."""

    def __init__(self, name, interior, L, steps, c=None, sources=None, decomp=(1, 1, 1), ghost=0, substeps=0):
        self.name = name
        self.n_interior = tuple(int(v) for v in interior)
        self.cpml = (int(L),) * 6 if np.isscalar(L) else tuple(int(v) for v in L)
        self.total = tuple(self.n_interior[a] + self.cpml[2 * a] + self.cpml[2 * a + 1] for a in range(3))
        self.steps = int(steps)
        self.c = c                                   # None = homogeneous c = 1
        self.c_max = 1.0 if c is None else float(np.max(c))
        self.dx = 1.0
        self.dt = COURANT * self.dx / self.c_max
        self.cpml_order = 2
        self.cpml_R0 = 1e-5
        self.cpml_kappa_max = 1.0
        self.cpml_alpha_max = math.pi * F0
        self.cpml_c_ref = self.c_max
        if sources is None:
            sources = np.array([[t // 2 for t in self.total]], np.int32)
        self.sources = np.ascontiguousarray(sources, np.int32).reshape(-1, 3)
        self.wavelets = np.tile(ricker(self.steps, self.dt), (self.sources.shape[0], 1))
        self.decomp, self.ghost, self.substeps = tuple(decomp), int(ghost), int(substeps)

    @property
    def points(self):
        return self.total[0] * self.total[1] * self.total[2]

    def cpml_kwargs(self):
        return dict(dx=self.dx, dt=self.dt, cpml_order=self.cpml_order, cpml_R0=self.cpml_R0,
                    cpml_kappa_max=self.cpml_kappa_max, cpml_alpha_max=self.cpml_alpha_max,
                    cpml_c_ref=self.cpml_c_ref)


def config(idx, scale=None, steps=None, **kw):
    """BASELINE.json configs 1..5.  `scale` = interior size override for the
    reduced parity cases (same structure, smaller cube)."""
    if idx == 1:
        n, L, st = scale or 64, 8, 100
        return Workload("config1", (n,) * 3, L, steps or st, **kw)
    if idx == 2:
        n, L, st = scale or 256, 16, 500
        return Workload("config2", (n,) * 3, L, steps or st, **kw)
    if idx == 3:
        n, L, st = scale or 512, 20, 1000
        tot = (n + 2 * L,) * 3
        c = smooth_medium(tot)
        src = seeded_sources(3, tot, margin=min(32, tot[0] // 4))
        return Workload("config3", (n,) * 3, L, steps or st, c=c, sources=src, **kw)
    if idx == 4:
        n, L, st = scale or 1536, 32, 200
        return Workload("config4", (n,) * 3, L, steps or st, **kw)
    if idx == 5:
        n, L, st = scale or 512, 20, 400
        kw.setdefault("decomp", (1, 2, 2))
        kw.setdefault("ghost", 8)
        kw.setdefault("substeps", 2)
        return Workload("config5", (n,) * 3, L, steps or st, **kw)
    raise ValueError("config index must be 1..5")
