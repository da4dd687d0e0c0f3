"""Seeded synthetic particle sets shaped like the paper's workloads.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2307_06345_b200.binding``).  It holds none of the method's
arithmetic (no keys, no sort, no tree logic): it only draws float64 coordinates
from ``numpy.random.Generator(PCG64(seed))`` and hands the *same* host buffers to
both sides.

The paper's own workloads are synthetic too: a 3D Gaussian density profile for
Table 1 and a 1/r sphere for Fig. 5.  The five
configurations below are the ones BASELINE.json names; they stand in for the
paper's workloads ("Input recipe").

All generators return three C-contiguous float64 arrays ``(x, y, z)`` of length
``n`` (structure-of-arrays, the layout the library consumes).
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field

import numpy as np

BASE_SEED = 230706345  # arXiv id 2307.06345

_CHUNK = 1 << 24  # generate in chunks to bound temporaries at N = 2^28


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def uniform(n: int, lo: float, hi: float, seed: int):
    """i.i.d. uniform in [lo, hi)^3 (configs 1 and 3)."""
    rng = _rng(seed)
    out = []
    for _ in range(3):
        c = np.empty(n, dtype=np.float64)
        for s in range(0, n, _CHUNK):
            e = min(n, s + _CHUNK)
            u = rng.random(e - s)
            c[s:e] = lo + (hi - lo) * u
        # guard the half-open interval against rounding of lo + (hi-lo)*u
        np.minimum(c, np.nextafter(hi, lo), out=c)
        out.append(c)
    return tuple(out)


def plummer(n: int, seed: int, a: float = 1.0, rmax: float = 100.0):
    """Plummer sphere, scale radius ``a``, truncated at ``rmax`` (configs 2 and 5).

    Radius by inverting the cumulative mass, r = a (u^(-2/3) - 1)^(-1/2); draws with
    r > rmax are rejected; direction isotropic (cos(theta) uniform in [-1, 1], phi
    uniform in [0, 2 pi)).
    """
    rng = _rng(seed)
    x = np.empty(n, dtype=np.float64)
    y = np.empty(n, dtype=np.float64)
    z = np.empty(n, dtype=np.float64)
    filled = 0
    while filled < n:
        m = min(_CHUNK, n - filled)
        m_draw = m + m // 512 + 64  # rejection rate is ~1.5e-4
        u = rng.random(m_draw)
        ct = rng.uniform(-1.0, 1.0, m_draw)
        phi = rng.uniform(0.0, 2.0 * np.pi, m_draw)
        with np.errstate(divide="ignore", invalid="ignore"):
            r = a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
        keep = np.flatnonzero(r <= rmax)[:m]
        k = keep.size
        r = r[keep]
        ct = ct[keep]
        phi = phi[keep]
        st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
        x[filled:filled + k] = r * st * np.cos(phi)
        y[filled:filled + k] = r * st * np.sin(phi)
        z[filled:filled + k] = r * ct
        filled += k
    return x, y, z


def blobs(n: int, seed: int, nblobs: int = 1000, blob_fraction: float = 0.9):
    """Mixture of isotropic Gaussian blobs plus a uniform background (config 4).

    Each particle is, independently, a blob particle with probability
    ``blob_fraction`` (blob chosen uniformly; centres uniform in [0,1)^3, sigma
    log-uniform in [1e-4, 1e-2]) or a uniform background particle; everything is
    clipped to [0, nextafter(1, 0)].  Particles are therefore in random memory
    order, as they would be before the first sort of a simulation.
    """
    rng = _rng(seed)
    centres = rng.random((nblobs, 3))
    sigma = 10.0 ** rng.uniform(-4.0, -2.0, nblobs)
    top = np.nextafter(1.0, 0.0)
    coords = [np.empty(n, dtype=np.float64) for _ in range(3)]
    for s in range(0, n, _CHUNK):
        e = min(n, s + _CHUNK)
        m = e - s
        is_blob = rng.random(m) < blob_fraction
        b = rng.integers(0, nblobs, m)
        for d in range(3):
            g = rng.standard_normal(m)
            u = rng.random(m)
            c = np.where(is_blob, centres[b, d] + sigma[b] * g, u)
            np.clip(c, 0.0, top, out=c)
            coords[d][s:e] = c
    return tuple(coords)


def gaussian(n: int, seed: int, sigma: float = 1.0):
    """Single isotropic 3D Gaussian density profile (the shape of the paper's
    Table 1 workload); used for the statistical tree-size pin."""
    rng = _rng(seed)
    out = []
    for _ in range(3):
        c = np.empty(n, dtype=np.float64)
        for s in range(0, n, _CHUNK):
            e = min(n, s + _CHUNK)
            c[s:e] = sigma * rng.standard_normal(e - s)
        out.append(c)
    return tuple(out)


def displace(x, y, z, sigma: float, seed: int):
    """Return copies of (x, y, z) with an i.i.d. N(0, sigma^2) step added to every
    coordinate (the incremental-rebuild steps of config 5)."""
    rng = _rng(seed)
    out = []
    for c in (x, y, z):
        d = np.array(c, dtype=np.float64, copy=True)
        n = d.shape[0]
        for s in range(0, n, _CHUNK):
            e = min(n, s + _CHUNK)
            d[s:e] += sigma * rng.standard_normal(e - s)
        out.append(d)
    return tuple(out)


def checksum(*arrays) -> str:
    """64-bit hex digest of the raw buffers (logged beside every measurement)."""
    h = hashlib.blake2b(digest_size=8)
    for a in arrays:
        h.update(np.ascontiguousarray(a).view(np.uint8))
    return h.hexdigest()


@dataclass
class Workload:
    name: str
    n: int
    bucket_sizes: tuple
    seed: int
    kind: str
    params: dict = field(default_factory=dict)
    incremental_steps: int = 0
    step_sigma: float = 0.0

    def generate(self, n: int | None = None):
        """Draw the coordinates; ``n`` overrides the size (same recipe, smaller)."""
        n = self.n if n is None else n
        if self.kind == "uniform":
            return uniform(n, self.params["lo"], self.params["hi"], self.seed)
        if self.kind == "plummer":
            return plummer(n, self.seed, a=1.0, rmax=100.0)
        if self.kind == "blobs":
            return blobs(n, self.seed)
        if self.kind == "gaussian":
            return gaussian(n, self.seed)
        raise ValueError(self.kind)

    def step(self, x, y, z, k: int):
        """Coordinates after incremental step ``k`` (1-based) applied to (x, y, z)."""
        return displace(x, y, z, self.step_sigma, self.seed + 1000 * k)


# BASELINE.json "configs", in order.  CONFIGS[3] (N = 2^26, blobs) is the headline.
CONFIGS = (
    Workload("c1_uniform_64k", 1 << 16, (64,), BASE_SEED + 1, "uniform", {"lo": 0.0, "hi": 1.0}),
    Workload("c2_plummer_1m", 1 << 20, (64,), BASE_SEED + 2, "plummer"),
    Workload("c3_uniform_16m", 1 << 24, (16, 64), BASE_SEED + 3, "uniform", {"lo": -1.0, "hi": 1.0}),
    Workload("c4_blobs_64m", 1 << 26, (64,), BASE_SEED + 4, "blobs"),
    Workload("c5_plummer_256m", 1 << 28, (64,), BASE_SEED + 5, "plummer",
             incremental_steps=10, step_sigma=1e-3),
)

HEADLINE = CONFIGS[3]
