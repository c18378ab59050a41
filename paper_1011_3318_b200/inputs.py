"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no Dirac operator, no clover
term, no solver): it only produces the gauge links and source vectors described
in DESIGN.md ("Input recipe"), which stand in for the paper's "random gauge
configuration" and "Gaussian noise vector eta" (Sec. 5).

Everything is generated on the host in fp64 by a counter-based generator
(splitmix64 of (seed, stream, element index) -> Box-Muller), so values do not
depend on generation order or chunking and the same arrays feed both sides.

Canonical layouts:
  site index i = x + Lx*(y + Ly*(z + Lz*t)), mu = 0..3 = x,y,z,t
  gauge  [V][4][3][3] complex128, (U psi)_a = sum_b U[a][b] psi_b
  spinor [V][4][3]    complex128 (spin, colour)
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(z: np.ndarray) -> np.ndarray:
    """One splitmix64 output step applied elementwise to uint64 counters."""
    with np.errstate(over="ignore"):
        z = z + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def _key(seed: int, stream: int) -> np.uint64:
    k = _splitmix64(np.array([seed], dtype=np.uint64))[0]
    with np.errstate(over="ignore"):
        k = _splitmix64(np.array([k ^ np.uint64(stream * 0x632BE59BD9B4E019 & 0xFFFFFFFFFFFFFFFF)],
                                 dtype=np.uint64))[0]
    return k


def uniform01(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count uniforms in (0,1), element index start..start+count-1 of (seed, stream)."""
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        bits = _splitmix64(_splitmix64(idx ^ _key(seed, stream)))
    return ((bits >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count N(0,1) deviates; deviate k uses uniforms 2k and 2k+1 (Box-Muller, cosine branch)."""
    u = uniform01(seed, stream, 2 * start, 2 * count)
    return np.sqrt(-2.0 * np.log(u[0::2])) * np.cos(2.0 * np.pi * u[1::2])


def complex_normal(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count complex deviates re,im ~ N(0,1) i.i.d.; element k uses normals 2k, 2k+1."""
    g = normal(seed, stream, 2 * start, 2 * count)
    return g[0::2] + 1j * g[1::2]


def volume(dims) -> int:
    return int(dims[0]) * int(dims[1]) * int(dims[2]) * int(dims[3])


_GAUGE_STREAM = 1000
_CHUNK = 1 << 18  # links per chunk


def _chunks(total: int, fn):
    """fn(start, count) for every chunk of the element range; the chunks run on a thread pool (numpy releases the GIL in
    its inner loops).  Values are functions of the element index only, so neither chunking nor scheduling changes them."""
    starts = list(range(0, total, _CHUNK))
    if len(starts) <= 1:
        for s in starts:
            fn(s, min(_CHUNK, total - s))
        return
    with ThreadPoolExecutor(max_workers=min(len(starts), os.cpu_count() or 1)) as ex:
        list(ex.map(lambda s: fn(s, min(_CHUNK, total - s)), starts))


def gauge_exp(dims, eps: float, seed: int) -> np.ndarray:
    """U = exp(i*eps*H), H = (G+G^dag)/2 - tr/3, G 3x3 complex Gaussian (configs 0,1,2,4)."""
    nlink = 4 * volume(dims)
    out = np.empty((nlink, 3, 3), dtype=np.complex128)
    eye = np.eye(3)

    def fill(s, n):
        g = complex_normal(seed, _GAUGE_STREAM, 9 * s, 9 * n).reshape(n, 3, 3)
        h = 0.5 * (g + np.conj(np.swapaxes(g, 1, 2)))
        tr = np.einsum("nii->n", h).real / 3.0
        h = h - tr[:, None, None] * eye
        w, v = np.linalg.eigh(h)
        out[s:s + n] = np.einsum("nij,nj,nkj->nik", v, np.exp(1j * eps * w), np.conj(v))

    _chunks(nlink, fill)
    return out.reshape(volume(dims), 4, 3, 3)


def gauge_haar(dims, seed: int) -> np.ndarray:
    """'Fully random' SU(3): Gram-Schmidt rows 1-2 of a complex Gaussian 3x3, row 3 = conj(row1 x row2) (config 3)."""
    nlink = 4 * volume(dims)
    out = np.empty((nlink, 3, 3), dtype=np.complex128)

    def fill(s, n):
        g = complex_normal(seed, _GAUGE_STREAM, 9 * s, 9 * n).reshape(n, 3, 3)
        a = g[:, 0] / np.linalg.norm(g[:, 0], axis=1)[:, None]
        b = g[:, 1] - a * np.einsum("ni,ni->n", np.conj(a), g[:, 1])[:, None]
        b = b / np.linalg.norm(b, axis=1)[:, None]
        c = np.conj(np.cross(a, b))
        out[s:s + n, 0], out[s:s + n, 1], out[s:s + n, 2] = a, b, c

    _chunks(nlink, fill)
    return out.reshape(volume(dims), 4, 3, 3)


def gauge_unit(dims) -> np.ndarray:
    """Free field U = 1."""
    out = np.zeros((volume(dims), 4, 3, 3), dtype=np.complex128)
    out[:, :, [0, 1, 2], [0, 1, 2]] = 1.0
    return out


def spinor(dims, seed: int, stream: int = 0) -> np.ndarray:
    """Gaussian source: 12 complex N(0,1)+iN(0,1) per site, [V][4][3]."""
    v = volume(dims)
    out = np.empty(12 * v, dtype=np.complex128)

    def fill(s, n):
        out[s:s + n] = complex_normal(seed, stream, s, n)

    _chunks(12 * v, fill)
    return out.reshape(v, 4, 3)


def su3_field(dims, seed: int, stream: int = 777) -> np.ndarray:
    """Random SU(3) matrix per site, [V][3][3] (for gauge-covariance tests)."""
    v = volume(dims)
    g = complex_normal(seed, stream, 0, 9 * v).reshape(v, 3, 3)
    a = g[:, 0] / np.linalg.norm(g[:, 0], axis=1)[:, None]
    b = g[:, 1] - a * np.einsum("ni,ni->n", np.conj(a), g[:, 1])[:, None]
    b = b / np.linalg.norm(b, axis=1)[:, None]
    c = np.conj(np.cross(a, b))
    return np.stack([a, b, c], axis=1)


# BASELINE.json:configs, as parameters.  "overlap" is s (extension per side), d = 2s.
CONFIGS = {
    0: dict(dims=(4, 4, 4, 4), kappa=0.12, csw=1.0, gauge=("exp", 0.5), seed=1,
            ras=[dict(domain=(2, 2, 2, 2), overlap=0, block_iters=4)]),
    1: dict(dims=(8, 8, 8, 8), kappa=0.12, csw=1.0, gauge=("exp", 0.5), seed=2,
            ras=[dict(domain=(4, 4, 4, 4), overlap=0, block_iters=4),
                 dict(domain=(4, 4, 4, 4), overlap=1, block_iters=4)]),
    2: dict(dims=(16, 16, 16, 16), kappa=0.122, csw=1.2, gauge=("exp", 0.7), seed=3,
            ras=[dict(domain=d, overlap=s, block_iters=4)
                 for d in ((4, 4, 4, 4), (8, 4, 4, 4)) for s in (0, 1, 2)]),
    3: dict(dims=(32, 32, 32, 32), kappa=0.1225, csw=1.0, gauge=("haar",), seed=4,
            ras=[dict(domain=(8, 8, 8, 8), overlap=0, block_iters=5),
                 dict(domain=(8, 8, 4, 4), overlap=0, block_iters=5)]),
    4: dict(dims=(48, 48, 48, 96), kappa=0.12, csw=1.0, gauge=("exp", 0.5), seed=5,
            ras=[dict(domain=(8, 8, 8, 8), overlap=1, block_iters=4)]),
}


def make_gauge(cfg: dict, dims=None) -> np.ndarray:
    dims = dims or cfg["dims"]
    if cfg["gauge"][0] == "exp":
        return gauge_exp(dims, cfg["gauge"][1], cfg["seed"])
    return gauge_haar(dims, cfg["seed"])
