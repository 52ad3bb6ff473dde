"""Counter-based seeded generators (splitmix64 -> Box-Muller), numpy only.

Draw number q of a stream is a pure function of (seed, q), so any sub-range of a field is
reproducible without generating the rest.  Cell (x,y,z), component c consumes draw
q = ((x*ny + y)*nz + z)*3 + c  (SURVEY.md 8(d) recipe: [x][y][z][c] order).
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return z ^ (z >> np.uint64(31))


def _uniform01(seed: int, counter: np.ndarray) -> np.ndarray:
    """Uniform in (0,1), 53 bits, from the counter."""
    with np.errstate(over="ignore"):
        key = _splitmix64(np.full(1, seed, dtype=np.uint64))[0]
        bits = _splitmix64(counter.astype(np.uint64) ^ key)
    return ((bits >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal_field(seed: int, count: int, start: int = 0, chunk: int = 1 << 24) -> np.ndarray:
    """count standard-normal draws q = start .. start+count-1 of stream `seed` (Box-Muller:
    draw q uses uniforms 2q and 2q+1)."""
    out = np.empty(count, dtype=np.float64)
    for lo in range(0, count, chunk):
        hi = min(count, lo + chunk)
        q = np.arange(start + lo, start + hi, dtype=np.uint64)
        u1 = _uniform01(seed, q * np.uint64(2))
        u2 = _uniform01(seed, q * np.uint64(2) + np.uint64(1))
        out[lo:hi] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


def random_unit_vectors(seed: int, n) -> np.ndarray:
    """i.i.d. standard-normal 3-vectors, normalised; shape [nx, ny, nz, 3] fp64."""
    nx, ny, nz = n
    v = normal_field(seed, nx * ny * nz * 3).reshape(nx, ny, nz, 3)
    v /= np.linalg.norm(v, axis=-1, keepdims=True)
    return v


def in_plane_state(seed: int, n, base=(1.0, 0.1, 0.0), noise=0.01) -> np.ndarray:
    """base/|base| plus `noise` * normal per component, renormalised (config 2)."""
    nx, ny, nz = n
    b = np.asarray(base, dtype=np.float64)
    b = b / np.linalg.norm(b)
    v = b + noise * normal_field(seed, nx * ny * nz * 3).reshape(nx, ny, nz, 3)
    v /= np.linalg.norm(v, axis=-1, keepdims=True)
    return v


def box_filter_renormalise(v: np.ndarray) -> np.ndarray:
    """One 3x3x3 box filter summing in-range neighbours only (no wrap), then renormalise
    (config 3, reading Q21: the neighbour count cancels in the normalisation)."""
    acc = v.copy()
    for axis in range(3):
        src = acc
        out = src.copy()
        sl_lo = [slice(None)] * 4
        sl_hi = [slice(None)] * 4
        sl_lo[axis] = slice(0, -1)
        sl_hi[axis] = slice(1, None)
        out[tuple(sl_hi)] += src[tuple(sl_lo)]
        out[tuple(sl_lo)] += src[tuple(sl_hi)]
        acc = out
    acc /= np.linalg.norm(acc, axis=-1, keepdims=True)
    return acc


def sample_cells(seed: int, n, count: int) -> np.ndarray:
    """`count` seeded flat cell indices plus the 8 corners, 6 face centres and body centre."""
    nx, ny, nz = n
    ncell = nx * ny * nz
    u = _uniform01(seed, np.arange(count, dtype=np.uint64))
    cells = list(np.minimum((u * ncell).astype(np.int64), ncell - 1))
    ex = [(0, nx - 1), (0, ny - 1), (0, nz - 1)]
    mid = (nx // 2, ny // 2, nz // 2)
    pts = [(a, b, c) for a in ex[0] for b in ex[1] for c in ex[2]]
    pts += [(a, mid[1], mid[2]) for a in ex[0]] + [(mid[0], b, mid[2]) for b in ex[1]]
    pts += [(mid[0], mid[1], c) for c in ex[2]] + [mid]
    cells += [(x * ny + y) * nz + z for x, y, z in pts]
    return np.unique(np.asarray(cells, dtype=np.int64))


def sparse_sources(seed: int, n, count: int):
    """`count` seeded source cells (always including cell 0 and the last cell) carrying
    random unit vectors; every other cell is exactly zero.  Returns (m, flat source ids)."""
    nx, ny, nz = n
    ncell = nx * ny * nz
    u = _uniform01(seed ^ 0x5A5A, np.arange(count, dtype=np.uint64))
    ids = np.unique(np.concatenate([np.minimum((u * ncell).astype(np.int64), ncell - 1),
                                    np.array([0, ncell - 1], dtype=np.int64)]))
    vec = normal_field(seed, len(ids) * 3).reshape(-1, 3)
    vec /= np.linalg.norm(vec, axis=-1, keepdims=True)
    m = np.zeros((nx, ny, nz, 3), dtype=np.float64)
    m.reshape(-1, 3)[ids] = vec
    return m, ids
