"""Seeded synthetic input generators (numpy, host side).

This module serves BOTH the CPU oracle and the CUDA path: it only produces the
input buffers of the five workloads (BASELINE.json:configs) and
holds none of the method's arithmetic (no map/reduce/filter/contract code).

Generator: a counter-based 64-bit mixer.  ``bits(seed, stream, i)`` is the
SplitMix64 output function applied to ``base(seed, stream) + (i+1)*GAMMA``
(mod 2^64), so every element depends only on (seed, stream, index) and the
buffers can be produced in chunks, in any order.

The paper's benchmark inputs were generated and are not described beyond
their sizes and element types ("omitting the time it takes to
generate the input"; DOUBLE vectors PAPER.md:289, REAL_32 vectors PAPER.md:246,
DOUBLE matrices PAPER.md:325, sizes up to 10^8 PAPER.md:430); these generators
stand in for them.
"""
from __future__ import annotations

import concurrent.futures
import os

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_MASK = (1 << 64) - 1
_CHUNK = 1 << 22


def _mix_int(z: int) -> int:
    z &= _MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)


def base(seed: int, stream: int) -> int:
    """Stream origin: two rounds of the mixer over (seed, stream)."""
    return _mix_int(_mix_int(seed * 0x9E3779B97F4A7C15 + 0x632BE59BD9B4E019) ^ (stream * 0xD1342543DE82EF95 + 1))


def bits_scalar(seed: int, stream: int, i: int) -> int:
    """bits(seed, stream, i) for one index (python ints; reference for the vector form)."""
    return _mix_int(base(seed, stream) + (i + 1) * 0x9E3779B97F4A7C15)


def bits(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """uint64[count]: bits(seed, stream, start .. start+count-1)."""
    b = np.uint64(base(seed, stream))
    with np.errstate(over="ignore"):
        z = (np.arange(start + 1, start + count + 1, dtype=np.uint64) * _GAMMA) + b
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def u01(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """float64 uniform on [0,1): (bits >> 11) * 2^-53."""
    return (bits(seed, stream, start, count) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _chunks(n: int):
    for s in range(0, n, _CHUNK):
        yield s, min(_CHUNK, n - s)


def _fill(out: np.ndarray, fn) -> np.ndarray:
    """out[s:s+c] = fn(s, c) for every chunk; chunks are independent (counter-based), so threads may fill them."""
    n = out.size
    chunks = list(_chunks(n))
    workers = min(len(chunks), os.cpu_count() or 1, 16)

    def job(sc):
        out[sc[0]:sc[0] + sc[1]] = fn(*sc)

    if workers <= 1:
        for sc in chunks:
            job(sc)
    else:
        with concurrent.futures.ThreadPoolExecutor(max_workers=workers) as ex:
            list(ex.map(job, chunks))
    return out


def uniform_pm1_f64(seed: int, stream: int, n: int) -> np.ndarray:
    """float64[n], 2*u01 - 1 in [-1, 1)  (configs 0 and 4)."""
    return _fill(np.empty(n, dtype=np.float64), lambda s, c: 2.0 * u01(seed, stream, s, c) - 1.0)


def normal_f32(seed: int, stream: int, n: int, start: int = 0) -> np.ndarray:
    """float32[n] ~ N(0,1): Box-Muller in float64 on counters (2i, 2i+1), one output per pair (config 1).  start: elements
    start .. start+n-1 of the same infinite sequence (a rank generates only its shard of a sharded collection)."""
    def chunk(s, c):
        u = u01(seed, stream, 2 * (start + s), 2 * c)
        u1 = 1.0 - u[0::2]          # (0, 1]
        u2 = u[1::2]
        return (np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)).astype(np.float32)

    return _fill(np.empty(n, dtype=np.float32), chunk)


def uniform_i31(seed: int, stream: int, n: int) -> np.ndarray:
    """int32[n] uniform on [0, 2^31): bits >> 33 (config 2)."""
    return _fill(np.empty(n, dtype=np.int32), lambda s, c: (bits(seed, stream, s, c) >> np.uint64(33)).astype(np.int32))


def sorted_cumsum_f32(seed: int, stream: int, n: int) -> np.ndarray:
    """float32[n], ascending: s_0 = u_0, s_i = s_{i-1} + u_i sequentially in float64, x_i = (float) s_i (config 3)."""
    out = np.empty(n, dtype=np.float32)
    carry = 0.0
    for s, c in _chunks(n):
        u = u01(seed, stream, s, c)
        u[0] += carry               # same sequential order as one long running sum
        cs = np.cumsum(u)           # numpy's cumsum is a sequential left-to-right accumulation
        carry = float(cs[-1])
        out[s:s + c] = cs.astype(np.float32)
    return out


def violation_index(seed: int, n: int) -> int:
    """Seeded index j in [1, n-2] of the injected sortedness violation (config 3)."""
    return 1 + bits_scalar(seed, 99, 0) % (n - 2)


def inject_unsorted(x: np.ndarray, j: int) -> None:
    """x[j] = 0.5f * x[j-1]: breaks only the pair (j-1, j) and keeps x >= 0 (config 3)."""
    x[j] = np.float32(0.5) * x[j - 1]


def boosted_matrix_f64(seed: int, stream: int, n: int, boost: float | None = None) -> np.ndarray:
    """float64[n, n] row-major, 2*u01 - 1 with the diagonal boosted by +n (config 4)."""
    m = uniform_pm1_f64(seed, stream, n * n).reshape(n, n)
    idx = np.arange(n)
    m[idx, idx] += float(n if boost is None else boost)
    return m


def checksum(a: np.ndarray) -> int:
    """64-bit xor/rotate checksum of a buffer's bytes (logged so both sides can be seen to use the same bytes)."""
    raw = np.ascontiguousarray(a).reshape(-1).view(np.uint8)
    pad = (-raw.size) % 8
    if pad:
        raw = np.concatenate([raw, np.zeros(pad, dtype=np.uint8)])
    w = raw.view(np.uint64)
    acc = 0
    for s, c in _chunks(w.size):
        blk = w[s:s + c]
        with np.errstate(over="ignore"):
            k = (np.arange(s + 1, s + c + 1, dtype=np.uint64) * _GAMMA)
            acc ^= int(np.bitwise_xor.reduce(blk * _M1 + k))
    return acc & _MASK
