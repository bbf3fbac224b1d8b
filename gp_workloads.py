"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module serves BOTH the oracle (`oracle/`) and the CUDA path
(`paper_2606_11402_b200/`).  It holds none of the method's arithmetic: no
covariance function, no ordering, no neighbour search, no conditioning.  It only
produces point clouds, white noise and cotangents from a counter-based generator,
so both sides see bit-identical arrays (recipe: DESIGN.md §4).

Generator: z = mix(seed*0x9E3779B97F4A7C15 + (stream << 40) + index) with `mix`
the splitmix64 finaliser.  Uniforms are (z >> 40) * 2^-24 (exact in fp32) for
fp32 data and (z >> 11) * 2^-53 for fp64 data.  Normals are Box-Muller in double
on uniforms offset by half a step (so log(0) never occurs), rounded once to the
working dtype.

The paper measures on synthetic points only ("drawn from a unit Gaussian in 3d",
PAPER.md:47); BASELINE.json's configs replace that blob with harder
shapes.  No public dataset is involved.
"""
from __future__ import annotations

import dataclasses
import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser (two xor-shift-multiply rounds and a final xor-shift)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def raw_u64(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """`count` 64-bit words for counters start..start+count-1 of (seed, stream)."""
    with np.errstate(over="ignore"):
        base = np.uint64(seed) * _GOLDEN + (np.uint64(stream) << np.uint64(40))
        idx = np.arange(start, start + count, dtype=np.uint64)
        return _mix(base + idx)


def uniform(seed: int, stream: int, start: int, count: int, dtype) -> np.ndarray:
    """U[0,1) on the dtype's own grid: 24 bits for fp32, 53 bits for fp64 (returned as float64)."""
    z = raw_u64(seed, stream, start, count)
    if np.dtype(dtype) == np.float32:
        return (z >> np.uint64(40)).astype(np.float64) * 2.0 ** -24
    return (z >> np.uint64(11)).astype(np.float64) * 2.0 ** -53


def normal(seed: int, stream: int, start: int, count: int, dtype) -> np.ndarray:
    """N(0,1) by Box-Muller in double (streams `stream` and `stream+1`), returned as float64."""
    half = 2.0 ** -25 if np.dtype(dtype) == np.float32 else 2.0 ** -54
    u1 = uniform(seed, stream, start, count, dtype) + half
    u2 = uniform(seed, stream + 1, start, count, dtype)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


@dataclasses.dataclass(frozen=True)
class Config:
    """One BASELINE.json configuration with the readings of SURVEY.md §8(c)/(d) filled in."""
    cid: int
    name: str
    n: int
    d: int
    k: int
    n0: int
    kind: str            # 'se' | 'matern32' | 'exp'
    sigma: float
    ell: float
    jitter: float        # RELATIVE nugget: K_jj = sigma^2 (1 + jitter)   (reading S-7)
    dtypes: tuple        # working dtypes exercised
    ops: tuple

    def with_n(self, n: int) -> "Config":
        return dataclasses.replace(self, n=int(n))


CONFIGS = {
    1: Config(1, "uniform3d_k8_se_fp64", 4096, 3, 8, 64, "se", 1.0, 0.1, 1e-6,
              ("f64",), ("forward", "inverse", "logdet", "vjp")),
    2: Config(2, "uniform3d_k16_matern32", 1 << 20, 3, 16, 1024, "matern32", 1.0, 0.05, 1e-4,
              ("f32", "f64"), ("forward", "inverse", "logdet")),
    3: Config(3, "clustered3d_k16_matern32", 1 << 24, 3, 16, 1024, "matern32", 1.0, 0.02, 1e-3,
              ("f32",), ("forward", "inverse", "logdet", "vjp")),
    4: Config(4, "radial2d_k32_exp", 1 << 24, 2, 32, 1024, "exp", 1.0, 0.01, 1e-4,
              ("f32",), ("forward", "inverse", "logdet")),
    5: Config(5, "shells3d_k16_matern32", 1 << 28, 3, 16, 1024, "matern32", 1.0, 0.005, 1e-3,
              ("f32",), ("forward", "inverse", "logdet", "vjp")),
}

KIND_ID = {"se": 0, "matern32": 1, "exp": 2}
NP_DTYPE = {"f32": np.float32, "f64": np.float64}

# stream numbers (each coordinate / decision draws from its own stream)
_S_X = 0          # 0..2   uniform coordinates
_S_SEL = 4        # background-vs-cluster selector
_S_CL = 5         # cluster id
_S_G = 8          # 8..13  three normals (2 streams each)
_S_CEN = 16       # 16..18 cluster centres
_S_SCALE = 20     # cluster scale / shell radius
_S_SHELL = 24     # 24..25 log-normal radial factor
_S_NOISE = 32     # 32..33 xi / v_bar normals


def _chunked(n, chunk=1 << 22):
    for s in range(0, n, chunk):
        yield s, min(chunk, n - s)


def _for_chunks(n, fill, chunk=1 << 21):
    """Run fill(start, count) over all chunks; large n uses a thread pool (every element depends on its own
    counter only, so the result does not depend on the chunking or on the thread count)."""
    chunks = list(_chunked(n, chunk))
    if len(chunks) < 4:
        for s, c in chunks:
            fill(s, c)
        return
    import os
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(chunks), os.cpu_count() or 1, 32)) as ex:
        list(ex.map(lambda sc: fill(*sc), chunks))


def make_points(cfg: Config, dtype: str, n: int | None = None) -> np.ndarray:
    """Points [n, d] in USER order, values on the grid of `dtype`, returned in that dtype.

    Seeds: points 1000+c.  Prefixes are nested: make_points(cfg, n=a)
    equals make_points(cfg, n=b)[:a] because every point depends on its own counter only.
    """
    n = cfg.n if n is None else int(n)
    dt = NP_DTYPE[dtype]
    seed = 1000 + cfg.cid
    out = np.empty((n, cfg.d), dtype=dt)
    if cfg.cid in (1, 2):                                   # i.i.d. U[0,1]^3
        def fill(s, c):
            for j in range(cfg.d):
                out[s:s + c, j] = uniform(seed, _S_X + j, s, c, dt)
    elif cfg.cid == 3:    # 90 % mixture of 4096 isotropic Gaussians + 10 % uniform background
        ncl = 4096
        cen = np.stack([uniform(seed, _S_CEN + j, 0, ncl, dt) for j in range(3)], axis=1)
        scale = 10.0 ** (-4.0 + 3.0 * uniform(seed, _S_SCALE, 0, ncl, dt))

        def fill(s, c):
            bg = uniform(seed, _S_SEL, s, c, dt) < 0.1
            cl = np.minimum((uniform(seed, _S_CL, s, c, dt) * ncl).astype(np.int64), ncl - 1)
            for j in range(3):
                u = uniform(seed, _S_X + j, s, c, dt)
                g = normal(seed, _S_G + 2 * j, s, c, dt)
                out[s:s + c, j] = np.where(bg, u, cen[cl, j] + scale[cl] * g)
    elif cfg.cid == 4:    # radial power law in 2-d: r = U^3, angle uniform
        def fill(s, c):
            r = uniform(seed, _S_X, s, c, dt) ** 3
            phi = 2.0 * np.pi * uniform(seed, _S_X + 1, s, c, dt)
            out[s:s + c, 0] = r * np.cos(phi)
            out[s:s + c, 1] = r * np.sin(phi)
    elif cfg.cid == 5:    # 50 % uniform + 50 % log-normal radial shells around 1024 centres
        ncl = 1024
        cen = np.stack([uniform(seed, _S_CEN + j, 0, ncl, dt) for j in range(3)], axis=1)
        rad = 10.0 ** (-3.0 + 2.0 * uniform(seed, _S_SCALE, 0, ncl, dt))

        def fill(s, c):
            bg = uniform(seed, _S_SEL, s, c, dt) < 0.5
            cl = np.minimum((uniform(seed, _S_CL, s, c, dt) * ncl).astype(np.int64), ncl - 1)
            g = np.stack([normal(seed, _S_G + 2 * j, s, c, dt) for j in range(3)], axis=1)
            gn = np.sqrt((g * g).sum(axis=1))
            gn[gn == 0.0] = 1.0
            rr = rad[cl] * np.exp(0.25 * normal(seed, _S_SHELL, s, c, dt))
            for j in range(3):
                u = uniform(seed, _S_X + j, s, c, dt)
                out[s:s + c, j] = np.where(bg, u, cen[cl, j] + rr * g[:, j] / gn)
    else:
        raise ValueError(f"unknown config {cfg.cid}")
    _for_chunks(n, fill)
    return out


def make_gaussian_blob(n: int, d: int, dtype: str, seed: int = 1100) -> np.ndarray:
    """The paper's own workload shape: points ~ unit Gaussian in d dims."""
    dt = NP_DTYPE[dtype]
    out = np.empty((n, d), dtype=dt)

    def fill(s, c):
        for j in range(d):
            out[s:s + c, j] = normal(seed, _S_G + 2 * j, s, c, dt)
    _for_chunks(n, fill)
    return out


def make_noise(cfg_id: int, n: int, dtype: str, what: str = "xi") -> np.ndarray:
    """White noise xi (seed 2000+c) or a cotangent v_bar (seed 3000+c), N(0,1), in `dtype`."""
    base = {"xi": 2000, "vbar": 3000}[what]
    dt = NP_DTYPE[dtype]
    out = np.empty(n, dtype=dt)

    def fill(s, c):
        out[s:s + c] = normal(base + cfg_id, _S_NOISE, s, c, dt)
    _for_chunks(n, fill)
    return out
