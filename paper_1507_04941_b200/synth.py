"""Seeded synthetic HI-like cubes: the input recipe of DESIGN.md ("Synthetic inputs").

This module holds NONE of the method's arithmetic (no taps, no filtering, no statistics); it only
makes inputs, for BOTH the CUDA path and the oracle (tests and bench.py hand the same tensor,
or a host copy of a brick of it, to each side).

Stand-in for the paper's simulated ASKAP/WALLABY cube (2048x2048x16384 fp32) and its
1024x1048x4096 cut-out, which are not available: fp32, noise dominated, frequency the
long axis, sources extended mostly along frequency.

Layout: torch tensor [nz, ny, nx] (or [batch, nz, ny, nx]); x is unit stride (reading C-0).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import numpy as np
import torch


@dataclass(frozen=True)
class Workload:
    """One entry of BASELINE.json `configs` (index i = 1..5 as in SURVEY.md)."""
    name: str
    dims: Tuple[int, int, int]                 # (nx, ny, nz) of one cube INCLUDING any halo
    batch: int
    halo: Tuple[int, int, int]
    seed: int
    n_sources: int                             # per (sub-)cube
    sigmas: Tuple[Tuple[float, float, float], ...]
    box_half: Tuple[int, int, int]
    k: float
    sxy_range: Tuple[float, float] = (1.0, 4.0)
    sz_range: Tuple[float, float] = (2.0, 20.0)
    amp_range: Tuple[float, float] = (0.3, 3.0)
    independent_sxy: bool = True               # "ellipsoidal": sx, sy drawn independently
    noise_ramp: Optional[Tuple[float, float]] = None   # per-channel noise std from..to across z
    truncate: float = 3.0

    @property
    def voxels(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2] * self.batch

    @property
    def core_voxels(self) -> int:
        return ((self.dims[0] - 2 * self.halo[0]) * (self.dims[1] - 2 * self.halo[1]) *
                (self.dims[2] - 2 * self.halo[2]) * self.batch)


_BANK3 = ((1.0, 1.0, 2.0), (2.0, 2.0, 4.0), (3.0, 3.0, 8.0))

WORKLOADS = {
    1: Workload("config1_64x64x128", (64, 64, 128), 1, (0, 0, 0), 0, 8, (_BANK3[0],), (4, 4, 8), 4.0,
                sxy_range=(1.0, 3.0), sz_range=(2.0, 8.0), amp_range=(0.5, 3.0), independent_sxy=False),
    2: Workload("config2_512x512x1024", (512, 512, 1024), 1, (0, 0, 0), 1, 200, _BANK3, (8, 8, 16), 4.0),
    3: Workload("config3_1024x1024x2048", (1024, 1024, 2048), 1, (0, 0, 0), 2, 1000,
                _BANK3 + ((4.0, 4.0, 16.0),), (16, 16, 32), 4.0, noise_ramp=(0.8, 1.2)),
    4: Workload("config4_64x(256x256x512+halo32)", (320, 320, 576), 64, (32, 32, 32), 3, 20, _BANK3,
                (8, 8, 16), 4.0),
    # reading C-12: spatial sigma 1..3 linearly spaced, paired in order with the spectral sigmas
    5: Workload("config5_2048x2048x512", (2048, 2048, 512), 1, (0, 0, 0), 4, 500,
                ((1.0, 1.0, 4.0), (1.5, 1.5, 8.0), (2.0, 2.0, 16.0), (2.5, 2.5, 24.0), (3.0, 3.0, 32.0)),
                (16, 16, 48), 4.0, sz_range=(8.0, 40.0)),
}


def scaled(w: Workload, dims: Tuple[int, int, int], batch: Optional[int] = None,
           n_sources: Optional[int] = None) -> Workload:
    """Same recipe on a smaller cube (for tests that the oracle must finish in seconds)."""
    from dataclasses import replace
    return replace(w, name=f"{w.name}@{dims[0]}x{dims[1]}x{dims[2]}", dims=tuple(dims),
                   batch=w.batch if batch is None else batch,
                   n_sources=w.n_sources if n_sources is None else n_sources)


def _draw_sources(rng: np.random.Generator, n: int, dims, sxy_range, sz_range, amp_range,
                  independent_sxy: bool):
    """Fixed draw order per source: cx, cy, cz, sx, [sy], sz, A."""
    nx, ny, nz = dims
    out = []
    for _ in range(n):
        cx = rng.uniform(0.0, nx)
        cy = rng.uniform(0.0, ny)
        cz = rng.uniform(0.0, nz)
        sx = rng.uniform(*sxy_range)
        sy = rng.uniform(*sxy_range) if independent_sxy else sx
        sz = rng.uniform(*sz_range)
        amp = rng.uniform(*amp_range)
        out.append((cx, cy, cz, sx, sy, sz, amp))
    return out


def _add_sources(cube: torch.Tensor, sources) -> None:
    """cube[z,y,x] += A exp(-0.5(dx^2/sx^2 + dy^2/sy^2 + dz^2/sz^2)) on |d| <= 5 sigma, clipped."""
    nz, ny, nx = cube.shape
    dev = cube.device
    for (cx, cy, cz, sx, sy, sz, amp) in sources:
        prof = []
        sl = []
        for c, s, n in ((cz, sz, nz), (cy, sy, ny), (cx, sx, nx)):
            a = max(0, int(np.floor(c - 5.0 * s)))
            b = min(n, int(np.ceil(c + 5.0 * s)) + 1)
            if b <= a:
                prof = None
                break
            t = torch.arange(a, b, dtype=torch.float64, device=dev)
            prof.append(torch.exp(-0.5 * ((t - c) / s) ** 2))
            sl.append(slice(a, b))
        if prof is None:
            continue
        blob = amp * prof[0][:, None, None] * prof[1][None, :, None] * prof[2][None, None, :]
        cube[sl[0], sl[1], sl[2]] += blob.to(torch.float32)


def make_cube(shape_zyx: Sequence[int], seed: int, n_sources: int, device="cpu",
              sxy_range=(1.0, 3.0), sz_range=(2.0, 8.0), amp_range=(0.5, 3.0),
              independent_sxy=False, noise_ramp=None, generator: Optional[torch.Generator] = None,
              source_rng: Optional[np.random.Generator] = None) -> torch.Tensor:
    """i.i.d. N(0,1) fp32 noise (torch generator on `device`, seeded `seed`) + injected Gaussian
    sources whose parameters come from numpy's default_rng(seed + 1000)."""
    nz, ny, nx = (int(v) for v in shape_zyx)
    dev = torch.device(device)
    g = generator
    if g is None:
        g = torch.Generator(device=dev)
        g.manual_seed(int(seed))
    cube = torch.randn((nz, ny, nx), generator=g, device=dev, dtype=torch.float32)
    if noise_ramp is not None:
        ramp = torch.linspace(noise_ramp[0], noise_ramp[1], nz, device=dev, dtype=torch.float32)
        cube *= ramp[:, None, None]
    rng = source_rng if source_rng is not None else np.random.default_rng(int(seed) + 1000)
    _add_sources(cube, _draw_sources(rng, n_sources, (nx, ny, nz), sxy_range, sz_range, amp_range,
                                     independent_sxy))
    return cube


def workload_sources(w: Workload):
    """The injected sources of a workload, exactly as make_workload draws them: one list per batch entry of
    (cx, cy, cz, sx, sy, sz, amplitude) tuples.  Input generation only (tests centre their parity bricks on the
    brightest sources)."""
    rng = np.random.default_rng(int(w.seed) + 1000)
    return [_draw_sources(rng, w.n_sources, w.dims, w.sxy_range, w.sz_range, w.amp_range, w.independent_sxy)
            for _ in range(w.batch)]


def make_workload(w: Workload, device="cpu") -> torch.Tensor:
    """The input tensor of a workload: [batch, nz, ny, nx] fp32 (batch dim kept even for 1)."""
    nx, ny, nz = w.dims
    dev = torch.device(device)
    g = torch.Generator(device=dev)
    g.manual_seed(int(w.seed))
    rng = np.random.default_rng(int(w.seed) + 1000)
    out = torch.empty((w.batch, nz, ny, nx), device=dev, dtype=torch.float32)
    for b in range(w.batch):
        out[b] = make_cube((nz, ny, nx), w.seed, w.n_sources, device=dev, sxy_range=w.sxy_range,
                           sz_range=w.sz_range, amp_range=w.amp_range,
                           independent_sxy=w.independent_sxy, noise_ramp=w.noise_ramp,
                           generator=g, source_rng=rng)
    return out
