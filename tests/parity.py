"""Comparison rules between the CUDA path and the oracle (reading C-13).

  filtered : max |gpu - oracle| <= 1e-5 (unit-variance noise input; BASELINE.json north_star)
  mask     : identical except voxels whose oracle |f - t| <= 1e-4 * local std for a scale that can
             explain the flip (their number is reported)
  count    : gpu count == popcount(gpu mask); differs from the oracle's by at most the band voxels
  mean/std : |mean_gpu - mean| <= 1e-5 * std, |var_gpu - var| <= 2e-5 * var, plus the fp32 rounding
             floor of the formula (see assert_stats_close)
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

FILTER_TOL = 1e-5
BAND = 1e-4
STATS_RTOL = 1e-5


@dataclass
class MaskReport:
    mismatches: int
    excused: int
    band_voxels: int

    @property
    def ok(self) -> bool:
        return self.mismatches == self.excused


def filter_maxdiff(gpu_f: np.ndarray, oracle_f: np.ndarray) -> float:
    return float(np.max(np.abs(gpu_f.astype(np.float64) - oracle_f))) if oracle_f.size else 0.0


def assert_filter_close(gpu_f, oracle_f, what="filtered", tol=FILTER_TOL):
    d = filter_maxdiff(gpu_f, oracle_f)
    assert d <= tol, f"{what}: max|diff| = {d:.3e} > {tol:g}"
    return d


def in_band(scale_result) -> np.ndarray:
    """Voxels of one scale whose decision is within rounding: |f - t| <= 1e-4 * std (oracle values)."""
    st = scale_result.stats
    return np.abs(scale_result.f - st.thr) <= BAND * st.std


def compare_mask(gpu_mask: np.ndarray, oracle_find, inside: np.ndarray | None = None) -> MaskReport:
    """gpu_mask vs the oracle's OR mask over the scales in `oracle_find` (a FindResult on the same
    region).  A mismatch is excused only if the scales that would have to flip are in their band:
      oracle 1 / gpu 0 : every scale the oracle selected must be in its band;
      oracle 0 / gpu 1 : at least one scale must be in its band.
    `inside` (bool) marks voxels outside the halo (mask there must be 0 on both sides)."""
    g = gpu_mask.astype(bool)
    o = oracle_find.mask.astype(bool)
    bands = [in_band(s) for s in oracle_find.scales]
    sels = [s.stats.mask.astype(bool) for s in oracle_find.scales]
    if inside is not None:
        assert not g[~inside].any(), "gpu mask set inside the halo"
    any_band = np.zeros(g.shape, bool)
    all_sel_in_band = np.ones(g.shape, bool)
    for b, s in zip(bands, sels):
        any_band |= b
        all_sel_in_band &= (~s) | b
    mism = g != o
    miss = mism & o          # oracle 1, gpu 0
    extra = mism & ~o        # oracle 0, gpu 1
    excused = int((miss & all_sel_in_band).sum() + (extra & any_band).sum())
    if inside is not None:
        any_band &= inside
    return MaskReport(int(mism.sum()), excused, int(any_band.sum()))


def assert_mask_ok(gpu_mask, oracle_find, inside=None, what="mask") -> MaskReport:
    rep = compare_mask(gpu_mask, oracle_find, inside)
    assert rep.ok, (f"{what}: {rep.mismatches} mismatching voxels, only {rep.excused} inside the "
                    f"1e-4*std band ({rep.band_voxels} band voxels)")
    return rep


def assert_stats_close(gpu_mean, gpu_std, stats, what="stats"):
    """mean within 1e-5*std, variance within 2e-5*var (= std within 1e-5 relative), each plus the
    fp32 rounding floor of the formula itself: m and S2/n - m^2 are formed from fp32 sums whose
    rounding error is a few 2^-24 of sqrt(E[f^2]) resp. E[f^2] = std^2 + mean^2 (DESIGN.md,
    "Tolerances").  For noise-like windows (|mean| <~ std) the floor is ~1e-6 of the value."""
    eps = 2.0 ** -24
    msq = stats.std ** 2 + stats.mean ** 2
    tol_m = STATS_RTOL * stats.std + 8 * eps * np.sqrt(msq) + 1e-30
    tol_v = 2 * STATS_RTOL * stats.std ** 2 + 16 * eps * msq + 1e-30
    dm = np.abs(gpu_mean.astype(np.float64) - stats.mean)
    dv = np.abs(gpu_std.astype(np.float64) ** 2 - stats.std ** 2)
    assert np.all(dm <= tol_m), f"{what}: mean off by {np.max(dm / tol_m):.2f} x tolerance"
    assert np.all(dv <= tol_v), f"{what}: variance off by {np.max(dv / tol_v):.2f} x tolerance"
    return float(np.max(dm / tol_m)), float(np.max(dv / tol_v))


def halo_inside(lo, hi, cube, halo) -> np.ndarray:
    zz = np.arange(lo[2], hi[2])[:, None, None]
    yy = np.arange(lo[1], hi[1])[None, :, None]
    xx = np.arange(lo[0], hi[0])[None, None, :]
    return ((xx >= halo[0]) & (xx < cube[0] - halo[0]) & (yy >= halo[1]) & (yy < cube[1] - halo[1]) &
            (zz >= halo[2]) & (zz < cube[2] - halo[2]))
