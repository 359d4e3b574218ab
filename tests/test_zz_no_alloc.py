"""pgsf_filter3d_noalloc: the entry point for callers that cannot allocate device memory (static device scratch).
Collected last on purpose (file name): the suite runs with pytest -x."""
import os
import re

import numpy as np
import pytest
import torch

import parity

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "paper_1507_04941_b200", "csrc", "pgsf_noalloc.cu")


def test_noalloc_source_calls_no_allocator():
    """The translation unit of the entry point names no allocating CUDA call and takes the scratch's device address
    from cudaGetSymbolAddress (comments stripped first)."""
    src = open(SRC).read()
    code = re.sub(r"//[^\n]*", "", re.sub(r"/\*.*?\*/", "", src, flags=re.S))
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMemcpy", "cudaMemset", "new ", "malloc(", "std::string",
                   "std::vector"):
        assert banned not in code, banned
    assert "static __device__ __align__(256)" in code and "cudaGetSymbolAddress" in code
    hdr = open(os.path.join(ROOT, "include", "pgsf.h")).read()
    assert "#define PGSF_NOALLOC_MAX_VOXELS (1 << 21)" in hdr


@pytest.fixture(scope="module")
def pg():
    from paper_1507_04941_b200 import binding, build
    build.build()
    binding.load_library()
    assert torch.cuda.is_available(), "no GPU: the product path has no CPU fallback"
    return binding


@pytest.mark.gpu
def test_noalloc_matches_filter3d_on_two_calls_in_a_row(pg):
    """Two calls in a row (the second on a smaller cube with other data and another sigma: stale scratch of the first
    call must not show), each against pgsf_filter3d of a plan on the tiled and on the generic kernels, within the
    filter tolerance of the parity tests (1e-5, tests/parity.py); the library call is handed its output buffer, and
    the device's free memory does not change across the calls."""
    from paper_1507_04941_b200 import synth
    cases = [((128, 96, 160), (2.0, 2.0, 4.0), 11), ((100, 52, 77), (1.0, 1.5, 8.0), 12)]
    inputs, outs, refs = [], [], []
    for dims, sigma, seed in cases:
        d = synth.make_cube((dims[2], dims[1], dims[0]), seed, 6, device="cuda")
        inputs.append(d)
        outs.append(torch.empty_like(d))
        r = []
        for flags in (0, pg.PGSF_FLAG_FORCE_GENERIC):
            with pg.Plan(dims, [sigma], (4, 4, 8), 3.0, flags=flags) as plan:
                r.append(plan.pgsf_filter3d(0, d[None])[0].clone())
        refs.append(r)
    torch.cuda.synchronize()
    pg.pgsf_filter3d_noalloc(inputs[0], cases[0][1], d_out=outs[0])        # (first call on the device: set-up)
    torch.cuda.synchronize()
    outs[0].zero_()
    free0 = torch.cuda.mem_get_info()[0]
    for (dims, sigma, seed), d, o in zip(cases, inputs, outs):             # the two calls in a row, one stream
        pg.pgsf_filter3d_noalloc(d, sigma, d_out=o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    for (dims, sigma, seed), o, r in zip(cases, outs, refs):
        got = o.cpu().numpy()
        assert float(np.abs(got).max()) > 0.1
        parity.assert_filter_close(got, r[0].cpu().numpy().astype(np.float64), f"noalloc vs tiled {dims}")
        parity.assert_filter_close(got, r[1].cpu().numpy().astype(np.float64), f"noalloc vs generic {dims}")
        assert torch.equal(o, r[1]), "same arithmetic as the generic kernels: bit for bit"


@pytest.mark.gpu
def test_noalloc_rejects_what_does_not_fit(pg):
    big = torch.zeros((129, 128, 128), device="cuda")                       # 1 plane above 2^21 voxels
    with pytest.raises(pg.PgsfError) as e:
        pg.pgsf_filter3d_noalloc(big, (1, 1, 2))
    assert e.value.status == pg.PGSF_ERR_UNSUPPORTED and "PGSF_NOALLOC_MAX_VOXELS = 2097152" in str(e.value)
    small = torch.zeros((8, 8, 8), device="cuda")
    with pytest.raises(pg.PgsfError) as e:
        pg.pgsf_filter3d_noalloc(small, (1, 1, 40))                         # radius 120 > 96
    assert e.value.status == pg.PGSF_ERR_UNSUPPORTED
    with pytest.raises(pg.PgsfError) as e:
        pg.pgsf_filter3d_noalloc(small, (1, -1, 2))
    assert e.value.status == pg.PGSF_ERR_INVALID_ARG
    with pytest.raises(pg.PgsfError) as e:
        pg.pgsf_filter3d_noalloc(small, (1, 1, 2), d_out=small)             # in place
    assert e.value.status == pg.PGSF_ERR_INVALID_ARG and "overlap" in str(e.value)
    full = torch.ones((128, 128, 128), device="cuda")                       # exactly the maximum
    out = pg.pgsf_filter3d_noalloc(full, (1, 1, 2))
    torch.cuda.synchronize()
    assert abs(float(out[64, 64, 64]) - 1.0) < 1e-6
