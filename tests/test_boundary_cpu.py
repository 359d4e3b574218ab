"""CPU-side tests of the boundary: the C-ABI library builds, loads and exports every symbol that
include/pgsf.h declares; argument validation; loud failure without a GPU; the parity checker
itself (against deliberately perturbed oracle outputs).  No compute calls."""
import ctypes
import os
import re

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1507_04941_b200 import build, binding
    build.build()
    return binding.load_library()


def test_library_exports_every_declared_symbol(lib):
    from paper_1507_04941_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "pgsf.h")).read()
    declared = sorted(set(re.findall(r"PGSF_API[^;]*?\b(pgsf_\w+)\s*\(", hdr)))
    assert declared == sorted(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    # the five calls BASELINE.json north_star names
    for name in ("pgsf_plan_create", "pgsf_filter3d", "pgsf_local_threshold", "pgsf_find_multiscale",
                 "pgsf_plan_destroy"):
        assert name in declared


def test_library_has_sm100a_code_only():
    import subprocess
    from paper_1507_04941_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def _desc(binding, **kw):
    d = dict(dims=(16, 16, 16), sigmas=[(1, 1, 2)], box_half=(2, 2, 2), k=4.0)
    d.update(kw)
    return d


@pytest.mark.parametrize("kw", [
    dict(dims=(0, 16, 16)), dict(dims=(16, -1, 16)), dict(batch=0), dict(sigmas=[]),
    dict(sigmas=[(1, 1, 2)] * 9), dict(sigmas=[(-1, 1, 2)]), dict(box_half=(-1, 2, 2)),
    dict(halo=(8, 0, 0)), dict(halo=(0, 0, -1)), dict(truncate=0.0), dict(k=-1.0),
    dict(sigmas=[(float("nan"), 1, 2)]),
])
def test_plan_create_rejects_bad_arguments(lib, kw):
    from paper_1507_04941_b200 import binding
    with pytest.raises(binding.PgsfError) as ei:
        binding.Plan(**{**dict(dims_xyz=(16, 16, 16), sigmas=[(1, 1, 2)], box_half=(2, 2, 2), k=4.0),
                        **({"dims_xyz": kw.pop("dims")} if "dims" in kw else {}), **kw})
    assert ei.value.status == binding.PGSF_ERR_INVALID_ARG


@pytest.mark.parametrize("kw", [dict(sigmas=[(1, 1, 40)]), dict(box_half=(2, 2, 200))])
def test_plan_create_unsupported(lib, kw):
    from paper_1507_04941_b200 import binding
    with pytest.raises(binding.PgsfError) as ei:
        binding.Plan(**{**dict(dims_xyz=(16, 16, 16), sigmas=[(1, 1, 2)], box_half=(2, 2, 2), k=4.0), **kw})
    assert ei.value.status == binding.PGSF_ERR_UNSUPPORTED


def test_null_plan_calls_do_not_crash(lib):
    assert lib.pgsf_plan_destroy(None) == 0
    assert lib.pgsf_plan_workspace_bytes(None) == 0
    assert lib.pgsf_filter3d(None, 0, None, None, None, None) == 1
    assert lib.pgsf_local_threshold(None, None, None, 0, None, None, None, None, None) == 1
    assert lib.pgsf_find_multiscale(None, None, None, None, None, None, None) == 1
    assert lib.pgsf_find_multiscale_host(None, None, None, None, None) == 1
    assert lib.pgsf_plan_launch_count(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_gpu_fails_loudly_no_cpu_fallback(lib):
    from paper_1507_04941_b200 import binding
    with pytest.raises(binding.PgsfError) as ei:
        binding.Plan((16, 16, 16), [(1, 1, 2)], (2, 2, 2), 4.0)
    assert ei.value.status == binding.PGSF_ERR_CUDA


# ------------------------------------------------------------------ host-only logic through PGSF_FLAG_DRY_RUN plans

def _dry(binding, dims=(64, 48, 80), sigmas=((1, 1, 2), (2, 2, 4)), box=(4, 4, 8), **kw):
    return binding.Plan(dims, sigmas, box, 4.0, flags=binding.PGSF_FLAG_DRY_RUN | kw.pop("flags", 0), **kw)


@pytest.mark.parametrize("dims,sigmas,box,flags,tiled,needle", [
    ((64, 48, 80), ((1, 1, 2),), (4, 4, 8), 0, True, "tiled"),
    ((100, 48, 80), ((1, 1, 2),), (12, 12, 24), 0, True, "k_xyb"),                # hx = 12, nx % 6 != 0: still tiled
    ((64, 48, 80), ((1, 1, 2),), (10, 4, 8), 0, False, "hx = 10"),
    ((64, 48, 80), ((1, 1, 2),), (4, 4, 8), 1, False, "FORCE_GENERIC"),
    ((62, 48, 80), ((1, 1, 2),), (4, 4, 8), 0, False, "nx % 4"),
    ((64, 48, 80), ((5, 1, 2),), (4, 4, 8), 0, False, "radii (15, 3, 6)"),        # x radius above the compiled 12
    ((64, 48, 80), ((1, 1, 2),), (200 // 2 - 36, 4, 8), 0, False, "hx = 64"),     # filter tiled, statistics not
    ((8, 4, 70000), ((1, 1, 2),), (4, 4, 8), 0, False, "65535"),                  # grid.z limit
    ((8, 70000, 4), ((1, 1, 2),), (4, 4, 8), 0, False, "65535"),
])
def test_plan_path_reports_the_dispatch_decision(lib, dims, sigmas, box, flags, tiled, needle):
    """Which kernels a plan runs is decided (and can be queried) at plan time, so a shape / radius / box that
    falls off the tiled kernels is visible to the caller and can never surface as a launch failure."""
    from paper_1507_04941_b200 import binding
    with _dry(binding, dims, sigmas, box, flags=flags) as plan:
        ok, text = plan.pgsf_plan_path()
        assert ok == tiled and needle in text, text
        assert plan.pgsf_plan_workspace_bytes() > 0


def test_find_multiscale_rejects_overlapping_buffers(lib):
    """pgsf_find_multiscale parks intermediate data in the d_filtered cubes, so every buffer must be disjoint
    (validated on the host before anything is enqueued; a dry-run plan then stops with PGSF_ERR_CUDA)."""
    from paper_1507_04941_b200 import binding
    with _dry(binding) as plan:
        n = plan.voxels
        ws = plan.pgsf_plan_workspace_bytes()
        base = 1 << 40                                # fake, well aligned "device" addresses; never dereferenced
        step = ((4 * n + 255) // 256 + 1) * 256
        d_in, f0, f1, mask, cnt, wsp = (base + i * step for i in range(6))
        wsp = base + 8 * step

        def call(d_in=d_in, f=(f0, f1), mask=mask, cnt=cnt, wsp=wsp):
            arr = (ctypes.c_void_p * 2)(*f) if f is not None else None
            return lib.pgsf_find_multiscale(plan._h, ctypes.c_void_p(d_in), arr, ctypes.c_void_p(mask),
                                            ctypes.c_void_p(cnt), ctypes.c_void_p(wsp), None)

        assert call() == binding.PGSF_ERR_CUDA                       # valid arguments, no device
        assert call(f=None) == binding.PGSF_ERR_CUDA
        for bad, who in [(dict(f=(d_in, f1)), "d_in"), (dict(f=(f0, f0 + 256)), "d_filtered[1]"),
                         (dict(mask=f1 + 4 * n - 16), "d_mask"), (dict(wsp=f0 + 256), "d_workspace"),
                         (dict(cnt=mask + 8), "d_count"), (dict(wsp=d_in - ws + 256), "d_workspace")]:
            assert call(**bad) == binding.PGSF_ERR_INVALID_ARG, bad
            msg = lib.pgsf_last_error(plan._h).decode()
            assert "overlaps" in msg and who in msg, msg
        assert call(d_in=d_in + 4) == binding.PGSF_ERR_INVALID_ARG    # misaligned


def test_statistics_kernel_and_tensor_flag_in_the_plan_path(lib):
    """The plan path names the statistics kernel that will run (k_xyb, or k_ymarch under PGSF_OPT_TUNE bit 1) and a
    dry-run plan accepts PGSF_FLAG_TENSOR_ZPASS without touching a device (the operands are built on a real one)."""
    from paper_1507_04941_b200 import binding
    with _dry(binding, dims=(64, 48, 80), sigmas=((1, 1, 2), (1, 1, 16)), box=(8, 8, 16),
              flags=binding.PGSF_FLAG_TENSOR_ZPASS) as plan:
        ok, text = plan.pgsf_plan_path()
        assert ok and "k_xyb" in text, text
        plan.pgsf_plan_set_option(binding.PGSF_OPT_TUNE, 2)
        ok, text = plan.pgsf_plan_path()
        assert ok and "k_ymarch" in text, text


def test_label_objects_validates_its_arguments(lib):
    from paper_1507_04941_b200 import binding
    with _dry(binding) as plan:
        n = plan.voxels
        base = 1 << 40
        call = lambda m, l, c: lib.pgsf_label_objects(plan._h, ctypes.c_void_p(m), ctypes.c_void_p(l), ctypes.c_void_p(c), None)
        assert call(base, base + (1 << 30), base + (1 << 31)) == binding.PGSF_ERR_CUDA     # valid, no device
        assert call(0, base, 0) == binding.PGSF_ERR_INVALID_ARG
        assert call(base, base + (1 << 30) + 4, 0) == binding.PGSF_ERR_INVALID_ARG          # misaligned labels
        assert call(base, base + n - 16, 0) == binding.PGSF_ERR_INVALID_ARG                 # labels overlap the mask
        assert "overlaps" in lib.pgsf_last_error(plan._h).decode()
    with _dry(binding, dims=(2048, 2048, 1100)) as plan:                                    # > 2^32 - 2 voxels per cube
        assert lib.pgsf_label_objects(plan._h, ctypes.c_void_p(1 << 40), ctypes.c_void_p(1 << 44), None, None) == \
            binding.PGSF_ERR_UNSUPPORTED


def test_plan_options_are_validated(lib):
    from paper_1507_04941_b200 import binding
    with _dry(binding, dims=(32, 32, 32), batch=5) as plan:
        plan.pgsf_plan_set_option(binding.PGSF_OPT_GROUP_CUBES, 2)
        plan.pgsf_plan_set_option(binding.PGSF_OPT_HOST_SECTION_PLANES, 16)
        plan.pgsf_plan_set_option(binding.PGSF_OPT_HOST_DEVICE_BUDGET, 1 << 30)
        plan.pgsf_plan_set_option(binding.PGSF_OPT_TUNE, 2 | 4)
        plan.pgsf_plan_set_option(binding.PGSF_OPT_TUNE, 0)
        for opt, val in [(binding.PGSF_OPT_GROUP_CUBES, 0), (binding.PGSF_OPT_GROUP_CUBES, 6),
                         (binding.PGSF_OPT_HOST_SECTION_PLANES, 33), (binding.PGSF_OPT_HOST_DEVICE_BUDGET, -1),
                         (binding.PGSF_OPT_TUNE, -1), (binding.PGSF_OPT_TUNE, 1 << 16), (99, 0)]:
            with pytest.raises(binding.PgsfError) as ei:
                plan.pgsf_plan_set_option(opt, val)
            assert ei.value.status == binding.PGSF_ERR_INVALID_ARG


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1507_04941_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|pgsf_oracle|oracle/|liboracle", src), \
                    f"{f} reaches into oracle/"
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".c")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import paper_1507_04941_b200" not in src and "from paper_1507_04941_b200" not in src


# ------------------------------------------------------------------------------ the checker itself

def test_parity_checker_detects_perturbations(oracle):
    from paper_1507_04941_b200 import synth
    import parity
    d = synth.make_cube((48, 32, 32), seed=3, n_sources=4, device="cpu").numpy()
    res = oracle.find_full(d, [(1, 1, 2), (2, 2, 4)], (3, 3, 6), 2.5)
    f0 = res.scales[0].f
    # exact copy passes
    parity.assert_filter_close(f0.astype(np.float32), f0)
    assert parity.compare_mask(res.mask, res).mismatches == 0
    # a 2e-5 bump on one voxel fails the filter tolerance
    bad = f0.astype(np.float32).copy()
    bad[10, 10, 10] += 2e-5
    with pytest.raises(AssertionError):
        parity.assert_filter_close(bad, f0)
    # flipping a voxel far from the threshold is NOT excused
    far = np.argwhere(~(parity.in_band(res.scales[0]) | parity.in_band(res.scales[1])))[0]
    m = res.mask.copy()
    m[tuple(far)] ^= 1
    rep = parity.compare_mask(m, res)
    assert rep.mismatches == 1 and rep.excused == 0 and not rep.ok
    # flipping a voxel inside the band IS excused: build one by moving f onto t
    import copy
    res2 = copy.deepcopy(res)
    v = tuple(np.argwhere(res.mask == 0)[5])
    for s in res2.scales:
        s.f[v] = s.stats.thr[v]
    m = res2.mask.copy()
    m[v] = 1
    rep = parity.compare_mask(m, res2)
    assert rep.mismatches == 1 and rep.excused == 1 and rep.ok
    # mean / std tolerance
    st = res.scales[0].stats
    parity.assert_stats_close(st.mean.astype(np.float32), st.std.astype(np.float32), st)
    with pytest.raises(AssertionError):
        parity.assert_stats_close(st.mean.astype(np.float32), (st.std * (1 + 1e-4)).astype(np.float32), st)


def test_synth_is_seeded_and_config_shaped():
    from paper_1507_04941_b200 import synth
    w = synth.scaled(synth.WORKLOADS[3], (32, 24, 40), n_sources=3)
    a = synth.make_workload(w, "cpu")
    b = synth.make_workload(w, "cpu")
    assert a.shape == (1, 40, 24, 32) and a.dtype == torch.float32
    assert torch.equal(a, b)
    noise_only = synth.make_workload(synth.scaled(synth.WORKLOADS[3], (32, 24, 40), n_sources=0), "cpu")
    # the per-channel ramp 0.8 -> 1.2 is there
    assert noise_only[0, :5].std() < noise_only[0, -5:].std()
    assert (a - noise_only).abs().max() > 0.25         # sources were injected
    w4 = synth.scaled(synth.WORKLOADS[4], (24, 24, 32), batch=3, n_sources=2)
    c = synth.make_workload(w4, "cpu")
    assert c.shape == (3, 32, 24, 24) and not torch.equal(c[0], c[1])
    assert synth.WORKLOADS[5].sigmas[-1] == (3.0, 3.0, 32.0) and synth.WORKLOADS[2].voxels == 2 ** 28


# ---------------------------------------------------------------------------------- N > 1: replicas only

def _replica_worker(rank, world, port, out):
    import os
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1507_04941_b200 import synth
    w = bench.replica_workload(synth.WORKLOADS[1], rank)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")       # rank 1 is the slow one
    out.put((rank, w.seed, ms, bench.aggregate_value(w.voxels, len(w.sigmas), world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_world_size_2_gloo():
    """bench.py --gpus N runs N independent replicas: seeds differ per rank, the step
    time is the max over ranks, the value is the whole-job aggregate.  No data-path collective exists."""
    import socket
    import torch.multiprocessing as mp
    from paper_1507_04941_b200 import synth
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_replica_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = synth.WORKLOADS[1]
    assert [r[1] for r in res] == [w.seed, w.seed + 100]
    assert all(abs(r[2] - 15.0) < 1e-12 for r in res)                # max over ranks on every rank
    expect = w.voxels * len(w.sigmas) * 2 / 15e-3 / 1e9
    assert all(abs(r[3] - expect) < 1e-9 * expect for r in res)
