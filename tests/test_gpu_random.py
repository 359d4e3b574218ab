"""Randomised sweeps against the oracle: seeded random shapes, scales, boxes, halos, batches and plan flags through
the same comparisons as tests/test_gpu_parity.py.  The hand-picked cases there cover what was thought of; these cover
what was not (round 2: the sweep found the Kahan residue of the per-scale statistics beside bright sources and the
mixed kernels of a streamed tensor-core march; both are regression tests in test_gpu_parity.py now).
Every case prints its workload, so a failure can be copied into a parametrised test."""
import random

import numpy as np
import pytest
import torch

import parity
import test_gpu_parity as T
from test_gpu_parity import pg, synth  # noqa: F401  (module-scoped fixtures)

pytestmark = pytest.mark.gpu


def _draw_workload(rng, synth, seed, it, shape_mode):
    from dataclasses import replace
    fast = rng.random() < 0.7
    nx = rng.choice([4, 8, 12, 16, 20, 28, 36, 60, 64, 100, 132, 200, 260, 300]) if fast else rng.randint(5, 150)
    ny, nz, ns = rng.randint(3, 120), rng.randint(3, 160), rng.randint(1, 4)
    if shape_mode == "long":        # one long axis: several x strips, y chunks (> 2048 rows), many z march steps
        ax = rng.choice("xyz")
        if ax == "x":
            nx, ny, nz = rng.choice([520, 772, 1024, 1300]), rng.randint(3, 24), rng.randint(3, 40)
        elif ax == "y":
            nx, ny, nz = rng.choice([8, 16, 36]), rng.choice([1600, 2100, 2600, 4200]), rng.randint(3, 24)
        else:
            nx, ny, nz = rng.choice([8, 16, 36]), rng.randint(3, 24), rng.choice([300, 700, 1100])
        ns = rng.randint(1, 2)
    sx = [rng.choice([1, 2, 3, 4]) if fast else rng.choice([0.5, 1, 1.5, 2, 2.7, 3.3]) for _ in range(ns)]
    sy = ([s if rng.random() < 0.6 else rng.choice([1, 2, 3, 4]) for s in sx] if fast
          else [rng.choice([0.5, 1, 2, 3.1]) for _ in range(ns)])
    sz = [rng.choice([2, 4, 8, 16]) if rng.random() < 0.8 else rng.choice([1, 3, 5, 7, 24, 32]) for _ in range(ns)]
    box = (rng.choice([4, 8, 12, 16]) if fast else rng.randint(1, 14), rng.randint(1, 18), rng.randint(1, 34))
    batch = rng.choice([1, 1, 2, 3])
    halo = (0, 0, 0)
    if rng.random() < 0.5:
        halo = (rng.randint(0, min(6, (nx - 1) // 2)), rng.randint(0, min(6, (ny - 1) // 2)),
                rng.randint(0, min(6, (nz - 1) // 2)))
    flags = rng.choice([0, 0, 0, 1, 8])
    w = replace(synth.scaled(synth.WORKLOADS[2], (nx, ny, nz), batch=batch, n_sources=rng.randint(0, 10)),
                sigmas=tuple(zip(sx, sy, sz)), box_half=box, k=rng.choice([2.5, 3.0, 3.5]), halo=halo,
                seed=1000 * seed + it)
    return w, flags


@pytest.mark.parametrize("seed,cases,shape_mode", [(101, 40, "any"), (102, 20, "long")])
def test_random_workloads_find_and_statistics(pg, synth, oracle, seed, cases, shape_mode):
    """pgsf_find_multiscale + the per-scale calls (filtered cubes, mean / sd, masks, counts) on random workloads,
    tiled / generic / tensor-core plans."""
    rng = random.Random(seed)
    for it in range(cases):
        w, flags = _draw_workload(rng, synth, seed, it, shape_mode)
        d = synth.make_workload(w, "cuda")
        print(f"[{seed}:{it}] dims={w.dims} sigmas={w.sigmas} box={w.box_half} batch={w.batch} halo={w.halo} "
              f"flags={flags} k={w.k} n_sources={w.n_sources} seed={w.seed}", flush=True)
        T._full_compare(pg, oracle, w, d, flags, check_stats=(flags != pg.PGSF_FLAG_TENSOR_ZPASS))


@pytest.mark.parametrize("seed,cases", [(201, 40)])
def test_random_workloads_other_entry_points(pg, synth, oracle, seed, cases):
    """The streamed host entry point against the resident call (bit for bit; random section sizes, pinned and
    pageable input), pgsf_label_objects, pgsf_filter3d_weighted and pgsf_filter3d_direct against the oracle."""
    from dataclasses import replace
    rng = random.Random(seed)
    for it in range(cases):
        kind = rng.choice(["host", "host", "label", "weighted", "direct"])
        nx = rng.choice([8, 16, 36, 64, 100, 132]) if rng.random() < 0.7 else rng.randint(5, 90)
        ny, nz, ns = rng.randint(3, 90), rng.randint(3, 420), rng.randint(1, 3)
        sig = tuple((rng.choice([1, 2, 3]), rng.choice([1, 2, 3]), rng.choice([1, 2, 4, 8, 16])) for _ in range(ns))
        box = (rng.choice([4, 8, 12, 16, 5]), rng.randint(1, 12), rng.randint(1, 40))
        batch = rng.choice([1, 1, 2])
        halo = (0, 0, 0)
        if rng.random() < 0.4:
            halo = (rng.randint(0, min(4, (nx - 1) // 2)), rng.randint(0, min(4, (ny - 1) // 2)),
                    rng.randint(0, min(9, (nz - 1) // 2)))
        flags = rng.choice([0, 0, 1, 8])
        w = replace(synth.scaled(synth.WORKLOADS[2], (nx, ny, nz), batch=batch, n_sources=rng.randint(1, 10)),
                    sigmas=sig, box_half=box, k=rng.choice([2.5, 3.0]), halo=halo, seed=7000 * seed + it)
        print(f"[{seed}:{it}] {kind} dims={w.dims} sigmas={sig} box={box} batch={batch} halo={halo} flags={flags} "
              f"k={w.k} n_sources={w.n_sources} seed={w.seed}", flush=True)
        d = synth.make_workload(w, "cuda")
        if kind == "host":
            section = min(nz, rng.choice([0, 64, 128, 192, 256]))
            keep, pinned = rng.random() < 0.5, rng.random() < 0.6
            with T._plan(pg, w, flags) as plan:
                mask, cnt, filt = plan.pgsf_find_multiscale(d, keep_filtered=True)
                torch.cuda.synchronize()
            h_in = d.cpu().pin_memory() if pinned else d.cpu()
            h_mask, count, hf = T._host_run(pg, w, h_in, section=section, keep=keep, flags=flags)
            assert count == int(cnt.item()) and torch.equal(h_mask, mask.cpu()), f"section {section}"
            if keep:
                for s in range(ns):
                    assert torch.equal(hf[s], filt[s].cpu()), f"section {section}: filtered cube {s} differs"
        elif kind == "label":
            with T._plan(pg, w, flags) as plan:
                mask, cnt, _ = plan.pgsf_find_multiscale(d)
                if rng.random() < 0.3:      # dense random masks: long merge chains
                    gen = torch.Generator(device="cuda").manual_seed(w.seed)
                    mask = (torch.rand(mask.shape, device="cuda", generator=gen) < rng.choice([0.02, 0.2, 0.6])).to(torch.uint8)
                labels, nobj = plan.pgsf_label_objects(mask)
                torch.cuda.synchronize()
            total = 0
            for b in range(batch):
                ref, nb = oracle.label26(mask[b].cpu().numpy())
                total += nb
                assert np.array_equal(labels[b].cpu().numpy().view(np.uint32), ref), f"labels of cube {b} differ"
            assert int(nobj.item()) == total
        elif kind == "weighted":
            w1, d1 = replace(w, batch=1), d[:1].contiguous()
            gen = torch.Generator(device="cuda").manual_seed(w.seed)
            wt = torch.empty_like(d1).uniform_(0.25, 2.0, generator=gen)
            if rng.random() < 0.5:
                wt[:, nz // 3] = 0.0
            mode = rng.choice([0, 1])
            with T._plan(pg, w1, flags & 1) as plan:
                for s in range(ns):
                    out = plan.pgsf_filter3d_weighted(s, d1, wt, mode)
                    torch.cuda.synchronize()
                    ref = oracle.wfilter_full(d1[0].cpu().numpy(), wt[0].cpu().numpy(), sig[s], mode)
                    got = out[0].cpu().numpy().astype(np.float64)
                    assert np.isfinite(got).all()
                    assert np.max(np.abs(got - ref)) <= T.WEIGHTED_TOL * np.max(np.abs(ref)), f"scale {s} mode {mode}"
        else:
            w1, d1 = replace(w, batch=1), d[:1].contiguous()
            fshape = (2 * rng.randint(0, 6) + 1, 2 * rng.randint(0, 3) + 1, 2 * rng.randint(0, 4) + 1)
            f = np.random.default_rng(w.seed).standard_normal(fshape).astype(np.float32)
            f /= np.abs(f).sum()
            fp64 = rng.random() < 0.5
            with T._plan(pg, w1) as plan:
                out = plan.pgsf_filter3d_direct(torch.from_numpy(f).cuda(), d1, fp64_accum=fp64)
                torch.cuda.synchronize()
            ref = oracle.filter_general(d1[0].cpu().numpy(), f.astype(np.float64))
            parity.assert_filter_close(out[0].cpu().numpy(), ref, f"direct filter {fshape} fp64={fp64}")
