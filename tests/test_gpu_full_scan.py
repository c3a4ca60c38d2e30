"""Whole-scan, per-pixel parity of the CUDA path with the fp64 oracle on C3 and C4 (BASELINE.json north_star:
"all five configs match the oracle within 1e-4 relative per pixel"), in the launch configuration bench.py times.

Every pixel of every compared projection goes through parity_util's three checks: integer ray table bit for bit,
line integrals within 1e-4 relative + 1e-6 of the image maximum, signal within 1e-4 relative.

    python -m pytest tests/test_gpu_full_scan.py -m gpu -q                  # every 15th / 82nd projection (~1 min)
    python -m pytest tests/test_gpu_full_scan.py -m gpu -q -s --full-scan   # all 360 + all 656 projections (~25 min)

With --full-scan each test writes its record to gpurun_out/full_parity_<config>.json; profiles/r02_full_parity.md
is the summary of one such run.
"""
import json
import os
import time

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
from parity_util import (LI_FLOOR, LI_RTOL, check_line_integrals, check_ray_table, check_signal,  # noqa: E402
                         face_tie_checker, siddon_sliver_checker)

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gdrr():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    import paper_1204_6367_b200 as g
    return g


def _record(name, rec):
    out = os.path.join(ROOT, "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, f"full_parity_{name}.json"), "w") as f:
        json.dump(rec, f, indent=1)


def _scan_parity(gdrr, w, name, projections, block, sampler=0, layout=2, method="trilinear"):
    """Projects `projections` (a list of indices into w's scan) in blocks, runs the oracle on every pixel of each
    block and applies the three checks; returns the record of the worst cases."""
    siddon = method == "siddon"
    rec = dict(config=name, method=method, sampler=sampler, layout=layout, projections=len(projections), pixels=0, samples=0,
               ray_table_differences=0, face_tie_entries=0, worst_rel_signal=0.0, worst_rel_li=0.0, li_floor_pixels=0,
               worst_projection=None, oracle_seconds=0.0, gpu_kernel_launches=0)
    t_start = time.time()
    kw = dict(method=gdrr.GDRR_METHOD_SIDDON) if siddon else {}
    with gdrr.Projector(w, layout=layout, sampler=sampler, **kw) as pr:
        for b in range(0, len(projections), block):
            idx = projections[b:b + block]
            contiguous = list(idx) == list(range(idx[0], idx[0] + len(idx)))
            if contiguous:                                   # one launch for the block, as bench.py launches
                sig, li, tab = pr.project(proj_begin=idx[0], proj_count=len(idx), want_li=True, want_table=True)
                sig, li, tab = sig.cpu().numpy(), li.cpu().numpy(), tab.cpu().numpy()
            else:
                outs = [pr.project(proj_begin=p, proj_count=1, want_li=True, want_table=True) for p in idx]
                sig = np.concatenate([o[0].cpu().numpy() for o in outs])
                li = np.concatenate([o[1].cpu().numpy() for o in outs])
                tab = np.concatenate([o[2].cpu().numpy() for o in outs])
            t0 = time.time()
            ref = oracle.project(w.with_phis(w.phis[idx]), method=method)
            rec["oracle_seconds"] += time.time() - t0
            what = f"{name} projections {idx[0]}..{idx[-1]}"
            check_ray_table(tab, ref["ray_table"], what)
            rec["face_tie_entries"] += int(np.count_nonzero((ref["line_integrals"] == 0.0) & (li != 0.0)))
            # (the face tie of reading Q9 belongs to the midpoint rule's sample positions; Siddon's walk has the sliver
            # tie of reading Q26 instead: the ray must be shown to cross two planes within 1e-3 mm of each other)
            slivers = []
            rel_li, n_floor = check_line_integrals(li, ref["line_integrals"], what,
                                                   siddon_sliver_checker(w, idx, slivers) if siddon
                                                   else face_tie_checker(w, idx))
            rec["sliver_tie_entries"] = rec.get("sliver_tie_entries", 0) + len(slivers)
            rel_sig = check_signal(sig, ref["signal"], what)
            rec["pixels"] += int(sig.size)
            rec["samples"] += int(ref["ray_table"][..., 1].sum())
            if siddon:
                rec["segments"] = rec.get("segments", 0) + int(ref["n_segments"].sum())
            rec["li_floor_pixels"] += n_floor
            rec["worst_rel_li"] = max(rec["worst_rel_li"], rel_li)
            if rel_sig > rec["worst_rel_signal"]:
                rec["worst_rel_signal"] = rel_sig
                per_proj = np.abs(sig - ref["signal"]).reshape(len(idx), -1) / ref["signal"].reshape(len(idx), -1)
                rec["worst_projection"] = int(idx[int(np.argmax(per_proj.max(axis=1)))])
        rec["gpu_kernel_launches"] = pr.kernel_launches()
    rec["seconds"] = time.time() - t_start
    rec["tolerances"] = dict(signal_rtol=1e-4, li_rtol=LI_RTOL, li_floor_of_max=LI_FLOOR, ray_table="bit-exact")
    return rec


def _projection_list(n_proj, full, stride):
    return list(range(n_proj)) if full else list(range(0, n_proj, stride))


def test_c3_whole_scan_per_pixel(gdrr, workloads_cache, request):
    """C3: all 360 projections with --full-scan (7.1e7 pixels, 7.8e10 samples), else every 15th, contiguous blocks
    of 8 projections per launch."""
    full = request.config.getoption("--full-scan")
    w = workloads_cache("C3")
    if full:
        rec = _scan_parity(gdrr, w, "C3", list(range(w.n_proj)), 8)
        _record("C3", rec)
    else:
        rec = _scan_parity(gdrr, w, "C3", _projection_list(w.n_proj, False, 15), 8)
    print(json.dumps(rec))
    assert rec["ray_table_differences"] == 0 and rec["worst_rel_signal"] <= 1e-4


def test_c4_whole_scan_per_pixel(gdrr, workloads_cache, request):
    """C4: all 656 projections with --full-scan (5.2e8 pixels, 4.9e11 samples), else every 82nd."""
    full = request.config.getoption("--full-scan")
    w = workloads_cache("C4")
    if full:
        rec = _scan_parity(gdrr, w, "C4", list(range(w.n_proj)), 4)
        _record("C4", rec)
    else:
        rec = _scan_parity(gdrr, w, "C4", _projection_list(w.n_proj, False, 82), 4)
    print(json.dumps(rec))
    assert rec["ray_table_differences"] == 0 and rec["worst_rel_signal"] <= 1e-4


@pytest.mark.parametrize("sampler,layout", [(1, 2), (2, 2), (0, 0), (0, 1)],
                         ids=["gather", "staged", "brick", "linear"])
def test_c3_full_projections_non_default_paths(gdrr, workloads_cache, request, sampler, layout):
    """The gather kernel, the staged kernel forced, and the two exact layouts at C3 size: every pixel of the
    projections at 0, 37 and 90 degrees against the oracle."""
    w = workloads_cache("C3")
    rec = _scan_parity(gdrr, w, "C3", [0, 37, 90], 1, sampler=sampler, layout=layout)
    if request.config.getoption("--full-scan"):
        _record(f"C3_{request.node.callspec.id}", rec)
    print(json.dumps(rec))


def test_c3_whole_scan_siddon_per_pixel(gdrr, workloads_cache, request):
    """GDRR_METHOD_SIDDON over the C3 scan against the oracle's Siddon option: all 360 projections
    with --full-scan (5.2e10 voxel segments), else every 30th."""
    full = request.config.getoption("--full-scan")
    w = workloads_cache("C3")
    if full:
        rec = _scan_parity(gdrr, w, "C3", list(range(w.n_proj)), 8, method="siddon")
        _record("C3_siddon", rec)
    else:
        rec = _scan_parity(gdrr, w, "C3", _projection_list(w.n_proj, False, 30), 8, method="siddon")
    print(json.dumps(rec))
    assert rec["ray_table_differences"] == 0 and rec["worst_rel_signal"] <= 1e-4


def test_c4_whole_scan_siddon_per_pixel(gdrr, workloads_cache, request):
    """The same on C4: all 656 projections with --full-scan (3.3e11 voxel segments), else every 82nd."""
    full = request.config.getoption("--full-scan")
    w = workloads_cache("C4")
    if full:
        rec = _scan_parity(gdrr, w, "C4", list(range(w.n_proj)), 4, method="siddon")
        _record("C4_siddon", rec)
    else:
        rec = _scan_parity(gdrr, w, "C4", _projection_list(w.n_proj, False, 82), 4, method="siddon")
    print(json.dumps(rec))
    assert rec["ray_table_differences"] == 0 and rec["worst_rel_signal"] <= 1e-4


def test_c3_whole_scan_staged_equals_gather(gdrr, workloads_cache):
    """All 360 projections of C3 through GDRR_SAMPLER_STAGED and GDRR_SAMPLER_GATHER (which shares no staging
    code): identical ray tables, signals within 2e-5 on every pixel (only the summation chunks and the re-basing
    of the position differ).  Needs no oracle time, so it always covers the whole scan."""
    w = workloads_cache("C3")
    worst = 0.0
    with gdrr.Projector(w, sampler=1) as a, gdrr.Projector(w, sampler=2) as b:
        for p in range(0, w.n_proj, 40):
            n = min(40, w.n_proj - p)
            sa, _, ta = a.project(proj_begin=p, proj_count=n, want_table=True)
            sb, _, tb = b.project(proj_begin=p, proj_count=n, want_table=True)
            assert torch.equal(ta, tb), f"ray tables differ in projections {p}..{p + n - 1}"
            rel = ((sa - sb).abs() / sa).max().item()
            worst = max(worst, rel)
            assert rel < 2e-5, f"projections {p}..{p + n - 1}: staged and gather differ by {rel:.2e}"
    print("C3 whole scan, staged vs gather: worst relative signal difference", worst)


def test_c4_subset_staged_equals_gather(gdrr, workloads_cache):
    w = workloads_cache("C4")
    with gdrr.Projector(w, sampler=1) as a, gdrr.Projector(w, sampler=2) as b:
        for p in range(0, w.n_proj, 41):
            sa, _, ta = a.project(proj_begin=p, proj_count=1, want_table=True)
            sb, _, tb = b.project(proj_begin=p, proj_count=1, want_table=True)
            assert torch.equal(ta, tb)
            assert ((sa - sb).abs() / sa).max().item() < 2e-5
