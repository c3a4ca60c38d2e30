"""Benchmark of the gDRR primary-signal projector on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl reference]

One "step" is one pass of the whole hot path over one synthetic scan: volume
ingest (a0) from device-resident (rho, material), then ray setup, tri-linear
sampling, energy sum and store (a1-a7) for every projection of the workload.
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "trilinear_samples_per_s"
UNIT = "samples/s"
METHODS = {"trilinear": ("trilinear_samples_per_s", "samples/s"),
           "texture": ("texture_filtered_samples_per_s", "samples/s"),   # the paper's own design, reported separately
           "siddon": ("siddon_voxel_segments_per_s", "segments/s")}   # the paper's optional line integral
SM_COUNT = 148
L1_BYTES_PER_CLK = 128          # per SM, DESIGN.md "Roofline"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback (B200_PROFILING.md)")


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for row in self.rows:
            parts = [p.strip() for p in row.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "power_w_max": float(max(power)) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def source_digest(files=None):
    """sha256 over device sources of csrc/: the stamp that ties a record of profiles/ncu_constants.json to the kernel it
    was captured on.  `files`: the kernel's own translation unit, the headers it includes and the ingest that lays out
    the volume it reads (the record lists them); None = every file but the host-side gdrr_api.cu."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1204_6367_b200", "csrc")
    if files is None:
        files = [n for n in os.listdir(csrc) if n.endswith((".cu", ".cuh", ".h")) and n != "gdrr_api.cu"]
    for name in sorted(files):
        with open(os.path.join(csrc, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()


def ncu_constants(kernel, workload):
    """Figures that only an `ncu --set full` capture can give (DRAM bytes, L2->SM bytes, the busy fraction of the bound),
    from profiles/ncu_constants.json, written by hand from the committed capture summaries.  They are quoted only if the
    capture was taken on the CUDA sources of this run (source_digest); else every figure is None."""
    path = os.path.join(ROOT, "profiles", "ncu_constants.json")
    none = {"dram_bytes_per_projection": None, "l2_to_sm_bytes_per_sample": None, "bound": "not profiled",
            "bound_busy_frac": None, "capture": None, "matches_this_build": False}
    if not os.path.exists(path):
        return none
    with open(path) as f:
        table = json.load(f)
    rec = table.get("kernels", {}).get(kernel, {}).get(workload)
    if rec is None:
        return none
    rec = dict(rec)
    # (a record stamped with its own source list is valid while THOSE files are unchanged; older records carry the
    # digest of all device sources)
    if "sources" in rec:
        rec["matches_this_build"] = rec.get("source_sha256") == source_digest(rec["sources"])
    else:
        rec["matches_this_build"] = table.get("source_sha256") == source_digest()
    if not rec["matches_this_build"]:
        for k in ("dram_bytes_per_projection", "l2_to_sm_bytes_per_sample", "bound_busy_frac"):
            rec[k] = None
        rec["bound"] = rec.get("bound", "") + " (capture is of older sources: figures withheld)"
    return rec


def cone_voxels(w, p):
    """Voxels of the volume whose centre projects onto the detector at projection p: the least a projection must read."""
    nx, ny, nz = w.dims
    phi = float(w.phis[p])
    c, s = np.cos(phi), np.sin(phi)
    x = (np.arange(nx) - 0.5 * (nx - 1)) * w.spacing[0]
    y = (np.arange(ny) - 0.5 * (ny - 1)) * w.spacing[1]
    z = (np.arange(nz) - 0.5 * (nz - 1)) * w.spacing[2]
    X, Y = np.meshgrid(x, y, indexing="xy")                       # [ny][nx]
    depth = X * c + Y * s + w.sad                                  # along the central ray, from the source
    u = (-X * s + Y * c) * w.sdd / depth - w.u_off
    in_u = (np.abs(u) <= 0.5 * w.nu * w.du) & (depth > 0)
    zmax = (0.5 * w.nv * w.dv + abs(w.v_off)) * depth / w.sdd     # |z| that still hits the detector, per (x, y)
    per_column = (np.abs(z)[:, None, None] <= zmax[None]) & in_u[None]
    return int(per_column.sum())


def workload_config(w, name, world, n_total, launch_proj):
    nx, ny, nz = w.dims
    return {"workload": name, "volume": [nx, ny, nz], "voxel_mm": list(w.spacing),
            "materials": w.n_materials, "energy_bins": w.n_energy, "detector": [w.nu, w.nv],
            "pixel_mm": w.du, "step_mm": w.step_mm, "projections_per_gpu": w.n_proj,
            "projections_total": n_total, "projections_per_launch": launch_proj,
            "parallelism": f"projection-sharded x{world}, no collective",
            "l2": "volume in device layout exceeds L2 (no flush needed)" if
                  (nx + 2) * (ny + 2) * (nz + 2) * 4 * (1 if w.n_materials == 1 else 2 if w.n_materials == 2 else 4)
                  > 126e6 else "L2 flushed between steps"}


# ---------------------------------------------------------------------------
# the reference arm and the cpu_baseline leg: the oracle, as it stands
# ---------------------------------------------------------------------------

def oracle_sample(w, rows, projection):
    """Pixel list: `rows` evenly spaced detector rows of one projection."""
    jj = np.linspace(0, w.nv - 1, rows).round().astype(np.int32)
    ii = np.arange(w.nu, dtype=np.int32)
    J, I = np.meshgrid(jj, ii, indexing="ij")
    return np.stack([np.full(J.size, projection, dtype=np.int32), I.ravel(), J.ravel()], axis=1)


def time_oracle(w, pix):
    import oracle
    t0 = time.perf_counter()
    out = oracle.project(w, pixels=pix, want_li=False, method=time_oracle.method)
    dt = time.perf_counter() - t0
    time_oracle.last_signal = out["signal"]                 # for the parity figure printed beside the timing
    units = out["n_segments"].sum() if time_oracle.method == "siddon" else out["ray_table"][:, 1].sum()
    return int(units), dt, oracle.n_threads_available()


time_oracle.method = "trilinear"


def sized_oracle_sample(w, seconds):
    """A pixel list of the workload worth about `seconds` of oracle time on this
    host: probe the rate on 16 rows of one projection, then take whole
    projections evenly spaced over the scan (or fewer rows of one projection)."""
    p = min(37, w.n_proj - 1)
    probe_rows = max(1, min(w.nv, 16))
    time_oracle(w, oracle_sample(w, probe_rows, p))            # touch the volume once
    n, dt, _ = time_oracle(w, oracle_sample(w, probe_rows, p))
    per_proj = n * (w.nv / probe_rows)
    want = max(1.0, seconds * (n / dt))
    n_proj = int(min(w.n_proj, max(1, round(want / per_proj))))
    if want >= per_proj:
        projs = np.linspace(0, w.n_proj - 1, n_proj).round().astype(int)
        pix = np.concatenate([oracle_sample(w, w.nv, int(q)) for q in projs])
        return pix, f"all {w.nv} x {w.nu} pixels of {n_proj} projection(s) evenly spaced over the scan"
    rows = int(max(1, min(w.nv, round(w.nv * want / per_proj))))
    return oracle_sample(w, rows, p), f"{rows} evenly spaced detector rows x {w.nu} columns of projection {p}"


def run_reference(args):
    """--impl reference: the oracle as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from workloads import make_workload
    w = make_workload(args.workload, phantom=args.phantom)
    if args.tissue_classes != 4:
        from workloads import with_tissue_classes
        w = with_tissue_classes(w, args.tissue_classes)
    pix, sample = sized_oracle_sample(w, args.ref_seconds)
    for _ in range(args.warmup):
        time_oracle(w, pix[: max(1, len(pix) // 16)])
    total, elapsed, cores = 0, 0.0, 1
    for _ in range(args.steps):
        n, dt, cores = time_oracle(w, pix)
        total += n
        elapsed += dt
    value = total / elapsed
    per_proj = n * (w.nu * w.nv / len(pix))
    sample = f"{sample}, per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * elapsed / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic (seeded phantom; DESIGN.md 'Input recipe')",
            "config": workload_config(w, args.workload, 1, w.n_proj, 0),
            "projections_per_s": value / per_proj,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------

def run_b200(args):
    import torch
    import paper_1204_6367_b200 as g
    from paper_1204_6367_b200 import dist as gd
    from workloads import make_workload, pure_cell_fraction

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU path")
    rank, local_rank, world = gd.init_process_group("nccl")
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but WORLD_SIZE is {world}")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    peaks = measured_peaks()

    # the N-GPU job is one scan of n_proj * N evenly spaced angles, sharded by projection
    w0 = make_workload(args.workload, phantom=args.phantom)
    if args.tissue_classes != 4:                            # more than four materials: groups of four (include/gdrr.h)
        from workloads import with_tissue_classes
        w0 = with_tissue_classes(w0, args.tissue_classes)
    per_gpu = w0.n_proj if args.projections <= 0 else args.projections
    n_total = per_gpu * world
    mine = gd.strided_shard(n_total, world, rank)
    if args.angle_deg is None:
        w = w0.with_phis(gd.scan_angles(n_total)[mine])
    else:                                                   # profiling aid: every projection at one angle
        w = w0.with_phis(np.full(per_gpu, np.deg2rad(args.angle_deg)))
    if args.u_off_mm:                                       # half-fan scan (detector shifted along u)
        import copy
        w = copy.copy(w)
        w.u_off = float(args.u_off_mm)
    if args.trajectory != "circle":                         # other source paths, same kernels
        from workloads import trajectories
        nz_mm = w.dims[2] * w.spacing[2]
        w = w.with_poses(trajectories.helical_poses(w.sad, w.sdd, w.phis, pitch_mm=0.5 * nz_mm, z0_mm=-0.25 * nz_mm)
                         if args.trajectory == "helix" else
                         trajectories.c_arm_poses(w.sad, w.sdd, w.phis, np.deg2rad(args.tilt_deg)))
    launch_proj = per_gpu if args.launch_proj <= 0 else min(args.launch_proj, per_gpu)

    pr = g.Projector(w, device=local_rank, layout=args.layout,
                     method={"siddon": g.GDRR_METHOD_SIDDON, "texture": g.GDRR_METHOD_TEXTURE,
                             "trilinear": g.GDRR_METHOD_TRILINEAR}[args.method],
                     sampler={"auto": g.GDRR_SAMPLER_AUTO, "gather": g.GDRR_SAMPLER_GATHER,
                              "staged": g.GDRR_SAMPLER_STAGED}[args.sampler])
    signal = torch.empty((per_gpu, w.nv, w.nu), dtype=torch.float32, device=dev)
    # (more than four materials: the library needs the line-integral output, one launch_proj batch of it)
    li_buf = (torch.empty((min(per_gpu, launch_proj), w.n_materials, w.nv, w.nu), dtype=torch.float32, device=dev)
              if w.n_materials > 4 else None)
    stream = torch.cuda.current_stream()
    if args.method == "siddon":                            # units = voxel segments of positive length
        n_samples = sum(int(pr.siddon_segments(b, min(32, per_gpu - b)).sum().item()) for b in range(0, per_gpu, 32))
    else:
        n_samples = pr.count_samples()
    ingest_launches_before = pr.kernel_launches()

    vw = 1 if w.n_materials == 1 else 2 if w.n_materials == 2 else 4
    nx, ny, nz = w.dims
    vol_bytes = (nx + 2) * (ny + 2) * (nz + 2) * (16 if args.layout == 2 else 4 * vw)
    flush = (torch.empty(256 << 20, dtype=torch.uint8, device=dev) if vol_bytes <= 126e6 else None)

    def step(events=None):
        if flush is not None:                              # inputs fit in L2: evict them
            flush.zero_()
        if events is not None:
            events[2].record(stream)
        pr.ingest()                                        # a0
        if events is not None:
            events[0].record(stream)
        for b in range(0, per_gpu, launch_proj):            # a1-a7
            cnt = min(launch_proj, per_gpu - b)
            g.gdrr_project(pr.ctx, pr.vol, b, cnt, signal[b:b + cnt], None if li_buf is None else li_buf[:cnt])
        if events is not None:
            events[1].record(stream)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    kev = [tuple(torch.cuda.Event(enable_timing=True) for _ in range(3)) for _ in range(args.steps)]
    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = pr.kernel_launches()
    gd.barrier()
    torch.cuda.synchronize()
    t_begin.record(stream)
    for k in range(args.steps):
        step(kev[k])
    t_end.record(stream)
    torch.cuda.synchronize()
    gd.barrier()
    launches = pr.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else None
    bracket_ms = t_begin.elapsed_time(t_end)
    if flush is not None:                                   # leave the L2 flushes out of the step time
        bracket_ms = float(np.sum([c.elapsed_time(b) for a, b, c in kev]))
    elapsed_ms = gd.max_over_ranks(bracket_ms, dev)
    kernel_ms = float(np.mean([a.elapsed_time(b) for a, b, c in kev]))     # all project launches of a step
    total_samples = gd.sum_over_ranks(n_samples, dev)
    checksum = float(signal.double().sum().item())

    value = total_samples * args.steps / (elapsed_ms * 1e-3)
    proj_per_s = n_total * args.steps / (elapsed_ms * 1e-3)

    # ---- e2e: the same step through the host-buffer entry points ------------------
    e2e = None
    if not args.no_e2e:
        rho_h = torch.from_numpy(w.rho).pin_memory()
        mat_h = torch.from_numpy(w.mat).pin_memory()
        out_h = torch.empty((per_gpu, w.nv, w.nu), dtype=torch.float32).pin_memory()
        stage_proj = min(per_gpu, args.e2e_stage)      # the library double-buffers: two batches of stage_proj / 2
        stage = torch.empty((stage_proj, w.nv, w.nu), dtype=torch.float32, device=dev)

        def e2e_step():
            pr.ingest_host(rho_h, mat_h)
            g.gdrr_project_host(pr.ctx, pr.vol, 0, per_gpu, out_h, stage, stage_proj)

        e2e_step()
        torch.cuda.synchronize()
        gd.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        t0 = time.perf_counter()
        for _ in range(args.steps):
            e2e_step()
        e1.record(stream)
        torch.cuda.synchronize()
        wall_ms = (time.perf_counter() - t0) * 1e3
        gd.barrier()
        e2e_ms = gd.max_over_ranks(max(e0.elapsed_time(e1), wall_ms), dev)
        same = bool(torch.equal(out_h, signal.cpu()))
        e2e = {"value": total_samples * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
               "projections_per_s": n_total * args.steps / (e2e_ms * 1e-3),
               "ms_per_step": e2e_ms / args.steps,
               "h2d_bytes_per_step": int(rho_h.numel() * 4 + mat_h.numel()),
               "d2h_bytes_per_step": int(out_h.numel() * 4),
               "bit_identical_to_device_path": same,
               "api": "gdrr_create_volume_host + gdrr_project_host (pinned host buffers)"}

    if rank != 0:
        pr.close()
        return

    # ---- roofline of the dominant kernel (gdrr_project_kernel) ----------------------
    picked = {g.GDRR_SAMPLER_STAGED: "gdrr_project_staged_kernel", g.GDRR_SAMPLER_GATHER: "gdrr_project_packed_kernel"}
    kname = ("gdrr_project_siddon_kernel" if args.method == "siddon" else
             "gdrr_project_texture_kernel" if args.method == "texture" else
             "gdrr_project_kernel" if args.layout != 2 else
             picked[g.gdrr_last_sampler(pr.ctx)])          # what --sampler auto launched (gdrr_last_sampler)
    corner_bytes = 4 if args.layout == 2 else 4 * vw        # packed word, or one float per material
    per_unit = 1 if args.method == "siddon" else 8          # one voxel per segment, 8 corners per sample
    l1_bytes = per_unit * corner_bytes * n_samples
    l1_peak = SM_COUNT * L1_BYTES_PER_CLK * peaks["sm_max_mhz"] * 1e6 / 1e9       # GB/s
    l1_achieved = l1_bytes / (kernel_ms * 1e-3) / 1e9
    # what only ncu can see comes from the committed capture of these very sources, or is None (never a stale constant)
    ncu = ncu_constants(kname, args.workload if args.phantom == "smooth" and args.trajectory == "circle"
                        and not args.u_off_mm and w.n_materials <= 4 else "-")
    dram_step = ncu["dram_bytes_per_projection"] * per_gpu if ncu["dram_bytes_per_projection"] else None
    # the least a projection must move: every voxel of its cone once as a 4-byte word, and its image
    hbm_min = None
    if w.poses is None:
        probes = sorted({0, per_gpu // 8, per_gpu // 3})
        hbm_min = float(np.mean([cone_voxels(w, p) for p in probes])) * 4.0 * per_gpu + per_gpu * w.nu * w.nv * 4.0
    roofline = {"kernel": kname, "bound": "l1tex", "achieved": l1_achieved, "peak": l1_peak,
                "unit": "GB/s", "frac": l1_achieved / l1_peak,
                "traffic": dram_step / (-(-per_gpu // launch_proj)) if dram_step else None,
                "kernel_ms_per_step": kernel_ms, "launches_per_step": -(-per_gpu // launch_proj),
                "peak_def": f"{SM_COUNT} SMs x {L1_BYTES_PER_CLK} B/clk x {peaks['sm_max_mhz']:.0f} MHz (max SM clock)",
                "algorithmic": f"{per_unit} voxel value(s) x {corner_bytes} B = {per_unit * corner_bytes} B per "
                               f"{'segment' if args.method == 'siddon' else 'sample'} through L1",
                "samples_per_clk_per_sm": n_samples / (kernel_ms * 1e-3) / (SM_COUNT * peaks["sm_max_mhz"] * 1e6),
                "ncu_identified_bound": ncu["bound"], "ncu_bound_busy_frac": ncu["bound_busy_frac"],
                "ncu_capture": ncu["capture"], "ncu_capture_matches_this_build": ncu["matches_this_build"],
                "l2_to_sm_bytes_per_sample": ncu["l2_to_sm_bytes_per_sample"],
                # HBM: MEASURED dram bytes (the capture's per-projection figure x projections) over the live kernel time
                "hbm": {"achieved": dram_step / (kernel_ms * 1e-3) / 1e9 if dram_step else None,
                        "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "frac": dram_step / (kernel_ms * 1e-3) / 1e9 / peaks["hbm_gbs"] if dram_step else None,
                        "peak_source": peaks["source"],
                        "dram_bytes_per_step": dram_step, "algorithmic_min_bytes_per_step": hbm_min,
                        "traffic_vs_algorithmic": dram_step / hbm_min if dram_step and hbm_min else None,
                        "algorithmic": "4 B per voxel of the projection's cone, once, + 4 B per pixel"}}

    # ---- cpu_baseline: the oracle on a bounded sample of the same workload -----------
    cpu = None
    if not args.no_cpu_baseline:
        pix, sample = sized_oracle_sample(w, args.cpu_seconds)
        n, dt, cores = time_oracle(w, pix)
        ref = time_oracle.last_signal
        got = signal.cpu().numpy()[pix[:, 0], pix[:, 2], pix[:, 1]].astype(np.float64)
        pos = ref > 0.0                                     # (a zero oracle signal must be met exactly)
        cpu = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"{sample} ({n} samples)",
               "max_rel_err_of_b200_signal_on_sample": float(np.max(np.abs(got[pos] - ref[pos]) / ref[pos])) if pos.any() else 0.0,
               "zero_signal_pixels_met_exactly": bool(np.all(got[~pos] == 0.0))}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "method": args.method, "sampler": args.sampler, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic (seeded phantom; DESIGN.md 'Input recipe')",
            "config": dict(workload_config(w, args.workload, world, n_total, launch_proj),
                           phantom=args.phantom, pure_cell_fraction=pure_cell_fraction(w.mat), u_off_mm=w.u_off,
                           tissue_classes=w.n_materials,
                           inputs_sha256=w.sha256(),
                           **({} if args.trajectory == "circle" else {"trajectory": args.trajectory})),
            "projections_per_s": proj_per_s, "samples_per_step": total_samples,
            "paper_context": "paper: 1.2-2.3 s per poly-energetic projection on a GTX 580 (PAPER.md:366-367)",
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu, "checksum": checksum, "library": g.LIBRARY_PATH}
    print(json.dumps(line), flush=True)
    pr.close()


def run_denoise(args):
    """--method denoise: the scatter denoiser of PAPER.md:199-218 on a scan of synthetic
    Poisson images; a step = n_iter sweeps of Eq. (5) on every image."""
    import torch
    import paper_1204_6367_b200 as g
    from workloads import make_workload
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU path")
    w = make_workload(args.workload)
    n_img = w.n_proj if args.projections <= 0 else args.projections
    n_iter, beta = 100, 0.2
    peaks = measured_peaks()
    gen = torch.Generator(device="cuda").manual_seed(12046367)
    jj = torch.arange(w.nv, device="cuda")[:, None].float()
    ii = torch.arange(w.nu, device="cuda")[None, :].float()
    truth = 40.0 * (0.4 + torch.exp(-((ii - 0.4 * w.nu) ** 2 / (0.1 * w.nu ** 2) + (jj - 0.6 * w.nv) ** 2 / (0.2 * w.nv ** 2))))
    s_hat = torch.poisson(truth.expand(n_img, -1, -1).contiguous(), generator=gen) + 1.0
    out, scratch = torch.empty_like(s_hat), torch.empty_like(s_hat)
    ctx = g.gdrr_create_context(0)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        g.gdrr_denoise_scatter(ctx, s_hat, out, scratch, beta, n_iter)
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    sampler.start()
    l0 = g.gdrr_kernel_launches(ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        g.gdrr_denoise_scatter(ctx, s_hat, out, scratch, beta, n_iter)
    e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = g.gdrr_kernel_launches(ctx) - l0
    units = n_img * w.nu * w.nv * n_iter
    value = units * args.steps / (ms * 1e-3)
    # e2e: host images in, denoised images out
    hin, hout = s_hat.cpu().pin_memory(), torch.empty(s_hat.shape).pin_memory()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        s_hat.copy_(hin, non_blocking=True)
        g.gdrr_denoise_scatter(ctx, s_hat, out, scratch, beta, n_iter)
        hout.copy_(out, non_blocking=True)
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    import oracle
    img = s_hat[0].cpu().numpy()
    t0 = time.perf_counter()
    ref = oracle.denoise(img, beta=beta, n_iter=n_iter)
    dt = time.perf_counter() - t0
    err = float(np.max(np.abs(out[0].cpu().numpy() - ref) / ref))
    bytes_per_unit = 12.0 / 4                                  # S and S_hat in, S out, once per 4 fused sweeps
    achieved = bytes_per_unit * units * args.steps / (ms * 1e-3) / 1e9
    line = {"metric": "denoise_pixel_sweeps_per_s", "value": value, "unit": "pixel-sweeps/s", "method": "denoise",
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic (seeded Poisson images of a smooth scatter-like field)",
            "config": {"workload": f"{args.workload} detector, scatter denoiser (PAPER.md:199-218)", "detector": [w.nu, w.nv],
                       "images": n_img, "sweeps": n_iter, "beta": beta, "omega": 0.8,
                       "l2": "three image stacks exceed L2 (no flush needed)" if 3 * s_hat.numel() * 4 > 126e6 else "fits L2"},
            "images_per_s": n_img * args.steps / (ms * 1e-3),
            "paper_context": "paper: 0.041 s per projection for denoising + noise calibration on a GTX 580 (PAPER.md:366)",
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": units * args.steps / (e2e_ms * 1e-3), "unit": "pixel-sweeps/s",
                    "h2d_bytes_per_step": int(hin.numel() * 4), "d2h_bytes_per_step": int(hout.numel() * 4)},
            "roofline": {"kernel": "gdrr_denoise_kernel", "bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"],
                         "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"], "traffic": None,
                         "algorithmic": "12 B per pixel per launch of 4 fused sweeps = 3 B per pixel-sweep",
                         "peak_source": peaks["source"]},
            "cpu_baseline": {"value": img.size * n_iter / dt, "unit": "pixel-sweeps/s", "cores": 1, "kind": "oracle",
                             "sample": "one image", "max_rel_err_of_b200_on_sample": err}}
    print(json.dumps(line), flush=True)
    g.gdrr_destroy_context(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="C3", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--projections", type=int, default=0, help="projections per GPU (0 = the workload's)")
    ap.add_argument("--launch-proj", type=int, default=0, help="projections per kernel launch (0 = all)")
    ap.add_argument("--e2e-stage", type=int, default=64, help="projections in the e2e arm's device staging buffer")
    ap.add_argument("--method", default="trilinear", choices=sorted(METHODS) + ["denoise"],
                    help="line integral: the paper's default tri-linear midpoint rule, or its Siddon option")
    ap.add_argument("--sampler", default="auto", choices=["auto", "gather", "staged"],
                    help="packed-quad sampling kernel: quads staged through shared memory by TMA (auto), or gathered through L1")
    ap.add_argument("--angle-deg", type=float, default=None,
                    help="profiling aid: all projections at this one gantry angle instead of an evenly spaced scan")
    ap.add_argument("--trajectory", default="circle", choices=["circle", "helix", "c_arm"],
                    help="source path: the paper's circle (the headline), a one-turn helix over half the volume's "
                         "height, or the circle tilted about x by --tilt-deg (gdrr_set_geometry_poses)")
    ap.add_argument("--tilt-deg", type=float, default=20.0)
    ap.add_argument("--u-off-mm", type=float, default=0.0,
                    help="detector offset along u (half-fan scan: e.g. 148 on C3, where the far rays cross a corner of the volume)")
    ap.add_argument("--phantom", default="smooth", choices=["smooth", "noisy1", "noisy3", "random"],
                    help="C2..C4: the BASELINE recipe (smooth), the same with 1 % / 3 % voxel noise before the material "
                         "thresholds, or materials drawn per voxel (workloads/configs.py); the pure-cell fraction is printed")
    ap.add_argument("--tissue-classes", type=int, default=4, choices=[4, 5, 6, 7, 8],
                    help="C2..C4 segmented into this many materials (workloads.with_tissue_classes); beyond four the library "
                         "samples one group of four materials per pass")
    ap.add_argument("--layout", type=int, default=2, help="0 brick (exact), 1 linear (exact), 2 packed quad")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the cpu_baseline sample")
    ap.add_argument("--ref-seconds", type=float, default=8.0, help="target oracle time per step of --impl reference")
    args = ap.parse_args()
    global METRIC, UNIT
    if args.method == "denoise":
        if args.impl == "reference" or args.gpus != 1:
            raise SystemExit("--method denoise is a single-GPU measurement of the b200 arm")
        return run_denoise(args)
    METRIC, UNIT = METHODS[args.method]
    time_oracle.method = "siddon" if args.method == "siddon" else "trilinear"
    if args.method == "texture":
        args.layout = 1                                     # the texture is built from the LINEAR layout
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
