"""The N > 1 host logic on CPU: two gloo ranks shard a scan by projection
(no data-path collective; only the harness's barrier, MAX of
the elapsed time and SUM of the work counters).  No GPU, no CUDA library."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DIST = os.path.join(ROOT, "paper_1204_6367_b200", "dist.py")


def _load_dist():
    # dist.py is host logic only; load it without importing the package (which
    # would load the CUDA library)
    import importlib.util
    spec = importlib.util.spec_from_file_location("gdrr_dist", DIST)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def test_strided_shard_partitions_the_scan():
    gd = _load_dist()
    for n_total, world in ((360, 1), (720, 2), (1440, 4), (2880, 8), (11, 3)):
        seen = np.concatenate([gd.strided_shard(n_total, world, r) for r in range(world)])
        assert sorted(seen.tolist()) == list(range(n_total))
        sizes = [len(gd.strided_shard(n_total, world, r)) for r in range(world)]
        assert max(sizes) - min(sizes) <= 1
    phis = gd.scan_angles(360)
    assert phis[0] == 0.0 and np.isclose(phis[-1], 2 * np.pi * 359 / 360)
    assert len(np.unique(np.round(np.diff(phis), 12))) == 1


WORKER = textwrap.dedent("""
    import importlib.util, json, os, sys
    import numpy as np
    sys.path.insert(0, {root!r})
    spec = importlib.util.spec_from_file_location("gdrr_dist", {dist!r})
    gd = importlib.util.module_from_spec(spec); spec.loader.exec_module(gd)
    import oracle
    from workloads import make_workload
    rank, local_rank, world = gd.init_process_group("gloo")
    n_total = 6
    mine = gd.strided_shard(n_total, world, rank)
    w = make_workload("C0").with_phis(gd.scan_angles(n_total)[mine])
    out = oracle.project(w, want_li=False)
    gd.barrier()
    samples = gd.sum_over_ranks(int(out["ray_table"][..., 1].sum()))
    worst = gd.max_over_ranks(10.0 + rank)
    np.save(os.path.join({tmp!r}, f"sig_{{rank}}.npy"), out["signal"])
    if rank == 0:
        print(json.dumps(dict(samples=samples, worst=worst, world=world)))
""")


def test_two_gloo_ranks_shard_projections(tmp_path):
    """Each rank projects its own angles (here with the CPU oracle standing in
    for the GPU); the union equals the single-process scan; the reductions the
    bench uses give SUM of samples and MAX of time."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, dist=DIST, tmp=str(tmp_path)))
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (so, se) in zip(procs, outs):
        assert p.returncode == 0, se[-2000:]
    import json
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["world"] == 2 and line["worst"] == 11.0

    import oracle
    from workloads import make_workload
    gd = _load_dist()
    full = oracle.project(make_workload("C0").with_phis(gd.scan_angles(6)), want_li=False)
    assert line["samples"] == int(full["ray_table"][..., 1].sum())
    for rank in range(2):
        sig = np.load(tmp_path / f"sig_{rank}.npy")
        assert np.array_equal(sig, full["signal"][rank::2])
