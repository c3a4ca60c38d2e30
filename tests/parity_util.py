"""Shared helpers of the GPU parity tests: tolerances (DESIGN.md 'Tolerances',
SURVEY.md Q14) and the element-by-element comparison of the CUDA path with the
CPU oracle on the same seeded inputs."""
import numpy as np

SIGNAL_RTOL = 1e-4          # BASELINE.json north_star: 1e-4 relative per pixel
LI_RTOL = 1e-4
LI_FLOOR = 1e-6             # x max(LI_ref): grazing rays, SURVEY.md Q14


def check_signal(sig_gpu, sig_ref, what=""):
    sig_gpu = np.asarray(sig_gpu, dtype=np.float64)
    sig_ref = np.asarray(sig_ref, dtype=np.float64)
    assert sig_gpu.shape == sig_ref.shape, (sig_gpu.shape, sig_ref.shape)
    assert np.all(np.isfinite(sig_gpu)), f"{what}: non-finite signal"
    rel = np.abs(sig_gpu - sig_ref) / np.abs(sig_ref)
    worst = float(rel.max()) if rel.size else 0.0
    assert worst <= SIGNAL_RTOL, f"{what}: max relative signal error {worst:.3e} > {SIGNAL_RTOL}"
    return worst


FACE_TIE = 2.0 ** -12       # DESIGN.md reading Q9: a sample this close to a cell face may fall in either cell


def oracle_midpoints(w, projection, i, j):
    """Index coordinates gi[n][3] of every midpoint sample of one ray, from the oracle's own ray record: sample k sits at
    the parameter (j0 + k + 1/2) step along the unit direction from the source, and gi = (x - centre) / d + (N - 1) / 2
    (oracle/gdrr_oracle.c index_coords).  Circular gantry or poses; tests/test_parity_util.py pins it to
    oracle.ray_samples."""
    import oracle
    if getattr(w, "poses", None) is not None:
        r = oracle.ray_pose(w, w.poses[projection], i, j)
    else:
        r = oracle.ray(w, float(w.phis[projection]), i, j)
    if not r["hit"] or r["n"] <= 0:
        return np.zeros((0, 3))
    t = (r["j0"] + np.arange(r["n"]) + 0.5) * float(w.step_mm)
    x = r["S"][None, :] + t[:, None] * r["dir"][None, :]
    d = np.asarray(w.spacing, dtype=np.float64)
    n = np.asarray(w.dims, dtype=np.float64)
    return (x - np.asarray(w.centre, dtype=np.float64)[None, :]) / d[None, :] + 0.5 * (n[None, :] - 1.0)


def face_tie_checker(w, projections):
    """near_face(index) for check_line_integrals on full images [P][M][nv][nu] of the workload `w` (P =
    len(projections), indices into w's projections): True iff the oracle's own fp64 positions of that ray have a
    sample within FACE_TIE of a cell face (reading Q9: the fp32 path may then take the neighbouring cell, whose other
    corners get a weight <= FACE_TIE)."""

    def near_face(index):
        p, _, j, i = (int(x) for x in index)
        gi = oracle_midpoints(w, int(projections[p]), i, j)
        if not len(gi):
            return False
        fr = gi - np.floor(gi)
        return bool(np.minimum(fr, 1.0 - fr).min() < FACE_TIE)
    return near_face


SLIVER_MM = 1e-3      # two lattice planes of different axes crossed within this length: their order is a tie (Q26)


def siddon_sliver_checker(w, projections, found=None):
    """near_face(index) for check_line_integrals on Siddon images [P][M][nv][nu] of the workload `w` (gantry or poses):
    True iff the ray of that pixel, in the oracle's own fp64 geometry, crosses two lattice planes of DIFFERENT axes
    within SLIVER_MM of path length at a lattice edge one of whose four voxels holds the entry's material with
    rho > 0.  The ray has a sliver of one of those voxels; fp32 can order the two crossings the other way round and
    then has a sliver of the diagonal neighbour instead (reading Q26: both are valid).  If that voxel is the ray's
    only piece of the material, its line integral is a non-zero sliver against an exact 0 (or the reverse), below the
    floor like every other error.  `found`: list that collects the entries asked about."""
    import oracle
    rho, mat = np.asarray(w.rho), np.asarray(w.mat)
    dims = [int(n) for n in w.dims]
    spacing = [float(d) for d in w.spacing]
    lo = [float(w.centre[a]) - 0.5 * dims[a] * spacing[a] for a in range(3)]

    def near_edge(index):
        p, m, j, i = (int(x) for x in index)
        if found is not None:
            found.append((int(projections[p]), m, j, i))
        if getattr(w, "poses", None) is not None:
            r = oracle.ray_pose(w, w.poses[projections[p]], i, j)
        else:
            r = oracle.ray(w, float(w.phis[projections[p]]), i, j)
        if not r["hit"]:
            return False
        S, d = r["S"], r["dir"]
        unit = float(np.linalg.norm(d))
        eps = SLIVER_MM / unit
        ts, ax = [], []
        for a in range(3):
            if d[a] == 0.0:
                continue
            t = (lo[a] + np.arange(dims[a] + 1) * spacing[a] - S[a]) / d[a]
            t = t[(t >= r["t_in"] - eps) & (t <= r["t_out"] + eps)]
            ts.append(t)
            ax.append(np.full(len(t), a))
        ts, ax = np.concatenate(ts), np.concatenate(ax)
        order = np.argsort(ts, kind="stable")
        ts, ax = ts[order], ax[order]
        ties = np.nonzero((np.diff(ts) * unit < SLIVER_MM) & (ax[1:] != ax[:-1]))[0]
        for k in ties:
            a, b = int(ax[k]), int(ax[k + 1])
            c = [(S[q] + 0.5 * (ts[k] + ts[k + 1]) * d[q] - lo[q]) / spacing[q] for q in range(3)]
            third = 3 - a - b
            for da in (-1, 0):
                for db in (-1, 0):
                    v = [0, 0, 0]
                    v[a], v[b], v[third] = int(round(c[a])) + da, int(round(c[b])) + db, int(np.floor(c[third]))
                    if all(0 <= v[q] < dims[q] for q in range(3)) \
                            and int(mat[v[2], v[1], v[0]]) == m and float(rho[v[2], v[1], v[0]]) > 0.0:
                        return True
        return False
    return near_edge


def check_line_integrals(li_gpu, li_ref, what="", near_face=None):
    li_gpu = np.asarray(li_gpu, dtype=np.float64)
    li_ref = np.asarray(li_ref, dtype=np.float64)
    assert li_gpu.shape == li_ref.shape, (li_gpu.shape, li_ref.shape)
    scale = float(li_ref.max()) if li_ref.size else 0.0
    err = np.abs(li_gpu - li_ref)
    tol = LI_RTOL * np.abs(li_ref) + LI_FLOOR * scale
    bad = err > tol
    assert not bad.any(), (f"{what}: {int(bad.sum())} line integrals out of tolerance, worst "
                           f"|err| {float(err.max()):.3e} (scale {scale:.3e})")
    # A material the ray never touches (or a ray that misses) must give exactly zero.  The one exception is the tie of
    # reading Q9: a midpoint within 2^-12 of a cell face may be sampled in the neighbouring cell, which brings in that
    # cell's far corners with a weight <= 2^-12; such an entry must be that ray (near_face says so from the oracle's
    # own positions) and stay below the floor like every other entry.
    zero_bad = np.argwhere((li_ref == 0.0) & (li_gpu != 0.0))
    if len(zero_bad):
        assert near_face is not None and len(zero_bad) <= 1000, \
            f"{what}: {len(zero_bad)} non-zero LI where the oracle has 0"
        for index in zero_bad:
            assert near_face(index), (f"{what}: non-zero LI {li_gpu[tuple(index)]:.3e} at {tuple(index)} where the "
                                      "oracle has 0, and no sample of that ray is within 2^-12 of a cell face")
    needed_floor = int(np.count_nonzero(err > LI_RTOL * np.abs(li_ref)))
    rel = float((err / np.maximum(np.abs(li_ref), 1e-300))[li_ref > 1e-3 * scale].max()) if scale else 0.0
    return rel, needed_floor


def check_ray_table(tab_gpu, tab_ref, what=""):
    tab_gpu = np.asarray(tab_gpu)
    tab_ref = np.asarray(tab_ref)
    assert tab_gpu.shape == tab_ref.shape, (tab_gpu.shape, tab_ref.shape)
    diff = np.count_nonzero(tab_gpu != tab_ref)
    assert diff == 0, f"{what}: {diff} integer ray-table entries differ (must be bit-exact)"


def compare_full(projector, w, oracle_out, what=""):
    """Full-image comparison of every output of gdrr_project with oracle.project(w)."""
    sig, li, tab = projector.project(want_li=True, want_table=True)
    sig, li, tab = sig.cpu().numpy(), li.cpu().numpy(), tab.cpu().numpy()
    check_ray_table(tab, oracle_out["ray_table"], what)
    near_face = face_tie_checker(w, list(range(w.n_proj)))
    worst_li, n_floor = check_line_integrals(li, oracle_out["line_integrals"], what, near_face)
    worst_sig = check_signal(sig, oracle_out["signal"], what)
    return dict(signal=worst_sig, li=worst_li, li_floor_pixels=n_floor)
