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


def check_line_integrals(li_gpu, li_ref, what=""):
    li_gpu = np.asarray(li_gpu, dtype=np.float64)
    li_ref = np.asarray(li_ref, dtype=np.float64)
    assert li_gpu.shape == li_ref.shape, (li_gpu.shape, li_ref.shape)
    scale = float(li_ref.max()) if li_ref.size else 0.0
    err = np.abs(li_gpu - li_ref)
    tol = LI_RTOL * np.abs(li_ref) + LI_FLOOR * scale
    bad = err > tol
    assert not bad.any(), (f"{what}: {int(bad.sum())} line integrals out of tolerance, worst "
                           f"|err| {float(err.max()):.3e} (scale {scale:.3e})")
    # rays that miss (or cross only empty voxels) must be exactly zero
    assert np.all(li_gpu[li_ref == 0.0] == 0.0), f"{what}: non-zero LI where the oracle has 0"
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
    worst_li, n_floor = check_line_integrals(li, oracle_out["line_integrals"], what)
    worst_sig = check_signal(sig, oracle_out["signal"], what)
    return dict(signal=worst_sig, li=worst_li, li_floor_pixels=n_floor)
