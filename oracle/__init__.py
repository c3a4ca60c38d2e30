"""ctypes loader for the CPU oracle (oracle/gdrr_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports
``paper_1204_6367_b200`` and shares no code with it.  This file only builds
and marshals; every number comes from gdrr_oracle.c.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gdrr_oracle.c")
_LIB = os.path.join(_HERE, "libgdrr_oracle.so")
_lib = None

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_float_p = ctypes.POINTER(ctypes.c_float)
_c_u8_p = ctypes.POINTER(ctypes.c_uint8)
_c_i32_p = ctypes.POINTER(ctypes.c_int32)


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99, fp64, no FMA contraction)."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-Wall", "-ffp-contract=off", "-fopenmp",
           "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        for name in ("gdrr_oracle_ray", "gdrr_oracle_trilinear", "gdrr_oracle_ray_samples",
                     "gdrr_oracle_project", "gdrr_oracle_project_siddon", "gdrr_oracle_project_literal",
                     "gdrr_oracle_project_poses", "gdrr_oracle_ray_pose", "gdrr_oracle_denoise",
                     "gdrr_oracle_project_general"):
            getattr(_lib, name).restype = ctypes.c_int
    return _lib


def _dp(a):
    return None if a is None else a.ctypes.data_as(_c_double_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _geom_args(w, step=None):
    nx, ny, nz = w.dims
    centre = _f64(w.centre)
    return centre, [
        ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz),
        ctypes.c_double(w.spacing[0]), ctypes.c_double(w.spacing[1]),
        ctypes.c_double(w.spacing[2]), _dp(centre)]


def _det_args(w, step=None):
    return [ctypes.c_double(w.sad), ctypes.c_double(w.sdd), ctypes.c_double(w.theta),
            ctypes.c_int(w.nu), ctypes.c_int(w.nv), ctypes.c_double(w.du),
            ctypes.c_double(w.dv), ctypes.c_double(w.u_off), ctypes.c_double(w.v_off)]


def ray(w, phi, i, j, step=None):
    """Geometry of one ray: dict(S, dir, L, t_in, t_out, j0, n, hit)."""
    lib = _load()
    centre, ga = _geom_args(w)
    out = np.zeros(9)
    tab = np.zeros(3, dtype=np.int32)
    rc = lib.gdrr_oracle_ray(*ga, *_det_args(w),
                             ctypes.c_double(w.step_mm if step is None else step),
                             ctypes.c_double(phi), ctypes.c_int(i), ctypes.c_int(j),
                             _dp(out), tab.ctypes.data_as(_c_i32_p))
    if rc:
        raise ValueError("gdrr_oracle_ray: invalid arguments")
    return dict(S=out[0:3].copy(), dir=out[3:6].copy(), L=out[6], t_in=out[7],
                t_out=out[8], j0=int(tab[0]), n=int(tab[1]), hit=bool(tab[2]))


def ray_pose(w, pose, i, j, step=None):
    """Geometry of one ray of a general pose (12 doubles: S, P, u_hat, v_hat); dict as ray()."""
    lib = _load()
    centre, ga = _geom_args(w)
    pose = _f64(pose).reshape(12)
    out = np.zeros(9)
    tab = np.zeros(3, dtype=np.int32)
    rc = lib.gdrr_oracle_ray_pose(*ga, ctypes.c_int(w.nu), ctypes.c_int(w.nv), ctypes.c_double(w.du),
                                  ctypes.c_double(w.dv), ctypes.c_double(w.u_off), ctypes.c_double(w.v_off),
                                  ctypes.c_double(w.step_mm if step is None else step), _dp(pose),
                                  ctypes.c_int(i), ctypes.c_int(j), _dp(out), tab.ctypes.data_as(_c_i32_p))
    if rc:
        raise ValueError("gdrr_oracle_ray_pose: invalid arguments")
    return dict(S=out[0:3].copy(), dir=out[3:6].copy(), L=out[6], t_in=out[7],
                t_out=out[8], j0=int(tab[0]), n=int(tab[1]), hit=bool(tab[2]))


def trilinear(rho, gi):
    """Clamp-to-edge tri-linear interpolant of rho[nz][ny][nx] at index points gi[n][3]."""
    lib = _load()
    rho = np.ascontiguousarray(rho, dtype=np.float32)
    gi = np.ascontiguousarray(gi, dtype=np.float64).reshape(-1, 3)
    nz, ny, nx = rho.shape
    out = np.zeros(gi.shape[0])
    lib.gdrr_oracle_trilinear(rho.ctypes.data_as(_c_float_p), nx, ny, nz,
                              ctypes.c_int(gi.shape[0]), _dp(gi), _dp(out))
    return out


def ray_samples(w, phi, i, j, step=None):
    """(gi[n][3] float64, cell[n][3] int32) of every midpoint sample of one ray."""
    lib = _load()
    r = ray(w, phi, i, j, step)
    n = max(r["n"], 1)
    gi = np.zeros((n, 3))
    cell = np.zeros((n, 3), dtype=np.int32)
    centre, ga = _geom_args(w)
    rc = lib.gdrr_oracle_ray_samples(*ga, *_det_args(w),
                                     ctypes.c_double(w.step_mm if step is None else step),
                                     ctypes.c_double(phi), ctypes.c_int(i), ctypes.c_int(j),
                                     ctypes.c_int(n), _dp(gi), cell.ctypes.data_as(_c_i32_p))
    if rc < 0:
        raise ValueError("gdrr_oracle_ray_samples: invalid arguments")
    return gi[:r["n"]], cell[:r["n"]]


def _project_common(w, step):
    rho = np.ascontiguousarray(w.rho, dtype=np.float32)
    mat = np.ascontiguousarray(w.mat, dtype=np.uint8)
    phis = _f64(w.phis)
    phi_w, resp, mu_hat = _f64(w.phi_weight), _f64(w.response), _f64(w.mu_hat)
    flu = None if w.fluence_map is None else np.ascontiguousarray(w.fluence_map, dtype=np.float32)
    bt_mu, bt_t = _f64(w.bowtie_mu), _f64(w.bowtie_thickness)
    centre, ga = _geom_args(w)
    keep = (rho, mat, phis, phi_w, resp, mu_hat, flu, bt_mu, bt_t, centre)
    args = ([rho.ctypes.data_as(_c_float_p), mat.ctypes.data_as(_c_u8_p)] + ga
            + [ctypes.c_int(w.n_materials)] + _det_args(w)
            + [ctypes.c_int(phis.shape[0]), _dp(phis),
               ctypes.c_double(w.step_mm if step is None else step),
               ctypes.c_int(phi_w.shape[0]), _dp(phi_w), _dp(resp), _dp(mu_hat),
               None if flu is None else flu.ctypes.data_as(_c_float_p),
               _dp(bt_mu), _dp(bt_t)])
    return keep, args


def project(w, pixels=None, step=None, want_li=True, want_table=True, n_threads=0, method="trilinear"):
    """Run the oracle on workload-like ``w``.  method: "trilinear" (the paper's default
    midpoint rule) or "siddon" (exact radiological path through homogeneous voxels; the
    result then also holds ``n_segments``).

    pixels: None (every pixel of every projection) or int array [n][3] of
    (projection, column i, row j).  Returns dict(signal, line_integrals,
    ray_table) with shapes [n_proj][nv][nu], [n_proj][M][nv][nu],
    [n_proj][nv][nu][2]  (or [n], [n][M], [n][2] for listed pixels).
    """
    lib = _load()
    poses = getattr(w, "poses", None)
    if getattr(w, "response_gain", None) is not None:
        return _project_general(lib, w, pixels, step, want_li, want_table, n_threads, method)
    if poses is not None:
        return _project_poses(lib, w, _f64(poses).reshape(-1, 12), pixels, step, want_li, want_table,
                              n_threads, method)
    keep, args = _project_common(w, step)
    M, n_proj = w.n_materials, len(w.phis)
    if pixels is None:
        n_pix, pix = 0, None
        signal = np.zeros((n_proj, w.nv, w.nu))
        li = np.zeros((n_proj, M, w.nv, w.nu)) if want_li else None
        tab = np.zeros((n_proj, w.nv, w.nu, 2), dtype=np.int32) if want_table else None
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 3)
        n_pix = pix.shape[0]
        signal = np.zeros(n_pix)
        li = np.zeros((n_pix, M)) if want_li else None
        tab = np.zeros((n_pix, 2), dtype=np.int32) if want_table else None
    common = (*args, ctypes.c_int64(n_pix),
              None if pix is None else pix.ctypes.data_as(_c_i32_p),
              _dp(signal), _dp(li), None if tab is None else tab.ctypes.data_as(_c_i32_p))
    if method == "siddon":
        nseg = np.zeros(signal.shape, dtype=np.int32)
        rc = lib.gdrr_oracle_project_siddon(*common, nseg.ctypes.data_as(_c_i32_p), ctypes.c_int(n_threads))
        out = dict(signal=signal, line_integrals=li, ray_table=tab, n_segments=nseg)
    elif method == "trilinear":
        rc = lib.gdrr_oracle_project(*common, ctypes.c_int(n_threads))
        out = dict(signal=signal, line_integrals=li, ray_table=tab)
    else:
        raise ValueError(f"unknown method {method!r}")
    if rc:
        raise ValueError("gdrr_oracle_project: invalid arguments")
    return out


def _project_general(lib, w, pixels, step, want_li, want_table, n_threads, method):
    """project() with a pixel-dependent detector response w.response_gain [n_energy][nv][nu] (reading Q32), on the
    circular gantry or on w.poses: same outputs."""
    if method not in ("trilinear", "siddon"):
        raise ValueError(f"unknown method {method!r}")
    rho = np.ascontiguousarray(w.rho, dtype=np.float32)
    mat = np.ascontiguousarray(w.mat, dtype=np.uint8)
    phi_w, resp, mu_hat = _f64(w.phi_weight), _f64(w.response), _f64(w.mu_hat)
    flu = None if w.fluence_map is None else np.ascontiguousarray(w.fluence_map, dtype=np.float32)
    bt_mu, bt_t = _f64(w.bowtie_mu), _f64(w.bowtie_thickness)
    gain = np.ascontiguousarray(w.response_gain, dtype=np.float32)
    if gain.shape != (phi_w.shape[0], w.nv, w.nu):
        raise ValueError("response_gain must be [n_energy][nv][nu]")
    poses = None if getattr(w, "poses", None) is None else _f64(w.poses).reshape(-1, 12)
    phis = None if poses is not None else _f64(w.phis)
    centre, ga = _geom_args(w)
    M, n_proj = w.n_materials, (poses.shape[0] if poses is not None else phis.shape[0])
    if pixels is None:
        n_pix, pix = 0, None
        signal = np.zeros((n_proj, w.nv, w.nu))
        li = np.zeros((n_proj, M, w.nv, w.nu)) if want_li else None
        tab = np.zeros((n_proj, w.nv, w.nu, 2), dtype=np.int32) if want_table else None
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 3)
        n_pix = pix.shape[0]
        signal = np.zeros(n_pix)
        li = np.zeros((n_pix, M)) if want_li else None
        tab = np.zeros((n_pix, 2), dtype=np.int32) if want_table else None
    nseg = np.zeros(signal.shape, dtype=np.int32)
    rc = lib.gdrr_oracle_project_general(
        ctypes.c_int(1 if method == "siddon" else 0),
        rho.ctypes.data_as(_c_float_p), mat.ctypes.data_as(_c_u8_p), *ga, ctypes.c_int(M), *_det_args(w),
        ctypes.c_int(n_proj), _dp(phis), _dp(poses), ctypes.c_double(w.step_mm if step is None else step),
        ctypes.c_int(phi_w.shape[0]), _dp(phi_w), _dp(resp), _dp(mu_hat),
        None if flu is None else flu.ctypes.data_as(_c_float_p), _dp(bt_mu), _dp(bt_t),
        gain.ctypes.data_as(_c_float_p),
        ctypes.c_int64(n_pix), None if pix is None else pix.ctypes.data_as(_c_i32_p),
        _dp(signal), _dp(li), None if tab is None else tab.ctypes.data_as(_c_i32_p),
        nseg.ctypes.data_as(_c_i32_p), ctypes.c_int(n_threads))
    if rc:
        raise ValueError("gdrr_oracle_project_general: invalid arguments")
    out = dict(signal=signal, line_integrals=li, ray_table=tab)
    if method == "siddon":
        out["n_segments"] = nseg
    return out


def _project_poses(lib, w, poses, pixels, step, want_li, want_table, n_threads, method):
    """project() on a general source path (w.poses): same outputs."""
    if method not in ("trilinear", "siddon"):
        raise ValueError(f"unknown method {method!r}")
    rho = np.ascontiguousarray(w.rho, dtype=np.float32)
    mat = np.ascontiguousarray(w.mat, dtype=np.uint8)
    phi_w, resp, mu_hat = _f64(w.phi_weight), _f64(w.response), _f64(w.mu_hat)
    flu = None if w.fluence_map is None else np.ascontiguousarray(w.fluence_map, dtype=np.float32)
    bt_mu, bt_t = _f64(w.bowtie_mu), _f64(w.bowtie_thickness)
    centre, ga = _geom_args(w)
    M, n_proj = w.n_materials, poses.shape[0]
    if pixels is None:
        n_pix, pix = 0, None
        signal = np.zeros((n_proj, w.nv, w.nu))
        li = np.zeros((n_proj, M, w.nv, w.nu)) if want_li else None
        tab = np.zeros((n_proj, w.nv, w.nu, 2), dtype=np.int32) if want_table else None
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 3)
        n_pix = pix.shape[0]
        signal = np.zeros(n_pix)
        li = np.zeros((n_pix, M)) if want_li else None
        tab = np.zeros((n_pix, 2), dtype=np.int32) if want_table else None
    nseg = np.zeros(signal.shape, dtype=np.int32)
    rc = lib.gdrr_oracle_project_poses(
        ctypes.c_int(1 if method == "siddon" else 0),
        rho.ctypes.data_as(_c_float_p), mat.ctypes.data_as(_c_u8_p), *ga, ctypes.c_int(M),
        ctypes.c_int(w.nu), ctypes.c_int(w.nv), ctypes.c_double(w.du), ctypes.c_double(w.dv),
        ctypes.c_double(w.u_off), ctypes.c_double(w.v_off), ctypes.c_int(n_proj), _dp(poses),
        ctypes.c_double(w.step_mm if step is None else step),
        ctypes.c_int(phi_w.shape[0]), _dp(phi_w), _dp(resp), _dp(mu_hat),
        None if flu is None else flu.ctypes.data_as(_c_float_p), _dp(bt_mu), _dp(bt_t),
        ctypes.c_int64(n_pix), None if pix is None else pix.ctypes.data_as(_c_i32_p),
        _dp(signal), _dp(li), None if tab is None else tab.ctypes.data_as(_c_i32_p),
        nseg.ctypes.data_as(_c_i32_p), ctypes.c_int(n_threads))
    if rc:
        raise ValueError("gdrr_oracle_project_poses: invalid arguments")
    out = dict(signal=signal, line_integrals=li, ray_table=tab)
    if method == "siddon":
        out["n_segments"] = nseg
    return out


def project_literal(w, pixels, step=None, n_threads=0):
    """Paper-literal per-energy ray traces on listed pixels: dict(signal[n], tau[n][n_energy])."""
    lib = _load()
    keep, args = _project_common(w, step)
    pix = np.ascontiguousarray(pixels, dtype=np.int32).reshape(-1, 3)
    n_pix = pix.shape[0]
    signal = np.zeros(n_pix)
    tau = np.zeros((n_pix, len(w.phi_weight)))
    rc = lib.gdrr_oracle_project_literal(
        *args, ctypes.c_int64(n_pix), pix.ctypes.data_as(_c_i32_p),
        _dp(signal), _dp(tau), ctypes.c_int(n_threads))
    if rc:
        raise ValueError("gdrr_oracle_project_literal: invalid arguments")
    return dict(signal=signal, tau=tau)


def denoise(s_hat, beta, n_iter, omega=0.8, floor=1e-12, s0=None):
    """Relaxed Jacobi sweeps of the paper's Eq. (5) on one image [nv][nu]; fp64."""
    lib = _load()
    s_hat = np.ascontiguousarray(s_hat, dtype=np.float64)
    nv, nu = s_hat.shape
    s0a = None if s0 is None else np.ascontiguousarray(s0, dtype=np.float64)
    out, work = np.zeros_like(s_hat), np.zeros_like(s_hat)
    rc = lib.gdrr_oracle_denoise(_dp(s_hat), _dp(s0a), ctypes.c_int(nu), ctypes.c_int(nv), ctypes.c_double(beta),
                                 ctypes.c_double(omega), ctypes.c_int(n_iter), ctypes.c_double(floor), _dp(out), _dp(work))
    if rc:
        raise ValueError("gdrr_oracle_denoise: invalid arguments")
    return out


def n_threads_available() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1
