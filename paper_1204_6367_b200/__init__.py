"""Python binding of libgdrr_b200.so, the C-ABI library declared in include/gdrr.h.

Argument marshalling only: every step of the projector (volume ingest, ray
setup, tri-linear sampling, energy sum) runs in the library's hand-written
sm_100a CUDA kernels.  PyTorch is used for device memory and streams.  There
is no CPU path and no other backend: if the library cannot be loaded this
module raises, it never falls back.  It never imports ``oracle``.

Functions carry the names of the C entry points and take torch CUDA tensors
(``*_dev`` arguments), numpy arrays (host tables) and plain numbers.
``Projector`` is a small convenience holder that keeps the tensors a volume
handle refers to alive.
"""
import ctypes
import os

import numpy as np

from . import build as _build

GDRR_OK = 0
GDRR_ERR_INVALID_ARG = -1
GDRR_ERR_NOT_READY = -2
GDRR_ERR_CUDA = -3
GDRR_ERR_WORKSPACE = -4
GDRR_ERR_UNSUPPORTED = -5
GDRR_LAYOUT_BRICK = 0
GDRR_LAYOUT_LINEAR = 1
GDRR_LAYOUT_PACKED_QUAD = 2
GDRR_SAMPLER_AUTO = 0
GDRR_SAMPLER_GATHER = 1
GDRR_SAMPLER_STAGED = 2
GDRR_METHOD_TRILINEAR = 0
GDRR_METHOD_SIDDON = 1
GDRR_METHOD_TEXTURE = 2
GDRR_MAX_MATERIALS = 16
GDRR_MAX_ENERGIES = 512
GDRR_DENOISE_STATIC_MAX_FLOATS = 4194304

EXPORTS = (
    "gdrr_create_context", "gdrr_destroy_context", "gdrr_last_error",
    "gdrr_volume_workspace_bytes", "gdrr_create_volume", "gdrr_create_volume_host",
    "gdrr_destroy_volume", "gdrr_set_geometry", "gdrr_set_spectrum", "gdrr_project",
    "gdrr_project_host", "gdrr_ray_setup", "gdrr_kernel_launches", "gdrr_version",
    "gdrr_set_method", "gdrr_siddon_segments", "gdrr_set_sampler", "gdrr_volume_attach_texture", "gdrr_denoise_scatter",
    "gdrr_denoise_scatter_static",
    "gdrr_set_geometry_poses", "gdrr_last_sampler", "gdrr_debug_set_skew", "gdrr_debug_ray_cells",
    "gdrr_set_response_gain", "gdrr_volume_status",
)


class GdrrError(RuntimeError):
    def __init__(self, code, message):
        super().__init__(f"gdrr error {code}: {message}")
        self.code = code


def _load():
    path = _build.LIB
    if not os.path.exists(path):
        # a source checkout on a machine with nvcc: build in-tree, else fail loudly
        path = _build.build()
    lib = ctypes.CDLL(path)
    vp, i, d, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    pp = ctypes.POINTER(ctypes.c_void_p)
    sig = {
        "gdrr_create_context": (i, [i, pp]),
        "gdrr_destroy_context": (i, [vp]),
        "gdrr_last_error": (ctypes.c_char_p, [vp]),
        "gdrr_volume_workspace_bytes": (i, [i, i, i, i, i, ctypes.POINTER(sz)]),
        "gdrr_create_volume": (i, [vp, vp, vp, i, i, i, d, d, d, vp, i, i, vp, sz, vp, pp]),
        "gdrr_create_volume_host": (i, [vp, vp, vp, i, i, i, d, d, d, vp, i, i, vp, vp, vp, sz, vp, pp]),
        "gdrr_destroy_volume": (i, [vp]),
        "gdrr_volume_status": (i, [vp, vp]),
        "gdrr_set_geometry": (i, [vp, d, d, d, i, i, d, d, d, d, i, vp, d]),
        "gdrr_set_geometry_poses": (i, [vp, i, i, d, d, d, d, i, vp, d]),
        "gdrr_set_spectrum": (i, [vp, i, i, vp, vp, vp, vp, vp, vp]),
        "gdrr_project": (i, [vp, vp, i, i, vp, vp, vp, vp]),
        "gdrr_project_host": (i, [vp, vp, i, i, vp, vp, i, vp]),
        "gdrr_ray_setup": (i, [vp, vp, i, i, vp, vp, vp]),
        "gdrr_set_method": (i, [vp, i]),
        "gdrr_set_sampler": (i, [vp, i]),
        "gdrr_volume_attach_texture": (i, [vp, vp, vp]),
        "gdrr_denoise_scatter": (i, [vp, vp, vp, vp, i, i, i, d, d, i, d, vp]),
        "gdrr_denoise_scatter_static": (i, [vp, vp, vp, i, i, i, d, d, i, d, vp]),
        "gdrr_siddon_segments": (i, [vp, vp, i, i, vp, vp]),
        "gdrr_set_response_gain": (i, [vp, vp]),
        "gdrr_last_sampler": (i, [vp]),
        "gdrr_debug_set_skew": (i, [vp, i]),
        "gdrr_debug_ray_cells": (i, [vp, vp, i, i, i, i, vp, i, vp, vp]),
        "gdrr_kernel_launches": (ctypes.c_ulonglong, [vp]),
        "gdrr_version": (ctypes.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        try:
            fn = getattr(lib, name)
        except AttributeError as e:
            raise ImportError(f"{path} does not export {name}: it is older than include/gdrr.h; rebuild it with "
                              "`python paper_1204_6367_b200/build.py --force`") from e
        fn.restype = res
        fn.argtypes = args
    return lib


_lib = _load()
LIBRARY_PATH = _build.LIB


def _check(rc, ctx=None):
    if rc != GDRR_OK:
        msg = _lib.gdrr_last_error(ctx)
        raise GdrrError(rc, msg.decode() if msg else "")


def _host(a, dtype):
    """Contiguous host array of `dtype` (or None) and its address."""
    if a is None:
        return None, None
    arr = np.ascontiguousarray(a, dtype=dtype)
    return arr, arr.ctypes.data


def _dev(t, dtype_name, min_numel=0, what="tensor"):
    """Address of a contiguous CUDA tensor (or None)."""
    if t is None:
        return None
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{what} must be a CUDA tensor")
    if str(t.dtype) != "torch." + dtype_name:
        raise TypeError(f"{what} must have dtype {dtype_name}, got {t.dtype}")
    if not t.is_contiguous():
        raise ValueError(f"{what} must be contiguous")
    if t.numel() < min_numel:
        raise ValueError(f"{what} has {t.numel()} elements, {min_numel} needed")
    return t.data_ptr()


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


# ---------------------------------------------------------------------------
# the C entry points, same names
# ---------------------------------------------------------------------------

def gdrr_version():
    return _lib.gdrr_version().decode()


class _Context(ctypes.c_void_p):
    """The gdrr_context* handle.  The C ABI cannot see the sizes of the caller's device buffers, so the binding
    remembers the detector shape and the material count it passed in and checks every output tensor against them."""
    nu = nv = n_mat = None


def _plane(ctx, proj_count, per_pixel=1, what="gdrr_set_geometry"):
    """Elements an output of `proj_count` projections needs (0 if the shape is not known on this side)."""
    if not isinstance(ctx, _Context) or ctx.nu is None:
        return 0
    return int(proj_count) * ctx.nu * ctx.nv * per_pixel


def gdrr_create_context(cuda_device=0):
    out = _Context()
    _check(_lib.gdrr_create_context(int(cuda_device), ctypes.byref(out)))
    return out


def gdrr_destroy_context(ctx):
    _check(_lib.gdrr_destroy_context(ctx))


def gdrr_last_error(ctx=None):
    msg = _lib.gdrr_last_error(ctx)
    return msg.decode() if msg else ""


def gdrr_volume_workspace_bytes(nx, ny, nz, n_materials, layout=GDRR_LAYOUT_PACKED_QUAD):
    out = ctypes.c_size_t()
    _check(_lib.gdrr_volume_workspace_bytes(nx, ny, nz, n_materials, layout, ctypes.byref(out)))
    return out.value


def gdrr_create_volume(ctx, rho_dev, material_dev, dims, spacing_mm, centre_mm, n_materials,
                       layout, workspace_dev, stream=None):
    """dims = (nx, ny, nz); rho_dev float32 / material_dev uint8 CUDA tensors of
    shape [nz][ny][nx]; workspace_dev a uint8 CUDA tensor of at least
    gdrr_volume_workspace_bytes.  Returns the volume handle."""
    nx, ny, nz = (int(x) for x in dims)
    nvox = nx * ny * nz
    centre, centre_p = _host(centre_mm, np.float64)
    out = ctypes.c_void_p()
    _check(_lib.gdrr_create_volume(
        ctx, _dev(rho_dev, "float32", nvox, "rho_dev"), _dev(material_dev, "uint8", nvox, "material_dev"),
        nx, ny, nz, float(spacing_mm[0]), float(spacing_mm[1]), float(spacing_mm[2]), centre_p,
        int(n_materials), int(layout), _dev(workspace_dev, "uint8", 0, "workspace_dev"),
        workspace_dev.numel(), _stream(stream), ctypes.byref(out)), ctx)
    return out


def gdrr_create_volume_host(ctx, rho_host, material_host, dims, spacing_mm, centre_mm, n_materials,
                            layout, rho_stage_dev, material_stage_dev, workspace_dev, stream=None):
    """As gdrr_create_volume, from host arrays (numpy, or pinned CPU torch tensors)."""
    nx, ny, nz = (int(x) for x in dims)
    nvox = nx * ny * nz
    rho_p = _host_ptr(rho_host, "float32", nvox)
    mat_p = _host_ptr(material_host, "uint8", nvox)
    centre, centre_p = _host(centre_mm, np.float64)
    out = ctypes.c_void_p()
    _check(_lib.gdrr_create_volume_host(
        ctx, rho_p, mat_p, nx, ny, nz, float(spacing_mm[0]), float(spacing_mm[1]),
        float(spacing_mm[2]), centre_p, int(n_materials), int(layout),
        _dev(rho_stage_dev, "float32", nvox, "rho_stage_dev"),
        _dev(material_stage_dev, "uint8", nvox, "material_stage_dev"),
        _dev(workspace_dev, "uint8", 0, "workspace_dev"), workspace_dev.numel(),
        _stream(stream), ctypes.byref(out)), ctx)
    return out


def _host_ptr(a, dtype_name, min_numel):
    """Address of a contiguous host buffer: numpy array or CPU torch tensor."""
    if isinstance(a, np.ndarray):
        if a.dtype != np.dtype(dtype_name) or not a.flags["C_CONTIGUOUS"] or a.size < min_numel:
            raise ValueError(f"host array must be C-contiguous {dtype_name} with >= {min_numel} elements")
        return a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor) and not a.is_cuda:
        if str(a.dtype) != "torch." + dtype_name or not a.is_contiguous() or a.numel() < min_numel:
            raise ValueError(f"host tensor must be contiguous {dtype_name} with >= {min_numel} elements")
        return a.data_ptr()
    raise TypeError("host buffer must be a numpy array or a CPU torch tensor")


def gdrr_volume_status(ctx, vol):
    """Waits for the volume's ingest; raises GdrrError(INVALID_ARG) if it met a material index >= n_materials."""
    _check(_lib.gdrr_volume_status(ctx, vol), ctx)


def gdrr_destroy_volume(vol):
    _check(_lib.gdrr_destroy_volume(vol))


def gdrr_set_geometry(ctx, sad_mm, sdd_mm, theta_rad, nu, nv, du_mm, dv_mm, u_offset_mm,
                      v_offset_mm, phi_rad, step_mm):
    phi, phi_p = _host(phi_rad, np.float64)
    _check(_lib.gdrr_set_geometry(ctx, float(sad_mm), float(sdd_mm), float(theta_rad), int(nu),
                                  int(nv), float(du_mm), float(dv_mm), float(u_offset_mm),
                                  float(v_offset_mm), int(phi.shape[0]), phi_p, float(step_mm)), ctx)
    if isinstance(ctx, _Context):
        ctx.nu, ctx.nv = int(nu), int(nv)


def gdrr_set_geometry_poses(ctx, nu, nv, du_mm, dv_mm, u_offset_mm, v_offset_mm, poses, step_mm):
    """poses: float64 [n_proj][12] = per projection source S, detector origin P, u_hat, v_hat (mm)."""
    ps, ps_p = _host(np.ascontiguousarray(poses, dtype=np.float64).reshape(-1, 12), np.float64)
    _check(_lib.gdrr_set_geometry_poses(ctx, int(nu), int(nv), float(du_mm), float(dv_mm), float(u_offset_mm),
                                        float(v_offset_mm), int(ps.shape[0]), ps_p, float(step_mm)), ctx)
    if isinstance(ctx, _Context):
        ctx.nu, ctx.nv = int(nu), int(nv)


def gdrr_set_spectrum(ctx, phi_weight, response, mu_hat, fluence_map=None, bowtie_mu=None,
                      bowtie_thickness_mm=None):
    mu, mu_p = _host(mu_hat, np.float64)
    if mu.ndim != 2:
        raise ValueError("mu_hat must be [n_materials][n_energy]")
    n_mat, n_e = mu.shape
    pw, pw_p = _host(phi_weight, np.float64)
    rs, rs_p = _host(response, np.float64)
    if pw.shape != (n_e,) or rs.shape != (n_e,):
        raise ValueError("phi_weight and response must be [n_energy]")
    fl, fl_p = _host(fluence_map, np.float32)
    bm, bm_p = _host(bowtie_mu, np.float64)
    bt, bt_p = _host(bowtie_thickness_mm, np.float64)
    if bm is not None and bm.shape != (n_e,):
        raise ValueError("bowtie_mu must be [n_energy]")
    _check(_lib.gdrr_set_spectrum(ctx, n_e, n_mat, pw_p, rs_p, mu_p, fl_p, bm_p, bt_p), ctx)
    if isinstance(ctx, _Context):
        ctx.n_mat = int(n_mat)


def gdrr_set_response_gain(ctx, gain):
    """gain: float32 [n_energy][nv][nu] (host) or None (= 1)."""
    g, g_p = _host(gain, np.float32)
    if g is not None and isinstance(ctx, _Context) and ctx.nu is not None and g.shape[1:] != (ctx.nv, ctx.nu):
        raise ValueError("gain must be [n_energy][nv][nu]")
    _check(_lib.gdrr_set_response_gain(ctx, g_p), ctx)


def gdrr_project(ctx, vol, proj_begin, proj_count, signal_dev, line_integrals_dev=None,
                 ray_table_dev=None, stream=None):
    n_mat = ctx.n_mat if isinstance(ctx, _Context) and ctx.n_mat else 0
    _check(_lib.gdrr_project(ctx, vol, int(proj_begin), int(proj_count),
                             _dev(signal_dev, "float32", _plane(ctx, proj_count), "signal_dev"),
                             _dev(line_integrals_dev, "float32", _plane(ctx, proj_count, n_mat), "line_integrals_dev"),
                             _dev(ray_table_dev, "int32", _plane(ctx, proj_count, 2), "ray_table_dev"),
                             _stream(stream)), ctx)


def gdrr_project_host(ctx, vol, proj_begin, proj_count, signal_host, signal_stage_dev, stage_proj,
                      stream=None):
    _check(_lib.gdrr_project_host(ctx, vol, int(proj_begin), int(proj_count),
                                  _host_ptr(signal_host, "float32", _plane(ctx, proj_count)),
                                  _dev(signal_stage_dev, "float32", _plane(ctx, stage_proj), "signal_stage_dev"),
                                  int(stage_proj), _stream(stream)), ctx)


def gdrr_ray_setup(ctx, vol, proj_begin, proj_count, ray_table_dev=None, n_samples_dev=None,
                   stream=None):
    _check(_lib.gdrr_ray_setup(ctx, vol, int(proj_begin), int(proj_count),
                               _dev(ray_table_dev, "int32", _plane(ctx, proj_count, 2), "ray_table_dev"),
                               _dev(n_samples_dev, "int64", 1, "n_samples_dev"), _stream(stream)), ctx)


def gdrr_set_method(ctx, method):
    _check(_lib.gdrr_set_method(ctx, int(method)), ctx)


def gdrr_volume_attach_texture(ctx, vol, stream=None):
    _check(_lib.gdrr_volume_attach_texture(ctx, vol, _stream(stream)), ctx)


def gdrr_denoise_scatter(ctx, s_hat_dev, s_dev, scratch_dev, beta, n_iter, omega=0.8, floor_value=1e-12, stream=None):
    """s_hat_dev, s_dev, scratch_dev: float32 CUDA tensors [n_images][nv][nu] (or [nv][nu])."""
    shape = tuple(s_hat_dev.shape)
    n_images, nv, nu = (1,) + shape if len(shape) == 2 else shape
    n = n_images * nv * nu
    _check(_lib.gdrr_denoise_scatter(ctx, _dev(s_hat_dev, "float32", n, "s_hat_dev"), _dev(s_dev, "float32", n, "s_dev"),
                                     _dev(scratch_dev, "float32", n, "scratch_dev"), nu, nv, n_images, float(beta),
                                     float(omega), int(n_iter), float(floor_value), _stream(stream)), ctx)


def gdrr_denoise_scatter_static(ctx, s_hat_dev, s_dev, beta, n_iter, omega=0.8, floor_value=1e-12, stream=None):
    """gdrr_denoise_scatter without a scratch tensor: the library's static scratch array (at most
    GDRR_DENOISE_STATIC_MAX_FLOATS pixels per call; calls that overlap on the GPU race on it)."""
    shape = tuple(s_hat_dev.shape)
    n_images, nv, nu = (1,) + shape if len(shape) == 2 else shape
    n = n_images * nv * nu
    _check(_lib.gdrr_denoise_scatter_static(ctx, _dev(s_hat_dev, "float32", n, "s_hat_dev"),
                                            _dev(s_dev, "float32", n, "s_dev"), nu, nv, n_images, float(beta),
                                            float(omega), int(n_iter), float(floor_value), _stream(stream)), ctx)


def gdrr_set_sampler(ctx, sampler):
    _check(_lib.gdrr_set_sampler(ctx, int(sampler)), ctx)


def gdrr_siddon_segments(ctx, vol, proj_begin, proj_count, n_segments_dev, stream=None):
    _check(_lib.gdrr_siddon_segments(ctx, vol, int(proj_begin), int(proj_count),
                                     _dev(n_segments_dev, "int32", _plane(ctx, proj_count), "n_segments_dev"),
                                     _stream(stream)), ctx)


def gdrr_last_sampler(ctx):
    return int(_lib.gdrr_last_sampler(ctx))


def gdrr_debug_set_skew(ctx, mode):
    _check(_lib.gdrr_debug_set_skew(ctx, int(mode)), ctx)


def gdrr_debug_ray_cells(ctx, vol, projection, i, j, sampler, cells_dev, count_dev, stream=None):
    """cells_dev: int32 CUDA tensor [max_samples][3]; count_dev: int32 CUDA tensor [1]."""
    _check(_lib.gdrr_debug_ray_cells(ctx, vol, int(projection), int(i), int(j), int(sampler),
                                     _dev(cells_dev, "int32", 0, "cells_dev"), int(cells_dev.numel() // 3),
                                     _dev(count_dev, "int32", 1, "count_dev"), _stream(stream)), ctx)


def gdrr_kernel_launches(ctx):
    return int(_lib.gdrr_kernel_launches(ctx))


# ---------------------------------------------------------------------------
# convenience holder (no arithmetic): keeps handles and their tensors together
# ---------------------------------------------------------------------------

class Projector:
    """Context + volume + the torch tensors they borrow, built from a
    workload-like object (attributes as workloads.Workload)."""

    def __init__(self, w, device=0, layout=GDRR_LAYOUT_PACKED_QUAD, from_host=False,
                 method=GDRR_METHOD_TRILINEAR, sampler=GDRR_SAMPLER_AUTO):
        import torch
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.w = w
        self.ctx = gdrr_create_context(device)
        self.vol = None
        self.layout = layout
        self.method = method
        gdrr_set_method(self.ctx, method)
        gdrr_set_sampler(self.ctx, sampler)
        if getattr(w, "poses", None) is not None:      # helical / C-arm / free source path
            gdrr_set_geometry_poses(self.ctx, w.nu, w.nv, w.du, w.dv, w.u_off, w.v_off, w.poses, w.step_mm)
        else:
            gdrr_set_geometry(self.ctx, w.sad, w.sdd, w.theta, w.nu, w.nv, w.du, w.dv, w.u_off, w.v_off,
                              w.phis, w.step_mm)
        gdrr_set_spectrum(self.ctx, w.phi_weight, w.response, w.mu_hat, w.fluence_map, w.bowtie_mu,
                          w.bowtie_thickness)
        if getattr(w, "response_gain", None) is not None:
            gdrr_set_response_gain(self.ctx, w.response_gain)
        nx, ny, nz = w.dims
        nbytes = gdrr_volume_workspace_bytes(nx, ny, nz, w.n_materials, layout)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self.rho_stage = torch.empty((nz, ny, nx), dtype=torch.float32, device=self.device)
            self.mat_stage = torch.empty((nz, ny, nx), dtype=torch.uint8, device=self.device)
            if not from_host:
                self.rho_stage.copy_(torch.from_numpy(w.rho))
                self.mat_stage.copy_(torch.from_numpy(w.mat))
                self.ingest()

    def ingest(self):
        """Step a0 from the device-resident (rho, material) staging tensors."""
        w = self.w
        if self.vol is not None:
            gdrr_destroy_volume(self.vol)
            self.vol = None
        with self.torch.cuda.device(self.device):
            self.vol = gdrr_create_volume(self.ctx, self.rho_stage, self.mat_stage, w.dims, w.spacing,
                                          w.centre, w.n_materials, self.layout, self.workspace)
            if self.method == GDRR_METHOD_TEXTURE:
                gdrr_volume_attach_texture(self.ctx, self.vol)

    def ingest_host(self, rho_host, mat_host):
        """Step a0 from host buffers (H2D copy inside the library call)."""
        w = self.w
        if self.vol is not None:
            gdrr_destroy_volume(self.vol)
            self.vol = None
        with self.torch.cuda.device(self.device):
            self.vol = gdrr_create_volume_host(self.ctx, rho_host, mat_host, w.dims, w.spacing, w.centre,
                                               w.n_materials, self.layout, self.rho_stage,
                                               self.mat_stage, self.workspace)
            if self.method == GDRR_METHOD_TEXTURE:
                gdrr_volume_attach_texture(self.ctx, self.vol)

    def project(self, proj_begin=0, proj_count=None, want_li=False, want_table=False, signal=None):
        torch, w = self.torch, self.w
        n = w.n_proj - proj_begin if proj_count is None else proj_count
        with torch.cuda.device(self.device):
            if signal is None:
                signal = torch.empty((n, w.nv, w.nu), dtype=torch.float32, device=self.device)
            li = (torch.empty((n, w.n_materials, w.nv, w.nu), dtype=torch.float32, device=self.device)
                  if want_li or w.n_materials > 4 else None)      # (more than four materials: required by the library)
            tab = (torch.empty((n, w.nv, w.nu, 2), dtype=torch.int32, device=self.device)
                   if want_table else None)
            gdrr_project(self.ctx, self.vol, proj_begin, n, signal, li, tab)
        return signal, li, tab

    def count_samples(self, proj_begin=0, proj_count=None):
        torch, w = self.torch, self.w
        n = w.n_proj - proj_begin if proj_count is None else proj_count
        with torch.cuda.device(self.device):
            total = torch.zeros(1, dtype=torch.int64, device=self.device)
            gdrr_ray_setup(self.ctx, self.vol, proj_begin, n, None, total)
            return int(total.item())

    def siddon_segments(self, proj_begin=0, proj_count=None):
        torch, w = self.torch, self.w
        n = w.n_proj - proj_begin if proj_count is None else proj_count
        with torch.cuda.device(self.device):
            out = torch.empty((n, w.nv, w.nu), dtype=torch.int32, device=self.device)
            gdrr_siddon_segments(self.ctx, self.vol, proj_begin, n, out)
        return out

    def kernel_launches(self):
        return gdrr_kernel_launches(self.ctx)

    def close(self):
        if self.vol is not None:
            gdrr_destroy_volume(self.vol)
            self.vol = None
        if self.ctx is not None:
            gdrr_destroy_context(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()
