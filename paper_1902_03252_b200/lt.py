"""Thin Python binding of liblt_gradient.so (include/lt_gradient.h): argument marshalling only.

Every step of the path (per-lens precompute, gradient kernels, mixed-rule flagging, fp64 recompute) runs in the CUDA
library; PyTorch is used here for device memory and streams.  There is NO CPU fallback: if the shared library is
missing or cannot be loaded this module raises (it never imports anything from oracle/).

Functions carry the C names; tensors stand for the pointers:
    lt_gradient_grid(lenses[n,7] f64 cuda, x_min, y_min, dx, nx, ny, mode, ...) -> out [ny, nx, 2]
"""
import ctypes
import os

import torch

LT_FP64, LT_FP32, LT_MIXED = 0, 1, 2
LT_OK = 0
LT_ERR_BAD_LENS_PARAMS = -9

_HERE = os.path.dirname(os.path.abspath(__file__))
# LT_GRADIENT_LIB: another build of the same library (csrc/build.py: defines / out) -- for kernel experiments
_LIB_PATH = os.environ.get("LT_GRADIENT_LIB") or os.path.join(_HERE, "liblt_gradient.so")

SYMBOLS = ["lt_version", "lt_error_string", "lt_last_cuda_error", "lt_mixed_defaults", "lt_workspace_bytes",
           "lt_gradient_grid", "lt_gradient_points", "lt_host_workspace_bytes", "lt_gradient_grid_host",
           "lt_gradient_grid_sie", "lt_gradient_points_sie", "lt_gradient_grid_sie_host", "lt_find_images", "lt_mixed_rule",
           "lt_source_barycentres", "lt_chi2",
           "lt_gradient_grid_nfw", "lt_gradient_points_nfw", "lt_gradient_grid_nfw_host",
           "lt_set_tuning", "lt_last_launch_count", "lt_set_kernel_events", "lt_last_status", "lt_mixed_last_stats", "lt_mixed_last_flags", "lt_mixed_last_sp_map", "lt_rule_audit", "lt_rule_audit_result", "lt_peak_probe",
           "lt_gradient_grid_noalloc", "lt_noalloc_last_status"]
LT_NOALLOC_MAX_LENSES = 4096
LT_ERR_NOALLOC_TOO_LARGE = -10


class lt_mixed_params(ctypes.Structure):
    _fields_ = [("m_max", ctypes.c_double), ("c28", ctypes.c_double), ("patch_halfwidth_cluster", ctypes.c_double),
                ("patch_halfwidth_galaxy", ctypes.c_double), ("b0_cluster_threshold", ctypes.c_double)]


class lt_mixed_stats(ctypes.Structure):
    _fields_ = [("n_pixels", ctypes.c_longlong), ("n_flagged", ctypes.c_longlong), ("n_patch", ctypes.c_longlong),
                ("n_eq25", ctypes.c_longlong), ("n_eq28", ctypes.c_longlong)]


LT_AUDIT_BINS = 9
AUDIT_BIN_EDGES_PX = (0, 1, 2, 4, 8, 16, 32, 64, 128)


class lt_audit_result(ctypes.Structure):
    _fields_ = [("n_pixels", ctypes.c_longlong), ("n_violating", ctypes.c_longlong),
                ("n_violating_flagged", ctypes.c_longlong), ("n_violating_missed", ctypes.c_longlong),
                ("n_flagged", ctypes.c_longlong), ("max_err", ctypes.c_double), ("max_err_in_patch", ctypes.c_double),
                ("max_err_outside_patch", ctypes.c_double), ("max_err_by_distance", ctypes.c_double * LT_AUDIT_BINS),
                ("implied_m_max", ctypes.c_double), ("implied_m_max_outside_patch", ctypes.c_double)]


class LtError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().lt_error_string(code).decode()
        if code == -8:
            msg += " [cudaError %d]" % lib().lt_last_cuda_error()
        super().__init__("%s: %s (%d)" % (where, msg, code))


_lib = None


def lib():
    """Loads the in-tree liblt_gradient.so (built by paper_1902_03252_b200.csrc.build).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError("liblt_gradient.so is not built: run `python -m paper_1902_03252_b200.csrc.build` "
                               "(or __graft_entry__.build()).  There is no CPU fallback.")
        L = ctypes.CDLL(_LIB_PATH)
        vp, ci, cd, cll, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_longlong, ctypes.c_size_t
        L.lt_version.restype = ci
        L.lt_error_string.restype = ctypes.c_char_p
        L.lt_error_string.argtypes = [ci]
        L.lt_last_cuda_error.restype = ci
        L.lt_mixed_defaults.argtypes = [ctypes.POINTER(lt_mixed_params)]
        L.lt_mixed_defaults.restype = None
        L.lt_workspace_bytes.argtypes = [ci, ci, ci, ci]
        L.lt_workspace_bytes.restype = sz
        L.lt_host_workspace_bytes.argtypes = [ci, ci, ci, ci]
        L.lt_host_workspace_bytes.restype = sz
        L.lt_gradient_grid.argtypes = [vp, ci, cd, cd, cd, ci, ci, ci, ctypes.POINTER(lt_mixed_params), vp, vp, sz, vp]
        L.lt_gradient_grid.restype = ci
        L.lt_gradient_grid_host.argtypes = L.lt_gradient_grid.argtypes
        L.lt_gradient_grid_host.restype = ci
        L.lt_gradient_points.argtypes = [vp, ci, vp, cll, vp, vp, sz, vp]
        L.lt_gradient_points.restype = ci
        for name in ("lt_gradient_grid_sie", "lt_gradient_grid_sie_host", "lt_gradient_grid_nfw", "lt_gradient_grid_nfw_host"):
            getattr(L, name).argtypes = L.lt_gradient_grid.argtypes
            getattr(L, name).restype = ci
        for name in ("lt_gradient_points_sie", "lt_gradient_points_nfw"):
            getattr(L, name).argtypes = L.lt_gradient_points.argtypes
            getattr(L, name).restype = ci
        L.lt_mixed_rule.argtypes = [vp, cd, cd, cd, ci, ci, vp, ci, ctypes.POINTER(lt_mixed_params), vp, vp, sz, vp]
        L.lt_mixed_rule.restype = ci
        L.lt_find_images.argtypes = [vp, cd, cd, cd, ci, ci, cd, vp, ci, vp, ci, vp, vp]
        L.lt_find_images.restype = ci
        L.lt_source_barycentres.argtypes = [vp, vp, vp, ci, cd, vp, vp]
        L.lt_source_barycentres.restype = ci
        L.lt_chi2.argtypes = [vp, vp, vp, ci, ci, vp, vp, ci, vp, vp, vp]
        L.lt_chi2.restype = ci
        L.lt_set_tuning.argtypes = [ci, ci, ci, ci, ci, ci]
        L.lt_last_launch_count.restype = ci
        L.lt_set_tuning.restype = ci
        L.lt_set_kernel_events.argtypes = [vp, vp]
        L.lt_set_kernel_events.restype = ci
        L.lt_last_status.argtypes = [vp, vp, ctypes.POINTER(ci)]
        L.lt_last_status.restype = ci
        L.lt_mixed_last_stats.argtypes = [vp, vp, ctypes.POINTER(lt_mixed_stats)]
        L.lt_mixed_last_stats.restype = ci
        L.lt_mixed_last_flags.argtypes = [vp, ci, ci, ci, vp, vp]
        L.lt_mixed_last_flags.restype = ci
        L.lt_mixed_last_sp_map.argtypes = [vp, ci, ci, ci, vp, vp]
        L.lt_mixed_last_sp_map.restype = ci
        L.lt_rule_audit.argtypes = [vp, vp, cd, cd, cd, ci, ci, vp, ci, vp, vp, vp, vp]
        L.lt_rule_audit.restype = ci
        L.lt_rule_audit_result.argtypes = [vp, cd, vp, ctypes.POINTER(lt_audit_result)]
        L.lt_rule_audit_result.restype = ci
        L.lt_peak_probe.argtypes = [ci, ci, ctypes.POINTER(cd), vp]
        L.lt_peak_probe.restype = ci
        L.lt_gradient_grid_noalloc.argtypes = [vp, ci, cd, cd, cd, ci, ci, ci, vp, vp]
        L.lt_gradient_grid_noalloc.restype = ci
        L.lt_noalloc_last_status.argtypes = [vp, ctypes.POINTER(ci)]
        L.lt_noalloc_last_status.restype = ci
        _lib = L
    return _lib


def _check(rc, where):
    if rc != LT_OK:
        raise LtError(rc, where)


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _keep(stream, *tensors):
    """A tensor this binding allocated (or a contiguous copy it made) on the current stream and hands to kernels enqueued
    on another `stream` must not go back to the caching allocator's pool before those kernels have run: record the use."""
    if stream is None or stream == torch.cuda.current_stream():
        return
    for t in tensors:
        if isinstance(t, torch.Tensor) and t.is_cuda:
            t.record_stream(stream)


def _lenses_dev(lenses, cols=7):
    if not (isinstance(lenses, torch.Tensor) and lenses.is_cuda and lenses.dtype == torch.float64):
        raise TypeError("lenses must be a CUDA float64 tensor [n_lens, %d]" % cols)
    lenses = lenses.reshape(-1, cols)
    if not lenses.is_contiguous():
        lenses = lenses.contiguous()
    return lenses


def _mixed_ptr(mixed):
    if mixed is None:
        return None
    if isinstance(mixed, lt_mixed_params):
        return ctypes.byref(mixed)
    return ctypes.byref(lt_mixed_params(*[float(v) for v in mixed]))


def lt_version():
    return int(lib().lt_version())


def lt_mixed_defaults():
    p = lt_mixed_params()
    lib().lt_mixed_defaults(ctypes.byref(p))
    return p


def lt_workspace_bytes(n_lens, nx, ny, mode):
    return int(lib().lt_workspace_bytes(int(n_lens), int(nx), int(ny), int(mode)))


def lt_host_workspace_bytes(n_lens, nx, ny, mode):
    return int(lib().lt_host_workspace_bytes(int(n_lens), int(nx), int(ny), int(mode)))


def lt_set_tuning(ppt64=0, ppt32=0, chunk64=0, chunk32=0, ctas_per_sm=0, single_launch=0):
    _check(lib().lt_set_tuning(int(ppt64), int(ppt32), int(chunk64), int(chunk32), int(ctas_per_sm),
                               int(single_launch)), "lt_set_tuning")


def lt_last_launch_count():
    return int(lib().lt_last_launch_count())


def lt_set_kernel_events(ev_start=None, ev_stop=None):
    """Measurement hook: two torch.cuda.Event(enable_timing=True) recorded by the next lt_gradient_grid calls around
    the dominant kernel's launch; None, None switches it off."""
    def handle(ev):
        if ev is None:
            return None
        if not ev.cuda_event:       # torch creates the cudaEvent lazily: force it
            ev.record()
        return ctypes.c_void_p(ev.cuda_event)
    _check(lib().lt_set_kernel_events(handle(ev_start), handle(ev_stop)), "lt_set_kernel_events")


def alloc_workspace(n_lens, nx, ny, mode, device="cuda", host=False):
    n = (lt_host_workspace_bytes if host else lt_workspace_bytes)(n_lens, nx, ny, mode)
    if n == 0:
        raise LtError(-2, "lt_workspace_bytes")
    return torch.empty(n, dtype=torch.uint8, device=device)


def lt_gradient_grid(lenses, x_min, y_min, dx, nx, ny, mode=LT_FP64, mixed=None, out=None, workspace=None,
                     stream=None, _fn="lt_gradient_grid", _cols=7):
    """Deflection map on the device.  Returns `out` ([ny, nx, 2]; float32 for LT_FP32, else float64).  Asynchronous."""
    lenses = _lenses_dev(lenses, _cols)
    n_lens = lenses.shape[0]
    dt = torch.float32 if mode == LT_FP32 else torch.float64
    if out is None:
        out = torch.empty((ny, nx, 2), dtype=dt, device=lenses.device)
    elif out.dtype != dt or out.numel() != nx * ny * 2 or not out.is_contiguous() or not out.is_cuda:
        raise TypeError("out must be a contiguous CUDA %s tensor with nx*ny*2 elements" % dt)
    if workspace is None:
        workspace = alloc_workspace(n_lens, nx, ny, mode, lenses.device)
    rc = getattr(lib(), _fn)(ctypes.c_void_p(lenses.data_ptr() if n_lens else None), n_lens, float(x_min),
                             float(y_min), float(dx), int(nx), int(ny), int(mode), _mixed_ptr(mixed),
                             ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(workspace.data_ptr()),
                             workspace.numel(), _stream(stream))
    _check(rc, _fn)
    _keep(stream, lenses, workspace, out)
    return out


def lt_gradient_grid_noalloc(lenses, x_min, y_min, dx, nx, ny, mode, out, stream=None):
    """lt_gradient_grid (LT_FP64 / LT_FP32, at most LT_NOALLOC_MAX_LENSES dPIE lenses) with the workspace in the library's
    built-in device array: neither this binding nor the library allocates.  `lenses` (CUDA float64 [n_lens, 7], contiguous)
    and `out` ([ny, nx, 2], float64 / float32) are the caller's.  Calls that overlap on the GPU race on the array."""
    if not (lenses.is_cuda and lenses.dtype == torch.float64 and lenses.is_contiguous() and lenses.dim() == 2 and
            lenses.shape[1] == 7):
        raise TypeError("lenses must be a contiguous CUDA float64 [n_lens, 7] tensor")
    dt = torch.float32 if mode == LT_FP32 else torch.float64
    if out.dtype != dt or out.numel() != nx * ny * 2 or not out.is_contiguous() or not out.is_cuda:
        raise TypeError("out must be a contiguous CUDA %s tensor with nx*ny*2 elements" % dt)
    n_lens = lenses.shape[0]
    _check(lib().lt_gradient_grid_noalloc(ctypes.c_void_p(lenses.data_ptr() if n_lens else None), n_lens, float(x_min),
                                          float(y_min), float(dx), int(nx), int(ny), int(mode),
                                          ctypes.c_void_p(out.data_ptr()), _stream(stream)), "lt_gradient_grid_noalloc")
    return out


def lt_noalloc_last_status(stream=None):
    """(code, first offending lens index or -1) of the last lt_gradient_grid_noalloc call on the current device."""
    bad = ctypes.c_int(-1)
    rc = lib().lt_noalloc_last_status(_stream(stream), ctypes.byref(bad))
    if rc not in (LT_OK, LT_ERR_BAD_LENS_PARAMS):
        raise LtError(rc, "lt_noalloc_last_status")
    return rc, bad.value


def lt_gradient_grid_sie(lenses, x_min, y_min, dx, nx, ny, mode=LT_FP64, mixed=None, out=None, workspace=None,
                         stream=None):
    """The same with the paper's SIE body (Algorithm 1); lenses: CUDA float64 [n_lens, 5] = (xc, yc, eps, Phi, b0)."""
    return lt_gradient_grid(lenses, x_min, y_min, dx, nx, ny, mode, mixed, out, workspace, stream,
                            _fn="lt_gradient_grid_sie", _cols=5)


def lt_gradient_grid_host(h_lenses, x_min, y_min, dx, nx, ny, mode, h_out, workspace, mixed=None, stream=None,
                          _fn="lt_gradient_grid_host", _cols=7):
    """End-to-end call with HOST buffers (CPU tensors, ideally pinned): H2D of the catalogue, the hot path, D2H of the
    map, all enqueued on the stream.  The caller synchronises before reading h_out."""
    if h_lenses.is_cuda or h_out.is_cuda or h_lenses.dtype != torch.float64 or not h_lenses.is_contiguous():
        raise TypeError("h_lenses / h_out must be contiguous CPU tensors (float64 catalogue)")
    n_lens = h_lenses.reshape(-1, _cols).shape[0]
    dt = torch.float32 if mode == LT_FP32 else torch.float64
    if h_out.dtype != dt or h_out.numel() != nx * ny * 2 or not h_out.is_contiguous():
        raise TypeError("h_out must be a contiguous CPU %s tensor with nx*ny*2 elements" % dt)
    rc = getattr(lib(), _fn)(ctypes.c_void_p(h_lenses.data_ptr() if n_lens else None), n_lens, float(x_min),
                             float(y_min), float(dx), int(nx), int(ny), int(mode), _mixed_ptr(mixed),
                             ctypes.c_void_p(h_out.data_ptr()), ctypes.c_void_p(workspace.data_ptr()),
                             workspace.numel(), _stream(stream))
    _check(rc, _fn)
    _keep(stream, workspace)
    return h_out


def lt_gradient_grid_sie_host(h_lenses, x_min, y_min, dx, nx, ny, mode, h_out, workspace, mixed=None, stream=None):
    return lt_gradient_grid_host(h_lenses, x_min, y_min, dx, nx, ny, mode, h_out, workspace, mixed, stream,
                                 _fn="lt_gradient_grid_sie_host", _cols=5)


def lt_gradient_points(lenses, points, out=None, workspace=None, stream=None, _fn="lt_gradient_points", _cols=7):
    """fp64 deflection at arbitrary points ([n, 2] float64 CUDA).  Returns [n, 2]."""
    lenses = _lenses_dev(lenses, _cols)
    n_lens = lenses.shape[0]
    if not (points.is_cuda and points.dtype == torch.float64):
        raise TypeError("points must be a CUDA float64 tensor [n, 2]")
    points = points.reshape(-1, 2).contiguous()
    n = points.shape[0]
    if out is None:
        out = torch.empty((n, 2), dtype=torch.float64, device=points.device)
    if workspace is None:
        workspace = alloc_workspace(n_lens, 1, 1, LT_FP64, points.device)
    rc = getattr(lib(), _fn)(ctypes.c_void_p(lenses.data_ptr() if n_lens else None), n_lens,
                             ctypes.c_void_p(points.data_ptr() if n else None), n,
                             ctypes.c_void_p(out.data_ptr() if n else None),
                             ctypes.c_void_p(workspace.data_ptr()), workspace.numel(), _stream(stream))
    _check(rc, _fn)
    _keep(stream, lenses, points, workspace, out)
    return out


def lt_gradient_grid_nfw(lenses, x_min, y_min, dx, nx, ny, mode=LT_FP64, mixed=None, out=None, workspace=None,
                         stream=None):
    """The same for pseudo-elliptical NFW lenses; lenses: CUDA float64 [n_lens, 6] = (xc, yc, eps, Phi, kappa_s, rs)."""
    return lt_gradient_grid(lenses, x_min, y_min, dx, nx, ny, mode, mixed, out, workspace, stream,
                            _fn="lt_gradient_grid_nfw", _cols=6)


def lt_gradient_grid_nfw_host(h_lenses, x_min, y_min, dx, nx, ny, mode, h_out, workspace, mixed=None, stream=None):
    return lt_gradient_grid_host(h_lenses, x_min, y_min, dx, nx, ny, mode, h_out, workspace, mixed, stream,
                                 _fn="lt_gradient_grid_nfw_host", _cols=6)


def lt_gradient_points_nfw(lenses, points, out=None, workspace=None, stream=None):
    return lt_gradient_points(lenses, points, out, workspace, stream, _fn="lt_gradient_points_nfw", _cols=6)


def lt_gradient_points_sie(lenses, points, out=None, workspace=None, stream=None):
    return lt_gradient_points(lenses, points, out, workspace, stream, _fn="lt_gradient_points_sie", _cols=5)


def lt_mixed_rule(sp_map, x_min, y_min, dx, centres, mixed=None, workspace=None, stream=None):
    """The mixed rule on a caller-supplied single precision map ([ny, nx, 2] float32 CUDA); centres: [n, 3] float64 CUDA
    (x, y, deflection scale).  Returns (flags uint8 [ny, nx], workspace)."""
    if not (sp_map.is_cuda and sp_map.dtype == torch.float32 and sp_map.is_contiguous() and sp_map.dim() == 3):
        raise TypeError("sp_map must be a contiguous CUDA float32 tensor [ny, nx, 2]")
    ny, nx = sp_map.shape[0], sp_map.shape[1]
    centres = centres.reshape(-1, 3).contiguous()
    n = centres.shape[0]
    if workspace is None:
        workspace = alloc_workspace(0, nx, ny, LT_MIXED, sp_map.device)
    flags = torch.empty((ny, nx), dtype=torch.uint8, device=sp_map.device)
    rc = lib().lt_mixed_rule(ctypes.c_void_p(sp_map.data_ptr()), float(x_min), float(y_min), float(dx), int(nx), int(ny),
                             ctypes.c_void_p(centres.data_ptr() if n else None), n, _mixed_ptr(mixed),
                             ctypes.c_void_p(flags.data_ptr()), ctypes.c_void_p(workspace.data_ptr()), workspace.numel(),
                             _stream(stream))
    _check(rc, "lt_mixed_rule")
    _keep(stream, centres, workspace, flags)
    return flags, workspace


HIT_DTYPE = [("source", "i4"), ("cell", "i4"), ("triangle", "i4"), ("reserved", "i4"), ("x", "f8"), ("y", "f8")]


def lt_find_images(grad, x_min, y_min, dx, dls_dos, sources, max_hits=1 << 16, hits=None, n_hits=None, stream=None):
    """Predicted images of the source points `sources` ([n, 2] float64 CUDA) on the fp64 map `grad` ([ny, nx, 2] float64
    CUDA).  Returns (hits, n_hits): a uint8 CUDA tensor [max_hits, 32] of lt_image_hit records and a 1-element int32
    CUDA tensor with the number found.  Asynchronous; decode with hits_to_numpy after synchronising."""
    if not (grad.is_cuda and grad.dtype == torch.float64 and grad.is_contiguous() and grad.dim() == 3):
        raise TypeError("grad must be a contiguous CUDA float64 tensor [ny, nx, 2]")
    ny, nx = grad.shape[0], grad.shape[1]
    if not (sources.is_cuda and sources.dtype == torch.float64):
        raise TypeError("sources must be a CUDA float64 tensor [n, 2]")
    sources = sources.reshape(-1, 2).contiguous()
    n = sources.shape[0]
    if hits is None:
        hits = torch.empty((max(int(max_hits), 1), 32), dtype=torch.uint8, device=grad.device)
    if n_hits is None:
        n_hits = torch.empty(1, dtype=torch.int32, device=grad.device)
    rc = lib().lt_find_images(ctypes.c_void_p(grad.data_ptr()), float(x_min), float(y_min), float(dx), int(nx), int(ny),
                              float(dls_dos), ctypes.c_void_p(sources.data_ptr() if n else None), n,
                              ctypes.c_void_p(hits.data_ptr()), int(max_hits), ctypes.c_void_p(n_hits.data_ptr()),
                              _stream(stream))
    _check(rc, "lt_find_images")
    _keep(stream, sources, hits, n_hits)
    return hits, n_hits


def hits_to_numpy(hits, n_hits):
    """(synchronises) the stored records as a numpy structured array sorted by (source, cell, triangle), and the count"""
    import numpy as np
    n = int(n_hits.item())
    a = hits.cpu().numpy().view(np.dtype(HIT_DTYPE)).reshape(-1)[: min(n, hits.shape[0])]
    return np.sort(a, order=["source", "cell", "triangle"]), n


def _offsets_dev(offsets, device):
    if not (isinstance(offsets, torch.Tensor) and offsets.is_cuda and offsets.dtype == torch.int32):
        raise TypeError("offsets must be a CUDA int32 tensor [n_systems + 1]")
    return offsets.contiguous()


def lt_source_barycentres(theta, alpha, offsets, dls_dos, out=None, stream=None):
    """Barycentre, per multiple-image system, of the observed images lensed back into the source plane (eq. 13).
    theta, alpha: [n_images, 2] float64 CUDA; offsets: [n_systems + 1] int32 CUDA.  Returns [n_systems, 2]."""
    for t in (theta, alpha):
        if not (t.is_cuda and t.dtype == torch.float64):
            raise TypeError("theta and alpha must be CUDA float64 tensors [n_images, 2]")
    theta, alpha = theta.reshape(-1, 2).contiguous(), alpha.reshape(-1, 2).contiguous()
    offsets = _offsets_dev(offsets, theta.device)
    n_sys = offsets.numel() - 1
    if out is None:
        out = torch.empty((n_sys, 2), dtype=torch.float64, device=theta.device)
    rc = lib().lt_source_barycentres(ctypes.c_void_p(theta.data_ptr() if theta.numel() else out.data_ptr()),
                                     ctypes.c_void_p(alpha.data_ptr() if alpha.numel() else out.data_ptr()),
                                     ctypes.c_void_p(offsets.data_ptr()), n_sys, float(dls_dos),
                                     ctypes.c_void_p(out.data_ptr() if n_sys else None), _stream(stream))
    _check(rc, "lt_source_barycentres")
    _keep(stream, theta, alpha, offsets, out)
    return out


def lt_chi2(theta_obs, sigma, offsets, hits, n_hits, terms=None, result=None, stream=None):
    """Eq. 11 with every observed image paired with the nearest predicted image of its system.  theta_obs [n_images, 2]
    and sigma [n_images] float64 CUDA, offsets [n_systems + 1] int32 CUDA, hits / n_hits as lt_find_images returned them.
    Returns (result, terms): a 32-byte uint8 CUDA tensor holding lt_chi2_result (decode with chi2_to_python) and the
    per-image terms (nan = no predicted image in that system).  Asynchronous."""
    if not (theta_obs.is_cuda and theta_obs.dtype == torch.float64 and sigma.is_cuda and sigma.dtype == torch.float64):
        raise TypeError("theta_obs and sigma must be CUDA float64 tensors")
    theta_obs, sigma = theta_obs.reshape(-1, 2).contiguous(), sigma.reshape(-1).contiguous()
    n_img = theta_obs.shape[0]
    if sigma.numel() != n_img:
        raise ValueError("sigma must have one entry per observed image")
    offsets = _offsets_dev(offsets, theta_obs.device)
    n_sys = offsets.numel() - 1
    if terms is None:
        terms = torch.empty(max(n_img, 1), dtype=torch.float64, device=theta_obs.device)[:n_img]
    if result is None:
        result = torch.empty(32, dtype=torch.uint8, device=theta_obs.device)
    rc = lib().lt_chi2(ctypes.c_void_p(theta_obs.data_ptr() if n_img else None),
                       ctypes.c_void_p(sigma.data_ptr() if n_img else None), ctypes.c_void_p(offsets.data_ptr()), n_sys,
                       n_img, ctypes.c_void_p(hits.data_ptr()), ctypes.c_void_p(n_hits.data_ptr()), int(hits.shape[0]),
                       ctypes.c_void_p(terms.data_ptr() if n_img else None), ctypes.c_void_p(result.data_ptr()),
                       _stream(stream))
    _check(rc, "lt_chi2")
    _keep(stream, theta_obs, sigma, offsets, hits, n_hits, terms, result)
    return result, terms


def chi2_to_python(result):
    """(synchronises) (chi2, n_matched, n_unmatched) from the 32-byte record lt_chi2 wrote"""
    import numpy as np
    raw = result.cpu().numpy().tobytes()
    return float(np.frombuffer(raw, np.float64, 1)[0]), int(np.frombuffer(raw, np.int64, 3, 8)[0]), \
        int(np.frombuffer(raw, np.int64, 3, 8)[1])


def lt_last_status(workspace, stream=None):
    """(code, first offending lens index or -1).  Synchronises the stream."""
    bad = ctypes.c_int(-1)
    rc = lib().lt_last_status(ctypes.c_void_p(workspace.data_ptr()), _stream(stream), ctypes.byref(bad))
    if rc not in (LT_OK, LT_ERR_BAD_LENS_PARAMS):
        raise LtError(rc, "lt_last_status")
    return rc, bad.value


def lt_mixed_last_stats(workspace, stream=None):
    s = lt_mixed_stats()
    _check(lib().lt_mixed_last_stats(ctypes.c_void_p(workspace.data_ptr()), _stream(stream), ctypes.byref(s)),
           "lt_mixed_last_stats")
    return {"n_flagged": s.n_flagged, "n_patch": s.n_patch, "n_eq25": s.n_eq25, "n_eq28": s.n_eq28}


def lt_mixed_last_flags(workspace, n_lens, nx, ny, stream=None):
    out = torch.empty((ny, nx), dtype=torch.uint8, device=workspace.device)
    _check(lib().lt_mixed_last_flags(ctypes.c_void_p(workspace.data_ptr()), int(n_lens), int(nx), int(ny),
                                     ctypes.c_void_p(out.data_ptr()), _stream(stream)), "lt_mixed_last_flags")
    return out


def lt_mixed_last_sp_map(workspace, n_lens, nx, ny, stream=None):
    """The single precision map ([ny, nx, 2] float32) the last LT_MIXED call on this workspace evaluated its rule on."""
    out = torch.empty((ny, nx, 2), dtype=torch.float32, device=workspace.device)
    _check(lib().lt_mixed_last_sp_map(ctypes.c_void_p(workspace.data_ptr()), int(n_lens), int(nx), int(ny),
                                      ctypes.c_void_p(out.data_ptr()), _stream(stream)), "lt_mixed_last_sp_map")
    return out


def lt_rule_audit(sp_map, dp_map, x_min, y_min, dx, centres=None, flags=None, want_violation=False, stream=None):
    """The paper's accuracy criterion |err_i| <= dx / (4 M_i) of a single precision map ([ny, nx, 2] float32
    CUDA) against a double precision map ([ny, nx, 2] float64 CUDA).  centres: [n, 3] float64 CUDA or None; flags: the
    rule's mask ([ny, nx] uint8 CUDA) or None.  Synchronises.  Returns (dict of lt_audit_result's fields, violation
    map [ny, nx] uint8 CUDA or None)."""
    if not (sp_map.is_cuda and sp_map.dtype == torch.float32 and sp_map.is_contiguous() and sp_map.dim() == 3):
        raise TypeError("sp_map must be a contiguous CUDA float32 tensor [ny, nx, 2]")
    if not (dp_map.is_cuda and dp_map.dtype == torch.float64 and dp_map.is_contiguous() and dp_map.shape == sp_map.shape):
        raise TypeError("dp_map must be a contiguous CUDA float64 tensor of sp_map's shape")
    ny, nx = sp_map.shape[0], sp_map.shape[1]
    n = 0
    if centres is not None:
        centres = centres.reshape(-1, 3).contiguous()
        n = centres.shape[0]
    if flags is not None and not (flags.is_cuda and flags.dtype == torch.uint8 and flags.is_contiguous() and flags.numel() == nx * ny):
        raise TypeError("flags must be a contiguous CUDA uint8 tensor [ny, nx]")
    viol = torch.empty((ny, nx), dtype=torch.uint8, device=sp_map.device) if want_violation else None
    d_res = torch.empty(ctypes.sizeof(lt_audit_result), dtype=torch.uint8, device=sp_map.device)
    _check(lib().lt_rule_audit(ctypes.c_void_p(sp_map.data_ptr()), ctypes.c_void_p(dp_map.data_ptr()), float(x_min),
                               float(y_min), float(dx), int(nx), int(ny),
                               ctypes.c_void_p(centres.data_ptr() if n else None), n,
                               ctypes.c_void_p(flags.data_ptr() if flags is not None else None),
                               ctypes.c_void_p(viol.data_ptr() if viol is not None else None),
                               ctypes.c_void_p(d_res.data_ptr()), _stream(stream)), "lt_rule_audit")
    _keep(stream, centres, d_res, viol)
    return d_res, viol


def lt_rule_audit_result(d_result, dx, stream=None):
    """(synchronises) the fields of the lt_audit_result that lt_rule_audit left in device memory, as a dict"""
    h = lt_audit_result()
    _check(lib().lt_rule_audit_result(ctypes.c_void_p(d_result.data_ptr()), float(dx), _stream(stream), ctypes.byref(h)),
           "lt_rule_audit_result")
    out = {name: getattr(h, name) for name, _ in lt_audit_result._fields_ if name != "max_err_by_distance"}
    out["max_err_by_distance"] = list(h.max_err_by_distance)
    return out


def lt_peak_probe(which, iters=1 << 16, stream=None):
    """Achieved FLOP/s of a dependent-free FMA-chain kernel (0 = fp64, 1 = fp32, 2 = fp32 packed pairs; 3 = fp64 and
    4 = packed fp32 with three distinct register sources per instruction).  Synchronises."""
    v = ctypes.c_double(0.0)
    _check(lib().lt_peak_probe(int(which), int(iters), ctypes.byref(v), _stream(stream)), "lt_peak_probe")
    return v.value
