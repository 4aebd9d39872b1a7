"""ctypes binding of include/smre.h: same names, argument marshalling only.

Every step of the projection runs in the CUDA kernels behind the C ABI.  There is no CPU
fallback: if libsmre.so is missing or cannot be loaded, importing callers get an exception.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import _build

SMRE_OK, SMRE_EINVAL, SMRE_EUNSUPPORTED, SMRE_ENOMEM, SMRE_ECUDA = range(5)
SMRE_STANDARD, SMRE_INCOMPLETE = 0, 1
SMRE_SCHED_AUTO, SMRE_SCHED_GRAPH, SMRE_SCHED_PERSISTENT, SMRE_SCHED_STRIPS = 0, 1, 2, 3
_STATUS = {0: "SMRE_OK", 1: "SMRE_EINVAL", 2: "SMRE_EUNSUPPORTED", 3: "SMRE_ENOMEM", 4: "SMRE_ECUDA"}

# every symbol include/smre.h declares
class AdmmParams(ctypes.Structure):
    """smre_admm_params of include/smre.h; defaults are App. B of the paper."""
    _fields_ = [("sigma_psf", ctypes.c_float), ("rho1", ctypes.c_float), ("rho2", ctypes.c_float),
                ("alpha1", ctypes.c_float), ("alpha2", ctypes.c_float), ("lam", ctypes.c_float),
                ("gamma", ctypes.c_float), ("delta", ctypes.c_float), ("max_iter", ctypes.c_int),
                ("n_sweeps", ctypes.c_int), ("check_every", ctypes.c_int)]


exported_symbols = (
    "smre_create", "smre_project", "smre_project_host", "smre_destroy", "smre_set_schedule",
    "smre_info", "smre_family", "smre_export_increments", "smre_last_launch", "smre_last_error",
    "smre_plan_check", "smre_project_noalloc", "smre_project_tol", "smre_export_tile_cycles", "smre_calibrate", "smre_cumulant2",
    "smre_shape", "smre_admm", "smre_psf_apply",
)


class SmreError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{_STATUS.get(status, status)}: {text}")
        self.status = status


def lib_path() -> str:
    return _build.LIB


_lib = None
_vp, _ip, _fp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_float)
_llp = ctypes.POINTER(ctypes.c_longlong)


def load_library(build_if_missing: bool = True):
    """dlopen libsmre.so (building it with nvcc first if the sources are newer)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build() if build_if_missing else _build.LIB
    if not os.path.exists(path):
        raise ImportError(f"{path} is missing: build it with `python -m paper_1503_03492_b200._build`")
    lib = ctypes.CDLL(path)
    lib.smre_create.argtypes = [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                _ip, ctypes.c_int, _fp, ctypes.c_int]
    lib.smre_project.argtypes = [_vp, _vp, _vp, ctypes.c_int, _vp]
    lib.smre_project_host.argtypes = [_vp, _vp, _vp, ctypes.c_int, _vp]
    lib.smre_destroy.argtypes = [_vp]
    lib.smre_set_schedule.argtypes = [_vp, ctypes.c_int]
    lib.smre_info.argtypes = [_vp, _ip, _llp, _llp]
    lib.smre_family.argtypes = [_vp, ctypes.c_int, _ip, _ip, _ip, _fp]
    lib.smre_export_increments.argtypes = [_vp, _vp, _vp]
    lib.smre_last_launch.argtypes = [_vp, _ip, _llp, _ip, _ip]
    lib.smre_plan_check.argtypes = [ctypes.c_int, ctypes.c_int, _ip, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                    _ip, _ip, _ip, _ip, _llp]
    lib.smre_project_noalloc.argtypes = [ctypes.c_int, ctypes.c_int, _ip, ctypes.c_int, _fp, _vp, _vp, ctypes.c_int, _vp]
    lib.smre_calibrate.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, ctypes.c_int, _vp, ctypes.c_float,
                                   _vp, _vp, _vp, _vp]
    lib.smre_cumulant2.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, _vp, _vp, _vp]
    lib.smre_project_tol.argtypes = [_vp, _vp, _vp, ctypes.c_int, ctypes.c_float, _vp, _vp]
    lib.smre_shape.argtypes = [_vp, _ip, _ip, _ip, _ip]
    lib.smre_admm.argtypes = [_vp, ctypes.c_int, ctypes.c_int, _vp, ctypes.POINTER(AdmmParams), _vp, _vp, _ip, _vp, _vp]
    lib.smre_psf_apply.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_float, _vp, _vp, _vp, _vp]
    lib.smre_export_tile_cycles.argtypes = [_vp, ctypes.c_int, _vp, _ip, _ip, _vp]
    for name in exported_symbols:
        getattr(lib, name).restype = ctypes.c_int
    lib.smre_last_error.restype = ctypes.c_char_p
    lib.smre_last_error.argtypes = []
    _lib = lib
    return lib


def smre_last_error() -> str:
    return load_library().smre_last_error().decode()


def _check(status):
    if status != SMRE_OK:
        raise SmreError(status, smre_last_error())


def smre_create(H, W, batch, sides, c_table, variant):
    """-> opaque handle (int).  sides: ints, c_table: float32 thresholds, one per side."""
    lib = load_library()
    sides = np.ascontiguousarray(sides, dtype=np.int32)
    c_table = np.ascontiguousarray(c_table, dtype=np.float32)
    if sides.ndim != 1 or sides.shape != c_table.shape:
        raise ValueError("sides and c_table must be 1-D and of equal length")
    h = _vp()
    _check(lib.smre_create(ctypes.byref(h), int(H), int(W), int(batch),
                           sides.ctypes.data_as(_ip), len(sides), c_table.ctypes.data_as(_fp),
                           int(variant)))
    return h.value


def smre_project(handle, y_ptr, x_out_ptr, n_sweeps, stream=0):
    """y_ptr / x_out_ptr: device addresses (tensor.data_ptr()); stream: cudaStream_t as int."""
    _check(load_library().smre_project(handle, y_ptr, x_out_ptr, int(n_sweeps), stream))


def smre_project_host(handle, y_ptr, x_out_ptr, n_sweeps, stream=0):
    """Host addresses (numpy .ctypes.data or pinned tensor.data_ptr()); blocks until done."""
    _check(load_library().smre_project_host(handle, y_ptr, x_out_ptr, int(n_sweeps), stream))


def smre_project_noalloc(H, W, sides, c_table, y_ptr, x_out_ptr, n_sweeps, stream=0):
    """Standard projection of one H x W image with the increment planes in the library's static device scratch
    (SMRE_NOALLOC_MAX_BYTES): allocates nothing.  y_ptr / x_out_ptr: device addresses."""
    sides = np.ascontiguousarray(sides, dtype=np.int32)
    c_table = np.ascontiguousarray(c_table, dtype=np.float32)
    if sides.ndim != 1 or sides.shape != c_table.shape:
        raise ValueError("sides and c_table must be 1-D and of equal length")
    _check(load_library().smre_project_noalloc(int(H), int(W), sides.ctypes.data_as(_ip), len(sides),
                                               c_table.ctypes.data_as(_fp), y_ptr, x_out_ptr, int(n_sweeps), stream))


def smre_project_tol(handle, y_ptr, x_out_ptr, max_sweeps, tol, sweeps_done_ptr=None, stream=0):
    """Projection under the paper's stop rules (Alg. 2 / Listing 3); sweeps_done_ptr: device int address or None."""
    _check(load_library().smre_project_tol(handle, y_ptr, x_out_ptr, int(max_sweeps), float(tol), sweeps_done_ptr, stream))


def smre_export_tile_cycles(handle, shift, out_ptr=None, stream=0):
    """-> (tiles_y, tiles_x) of the shift; copies the per-tile cycle counts to out_ptr (device ints) if given."""
    ty, tx = ctypes.c_int(), ctypes.c_int()
    _check(load_library().smre_export_tile_cycles(handle, int(shift), out_ptr, ctypes.byref(ty), ctypes.byref(tx), stream))
    return ty.value, tx.value


def smre_calibrate(H, W, n_frames, sides, noise_ptr, alpha, q_stat_ptr, q_alpha_ptr, c_table_ptr, stream=0):
    """Thresholds from simulated noise (sec. 2.1); all *_ptr are device addresses."""
    sides = np.ascontiguousarray(sides, dtype=np.int32)
    _check(load_library().smre_calibrate(int(H), int(W), int(n_frames), sides.ctypes.data_as(_ip), len(sides), noise_ptr,
                                         float(alpha), q_stat_ptr, q_alpha_ptr, c_table_ptr, stream))


def calibrate(noise, sides, alpha):
    """noise: float32 CUDA tensor [n,H,W] of unit-variance noise -> (c_table [n_sides], q_alpha [1], Q [n]) tensors."""
    import torch
    if not (noise.is_cuda and noise.dtype == torch.float32 and noise.is_contiguous() and noise.dim() == 3):
        raise ValueError("noise must be a contiguous float32 CUDA tensor [n, H, W]")
    n, H, W = noise.shape
    q = torch.empty(n, dtype=torch.float32, device=noise.device)
    qa = torch.empty(1, dtype=torch.float32, device=noise.device)
    c = torch.empty(len(sides), dtype=torch.float32, device=noise.device)
    smre_calibrate(H, W, n, sides, noise.data_ptr(), alpha, q.data_ptr(), qa.data_ptr(), c.data_ptr(),
                   torch.cuda.current_stream(noise.device).cuda_stream)
    return c, qa, q


def smre_cumulant2(H, W, n_frames, stack_ptr, out_ptr, stream=0):
    """C_2 = <F^2> - <F>^2 per pixel over a stack (Eq. 19); device addresses."""
    _check(load_library().smre_cumulant2(int(H), int(W), int(n_frames), stack_ptr, out_ptr, stream))


def smre_admm(handle, H, W, I_ptr, params, x_ptr, eps_ptr=None, hist_ptr=None, stream=0):
    """The ADMM around the projection (include/smre.h); device addresses; returns the iterations done."""
    it = ctypes.c_int(0)
    _check(load_library().smre_admm(handle, int(H), int(W), I_ptr, ctypes.byref(params), x_ptr, eps_ptr,
                                    ctypes.byref(it), hist_ptr, stream))
    return it.value


def smre_psf_apply(H, W, sigma, in_ptr, tmp_ptr, out_ptr, stream=0):
    _check(load_library().smre_psf_apply(int(H), int(W), float(sigma), in_ptr, tmp_ptr, out_ptr, stream))


def admm(solver, image, sigma_psf, gamma, delta=1e-3, max_iter=10000, n_sweeps=200, rho1=6.192, rho2=1.8, alpha1=1.2,
         alpha2=0.12, lam=1.0, check_every=8, return_history=False):
    """image: float32 CUDA tensor [H,W]; solver: a Solver with batch 1.  Returns (x, eps, iterations[, hist])."""
    import torch
    if not (image.is_cuda and image.dtype == torch.float32 and image.is_contiguous() and image.dim() == 2):
        raise ValueError("image must be a contiguous float32 CUDA tensor [H,W]")
    H, W = image.shape
    p = AdmmParams(sigma_psf, rho1, rho2, alpha1, alpha2, lam, gamma, delta, int(max_iter), int(n_sweeps), int(check_every))
    x = torch.empty_like(image)
    eps = torch.empty_like(image)
    hist = torch.zeros(2 * int(max_iter), device=image.device) if return_history else None
    it = smre_admm(solver.handle, H, W, image.data_ptr(), p, x.data_ptr(), eps.data_ptr(),
                   hist.data_ptr() if return_history else None, torch.cuda.current_stream(image.device).cuda_stream)
    if return_history:
        return x, eps, it, hist[:2 * it].reshape(it, 2)
    return x, eps, it


def psf_apply(image, sigma_psf):
    import torch
    if not (image.is_cuda and image.dtype == torch.float32 and image.is_contiguous() and image.dim() == 2):
        raise ValueError("image must be a contiguous float32 CUDA tensor [H,W]")
    tmp = torch.empty_like(image)
    out = torch.empty_like(image)
    smre_psf_apply(image.shape[0], image.shape[1], sigma_psf, image.data_ptr(), tmp.data_ptr(), out.data_ptr(),
                   torch.cuda.current_stream(image.device).cuda_stream)
    return out


def cumulant2(stack):
    """stack: float32 CUDA tensor [n,H,W] -> float32 tensor [H,W]."""
    import torch
    if not (stack.is_cuda and stack.dtype == torch.float32 and stack.is_contiguous() and stack.dim() == 3):
        raise ValueError("stack must be a contiguous float32 CUDA tensor [n, H, W]")
    n, H, W = stack.shape
    out = torch.empty((H, W), dtype=torch.float32, device=stack.device)
    smre_cumulant2(H, W, n, stack.data_ptr(), out.data_ptr(), torch.cuda.current_stream(stack.device).cuda_stream)
    return out


def smre_destroy(handle):
    _check(load_library().smre_destroy(handle))


def smre_set_schedule(handle, schedule):
    _check(load_library().smre_set_schedule(handle, int(schedule)))


def smre_info(handle):
    n, w, b = ctypes.c_int(), ctypes.c_longlong(), ctypes.c_longlong()
    _check(load_library().smre_info(handle, ctypes.byref(n), ctypes.byref(w), ctypes.byref(b)))
    return n.value, w.value, b.value


def smre_family(handle, idx):
    s, oy, ox, c = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_float()
    _check(load_library().smre_family(handle, int(idx), ctypes.byref(s), ctypes.byref(oy),
                                      ctypes.byref(ox), ctypes.byref(c)))
    return s.value, oy.value, ox.value, c.value


def smre_export_increments(handle, q_out_ptr, stream=0):
    _check(load_library().smre_export_increments(handle, q_out_ptr, stream))


def smre_last_launch(handle):
    s, n, ty, tx = ctypes.c_int(), ctypes.c_longlong(), ctypes.c_int(), ctypes.c_int()
    _check(load_library().smre_last_launch(handle, ctypes.byref(s), ctypes.byref(n),
                                           ctypes.byref(ty), ctypes.byref(tx)))
    return s.value, n.value, ty.value, tx.value


def smre_plan_check(H, W, sides, n_sweeps, max_ctas=148):
    """Host-only: -> (tiles_y, tiles_x, max_tile_h, max_tile_w, table_bytes) of the conveyor plan."""
    sides = np.ascontiguousarray(sides, dtype=np.int32)
    ty, tx, mh, mw, tb = (ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int(),
                          ctypes.c_longlong())
    _check(load_library().smre_plan_check(int(H), int(W), sides.ctypes.data_as(_ip), len(sides),
                                          int(n_sweeps), int(max_ctas), ctypes.byref(ty), ctypes.byref(tx),
                                          ctypes.byref(mh), ctypes.byref(mw), ctypes.byref(tb)))
    return ty.value, tx.value, mh.value, mw.value, tb.value


class Solver:
    """Convenience owner of one handle for torch tensors (marshalling only)."""

    def __init__(self, H, W, sides, c_table, variant="standard", batch=1, schedule=SMRE_SCHED_AUTO):
        v = {"standard": SMRE_STANDARD, "incomplete": SMRE_INCOMPLETE}.get(variant, variant)
        self.H, self.W, self.batch, self.variant = int(H), int(W), int(batch), v
        self.handle = smre_create(H, W, batch, sides, c_table, v)
        if schedule != SMRE_SCHED_AUTO:
            smre_set_schedule(self.handle, schedule)

    def project(self, y, n_sweeps, out=None, stream=None):
        import torch
        if not (y.is_cuda and y.dtype == torch.float32 and y.is_contiguous()):
            raise ValueError("y must be a contiguous float32 CUDA tensor")
        if y.numel() != self.batch * self.H * self.W:
            raise ValueError("y has the wrong number of elements")
        if out is None:
            out = torch.empty_like(y)
        elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
                  and out.numel() == y.numel()):
            raise ValueError("out must be a contiguous float32 CUDA tensor of y's size")
        st = torch.cuda.current_stream(y.device) if stream is None else stream
        smre_project(self.handle, y.data_ptr(), out.data_ptr(), n_sweeps, st.cuda_stream)
        return out

    def project_tol(self, y, max_sweeps, tol, out=None):
        """-> (x, sweeps_done int32 tensor: [batch] for the standard variant, [1] = largest tile count for ICD)."""
        import torch
        if not (y.is_cuda and y.dtype == torch.float32 and y.is_contiguous()) or y.numel() != self.batch * self.H * self.W:
            raise ValueError("y must be a contiguous float32 CUDA tensor of batch*H*W elements")
        if out is None:
            out = torch.empty_like(y)
        done = torch.zeros(self.batch if self.variant == SMRE_STANDARD else 1, dtype=torch.int32, device=y.device)
        st = torch.cuda.current_stream(y.device)
        smre_project_tol(self.handle, y.data_ptr(), out.data_ptr(), max_sweeps, tol, done.data_ptr(), st.cuda_stream)
        return out, done

    def tile_cycles(self):
        """ICD: list per shift of int32 tensors [batch, tiles_y, tiles_x] of the last project_tol."""
        import torch
        res, i = [], 0
        while True:
            try:
                ty, tx = smre_export_tile_cycles(self.handle, i)
            except SmreError:
                break
            t = torch.zeros((self.batch, ty, tx), dtype=torch.int32, device="cuda")
            smre_export_tile_cycles(self.handle, i, t.data_ptr(), torch.cuda.current_stream().cuda_stream)
            res.append(t)
            i += 1
        return res

    def project_host(self, y_np, n_sweeps, out=None, stream=0):
        y_np = np.ascontiguousarray(y_np, dtype=np.float32)
        if y_np.size != self.batch * self.H * self.W:
            raise ValueError("y has the wrong number of elements")
        if out is None:
            out = np.empty_like(y_np)
        smre_project_host(self.handle, y_np.ctypes.data, out.ctypes.data, n_sweeps, stream)
        return out

    def increments(self):
        import torch
        F, _, _ = smre_info(self.handle)
        q = torch.empty((F, self.batch, self.H, self.W), dtype=torch.float32, device="cuda")
        smre_export_increments(self.handle, q.data_ptr(), torch.cuda.current_stream().cuda_stream)
        return q

    info = property(lambda self: smre_info(self.handle))
    last_launch = property(lambda self: smre_last_launch(self.handle))

    def families(self):
        return [smre_family(self.handle, i) for i in range(self.info[0])]

    def close(self):
        if self.handle:
            smre_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
