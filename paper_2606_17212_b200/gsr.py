"""Thin ctypes binding of libgsr.so (include/gsr.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device
memory and streams only.  There is NO CPU fallback: importing this module without the built
extension, or calling it without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libgsr.so"

GSR_OK, GSR_E_INVALID_ARG, GSR_E_INVALID_LEVEL, GSR_E_WORKSPACE_TOO_SMALL, GSR_E_CUDA = 0, -1, -2, -3, -4


class GsrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gsr error {code}: {msg}")
        self.code = code


class SceneDesc(C.Structure):
    _fields_ = [("C", C.c_int32), ("N", C.c_int32), ("sh_degree", C.c_int32), ("R", C.c_int32),
                ("group_off", C.c_void_p), ("mean", C.c_void_p), ("log_scale", C.c_void_p), ("quat", C.c_void_p),
                ("opacity_logit", C.c_void_p), ("sh_base", C.c_void_p), ("sh_res", C.c_void_p),
                ("motion_q", C.c_void_p), ("A0", C.c_void_p), ("A1", C.c_void_p), ("motion_scale", C.c_void_p),
                ("background", C.c_float * 3), ("delta2", C.c_void_p), ("delta3", C.c_void_p),
                ("d_log_scale", C.c_void_p), ("d_quat", C.c_void_p), ("d_opacity_logit", C.c_void_p),
                ("d_sh", C.c_void_p), ("affine_on_covariance", C.c_int32)]


class CameraC(C.Structure):
    _fields_ = [("R_wc", C.c_float * 9), ("t_wc", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("W", C.c_int32), ("H", C.c_int32), ("znear", C.c_float)]


class LossModel(C.Structure):
    _fields_ = [("p_iid", C.c_double), ("p_gb", C.c_double), ("p_bg", C.c_double), ("e_good", C.c_double),
                ("e_bad", C.c_double), ("seed", C.c_uint64)]


UTILITY_DTYPE = np.dtype([(n, np.float64) for n in
                          ("mean_mse", "q10_mse", "std_mse", "risk_mse", "mean_db", "q10_db", "std_db", "risk_db",
                           "count")])

_lib = None


def lib():
    """Loads libgsr.so; fails loudly if it has not been built (python -m paper_2606_17212_b200.build)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_17212_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, i32, i64, sz, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_size_t, C.c_float
        L.gsr_last_error.restype = C.c_char_p
        L.gsr_version.restype = C.c_char_p
        L.gsr_load_scene.argtypes = [C.POINTER(SceneDesc), C.POINTER(vp)]
        L.gsr_free_scene.argtypes = [vp]
        L.gsr_free_scene.restype = None
        L.gsr_workspace_bytes.argtypes = [vp, C.POINTER(CameraC), i32]
        L.gsr_workspace_bytes.restype = sz
        L.gsr_workspace_bytes_ex.argtypes = [vp, C.POINTER(CameraC), i32, i64]
        L.gsr_workspace_bytes_ex.restype = sz
        L.gsr_render_states.argtypes = [vp, C.POINTER(CameraC), f32, vp, i32, vp, vp, sz, vp]
        L.gsr_render_states_ex.argtypes = [vp, C.POINTER(CameraC), f32, vp, i32, vp, vp, vp, vp, vp, sz, vp]
        L.gsr_workspace_status.argtypes = [vp, C.POINTER(i64), vp]
        L.gsr_distortion_workspace_bytes.argtypes = [i32, i32, i32]
        L.gsr_distortion_workspace_bytes.restype = sz
        L.gsr_distortion.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, sz, vp]
        L.gsr_distortion_static.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp]
        L.gsr_distortion_static_max_partials.argtypes = []
        L.gsr_distortion_static_max_partials.restype = i64
        L.gsr_group_utility.argtypes = [vp, vp, vp, vp, vp, i32, i32, vp, vp, vp, vp]
        L.gsr_group_utility_b.argtypes = [vp, vp, i32, vp, vp, vp, i32, i32, vp, vp, vp, vp]
        L.gsr_index_status.argtypes = [vp]
        L.gsr_num_records.argtypes = [vp]
        L.gsr_num_records.restype = i64
        L.gsr_render_backward.argtypes = [vp, vp, vp, vp, i32, vp, vp]
        L.gsr_distortion_backward.argtypes = [vp, vp, i32, i32, i32, vp, C.c_double, vp, vp, sz, vp]
        L.gsr_distortion_backward_workspace_bytes.argtypes = [i32, i32]
        L.gsr_distortion_backward_workspace_bytes.restype = sz
        L.gsr_objective_weights.argtypes = [vp, i32, C.c_double, C.c_double, C.c_double, vp, vp, i32, C.c_double, vp, vp]
        L.gsr_flicker_backward.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, vp, vp]
        L.gsr_project_backward_full.argtypes = [vp, C.POINTER(CameraC), f32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gsr_project_backward.argtypes = [vp, C.POINTER(CameraC), f32, vp, vp, vp, vp, vp, vp]
        L.gsr_close_levels.argtypes = [vp, i64, vp, vp, vp]
        L.gsr_frame_workspace_bytes.argtypes = [vp, C.POINTER(CameraC), i32, i32, i32, i32]
        L.gsr_frame_workspace_bytes.restype = sz
        L.gsr_utility_frame_host.argtypes = [vp, C.POINTER(CameraC), f32, vp, i32, vp, vp, vp, i32, i32, vp, vp, vp,
                                             i32, vp, vp, sz, vp]
        L.gsr_debug_projection.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.gsr_debug_keys.argtypes = [vp, vp, i32, i64, vp, vp, vp, C.POINTER(i64), vp]
        L.gsr_debug_state_counts.argtypes = [vp, vp, vp, vp]
        L.gsr_debug_closure.argtypes = [vp, vp, vp, vp]
        L.gsr_set_option.argtypes = [C.c_char_p, i32]
        L.gsr_render_states_vs_full.argtypes = [vp, C.POINTER(CameraC), f32, vp, i32, vp, vp, vp, vp, vp, sz, vp]
        L.gsr_debug_pair_counts.argtypes = [vp, vp, vp, vp]
        L.gsr_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(i32)]
        L.gsr_launch_count.restype = i64
        L.gsr_profile_read_phases.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(i32)]
        L.gsr_measure_fp32_peak.argtypes = [C.POINTER(C.c_double), vp]
        L.gsr_group_wire_bytes.argtypes = [vp, i32, vp, vp]
        L.gsr_frontier_order.argtypes = [vp, vp, i32, i32, vp, vp, vp]
        L.gsr_frontier_states.argtypes = [vp, vp, i32, vp, i32, vp, vp, vp, vp]
        L.gsr_state_bytes.argtypes = [vp, i32, i32, vp, vp, vp]
        L.gsr_best_state_under_budget.argtypes = [vp, vp, i32, vp, i32, vp, vp]
        L.gsr_distortion_ssim.argtypes = [vp, vp, i32, i32, i32, vp, vp, vp, vp, sz, vp]
        L.gsr_flicker.argtypes = [vp, vp, vp, vp, i32, i32, i32, vp, vp, sz, vp]
        L.gsr_risk_reduce.argtypes = [vp, i32, i32, C.c_double, i32, vp, vp]
        L.gsr_prefix_monotonicity.argtypes = [vp, vp, vp, i32, vp, vp, vp]
        L.gsr_prefix_monotonicity_n.argtypes = [vp, i32, vp, vp, i32, vp, vp, vp]
        L.gsr_delivery_workspace_bytes.argtypes = [i32]
        L.gsr_delivery_workspace_bytes.restype = sz
        L.gsr_sample_delivery.argtypes = [vp, vp, i32, C.POINTER(LossModel), vp, i32, i32, vp, vp, vp, sz, vp]
        _lib = L
    return _lib


def _check(rc: int):
    if rc != GSR_OK:
        raise GsrError(rc, lib().gsr_last_error().decode())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("gsr needs a CUDA device (no CPU fallback)")
    return torch


def _stream():
    return C.c_void_p(_torch().cuda.current_stream().cuda_stream)


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


def _hp(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _dp(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def camera_struct(cam) -> CameraC:
    if isinstance(cam, CameraC):
        return cam
    c = CameraC()
    c.R_wc[:] = [float(v) for v in np.asarray(cam.R_wc, np.float32).reshape(9)]
    c.t_wc[:] = [float(v) for v in np.asarray(cam.t_wc, np.float32).reshape(3)]
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    c.W, c.H, c.znear = int(cam.W), int(cam.H), float(cam.znear)
    return c


def set_option(name: str, value: int):
    _check(lib().gsr_set_option(name.encode(), int(value)))


def profile_read():
    """gsr_profile_read -> (sum of compositing-kernel ms, launches) since the last read."""
    ms, n = C.c_double(0), C.c_int32(0)
    _check(lib().gsr_profile_read(C.byref(ms), C.byref(n)))
    return float(ms.value), int(n.value)


def profile_read_phases():
    """gsr_profile_read_phases -> (projection ms, binning + sort ms, frames) since the last read."""
    a, b, n = C.c_double(0), C.c_double(0), C.c_int32(0)
    _check(lib().gsr_profile_read_phases(C.byref(a), C.byref(b), C.byref(n)))
    return float(a.value), float(b.value), int(n.value)


def launch_count() -> int:
    return int(lib().gsr_launch_count())


def measure_fp32_peak() -> float:
    _torch()
    tf = C.c_double(0)
    _check(lib().gsr_measure_fp32_peak(C.byref(tf), _stream()))
    return float(tf.value)


class Scene:
    """gsr_load_scene / gsr_free_scene.  `sc` carries the arrays of gsr_scene_desc as numpy attributes."""

    def __init__(self, sc):
        _torch().cuda.init()
        self.C, self.N, self.R, self.sh_degree = int(sc.C), int(sc.N), int(sc.R), int(sc.sh_degree)
        keep = dict(group_off=_np(sc.group_off, np.int32), mean=_np(sc.mean, np.float32),
                    log_scale=_np(sc.log_scale, np.float32), quat=_np(sc.quat, np.float32),
                    opacity_logit=_np(sc.opacity_logit, np.float32), sh_base=_np(sc.sh_base, np.float32),
                    sh_res=_np(sc.sh_res, np.float32), motion_q=_np(sc.motion_q, np.int8),
                    A0=_np(sc.A0, np.float32), A1=_np(sc.A1, np.float32),
                    motion_scale=_np(sc.motion_scale, np.float32))
        d = SceneDesc()
        d.C, d.N, d.sh_degree, d.R = self.C, self.N, self.sh_degree, self.R
        for k, v in keep.items():
            setattr(d, k, v.ctypes.data)
        d.background[:] = [float(v) for v in np.asarray(sc.background, np.float32)]
        d.affine_on_covariance = 1 if getattr(sc, "affine_on_covariance", False) else 0
        self.V = 2                                   # projected records per Gaussian
        # optional position residual levels of Eq. (1) and per-level scale / rotation / opacity refinements
        for name in ("delta2", "delta3", "d_log_scale", "d_quat", "d_opacity_logit", "d_sh"):
            a = getattr(sc, name, None)
            if a is not None:
                keep[name] = _np(a, np.float32)
                setattr(d, name, keep[name].ctypes.data)
                self.V = 4
        h = C.c_void_p()
        _check(lib().gsr_load_scene(C.byref(d), C.byref(h)))
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            lib().gsr_free_scene(self.handle)
            self.handle = None

    __del__ = close

    # ---- workspace
    def workspace_bytes(self, cam, B: int, key_capacity: int = 0) -> int:
        n = lib().gsr_workspace_bytes_ex(self.handle, C.byref(camera_struct(cam)), int(B), int(key_capacity))
        if n == 0:
            raise GsrError(GSR_E_INVALID_ARG, "gsr_workspace_bytes: invalid arguments")
        return int(n)

    def new_workspace(self, cam, B: int, key_capacity: int = 0):
        torch = _torch()
        return torch.empty(self.workspace_bytes(cam, B, key_capacity), dtype=torch.uint8, device="cuda")

    # ---- hot path
    def render_states(self, cam, t: float, levels, out=None, workspace=None, ref=None, mse=None, psnr=None,
                      want_images: bool = True):
        """gsr_render_states(_ex).  levels: cuda int8 [B,C].  Returns (out, mse, psnr) (entries may be None)."""
        torch = _torch()
        B = int(levels.shape[0])
        assert levels.dtype == torch.int8 and levels.is_cuda and levels.is_contiguous()
        assert levels.shape[1] == self.C
        if workspace is None:
            workspace = self.new_workspace(cam, B)
        if out is None and want_images:
            out = torch.empty((B, cam.H, cam.W, 3), dtype=torch.float32, device="cuda")
        if ref is not None:
            assert ref.dtype == torch.float32 and ref.is_cuda and ref.is_contiguous()
            if mse is None:
                mse = torch.empty(B, dtype=torch.float64, device="cuda")
            if psnr is None:
                psnr = torch.empty(B, dtype=torch.float32, device="cuda")
        _check(lib().gsr_render_states_ex(self.handle, C.byref(camera_struct(cam)), C.c_float(t), _dp(levels), B,
                                          _dp(out), _dp(ref), _dp(mse), _dp(psnr), _dp(workspace),
                                          workspace.numel(), _stream()))
        return out, mse, psnr

    def render_states_vs_full(self, cam, t: float, levels, workspace, ref_out, mse, psnr, out=None):
        """gsr_render_states_vs_full: all buffers are caller-provided device tensors (nothing allocated)."""
        B = int(levels.shape[0])
        _check(lib().gsr_render_states_vs_full(self.handle, C.byref(camera_struct(cam)), C.c_float(t), _dp(levels),
                                               B, _dp(out), _dp(ref_out), _dp(mse), _dp(psnr), _dp(workspace),
                                               workspace.numel(), _stream()))

    def num_records(self) -> int:
        return int(lib().gsr_num_records(self.handle))

    def render_backward(self, workspace, images, dL_dimages, grad=None):
        """gsr_render_backward after a forward call on `workspace`: images, dL_dimages cuda float32 [B,H,W,3] ->
        cuda float32 [num_records, 12] (see include/gsr.h for the columns); `grad` reuses a buffer."""
        torch = _torch()
        for t in (images, dL_dimages):
            assert t.dtype == torch.float32 and t.is_cuda and t.is_contiguous() and t.shape == images.shape
        if grad is None:
            grad = torch.empty((self.num_records(), 12), dtype=torch.float32, device="cuda")
        assert grad.dtype == torch.float32 and grad.is_cuda and grad.is_contiguous() and tuple(grad.shape) == (self.num_records(), 12)
        _check(lib().gsr_render_backward(self.handle, _dp(workspace), _dp(images), _dp(dL_dimages),
                                         int(images.shape[0]), _dp(grad), _stream()))
        return grad

    def project_backward(self, cam, t: float, grad_records, out=None):
        """gsr_project_backward: grad_records cuda float32 [num_records, 12] (from render_backward, same cam and t)
        -> dict of cuda float32 gradients: gauss [N,14] (mean 3, rho 3, log_scale 3, quat 4, opacity_logit),
        sh_base / sh_res [N,K,3], cluster [C,13] (A_c(t) 3x4, s_c); `out` reuses the dict of a previous call."""
        torch = _torch()
        assert grad_records.dtype == torch.float32 and grad_records.is_cuda and grad_records.is_contiguous()
        assert tuple(grad_records.shape) == (self.num_records(), 12)
        K = (self.sh_degree + 1) ** 2
        if out is None:
            out = {"gauss": torch.empty((self.N, 14), dtype=torch.float32, device="cuda"),
                   "sh_base": torch.empty((self.N, K, 3), dtype=torch.float32, device="cuda"),
                   "sh_res": torch.empty((self.N, K, 3), dtype=torch.float32, device="cuda"),
                   "cluster": torch.empty((self.C, 13), dtype=torch.float32, device="cuda")}
        for name, shape in (("gauss", (self.N, 14)), ("sh_base", (self.N, K, 3)), ("sh_res", (self.N, K, 3)),
                            ("cluster", (self.C, 13))):
            v = out[name]
            assert v.dtype == torch.float32 and v.is_cuda and v.is_contiguous() and tuple(v.shape) == shape
        _check(lib().gsr_project_backward(self.handle, C.byref(camera_struct(cam)), float(t), _dp(grad_records),
                                          _dp(out["gauss"]), _dp(out["sh_base"]), _dp(out["sh_res"]),
                                          _dp(out["cluster"]), _stream()))
        return out

    def project_backward_full(self, cam, t: float, grad_records, out=None):
        """gsr_project_backward_full: like project_backward, for every scene; adds "delta" [N,6], "attr" [3,N,8]
        (log_scale 3, quat 4, opacity_logit per refinement level) and "d_sh" [3,N,K,3]."""
        torch = _torch()
        assert grad_records.dtype == torch.float32 and grad_records.is_cuda and grad_records.is_contiguous()
        assert tuple(grad_records.shape) == (self.num_records(), 12)
        K = (self.sh_degree + 1) ** 2
        e = lambda *shape: torch.empty(shape, dtype=torch.float32, device="cuda")
        if out is None:                                      # `out` reuses the dict of a previous call
            out = {"gauss": e(self.N, 14), "sh_base": e(self.N, K, 3), "sh_res": e(self.N, K, 3), "cluster": e(self.C, 13),
                   "delta": e(self.N, 6), "attr": e(3, self.N, 8), "d_sh": e(3, self.N, K, 3)}
        _check(lib().gsr_project_backward_full(self.handle, C.byref(camera_struct(cam)), float(t), _dp(grad_records),
                                               _dp(out["gauss"]), _dp(out["sh_base"]), _dp(out["sh_res"]),
                                               _dp(out["cluster"]), _dp(out["delta"]), _dp(out["attr"]), _dp(out["d_sh"]),
                                               _stream()))
        return out

    def debug_pair_counts(self, workspace) -> np.ndarray:
        c = np.zeros(3, np.int64)
        _check(lib().gsr_debug_pair_counts(self.handle, _dp(workspace), _hp(c), _stream()))
        return c

    def status(self, workspace) -> int:
        """gsr_workspace_status: synchronises; raises on a latched device-side error; returns #keys."""
        n = C.c_int64(0)
        _check(lib().gsr_workspace_status(_dp(workspace), C.byref(n), _stream()))
        return int(n.value)

    # ---- host-buffer convenience call
    def utility_frame_host(self, cam, t: float, levels_host: np.ndarray, idx_without, idx_with, group_id, G: int,
                           workspace=None, want_images: bool = False, materialise: bool = False, bufs=None):
        """gsr_utility_frame_host.  want_images copies the [B,H,W,3] images back to the host; materialise
        only writes them on the device (what gsr_render_states does).  `bufs` = (mse, psnr, util) host
        arrays to reuse (e.g. views of pinned memory)."""
        torch = _torch()
        lv = _np(levels_host, np.int8)
        B = lv.shape[0]
        iwo, iw, gid = _np(idx_without, np.int32), _np(idx_with, np.int32), _np(group_id, np.int32)
        n_pairs = int(iwo.size)
        camc = camera_struct(cam)
        mat = int(bool(want_images or materialise))
        need = lib().gsr_frame_workspace_bytes(self.handle, C.byref(camc), B, n_pairs, G, mat)
        if workspace is None or workspace.numel() < need:
            workspace = torch.empty(need, dtype=torch.uint8, device="cuda")
        if bufs is None:
            mse, psnr, util = np.empty(B, np.float64), np.empty(B, np.float32), np.zeros(max(G, 1), UTILITY_DTYPE)
        else:
            mse, psnr, util = bufs
        out = np.empty((B, cam.H, cam.W, 3), np.float32) if want_images else None
        _check(lib().gsr_utility_frame_host(self.handle, C.byref(camc), C.c_float(t), _hp(lv), B, _hp(iwo), _hp(iw),
                                            _hp(gid), n_pairs, G, _hp(mse), _hp(psnr), _hp(util), mat,
                                            _hp(out) if out is not None else None, _dp(workspace),
                                            workspace.numel(), _stream()))
        return mse, psnr, util[:G], out, workspace

    # ---- debug / parity exports
    def debug_projection(self, workspace) -> dict:
        n = self.V * self.N
        o = dict(valid=np.zeros(n, np.uint8), radius=np.zeros(n, np.int32), rect=np.zeros((n, 4), np.int32),
                 depth_bits=np.zeros(n, np.uint32), count=np.zeros(n, np.int32), mean2d=np.zeros((n, 2), np.float32),
                 conic=np.zeros((n, 3), np.float32), rgb_base=np.zeros((n, 3), np.float32),
                 rgb_res=np.zeros((n, 3), np.float32))
        _check(lib().gsr_debug_projection(self.handle, _dp(workspace), _hp(o["valid"]), _hp(o["radius"]),
                                          _hp(o["rect"]), _hp(o["depth_bits"]), _hp(o["count"]), _hp(o["mean2d"]),
                                          _hp(o["conic"]), _hp(o["rgb_base"]), _hp(o["rgb_res"]), _stream()))
        return o

    def debug_keys(self, workspace, b: int, cap: int):
        tile = np.zeros(max(cap, 1), np.uint32)
        dbits = np.zeros(max(cap, 1), np.uint32)
        gi = np.zeros(max(cap, 1), np.int32)
        n = C.c_int64(0)
        _check(lib().gsr_debug_keys(self.handle, _dp(workspace), int(b), int(cap), _hp(tile), _hp(dbits), _hp(gi),
                                    C.byref(n), _stream()))
        m = min(int(n.value), cap)
        return tile[:m], dbits[:m], gi[:m], int(n.value)

    def debug_state_counts(self, workspace, B: int) -> np.ndarray:
        c = np.zeros(B, np.int64)
        _check(lib().gsr_debug_state_counts(self.handle, _dp(workspace), _hp(c), _stream()))
        return c

    def debug_closure(self, workspace, B: int) -> np.ndarray:
        d = np.zeros((B, self.C), np.int8)
        _check(lib().gsr_debug_closure(self.handle, _dp(workspace), _hp(d), _stream()))
        return d


def distortion(imgs, ref, workspace=None):
    """gsr_distortion: imgs cuda f32 [B,H,W,3], ref cuda f32 [H,W,3] -> (mse f64 [B], psnr f32 [B]) on device."""
    torch = _torch()
    B, H, W = int(imgs.shape[0]), int(imgs.shape[1]), int(imgs.shape[2])
    assert imgs.dtype == torch.float32 and imgs.is_contiguous() and ref.is_contiguous()
    need = lib().gsr_distortion_workspace_bytes(B, H, W)
    if workspace is None or workspace.numel() < need:
        workspace = torch.empty(need, dtype=torch.uint8, device="cuda")
    mse = torch.empty(B, dtype=torch.float64, device="cuda")
    psnr = torch.empty(B, dtype=torch.float32, device="cuda")
    _check(lib().gsr_distortion(_dp(imgs), _dp(ref), B, H, W, _dp(mse), _dp(psnr), _dp(workspace),
                                workspace.numel(), _stream()))
    return mse, psnr


def distortion_static(imgs, ref, mse, psnr):
    """gsr_distortion_static: like `distortion`, but the library allocates nothing — the outputs mse (cuda f64 [B])
    and psnr (cuda f32 [B]) are the caller's, the scratch is built into the library (B * tiles <= 2^20)."""
    torch = _torch()
    B, H, W = int(imgs.shape[0]), int(imgs.shape[1]), int(imgs.shape[2])
    assert imgs.dtype == torch.float32 and imgs.is_cuda and imgs.is_contiguous()
    assert ref.dtype == torch.float32 and ref.is_cuda and ref.is_contiguous() and tuple(ref.shape) == (H, W, 3)
    assert mse.dtype == torch.float64 and mse.is_cuda and mse.is_contiguous() and mse.numel() == B
    assert psnr.dtype == torch.float32 and psnr.is_cuda and psnr.is_contiguous() and psnr.numel() == B
    _check(lib().gsr_distortion_static(_dp(imgs), _dp(ref), B, H, W, _dp(mse), _dp(psnr), _stream()))
    return mse, psnr


def group_utility(mse, psnr, idx_without, idx_with, group_id, G: int, want_deltas: bool = True):
    """gsr_group_utility on device tensors.  Returns (util structured array [G], delta_mse, delta_db)."""
    torch = _torch()
    n_pairs = int(idx_without.numel())
    util = torch.zeros((max(G, 1), 9), dtype=torch.float64, device="cuda")
    dm = torch.empty(max(n_pairs, 1), dtype=torch.float64, device="cuda") if want_deltas else None
    dd = torch.empty(max(n_pairs, 1), dtype=torch.float64, device="cuda") if want_deltas else None
    for t in (idx_without, idx_with, group_id):
        assert t.dtype == torch.int32 and t.is_cuda and t.is_contiguous()
    _check(lib().gsr_group_utility_b(_dp(mse), _dp(psnr), int(mse.numel()), _dp(idx_without), _dp(idx_with),
                                     _dp(group_id), n_pairs, G, _dp(util), _dp(dm), _dp(dd), _stream()))
    index_status()
    u = util[:G].cpu().numpy().view(UTILITY_DTYPE).reshape(G)
    return u, (dm[:n_pairs] if dm is not None else None), (dd[:n_pairs] if dd is not None else None)


def group_utility_into(mse, psnr, idx_without, idx_with, group_id, G: int, util_out):
    """gsr_group_utility_b with a caller-provided cuda float64 [G,9] output (no allocation, no sync; range errors of
    the pair lists stay latched until index_status() is called)."""
    _check(lib().gsr_group_utility_b(_dp(mse), _dp(psnr), int(mse.numel()), _dp(idx_without), _dp(idx_with),
                                     _dp(group_id), int(idx_without.numel()), G, _dp(util_out), None, None, _stream()))


def index_status():
    """gsr_index_status: synchronises the stream; raises if a device-side index check refused an entry."""
    _check(lib().gsr_index_status(_stream()))


def close_levels(mask):
    """gsr_close_levels: cuda uint8 masks -> (depth int8, closure uint8) on device."""
    torch = _torch()
    assert mask.dtype == torch.uint8 and mask.is_cuda and mask.is_contiguous()
    depth = torch.empty(mask.shape, dtype=torch.int8, device="cuda")
    closure = torch.empty(mask.shape, dtype=torch.uint8, device="cuda")
    _check(lib().gsr_close_levels(_dp(mask), mask.numel(), _dp(depth), _dp(closure), _stream()))
    return depth, closure


# ---- scheduling frontier / partial-state atlas (include/gsr.h): marshalling only
POLICY_UTILITY, POLICY_NOMINAL, POLICY_BYTE_GREEDY = 0, 1, 2


def group_wire_bytes(raw_bytes):
    """gsr_group_wire_bytes: cuda int64 [4C] -> cuda int64 [4C]."""
    torch = _torch()
    assert raw_bytes.dtype == torch.int64 and raw_bytes.is_cuda and raw_bytes.is_contiguous()
    wire = torch.empty_like(raw_bytes)
    _check(lib().gsr_group_wire_bytes(_dp(raw_bytes), raw_bytes.numel() // 4, _dp(wire), _stream()))
    return wire


def frontier_order(score, wire, policy: int):
    """gsr_frontier_order -> (order int32 [4C], cum_bytes int64 [4C]) on device."""
    torch = _torch()
    n = wire.numel()
    assert wire.dtype == torch.int64 and wire.is_cuda and wire.is_contiguous()
    if score is not None:
        assert score.dtype == torch.float64 and score.is_cuda and score.is_contiguous() and score.numel() == n
    order = torch.empty(n, dtype=torch.int32, device="cuda")
    cum = torch.empty(n, dtype=torch.int64, device="cuda")
    _check(lib().gsr_frontier_order(_dp(score), _dp(wire), n // 4, int(policy), _dp(order), _dp(cum), _stream()))
    return order, cum


def frontier_states(order, wire, budgets, levels_out=None):
    """gsr_frontier_states -> (levels int8 [nb, C], used int64 [nb], n_groups int32 [nb]) on device."""
    torch = _torch()
    Cn, nb = wire.numel() // 4, budgets.numel()
    assert budgets.dtype == torch.int64 and budgets.is_cuda and order.dtype == torch.int32
    levels = levels_out if levels_out is not None else torch.empty((nb, Cn), dtype=torch.int8, device="cuda")
    used = torch.empty(nb, dtype=torch.int64, device="cuda")
    ng = torch.empty(nb, dtype=torch.int32, device="cuda")
    _check(lib().gsr_frontier_states(_dp(order), _dp(wire), Cn, _dp(budgets), nb, _dp(levels), _dp(used), _dp(ng),
                                     _stream()))
    return levels, used, ng


def state_bytes(levels, wire, out=None):
    """gsr_state_bytes: cuda int8 [B, C] -> cuda int64 [B]."""
    torch = _torch()
    B, Cn = int(levels.shape[0]), int(levels.shape[1])
    assert levels.dtype == torch.int8 and levels.is_cuda and levels.is_contiguous() and wire.numel() == 4 * Cn
    if out is None:
        out = torch.empty(B, dtype=torch.int64, device="cuda")
    _check(lib().gsr_state_bytes(_dp(levels), B, Cn, _dp(wire), _dp(out), _stream()))
    return out


def best_state_under_budget(psnr, bytes_per_state, budgets, out=None):
    """gsr_best_state_under_budget -> cuda int32 [nb]."""
    torch = _torch()
    assert psnr.dtype == torch.float32 and bytes_per_state.dtype == torch.int64 and budgets.dtype == torch.int64
    if out is None:
        out = torch.empty(budgets.numel(), dtype=torch.int32, device="cuda")
    _check(lib().gsr_best_state_under_budget(_dp(psnr), _dp(bytes_per_state), psnr.numel(), _dp(budgets),
                                             budgets.numel(), _dp(out), _stream()))
    return out


# ---- richer distortion / risk reductions (include/gsr.h): marshalling only
RISK_DTYPE = np.dtype([(n, np.float64) for n in ("mean", "cvar", "quantile", "worst", "count")])


def _tile_workspace(B, H, W, workspace):
    torch = _torch()
    need = lib().gsr_distortion_workspace_bytes(B, H, W)
    if workspace is None or workspace.numel() < need:
        workspace = torch.empty(need, dtype=torch.uint8, device="cuda")
    return workspace


def distortion_ssim(imgs, ref, mse=None, workspace=None):
    """gsr_distortion_ssim -> (ssim f64 [B], d_mix f64 [B] or None) on device."""
    torch = _torch()
    B, H, W = int(imgs.shape[0]), int(imgs.shape[1]), int(imgs.shape[2])
    assert imgs.dtype == torch.float32 and imgs.is_contiguous() and ref.is_contiguous()
    workspace = _tile_workspace(B, H, W, workspace)
    ssim = torch.empty(B, dtype=torch.float64, device="cuda")
    dmix = torch.empty(B, dtype=torch.float64, device="cuda") if mse is not None else None
    _check(lib().gsr_distortion_ssim(_dp(imgs), _dp(ref), B, H, W, _dp(mse), _dp(ssim), _dp(dmix), _dp(workspace),
                                     workspace.numel(), _stream()))
    return ssim, dmix


def distortion_backward(imgs, ref, weight=None, lambda_ssim: float = 0.20, out=None, workspace=None):
    """gsr_distortion_backward: d/d(imgs) of sum_b weight[b] (MSE_b + lambda_ssim (1 - SSIM_b)) -> cuda float32
    [B,H,W,3].  weight: cuda float64 [B] or None (= 1 per state); workspace: cuda uint8 of
    gsr_distortion_backward_workspace_bytes(H, W) bytes (allocated here if None)."""
    torch = _torch()
    B, H, W = int(imgs.shape[0]), int(imgs.shape[1]), int(imgs.shape[2])
    assert imgs.dtype == torch.float32 and imgs.is_cuda and imgs.is_contiguous()
    assert ref.dtype == torch.float32 and ref.is_cuda and ref.is_contiguous() and tuple(ref.shape) == (H, W, 3)
    if weight is not None:
        assert weight.dtype == torch.float64 and weight.is_cuda and weight.is_contiguous() and weight.numel() == B
    if out is None:
        out = torch.empty_like(imgs)
    assert out.dtype == torch.float32 and out.is_cuda and out.is_contiguous() and out.shape == imgs.shape
    if workspace is None:
        workspace = torch.empty(int(lib().gsr_distortion_backward_workspace_bytes(H, W)), dtype=torch.uint8, device="cuda")
    _check(lib().gsr_distortion_backward(_dp(imgs), _dp(ref), B, H, W, _dp(weight), float(lambda_ssim), _dp(out),
                                         _dp(workspace), workspace.numel(), _stream()))
    return out


def objective_weights(d, w_mean: float = 1.0, w_cvar: float = 0.30, alpha: float = 0.05, idx_prev=None, idx_next=None,
                      w_mono: float = 0.0, out=None):
    """gsr_objective_weights: d cuda float64 [n] -> dL/dD_b of w_mean mean + w_cvar CVaR_alpha + w_mono M, cuda float64 [n]."""
    torch = _torch()
    assert d.dtype == torch.float64 and d.is_cuda and d.is_contiguous()
    n = int(d.numel())
    n_pairs = 0 if idx_prev is None else int(idx_prev.numel())
    if n_pairs:
        for t in (idx_prev, idx_next):
            assert t.dtype == torch.int32 and t.is_cuda and t.is_contiguous() and t.numel() == n_pairs
    if out is None:
        out = torch.empty(n, dtype=torch.float64, device="cuda")
    _check(lib().gsr_objective_weights(_dp(d), n, float(w_mean), float(w_cvar), float(alpha), _dp(idx_prev) if n_pairs else None,
                                       _dp(idx_next) if n_pairs else None, n_pairs, float(w_mono), _dp(out), _stream()))
    return out


def flicker_backward(imgs_t1, imgs_t2, ref_t1, ref_t2, weight=None):
    """gsr_flicker_backward -> (g_t1, g_t2) cuda float32 [B,H,W,3]."""
    torch = _torch()
    B, H, W = int(imgs_t1.shape[0]), int(imgs_t1.shape[1]), int(imgs_t1.shape[2])
    for t in (imgs_t1, imgs_t2, ref_t1, ref_t2):
        assert t.dtype == torch.float32 and t.is_cuda and t.is_contiguous()
    g1, g2 = torch.empty_like(imgs_t1), torch.empty_like(imgs_t2)
    _check(lib().gsr_flicker_backward(_dp(imgs_t1), _dp(imgs_t2), _dp(ref_t1), _dp(ref_t2), B, H, W, _dp(weight),
                                      _dp(g1), _dp(g2), _stream()))
    return g1, g2


def flicker(imgs_t1, imgs_t2, ref_t1, ref_t2, workspace=None):
    """gsr_flicker -> f64 [B] on device."""
    torch = _torch()
    B, H, W = int(imgs_t1.shape[0]), int(imgs_t1.shape[1]), int(imgs_t1.shape[2])
    for t in (imgs_t1, imgs_t2, ref_t1, ref_t2):
        assert t.dtype == torch.float32 and t.is_cuda and t.is_contiguous()
    workspace = _tile_workspace(B, H, W, workspace)
    out = torch.empty(B, dtype=torch.float64, device="cuda")
    _check(lib().gsr_flicker(_dp(imgs_t1), _dp(imgs_t2), _dp(ref_t1), _dp(ref_t2), B, H, W, _dp(out), _dp(workspace),
                             workspace.numel(), _stream()))
    return out


def risk_reduce(values, alpha: float, upper_tail: bool):
    """gsr_risk_reduce on a cuda float64 / float32 vector -> structured numpy record (synchronises)."""
    torch = _torch()
    assert values.is_cuda and values.is_contiguous() and values.dtype in (torch.float64, torch.float32)
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    _check(lib().gsr_risk_reduce(_dp(values), 1 if values.dtype == torch.float32 else 0, values.numel(),
                                 C.c_double(alpha), int(bool(upper_tail)), _dp(out), _stream()))
    return out.cpu().numpy().view(RISK_DTYPE)[0]


def prefix_monotonicity(d, idx_prev, idx_next):
    """gsr_prefix_monotonicity -> (M, violations) (synchronises)."""
    torch = _torch()
    assert d.dtype == torch.float64 and idx_prev.dtype == torch.int32 and idx_next.dtype == torch.int32
    m = torch.zeros(1, dtype=torch.float64, device="cuda")
    v = torch.zeros(1, dtype=torch.int32, device="cuda")
    _check(lib().gsr_prefix_monotonicity_n(_dp(d), int(d.numel()), _dp(idx_prev), _dp(idx_next), idx_prev.numel(),
                                           _dp(m), _dp(v), _stream()))
    index_status()
    return float(m.item()), int(v.item())


# ---- delivery-mask sampler (include/gsr.h): marshalling only
def sample_delivery(raw_bytes, order, model: dict, W: int, packet_budget=None, world0: int = 0, want_levels=True):
    """gsr_sample_delivery -> (mask uint8 [W, C], levels int8 [W, C] or None) on device.
    model: dict(p_iid, p_gb, p_bg, e_good, e_bad, seed)."""
    torch = _torch()
    Cn = raw_bytes.numel() // 4
    assert raw_bytes.dtype == torch.int64 and order.dtype == torch.int32 and raw_bytes.is_cuda and order.is_cuda
    if packet_budget is not None:
        assert packet_budget.dtype == torch.int32 and packet_budget.is_cuda and packet_budget.numel() == W
    m = LossModel(float(model["p_iid"]), float(model["p_gb"]), float(model["p_bg"]), float(model["e_good"]),
                  float(model["e_bad"]), int(model["seed"]))
    mask = torch.empty((W, Cn), dtype=torch.uint8, device="cuda")
    levels = torch.empty((W, Cn), dtype=torch.int8, device="cuda") if want_levels else None
    ws = torch.empty(lib().gsr_delivery_workspace_bytes(Cn), dtype=torch.uint8, device="cuda")
    _check(lib().gsr_sample_delivery(_dp(raw_bytes), _dp(order), Cn, C.byref(m), _dp(packet_budget), int(W),
                                     int(world0), _dp(mask), _dp(levels), _dp(ws), ws.numel(), _stream()))
    return mask, levels
