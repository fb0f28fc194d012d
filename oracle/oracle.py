"""ctypes front-end of the CPU oracle (oracle/gsr_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs — never from the product package.  It does not import the
product package either; scenes and cameras are duck-typed objects carrying numpy arrays (see
paper_2606_17212_b200/synth.py for the attribute names).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "gsr_oracle.c"
_LIB = _HERE / "libgsr_oracle.so"
# GSR_ORACLE_SANITIZE=1 (tests/test_oracle_sanitized.py): the same source under -fsanitize=address,undefined, as a
# separate library; the process must then run with libasan preloaded
if os.environ.get("GSR_ORACLE_SANITIZE") == "1":
    _LIB = _HERE / "libgsr_oracle_san.so"

CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-mfma", "-fopenmp", "-shared", "-fPIC", "-std=c11",
          "-D_GNU_SOURCE", "-Wall"]


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (no CUDA involved)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        extra = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-g"] if _LIB.name.endswith("_san.so") else []
        subprocess.check_call(["gcc", *CFLAGS, *extra, str(_SRC), "-o", str(tmp), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Scene(C.Structure):
    _fields_ = [("C", C.c_int32), ("N", C.c_int32), ("K", C.c_int32), ("R", C.c_int32),
                ("group_off", C.c_void_p), ("mean", C.c_void_p), ("cov3d", C.c_void_p),
                ("opacity", C.c_void_p), ("tau", C.c_void_p), ("sh_base", C.c_void_p),
                ("sh_res", C.c_void_p), ("motion_q", C.c_void_p), ("A0", C.c_void_p), ("A1", C.c_void_p),
                ("motion_scale", C.c_void_p), ("delta2", C.c_void_p), ("delta3", C.c_void_p),
                ("cov3d_lv", C.c_void_p), ("opacity_lv", C.c_void_p), ("tau_lv", C.c_void_p), ("d_sh", C.c_void_p),
                ("affine_cov", C.c_int32), ("pad_", C.c_int32),
                ("background", C.c_float * 3)]


class _Camera(C.Structure):
    _fields_ = [("R", C.c_float * 9), ("t", C.c_float * 3), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("W", C.c_int32), ("H", C.c_int32),
                ("znear", C.c_float)]


PROJ_DTYPE = np.dtype([("valid", np.int32), ("mu", np.float32, 3), ("z", np.float32), ("mx", np.float32),
                       ("my", np.float32), ("qa", np.float32), ("qb", np.float32), ("qc", np.float32),
                       ("cov2d", np.float32, 3), ("radius", np.int32), ("rect", np.int32, 4),
                       ("depth_bits", np.uint32), ("count", np.int32), ("rgb", np.float64, 3),
                       ("opacity", np.float32), ("tau", np.float32), ("pad_", np.float32, 2)], align=True)

_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
        _lib.orc_keys_state.restype = C.c_int64
        _lib.orc_trace_pixel.restype = C.c_int64
        _lib.orc_sizeof_proj.restype = C.c_int32
        _lib.orc_num_threads.restype = C.c_int32
        _lib.orc_project_backward_O9.restype = C.c_int32
        assert _lib.orc_sizeof_proj() == PROJ_DTYPE.itemsize, (_lib.orc_sizeof_proj(), PROJ_DTYPE.itemsize)
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    return np.ascontiguousarray(a, dtype=dtype)


# ------------------------------------------------------------------------------------------------
def close_levels(mask) -> tuple[np.ndarray, np.ndarray]:
    """O-1: raw 4-bit delivery masks -> (delivered depth int8 in -1..3, closure bitmask uint8)."""
    m = _c(mask, np.uint8)
    depth = np.empty(m.shape, np.int8)
    closure = np.empty(m.shape, np.uint8)
    lib().orc_close_levels(_p(m), C.c_int64(m.size), _p(depth), _p(closure))
    return depth, closure


def basis(t: float, R: int) -> np.ndarray:
    b = np.empty(R, np.float32)
    lib().orc_basis(C.c_float(t), C.c_int32(R), _p(b))
    return b


def sh_basis(K: int, d) -> np.ndarray:
    Y = np.zeros(16, np.float64)
    lib().orc_sh_basis(C.c_int32(K), C.c_double(d[0]), C.c_double(d[1]), C.c_double(d[2]), _p(Y))
    return Y[:K]


def sh_basis_grad(K: int, d) -> np.ndarray:
    """[3, K]: partial derivatives of the SH basis with respect to x, y, z taken as independent variables."""
    g = np.zeros((3, 16), np.float64)
    lib().orc_sh_basis_grad(C.c_int32(K), C.c_double(d[0]), C.c_double(d[1]), C.c_double(d[2]), _p(g[0]), _p(g[1]),
                            _p(g[2]))
    return g[:, :K]


def make_camera(cam) -> _Camera:
    c = _Camera()
    c.R[:] = [float(v) for v in np.asarray(cam.R_wc, np.float32).reshape(9)]
    c.t[:] = [float(v) for v in np.asarray(cam.t_wc, np.float32).reshape(3)]
    c.fx, c.fy, c.cx, c.cy = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy)
    c.W, c.H, c.znear = int(cam.W), int(cam.H), float(cam.znear)
    return c


class OracleScene:
    """Activated scene (O-0) + the per-state / per-batch oracle calls."""

    def __init__(self, sc):
        L = lib()
        self.C, self.N, self.R = int(sc.C), int(sc.N), int(sc.R)
        self.K = (int(sc.sh_degree) + 1) ** 2
        self.group_off = _c(sc.group_off, np.int32)
        self.mean = _c(sc.mean, np.float32)
        self.sh_base = _c(sc.sh_base, np.float32)
        self.sh_res = _c(sc.sh_res, np.float32)
        self.motion_q = _c(sc.motion_q, np.int8)
        self.A0 = _c(sc.A0, np.float32)
        self.A1 = _c(sc.A1, np.float32)
        self.motion_scale = _c(sc.motion_scale, np.float32)
        self.cov3d = np.empty((self.N, 6), np.float32)
        self.opacity = np.empty(self.N, np.float32)
        self.tau = np.empty(self.N, np.float32)
        ls, qt, lg = _c(sc.log_scale, np.float32), _c(sc.quat, np.float32), _c(sc.opacity_logit, np.float32)
        self.log_scale, self.quat, self.opacity_logit = ls, qt, lg   # raw parameters (O-9 differentiates them)
        L.orc_activate(C.c_int64(self.N), _p(ls), _p(qt), _p(lg), _p(self.cov3d), _p(self.opacity),
                       _p(self.tau))
        s = _Scene()
        s.C, s.N, s.K, s.R = self.C, self.N, self.K, self.R
        for name in ("group_off", "mean", "cov3d", "opacity", "tau", "sh_base", "sh_res", "motion_q", "A0",
                     "A1", "motion_scale"):
            setattr(s, name, getattr(self, name).ctypes.data)
        # optional level-2 / level-3 position residuals of Eq. (1) (None = zero)
        self.delta2 = _c(sc.delta2, np.float32) if getattr(sc, "delta2", None) is not None else None
        self.delta3 = _c(sc.delta3, np.float32) if getattr(sc, "delta3", None) is not None else None
        s.delta2 = self.delta2.ctypes.data if self.delta2 is not None else None
        s.delta3 = self.delta3.ctypes.data if self.delta3 is not None else None
        # optional per-level refinements of log-scale / quaternion / opacity logit (reading I2):
        # the attributes at delivered depth v are the base plus the residuals of levels 1..v, summed in level
        # order in binary32, then activated exactly like the base (O-0)
        refs = [getattr(sc, n, None) for n in ("d_log_scale", "d_quat", "d_opacity_logit")]
        s.cov3d_lv = s.opacity_lv = s.tau_lv = None
        self.raw_lv = None
        if any(r is not None for r in refs):
            cur = [ls.copy(), qt.copy(), lg.copy()]
            self.cov3d_lv = np.empty((4, self.N, 6), np.float32)
            self.opacity_lv = np.empty((4, self.N), np.float32)
            self.tau_lv = np.empty((4, self.N), np.float32)
            self.raw_lv = [np.empty((4,) + c.shape, np.float32) for c in cur]   # raw attributes per delivered depth
            for v in range(4):
                if v >= 1:
                    for k, r in enumerate(refs):
                        if r is not None:
                            cur[k] = (cur[k] + _c(r[v - 1], np.float32).reshape(cur[k].shape)).astype(np.float32)
                for k in range(3):
                    self.raw_lv[k][v] = cur[k]
                L.orc_activate(C.c_int64(self.N), _p(_c(cur[0], np.float32)), _p(_c(cur[1], np.float32)),
                               _p(_c(cur[2], np.float32)), _p(self.cov3d_lv[v]), _p(self.opacity_lv[v]),
                               _p(self.tau_lv[v]))
            s.cov3d_lv, s.opacity_lv, s.tau_lv = (self.cov3d_lv.ctypes.data, self.opacity_lv.ctypes.data,
                                                   self.tau_lv.ctypes.data)
        self.d_sh = _c(sc.d_sh, np.float32) if getattr(sc, "d_sh", None) is not None else None
        s.d_sh = self.d_sh.ctypes.data if self.d_sh is not None else None
        s.affine_cov = 1 if getattr(sc, "affine_on_covariance", False) else 0
        s.background[:] = [float(v) for v in np.asarray(sc.background, np.float32)]
        self._s = s

    # -- O-2/O-3
    def project(self, cam, t: float, depth) -> np.ndarray:
        d = _c(depth, np.int8)
        assert d.shape == (self.C,)
        out = np.zeros(self.N, PROJ_DTYPE)
        lib().orc_project_state(C.byref(self._s), C.byref(make_camera(cam)), C.c_float(t), _p(d), _p(out))
        return out

    # -- O-4
    def keys(self, proj: np.ndarray, cam) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
        TX = (int(cam.W) + 15) // 16
        total = int(proj["count"][proj["valid"] == 1].sum())
        tile = np.empty(max(total, 1), np.uint32)
        dbits = np.empty(max(total, 1), np.uint32)
        idx = np.empty(max(total, 1), np.int32)
        n = lib().orc_keys_state(_p(proj), C.c_int32(self.N), C.c_int32(TX), C.c_int64(total), _p(tile),
                                 _p(dbits), _p(idx))
        assert n == total
        return tile[:n], dbits[:n], idx[:n]

    # -- O-5
    def render(self, cam, t: float, depth, brute_force: bool = False, t_stop: float = 1e-4,
               want_T: bool = False, proj: np.ndarray | None = None):
        if proj is None:
            proj = self.project(cam, t, depth)
        img = np.zeros((cam.H, cam.W, 3), np.float64)
        stats = np.zeros(2, np.int64)
        Tf = np.zeros((cam.H, cam.W), np.float64) if want_T else None
        fn = lib().orc_render_O1 if brute_force else lib().orc_render_O2
        fn(C.byref(self._s), C.byref(make_camera(cam)), _p(proj), C.c_double(t_stop), _p(img), _p(stats),
           _p(Tf) if want_T else None)
        return (img, stats, Tf) if want_T else (img, stats)

    def backward(self, cam, t: float, depth, g_img, t_stop: float = 1e-4, proj: np.ndarray | None = None,
                 want_abs: bool = False):
        """orc_backward_O1: g_img = dL/d(image) double [H,W,3] of ONE state -> double [N,9] =
        (drgb[3], dopacity, dqa, dqb, dqc, dmx, dmy) per Gaussian of that state; want_abs adds the same sums
        with every per-pixel contribution in absolute value."""
        if proj is None:
            proj = self.project(cam, t, depth)
        g = _c(g_img, np.float64)
        assert g.shape == (cam.H, cam.W, 3)
        grad = np.zeros((self.N, 9), np.float64)
        gabs = np.zeros((self.N, 9), np.float64) if want_abs else None
        lib().orc_backward_O1(C.byref(self._s), C.byref(make_camera(cam)), _p(proj), C.c_double(t_stop), _p(g), _p(grad),
                              _p(gabs) if want_abs else None)
        return (grad, gabs) if want_abs else grad

    PARAM_GRADS = ("mean", "rho", "log_scale", "quat", "opacity_logit", "sh_base", "sh_res", "A", "motion_scale")
    FULL_GRADS = ("delta2", "delta3", "d_log_scale", "d_quat", "d_opacity_logit", "d_sh")

    def project_backward(self, cam, t: float, depth, g9, into: dict | None = None):
        """orc_project_backward_O9: g9 = dL/d(rgb[3], opacity, A, B, Cq, m_x, m_y) double [N,9] of ONE state (the
        output of `backward`) -> dict of double gradients with respect to the scene's parameters (PARAM_GRADS:
        mean [N,3], rho [N,3] (motion residual vector), log_scale [N,3], quat [N,4], opacity_logit [N],
        sh_base / sh_res [N,K,3], A [C,3,4] (A_c(t)), motion_scale [C]; and, where the scene has them, FULL_GRADS:
        delta2 / delta3 [N,3], d_log_scale [3,N,3], d_quat [3,N,4], d_opacity_logit [3,N], d_sh [3,N,K,3]) plus
        "margin" [N].  `into` accumulates."""
        d = _c(depth, np.int8)
        g = _c(g9, np.float64)
        assert d.shape == (self.C,) and g.shape == (self.N, 9)
        N, K = self.N, self.K
        out = into if into is not None else {
            "mean": np.zeros((N, 3)), "rho": np.zeros((N, 3)), "log_scale": np.zeros((N, 3)),
            "quat": np.zeros((N, 4)), "opacity_logit": np.zeros(N),
            "sh_base": np.zeros((N, K, 3)), "sh_res": np.zeros((N, K, 3)),
            "A": np.zeros((self.C, 3, 4)), "motion_scale": np.zeros(self.C), "margin": np.full(N, np.inf),
            "delta2": np.zeros((N, 3)), "delta3": np.zeros((N, 3)), "d_log_scale": np.zeros((3, N, 3)),
            "d_quat": np.zeros((3, N, 4)), "d_opacity_logit": np.zeros((3, N)), "d_sh": np.zeros((3, N, K, 3))}
        margin = np.full(N, np.inf)
        lv = self.raw_lv is not None
        # per-depth attribute gradients of this state (row = the state's depth of the Gaussian's cluster)
        g_ls = np.zeros((4, N, 3)) if lv else out["log_scale"]
        g_qt = np.zeros((4, N, 4)) if lv else out["quat"]
        g_lg = np.zeros((4, N)) if lv else out["opacity_logit"]
        rc = lib().orc_project_backward_O9(
            C.byref(self._s), _p(self.log_scale), _p(self.quat), _p(self.opacity_logit), C.byref(make_camera(cam)),
            C.c_float(t), _p(d), _p(g), _p(out["mean"]), _p(out["rho"]), _p(g_ls), _p(g_qt), _p(g_lg),
            _p(out["sh_base"]), _p(out["sh_res"]), _p(out["A"]), _p(out["motion_scale"]), _p(margin),
            _p(self.raw_lv[0]) if lv else None, _p(self.raw_lv[1]) if lv else None, _p(self.raw_lv[2]) if lv else None,
            _p(out["delta2"]), _p(out["delta3"]), _p(out["d_sh"]))
        if rc != 0:
            raise ValueError("orc_project_backward_O9: inconsistent optional arrays")
        if lv:   # fold: the attributes at depth v are base + levels 1..v
            for name, arr in (("log_scale", g_ls), ("quat", g_qt), ("opacity_logit", g_lg)):
                out[name] += arr.sum(0)
                for l in (1, 2, 3):
                    out["d_" + name][l - 1] += arr[l:].sum(0)
        out["margin"] = np.minimum(out["margin"], margin)
        return out

    def trace_pixel(self, cam, t: float, depth, x: int, y: int, t_stop: float = 1e-4, cap: int = 4096):
        proj = self.project(cam, t, depth)
        g = np.zeros(cap, np.int32)
        a = np.zeros(cap, np.float64)
        T = np.zeros(cap, np.float64)
        n = lib().orc_trace_pixel(C.byref(self._s), C.byref(make_camera(cam)), _p(proj), C.c_double(t_stop),
                                  C.c_int32(x), C.c_int32(y), C.c_int64(cap), _p(g), _p(a), _p(T))
        n = min(int(n), cap)
        return g[:n], a[:n], T[:n]

    def render_batch(self, cam, t: float, levels, brute_force: bool = False, t_stop: float = 1e-4):
        lv = _c(levels, np.int8)
        B = lv.shape[0]
        assert lv.shape == (B, self.C)
        img = np.zeros((B, cam.H, cam.W, 3), np.float64)
        stats = np.zeros((B, 2), np.int64)
        lib().orc_render_batch(C.byref(self._s), C.byref(make_camera(cam)), C.c_float(t), _p(lv), C.c_int32(B),
                               C.c_double(t_stop), _p(img), _p(stats), C.c_int32(1 if brute_force else 0))
        return img, stats


# -- O-6
def distortion(imgs, ref) -> tuple[np.ndarray, np.ndarray]:
    im = _c(imgs, np.float64)
    B = im.shape[0]
    rf = _c(ref, np.float64).reshape(-1)
    im = im.reshape(B, -1)
    assert im.shape[1] == rf.size
    mse = np.empty(B, np.float64)
    psnr = np.empty(B, np.float64)
    lib().orc_distortion(_p(im), _p(rf), C.c_int32(B), C.c_int64(rf.size), _p(mse), _p(psnr))
    return mse, psnr


# -- O-7
UTIL_FIELDS = ("mean_mse", "q10_mse", "std_mse", "risk_mse", "mean_db", "q10_db", "std_db", "risk_db", "count")


def group_utility(mse, psnr_db, idx_without, idx_with, group_id, G: int):
    m, p = _c(mse, np.float64), _c(psnr_db, np.float64)
    a, b, g = _c(idx_without, np.int32), _c(idx_with, np.int32), _c(group_id, np.int32)
    n = a.size
    dm = np.empty(max(n, 1), np.float64)
    dd = np.empty(max(n, 1), np.float64)
    util = np.zeros((G, 9), np.float64)
    lib().orc_group_utility(_p(m), _p(p), _p(a), _p(b), _p(g), C.c_int64(n), C.c_int32(G), _p(dm), _p(dd),
                            _p(util))
    return dm[:n], dd[:n], util


def num_threads() -> int:
    return int(lib().orc_num_threads())
