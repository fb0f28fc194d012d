"""Small hand-built scenes for the oracle pins and the GPU parity tests (inputs only)."""
import numpy as np

from paper_2606_17212_b200 import synth

Y0 = 0.5 * np.sqrt(1.0 / np.pi)


def tiny_scene(means, scales, quats=None, logits=None, colors=None, levels=None, clusters=None, C=None,
               sh_degree=0, R=1, background=(0.0, 0.0, 0.0), A0=None, A1=None, motion_q=None,
               motion_scale=None, sh_base=None, sh_res=None):
    """Scene from explicit per-Gaussian values.  Gaussians are re-sorted by (cluster, level)."""
    means = np.asarray(means, np.float64).reshape(-1, 3)
    N = means.shape[0]
    scales = np.broadcast_to(np.asarray(scales, np.float64), (N, 3)) if np.ndim(scales) < 2 else np.asarray(scales)
    quats = np.tile([1.0, 0, 0, 0], (N, 1)) if quats is None else np.asarray(quats, np.float64).reshape(N, 4)
    logits = np.zeros(N) if logits is None else np.broadcast_to(np.asarray(logits, np.float64), (N,))
    levels = np.zeros(N, np.int64) if levels is None else np.asarray(levels, np.int64)
    clusters = np.zeros(N, np.int64) if clusters is None else np.asarray(clusters, np.int64)
    C = int(clusters.max()) + 1 if C is None else C
    K = (sh_degree + 1) ** 2
    if sh_base is None:
        sh_base = np.zeros((N, K, 3))
        col = np.full((N, 3), 0.5) if colors is None else np.broadcast_to(np.asarray(colors, np.float64), (N, 3))
        sh_base[:, 0, :] = (col - 0.5) / Y0
    sh_res = np.zeros((N, K, 3)) if sh_res is None else np.asarray(sh_res)
    motion_q = np.zeros((N, R, 3), np.int8) if motion_q is None else np.asarray(motion_q, np.int8)
    order = np.lexsort((np.arange(N), levels, clusters))
    counts = np.zeros((C, 4), np.int64)
    for c, l in zip(clusters, levels):
        counts[c, l] += 1
    off = np.zeros(4 * C + 1, np.int32)
    off[1:] = np.cumsum(counts.reshape(-1))
    if A0 is None:
        A0 = np.zeros((C, 3, 4)); A0[:, :, :3] = np.eye(3)
    A1 = np.zeros((C, 3, 4)) if A1 is None else A1
    motion_scale = np.ones(C) if motion_scale is None else motion_scale
    f32 = lambda a: np.ascontiguousarray(a, np.float32)
    sc = synth.Scene(C=C, N=N, sh_degree=sh_degree, R=R, group_off=off, mean=f32(means[order]),
                     log_scale=f32(np.log(scales)[order]), quat=f32(quats[order]),
                     opacity_logit=f32(logits[order]), sh_base=f32(np.asarray(sh_base)[order]),
                     sh_res=f32(sh_res[order]), motion_q=np.ascontiguousarray(motion_q[order]),
                     A0=f32(A0), A1=f32(A1), motion_scale=f32(motion_scale), background=f32(background))
    return sc, order


def axis_camera(W=128, H=128, f=100.0, z0=4.0, cx=None, cy=None):
    """Camera at (0,0,-z0) looking down +z, R = I."""
    cam = synth.make_camera(np.eye(3, dtype=np.float32), np.array([0, 0, z0], np.float32), W, H, f)
    if cx is not None:
        cam.cx = cx
    if cy is not None:
        cam.cy = cy
    return cam
