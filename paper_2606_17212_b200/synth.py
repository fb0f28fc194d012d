"""Seeded synthetic input generators (scenes, cameras, state batches, utility pairs).

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench).  It
holds none of the method's arithmetic: it only draws the *inputs* of the method
(canonical Gaussian parameters, motion payloads, camera poses, delivered-depth
vectors, pair index lists) with numpy's PCG64 generator.  Nothing here imports
`oracle/` or the CUDA binding.

Recipes follow SURVEY.md §8(d) / DESIGN.md §4 (stand-ins for the D-NeRF / HyperNeRF
shaped workloads of BASELINE.json:configs[0..4]; the real datasets are not used and
nothing from them is reproduced).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

BASE_SEED = 26061721

# per-level delivery probabilities (BASELINE.json:configs[1])
LEVEL_PROB = (0.95, 0.8, 0.6, 0.4)

# value of the degree-0 real spherical harmonic; used only to place the DC coefficient so
# that the synthetic base colour lands in [0.1, 0.9] (an input recipe, not method code)
_SH_DC = 0.28209479177387814


@dataclass
class Scene:
    C: int
    N: int
    sh_degree: int
    R: int
    group_off: np.ndarray      # int32 [4C+1]; Gaussians sorted by (cluster, level)
    mean: np.ndarray           # f32 [N,3] canonical positions
    log_scale: np.ndarray      # f32 [N,3]
    quat: np.ndarray           # f32 [N,4] wxyz (not normalised)
    opacity_logit: np.ndarray  # f32 [N]
    sh_base: np.ndarray        # f32 [N,K,3]
    sh_res: np.ndarray         # f32 [N,K,3] level-3 payload
    motion_q: np.ndarray       # int8 [N,R,3] level-1 payload
    A0: np.ndarray             # f32 [C,3,4]
    A1: np.ndarray             # f32 [C,3,4]
    motion_scale: np.ndarray   # f32 [C]
    background: np.ndarray     # f32 [3]
    delta2: np.ndarray | None = None   # f32 [N,3] level-2 position residual of Eq. (1) (None = zero)
    delta3: np.ndarray | None = None   # f32 [N,3] level-3 position residual of Eq. (1) (None = zero)
    # per-level refinements (levels 1..3) of log-scale / raw quaternion / opacity logit, or None
    d_log_scale: np.ndarray | None = None      # f32 [3,N,3]
    d_quat: np.ndarray | None = None           # f32 [3,N,4]
    d_opacity_logit: np.ndarray | None = None  # f32 [3,N]
    d_sh: np.ndarray | None = None             # f32 [3,N,K,3] per-level colour residuals
    affine_on_covariance: bool = False         # the cluster affine also transforms Sigma (reading I4)

    @property
    def K(self) -> int:
        return (self.sh_degree + 1) ** 2

    def cluster_of(self) -> np.ndarray:
        out = np.empty(self.N, np.int32)
        for g in range(4 * self.C):
            out[self.group_off[g]:self.group_off[g + 1]] = g // 4
        return out

    def level_of(self) -> np.ndarray:
        out = np.empty(self.N, np.int8)
        for g in range(4 * self.C):
            out[self.group_off[g]:self.group_off[g + 1]] = g % 4
        return out


@dataclass
class Camera:
    R_wc: np.ndarray   # f32 [3,3] world->camera rotation (rows: right, down, forward)
    t_wc: np.ndarray   # f32 [3]
    fx: float
    fy: float
    cx: float
    cy: float
    W: int
    H: int
    znear: float = 0.2


@dataclass
class Workload:
    name: str
    scene: Scene
    frames: List[Tuple[Camera, float]]          # (camera, t) per frame
    levels: List[np.ndarray]                    # per frame: int8 [B,C] delivered depth -1..3
    # utility pairs per frame (indices into that frame's batch); may be empty arrays
    idx_without: List[np.ndarray] = field(default_factory=list)
    idx_with: List[np.ndarray] = field(default_factory=list)
    group_id: List[np.ndarray] = field(default_factory=list)
    G: int = 0


# ----------------------------------------------------------------------------- helpers
def _rng(cfg: int, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64([BASE_SEED + cfg, stream]))


def focal_from_fov(extent_px: int, fov_deg: float) -> float:
    return float(0.5 * extent_px / np.tan(np.deg2rad(0.5 * fov_deg)))


def look_at(pos, target=(0.0, 0.0, 0.0), down_hint=(0.0, 1.0, 0.0)):
    """World->camera pose, OpenCV axes (x right, y down, z forward); world +y is 'down'."""
    pos = np.asarray(pos, np.float64)
    f = np.asarray(target, np.float64) - pos
    f /= np.linalg.norm(f)
    r = np.cross(np.asarray(down_hint, np.float64), f)
    if np.linalg.norm(r) < 1e-6:
        r = np.cross(np.array([1.0, 0.0, 0.0]), f)
    r /= np.linalg.norm(r)
    d = np.cross(f, r)
    R = np.stack([r, d, f]).astype(np.float32)
    t = (-(R.astype(np.float64) @ pos)).astype(np.float32)
    return R, t


def make_camera(R, t, W, H, f) -> Camera:
    return Camera(R_wc=np.ascontiguousarray(R, np.float32), t_wc=np.ascontiguousarray(t, np.float32),
                  fx=float(np.float32(f)), fy=float(np.float32(f)),
                  cx=0.5 * W, cy=0.5 * H, W=int(W), H=int(H), znear=0.2)


def _split_counts(n_c: int, fracs) -> List[int]:
    cnt = [int(round(n_c * fr)) for fr in fracs[1:]]
    return [n_c - sum(cnt)] + cnt


def _common_attributes(rng, N, sh_degree, R):
    K = (sh_degree + 1) ** 2
    quat = rng.standard_normal((N, 4)).astype(np.float32)
    logit = rng.standard_normal(N).astype(np.float32)
    base_col = rng.uniform(0.1, 0.9, (N, 3))
    sh_base = (0.05 * rng.standard_normal((N, K, 3))).astype(np.float32)
    sh_base[:, 0, :] = ((base_col - 0.5) / _SH_DC).astype(np.float32)
    sh_res = (0.05 * rng.standard_normal((N, K, 3))).astype(np.float32)
    q = np.clip(np.rint(40.0 * rng.standard_normal((N, R, 3))), -127, 127).astype(np.int8)
    return quat, logit, sh_base, sh_res, q


def _motion(rng, C, R):
    A0 = np.zeros((C, 3, 4), np.float32)
    A0[:, :, :3] = np.eye(3, dtype=np.float32)
    A1 = rng.standard_normal((C, 3, 4))
    A1 /= np.linalg.norm(A1.reshape(C, -1), axis=1)[:, None, None]
    A1 = (A1 * (0.1 * rng.uniform(0.0, 1.0, (C, 1, 1)))).astype(np.float32)
    # residual RMS ~ 0.02: q has std 40, the cosine basis has RMS 1/sqrt(2)
    s = 0.02 / (40.0 * np.sqrt(R / 2.0)) * rng.uniform(0.5, 1.5, C)
    return A0, A1, s.astype(np.float32)


def _group_offsets(counts_per_cluster_level: np.ndarray) -> np.ndarray:
    off = np.zeros(counts_per_cluster_level.size + 1, np.int64)
    np.cumsum(counts_per_cluster_level.reshape(-1), out=off[1:])
    return off.astype(np.int32)


def sample_levels(rng, B: int, C: int, probs=LEVEL_PROB) -> np.ndarray:
    """i.i.d. per-level delivery, then dependency closure -> delivered depth in -1..3.

    Drawing the Bernoulli bits and counting the leading run of delivered levels is input
    generation (the method's own closure is `gsr_close_levels` / `orc_close_levels`)."""
    bits = rng.uniform(size=(B, C, 4)) < np.asarray(probs)[None, None, :]
    run = np.cumprod(bits, axis=2).sum(axis=2)
    return (run - 1).astype(np.int8)


def sample_masks(rng, n: int, probs=LEVEL_PROB) -> np.ndarray:
    """Raw 4-bit delivery masks (bit l = level l delivered), NOT closed."""
    bits = rng.uniform(size=(n, 4)) < np.asarray(probs)[None, :]
    return (bits * (1 << np.arange(4))[None, :]).sum(axis=1).astype(np.uint8)


def make_pairs(rng, contexts: np.ndarray):
    """For each context m pick a group g=(c, d_c+1) with d_c<3 and return (m, m∪g, group id).

    group id = 4*c + level.  Contexts with every cluster complete get cluster 0 lowered first."""
    B, C = contexts.shape
    ctx = contexts.copy()
    partner = contexts.copy()
    gid = np.empty(B, np.int32)
    for b in range(B):
        cand = np.nonzero(ctx[b] < 3)[0]
        if cand.size == 0:
            ctx[b, 0] = 2
            partner[b, 0] = 2
            cand = np.array([0])
        c = int(cand[rng.integers(cand.size)])
        partner[b, c] = ctx[b, c] + 1
        gid[b] = 4 * c + int(partner[b, c])
    return ctx, partner, gid


# ----------------------------------------------------------------------------- scenes
def scene_cfg0() -> Scene:
    """BASELINE.json:configs[0] — tiny oracle scene (4 clusters x (64 + 3x32), SH degree 1, R=4)."""
    rng = _rng(0)
    C, R, deg = 4, 4, 1
    counts = np.tile(np.array([64, 32, 32, 32]), (C, 1))
    off = _group_offsets(counts)
    N = int(off[-1])
    mean = rng.uniform(-1.0, 1.0, (N, 3)).astype(np.float32)
    log_scale = (-3.0 + 0.3 * rng.standard_normal((N, 3))).astype(np.float32)
    quat, logit, sh_base, sh_res, q = _common_attributes(rng, N, deg, R)
    A0, A1, s = _motion(rng, C, R)
    return Scene(C, N, deg, R, off, mean, log_scale, quat, logit, sh_base, sh_res, q, A0, A1, s,
                 np.zeros(3, np.float32))


def _object_scene(cfg: int, C: int, per_cluster: float, f: float, background, size_mul: float = 1.0) -> Scene:
    rng = _rng(cfg)
    R, deg = 8, 3
    n_c = np.rint(per_cluster * rng.uniform(0.8, 1.2, C)).astype(np.int64)
    counts = np.array([_split_counts(int(n), (0.60, 0.15, 0.15, 0.10)) for n in n_c])
    off = _group_offsets(counts)
    N = int(off[-1])
    centres = rng.uniform(-0.8, 0.8, (C, 3))
    cl = np.repeat(np.arange(C), counts.sum(axis=1))
    mean = np.clip(centres[cl] + 0.2 * rng.standard_normal((N, 3)), -1.0, 1.0).astype(np.float32)
    log_scale = (np.log(size_mul * 2.5 * 4.0 / f) + 0.3 * rng.standard_normal((N, 3))).astype(np.float32)
    quat, logit, sh_base, sh_res, q = _common_attributes(rng, N, deg, R)
    A0, A1, s = _motion(rng, C, R)
    return Scene(C, N, deg, R, off, mean, log_scale, quat, logit, sh_base, sh_res, q, A0, A1, s,
                 np.asarray(background, np.float32))


def scene_cfg1() -> Scene:
    """configs[1]: 32 clusters x ~3k Gaussians (~100k), SH3, R=8, white background."""
    return _object_scene(1, 32, 3125.0, focal_from_fov(800, 40.0), (1.0, 1.0, 1.0))


def scene_cfg4() -> Scene:
    """configs[4]: 128 clusters, ~1M Gaussians, SH3, R=8 (reading A23), black background."""
    return _object_scene(4, 128, 7812.5, focal_from_fov(1920, 50.0), (0.0, 0.0, 0.0))


def scene_cfg2() -> Scene:
    """configs[2]: 64 clusters, ~300k Gaussians, forward-facing, 536x960 portrait."""
    rng = _rng(2)
    C, R, deg = 64, 8, 3
    W, H = 536, 960
    f = focal_from_fov(H, 50.0)
    n_c = np.rint(4687.5 * rng.uniform(0.8, 1.2, C)).astype(np.int64)
    counts = np.array([_split_counts(int(n), (0.60, 0.15, 0.15, 0.10)) for n in n_c])
    off = _group_offsets(counts)
    N = int(off[-1])
    cl = np.repeat(np.arange(C), counts.sum(axis=1))
    # clusters = 4x4x4 grid cells in (u, v, log z)
    gu, gv, gz = cl % 4, (cl // 4) % 4, cl // 16
    u = (gu + rng.uniform(0, 1, N)) / 4.0 * 2.0 - 1.0          # [-1,1] across the frustum
    v = (gv + rng.uniform(0, 1, N)) / 4.0 * 2.0 - 1.0
    lz = np.log(0.5) + (gz + rng.uniform(0, 1, N)) / 4.0 * (np.log(10.0) - np.log(0.5))
    z = np.exp(lz)
    x = 1.1 * u * (0.5 * W / f) * z
    y = 1.1 * v * (0.5 * H / f) * z
    mean = np.stack([x, y, z], axis=1).astype(np.float32)
    log_scale = (np.log(2.5 * z / f)[:, None] + 0.3 * rng.standard_normal((N, 3))).astype(np.float32)
    quat, logit, sh_base, sh_res, q = _common_attributes(rng, N, deg, R)
    A0, A1, s = _motion(rng, C, R)
    # forward-facing scenes are metres deep: scale the motion to the depth so it stays ~pixels
    return Scene(C, N, deg, R, off, mean, log_scale, quat, logit, sh_base, sh_res, q, A0, A1, s,
                 np.zeros(3, np.float32))


# ----------------------------------------------------------------------------- cameras
def camera_cfg0() -> Tuple[Camera, float]:
    W = H = 128
    R = np.eye(3, dtype=np.float32)
    t = np.array([0.0, 0.0, 4.0], np.float32)   # camera at (0,0,-4) looking down +z
    return make_camera(R, t, W, H, focal_from_fov(W, 50.0)), 0.5


def sphere_cameras(cfg: int, n: int, W: int, H: int, fov_deg: float, radius: float = 4.0):
    rng = _rng(cfg, 1)
    f = focal_from_fov(W, fov_deg)
    cams = []
    for _ in range(n):
        v = rng.standard_normal(3)
        v /= np.linalg.norm(v)
        R, t = look_at(radius * v)
        cams.append(make_camera(R, t, W, H, f))
    return cams


def jitter_cameras(cfg: int, n: int, W: int, H: int, f: float, max_deg: float = 5.0):
    rng = _rng(cfg, 1)
    cams = []
    for _ in range(n):
        yaw, pitch = np.deg2rad(rng.uniform(-max_deg, max_deg, 2))
        Ry = np.array([[np.cos(yaw), 0, np.sin(yaw)], [0, 1, 0], [-np.sin(yaw), 0, np.cos(yaw)]])
        Rx = np.array([[1, 0, 0], [0, np.cos(pitch), -np.sin(pitch)], [0, np.sin(pitch), np.cos(pitch)]])
        cams.append(make_camera((Rx @ Ry).astype(np.float32), np.zeros(3, np.float32), W, H, f))
    return cams


# ----------------------------------------------------------------------------- workloads
def all_closed_states(C: int) -> np.ndarray:
    """All 5^C depth vectors in lexicographic order (configs[0]: 625 states for C=4)."""
    grids = np.meshgrid(*[np.arange(-1, 4)] * C, indexing="ij")
    return np.stack([g.reshape(-1) for g in grids], axis=1).astype(np.int8)


def workload_cfg0() -> Workload:
    sc = scene_cfg0()
    cam, t = camera_cfg0()
    lv = all_closed_states(sc.C)
    return Workload("cfg0_tiny", sc, [(cam, t)], [lv])


def _paired_frame_batches(cfg, scene, n_frames, B):
    """Per frame: B/2 contexts sampled with the per-level law + their B/2 'with group' partners
    (reading A25).  Batch layout: [contexts..., partners...]."""
    rng = _rng(cfg, 2)
    levels, iw, iwith, gid = [], [], [], []
    half = B // 2
    for _ in range(n_frames):
        ctx = sample_levels(rng, half, scene.C)
        ctx, partner, g = make_pairs(rng, ctx)
        levels.append(np.concatenate([ctx, partner], axis=0))
        iw.append(np.arange(half, dtype=np.int32))
        iwith.append(np.arange(half, B, dtype=np.int32))
        gid.append(g)
    return levels, iw, iwith, gid


def workload_cfg1(n_frames: int = 150, B: int = 256, scene: Scene | None = None) -> Workload:
    sc = scene if scene is not None else scene_cfg1()
    cams = sphere_cameras(1, n_frames, 800, 800, 40.0)
    frames = [(cams[n], float(np.float32((n + 0.5) / 150.0))) for n in range(n_frames)]
    levels, iw, iwith, gid = _paired_frame_batches(1, sc, n_frames, B)
    return Workload("cfg1_object_centric_800x800_B256", sc, frames, levels, iw, iwith, gid, 4 * sc.C)


def workload_train(n_frames: int = 3, B: int = 128, n_gaussians: float = 2.7e6, scene: Scene | None = None) -> Workload:
    """The size of the paper's forward-plus-backward benchmark ("2.7M primitives", up to 128 worlds, PAPER.md:148,
    238-249; its scene, resolution and masks are not given): the cfg1 recipe at 32 clusters x 84 k Gaussians, 800 x
    800, B = 128 sampled states per frame, the Gaussians' extents scaled by sqrt(N_cfg1 / N) so that the summed
    footprint — hence the depth complexity of a pixel — stays that of cfg1."""
    C = 32
    sc = scene if scene is not None else _object_scene(7, C, n_gaussians / C, focal_from_fov(800, 40.0), (1.0, 1.0, 1.0),
                                                       size_mul=float(np.sqrt(1.0e5 / n_gaussians)))
    cams = sphere_cameras(7, n_frames, 800, 800, 40.0)
    frames = [(cams[n], float(np.float32((n + 0.5) / max(n_frames, 1)))) for n in range(n_frames)]
    levels, iw, iwith, gid = _paired_frame_batches(7, sc, n_frames, B)
    return Workload("train_object_centric_800x800_B%d_N%d" % (B, sc.N), sc, frames, levels, iw, iwith, gid, 4 * sc.C)


def workload_cfg2(n_frames: int = 4, B: int = 512, scene: Scene | None = None) -> Workload:
    sc = scene if scene is not None else scene_cfg2()
    cams = jitter_cameras(2, n_frames, 536, 960, focal_from_fov(960, 50.0))
    frames = [(cams[n], float(np.float32((n + 0.5) / n_frames))) for n in range(n_frames)]
    levels, iw, iwith, gid = _paired_frame_batches(2, sc, n_frames, B)
    return Workload("cfg2_forward_facing_536x960_B512", sc, frames, levels, iw, iwith, gid, 4 * sc.C)


def workload_cfg3(n_views: int = 8, n_ctx: int = 16, scene: Scene | None = None,
                  clusters: int | None = None) -> Workload:
    """configs[3]: per view, for every (cluster c, refinement level l in 1..3) and n_ctx sampled
    contexts: the context with cluster c forced to l-1 and to l (reading A18)."""
    sc = scene if scene is not None else scene_cfg2()
    rng = _rng(3, 2)
    Cn = sc.C if clusters is None else clusters
    cams = jitter_cameras(3, n_views, 536, 960, focal_from_fov(960, 50.0))
    frames = [(cams[v], float(np.float32((v + 0.5) / n_views))) for v in range(n_views)]
    levels, iw, iwith, gid = [], [], [], []
    for _ in range(n_views):
        n_pairs = Cn * 3 * n_ctx
        ctx = sample_levels(rng, n_pairs, sc.C)
        wo, wi = ctx.copy(), ctx.copy()
        g = np.empty(n_pairs, np.int32)
        k = 0
        for c in range(Cn):
            for l in (1, 2, 3):
                for _j in range(n_ctx):
                    wo[k, c] = l - 1
                    wi[k, c] = l
                    g[k] = 4 * c + l
                    k += 1
        levels.append(np.concatenate([wo, wi], axis=0))
        iw.append(np.arange(n_pairs, dtype=np.int32))
        iwith.append(np.arange(n_pairs, 2 * n_pairs, dtype=np.int32))
        gid.append(g)
    return Workload("cfg3_utility_sweep_536x960", sc, frames, levels, iw, iwith, gid, 4 * sc.C)


def workload_cfg4(scene: Scene | None = None, B_per_t: int = 256) -> Workload:
    sc = scene if scene is not None else scene_cfg4()
    cams = sphere_cameras(4, 4, 1920, 1080, 50.0)
    ts = [0.125, 0.375, 0.625, 0.875]
    frames = [(cams[n], ts[n]) for n in range(4)]
    levels, iw, iwith, gid = _paired_frame_batches(4, sc, 4, B_per_t)
    return Workload("cfg4_stress_1920x1080_B1024", sc, frames, levels, iw, iwith, gid, 4 * sc.C)


def scaled_object_workload(seed_cfg: int, C: int, per_cluster: float, W: int, H: int, fov: float,
                           n_frames: int, B: int, background=(1.0, 1.0, 1.0)) -> Workload:
    """A reduced object-centric workload with the cfg1 recipe (parity tests at oracle-friendly sizes)."""
    sc = _object_scene(seed_cfg, C, per_cluster, focal_from_fov(W, fov), background)
    cams = sphere_cameras(seed_cfg, n_frames, W, H, fov)
    frames = [(cams[n], float(np.float32((n + 0.5) / max(n_frames, 1)))) for n in range(n_frames)]
    levels, iw, iwith, gid = _paired_frame_batches(seed_cfg, sc, n_frames, B)
    return Workload(f"scaled_cfg{seed_cfg}_{W}x{H}_B{B}", sc, frames, levels, iw, iwith, gid, 4 * sc.C)


# ----------------------------------------------------------------------------- scheduling frontier / atlas inputs
def group_raw_bytes(sc: Scene) -> np.ndarray:
    """Synthetic raw stream bytes of the 4C completion groups (input recipe): a Gaussian of
    a group costs its fp32 attributes (mean 3, log-scale 3, quaternion 4, opacity 1, base SH 3K); the
    level-1 group also carries the int8 motion coefficients (3R) of the level-0 and level-1 Gaussians,
    levels 2 and 3 those of their own Gaussians; the level-3 group also carries the fp32 SH residuals (3K)
    of every Gaussian of the cluster."""
    K = (sc.sh_degree + 1) ** 2
    attr = 4 * (11 + 3 * K)
    n = np.diff(np.asarray(sc.group_off, np.int64)).reshape(sc.C, 4)
    raw = np.zeros((sc.C, 4), np.int64)
    raw[:, 0] = n[:, 0] * attr
    raw[:, 1] = n[:, 1] * attr + (n[:, 0] + n[:, 1]) * 3 * sc.R
    raw[:, 2] = n[:, 2] * (attr + 3 * sc.R)
    raw[:, 3] = n[:, 3] * (attr + 3 * sc.R) + n.sum(axis=1) * 12 * K
    return raw.reshape(-1)


@dataclass
class AtlasWorkload:
    """Partial-state atlas + scheduling frontier on one scene.
    Per view: a utility sweep (all 4 groups of every cluster x n_ctx contexts, with / without), then
    n_atlas sampled closed states + the 5 complete prefixes, then 3 policies x len(budget_fracs) frontier
    states (built on the device from the measured utilities)."""
    name: str
    scene: Scene
    frames: List[Tuple[Camera, float]]
    sweep_levels: List[np.ndarray]       # per view int8 [2*n_pairs, C]
    idx_without: List[np.ndarray]
    idx_with: List[np.ndarray]
    group_id: List[np.ndarray]
    G: int
    atlas_levels: List[np.ndarray]       # per view int8 [n_atlas + 5, C]
    raw_bytes: np.ndarray                # int64 [4C]
    budget_fracs: Tuple[float, ...]      # budgets = floor(frac * total wire bytes)


def workload_atlas(n_views: int = 2, n_ctx: int = 8, n_atlas: int = 8192, scene: Scene | None = None,
                   W: int = 800, H: int = 800, fov: float = 40.0, seed_cfg: int = 5,
                   budget_fracs=(0.2, 0.4, 0.6, 0.8)) -> AtlasWorkload:
    """The paper samples 8,197 dependency-closed states per scene: here n_atlas = 8192
    sampled with the per-level law plus the 5 complete prefixes (all clusters at depth -1, 0, 1, 2, 3)."""
    sc = scene if scene is not None else scene_cfg1()
    rng = _rng(seed_cfg, 2)
    cams = sphere_cameras(seed_cfg, n_views, W, H, fov)
    frames = [(cams[v], float(np.float32((v + 0.5) / n_views))) for v in range(n_views)]
    sweep, iw, iwith, gid, atlas = [], [], [], [], []
    for _ in range(n_views):
        n_pairs = sc.C * 4 * n_ctx
        ctx = sample_levels(rng, n_pairs, sc.C)
        wo, wi = ctx.copy(), ctx.copy()
        g = np.empty(n_pairs, np.int32)
        k = 0
        for c in range(sc.C):
            for l in range(4):
                wo[k:k + n_ctx, c] = l - 1
                wi[k:k + n_ctx, c] = l
                g[k:k + n_ctx] = 4 * c + l
                k += n_ctx
        sweep.append(np.concatenate([wo, wi], axis=0))
        iw.append(np.arange(n_pairs, dtype=np.int32))
        iwith.append(np.arange(n_pairs, 2 * n_pairs, dtype=np.int32))
        gid.append(g)
        prefixes = np.stack([np.full(sc.C, d, np.int8) for d in range(-1, 4)])
        atlas.append(np.concatenate([sample_levels(rng, n_atlas, sc.C), prefixes], axis=0))
    return AtlasWorkload(f"atlas_{W}x{H}_B{n_atlas + 5}", sc, frames, sweep, iw, iwith, gid, 4 * sc.C, atlas,
                         group_raw_bytes(sc), tuple(budget_fracs))


def with_position_residuals(sc: Scene, seed_cfg: int = 6, sigma2: float = 0.006, sigma3: float = 0.003) -> Scene:
    """The same scene with level-2 / level-3 position residuals delta^(2), delta^(3) of Eq. (1):
    N(0, sigma^2) per coordinate, finer at level 3 (input recipe; no config of BASELINE.json defines them)."""
    import dataclasses
    rng = _rng(seed_cfg, 7)
    d2 = rng.normal(0.0, sigma2, (sc.N, 3)).astype(np.float32)
    d3 = rng.normal(0.0, sigma3, (sc.N, 3)).astype(np.float32)
    return dataclasses.replace(sc, delta2=d2, delta3=d3)


def with_attribute_refinements(sc: Scene, seed_cfg: int = 6, s_scale: float = 0.08, s_quat: float = 0.05,
                               s_logit: float = 0.3) -> Scene:
    """The same scene with per-level refinements of scale, rotation and opacity ("Scale, rotation,
    opacity, and colour use a base plus three learned refinements"): additive residuals on log-scale, raw
    quaternion and opacity logit, N(0, (s / 2^(l-1))^2) at level l = 1..3 (finer planes at later levels), and
    per-level SH colour residuals of the same decay."""
    import dataclasses
    rng = _rng(seed_cfg, 8)
    f = np.array([1.0, 0.5, 0.25])[:, None, None]
    dls = (rng.normal(0.0, 1.0, (3, sc.N, 3)) * s_scale * f).astype(np.float32)
    dq = (rng.normal(0.0, 1.0, (3, sc.N, 4)) * s_quat * f).astype(np.float32)
    dlg = (rng.normal(0.0, 1.0, (3, sc.N)) * s_logit * f[:, :, 0]).astype(np.float32)
    K = (sc.sh_degree + 1) ** 2
    dsh = (rng.normal(0.0, 1.0, (3, sc.N, K, 3)) * 0.03 * f[:, :, :, None]).astype(np.float32)
    return dataclasses.replace(sc, d_log_scale=dls, d_quat=dq, d_opacity_logit=dlg, d_sh=dsh)
