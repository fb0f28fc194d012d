"""Frames in flight (include/gsr.h: "the scene handle is immutable after load and usable from
several streams"): frames rendered concurrently on separate CUDA streams, each with its own workspace and
outputs, give BITWISE the results of the same frames rendered one at a time — through the device call
(gsr_render_states_vs_full + gsr_group_utility) and through the blocking host call driven from threads."""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from paper_2606_17212_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def gsr(torch_mod):
    from paper_2606_17212_b200 import gsr as G
    G.lib()
    return G


@pytest.fixture(scope="module")
def workload():
    return synth.scaled_object_workload(41, C=8, per_cluster=900.0, W=200, H=152, fov=40.0, n_frames=6, B=48)


def _bufs(torch, scene, cam, B, G):
    return {"ws": scene.new_workspace(cam, B),
            "out": torch.empty((B, cam.H, cam.W, 3), dtype=torch.float32, device="cuda"),
            "ref": torch.empty((cam.H, cam.W, 3), dtype=torch.float32, device="cuda"),
            "mse": torch.empty(B, dtype=torch.float64, device="cuda"),
            "psnr": torch.empty(B, dtype=torch.float32, device="cuda"),
            "util": torch.zeros((max(G, 1), 9), dtype=torch.float64, device="cuda")}


def test_frames_on_concurrent_streams_equal_serial_bitwise(gsr, torch_mod, workload):
    torch = torch_mod
    wl = workload
    scene = gsr.Scene(wl.scene)
    cam0, _ = wl.frames[0]
    B, G = wl.levels[0].shape[0], wl.G
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).cuda()
    lv = [dev(l, np.int8) for l in wl.levels]
    iwo, iw, gid = ([dev(a, np.int32) for a in x] for x in (wl.idx_without, wl.idx_with, wl.group_id))
    cams = [gsr.camera_struct(c) for c, _ in wl.frames]
    ts = [float(t) for _, t in wl.frames]
    n = len(cams)

    def frame(b, f):
        scene.render_states_vs_full(cams[f], ts[f], lv[f], b["ws"], b["ref"], b["mse"], b["psnr"], out=b["out"])
        if G > 0:
            gsr.group_utility_into(b["mse"], b["psnr"], iwo[f], iw[f], gid[f], G, b["util"])

    # serial: one frame at a time on the current stream
    b0 = _bufs(torch, scene, cam0, B, G)
    want = []
    for f in range(n):
        frame(b0, f)
        torch.cuda.synchronize()
        want.append({k: b0[k].clone() for k in ("out", "ref", "mse", "psnr", "util")})
    # pipelined: frame f on stream f mod 3; several rounds so that kernels of different frames really overlap
    F = 3
    lanes = [dict(_bufs(torch, scene, cam0, B, G), stream=torch.cuda.Stream()) for _ in range(F)]
    for rounds in range(3):
        got = [None] * n
        for f0 in range(0, n, F):
            for i in range(F):
                if f0 + i < n:
                    with torch.cuda.stream(lanes[i]["stream"]):
                        frame(lanes[i], f0 + i)
            torch.cuda.synchronize()
            for i in range(F):
                if f0 + i < n:
                    got[f0 + i] = {k: lanes[i][k].clone() for k in ("out", "ref", "mse", "psnr", "util")}
        for f in range(n):
            for k in want[f]:
                assert torch.equal(got[f][k], want[f][k]), (rounds, f, k)
    for lane in lanes:
        scene.status(lane["ws"])
    scene.close()


def test_host_call_from_threads_equals_serial_bitwise(gsr, torch_mod, workload):
    torch = torch_mod
    wl = workload
    scene = gsr.Scene(wl.scene)
    n, G = len(wl.frames), wl.G

    def call(f, ws=None):
        cam, t = wl.frames[f]
        mse, psnr, util, _, ws = scene.utility_frame_host(cam, t, wl.levels[f], wl.idx_without[f], wl.idx_with[f],
                                                          wl.group_id[f], G, workspace=ws, materialise=True)
        return mse.copy(), psnr.copy(), np.array(util, copy=True), ws

    want = [call(f)[:3] for f in range(n)]
    streams = [torch.cuda.Stream() for _ in range(3)]

    def task(f):
        with torch.cuda.stream(streams[f % 3]):
            return call(f)[:3]

    with ThreadPoolExecutor(max_workers=3) as pool:
        for _ in range(2):
            got = list(pool.map(task, range(n)))
            for f in range(n):
                assert np.array_equal(got[f][0], want[f][0]) and np.array_equal(got[f][1], want[f][1])
                assert got[f][2].tobytes() == want[f][2].tobytes()
    scene.close()


def test_options_belong_to_the_calling_thread(gsr, torch_mod, workload):
    """include/gsr.h: "state_block" and "dedup" steer the calls of the thread that set them.  Three threads render the
    same frames at the same time with different state blocks (one of them without dedup); every one of them gets
    the bits of the serial default render, and the main thread's options are untouched.  "profile" is refused
    while a call is in flight and never makes another thread's calls record events."""
    import threading
    torch = torch_mod
    wl = workload
    scene = gsr.Scene(wl.scene)
    n = len(wl.frames)
    dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a, dt)).cuda()
    lv = [dev(l, np.int8) for l in wl.levels]
    cams = [gsr.camera_struct(c) for c, _ in wl.frames]
    ts = [float(t) for _, t in wl.frames]
    cam0, _ = wl.frames[0]
    B = wl.levels[0].shape[0]

    def render_all(b):
        res = []
        for f in range(n):
            scene.render_states_vs_full(cams[f], ts[f], lv[f], b["ws"], b["ref"], b["mse"], b["psnr"], out=b["out"])
            torch.cuda.current_stream().synchronize()
            res.append((b["out"].clone(), b["mse"].clone()))
        return res

    want = render_all(_bufs(torch, scene, cam0, B, 0))
    settings = [(4, 1), (16, 1), (8, 0)]
    got, errors = [None] * len(settings), []
    start = threading.Barrier(len(settings))

    def worker(k):
        try:
            torch.cuda.set_device(0)
            S, dedup = settings[k]
            gsr.set_option("state_block", S)
            gsr.set_option("dedup", dedup)
            b = _bufs(torch, scene, cam0, B, 0)
            start.wait()
            with torch.cuda.stream(torch.cuda.Stream()):
                for _ in range(3):
                    got[k] = render_all(b)
        except Exception as e:  # noqa: BLE001
            errors.append(repr(e))

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(len(settings))]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    assert not errors, errors
    for k in range(len(settings)):
        for f in range(n):
            assert torch.equal(got[k][f][0], want[f][0]) and torch.equal(got[k][f][1], want[f][1]), (settings[k], f)
    # the main thread still renders with its own (default) options, and profiling stays with the thread that asked
    gsr.set_option("profile", 1)
    done = []
    th = threading.Thread(target=lambda: done.append(render_all(_bufs(torch, scene, cam0, B, 0))))
    th.start()
    th.join()
    ms, launches = gsr.profile_read()
    assert launches == 0                                   # the other thread's calls recorded nothing
    render_all(_bufs(torch, scene, cam0, B, 0))
    ms, launches = gsr.profile_read()
    assert launches == 2 * n                               # reference + batch per frame, this thread's calls
    gsr.set_option("profile", 0)
    scene.close()
