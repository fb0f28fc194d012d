"""GPU mirrors of the oracle pins P21-P24 (tests/test_oracle_pins.py): the four scenes that exercise the SH view
direction, the alpha cap 0.99, the Jacobian clamp 1.3 lim and the lambda floor 0.1 go through the C ABI and are
compared with the oracle at the bars of DESIGN.md §3.8 — projection integers and decision-feeding fp32 bit-exact,
colours <= 2e-6, pixels <= 2e-4 — and with the closed forms the pins use."""
import numpy as np
import pytest

from tests.test_gpu_parity import PIX_TOL, _check_projection, _render, gsr, torch_mod  # noqa: F401  (fixtures)
from tests.test_oracle_pins import (pin_scene_alpha_cap, pin_scene_jacobian_clamp, pin_scene_lambda_floor,
                                    pin_scene_sh_view_direction)

pytestmark = pytest.mark.gpu


def _pixels_vs_oracle(gsr, torch_mod, oracle_mod, scn, cam):
    scene = gsr.Scene(scn)
    lv = np.zeros((1, scn.C), np.int8)
    out, _, _, _ = _render(torch_mod, scene, cam, 0.0, lv)
    img, _ = oracle_mod.OracleScene(scn).render(cam, 0.0, lv[0])
    got = out[0].cpu().numpy()
    assert np.abs(got - img).max() <= PIX_TOL
    scene.close()
    return got


def test_sh_view_direction(gsr, torch_mod, oracle_mod):
    scn, cam, eye, mu, k = pin_scene_sh_view_direction()
    _check_projection(gsr, torch_mod, oracle_mod, scn, cam, 0.0)
    scene = gsr.Scene(scn)
    _, _, _, ws = _render(torch_mod, scene, cam, 0.0, np.zeros((1, 1), np.int8))
    rgb = scene.debug_projection(ws)["rgb_base"][0]          # record 2*0 + 0: the depth-0 variant
    d = mu.astype(np.float32).astype(np.float64) - eye
    d /= np.linalg.norm(d)
    expect = 0.5 + np.sqrt(3.0 / (4.0 * np.pi)) * k * d
    assert np.abs(rgb - expect).max() < 4e-6                  # fp32 colour on the GPU + fp32 rounding of t_wc
    scene.close()
    _pixels_vs_oracle(gsr, torch_mod, oracle_mod, scn, cam)


@pytest.mark.parametrize("bg", [(0.0, 0.0, 0.0), (1.0, 1.0, 1.0)])
def test_alpha_cap(gsr, torch_mod, oracle_mod, bg):
    scn, cam, col = pin_scene_alpha_cap(bg)
    _check_projection(gsr, torch_mod, oracle_mod, scn, cam, 0.0)
    got = _pixels_vs_oracle(gsr, torch_mod, oracle_mod, scn, cam)
    assert np.abs(got[32, 32] - (0.99 * np.array(col) + 0.01 * np.array(bg))).max() < 1e-5


def test_jacobian_clamp(gsr, torch_mod, oracle_mod):
    scn, cam, lim, s, f, z = pin_scene_jacobian_clamp()
    _check_projection(gsr, torch_mod, oracle_mod, scn, cam, 0.0)        # conic, radius, rectangle bit-exact
    _pixels_vs_oracle(gsr, torch_mod, oracle_mod, scn, cam)


def test_lambda_floor(gsr, torch_mod, oracle_mod):
    scn, cam = pin_scene_lambda_floor()
    _check_projection(gsr, torch_mod, oracle_mod, scn, cam, 0.0)
    scene = gsr.Scene(scn)
    _, _, _, ws = _render(torch_mod, scene, cam, 0.0, np.zeros((1, 1), np.int8))
    P = scene.debug_projection(ws)
    assert P["radius"][0] == 5 and P["rect"][0].tolist() == [3, 3, 5, 5]
    scene.close()
    _pixels_vs_oracle(gsr, torch_mod, oracle_mod, scn, cam)
