"""GPU parity of the backward pass (ms_backward; S:Sec.8(f) NEXT-4) against the fp64 oracle of oracle/mso_grad.c on the
same seeded inputs and the same dL/dC.  Bar: every gradient within 1e-2 of the largest gradient of
its family (weights, centres, semi-axes, quaternions).  The bar is set by the FORWARD geometry, not by the backward
arithmetic: the GPU differentiates the render it runs -- canonical fp32 geometry -- while the oracle's
backward is fp64 throughout; a sample position that differs by 1 ulp of the eye distance moves the top encoding band's
phase by 2^(L-1) pi times that (1e-4 at L = 4), and grazing chords carry 1/sqrt(disc).  Measured: <= 5e-3 at L = 4,
<= 6e-4 at L = 2 (held to 2e-3 there, which a dropped or mis-signed term of the chain rule would break); at L = 6 the
top band's phase error is four times that of L = 4 (measured 1.4e-2; held to 3e-2).  Wide or deep random networks
amplify the same position error (64 and 128 wide at L = 2: up to 8e-3 on the geometry families, set by one or two
grazing chords of the scene), so the tight bar is held by every kernel variant on networks up to 32 wide and the 1e-2
bar on the wide ones."""
import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth

pytestmark = pytest.mark.gpu

TOL_REL = 1e-2
TOL_REL_L2 = 2e-3
TOL_REL_L6 = 3e-2


def _api():
    from paper_2606_03877_b200 import api
    return api


def with_biases(sc, mlp, seed):
    """non-zero biases: keeps samples off the exact ReLU kink (pre-activation == bias == 0), where one-sided
    derivatives are a convention (tests/test_oracle_grad_pins.py)"""
    rng = np.random.default_rng(seed + 77)
    w = sc.weights.copy()
    off = 0
    for i, o in mlp.layer_dims:
        off += i * o
        w[:, off:off + o] += rng.uniform(-0.3, 0.3, (w.shape[0], o)).astype(np.float32)
        off += o
    return synth.custom_scene(sc.center, sc.quat, sc.scale, w, mlp)


def compare(sc, cam, H, W, K, t_stop=1e-4, seed=0, tol=TOL_REL):
    api = _api()
    rng = np.random.default_rng(seed)
    g_in = rng.normal(size=(H * W, 3))
    ref = mso.loss_grad_f64(sc, cam, H, W, K, g_in=g_in, t_stop=t_stop)
    gs = api.Scene(sc)
    d_rgb = torch.from_numpy(g_in.astype(np.float32)).cuda().reshape(H, W, 3)
    gw, gc, gq, gsc = gs.backward(cam, H, W, K, d_rgb, t_stop=t_stop)
    torch.cuda.synchronize()
    out = {}
    for name, g, r in (("weights", gw, ref["g_weights"]), ("center", gc, ref["g_center"]),
                       ("quat", gq, ref["g_quat"]), ("scale", gsc, ref["g_scale"])):
        g = g.cpu().numpy().astype(np.float64)
        scale = np.abs(r).max()
        assert scale > 0
        err = np.abs(g - r).max() / scale
        out[name] = err
        assert err <= tol, (name, err, scale)
    # accumulation: a second call adds the same gradient again
    gs.backward(cam, H, W, K, d_rgb, t_stop=t_stop, grads=(gw, gc, gq, gsc))
    torch.cuda.synchronize()
    assert np.abs(gw.cpu().numpy() - 2 * ref["g_weights"]).max() <= 2 * tol * np.abs(ref["g_weights"]).max()
    return out


def test_backward_cfg1_shape():
    """BASELINE.json configs[0]'s scene and MLP (27-32-32-4, K = 8), 48 x 48"""
    cfg = synth.shrink(synth.CONFIGS["cfg1"], 48, 48)
    sc = with_biases(synth.make_scene(cfg), cfg.mlp, 0)
    compare(sc, synth.make_cameras(cfg)[0], 48, 48, cfg.K)


@pytest.mark.parametrize("seed,viewdir,width,nh,L", [(3, 0, 8, 2, 2), (5, 1, 16, 3, 2), (7, 1, 64, 3, 4), (11, 1, 32, 2, 2),
                                                     (13, 0, 24, 2, 2), (9, 0, 128, 3, 2), (9, 0, 128, 3, 6),
                                                     (15, 1, 64, 4, 2), (17, 0, 16, 1, 2), (19, 0, 64, 2, 2),
                                                     (21, 0, 32, 3, 2), (23, 0, 64, 1, 2)])
def test_backward_overlapping_primitives(seed, viewdir, width, nh, L):
    """heavily overlapping supports (interleaved samples of several primitives on every ray), ragged image,
    with and without the view-direction input: CFG3's 30-64-64-64-4, CFG4's 39-128-128-128-4 (two 64-sample passes
    per row block), widths served by the generic one-thread-per-sample kernel (8, 24; 64 with four hidden layers)"""
    mlp = synth.MLPSpec(L, viewdir, nh, width, 0, False)
    cfg = synth.SceneConfig(f"b{seed}", seed, 9, 0.6, 0.35, 0.8, mlp, 37, 23, 50.0, 3.0, 5)
    sc = with_biases(synth.make_scene(cfg), mlp, seed)
    compare(sc, synth.make_cameras(cfg)[0], cfg.height, cfg.width, cfg.K, seed=seed,
            tol=TOL_REL_L6 if L == 6 else (TOL_REL_L2 if L == 2 and width <= 32 else TOL_REL))


def test_backward_stops_at_the_early_termination():
    """opaque scene: samples behind the stop carry no gradient on either side (Q9).  A ray whose T lands within
    rounding of the threshold may stop one sample apart (Q25): its gradient differs by < t_stop, far inside the bar."""
    sc, cfg = synth.dense_scene()
    sc = with_biases(sc, cfg.mlp, 1)
    cam = synth.make_cameras(cfg)[0]
    compare(sc, cam, 40, 48, cfg.K, t_stop=1e-4)
    compare(sc, cam, 40, 48, cfg.K, t_stop=0.0)


def test_backward_refuses_what_it_does_not_cover():
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["next1"], 32, 18)       # contact-point mode: no backward
    gs = api.Scene(synth.make_scene(cfg))
    with pytest.raises(api.MsError) as e:
        gs.backward(synth.make_cameras(cfg)[0], 18, 32, 1, torch.zeros((18, 32, 3), device="cuda"))
    assert e.value.code == -4
