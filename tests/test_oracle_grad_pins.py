"""Pins of the backward-pass oracle (oracle/mso_grad.c; S:Sec.8(f) NEXT-4), written before any backward kernel.
What fixes it, other than itself: (1) its fp64 forward is the render of mso.c (canonical fp32 geometry) to rounding;
(2) central finite differences of that forward in every parameter family -- MLP weights of every layer, centres,
semi-axes, quaternions (the losses need dL/dtheta and dL/d(mu, s, q)); (3) the closed form of one constant
primitive, C = c (1 - exp(-sigma L)) (north_star; Eq.6), differentiated by hand; (4) no gradient behind the
early stop."""
import numpy as np
import pytest

from oracle import mso
from paper_2606_03877_b200 import synth


def tiny(seed=3, n=7, K=4, W=14, H=10, mlp=None, sigma_bias=0.5):
    mlp = mlp or synth.MLPSpec(2, 0, 2, 8, 0, False)
    cfg = synth.SceneConfig(f"g{seed}", seed, n, 0.6, 0.35, 0.8, mlp, W, H, 50.0, 3.0, K, sigma_bias=sigma_bias)
    sc = synth.make_scene(cfg)
    # non-zero biases: with the generator's zero biases a sample whose first hidden layer is all off sits EXACTLY on
    # the ReLU kink of the second (pre-activation = bias = 0), where the one-sided derivative 0 the oracle takes and a
    # central difference disagree
    rng = np.random.default_rng(seed + 77)
    w = sc.weights.copy()
    off = 0
    for i, o in mlp.layer_dims:
        off += i * o
        w[:, off:off + o] += rng.uniform(-0.3, 0.3, (w.shape[0], o)).astype(np.float32)
        off += o
    sc = synth.custom_scene(sc.center, sc.quat, sc.scale, w, mlp)
    return sc, synth.make_cameras(cfg)[0], cfg


def test_fp64_forward_is_the_oracle_render():
    for mlp in (synth.MLPSpec(2, 0, 2, 8, 0, False), synth.MLPSpec(4, 1, 3, 16, 0, False)):
        sc, cam, cfg = tiny(mlp=mlp)
        o_rgb, o_alpha, _, st = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, cfg.K, tile=0)
        r = mso.loss_grad_f64(sc, cam, cfg.height, cfg.width, cfg.K, want_grad=False)
        assert st.n_intervals > 100
        d = np.abs(r["rgb"] - o_rgb)                         # fp32 vs fp64 geometry: grazing chords lose digits
        assert d.max() < 1e-4 and d.mean() < 2e-6 and np.median(d[o_rgb > 0]) < 2e-6


def fd(sc, cam, cfg, name, arr, idx, h, target, t_stop=1e-4):
    kw = {k: None for k in ("center", "quat", "scale", "weights")}
    out = []
    for sgn in (+1, -1):
        a = arr.copy()
        a.flat[idx] += sgn * h
        kw[name] = a
        out.append(mso.loss_grad_f64(sc, cam, cfg.height, cfg.width, cfg.K, target=target, want_grad=False,
                                     t_stop=t_stop, **kw)["loss"])
    return (out[0] - out[1]) / (2 * h)


@pytest.mark.parametrize("seed,viewdir", [(3, 0), (5, 1)])
def test_gradients_against_central_finite_differences(seed, viewdir):
    sc, cam, cfg = tiny(seed=seed, mlp=synth.MLPSpec(2, viewdir, 2, 8, 0, False))
    rng = np.random.default_rng(seed)
    H, W = cfg.height, cfg.width
    target = rng.uniform(0, 1, (H * W, 3))
    r = mso.loss_grad_f64(sc, cam, H, W, cfg.K, target=target)
    assert r["loss"] > 1.0
    fams = {"center": (np.asarray(sc.center, np.float64), r["g_center"], 1e-6),
            "scale": (np.asarray(sc.scale, np.float64), r["g_scale"], 1e-6),
            "quat": (np.asarray(sc.quat, np.float64), r["g_quat"], 1e-6),
            "weights": (np.asarray(sc.weights, np.float64), r["g_weights"], 1e-6)}
    for name, (arr, g, h) in fams.items():
        idxs = np.arange(arr.size) if arr.size <= 40 else rng.choice(arr.size, 60, replace=False)
        scale = max(1.0, np.abs(g).max())
        worst = 0.0
        for i in idxs:
            num = fd(sc, cam, cfg, name, arr, int(i), h, target)
            worst = max(worst, abs(num - g.flat[int(i)]))
        # the L1 loss is piecewise smooth: a pixel whose C - target changes sign inside +-h would break it; none does
        assert worst <= 2e-5 * scale, (name, worst, scale)
    # every parameter family is live (a dropped term would leave zeros)
    assert all(np.abs(fams[k][1]).max() > 1e-3 for k in fams)
    # the quaternion gradient is tangent to the unit sphere (q enters only through q / |q|)
    assert np.abs((r["g_quat"] * np.asarray(sc.quat, np.float64)).sum(axis=1)).max() < 1e-9


def test_constant_primitive_closed_form():
    """One sphere of radius s whose MLP outputs constants: through its centre C = c (1 - exp(-sigma 2 s)),
    c = sigmoid(b_rgb), sigma = softplus(b_sigma) -- for every K (north_star).  By hand:
    dC/db_sigma = c 2s exp(-2 s sigma) sigmoid(b_sigma);  dC/db_rgb = c (1 - c) (1 - exp(-2 s sigma));
    dC/ds (all three semi-axes together) = c sigma 2 exp(-2 s sigma)."""
    mlp = synth.MLPSpec(1, 0, 1, 4, 0, False)
    b = np.array([0.3, -0.2, 0.9, 0.7], np.float32).astype(np.float64)    # the values the float32 scene arrays hold
    w = synth.constant_mlp_weights(mlp, b)
    s = float(np.float32(0.4))
    sc = synth.custom_scene([[0, 0, 0.0]], [[1, 0, 0, 0]], [[s, s, s]], w[None], mlp)
    W = H = 1                                                  # the single pixel looks down the optical axis
    cam = synth.pinhole(W, H, 40.0, synth.look_at([0, 0, 3.0]))
    g_in = np.array([[1.0, 0.0, 0.0]])                         # dL/dC = e_r: picks the red channel
    for K in (1, 3, 8):
        r = mso.loss_grad_f64(sc, cam, H, W, K, g_in=g_in)
        c = 1 / (1 + np.exp(-b[:3]))
        sigma = np.log1p(np.exp(b[3]))
        ex = np.exp(-2 * s * sigma)
        assert np.allclose(r["rgb"][0], c * (1 - ex), rtol=0, atol=1e-12)
        gw = r["g_weights"][0]
        assert np.isclose(gw[-1], c[0] * 2 * s * ex / (1 + np.exp(-b[3])), rtol=1e-10)     # b_sigma
        assert np.isclose(gw[-4], c[0] * (1 - c[0]) * (1 - ex), rtol=1e-10)                # b_r
        assert gw[-3] == 0.0 and gw[-2] == 0.0                                             # b_g, b_b: not in the loss
        assert np.isclose(r["g_scale"][0].sum(), c[0] * sigma * 2 * ex, rtol=1e-9)
        assert np.abs(r["g_center"][0][:2]).max() < 1e-9       # the chord through the centre is stationary sideways


def test_no_gradient_behind_the_early_stop():
    """Opaque front primitive, a second one well behind it: every ray through both stops inside the first, so the
    second receives no gradient at all; with the threshold off it does (Q9)."""
    mlp = synth.MLPSpec(1, 0, 1, 4, 0, False)
    w = synth.constant_mlp_weights(mlp, np.array([0.2, 0.1, -0.3, 12.0]))
    sc = synth.custom_scene([[0, 0, 1.0], [0, 0, -1.0]], [[1, 0, 0, 0]] * 2, [[0.9, 0.9, 0.5], [0.3, 0.3, 0.3]],
                            np.stack([w, w]), mlp)
    W, H = 9, 7
    cam = synth.pinhole(W, H, 20.0, synth.look_at([0, 0, 6.0]))
    tgt = np.zeros((H * W, 3))
    r = mso.loss_grad_f64(sc, cam, H, W, 8, target=tgt, t_stop=1e-4)
    assert np.abs(r["g_weights"][0]).max() > 1e-3
    assert not r["g_weights"][1].any() and not r["g_center"][1].any() and not r["g_scale"][1].any()
    r0 = mso.loss_grad_f64(sc, cam, H, W, 8, target=tgt, t_stop=0.0)
    assert np.abs(r0["g_weights"][1]).max() > 0.0
