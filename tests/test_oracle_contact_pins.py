"""Pins for the oracle's contact-point mode (S:Sec.8(f) NEXT-1; the paper's own variant)
against things other than itself: Eq.2's t* and the Lambda quadratic form from scipy's rotation,
Eq.5's layout from numpy, the MLP from torch fp64, closed forms of Eq.6 with the two readings
(chord length, Gaussian falloff) written out, brute force without binning.  CPU only."""
import math

import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth
from test_oracle_pins import chord64, chord_tol, lam, ray64, sigmoid, softplus

MLP_C = synth.MLPSpec(3, 0, 1, 8, 0, False, synth.MODE_CONTACT)       # 36-8-4
MLP_PAPER = synth.MLPSpec(6, 0, 2, 32, 0, False, synth.MODE_CONTACT)   # 72-32-32-4


def one_prim(mu, q, s, raw_out, mlp=MLP_C):
    w = synth.constant_mlp_weights(mlp, raw_out)
    return synth.custom_scene([mu], [q], [s], w[None], mlp)


def test_paper_mlp_has_3524_parameters():
    """72-d encoded input, two hidden layers of 32, 4 outputs -> 72*32+32 + 32*32+32 + 32*4+4."""
    assert MLP_PAPER.in_dim == 72 and MLP_PAPER.params_per_prim == 3524


def test_contact_point_is_eq2_and_the_chord_midpoint():
    """Eq.2: t* = d^T Lambda (mu - o) / d^T Lambda d, Lambda from scipy; for a ray that
    starts outside the support it is also the midpoint of the chord."""
    mu, q, s = [0.2, -0.1, 0.3], [0.9, 0.1, -0.3, 0.2], [0.5, 0.25, 0.8]
    sc = one_prim(mu, q, s, [0.3, -0.2, 0.1, 0.7])
    orc = mso.OracleScene(sc)
    W, H = 48, 40
    cam = synth.pinhole(W, H, 45.0, synth.look_at([0.5, 0.4, 4.0]))
    L, _ = lam(q, s)
    n = 0
    for pixel in range(0, W * H, 3):
        prim, k, t = orc.ray_samples(cam, H, W, 1, pixel)
        o, d = ray64(cam, pixel % W, pixel // W)
        ch = chord64(o, d, mu, L)
        if ch is None or ch[1] - ch[0] < 1e-3:
            assert len(t) <= 1
            continue
        assert len(t) == 1 and k[0] == 0
        t_star = d @ L @ (np.asarray(mu) - o) / (d @ L @ d)
        tol = chord_tol(t_star, ch[1] - ch[0])
        assert abs(t[0] - t_star) <= tol and abs(t[0] - 0.5 * (ch[0] + ch[1])) <= tol
        n += 1
    assert n > 20


def test_eye_inside_the_support_clamps_t_star_to_zero():
    """Eq.2's max(0, .): the eye is inside the ellipsoid and past its centre along the ray -> p* = o."""
    mu, s = [0.0, 0.0, 0.0], [1.5, 1.5, 1.5]
    sc = one_prim(mu, [1, 0, 0, 0], s, [0, 0, 0, 0.5])
    orc = mso.OracleScene(sc)
    cam = synth.pinhole(9, 9, 40.0, synth.look_at([0, 0, -0.5], target=[0, 0, -3.0]))   # looking away from mu
    prim, k, t = orc.ray_samples(cam, 9, 9, 1, 40)
    assert len(t) == 1 and t[0] == 0.0


def test_single_constant_primitive_closed_form():
    """Eq.6 with one primitive: pixel = c alpha, alpha = (1 - exp(-sigma l)) g with the readings
    l = chord length, g = exp(-(9/2) r^2), r^2 = |p* - mu|^2_Lambda -- all from the Lambda quadratic."""
    mu, q, s = [0.1, 0.2, -0.2], [0.7, -0.2, 0.5, 0.4], [0.6, 0.9, 0.4]
    raw = [0.4, -1.0, 2.0, 1.3]
    sc = one_prim(mu, q, s, raw)
    W, H = 40, 30
    cam = synth.pinhole(W, H, 50.0, synth.look_at([2.5, 1.0, 2.0]))
    rgb, alpha, _, st = mso.OracleScene(sc).render(cam, H, W, 1, tile=0)
    L, _ = lam(q, s)
    hit = 0
    for pixel in range(W * H):
        o, d = ray64(cam, pixel % W, pixel // W)
        ch = chord64(o, d, mu, L)
        if ch is None or ch[1] - ch[0] < 1e-3:
            continue
        ts = d @ L @ (np.asarray(mu) - o) / (d @ L @ d)
        v = o + ts * d - np.asarray(mu)
        g = math.exp(-4.5 * (v @ L @ v))
        a = (1.0 - math.exp(-softplus(raw[3]) * (ch[1] - ch[0]))) * g
        tol = 4 * chord_tol(ts, ch[1] - ch[0]) * softplus(raw[3]) + 1e-6
        assert abs(alpha[pixel] - a) <= tol
        assert np.abs(rgb[pixel] - sigmoid(raw[:3]) * a).max() <= tol
        hit += 1
    assert hit > 100 and st.n_intervals >= hit


def test_encoding_layout_mlp_and_falloff_argument():
    """gamma([d; delta]) index 2L j + 2l (+1) = sin / cos (2^l pi z_j) (Eq.5), delta = mu - p*
    (Eq.3); the MLP against torch fp64; r^2 against the Lambda quadratic form."""
    cfg = synth.shrink(synth.CONFIGS["next1"], 32, 18)
    sc = synth.make_scene(cfg)
    orc = mso.OracleScene(sc)
    rng = np.random.default_rng(3)
    Lf = cfg.mlp.n_freq
    for prim in (0, 17, 2047):
        o = rng.uniform(-1, 1, 3).astype(np.float32)
        d = rng.normal(size=3)
        d = (d / np.linalg.norm(d)).astype(np.float32)
        t = np.float32(rng.uniform(0.5, 3.0))
        x, raw, act, r2 = orc.contact_eval(prim, o, d, float(t))
        p = o.astype(np.float64) + float(t) * d.astype(np.float64)
        z = np.concatenate([d.astype(np.float64), sc.center[prim].astype(np.float64) - p])
        ref = np.zeros(12 * Lf)
        for j in range(6):
            for l in range(Lf):
                ref[2 * Lf * j + 2 * l] = np.sin(2.0 ** l * np.pi * z[j])
                ref[2 * Lf * j + 2 * l + 1] = np.cos(2.0 ** l * np.pi * z[j])
        assert np.abs(x - ref).max() <= 2.0 ** (Lf - 1) * np.pi * 4e-7 + 1e-12    # p* is rounded to fp32
        h = torch.tensor(x, dtype=torch.float64)
        w = torch.tensor(sc.weights[prim].astype(np.float64))
        off = 0
        dims = cfg.mlp.layer_dims
        for li, (i, oo) in enumerate(dims):
            Wm = w[off:off + i * oo].reshape(i, oo); off += i * oo
            b = w[off:off + oo]; off += oo
            h = h @ Wm + b
            if li < len(dims) - 1:
                h = torch.relu(h)
        assert np.abs(raw - h.numpy()).max() <= 1e-10
        assert np.abs(act[:3] - torch.sigmoid(h[:3]).numpy()).max() <= 1e-12
        assert abs(act[3] - float(torch.nn.functional.softplus(h[3]))) <= 1e-12
        Lm, _ = lam(sc.quat[prim], sc.scale[prim])
        v = p - sc.center[prim].astype(np.float64)
        assert abs(r2 - v @ Lm @ v) <= 1e-4 * max(1.0, v @ Lm @ v)


def test_two_disjoint_primitives_front_to_back_and_id_swap():
    """Eq.6: C = a1 c1 + (1 - a1) a2 c2 in the order of t*, whatever the primitive ids."""
    raws = [[1.0, -1.0, 0.0, 2.0], [-0.5, 0.7, 1.5, 0.8]]
    mus, ss = [[0, 0, 1.0], [0, 0, -1.0]], [[0.4] * 3, [0.6] * 3]
    cam = synth.pinhole(1, 1, 30.0, synth.look_at([0, 0, 4.0]))          # the ray runs along -z through both centres
    out = []
    for order in ((0, 1), (1, 0)):
        w = np.stack([synth.constant_mlp_weights(MLP_C, raws[i]) for i in order])
        sc = synth.custom_scene([mus[i] for i in order], [[1, 0, 0, 0]] * 2, [ss[i] for i in order], w, MLP_C)
        rgb, alpha, _, _ = mso.OracleScene(sc).render(cam, 1, 1, 1, tile=0)
        out.append((rgb[0], alpha[0]))
    a = [1.0 - math.exp(-softplus(raws[i][3]) * 2 * ss[i][0]) for i in (0, 1)]   # through the centre: r^2 = 0, g = 1
    c = [sigmoid(raws[i][:3]) for i in (0, 1)]
    expect = a[0] * c[0] + (1 - a[0]) * a[1] * c[1]
    for rgb, alpha in out:
        assert np.abs(rgb - expect).max() <= 1e-5 and abs(alpha - (1 - (1 - a[0]) * (1 - a[1]))) <= 1e-5


def test_binned_equals_brute_force_and_invariants():
    cfg = synth.shrink(synth.CONFIGS["next1"], 96, 54)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    rgb, alpha, _, st = orc.render(cam, 54, 96, 1, tile=16)
    rgb0, alpha0, _, st0 = orc.render(cam, 54, 96, 1, tile=0)
    assert np.array_equal(rgb, rgb0) and np.array_equal(alpha, alpha0) and st.n_intervals == st0.n_intervals
    assert alpha.min() >= 0 and alpha.max() <= 1 and (rgb <= alpha[:, None] + 1e-12).all()
    assert st.n_samples == st.n_intervals                       # one evaluation per (ray, primitive)
    with pytest.raises(Exception):
        orc.render(cam, 54, 96, 2)                              # K samples per interval is the other mode


def test_tile_centre_order_pins():
    """P:109 / P:148 shared per-tile order (MSO_ORDER_TILE): (i) alpha = 1 - prod(1 - alpha_i) does not depend on
    the order; (ii) the tile lists are sorted by Eq.2's t* of the tile-centre ray, recomputed from the
    Lambda quadratic in fp64; (iii) a pixel's colour equals an independent fp64 re-compositing of its
    hits in tile-list order; (iv) one primitive: identical to the exact order."""
    cfg = synth.shrink(synth.CONFIGS["next1"], 96, 54)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    H, W, T = 54, 96, 8
    orc = mso.OracleScene(sc)
    rgb_e, alpha_e, _, st_e = orc.render(cam, H, W, 1, tile=T)
    orc.set_order(1)
    rgb_t, alpha_t, _, st_t = orc.render(cam, H, W, 1, tile=T)
    assert st_t.n_intervals == st_e.n_intervals
    assert np.abs(alpha_t - alpha_e).max() <= 1e-12                        # (i)
    assert np.abs(rgb_t - rgb_e).max() > 1e-3                              # and the colours do differ
    off, prim, zb = orc.tile_lists(cam, H, W, T)
    tiles_x = (W + T - 1) // T
    checked = 0
    for t in range(0, len(off) - 1, 5):                                    # (ii)
        ids = prim[off[t]:off[t + 1]]
        if len(ids) < 2:
            continue
        o, d = ray64(cam, (t % tiles_x) * T + T / 2 - 0.5, (t // tiles_x) * T + T / 2 - 0.5)   # ray64 adds the half pixel
        ts = []
        for i in ids:
            L, _ = lam(sc.quat[i], sc.scale[i])
            ts.append(max(0.0, d @ L @ (sc.center[i].astype(np.float64) - o) / (d @ L @ d)))
        ts = np.array(ts)
        assert np.all(np.diff(ts) >= -1e-4 * np.maximum(1.0, ts[1:]))
        assert np.abs(zb[off[t]:off[t + 1]].view(np.float32) - ts).max() <= 1e-4 * max(1.0, ts.max())
        checked += 1
    assert checked > 10
    for pixel in (W * 20 + 31, W * 33 + 70, W * 41 + 12):                  # (iii)
        x, y = pixel % W, pixel // W
        t = (y // T) * tiles_x + x // T
        order = list(prim[off[t]:off[t + 1]])
        hp, ht, hl = orc.ray_intervals(cam, H, W, 1, pixel, tile=T)
        hits = sorted(zip(hp, ht, hl), key=lambda h: order.index(h[0]))
        o32, d32 = mso.ray(cam, x, y)
        Tr, C = 1.0, np.zeros(3)
        for p, tstar, chord in hits:
            _, _, act, r2 = orc.contact_eval(int(p), o32, d32, float(tstar))
            a = (1.0 - math.exp(-act[3] * float(chord))) * math.exp(-4.5 * r2)
            C += Tr * a * act[:3]
            Tr *= 1.0 - a
        assert len(hits) >= 2 and np.abs(C - rgb_t[pixel]).max() <= 1e-12 and abs((1 - Tr) - alpha_t[pixel]) <= 1e-12
    w = synth.constant_mlp_weights(MLP_C, [0.3, -0.2, 0.1, 0.7])           # (iv)
    one = synth.custom_scene([[0, 0, 0]], [[1, 0, 0, 0]], [[0.8, 0.5, 0.6]], w[None], MLP_C)
    cam1 = synth.pinhole(32, 24, 50.0, synth.look_at([0.5, 0.4, 3.0]))
    o1 = mso.OracleScene(one)
    a = o1.render(cam1, 24, 32, 1, tile=8)
    o1.set_order(1)
    b = o1.render(cam1, 24, 32, 1, tile=8)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    with pytest.raises(Exception):
        o1.render(cam1, 24, 32, 1, tile=0)                                 # the shared order needs tiles
