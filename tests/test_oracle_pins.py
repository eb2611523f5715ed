"""Pins for the CPU oracle (oracle/mso.c) against things OTHER than itself:
closed forms (Eq.6 / Eq.14), the paper's Lambda and t*
formulas, invariants, brute force without binning, library routines
(scipy Rotation, torch fp64 matmul / softplus / sigmoid) and an independent
re-compositing loop.  SURVEY.md Sec.8(c) pins P1-P12.  CPU only.
"""
import math

import numpy as np
import pytest
import torch
from scipy.spatial.transform import Rotation

from oracle import mso
from paper_2606_03877_b200 import synth

MLP_SMALL = synth.MLPSpec(2, 0, 1, 8, 0, False)


# ----------------------------------------------------------------------------
# independent fp64 helpers (paper formulas, not the oracle's code path)
# ----------------------------------------------------------------------------
def lam(q_wxyz, s):
    """Lambda_i = R(q) diag(s^2)^-1 R(q)^T, R from scipy (library)."""
    q = np.asarray(q_wxyz, np.float64)
    q = q / np.linalg.norm(q)
    R = Rotation.from_quat([q[1], q[2], q[3], q[0]]).as_matrix()
    return R @ np.diag(1.0 / np.asarray(s, np.float64) ** 2) @ R.T, R


def ray64(cam, x, y):
    m = np.asarray(cam.c2w, np.float64).reshape(3, 4)
    dc = np.array([(x + 0.5 - cam.cx) / cam.fx, (y + 0.5 - cam.cy) / cam.fy, 1.0])
    d = m[:, :3] @ dc
    return m[:, 3].copy(), d / np.linalg.norm(d)


def chord64(o, d, mu, L):
    """roots of |o + t d - mu|^2_Lambda = 1 -> (t0, t1) or None."""
    v = o - np.asarray(mu, np.float64)
    a, b, c = d @ L @ d, d @ L @ v, v @ L @ v - 1.0
    disc = b * b - a * c
    if disc <= 0:
        return None
    return (-b - math.sqrt(disc)) / a, (-b + math.sqrt(disc)) / a


def chord_tol(t_mid, L):
    """fp32 conditioning of the chord: disc = b^2 - a c cancels, so the absolute error of
    L = 2 sqrt(disc)/a is about 2 eps t_mid^2 / L (eps = 2^-24); 4x margin."""
    return 8 * 2.0 ** -24 * t_mid * t_mid / L + 2e-6


def sigmoid(x):
    return 1.0 / (1.0 + np.exp(-np.asarray(x, np.float64)))


def softplus(x):
    return float(torch.nn.functional.softplus(torch.tensor(float(x), dtype=torch.float64)))


def const_scene(prims, mlp=MLP_SMALL):
    """prims: list of (center, quat, scale, raw_out)."""
    w = [synth.constant_mlp_weights(mlp, p[3]) for p in prims]
    return synth.custom_scene([p[0] for p in prims], [p[1] for p in prims],
                              [p[2] for p in prims], np.stack(w), mlp)


def front_camera(W=33, H=21, fov=40.0, dist=4.0):
    return synth.pinhole(W, H, fov, synth.look_at([0.0, 0.0, dist]))


# ----------------------------------------------------------------------------
# geometry pieces
# ----------------------------------------------------------------------------
def test_support_metric_matches_paper_lambda():
    """A^T A == Lambda and M == A^-1, for random primitives."""
    sc = synth.make_scene(synth.CONFIGS["cfg1"])
    A, M = mso.OracleScene(sc).frames()
    for i in range(sc.n):
        L, R = lam(sc.quat[i], sc.scale[i])
        A64 = A[i].astype(np.float64)
        np.testing.assert_allclose(A64.T @ A64, L, rtol=2e-5, atol=1e-5)
        np.testing.assert_allclose(M[i].astype(np.float64) @ A64, np.eye(3), atol=2e-5)
        np.testing.assert_allclose(M[i], R * sc.scale[i][None, :], rtol=1e-5, atol=1e-6)


def test_quaternion_convention_is_wxyz_hamilton():
    """90 deg about +z, (w,x,y,z) = (c,0,0,s): x axis -> y axis (library: scipy)."""
    c = math.sqrt(0.5)
    sc = const_scene([([0, 0, 0], [c, 0, 0, c], [1, 2, 3], [0, 0, 0, 0])])
    _, M = mso.OracleScene(sc).frames()
    np.testing.assert_allclose(M[0] @ np.array([1.0, 0, 0]), [0, 1, 0], atol=1e-6)
    np.testing.assert_allclose(M[0] @ np.array([0, 1.0, 0]), [-2, 0, 0], atol=1e-6)


def test_zero_quaternion_and_bad_scale_rejected():
    with pytest.raises(ValueError):
        mso.OracleScene(const_scene([([0, 0, 0], [0, 0, 0, 0], [1, 1, 1], [0, 0, 0, 0])]))
    with pytest.raises(ValueError):
        mso.OracleScene(const_scene([([0, 0, 0], [1, 0, 0, 0], [1, 0, 1], [0, 0, 0, 0])]))


def test_camera_rays():
    cfg = synth.CONFIGS["cfg1"]
    cam = synth.make_cameras(cfg)[0]
    m = cam.c2w.reshape(3, 4).astype(np.float64)
    W, H = cfg.width, cfg.height
    for (x, y) in [(0, 0), (W - 1, 0), (0, H - 1), (W // 2, H // 2), (17, 5)]:
        o, d = mso.ray(cam, x, y)
        o64, d64 = ray64(cam, x, y)
        np.testing.assert_allclose(o, m[:, 3], atol=0)
        np.testing.assert_allclose(d, d64, atol=3e-7)
        assert abs(np.linalg.norm(d.astype(np.float64)) - 1) < 3e-7
    # horizontal FOV: angle between first and last pixel-centre columns on the middle row
    _, dl = mso.ray(cam, 0, H // 2)
    _, dr = mso.ray(cam, W - 1, H // 2)
    yoff = (H // 2 + 0.5 - cam.cy) / cam.fy
    half = (W / 2 - 0.5) / cam.fx
    expect = (yoff * yoff + 1 - half * half) / (yoff * yoff + 1 + half * half)
    assert abs(float(dl.astype(np.float64) @ dr.astype(np.float64)) - expect) < 1e-6
    # the eye sits at radius 3 and the optical axis points at the origin
    assert abs(np.linalg.norm(m[:, 3]) - cfg.radius) < 1e-6
    np.testing.assert_allclose(m[:, 2], -m[:, 3] / np.linalg.norm(m[:, 3]), atol=1e-6)
    # fx from the horizontal FOV (Q14)
    assert abs(cam.fx - 0.5 * W / math.tan(math.radians(cfg.fov_deg) / 2)) < 1e-4


def test_chord_matches_paper_quadratic_and_contact_point():
    """P2: t_in/t_out solve |o+td-mu|_Lambda = 1; Eq.2's t* is the chord midpoint."""
    cfg = synth.CONFIGS["cfg1"]
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    n_checked = 0
    for pixel in range(0, cfg.width * cfg.height, 7):
        prim, t_in, delta = orc.ray_intervals(cam, cfg.height, cfg.width, cfg.K, pixel, tile=0)
        o, d = ray64(cam, pixel % cfg.width, pixel // cfg.width)
        expect = {}
        for i in range(sc.n):
            L, _ = lam(sc.quat[i], sc.scale[i])
            r = chord64(o, d, sc.center[i], L)
            if r and r[1] > 0:
                expect[i] = (r, L)
        # grazing rays may differ between fp32 and fp64; everything else must agree
        for i, ti, de in zip(prim, t_in, delta):
            assert i in expect or de * cfg.K < 1e-2
            if i in expect:
                (t0, t1), L = expect[i]
                if t1 - t0 < 1e-2:
                    continue
                assert abs(ti - max(t0, 0)) < 2e-5 * max(1, t1)
                assert abs(ti + de * cfg.K - t1) < 2e-5 * max(1, t1)
                tstar = max(0.0, d @ L @ (sc.center[i] - o) / (d @ L @ d))     # Eq.2
                assert abs(tstar - (ti + 0.5 * de * cfg.K)) < 3e-5 * max(1, t1)
                n_checked += 1
        for i, ((t0, t1), _) in expect.items():
            assert i in prim or (t1 - t0) < 1e-2
    assert n_checked > 100


def test_sphere_chord_closed_form():
    """P2: sphere of radius s: L = 2 sqrt(s^2 - dist(ray, mu)^2)."""
    s = 0.7
    sc = const_scene([([0.1, -0.2, 0.3], [1, 0, 0, 0], [s, s, s], [0, 0, 0, 0])])
    cam = front_camera()
    orc = mso.OracleScene(sc)
    hits = 0
    for pixel in range(33 * 21):
        prim, t_in, delta = orc.ray_intervals(cam, 21, 33, 5, pixel, tile=0)
        o, d = ray64(cam, pixel % 33, pixel // 33)
        v = np.array([0.1, -0.2, 0.3]) - o
        dist2 = v @ v - (v @ d) ** 2
        if dist2 < s * s - 1e-4:
            assert len(prim) == 1
            L = 2 * math.sqrt(s * s - dist2)
            assert abs(delta[0] * 5 - L) < chord_tol(v @ d, L)
            hits += 1
        elif dist2 > s * s + 1e-4:
            assert len(prim) == 0
    assert hits > 20


def test_midpoint_samples_and_order():
    """t_k = t_in + (k+1/2) delta; the sequence is a permutation of all (prim,k) sorted by
    (t, prim id, k)  (NS (c),(e); Q12)."""
    cfg = synth.CONFIGS["cfg3"]
    cfg = synth.shrink(cfg, 40, 28)
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    seen_multi = 0
    for pixel in range(0, 40 * 28, 37):
        prim, t_in, delta = orc.ray_intervals(cam, 28, 40, cfg.K, pixel)
        sp, sk, st = orc.ray_samples(cam, 28, 40, cfg.K, pixel)
        assert len(sp) == len(prim) * cfg.K
        lut = {int(p): (a, b) for p, a, b in zip(prim, t_in, delta)}
        assert sorted(zip(sp.tolist(), sk.tolist())) == [(int(p), k) for p in sorted(lut) for k in range(cfg.K)]
        for p, k, t in zip(sp, sk, st):
            a, b = lut[int(p)]
            assert t == np.float32(a + np.float32(np.float32(k + 0.5) * b))      # canonical fp32
            assert abs(float(t) - (float(a) + (k + 0.5) * float(b))) < 1e-5
        keys = list(zip(st.tolist(), sp.tolist(), sk.tolist()))
        assert keys == sorted(keys)
        seen_multi += len(prim) > 3
    assert seen_multi > 5


# ----------------------------------------------------------------------------
# P1, P3, P4: closed forms of Eq.6 / Eq.14
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("K", [1, 3, 8, 16])
def test_single_constant_primitive_closed_form(K):
    """P1: pixel = sigmoid(b_rgb) (1 - exp(-softplus(b_sigma) L)) for every K."""
    raw = [0.3, -1.2, 2.0, 0.7]
    q = [0.9, 0.1, -0.3, 0.2]
    s = [0.5, 0.9, 0.3]
    mu = [0.2, 0.1, -0.1]
    sc = const_scene([(mu, q, s, raw)])
    cam = front_camera()
    rgb, alpha, _, st = mso.OracleScene(sc).render(cam, 21, 33, K, tile=8)
    L, _ = lam(q, s)
    sig = softplus(raw[3])
    n_hit = 0
    for pixel in range(33 * 21):
        o, d = ray64(cam, pixel % 33, pixel // 33)
        r = chord64(o, d, mu, L)
        if r is None or r[1] - r[0] < 1e-3:
            continue
        a = 1.0 - math.exp(-sig * (r[1] - r[0]))
        tol = sig * chord_tol(0.5 * (r[0] + r[1]), r[1] - r[0])
        assert abs(alpha[pixel] - a) < tol
        np.testing.assert_allclose(rgb[pixel], sigmoid(raw[:3]) * a, atol=tol)
        n_hit += 1
    assert n_hit > 30 and st.n_intervals >= n_hit


def test_eye_inside_support_starts_at_t_near():
    """Q13: camera inside the ellipsoid -> interval [t_near, t_out]."""
    raw = [0.0, 0.0, 0.0, 1.0]
    sc = const_scene([([0, 0, 3.5], [1, 0, 0, 0], [1.0, 1.0, 1.0], raw)])   # eye at z=4 is inside
    cam = front_camera()
    rgb, alpha, _, _ = mso.OracleScene(sc).render(cam, 21, 33, 4, tile=8)
    L, _ = lam([1, 0, 0, 0], [1, 1, 1])
    for pixel in [0, 16, 33 * 10 + 16, 33 * 21 - 1]:
        o, d = ray64(cam, pixel % 33, pixel // 33)
        t0, t1 = chord64(o, d, [0, 0, 3.5], L)
        assert t0 < 0 < t1
        assert abs(alpha[pixel] - (1 - math.exp(-softplus(1.0) * t1))) < 5e-6
    cam2 = synth.pinhole(33, 21, 40.0, synth.look_at([0.0, 0.0, 4.0]), t_near=0.25)
    _, alpha2, _, _ = mso.OracleScene(sc).render(cam2, 21, 33, 4, tile=8)
    o, d = ray64(cam2, 16, 10)
    t0, t1 = chord64(o, d, [0, 0, 3.5], L)
    assert abs(alpha2[33 * 10 + 16] - (1 - math.exp(-softplus(1.0) * (t1 - 0.25)))) < 5e-6


def test_primitive_behind_camera_is_invisible():
    sc = const_scene([([0, 0, 6.0], [1, 0, 0, 0], [0.5, 0.5, 0.5], [1, 1, 1, 3.0])])
    cam = front_camera()                                    # eye at z=4 looking toward -z
    for tile in (0, 8):
        rgb, alpha, _, st = mso.OracleScene(sc).render(cam, 21, 33, 4, tile=tile)
        assert st.n_intervals == 0 and not rgb.any() and not alpha.any()


def test_two_disjoint_primitives_front_to_back():
    """P3: C = a1 c1 + (1-a1) a2 c2 (Eq.6); primitive ids must not matter."""
    p_near = ([0, 0, 1.0], [1, 0, 0, 0], [0.4, 0.4, 0.4], [2.0, -1.0, 0.5, 1.5])
    p_far = ([0, 0, -1.0], [1, 0, 0, 0], [0.6, 0.6, 0.6], [-0.7, 0.9, 0.1, 0.2])
    cam = front_camera()
    pix = 33 * 10 + 16                                     # central ray: along -z through both
    out = []
    for order in ([p_near, p_far], [p_far, p_near]):
        rgb, alpha, _, _ = mso.OracleScene(const_scene(order)).render(cam, 21, 33, 8, tile=0, pixels=[pix])
        out.append((rgb[0], alpha[0]))
    o, d = ray64(cam, 16, 10)
    L1, _ = lam([1, 0, 0, 0], p_near[2])
    L2, _ = lam([1, 0, 0, 0], p_far[2])
    c1 = chord64(o, d, p_near[0], L1)
    c2 = chord64(o, d, p_far[0], L2)
    a1 = 1 - math.exp(-softplus(p_near[3][3]) * (c1[1] - c1[0]))
    a2 = 1 - math.exp(-softplus(p_far[3][3]) * (c2[1] - c2[0]))
    expect = a1 * sigmoid(p_near[3][:3]) + (1 - a1) * a2 * sigmoid(p_far[3][:3])
    for rgb, alpha in out:
        np.testing.assert_allclose(rgb, expect, atol=5e-6)
        assert abs(alpha - (a1 + (1 - a1) * a2)) < 5e-6
    np.testing.assert_allclose(out[0][0], out[1][0], atol=1e-15)


def test_coincident_primitives_tie_break_by_id():
    """P4: two coincident constant primitives: samples interleave 0,1,0,1,... and
    C = [a1 c1 + e1 a2 c2] (1 - q^K)/(1 - q), q = e1 e2; swapping ids swaps the roles."""
    K = 6
    geo = ([0.1, 0, 0], [0.8, 0.2, 0.1, -0.4], [0.5, 0.7, 0.4])
    rawA, rawB = [1.0, -2.0, 0.3, 0.9], [-0.5, 0.8, 1.7, -0.3]
    cam = front_camera()
    pix = 33 * 10 + 17
    o, d = ray64(cam, 17, 10)
    L, _ = lam(geo[1], geo[2])
    t0, t1 = chord64(o, d, geo[0], L)
    dl = (t1 - t0) / K
    for first, second in ((rawA, rawB), (rawB, rawA)):
        sc = const_scene([(*geo, first), (*geo, second)])
        orc = mso.OracleScene(sc)
        sp, sk, st = orc.ray_samples(cam, 21, 33, K, pix, tile=0)
        assert sp.tolist() == [0, 1] * K and sk.tolist() == [k for k in range(K) for _ in (0, 1)]
        rgb, alpha, _, _ = orc.render(cam, 21, 33, K, tile=0, pixels=[pix])
        e1 = math.exp(-softplus(first[3]) * dl)
        e2 = math.exp(-softplus(second[3]) * dl)
        q = e1 * e2
        geom = (1 - q ** K) / (1 - q)
        expect = ((1 - e1) * sigmoid(first[:3]) + e1 * (1 - e2) * sigmoid(second[:3])) * geom
        np.testing.assert_allclose(rgb[0], expect, atol=5e-6)
        assert abs(alpha[0] - (1 - q ** K)) < 5e-6


# ----------------------------------------------------------------------------
# P5-P7, P11: invariants, brute force, tile-size independence
# ----------------------------------------------------------------------------
def _feat_alpha_scene(cfg):
    """cfg scene with an extra feature head whose weights are 0 and bias 1 (pin P11)."""
    mlp = synth.MLPSpec(cfg.mlp.n_freq, cfg.mlp.use_viewdir, cfg.mlp.n_hidden, cfg.mlp.width, 2, False)
    base = synth.make_scene(cfg)
    dims = cfg.mlp.layer_dims
    n_head_in = dims[-1][0]
    body = sum(i * o + o for i, o in dims[:-1])
    w_old = base.weights
    n = base.n
    Wh = w_old[:, body:body + n_head_in * 4].reshape(n, n_head_in, 4)
    bh = w_old[:, body + n_head_in * 4:]
    Wh2 = np.concatenate([Wh, np.zeros((n, n_head_in, 2), np.float32)], axis=2)
    bh2 = np.concatenate([bh, np.ones((n, 2), np.float32)], axis=1)
    w_new = np.concatenate([w_old[:, :body], Wh2.reshape(n, -1), bh2], axis=1)
    return synth.custom_scene(base.center, base.quat, base.scale, w_new, mlp)


def test_invariants_and_feature_weights_cfg1():
    """P5 + P11: alpha in [0,1], rgb <= alpha, rays missing every support are exactly 0,
    and a constant-1 feature composites to exactly out_alpha (same weights T*alpha)."""
    cfg = synth.CONFIGS["cfg1"]
    sc = _feat_alpha_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    rgb, alpha, feat, st = orc.render(cam, cfg.height, cfg.width, cfg.K, tile=16)
    hits = orc.hit_counts(cam, cfg.height, cfg.width, cfg.K, tile=16)
    assert st.n_intervals == hits.sum() == 1378        # 0.34 hits/ray at cfg1
    assert np.all(alpha >= 0) and np.all(alpha <= 1) and np.all(rgb >= 0)
    assert np.all(rgb <= alpha[:, None] + 1e-15)
    miss = hits == 0
    assert 0.6 < miss.mean() < 0.8
    assert not rgb[miss].any() and not alpha[miss].any() and not feat[miss].any()
    np.testing.assert_allclose(feat[:, 0], alpha, atol=1e-14)
    np.testing.assert_allclose(feat[:, 1], alpha, atol=1e-14)
    assert alpha.max() > 0.5


def test_transmittance_monotone_and_recomposited():
    """P5: recomposite a few rays in Python from the oracle's sample list + MLP outputs:
    T is non-increasing, weights telescope to 1 - T, and the sum equals the render."""
    cfg = synth.shrink(synth.CONFIGS["cfg3"], 48, 32)
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    A, _ = orc.frames()
    pix = [5, 48 * 16 + 24, 48 * 20 + 7, 48 * 31 + 40]
    rgb, alpha, _, _ = orc.render(cam, 32, 48, cfg.K, pixels=pix)
    for q, pixel in enumerate(pix):
        prim, t_in, delta = orc.ray_intervals(cam, 32, 48, cfg.K, pixel)
        dl = {int(p): float(b) for p, b in zip(prim, delta)}
        sp, sk, st = orc.ray_samples(cam, 32, 48, cfg.K, pixel)
        o, d = mso.ray(cam, pixel % 48, pixel // 48)
        T, C, wsum, prevT = 1.0, np.zeros(3), 0.0, 1.0
        for p, t in zip(sp, st):
            pos = o.astype(np.float64) + float(t) * d.astype(np.float64)
            u = A[p].astype(np.float64) @ (pos - sc.center[p].astype(np.float64))
            _, act = orc.mlp_eval(int(p), u.astype(np.float32), d)
            e = math.exp(-act[3] * dl[int(p)])
            C += T * (1 - e) * act[:3]
            wsum += T * (1 - e)
            T *= e
            assert T <= prevT
            prevT = T
        assert abs(wsum - (1 - T)) < 1e-12
        # u is recomputed here in fp64 while the oracle uses canonical fp32: loose tolerance
        np.testing.assert_allclose(rgb[q], C, atol=2e-4)
        assert abs(alpha[q] - (1 - T)) < 2e-4


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_binned_equals_brute_force_random_tiny_scenes(seed):
    """P6: every primitive tested against every ray (no binning) gives bitwise the same image,
    with the eye inside the primitive cloud (supports straddle the eye plane / image border)."""
    sc, cam, cfg = synth.random_tiny_scene(seed)
    orc = mso.OracleScene(sc)
    H, W = cfg.height, cfg.width
    ref = orc.render(cam, H, W, cfg.K, tile=0)
    hc0 = orc.hit_counts(cam, H, W, cfg.K, tile=0)
    assert ref[3].n_intervals > 50
    for tile in (4, 8, 16):
        out = orc.render(cam, H, W, cfg.K, tile=tile)
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])
        assert np.array_equal(orc.hit_counts(cam, H, W, cfg.K, tile=tile), hc0)


def test_binned_equals_brute_force_cfg1_and_tile_size_irrelevant():
    """P6 + P7 on the tiny oracle scene of BASELINE.json configs[0]."""
    cfg = synth.CONFIGS["cfg1"]
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    ref = orc.render(cam, cfg.height, cfg.width, cfg.K, tile=0)
    sizes = set()
    for tile in (8, 16, 32):
        out = orc.render(cam, cfg.height, cfg.width, cfg.K, tile=tile)
        assert np.array_equal(out[0], ref[0]) and np.array_equal(out[1], ref[1])
        sizes.add(out[3].n_pairs)
    assert len(sizes) == 3                      # the tile lists do differ


def test_projection_aabb_is_conservative_and_tight():
    """Points ON each ellipsoid, projected in fp64, must land inside the AABB; for supports
    well in front of the eye the AABB is no more than ~2 px larger than the sampled extent."""
    cfg = synth.CONFIGS["cfg3"]
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    W, H = cfg.width, cfg.height
    m = cam.c2w.reshape(3, 4).astype(np.float64)
    rng = np.random.default_rng(0)
    w = rng.normal(size=(4000, 3))
    w /= np.linalg.norm(w, axis=1, keepdims=True)
    n_tight = n_full = n_cull = 0
    for i in range(0, sc.n, 3):
        _, R = lam(sc.quat[i], sc.scale[i])
        pts = sc.center[i].astype(np.float64) + (w * sc.scale[i].astype(np.float64)) @ R.T
        pc = (pts - m[:, 3]) @ m[:, :3]
        vis, (x0, x1, y0, y1), z = orc.project(cam, H, W, i)
        front = pc[:, 2] > 1e-6
        if not front.any():
            assert not vis
            n_cull += 1
            continue
        px = cam.fx * pc[front, 0] / pc[front, 2] + cam.cx - 0.5      # pixel index whose centre is hit
        py = cam.fy * pc[front, 1] / pc[front, 2] + cam.cy - 0.5
        inside = (px >= -0.5) & (px <= W - 0.5) & (py >= -0.5) & (py <= H - 0.5)
        if inside.any():
            assert vis
            assert x0 <= np.floor(px[inside].min() + 0.5) and x1 >= np.ceil(px[inside].max() - 0.5)
            assert y0 <= np.floor(py[inside].min() + 0.5) and y1 >= np.ceil(py[inside].max() - 0.5)
        assert z <= pc[:, 2].min() + 1e-5 or z == 0.0
        if front.all() and pc[:, 2].min() > 0.5 and vis:
            if (x0, x1, y0, y1) == (0, W - 1, 0, H - 1):
                n_full += 1
                continue
            if px.min() > 2 and px.max() < W - 3:
                assert x0 >= px.min() - 3 and x1 <= px.max() + 3
                n_tight += 1
    assert n_tight > 50


def test_near_eye_box_bound_is_conservative_and_beats_the_whole_image():
    """Q13: a support that touches or straddles the eye plane is bounded by its camera-space box
    clipped at the depth in front of which everything projects off the image.  Eye INSIDE CFG4's primitive cloud:
    points on every such ellipsoid, projected in fp64, land inside the rectangle whenever they land on the image;
    most of these supports no longer cover the whole image."""
    cfg = synth.shrink(synth.CONFIGS["cfg4_inside"], 480, 270)
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    W, H = cfg.width, cfg.height
    m = cam.c2w.reshape(3, 4).astype(np.float64)
    rng = np.random.default_rng(1)
    w = rng.normal(size=(6000, 3))
    w /= np.linalg.norm(w, axis=1, keepdims=True)
    n_near = n_full = n_small = 0
    for i in range(sc.n):
        _, R = lam(sc.quat[i], sc.scale[i])
        # surface and interior points: the clip argument is about every point of the support
        rad = np.concatenate([np.ones(3000), rng.uniform(0, 1, 3000) ** (1 / 3)])[:, None]
        pts = sc.center[i].astype(np.float64) + (w * rad * sc.scale[i].astype(np.float64)) @ R.T
        pc = (pts - m[:, 3]) @ m[:, :3]
        rz = np.linalg.norm((R * sc.scale[i].astype(np.float64)).T @ m[:, 2])      # |row_z(M_c)|
        cz = (sc.center[i].astype(np.float64) - m[:, 3]) @ m[:, 2]
        if not (cz + rz > 0 and cz - rz <= 0.01 * rz):
            continue                                              # not the near-eye branch
        n_near += 1
        vis, (x0, x1, y0, y1), z = orc.project(cam, H, W, i)
        front = pc[:, 2] > 1e-9
        px = cam.fx * pc[front, 0] / pc[front, 2] + cam.cx - 0.5
        py = cam.fy * pc[front, 1] / pc[front, 2] + cam.cy - 0.5
        inside = (px >= -0.5) & (px <= W - 0.5) & (py >= -0.5) & (py <= H - 0.5)
        if inside.any():
            assert vis
            assert x0 <= np.floor(px[inside].min() + 0.5) and x1 >= np.ceil(px[inside].max() - 0.5)
            assert y0 <= np.floor(py[inside].min() + 0.5) and y1 >= np.ceil(py[inside].max() - 0.5)
        if vis and (x0, x1, y0, y1) == (0, W - 1, 0, H - 1):
            n_full += 1
        else:
            n_small += 1
    assert n_near > 100 and n_small > 0.6 * n_near, (n_near, n_full, n_small)
    # and the image does not notice: binned == brute force bitwise on a sample of pixels
    pix = rng.choice(W * H, 400, replace=False).astype(np.int32)
    a = orc.render(cam, H, W, 4, tile=16, pixels=pix)
    b = orc.render(cam, H, W, 4, tile=0, pixels=pix)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and a[3].n_intervals == b[3].n_intervals


def test_tile_lists_sorted_by_tile_depth_id():
    """NS (a),(b): keys = (tile, z_entry bits, primitive id) ascending; rebuilt here from the
    per-primitive AABBs with numpy lexsort (library)."""
    cfg = synth.shrink(synth.CONFIGS["cfg3"], 160, 96)
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    tile = 16
    off, prim, zb = orc.tile_lists(cam, 96, 160, tile)
    tx = (160 + tile - 1) // tile
    keys = []
    for i in range(sc.n):
        vis, (x0, x1, y0, y1), z = orc.project(cam, 96, 160, i)
        if not vis:
            continue
        bits = int(np.float32(z).view(np.uint32))
        for b in range(y0 // tile, y1 // tile + 1):
            for a in range(x0 // tile, x1 // tile + 1):
                keys.append((b * tx + a, bits, i))
    keys = np.array(keys, dtype=np.int64)
    order = np.lexsort((keys[:, 2], keys[:, 1], keys[:, 0]))
    keys = keys[order]
    assert len(keys) == len(prim) == off[-1]
    assert np.array_equal(keys[:, 2], prim) and np.array_equal(keys[:, 1], zb.astype(np.int64))
    counts = np.bincount(keys[:, 0], minlength=len(off) - 1)
    assert np.array_equal(np.diff(off), counts)
    # depth is non-decreasing inside each tile
    for t in range(len(off) - 1):
        z = zb[off[t]:off[t + 1]].view(np.float32)
        assert np.all(np.diff(z) >= 0)


# ----------------------------------------------------------------------------
# P8: MLP against torch fp64 (library special case)
# ----------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg4", "cfg5"])
def test_mlp_and_posenc_vs_torch_fp64(name):
    cfg = synth.CONFIGS[name]
    mlp = cfg.mlp
    small = synth.SceneConfig("t", cfg.seed, 5, cfg.box, cfg.s_min, cfg.s_max, mlp, 8, 8, 60.0, 3.0, 4)
    sc = synth.make_scene(small)
    orc = mso.OracleScene(sc)
    rng = np.random.default_rng(3)
    for prim in range(sc.n):
        u = rng.uniform(-1, 1, 3).astype(np.float32)
        d = rng.normal(size=3)
        d = (d / np.linalg.norm(d)).astype(np.float32)
        # Eq.5 with identity first, blocks [sin(2^l pi u) (xyz), cos(2^l pi u) (xyz)] (Q3)
        u64 = u.astype(np.float64)
        x = [u64]
        for lvl in range(mlp.n_freq):
            x += [np.sin(2.0 ** lvl * np.pi * u64), np.cos(2.0 ** lvl * np.pi * u64)]
        if mlp.use_viewdir:
            x.append(d.astype(np.float64))
        x = np.concatenate(x)
        assert x.size == mlp.in_dim
        np.testing.assert_allclose(orc.encode(u, d), x, atol=1e-13)
        h = torch.tensor(x, dtype=torch.float64)
        w = torch.tensor(sc.weights[prim], dtype=torch.float64)
        pos = 0
        layers = mlp.layer_dims
        for li, (i, o) in enumerate(layers):
            W = w[pos:pos + i * o].reshape(i, o)
            pos += i * o
            b = w[pos:pos + o]
            pos += o
            h = h @ W + b
            if li < len(layers) - 1:
                h = torch.relu(h)
        assert pos == mlp.params_per_prim
        raw, act = orc.mlp_eval(prim, u, d)
        np.testing.assert_allclose(raw, h.numpy(), rtol=1e-12, atol=1e-12)
        np.testing.assert_allclose(act[:3], torch.sigmoid(h[:3]).numpy(), atol=1e-14)
        assert abs(act[3] - float(torch.nn.functional.softplus(h[3]))) < 1e-14
        np.testing.assert_allclose(act[4:], h[4:].numpy(), atol=0)


def test_softplus_is_stable_for_large_inputs():
    mlp = MLP_SMALL
    for r in (-60.0, -5.0, 0.0, 5.0, 60.0, 800.0):
        sc = const_scene([([0, 0, 0], [1, 0, 0, 0], [1, 1, 1], [0, 0, 0, r])], mlp)
        _, act = mso.OracleScene(sc).mlp_eval(0, [0.1, 0.2, 0.3])
        assert abs(act[3] - softplus(r)) <= 1e-12 * max(1.0, abs(r))


# ----------------------------------------------------------------------------
# P9: early termination
# ----------------------------------------------------------------------------
def test_early_termination_constant_density_stop_index():
    """Constant sigma: T after n samples = exp(-n sigma delta); the ray stops at the smallest n
    with T < 1e-4 and alpha_out = 1 - T_n exactly there (NS (e), Q9)."""
    K = 64
    raw = [0.2, 0.4, -0.3, 30.0]
    s = 1.0
    sc = const_scene([([0, 0, 0], [1, 0, 0, 0], [s, s, s], raw)])
    cam = front_camera()
    pix = 33 * 10 + 16
    orc = mso.OracleScene(sc)
    rgb, alpha, _, st = orc.render(cam, 21, 33, K, tile=8, pixels=[pix])
    o, d = ray64(cam, 16, 10)
    L, _ = lam([1, 0, 0, 0], [s, s, s])
    t0, t1 = chord64(o, d, [0, 0, 0], L)
    sd = softplus(raw[3]) * (t1 - t0) / K
    n_stop = next(n for n in range(1, K + 1) if math.exp(-n * sd) < 1e-4)
    assert 1 < n_stop < K
    assert st.n_terminated == 1 and st.n_mlp_evals == n_stop
    assert abs(alpha[0] - (1 - math.exp(-n_stop * sd))) < 1e-9
    np.testing.assert_allclose(rgb[0], sigmoid(raw[:3]) * (1 - math.exp(-n_stop * sd)), atol=1e-9)
    # with the threshold disabled the full sum is returned
    _, alpha_full, _, st2 = orc.render(cam, 21, 33, K, tile=8, pixels=[pix], t_stop=0.0)
    assert st2.n_terminated == 0 and st2.n_mlp_evals == K
    assert abs(alpha_full[0] - (1 - math.exp(-K * sd))) < 1e-9


def test_early_termination_dense_scene_equals_truncated_sum():
    """P9: on an opaque scene the render equals the full front-to-back sum truncated after the
    first sample with T < 1e-4 (none of cfg1-5 terminates, so this scene covers the branch)."""
    sc, cfg = synth.dense_scene()
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    H, W = cfg.height, cfg.width
    rgb, alpha, _, st = orc.render(cam, H, W, cfg.K)
    assert st.n_terminated > 200 and st.n_mlp_evals < st.n_samples
    A, _ = orc.frames()
    checked = 0
    for pixel in range(W * (H // 2) + 3, W * (H // 2) + W, 9):
        prim, t_in, delta = orc.ray_intervals(cam, H, W, cfg.K, pixel)
        if len(prim) == 0:
            continue
        dl = {int(p): float(b) for p, b in zip(prim, delta)}
        sp, sk, stt = orc.ray_samples(cam, H, W, cfg.K, pixel)
        o, d = mso.ray(cam, pixel % W, pixel // W)
        T, C, stopped = 1.0, np.zeros(3), False
        for p, t in zip(sp, stt):
            # canonical fp32 u, as the oracle defines it (p = o + t d; u = A (p - mu))
            pos = (o + np.float32(t) * d).astype(np.float32)
            wv = (pos - sc.center[p]).astype(np.float32)
            u = np.array([np.float32(np.float32(A[p][r, 0] * wv[0] + A[p][r, 1] * wv[1]) + A[p][r, 2] * wv[2])
                          for r in range(3)], np.float32)
            _, act = orc.mlp_eval(int(p), u, d)
            e = math.exp(-act[3] * dl[int(p)])
            C += T * (1 - e) * act[:3]
            T *= e
            if T < np.float32(1e-4):
                stopped = True
                break
        np.testing.assert_allclose(rgb[pixel], C, atol=1e-12)
        assert abs(alpha[pixel] - (1 - T)) < 1e-12
        checked += stopped
    assert checked >= 3


# ----------------------------------------------------------------------------
# P10, P12: rigid invariance, K refinement
# ----------------------------------------------------------------------------
def test_rigid_transform_of_scene_and_camera_leaves_image_unchanged():
    cfg = synth.CONFIGS["cfg1"]
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    ref = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, cfg.K)
    G = Rotation.from_rotvec([0.4, -0.9, 0.3])
    tvec = np.array([0.7, -0.2, 1.1])
    center2 = G.apply(sc.center.astype(np.float64)) + tvec
    qs = Rotation.from_quat(sc.quat[:, [1, 2, 3, 0]].astype(np.float64))
    q2 = (G * qs).as_quat()[:, [3, 0, 1, 2]]
    sc2 = synth.custom_scene(center2, q2, sc.scale, sc.weights, sc.mlp)
    m = cam.c2w.reshape(3, 4).astype(np.float64)
    m2 = np.concatenate([G.as_matrix() @ m[:, :3], (G.apply(m[:, 3]) + tvec)[:, None]], axis=1)
    cam2 = synth.Camera(cam.fx, cam.fy, cam.cx, cam.cy, m2.reshape(-1).astype(np.float32), 0.0,
                        cam.width, cam.height)
    out = mso.OracleScene(sc2).render(cam2, cfg.height, cfg.width, cfg.K)
    assert abs(out[3].n_intervals - ref[3].n_intervals) <= 3            # grazing rays only
    d = np.abs(out[0] - ref[0])
    assert np.quantile(d, 0.999) < 2e-4 and d.max() < 5e-3
    assert np.quantile(np.abs(out[1] - ref[1]), 0.999) < 2e-4


def test_k_refinement_converges():
    """P12 (sanity): for a smooth field the image converges as K doubles."""
    mlp = synth.MLPSpec(1, 0, 1, 8, 0, False)
    cfg = synth.SceneConfig("smooth", 11, 6, 0.6, 0.4, 0.8, mlp, 24, 16, 45.0, 3.0, 4)
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    imgs = [orc.render(cam, 16, 24, K)[0] for K in (2, 4, 8, 16, 32, 64)]
    errs = [np.abs(a - imgs[-1]).max() for a in imgs[:-1]]
    assert errs[-1] < errs[0] / 20 and all(errs[i + 1] < errs[i] for i in range(len(errs) - 1))


# ----------------------------------------------------------------------------
# regression snapshot written by tests/golden/make_golden.py (calls only oracle/)
# ----------------------------------------------------------------------------
def test_cfg1_matches_stored_oracle_snapshot():
    import json
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg1_oracle.json")
    g = json.load(open(path))
    cfg = synth.CONFIGS["cfg1"]
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    rgb, alpha, _, st = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, cfg.K)
    assert st.n_intervals == g["n_intervals"] and st.n_pairs == g["n_pairs"]
    pix = np.array(g["pixels"])
    np.testing.assert_allclose(rgb[pix], np.array(g["rgb"]), atol=1e-11)
    np.testing.assert_allclose(alpha[pix], np.array(g["alpha"]), atol=1e-11)
