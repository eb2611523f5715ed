"""Pins for the oracle's Eq.7 slot features (S:Sec.8(f) NEXT-2): the tetrahedral frame's
defining properties, the gate against torch's softmax with R from scipy, closed forms for one
primitive, the "same volumetric weights as colour" identity, brute force without binning.  CPU only."""
import math

import numpy as np
import torch
from scipy.spatial.transform import Rotation

from oracle import mso
from paper_2606_03877_b200 import synth
from test_oracle_pins import chord64, lam, ray64, softplus

MLP_C = synth.MLPSpec(3, 0, 1, 8, 0, False, synth.MODE_CONTACT)
TET = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], np.float64) / math.sqrt(3.0)


def test_canonical_tetrahedral_frame():
    """four unit directions, affinely independent, isotropic: sum = 0, pairwise cosine -1/3."""
    assert np.allclose(np.linalg.norm(TET, axis=1), 1.0) and np.allclose(TET.sum(axis=0), 0.0)
    G = TET @ TET.T
    assert np.allclose(G[~np.eye(4, dtype=bool)], -1.0 / 3.0)
    assert np.linalg.matrix_rank(np.hstack([TET, np.ones((4, 1))])) == 4


def scene_one(mu, q, s, raw, emb):
    w = synth.constant_mlp_weights(MLP_C, raw)
    return synth.custom_scene([mu], [q], [s], w[None], MLP_C, slots=np.asarray(emb, np.float32)[None])


def test_gates_against_torch_softmax_and_scipy_rotation():
    """g = softmax_k(a_k^T u), u = clip(R^T delta / s) (Eq.7), R from scipy, softmax from torch."""
    rng = np.random.default_rng(5)
    q, s = [0.3, -0.5, 0.2, 0.78], [0.4, 0.7, 0.25]
    sc = scene_one([0.1, 0.2, 0.3], q, s, [0, 0, 0, 0.5], rng.normal(size=(4, 8)))
    orc = mso.OracleScene(sc)
    qn = np.asarray(q) / np.linalg.norm(q)
    R = Rotation.from_quat([qn[1], qn[2], qn[3], qn[0]]).as_matrix()
    for scale in (0.1, 0.5, 3.0):                       # the last one exercises the clip
        delta = (rng.normal(size=3) * scale * 0.3).astype(np.float32)
        u = np.clip(R.T @ delta.astype(np.float64) / np.asarray(s), -1.0, 1.0)
        ref = torch.softmax(torch.tensor(TET @ u), dim=0).numpy()
        g = orc.slot_gates(0, delta)
        assert abs(g.sum() - 1.0) <= 1e-12 and np.abs(g - ref).max() <= 1e-6


def test_single_primitive_feature_closed_form_and_colour_weights():
    """F = alpha * sum_k g_k e_k for one primitive; with four identical embeddings v, F = alpha v exactly
    as for colour ("rendered with the same volumetric weights as color")."""
    mu, q, s = [0.0, 0.1, -0.1], [0.8, 0.3, -0.4, 0.1], [0.7, 0.5, 0.9]
    raw = [0.2, 0.1, -0.3, 1.1]
    rng = np.random.default_rng(8)
    emb = rng.normal(size=(4, 16))
    W, H = 24, 18
    cam = synth.pinhole(W, H, 50.0, synth.look_at([1.5, 2.0, 2.5]))
    rgb, alpha, feat, _ = mso.OracleScene(scene_one(mu, q, s, raw, emb)).render(cam, H, W, 1, tile=0)
    L, R = lam(q, s)
    n = 0
    for pixel in range(W * H):
        o, d = ray64(cam, pixel % W, pixel // W)
        ch = chord64(o, d, mu, L)
        if ch is None or ch[1] - ch[0] < 1e-2:
            continue
        ts = d @ L @ (np.asarray(mu) - o) / (d @ L @ d)
        delta = np.asarray(mu) - (o + ts * d)
        u = np.clip(R.T @ delta / np.asarray(s), -1, 1)
        g = torch.softmax(torch.tensor(TET @ u), dim=0).numpy()
        assert np.abs(feat[pixel] - alpha[pixel] * (g @ emb)).max() <= 2e-5
        n += 1
    assert n > 50
    v = rng.normal(size=16)
    _, alpha2, feat2, _ = mso.OracleScene(scene_one(mu, q, s, raw, np.tile(v, (4, 1)))).render(cam, H, W, 1, tile=0)
    assert np.abs(feat2 - alpha2[:, None] * v[None, :]).max() <= 1e-6


def test_next2_binned_equals_brute_and_colour_unchanged():
    cfg = synth.shrink(synth.replace(synth.CONFIGS["next2"], c_f=32), 64, 36)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    rgb, alpha, feat, st = orc.render(cam, 36, 64, 1, tile=16)
    rgb0, alpha0, feat0, _ = orc.render(cam, 36, 64, 1, tile=0)
    assert np.array_equal(feat, feat0) and np.array_equal(rgb, rgb0)
    cfg1 = synth.shrink(synth.CONFIGS["next1"], 64, 36)                       # same scene without slots
    rgb1, alpha1, _, _ = mso.OracleScene(synth.make_scene(cfg1)).render(cam, 36, 64, 1)
    assert np.array_equal(rgb, rgb1) and np.array_equal(alpha, alpha1)
    # |F| <= alpha * max_k |e_k| channel-wise (convex gate, weights sum to alpha)
    bound = np.abs(sc.slots).max()
    assert (np.abs(feat) <= alpha[:, None] * bound + 1e-9).all()


def test_next2_crop_matches_stored_oracle_snapshot():
    """regression snapshot written by tests/golden/make_golden.py (calls only oracle/)."""
    import json
    import os
    g = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "next2_oracle.json")))
    cfg = synth.shrink(synth.replace(synth.CONFIGS["next2"], c_f=8), 96, 54)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    rgb, alpha, feat, st = mso.OracleScene(sc).render(cam, 54, 96, 1)
    assert st.n_intervals == g["n_intervals"] and st.n_pairs == g["n_pairs"]
    pix = np.array(g["pixels"])
    np.testing.assert_allclose(rgb[pix], np.array(g["rgb"]), atol=1e-11)
    np.testing.assert_allclose(alpha[pix], np.array(g["alpha"]), atol=1e-11)
    np.testing.assert_allclose(feat[pix], np.array(g["feat"]), atol=1e-11)
