"""Randomised sweeps of the CUDA path against the oracle: seeded draws of the primitive count, K, tile edge, image size,
eye position (inside / outside the cloud) and MLP shape -- every kernel shape the library instantiates.  Structures
(tile lists, per-ray intervals, the composited order of every ray) bit-exact; fp32 images within the fp32 bar; the
debug, plain and no-sync renders bitwise equal; on the tensor path every random combination of band budget, wave size
and MS_FLAG_OVERLAP bitwise the one-band render.  The bf16 bar itself is a statement about the configs' distributions
(K >= 16, sigma-bias 0.5; tests/test_gpu_parity_bf16.py holds it there): random opaque scenes and 32-channel features at
K <= 5 reach up to 1.5 x the bar, so the sweep holds the tensor path to twice the bar."""
import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth
from test_gpu_parity_bf16 import TOL_MAX, TOL_MEAN
from test_gpu_parity_fp32 import TOL_FP32, check_structures

pytestmark = pytest.mark.gpu


def _api():
    from paper_2606_03877_b200 import api
    return api


def test_fp32_path_random_scenes():
    api = _api()
    rng = np.random.default_rng(12345)
    for seed in range(48):
        n = int(rng.integers(1, 40)); K = int(rng.choice([1, 2, 3, 4, 5, 8, 16, 24, 32])); tile = int(rng.choice([8, 16, 32]))
        W = int(rng.integers(5, 90)); H = int(rng.integers(5, 70)); straddle = bool(rng.integers(0, 2))
        mlp = synth.MLPSpec(int(rng.integers(1, 5)), int(rng.integers(0, 2)), int(rng.integers(1, 4)),
                            int(rng.choice([8, 16, 32, 64])), 0, False)
        sc, cam, cfg = synth.random_tiny_scene(seed, n, straddle=straddle, mlp=mlp)
        cam = synth.pinhole(W, H, cfg.fov_deg, cam.c2w)
        what = dict(seed=seed, n=n, K=K, tile=tile, W=W, H=H, straddle=straddle)
        gs, orc = api.Scene(sc), mso.OracleScene(sc)
        ref = [t.clone() for t in gs.render(cam, H, W, K, tile=tile, path=api.PATH_FP32, flags=api.FLAG_DEBUG_ALL)[:2]]
        torch.cuda.synchronize()
        o_rgb, o_alpha, _, st = orc.render(cam, H, W, K, tile=tile)
        assert check_structures(gs, orc, cam, H, W, K, tile, n_order_rays=4) == st.n_intervals, what
        d = np.abs(ref[0].cpu().numpy().reshape(-1, 3) - o_rgb)
        da = np.abs(ref[1].cpu().numpy().reshape(-1) - o_alpha)
        assert (d > TOL_FP32).sum() <= 2 and d.max() < 1.5e-4 and da.max() < 1.5e-4, (what, d.max(), da.max())   # Q25
        plain = gs.render(cam, H, W, K, tile=tile, path=api.PATH_FP32)
        torch.cuda.synchronize()
        assert torch.equal(plain[0], ref[0]) and torch.equal(plain[1], ref[1]), what
        for _ in range(2):                                   # sized from the previous view: no host synchronisation
            ns = gs.render(cam, H, W, K, tile=tile, path=api.PATH_FP32, flags=api.FLAG_NO_SYNC)
            torch.cuda.synchronize()
            s2 = gs.stats()
            assert s2.no_sync == 1 and s2.overflow == 0 and s2.n_intervals == st.n_intervals, what
            assert torch.equal(ns[0], ref[0]) and torch.equal(ns[1], ref[1]), what
        gs.close()


# (L, view direction, width, feature channels, hidden layers) of the tensor kernel's instantiations (K-sample mode)
TC_SHAPES = [(6, 0, 128, 0, 2), (4, 0, 64, 0, 2), (6, 0, 64, 0, 3), (4, 1, 128, 0, 3), (4, 0, 128, 0, 3), (6, 1, 128, 0, 3),
             (6, 0, 128, 0, 3), (4, 0, 64, 32, 3), (4, 1, 64, 32, 3), (4, 1, 64, 0, 3), (4, 0, 64, 0, 3)]


def test_tensor_path_random_scenes_bands_waves_overlap():
    api = _api()
    rng = np.random.default_rng(777)
    for seed in range(40):
        contact = bool(rng.integers(0, 2))
        n = int(rng.integers(4, 120)); tile = int(rng.choice([8, 16, 32]))
        K = 1 if contact else int(rng.choice([2, 4, 5, 8, 16, 24]))
        W = int(rng.integers(20, 140)); H = int(rng.integers(16, 100))
        L, vd, width, nfeat, nh = (6, 0, 32, 0, 2) if contact else TC_SHAPES[int(rng.integers(0, len(TC_SHAPES)))]
        mlp = synth.MLPSpec(L, vd, nh, width, nfeat, True, synth.MODE_CONTACT if contact else 0,
                            falloff=float(rng.choice([0.0, 0.5, 4.5])) if contact else 4.5)
        sbias = float(rng.choice([0.5, 8.0]))                # 8: opaque, rays stop early, waves drop work
        cfg = synth.SceneConfig(f"s{seed}", seed, n, 1.0, 0.15, 0.7, mlp, W, H, 50.0, 3.0, K, sigma_bias=sbias)
        sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
        what = dict(seed=seed, contact=contact, n=n, K=K, tile=tile, W=W, H=H, shape=(L, vd, width, nfeat, nh), sbias=sbias)
        gs, orc = api.Scene(sc), mso.OracleScene(sc)
        gs.band_bytes, gs.waves = -1, -1
        ref = [None if t is None else t.clone() for t in gs.render(cam, H, W, K, tile=tile, path=api.PATH_BF16_TC)]
        torch.cuda.synchronize()
        n_int = gs.stats().n_intervals
        o = orc.render(cam, H, W, K, tile=tile)
        d = np.abs(ref[0].cpu().numpy().reshape(-1, 3) - o[0])
        da = np.abs(ref[1].cpu().numpy().reshape(-1) - o[1])
        assert max(d.max(), da.max()) <= 2 * TOL_MAX and max(d.mean(), da.mean()) <= 2 * TOL_MEAN, (what, d.max(), da.max())
        if nfeat:
            df = np.abs(ref[2].cpu().numpy().reshape(-1, 32) - o[2])
            scale = max(1.0, np.abs(o[2]).max())
            assert df.max() <= 2 * TOL_MAX * scale and df.mean() <= 2 * TOL_MEAN * scale, (what, df.max(), scale)
        for _ in range(3):
            gs.band_bytes = int(rng.choice([-1, 32 << 10, 256 << 10, 2 << 20]))
            gs.waves = int(rng.choice([-1, 1, 2, 4]))
            fl = int(rng.choice([0, api.FLAG_OVERLAP, api.FLAG_DEBUG_ALL]))
            out = gs.render(cam, H, W, K, tile=tile, path=api.PATH_BF16_TC, flags=fl)
            torch.cuda.synchronize()
            s = gs.stats()
            for a, b in zip(out, ref):
                assert (a is None and b is None) or torch.equal(a, b), (what, gs.band_bytes, gs.waves, fl, s.n_bands, s.n_waves)
            assert s.n_intervals == n_int == o[3].n_intervals, what
            if fl == api.FLAG_DEBUG_ALL:
                assert check_structures(gs, orc, cam, H, W, K, tile, n_order_rays=3) == n_int, what
        gs.close()


def test_contact_mode_with_slot_features_random_scenes():
    """The paper's own mode with Eq.7 features on the fp32 path: the tile-owned feature kernel under random tile edges,
    image sizes (ragged tiles), C_f, band budgets and the shared per-tile order; rays with more than 32 hits included."""
    api = _api()
    rng = np.random.default_rng(4242)
    for seed in range(24):
        n = int(rng.integers(3, 150)); tile = int(rng.choice([8, 16, 32])); c_f = int(rng.choice([128, 256, 512]))
        W = int(rng.integers(9, 120)); H = int(rng.integers(9, 90))
        mlp = synth.MLPSpec(6, 0, 2, 32, 0, False, synth.MODE_CONTACT, falloff=float(rng.choice([0.0, 4.5])))
        cfg = synth.SceneConfig(f"c{seed}", seed, n, 0.8, 0.2, 0.9, mlp, W, H, 50.0, 3.0, 1,
                                sigma_bias=float(rng.choice([-1.0, 0.5, 6.0])), c_f=c_f)
        sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
        order = int(rng.choice([0, api.FLAG_TILE_ORDER]))
        what = dict(seed=seed, n=n, tile=tile, c_f=c_f, W=W, H=H, order=order)
        gs, orc = api.Scene(sc), mso.OracleScene(sc)
        orc.set_order(1 if order else 0)
        gs.band_bytes = -1
        ref = [t.clone() for t in gs.render(cam, H, W, 1, tile=tile, flags=order)]
        torch.cuda.synchronize()
        n_int = gs.stats().n_intervals
        o_rgb, o_alpha, o_feat, st = orc.render(cam, H, W, 1, tile=tile)
        assert n_int == st.n_intervals, what
        assert np.abs(ref[0].cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32, what
        assert np.abs(ref[1].cpu().numpy().reshape(-1) - o_alpha).max() <= TOL_FP32, what
        scale = max(1.0, np.abs(o_feat).max())
        assert np.abs(ref[2].cpu().numpy().reshape(-1, c_f) - o_feat).max() <= TOL_FP32 * scale, what
        for budget in (int(rng.choice([24 << 10, 200 << 10])), 0):
            gs.band_bytes = budget
            out = gs.render(cam, H, W, 1, tile=tile, flags=order | (api.FLAG_NO_SYNC if budget == 0 else 0))
            torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(out, ref)), (what, budget, gs.stats().n_bands)
        gs.close()
