"""Banded rendering and depth waves (S:Sec.8(f) NEXT-3; "The sorted primitives are processed sequentially ...
early t[ermination]"): neither may change a single bit of the image; bands bound the staging buffer; waves skip the
MLP work of rays that have already stopped -- never a sample the oracle evaluates."""
import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth
from test_gpu_parity_fp32 import TOL_FP32, check_structures

pytestmark = pytest.mark.gpu


def _api():
    from paper_2606_03877_b200 import api
    return api


def _render(gs, cam, H, W, K, **kw):
    out = gs.render(cam, H, W, K, **kw)
    torch.cuda.synchronize()
    return [None if t is None else t.clone() for t in out]


@pytest.mark.parametrize("name,W,H,path", [("cfg4", 240, 135, "tc"), ("cfg3", 158, 104, "fp32"), ("cfg5", 120, 68, "tc")])
def test_bands_leave_the_image_bitwise_unchanged(name, W, H, path):
    api = _api()
    cfg = synth.shrink(synth.CONFIGS[name], W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    p = api.PATH_BF16_TC if path == "tc" else api.PATH_FP32
    gs = api.Scene(sc)
    gs.band_bytes = -1                                   # one band: the whole frame staged at once
    ref = _render(gs, cam, H, W, cfg.K, path=p)
    st1 = gs.stats()
    assert st1.n_bands == 1
    for budget in (1 << 20, 300 << 10, 64 << 10):       # many bands, down to a few tiles each
        gs.band_bytes = budget
        out = _render(gs, cam, H, W, cfg.K, path=p, flags=api.FLAG_DEBUG_ALL)
        st = gs.stats()
        assert st.n_bands > 1 and st.n_intervals == st1.n_intervals and st.n_blocks >= st1.n_blocks
        assert st.staging_bytes < st1.staging_bytes
        for a, b in zip(out, ref):
            assert (a is None and b is None) or torch.equal(a, b)
        # MS_FLAG_OVERLAP: stage (e) of a band on a second stream beside stage (d) of the next, two staging halves
        ser = _render(gs, cam, H, W, cfg.K, path=p, flags=api.FLAG_OVERLAP)
        st_s = gs.stats()
        assert st_s.n_bands >= st.n_bands and st_s.n_intervals == st1.n_intervals
        for a, b in zip(ser, ref):
            assert (a is None and b is None) or torch.equal(a, b)
    # the structures of a banded frame against the oracle (tile lists, per-ray intervals, sample order of every ray)
    orc = mso.OracleScene(sc)
    assert check_structures(gs, orc, cam, H, W, cfg.K, 16, n_order_rays=4) == st1.n_intervals


def test_bands_on_ragged_image_with_eye_inside_the_cloud():
    """odd image size (tiles overhanging the border), supports that cover the whole image, 8-pixel tiles"""
    api = _api()
    sc, cam, cfg = synth.random_tiny_scene(2)
    H, W = 37, 53
    cam = synth.pinhole(W, H, cfg.fov_deg, cam.c2w)
    gs = api.Scene(sc)
    gs.band_bytes = -1
    ref = _render(gs, cam, H, W, cfg.K, path=api.PATH_FP32, tile=8)
    gs.band_bytes = 4 << 10
    out = _render(gs, cam, H, W, cfg.K, path=api.PATH_FP32, tile=8, flags=api.FLAG_DEBUG_ALL)
    assert gs.stats().n_bands > 2
    assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])
    orc = mso.OracleScene(sc)
    o_rgb, o_alpha, _, st = orc.render(cam, H, W, cfg.K, tile=8)
    assert check_structures(gs, orc, cam, H, W, cfg.K, 8, n_order_rays=4) == st.n_intervals
    assert np.abs(out[0].cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32


@pytest.mark.parametrize("path", ["fp32", "tc"])
@pytest.mark.parametrize("waves,band_bytes", [(1, -1), (2, -1), (2, 256 << 10), (4, 1 << 20)])
def test_depth_waves_skip_work_but_not_a_bit_of_the_image(path, waves, band_bytes):
    """Opaque scene (sigma-bias 8): most rays stop after a few hits.  With depth waves the intervals of stopped rays
    are never encoded: fewer samples evaluated than the frame holds, never fewer than the oracle evaluates, and
    the image is bitwise the one rendered without waves."""
    api = _api()
    if path == "tc":
        cfg = synth.SceneConfig("dense_tc", 7, 48, 1.0, 0.3, 0.8, synth.MLPSpec(6, 0, 2, 128, 0, True),
                                96, 80, 50.0, 3.0, 8, sigma_bias=8.0)
        sc = synth.make_scene(cfg)
        p = api.PATH_BF16_TC
    else:
        sc, cfg = synth.dense_scene()
        p = api.PATH_FP32
    cam = synth.make_cameras(cfg)[0]
    H, W, K = cfg.height, cfg.width, cfg.K
    gs = api.Scene(sc)
    gs.waves, gs.band_bytes = -1, -1
    ref = _render(gs, cam, H, W, K, path=p)
    st0 = gs.stats()
    assert st0.n_waves == 1 and st0.n_samples_evaluated == st0.n_samples and st0.n_dead_rays == 0
    gs.waves, gs.band_bytes = waves, band_bytes
    out = _render(gs, cam, H, W, K, path=p, flags=api.FLAG_DEBUG_ALL)
    st = gs.stats()
    assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])
    assert st.n_waves > 1 and st.n_dead_rays > 100
    _, _, _, ost = mso.OracleScene(sc).render(cam, H, W, K)
    assert ost.n_terminated > 200
    assert ost.n_mlp_evals <= st.n_samples_evaluated < 0.97 * st.n_samples
    assert st.n_samples == ost.n_samples
    # structures are those of the oracle whatever the wave layout
    orc = mso.OracleScene(sc)
    assert check_structures(gs, orc, cam, H, W, K, 16, n_order_rays=4) == ost.n_intervals


def test_waves_auto_switch_on_after_a_view_with_stopped_rays():
    api = _api()
    sc, cfg = synth.dense_scene()
    cam = synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)                                   # waves = 0: MS_WAVES_AUTO
    a = _render(gs, cam, cfg.height, cfg.width, cfg.K, path=api.PATH_FP32)
    assert gs.stats().n_waves == 1                       # no history yet
    b = _render(gs, cam, cfg.height, cfg.width, cfg.K, path=api.PATH_FP32)
    st = gs.stats()
    assert st.n_waves > 1 and st.n_samples_evaluated < st.n_samples
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])
    # a scene whose rays never stop stays on the single-wave path
    cfg1 = synth.CONFIGS["cfg1"]
    gs1 = api.Scene(synth.make_scene(cfg1))
    for _ in range(2):
        _render(gs1, synth.make_cameras(cfg1)[0], cfg1.height, cfg1.width, cfg1.K)
    assert gs1.stats().n_waves == 1


def test_waves_never_drop_a_sample_in_front_of_the_stop():
    """Waves with t_stop = 0 are off (nothing may ever be skipped); with a huge threshold rays stop at their first
    samples and still agree bitwise."""
    api = _api()
    sc, cfg = synth.dense_scene()
    cam = synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    gs.waves = 1
    _render(gs, cam, cfg.height, cfg.width, cfg.K, path=api.PATH_FP32, t_stop=0.0)
    assert gs.stats().n_waves == 1
    for t_stop in (0.3, 1e-2, 1e-6):
        gs.waves = -1
        ref = _render(gs, cam, cfg.height, cfg.width, cfg.K, path=api.PATH_FP32, t_stop=t_stop)
        gs.waves = 1
        out = _render(gs, cam, cfg.height, cfg.width, cfg.K, path=api.PATH_FP32, t_stop=t_stop)
        assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])


@pytest.mark.parametrize("case", ["contact_fp32", "contact_tc_slots", "feat_tc_tile8", "k64_tile32", "k5_ragged"])
def test_bands_and_waves_across_modes(case):
    """Bands x waves in every mode that reaches stages (d), (e): the paper's contact-point mode (K = 1, with and
    without Eq.7 slot features), the widened feature head on the tensor path, the tile sizes 8 and 32, K = 64 and a K
    that does not divide the 128-row block -- opaque media, so the waves do drop intervals.  Always: bitwise the
    image (and features) of the one-band, no-wave render, fewer samples evaluated, structures those of the oracle."""
    api = _api()
    tile, K, path = 16, 8, api.PATH_FP32
    if case == "contact_fp32":
        mlp = synth.MLPSpec(6, 0, 2, 32, 0, False, synth.MODE_CONTACT, falloff=0.0)   # no falloff (Q29's parameter): opaque hits
        cfg = synth.SceneConfig(case, 21, 160, 1.0, 0.2, 0.6, mlp, 80, 60, 50.0, 3.0, 1, sigma_bias=9.0)
        K = 1
    elif case == "contact_tc_slots":
        mlp = synth.MLPSpec(6, 0, 2, 32, 0, True, synth.MODE_CONTACT, falloff=0.5)
        cfg = synth.SceneConfig(case, 22, 160, 1.0, 0.2, 0.6, mlp, 80, 60, 50.0, 3.0, 1, sigma_bias=9.0, c_f=128)
        K, path = 1, api.PATH_BF16_TC
    elif case == "feat_tc_tile8":
        mlp = synth.MLPSpec(4, 1, 3, 64, 32, True)
        cfg = synth.SceneConfig(case, 23, 64, 1.0, 0.3, 0.8, mlp, 72, 50, 50.0, 3.0, 6, sigma_bias=8.0)
        tile, K, path = 8, 6, api.PATH_BF16_TC
    elif case == "k64_tile32":
        mlp = synth.MLPSpec(4, 0, 2, 32, 0, False)
        cfg = synth.SceneConfig(case, 24, 40, 1.0, 0.3, 0.8, mlp, 70, 45, 50.0, 3.0, 64, sigma_bias=6.0)
        tile, K = 32, 64
    else:
        mlp = synth.MLPSpec(4, 0, 3, 64, 0, True)
        cfg = synth.SceneConfig(case, 25, 64, 1.0, 0.3, 0.8, mlp, 61, 47, 50.0, 3.0, 5, sigma_bias=8.0)
        K, path = 5, api.PATH_BF16_TC
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    H, W = cfg.height, cfg.width
    gs = api.Scene(sc)
    gs.waves, gs.band_bytes = -1, -1
    ref = _render(gs, cam, H, W, K, path=path, tile=tile)
    st0 = gs.stats()
    for waves, band_bytes, fl in ((2, -1, 0), (1, 96 << 10, 0), (3, 512 << 10, 0), (2, 96 << 10, api.FLAG_OVERLAP)):
        gs.waves, gs.band_bytes = waves, band_bytes
        out = _render(gs, cam, H, W, K, path=path, tile=tile, flags=api.FLAG_DEBUG_ALL | fl)
        st = gs.stats()
        for a, b in zip(out, ref):
            assert (a is None and b is None) or torch.equal(a, b)
        assert st.n_waves > 1 and st.n_samples == st0.n_samples
        assert st.n_samples_evaluated < st.n_samples and st.n_dead_rays > 0
        if band_bytes > 0:
            assert st.n_bands > 1
    orc = mso.OracleScene(sc)
    _, _, _, ost = orc.render(cam, H, W, K, tile=tile)
    assert ost.n_mlp_evals <= st.n_samples_evaluated
    assert check_structures(gs, orc, cam, H, W, K, tile, n_order_rays=4) == ost.n_intervals
