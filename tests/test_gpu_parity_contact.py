"""GPU parity, contact-point mode (S:Sec.8(f) NEXT-1; the paper's own variant P:80-105): the CUDA
render through the C ABI against the oracle's contact mode on the same seeded inputs.  Same bar as
the fp32 path: tile lists, hit lists (t*, chord length) and the per-ray order bit-exact; rgb/alpha
within 1e-5 max abs."""
import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth
from test_gpu_parity_fp32 import TOL_FP32, render_both

pytestmark = pytest.mark.gpu


def _api():
    from paper_2606_03877_b200 import api
    return api


@pytest.mark.parametrize("W,H,tile", [(160, 90, 16), (97, 61, 8), (64, 36, 32)])
def test_next1_shrunk(W, H, tile):
    cfg = synth.shrink(synth.CONFIGS["next1"], W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    g, o, st = render_both(sc, cam, H, W, 1, tile=tile)
    assert st.n_intervals > 2 * W * H and st.n_samples == st.n_intervals
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32 and np.abs(g[1] - o[1]).max() <= TOL_FP32


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_contact_eye_inside_cloud(seed):
    """t* clamps to t_near when the eye is inside a support; supports straddle the eye plane."""
    mlp = synth.MLPSpec(3, 0, 1, 16, 0, False, synth.MODE_CONTACT)
    sc, cam, cfg = synth.random_tiny_scene(seed, n=16, mlp=mlp)
    g, o, st = render_both(sc, cam, cfg.height, cfg.width, 1, tile=8)
    assert st.n_intervals > 0
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32 and np.abs(g[1] - o[1]).max() <= TOL_FP32


def test_next1_full_size_sampled_pixels():
    """The bench configuration at its full 1280x720 size; the oracle computes a seeded pixel sample."""
    api = _api()
    cfg = synth.CONFIGS["next1"]
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, cfg.height, cfg.width, 1)
    torch.cuda.synchronize()
    pix = np.random.default_rng(2).choice(cfg.width * cfg.height, 20000, replace=False).astype(np.int32)
    o_rgb, o_alpha, _, st = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, 1, pixels=pix)
    assert st.n_intervals > 3 * len(pix)
    assert np.abs(rgb.cpu().numpy().reshape(-1, 3)[pix] - o_rgb).max() <= TOL_FP32
    assert np.abs(alpha.cpu().numpy().reshape(-1)[pix] - o_alpha).max() <= TOL_FP32
    a = alpha.cpu().numpy()
    assert a.min() >= 0 and a.max() <= 1 and (rgb.cpu().numpy() <= a[..., None] + 1e-6).all()


def test_contact_mode_argument_checks():
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["next1"], 32, 18)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    with pytest.raises(api.MsError):
        gs.render(cam, 18, 32, 4)                                   # K samples per chord is the other mode
    with pytest.raises(api.MsError):
        gs.render(cam, 18, 32, 1, path=api.PATH_BF16_TC)            # fp32 weights: no tensor image was packed


def test_contact_dense_scene_early_termination_and_t_near():
    """Opaque primitives (sigma-bias 8): rays stop at T < 1e-4 in contact mode too; and a camera with
    t_near > 0 (t* clamps to t_near, supports in front of it only)."""
    from dataclasses import replace
    cfg = synth.SceneConfig("dense_c", 9, 64, 1.0, 0.3, 0.8, synth.MLPSpec(4, 0, 2, 32, 0, False, synth.MODE_CONTACT),
                            96, 80, 50.0, 3.0, 1, sigma_bias=8.0)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    g, o, st = render_both(sc, cam, cfg.height, cfg.width, 1)
    assert st.n_terminated > 100
    d = np.maximum(np.abs(g[0] - o[0]).max(axis=1), np.abs(g[1] - o[1]))
    assert (d > TOL_FP32).sum() <= 2 and d.max() < 1.5e-4          # DESIGN.md Q25: stop decision fp32 vs fp64
    cam2 = replace(cam, t_near=2.6)
    g2, o2, st2 = render_both(sc, cam2, cfg.height, cfg.width, 1)
    assert 0 < st2.n_intervals < st.n_intervals
    d2 = np.maximum(np.abs(g2[0] - o2[0]).max(axis=1), np.abs(g2[1] - o2[1]))
    assert (d2 > TOL_FP32).sum() <= 2 and d2.max() < 1.5e-4


@pytest.mark.parametrize("c_f,W,H,tile", [(128, 96, 54, 16), (512, 64, 36, 16), (256, 53, 37, 8), (128, 70, 45, 32)])
def test_next2_slot_features(c_f, W, H, tile):
    """Eq.7 slot features (S:Sec.8(f) NEXT-2): gates, embeddings and the colour weights; C_f = 512 is the
    paper's width.  Features are linear in O(1) embeddings: 1e-5 relative to their range.  Tile edges 8 and
    32 on ragged images: a CTA of the feature kernel owns a whole 64-slot tile, or a quarter of a 1 024-slot one."""
    from dataclasses import replace
    api = _api()
    cfg = synth.shrink(replace(synth.CONFIGS["next2"], c_f=c_f), W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, feat = gs.render(cam, H, W, 1, tile=tile)
    torch.cuda.synchronize()
    o_rgb, o_alpha, o_feat, st = mso.OracleScene(sc).render(cam, H, W, 1, tile=tile)
    assert feat.shape == (H, W, c_f) and gs.stats().n_intervals == st.n_intervals
    assert np.abs(rgb.cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32
    assert np.abs(alpha.cpu().numpy().reshape(-1) - o_alpha).max() <= TOL_FP32
    scale = max(1.0, np.abs(o_feat).max())
    assert np.abs(feat.cpu().numpy().reshape(-1, c_f) - o_feat).max() <= TOL_FP32 * scale


def test_slot_argument_checks():
    api = _api()
    from dataclasses import replace
    cfg = synth.shrink(replace(synth.CONFIGS["next2"], c_f=96), 32, 18)        # not a multiple of 128
    with pytest.raises(api.MsError) as e:
        api.Scene(synth.make_scene(cfg))
    assert e.value.code == -4
    cfg2 = synth.shrink(synth.CONFIGS["cfg1"], 32, 18)                          # not a contact-mode scene
    sc2 = synth.make_scene(cfg2)
    sc2.slots = np.zeros((sc2.n, 4, 128), np.float32)
    with pytest.raises(api.MsError):
        api.Scene(sc2)


@pytest.mark.parametrize("W,H", [(160, 90), (97, 61)])
def test_next1_tensor_path(W, H):
    """Contact-point mode on the tcgen05 path (bf16 weights, 72-32-32-4): structures bit-exact,
    rgb/alpha at the bf16 bar of the north star (3e-3 max, 5e-4 mean per channel)."""
    from test_gpu_parity_bf16 import assert_bf16_bar
    from test_gpu_parity_fp32 import check_structures
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["next1b"], W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, H, W, 1, path=api.PATH_BF16_TC, flags=api.FLAG_DEBUG_ALL)
    torch.cuda.synchronize()
    o_rgb, o_alpha, _, st = orc.render(cam, H, W, 1)
    assert check_structures(gs, orc, cam, H, W, 1, 16, n_order_rays=8) == st.n_intervals
    assert_bf16_bar(rgb.cpu().numpy().reshape(-1, 3), alpha.cpu().numpy().reshape(-1), o_rgb, o_alpha)
    rgb32, alpha32, _ = gs.render(cam, H, W, 1, path=api.PATH_FP32)       # same scene, fp32 path: far tighter
    torch.cuda.synchronize()
    assert np.abs(rgb32.cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32


def test_contact_tensor_path_large_world_units():
    """delta = mu - p* is in world units.  Primitives with semi-axes 4-10 (delta up to ~10): the tensor
    path reduces z to [-1, 1] before the SFU sin / cos, so the top encoding bands keep the bf16 bar."""
    from test_gpu_parity_bf16 import assert_bf16_bar
    api = _api()
    mlp = synth.MLPSpec(6, 0, 2, 32, 0, True, synth.MODE_CONTACT)
    cfg = synth.SceneConfig("big_contact", 11, 24, 20.0, 4.0, 10.0, mlp, 96, 54, 60.0, 60.0, 1)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, 54, 96, 1, path=api.PATH_BF16_TC)
    torch.cuda.synchronize()
    o_rgb, o_alpha, _, st = mso.OracleScene(sc).render(cam, 54, 96, 1)
    assert st.n_intervals > 2000
    assert_bf16_bar(rgb.cpu().numpy().reshape(-1, 3), alpha.cpu().numpy().reshape(-1), o_rgb, o_alpha)


def test_contact_fp32_path_large_world_units():
    """The same scene on the fp32 path: its encode reduces 2^l z exactly to [-1, 1] before the SFU sin / cos (absolute
    error 2^-21 whatever |z|), so the 1e-5 bar holds with delta up to ~10 world units (2^5 z up to ~300)."""
    api = _api()
    mlp = synth.MLPSpec(6, 0, 2, 32, 0, False, synth.MODE_CONTACT)
    cfg = synth.SceneConfig("big_contact32", 11, 24, 20.0, 4.0, 10.0, mlp, 96, 54, 60.0, 60.0, 1)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, 54, 96, 1, path=api.PATH_FP32)
    torch.cuda.synchronize()
    o_rgb, o_alpha, _, st = mso.OracleScene(sc).render(cam, 54, 96, 1)
    assert st.n_intervals > 2000
    assert np.abs(rgb.cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32
    assert np.abs(alpha.cpu().numpy().reshape(-1) - o_alpha).max() <= TOL_FP32


def test_next1b_full_size_sampled_pixels():
    from test_gpu_parity_bf16 import assert_bf16_bar
    api = _api()
    cfg = synth.CONFIGS["next1b"]
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, cfg.height, cfg.width, 1)               # AUTO -> tensor path
    torch.cuda.synchronize()
    pix = np.random.default_rng(4).choice(cfg.width * cfg.height, 20000, replace=False).astype(np.int32)
    o_rgb, o_alpha, _, _ = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, 1, pixels=pix)
    assert_bf16_bar(rgb.cpu().numpy().reshape(-1, 3)[pix], alpha.cpu().numpy().reshape(-1)[pix], o_rgb, o_alpha)


def test_next2_slot_features_tensor_path():
    """Slot features with the MLPs on the tensor path: the gates come from the canonical fp32 geometry,
    the weights T alpha from bf16 MLPs -> the bf16 bar, relative to the features' range."""
    from dataclasses import replace
    from test_gpu_parity_bf16 import TOL_MAX, TOL_MEAN, assert_bf16_bar
    api = _api()
    cfg = synth.shrink(replace(synth.CONFIGS["next2b"], c_f=128), 96, 54)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    rgb, alpha, feat = gs.render(cam, 54, 96, 1)                            # AUTO -> tensor path
    torch.cuda.synchronize()
    o_rgb, o_alpha, o_feat, _ = mso.OracleScene(sc).render(cam, 54, 96, 1)
    assert_bf16_bar(rgb.cpu().numpy().reshape(-1, 3), alpha.cpu().numpy().reshape(-1), o_rgb, o_alpha)
    d = np.abs(feat.cpu().numpy().reshape(-1, 128) - o_feat)
    scale = max(1.0, np.abs(o_feat).max())
    assert d.max() <= TOL_MAX * scale and np.all(d.mean(axis=0) <= TOL_MEAN * scale)


@pytest.mark.parametrize("tile", [8, 16])
def test_tile_centre_order(tile):
    """MS_FLAG_TILE_ORDER: tile lists sorted by the tile-centre ray's t*, every pixel of a
    tile composited in that order -- bit-exact lists and order, rgb/alpha <= 1e-5 against the oracle's
    MSO_ORDER_TILE; and the A.4 trade-off: the image differs from the exact order, alpha does not."""
    from test_gpu_parity_fp32 import check_structures
    api = _api()
    W, H = 160, 90
    cfg = synth.shrink(synth.CONFIGS["next1"], W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    orc = mso.OracleScene(sc)
    o_rgb_e, o_alpha_e, _, _ = orc.render(cam, H, W, 1, tile=tile)
    orc.set_order(1)
    o_rgb, o_alpha, _, st = orc.render(cam, H, W, 1, tile=tile)
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, H, W, 1, tile=tile, flags=api.FLAG_DEBUG_ALL | api.FLAG_TILE_ORDER)
    torch.cuda.synchronize()
    assert check_structures(gs, orc, cam, H, W, 1, tile, n_order_rays=12) == st.n_intervals
    g_rgb, g_alpha = rgb.cpu().numpy().reshape(-1, 3), alpha.cpu().numpy().reshape(-1)
    assert np.abs(g_rgb - o_rgb).max() <= TOL_FP32 and np.abs(g_alpha - o_alpha).max() <= TOL_FP32
    assert np.abs(g_alpha - o_alpha_e).max() <= TOL_FP32 and np.abs(g_rgb - o_rgb_e).max() > 1e-3
    cfg1 = synth.shrink(synth.CONFIGS["cfg1"], 32, 18)
    with pytest.raises(api.MsError):
        api.Scene(synth.make_scene(cfg1)).render(synth.make_cameras(cfg1)[0], 18, 32, 8, flags=api.FLAG_TILE_ORDER)


def test_more_than_32_hits_per_ray_with_slot_features():
    """48 nested / overlapping supports around one point: the central rays carry 40+ hits, which takes the
    general merge of stage (e) (no lane-per-hit fast path) and hit-list cursors far into the tile list in the feature kernel."""
    api = _api()
    mlp = synth.MLPSpec(3, 0, 1, 16, 0, False, synth.MODE_CONTACT)
    rng = np.random.default_rng(21)
    n = 48
    center = rng.normal(size=(n, 3)) * 0.05
    quat = rng.normal(size=(n, 4))
    scale = rng.uniform(0.4, 1.2, size=(n, 3))
    w = synth.draw_weights(rng, n, mlp, -2.0)                 # low density: the rays do not terminate early
    slots = rng.normal(size=(n, 4, 128)).astype(np.float32)
    sc = synth.custom_scene(center, quat, scale, w, mlp, slots=slots)
    W, H = 40, 30
    cam = synth.pinhole(W, H, 40.0, synth.look_at([0.3, 0.2, 4.0]))
    gs = api.Scene(sc)
    rgb, alpha, feat = gs.render(cam, H, W, 1, flags=api.FLAG_DEBUG_ALL)
    torch.cuda.synchronize()
    orc = mso.OracleScene(sc)
    o_rgb, o_alpha, o_feat, st = orc.render(cam, H, W, 1)
    h_off, _, _, _ = gs.debug_intervals(H * W)
    assert np.diff(h_off).max() > 32 and gs.stats().n_intervals == st.n_intervals
    assert np.abs(rgb.cpu().numpy().reshape(-1, 3) - o_rgb).max() <= TOL_FP32
    assert np.abs(alpha.cpu().numpy().reshape(-1) - o_alpha).max() <= TOL_FP32
    scale_f = max(1.0, np.abs(o_feat).max())
    assert np.abs(feat.cpu().numpy().reshape(-1, 128) - o_feat).max() <= TOL_FP32 * scale_f
    ray = int(np.argmax(np.diff(h_off)))
    gp, gk, gt = gs.debug_sample_order(ray)
    op, ok, ot = orc.ray_samples(cam, H, W, 1, ray)
    assert np.array_equal(gp, op) and np.array_equal(gt.view(np.uint32), ot.view(np.uint32))
