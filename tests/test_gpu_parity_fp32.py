"""GPU parity, fp32 SIMT path: the CUDA render (through the C ABI) against the CPU oracle on the
same seeded inputs.  NS bar: tile lists, interval counts, sample order bit-exact; rgb/alpha
within 1e-5 max abs."""
import numpy as np
import pytest
import torch

from oracle import mso
from paper_2606_03877_b200 import synth

pytestmark = pytest.mark.gpu

TOL_FP32 = 1e-5      # NS: "rgb/alpha within 1e-5 max abs for the fp32 path"


def _api():
    from paper_2606_03877_b200 import api
    return api


def check_structures(gs, orc, cam, H, W, K, tile, n_order_rays=24):
    """bit-exact: tile lists, per-ray interval lists, and the order stage (e) composited EVERY ray's samples in
    (recorded by the composite kernel itself under FLAG_KEEP_ORDER); sample positions t on the busiest rays."""
    n_tiles = ((W + tile - 1) // tile) * ((H + tile - 1) // tile)
    g_off, g_prim, g_z = gs.debug_tile_lists(n_tiles)
    o_off, o_prim, o_z = orc.tile_lists(cam, H, W, tile)
    assert np.array_equal(g_off, o_off)
    assert np.array_equal(g_prim, o_prim)
    assert np.array_equal(g_z, o_z)
    h_off, h_prim, h_tin, h_dl = gs.debug_intervals(H * W)
    r_off, r_prim, r_tin, r_dl = orc.intervals_all(cam, H, W, K, tile)
    assert np.array_equal(h_off, r_off)                      # interval counts per ray
    # the GPU lists are in tile-list order; the oracle dump is sorted by primitive id
    ray_of = np.repeat(np.arange(H * W), np.diff(h_off))
    order = np.lexsort((h_prim, ray_of))
    assert np.array_equal(h_prim[order], r_prim)
    assert np.array_equal(h_tin[order].view(np.uint32), r_tin.view(np.uint32))
    assert np.array_equal(h_dl[order].view(np.uint32), r_dl.view(np.uint32))
    # sample ordering, every ray: (primitive, k) by rank
    s_prim, s_k = gs.debug_sample_order_all()
    q_prim, q_k = orc.samples_all(cam, H, W, K, tile)
    assert s_prim.size == int(h_off[-1]) * K
    assert np.array_equal(s_prim, q_prim) and np.array_equal(s_k, q_k)
    counts = np.diff(h_off)
    busiest = np.argsort(-counts, kind="stable")[:n_order_rays]
    for ray in busiest:
        if counts[ray] == 0:
            continue
        gp, gk, gt = gs.debug_sample_order(int(ray))
        op, ok, ot = orc.ray_samples(cam, H, W, K, int(ray), tile)
        assert np.array_equal(gp, op) and np.array_equal(gk, ok)
        assert np.array_equal(gt.view(np.uint32), ot.view(np.uint32))
    return int(h_off[-1])


def render_both(sc, cam, H, W, K, tile=16, path=None, t_stop=1e-4, structures=True):
    api = _api()
    path = api.PATH_FP32 if path is None else path
    orc = mso.OracleScene(sc)
    gs = api.Scene(sc)
    rgb, alpha, feat = gs.render(cam, H, W, K, tile=tile, path=path, t_stop=t_stop,
                                 flags=api.FLAG_DEBUG_ALL)
    torch.cuda.synchronize()
    o_rgb, o_alpha, o_feat, st = orc.render(cam, H, W, K, tile=tile, t_stop=t_stop)
    if structures:
        n_hits = check_structures(gs, orc, cam, H, W, K, tile)
        assert n_hits == st.n_intervals == gs.stats().n_intervals
        assert gs.stats().n_pairs == st.n_pairs
    g_rgb = rgb.cpu().numpy().reshape(-1, 3).astype(np.float64)
    g_alpha = alpha.cpu().numpy().reshape(-1).astype(np.float64)
    g_feat = feat.cpu().numpy().reshape(H * W, -1).astype(np.float64) if feat is not None else None
    gs.close()
    return (g_rgb, g_alpha, g_feat), (o_rgb, o_alpha, o_feat), st


def test_prim_frames_bit_exact():
    api = _api()
    sc = synth.make_scene(synth.CONFIGS["cfg3"])
    A, M = api.Scene(sc).debug_prim_frames()
    oA, oM = mso.OracleScene(sc).frames()
    assert np.array_equal(A.view(np.uint32), oA.view(np.uint32))
    assert np.array_equal(M.view(np.uint32), oM.view(np.uint32))


@pytest.mark.parametrize("tile", [8, 16, 32])
def test_cfg1_fp32(tile):
    """BASELINE.json configs[0]: 16 primitives, 27-32-32-4 fp32, 64x64, K=8."""
    cfg = synth.CONFIGS["cfg1"]
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    g, o, st = render_both(sc, cam, cfg.height, cfg.width, cfg.K, tile=tile)
    assert st.n_intervals == 1378
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32
    assert np.abs(g[1] - o[1]).max() <= TOL_FP32
    miss = o[1] == 0
    assert not g[0][miss].any() and not g[1][miss].any()       # exact zeros off every support


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
@pytest.mark.parametrize("tile", [8, 16])
def test_random_tiny_scenes_eye_inside_cloud(seed, tile):
    """supports behind / around / straddling the eye plane and the image border; ragged tiles."""
    sc, cam, cfg = synth.random_tiny_scene(seed)
    g, o, st = render_both(sc, cam, cfg.height, cfg.width, cfg.K, tile=tile)
    assert st.n_intervals > 50
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32
    assert np.abs(g[1] - o[1]).max() <= TOL_FP32


@pytest.mark.parametrize("name,W,H", [("cfg2", 200, 200), ("cfg3", 158, 104), ("cfg4", 240, 135)])
def test_shrunk_configs_fp32_path(name, W, H):
    """cfg2-4 scenes and poses at a reduced image (several tiles + a ragged tail), fp32 math on
    the same (bf16-valued) weights."""
    cfg = synth.shrink(synth.CONFIGS[name], W, H)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    g, o, st = render_both(sc, cam, H, W, cfg.K)
    assert st.n_intervals > 1000
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32
    assert np.abs(g[1] - o[1]).max() <= TOL_FP32


def test_feature_head_fp32_path():
    """cfg5 head (4 + 32 linear feature channels), composited with the same weights."""
    cfg = synth.shrink(synth.CONFIGS["cfg5"], 120, 68)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[1]
    g, o, st = render_both(sc, cam, 68, 120, cfg.K)
    assert g[2].shape == (68 * 120, 32)
    assert np.abs(g[0] - o[0]).max() <= TOL_FP32
    assert np.abs(g[1] - o[1]).max() <= TOL_FP32
    # features are unbounded linear outputs: same relative bar, scaled by their magnitude
    assert np.abs(g[2] - o[2]).max() <= TOL_FP32 * max(1.0, np.abs(o[2]).max())


def test_dense_scene_early_termination():
    """pin P9 on the GPU: rays stop once T < 1e-4.  The stop decision is taken in fp32 on the GPU
    and fp64 in the oracle (Q25): a ray whose T lands within rounding of the threshold
    may stop one sample apart, which changes the pixel by < t_stop."""
    sc, cfg = synth.dense_scene()
    cam = synth.make_cameras(cfg)[0]
    g, o, st = render_both(sc, cam, cfg.height, cfg.width, cfg.K)
    assert st.n_terminated > 200
    d = np.maximum(np.abs(g[0] - o[0]).max(axis=1), np.abs(g[1] - o[1]))
    assert (d > TOL_FP32).sum() <= 2 and d.max() < 1.5e-4
    # disabling the threshold must change the terminated rays, identically on both sides
    g2, o2, st2 = render_both(sc, cam, cfg.height, cfg.width, cfg.K, t_stop=0.0, structures=False)
    assert st2.n_terminated == 0
    assert np.abs(g2[0] - o2[0]).max() <= TOL_FP32 and np.abs(g2[1] - o2[1]).max() <= TOL_FP32
    assert np.abs(o2[1] - o[1]).max() > 1e-6


def test_empty_and_degenerate_inputs():
    api = _api()
    mlp = synth.MLPSpec(2, 0, 1, 8, 0, False)
    w = synth.constant_mlp_weights(mlp, [0, 0, 0, 1.0])
    # a primitive entirely behind the camera: nothing visible, zero pairs, all-zero image
    sc = synth.custom_scene([[0, 0, 9.0]], [[1, 0, 0, 0]], [[0.5, 0.5, 0.5]], w[None], mlp)
    cam = synth.pinhole(19, 7, 50.0, synth.look_at([0, 0, 4.0]))
    gs = api.Scene(sc)
    rgb, alpha, _ = gs.render(cam, 7, 19, 4, path=api.PATH_FP32)
    torch.cuda.synchronize()
    assert gs.stats().n_pairs == 0 and gs.stats().n_intervals == 0
    assert not rgb.any().item() and not alpha.any().item()
    # 1x1 image, K = 1
    sc1 = synth.custom_scene([[0, 0, 0.0]], [[1, 0, 0, 0]], [[0.5, 0.5, 0.5]], w[None], mlp)
    g, o, st = render_both(sc1, synth.pinhole(1, 1, 50.0, synth.look_at([0, 0, 4.0])), 1, 1, 1)
    assert st.n_intervals == 1 and abs(g[1][0] - o[1][0]) <= TOL_FP32
    # invalid arguments are reported, never crash
    with pytest.raises(api.MsError):
        api.Scene(synth.custom_scene([[0, 0, 0]], [[0, 0, 0, 0]], [[1, 1, 1]], w[None], mlp))
    with pytest.raises(api.MsError):
        api.Scene(synth.custom_scene([[0, 0, 0]], [[1, 0, 0, 0]], [[1, -1, 1]], w[None], mlp))
    with pytest.raises(api.MsError):
        gs.render(cam, 7, 19, 0, path=api.PATH_FP32)
    with pytest.raises(api.MsError):
        gs.render(cam, 7, 19, 4, tile=12, path=api.PATH_FP32)


def test_render_batch_and_host_entry_match_single_view():
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["cfg5"], 64, 36)
    sc, cams = synth.make_scene(cfg), synth.make_cameras(cfg)[:5]     # five views: the host entry's two output buffers
    gs = api.Scene(sc)                                                # are each reused (copy of view v beside view v + 1)
    singles = [gs.render(c, 36, 64, cfg.K, path=api.PATH_FP32) for c in cams]
    singles = [[t.clone() for t in s] for s in singles]
    rgb, alpha, feat = gs.render_batch(cams, 36, 64, cfg.K, path=api.PATH_FP32)
    h_rgb, h_alpha, h_feat = gs.render_host(cams, 36, 64, cfg.K, path=api.PATH_FP32)
    h1 = gs.render_host(cams[3:4], 36, 64, cfg.K, path=api.PATH_FP32)          # one view: no second stream
    torch.cuda.synchronize()
    assert torch.equal(h1[0][0], singles[3][0].cpu()) and torch.equal(h1[2][0], singles[3][2].cpu())
    for v, s in enumerate(singles):
        assert torch.equal(rgb[v], s[0]) and torch.equal(alpha[v], s[1]) and torch.equal(feat[v], s[2])
        assert torch.equal(h_rgb[v], s[0].cpu()) and torch.equal(h_alpha[v], s[1].cpu())
        assert torch.equal(h_feat[v], s[2].cpu())


@pytest.mark.parametrize("K,t_stop", [(16, 1e-4), (16, 0.0), (3, 1e-4)])
def test_more_than_32_hits_and_multi_window_rays(K, t_stop):
    """48 overlapping supports around one point: the central rays carry 40+ hits and, at K = 16, more than
    448 samples -- the uncached-hit branch of the merge and the windowed compositing of stage (e),
    with and without early termination inside a later window."""
    mlp = synth.MLPSpec(2, 0, 2, 32, 0, False)
    rng = np.random.default_rng(33)
    n = 48
    center = rng.normal(size=(n, 3)) * 0.05
    quat = rng.normal(size=(n, 4))
    scale = rng.uniform(0.4, 1.2, size=(n, 3))
    w = synth.draw_weights(rng, n, mlp, -1.0 if t_stop == 0.0 else 1.0)
    sc = synth.custom_scene(center, quat, scale, w, mlp)
    W, H = 24, 18
    cam = synth.pinhole(W, H, 40.0, synth.look_at([0.3, 0.2, 4.0]))
    g, o, st = render_both(sc, cam, H, W, K, t_stop=t_stop)
    assert st.n_intervals > 32 * 20 and (K < 16 or st.n_samples / (W * H) > 448 * 0.5)
    d = np.maximum(np.abs(g[0] - o[0]).max(axis=1), np.abs(g[1] - o[1]))
    if t_stop == 0.0:
        assert d.max() <= TOL_FP32                                  # no stop decision: the plain north-star bar
    else:
        assert (d > TOL_FP32).sum() <= 2 and d.max() < 1.5e-4      # Q25: stop decision fp32 vs fp64
