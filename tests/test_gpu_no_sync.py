"""MS_FLAG_NO_SYNC (S:Sec.3 "no device->host sync inside ms_render"): a view enqueued without any
host synchronisation, its scratch sized from the previous view -- bitwise the synchronising render; a view that does
not fit is reported, never silently wrong."""
import numpy as np
import pytest
import torch

from paper_2606_03877_b200 import synth

pytestmark = pytest.mark.gpu


def _api():
    from paper_2606_03877_b200 import api
    return api


@pytest.mark.parametrize("name,W,H,path", [("cfg1", 64, 64, "fp32"), ("cfg2", 200, 200, "tc"), ("cfg5", 120, 68, "tc"),
                                           ("next2", 96, 54, "fp32")])
def test_no_sync_view_equals_the_synchronising_one(name, W, H, path):
    api = _api()
    from dataclasses import replace
    cfg = synth.shrink(synth.CONFIGS[name], W, H)
    if cfg.c_f:
        cfg = replace(cfg, c_f=128)
    sc, cams = synth.make_scene(cfg), synth.make_cameras(cfg)
    p = api.PATH_BF16_TC if path == "tc" else api.PATH_FP32
    gs = api.Scene(sc)
    ref = [t.clone() if t is not None else None for t in gs.render(cams[0], H, W, cfg.K, path=p)]
    torch.cuda.synchronize()
    st0 = gs.stats()
    assert st0.no_sync == 0 and st0.n_bands == 1
    for _ in range(3):
        out = gs.render(cams[0], H, W, cfg.K, path=p, flags=api.FLAG_NO_SYNC)
        torch.cuda.synchronize()
        st = gs.stats()
        assert st.no_sync == 1 and st.overflow == 0
        assert (st.n_pairs, st.n_intervals, st.n_samples) == (st0.n_pairs, st0.n_intervals, st0.n_samples)
        for a, b in zip(out, ref):
            assert (a is None and b is None) or torch.equal(a, b)
    # another pose of the same shape: still no synchronisation, and equal to its own synchronising render
    cam2 = cams[1] if len(cams) > 1 else synth.pinhole(W, H, cfg.fov_deg, synth.look_at(synth.eye_from_angles(cfg.radius, 50.0, 12.0)))
    out = [t.clone() if t is not None else None for t in gs.render(cam2, H, W, cfg.K, path=p, flags=api.FLAG_NO_SYNC)]
    torch.cuda.synchronize()
    st = gs.stats()
    ref2 = gs.render(cam2, H, W, cfg.K, path=p)
    torch.cuda.synchronize()
    if st.overflow:
        assert st.no_sync == 1                      # reported; the synchronising render above has regrown the scratch
    else:
        for a, b in zip(out, ref2):
            assert (a is None and b is None) or torch.equal(a, b)


def test_no_sync_overflow_is_reported_and_recovered():
    """History from a view that sees the scene from far away, then a view full of primitives: it cannot fit, says so
    (ms_last_stats: MS_ERR_CAPACITY, overflow = 1), and the next render sizes again."""
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["cfg3"], 158, 104)
    sc = synth.make_scene(cfg)
    W, H = cfg.width, cfg.height
    away = synth.pinhole(W, H, 20.0, synth.look_at([0.0, 0.0, 90.0]))     # the whole scene in a few pixels
    cam = synth.make_cameras(cfg)[0]
    gs = api.Scene(sc)
    gs.render(away, H, W, cfg.K, path=api.PATH_FP32)
    torch.cuda.synchronize()
    assert 10 < gs.stats().n_intervals < 20000
    gs.render(cam, H, W, cfg.K, path=api.PATH_FP32, flags=api.FLAG_NO_SYNC)
    torch.cuda.synchronize()
    st = gs.stats()
    assert st.no_sync == 1 and st.overflow == 1
    ref = [t.clone() for t in gs.render(cam, H, W, cfg.K, path=api.PATH_FP32, flags=api.FLAG_NO_SYNC)[:2]]   # no history: synchronises
    torch.cuda.synchronize()
    st = gs.stats()
    assert st.no_sync == 0 and st.overflow == 0 and st.n_intervals > 1000
    out = gs.render(cam, H, W, cfg.K, path=api.PATH_FP32, flags=api.FLAG_NO_SYNC)
    torch.cuda.synchronize()
    assert gs.stats().no_sync == 1 and gs.stats().overflow == 0
    assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])


def test_no_sync_small_frame_in_tile_order_and_with_nothing_in_view():
    """The fused small-frame launches (stages (a) + (b) by one CTA; ray scan, tile statistics and pair order by one CTA)
    in the paper's shared per-tile order (MS_FLAG_TILE_ORDER: keys carry the tile-centre contact depth), and on a view
    that sees no primitive at all after one that saw many (zero pairs: every list empty, background only)."""
    api = _api()
    cfg = synth.shrink(synth.CONFIGS["next1"], 96, 54)
    sc, cam = synth.make_scene(cfg), synth.make_cameras(cfg)[0]
    H, W = cfg.height, cfg.width
    gs = api.Scene(sc)
    fl = api.FLAG_TILE_ORDER
    ref = [t.clone() for t in gs.render(cam, H, W, 1, flags=fl)[:2]]
    torch.cuda.synchronize()
    assert gs.stats().no_sync == 0 and 0 < gs.stats().n_pairs <= 16384
    launches = []
    for _ in range(2):
        n0 = api.launch_count()
        out = gs.render(cam, H, W, 1, flags=fl | api.FLAG_NO_SYNC)
        launches.append(api.launch_count() - n0)
        torch.cuda.synchronize()
        assert gs.stats().no_sync == 1 and gs.stats().overflow == 0
        assert torch.equal(out[0], ref[0]) and torch.equal(out[1], ref[1])
    assert launches[-1] <= 8, launches                     # fused (a)+(b), count, order, fill, MLP, composite (+ scan)
    # the same scene seen from behind the camera plane: nothing projects
    away = synth.pinhole(W, H, cfg.fov_deg, synth.look_at([0.0, 0.0, 60.0], target=[0.0, 0.0, 120.0]))
    blank = gs.render(away, H, W, 1, flags=fl | api.FLAG_NO_SYNC)
    torch.cuda.synchronize()
    st = gs.stats()
    assert st.no_sync == 1 and st.overflow == 0 and st.n_pairs == 0 and st.n_intervals == 0
    assert float(blank[0].abs().max()) == 0.0 and float(blank[1].abs().max()) == 0.0
    back = gs.render(cam, H, W, 1, flags=fl | api.FLAG_NO_SYNC)          # and the scratch still serves the full view
    torch.cuda.synchronize()
    assert gs.stats().overflow == 0 and torch.equal(back[0], ref[0])
