"""ctypes loader for the CPU oracle (oracle/libmso.so).

TEST INFRASTRUCTURE ONLY -- see oracle/mso.h.  Allowed importers: tests/,
__graft_entry__.smoke(), bench.py's cpu_baseline and `--impl reference` legs.
This module never imports the CUDA binding; it takes plain numpy arrays.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build


class _Prims(C.Structure):
    _fields_ = [("n", C.c_int32), ("center", C.c_void_p), ("quat", C.c_void_p), ("scale", C.c_void_p)]


class _MLP(C.Structure):
    _fields_ = [("n_freq", C.c_int32), ("use_viewdir", C.c_int32), ("n_hidden", C.c_int32),
                ("width", C.c_int32), ("n_feat", C.c_int32), ("weights", C.c_void_p), ("mode", C.c_int32),
                ("falloff", C.c_float)]


class _Camera(C.Structure):
    _fields_ = [("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("c2w", C.c_float * 12), ("t_near", C.c_float)]


class _Opts(C.Structure):
    _fields_ = [("K", C.c_int32), ("t_stop", C.c_float), ("tile", C.c_int32), ("n_threads", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("n_pixels", C.c_int64), ("n_intervals", C.c_int64), ("n_samples", C.c_int64),
                ("n_mlp_evals", C.c_int64), ("n_terminated", C.c_int64), ("n_pairs", C.c_int64),
                ("min_T", C.c_double)]


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.mso_scene_create.restype = C.c_int
        _lib.mso_scene_destroy.restype = None
        _lib.mso_scene_destroy.argtypes = [C.c_void_p]
    return _lib


def _ptr(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _cam(cam) -> _Camera:
    c = _Camera(cam.fx, cam.fy, cam.cx, cam.cy, (C.c_float * 12)(*[float(v) for v in cam.c2w]),
                cam.t_near)
    return c


@dataclass
class Stats:
    n_pixels: int
    n_intervals: int
    n_samples: int
    n_mlp_evals: int
    n_terminated: int
    n_pairs: int
    min_T: float


class OracleScene:
    """Owns an mso_scene built from a synth.Scene-like object (numpy arrays)."""

    def __init__(self, scene):
        self._keep = (np.ascontiguousarray(scene.center, np.float32),
                      np.ascontiguousarray(scene.quat, np.float32),
                      np.ascontiguousarray(scene.scale, np.float32),
                      np.ascontiguousarray(scene.weights, np.float32))
        self.mlp = scene.mlp
        self.n = int(self._keep[0].shape[0])
        p = _Prims(self.n, _ptr(self._keep[0]), _ptr(self._keep[1]), _ptr(self._keep[2]))
        m = _MLP(scene.mlp.n_freq, scene.mlp.use_viewdir, scene.mlp.n_hidden, scene.mlp.width,
                 scene.mlp.n_feat, _ptr(self._keep[3]), int(getattr(scene.mlp, "mode", 0)),
                 float(getattr(scene.mlp, "falloff", 4.5)))
        h = C.c_void_p()
        rc = lib().mso_scene_create(C.byref(p), C.byref(m), C.byref(h))
        if rc != 0:
            raise ValueError(f"mso_scene_create failed: {rc}")
        self._h = h
        self.c_f = 0
        slots = getattr(scene, "slots", None)
        if slots is not None:
            emb = np.ascontiguousarray(slots, np.float32)
            assert emb.shape[:2] == (self.n, 4)
            rc = lib().mso_scene_set_slots(self._h, C.c_int32(emb.shape[2]), _ptr(emb))
            if rc != 0:
                raise ValueError(f"mso_scene_set_slots failed: {rc}")
            self.c_f = int(emb.shape[2])

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            lib().mso_scene_destroy(h)
            self._h = None

    # -- render ------------------------------------------------------------
    def render(self, cam, H, W, K, *, t_stop=1e-4, tile=16, pixels=None, n_threads=0,
               want_feat=True):
        """Returns (rgb[n,3], alpha[n], feat[n,F] or None, Stats); fp64."""
        if pixels is not None:
            pixels = np.ascontiguousarray(pixels, np.int32)
            n = int(pixels.size)
        else:
            n = H * W
        rgb = np.zeros((n, 3), np.float64)
        alpha = np.zeros((n,), np.float64)
        nf = self.c_f or self.mlp.n_feat
        feat = np.zeros((n, nf), np.float64) if (nf and want_feat) else None
        st = _Stats()
        o = _Opts(K, t_stop, tile, n_threads)
        c = _cam(cam)
        rc = lib().mso_render(self._h, C.byref(c), C.c_int(H), C.c_int(W), C.byref(o),
                              _ptr(pixels), C.c_int64(n), _ptr(rgb), _ptr(alpha), _ptr(feat),
                              C.byref(st))
        if rc != 0:
            raise RuntimeError(f"mso_render failed: {rc}")
        stats = Stats(st.n_pixels, st.n_intervals, st.n_samples, st.n_mlp_evals, st.n_terminated,
                      st.n_pairs, st.min_T)
        return rgb, alpha, feat, stats

    # -- parity artefacts ----------------------------------------------------
    def tile_lists(self, cam, H, W, tile):
        n = C.c_size_t(0)
        c = _cam(cam)
        tiles = ((W + tile - 1) // tile) * ((H + tile - 1) // tile)
        off = np.zeros(tiles + 1, np.int64)
        rc = lib().mso_tile_lists(self._h, C.byref(c), H, W, tile, None, None, None,
                                  C.c_size_t(0), C.byref(n))
        if rc not in (0, -3):
            raise RuntimeError(f"mso_tile_lists failed: {rc}")
        prim = np.zeros(max(n.value, 1), np.int32)
        zb = np.zeros(max(n.value, 1), np.uint32)
        rc = lib().mso_tile_lists(self._h, C.byref(c), H, W, tile, _ptr(off), _ptr(prim), _ptr(zb),
                                  C.c_size_t(prim.size), C.byref(n))
        if rc != 0:
            raise RuntimeError(f"mso_tile_lists failed: {rc}")
        return off, prim[:n.value], zb[:n.value]

    def hit_counts(self, cam, H, W, K, tile=16, n_threads=0):
        out = np.zeros(H * W, np.int32)
        o = _Opts(K, 1e-4, tile, n_threads)
        c = _cam(cam)
        rc = lib().mso_hit_counts(self._h, C.byref(c), H, W, C.byref(o), _ptr(out))
        if rc != 0:
            raise RuntimeError(f"mso_hit_counts failed: {rc}")
        return out

    def ray_intervals(self, cam, H, W, K, pixel, tile=16):
        cap = self.n
        prim = np.zeros(cap, np.int32)
        t_in = np.zeros(cap, np.float32)
        delta = np.zeros(cap, np.float32)
        n = C.c_size_t(0)
        o = _Opts(K, 1e-4, tile, 1)
        c = _cam(cam)
        rc = lib().mso_ray_intervals(self._h, C.byref(c), H, W, C.byref(o), C.c_int32(pixel),
                                     _ptr(prim), _ptr(t_in), _ptr(delta), C.c_size_t(cap),
                                     C.byref(n))
        if rc != 0:
            raise RuntimeError(f"mso_ray_intervals failed: {rc}")
        return prim[:n.value], t_in[:n.value], delta[:n.value]

    def intervals_all(self, cam, H, W, K, tile=16):
        """(offsets[H*W+1], prim, t_in, delta), each ray's hits sorted by primitive id."""
        off = np.zeros(H * W + 1, np.int64)
        n = C.c_size_t(0)
        o = _Opts(K, 1e-4, tile, 1)
        c = _cam(cam)
        rc = lib().mso_intervals_all(self._h, C.byref(c), H, W, C.byref(o), _ptr(off), None, None,
                                     None, C.c_size_t(0), C.byref(n))
        if rc not in (0, -3):
            raise RuntimeError(f"mso_intervals_all failed: {rc}")
        prim = np.zeros(max(n.value, 1), np.int32)
        t_in = np.zeros(max(n.value, 1), np.float32)
        delta = np.zeros(max(n.value, 1), np.float32)
        rc = lib().mso_intervals_all(self._h, C.byref(c), H, W, C.byref(o), _ptr(off), _ptr(prim),
                                     _ptr(t_in), _ptr(delta), C.c_size_t(prim.size), C.byref(n))
        if rc != 0:
            raise RuntimeError(f"mso_intervals_all failed: {rc}")
        return off, prim[:n.value], t_in[:n.value], delta[:n.value]

    def samples_all(self, cam, H, W, K, tile=16):
        """(prim, k) of every sample of every pixel in compositing order (aligned with intervals_all's offsets * K)."""
        n = C.c_size_t(0)
        o = _Opts(K, 1e-4, tile, 1)
        c = _cam(cam)
        rc = lib().mso_samples_all(self._h, C.byref(c), H, W, C.byref(o), None, None, C.c_size_t(0), C.byref(n))
        if rc not in (0, -3):
            raise RuntimeError(f"mso_samples_all failed: {rc}")
        prim = np.zeros(max(n.value, 1), np.int32)
        k = np.zeros(max(n.value, 1), np.int32)
        rc = lib().mso_samples_all(self._h, C.byref(c), H, W, C.byref(o), _ptr(prim), _ptr(k),
                                   C.c_size_t(prim.size), C.byref(n))
        if rc != 0:
            raise RuntimeError(f"mso_samples_all failed: {rc}")
        return prim[:n.value], k[:n.value]

    def set_eye_guard(self, g: float):
        rc = lib().mso_scene_set_eye_guard(self._h, C.c_float(g))
        if rc != 0:
            raise ValueError(f"mso_scene_set_eye_guard failed: {rc}")

    def ray_samples(self, cam, H, W, K, pixel, tile=16):
        cap = self.n * K
        prim = np.zeros(cap, np.int32)
        k = np.zeros(cap, np.int32)
        t = np.zeros(cap, np.float32)
        n = C.c_size_t(0)
        o = _Opts(K, 1e-4, tile, 1)
        c = _cam(cam)
        rc = lib().mso_ray_samples(self._h, C.byref(c), H, W, C.byref(o), C.c_int32(pixel),
                                   _ptr(prim), _ptr(k), _ptr(t), C.c_size_t(cap), C.byref(n))
        if rc != 0:
            raise RuntimeError(f"mso_ray_samples failed: {rc}")
        return prim[:n.value], k[:n.value], t[:n.value]

    # -- pieces --------------------------------------------------------------
    def frames(self):
        A = np.zeros((self.n, 3, 3), np.float32)
        M = np.zeros((self.n, 3, 3), np.float32)
        lib().mso_prim_frames(self._h, _ptr(A), _ptr(M))
        return A, M

    def project(self, cam, H, W, prim):
        vis = C.c_int32(0)
        rect = (C.c_int32 * 4)()
        z = C.c_float(0)
        c = _cam(cam)
        rc = lib().mso_project(self._h, C.byref(c), H, W, C.c_int32(prim), C.byref(vis), rect,
                               C.byref(z))
        if rc != 0:
            raise RuntimeError(f"mso_project failed: {rc}")
        return bool(vis.value), tuple(rect), z.value

    def mlp_eval(self, prim, u, d=None):
        u = np.ascontiguousarray(u, np.float32)
        d = np.ascontiguousarray(d if d is not None else [0, 0, 1], np.float32)
        raw = np.zeros(self.mlp.out_dim, np.float64)
        act = np.zeros(self.mlp.out_dim, np.float64)
        rc = lib().mso_mlp_eval(self._h, C.c_int32(prim), _ptr(u), _ptr(d), _ptr(raw), _ptr(act))
        if rc != 0:
            raise RuntimeError(f"mso_mlp_eval failed: {rc}")
        return raw, act

    def set_order(self, order: int):
        """0: exact per-ray order; 1: the paper's shared per-tile order of the tile-centre ray (contact mode)."""
        rc = lib().mso_scene_set_order(self._h, C.c_int32(order))
        if rc != 0:
            raise ValueError(f"mso_scene_set_order failed: {rc}")

    def slot_gates(self, prim, delta):
        g = np.zeros(4, np.float64)
        dl = np.ascontiguousarray(delta, np.float32)
        rc = lib().mso_slot_gates(self._h, C.c_int32(prim), _ptr(dl), _ptr(g))
        if rc != 0:
            raise RuntimeError(f"mso_slot_gates failed: {rc}")
        return g

    def contact_eval(self, prim, o, d, t):
        """contact mode: (x, raw, act, r2) of primitive prim at o + t d."""
        o = np.ascontiguousarray(o, np.float32)
        d = np.ascontiguousarray(d, np.float32)
        x = np.zeros(self.mlp.in_dim, np.float64)
        raw = np.zeros(self.mlp.out_dim, np.float64)
        act = np.zeros(self.mlp.out_dim, np.float64)
        r2 = C.c_double()
        rc = lib().mso_contact_eval(self._h, C.c_int32(prim), _ptr(o), _ptr(d), C.c_float(t), _ptr(x), _ptr(raw),
                                    _ptr(act), C.byref(r2))
        if rc != 0:
            raise RuntimeError(f"mso_contact_eval failed: {rc}")
        return x, raw, act, r2.value

    def encode(self, u, d=None):
        u = np.ascontiguousarray(u, np.float32)
        d = np.ascontiguousarray(d if d is not None else [0, 0, 1], np.float32)
        x = np.zeros(self.mlp.in_dim, np.float64)
        rc = lib().mso_encode(self._h, _ptr(u), _ptr(d), _ptr(x))
        if rc != 0:
            raise RuntimeError(f"mso_encode failed: {rc}")
        return x


def ray(cam, x, y):
    o = np.zeros(3, np.float32)
    d = np.zeros(3, np.float32)
    c = _cam(cam)
    lib().mso_ray(C.byref(c), C.c_int(x), C.c_int(y), _ptr(o), _ptr(d))
    return o, d


def loss_grad_f64(scene, cam, H, W, K, *, center=None, quat=None, scale=None, weights=None, t_stop=1e-4,
                  pixels=None, target=None, g_in=None, want_grad=True):
    """fp64 forward (+ backward) of the render (mso_grad.c).  The scene's arrays may be overridden by fp64 arrays
    (the finite-difference pins perturb those).  Returns dict(loss, rgb, g_weights, g_center, g_quat, g_scale)."""
    n = int(scene.center.shape[0])
    c64 = np.ascontiguousarray(scene.center if center is None else center, np.float64)
    q64 = np.ascontiguousarray(scene.quat if quat is None else quat, np.float64)
    s64 = np.ascontiguousarray(scene.scale if scale is None else scale, np.float64)
    w64 = np.ascontiguousarray(scene.weights if weights is None else weights, np.float64)
    m = _MLP(scene.mlp.n_freq, scene.mlp.use_viewdir, scene.mlp.n_hidden, scene.mlp.width, scene.mlp.n_feat,
             None, int(getattr(scene.mlp, "mode", 0)), float(getattr(scene.mlp, "falloff", 4.5)))
    if pixels is not None:
        pixels = np.ascontiguousarray(pixels, np.int32)
        npx = int(pixels.size)
    else:
        npx = H * W
    tgt = None if target is None else np.ascontiguousarray(target, np.float64).reshape(npx, 3)
    gin = None if g_in is None else np.ascontiguousarray(g_in, np.float64).reshape(npx, 3)
    loss = C.c_double(0.0)
    rgb = np.zeros((npx, 3), np.float64)
    gw = np.zeros_like(w64) if want_grad else None
    gc = np.zeros_like(c64) if want_grad else None
    gq = np.zeros_like(q64) if want_grad else None
    gs = np.zeros_like(s64) if want_grad else None
    c = _cam(cam)
    rc = lib().mso_loss_grad_f64(C.c_int32(n), _ptr(c64), _ptr(q64), _ptr(s64), _ptr(w64), C.byref(m), C.byref(c),
                                 C.c_int(H), C.c_int(W), C.c_int(K), C.c_double(t_stop), _ptr(pixels),
                                 C.c_int64(npx), _ptr(tgt), _ptr(gin), C.byref(loss), _ptr(rgb), _ptr(gw), _ptr(gc),
                                 _ptr(gq), _ptr(gs))
    if rc != 0:
        raise RuntimeError(f"mso_loss_grad_f64 failed: {rc}")
    return dict(loss=loss.value, rgb=rgb, g_weights=gw, g_center=gc, g_quat=gq, g_scale=gs)
