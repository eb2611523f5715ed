"""Thin Python binding of the C ABI in include/mlpsplat.h (argument marshalling only: every
step of the render runs in the CUDA kernels of csrc/).  torch is used for device buffers and
streams.  There is NO CPU fallback: importing this module without the built CUDA library
raises, and so does calling it without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libmlpsplat.so")

MS_F32, MS_BF16 = 0, 1
PATH_AUTO, PATH_FP32, PATH_BF16_TC = 0, 1, 2
FLAG_KEEP_DEBUG, FLAG_STAGE_TIMES = 1, 2
FLAG_KEEP_ORDER = 8     # stage (e) records the order it composited in (ms_debug_sample_order*)
FLAG_NO_SYNC = 16        # no host synchronisation when the previous view sized the scratch (ms_opts.flags)
FLAG_OVERLAP = 32       # banded views: stage (e) of a band on a second stream beside stage (d) of the next (off by default)
FLAG_DEBUG_ALL = FLAG_KEEP_DEBUG | FLAG_KEEP_ORDER
FLAG_TILE_ORDER = 4     # contact mode: the paper's shared per-tile order instead of the exact per-ray order
STAGES = ("bin", "sort", "isect", "mlp", "composite")

EXPORTS = ["ms_scene_create", "ms_scene_set_slots", "ms_scene_destroy", "ms_render", "ms_render_batch", "ms_render_host",
           "ms_backward", "ms_last_stats", "ms_last_stage_ms", "ms_stage_accum", "ms_debug_tile_lists", "ms_debug_intervals",
           "ms_debug_sample_order", "ms_debug_sample_order_all", "ms_debug_prim_frames", "ms_launch_count_total", "ms_error_string", "ms_last_cuda_error",
           "ms_exclusive_scan_device", "ms_exclusive_scan_static"]


class _Prims(C.Structure):
    _fields_ = [("n", C.c_int32), ("center", C.c_void_p), ("quat", C.c_void_p), ("scale", C.c_void_p)]


class _MLP(C.Structure):
    _fields_ = [("n_freq", C.c_int32), ("use_viewdir", C.c_int32), ("n_hidden", C.c_int32),
                ("width", C.c_int32), ("n_feat", C.c_int32), ("dtype", C.c_int32),
                ("weights", C.c_void_p), ("n_weights", C.c_size_t), ("mode", C.c_int32), ("falloff", C.c_float)]


class _Camera(C.Structure):
    _fields_ = [("fx", C.c_float), ("fy", C.c_float), ("cx", C.c_float), ("cy", C.c_float),
                ("c2w", C.c_float * 12), ("t_near", C.c_float)]


class _Opts(C.Structure):
    _fields_ = [("K", C.c_int32), ("t_stop", C.c_float), ("tile", C.c_int32), ("path", C.c_int32),
                ("stream", C.c_void_p), ("flags", C.c_int32), ("band_bytes", C.c_int64), ("waves", C.c_int32),
                ("eye_guard", C.c_float)]


class _Stats(C.Structure):
    _fields_ = [("n_visible", C.c_int64), ("n_pairs", C.c_int64), ("n_intervals", C.c_int64),
                ("n_samples", C.c_int64), ("n_blocks", C.c_int64), ("scratch_bytes", C.c_int64),
                ("n_launches", C.c_int64), ("n_samples_evaluated", C.c_int64), ("n_dead_rays", C.c_int64),
                ("n_bands", C.c_int64), ("n_waves", C.c_int64), ("staging_bytes", C.c_int64), ("overflow", C.c_int64),
                ("no_sync", C.c_int64)]


def _load() -> C.CDLL:
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2606_03877_b200.build` "
            "(or __graft_entry__.build()). There is no CPU or PyTorch fallback.")
    lib = C.CDLL(_LIB_PATH)
    for name in EXPORTS:
        getattr(lib, name)  # fail loudly on a stale library
    lib.ms_error_string.restype = C.c_char_p
    lib.ms_launch_count_total.restype = C.c_int64
    lib.ms_scene_destroy.argtypes = [C.c_void_p]
    lib.ms_scene_set_slots.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    for name in ("ms_exclusive_scan_device", "ms_exclusive_scan_static"):
        getattr(lib, name).argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
    return lib


_lib = _load()


def launch_count() -> int:
    """Kernels this host thread has launched through the library so far (ms_launch_count_total)."""
    return int(_lib.ms_launch_count_total())


class MsError(RuntimeError):
    def __init__(self, code: int, where: str, cuda: int = 0):
        self.code = code
        self.cuda = cuda
        msg = _lib.ms_error_string(code).decode()
        super().__init__(f"{where}: {msg} ({code})" + (f", cudaError {cuda}" if cuda else ""))


SCAN_STATIC_MAX = 1 << 24   # MS_SCAN_STATIC_MAX: the largest n ms_exclusive_scan_static covers


def exclusive_scan(counts: "torch.Tensor", out: "torch.Tensor | None" = None, static: bool = False, stream=None):
    """out[i] = sum(counts[:i]) for i in [0, n] (uint32 arithmetic on int32 CUDA tensors): the offset scan of stages
    (a), (c), (d).  static=False: ms_exclusive_scan_device (the render's path; allocates its scratch and synchronises).
    static=True: ms_exclusive_scan_static -- allocates nothing, scratch in a fixed device array, n <= SCAN_STATIC_MAX,
    calls must not overlap on the GPU (include/mlpsplat.h).  Argument marshalling only."""
    if not (counts.is_cuda and counts.dtype == torch.int32 and counts.is_contiguous() and counts.dim() == 1):
        raise ValueError("counts: contiguous 1-D int32 CUDA tensor")
    n = counts.numel()
    if out is None:
        out = torch.empty(n + 1, dtype=torch.int32, device=counts.device)
    if not (out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() >= n + 1):
        raise ValueError("out: contiguous int32 CUDA tensor of n + 1 elements")
    s = torch.cuda.current_stream(counts.device).cuda_stream if stream is None else stream
    fn = _lib.ms_exclusive_scan_static if static else _lib.ms_exclusive_scan_device
    with torch.cuda.device(counts.device):
        rc = fn(_ptr(counts), _ptr(out), n, C.c_void_p(s))
    if rc != 0:
        raise MsError(rc, "ms_exclusive_scan_static" if static else "ms_exclusive_scan_device")
    return out


def _ptr(a):
    if a is None:
        return None
    if isinstance(a, torch.Tensor):
        return C.c_void_p(a.data_ptr())
    return a.ctypes.data_as(C.c_void_p)


def _cam_struct(cam) -> _Camera:
    return _Camera(cam.fx, cam.fy, cam.cx, cam.cy, (C.c_float * 12)(*[float(v) for v in cam.c2w]),
                   float(cam.t_near))


@dataclass
class Stats:
    n_pairs: int
    n_intervals: int
    n_samples: int
    n_blocks: int
    scratch_bytes: int
    n_launches: int
    n_visible: int = 0
    n_samples_evaluated: int = 0
    n_dead_rays: int = 0
    n_bands: int = 1
    n_waves: int = 1
    staging_bytes: int = 0
    overflow: int = 0
    no_sync: int = 0


class Scene:
    """Device-resident scene (ms_scene_create).  `scene` needs center/quat/scale/weights arrays
    and an `mlp` spec (see synth.Scene)."""

    def __init__(self, scene, dtype: int | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_03877_b200 needs a CUDA device; there is no CPU fallback")
        torch.cuda.init()
        torch.zeros(1, device="cuda")  # make sure the primary context exists
        self.mlp = scene.mlp
        self.n = int(scene.center.shape[0])
        center = np.ascontiguousarray(scene.center, np.float32)
        quat = np.ascontiguousarray(scene.quat, np.float32)
        scale = np.ascontiguousarray(scene.scale, np.float32)
        weights = np.ascontiguousarray(scene.weights, np.float32)
        if dtype is None:
            dtype = MS_BF16 if scene.mlp.bf16 else MS_F32
        self.dtype = dtype
        p = _Prims(self.n, _ptr(center), _ptr(quat), _ptr(scale))
        m = _MLP(scene.mlp.n_freq, scene.mlp.use_viewdir, scene.mlp.n_hidden, scene.mlp.width,
                 scene.mlp.n_feat, dtype, _ptr(weights), weights.size, int(getattr(scene.mlp, "mode", 0)),
                 float(getattr(scene.mlp, "falloff", 4.5)))
        h = C.c_void_p()
        rc = _lib.ms_scene_create(C.byref(p), C.byref(m), C.byref(h))
        if rc != 0:
            raise MsError(rc, "ms_scene_create")
        self._h = h
        self.c_f = 0                                   # Eq.7 slot features (ms_scene_set_slots)
        slots = getattr(scene, "slots", None)
        if slots is not None:
            emb = np.ascontiguousarray(slots, np.float32)
            if emb.ndim != 3 or emb.shape[:2] != (self.n, 4):
                raise ValueError("slots must be [n][4][c_f]")
            rc = _lib.ms_scene_set_slots(self._h, int(emb.shape[2]), _ptr(emb))
            if rc != 0:
                raise MsError(rc, "ms_scene_set_slots")
            self.c_f = int(emb.shape[2])

    def close(self):
        h = getattr(self, "_h", None)
        if h and _lib is not None:
            _lib.ms_scene_destroy(h)
        self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, where: str):
        if rc != 0:
            raise MsError(rc, where, _lib.ms_last_cuda_error(self._h))

    # band_bytes / waves / eye_guard of every render of this scene (ms_opts; 0 = the library's defaults)
    band_bytes: int = 0
    waves: int = 0
    eye_guard: float = 0.0

    def _opts(self, K, t_stop, tile, path, flags, stream=None) -> _Opts:
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        return _Opts(K, t_stop, tile, path, C.c_void_p(stream), flags, int(self.band_bytes), int(self.waves),
                     float(self.eye_guard))

    # -- rendering ---------------------------------------------------------------
    def render(self, cam, H, W, K, *, t_stop=1e-4, tile=16, path=PATH_AUTO, flags=0, out=None,
               want_feat=True, stream=None):
        """One view -> (rgb [H,W,3], alpha [H,W], feat [H,W,F] | None) float32 CUDA tensors."""
        nf = (self.c_f or self.mlp.n_feat) if want_feat else 0
        if out is None:
            rgb = torch.empty((H, W, 3), dtype=torch.float32, device="cuda")
            alpha = torch.empty((H, W), dtype=torch.float32, device="cuda")
            feat = torch.empty((H, W, nf), dtype=torch.float32, device="cuda") if nf else None
        else:
            rgb, alpha, feat = out
        o = self._opts(K, t_stop, tile, path, flags, stream)
        c = _cam_struct(cam)
        self._check(_lib.ms_render(self._h, C.byref(c), C.c_int32(H), C.c_int32(W), C.byref(o),
                                   _ptr(rgb), _ptr(alpha), _ptr(feat)), "ms_render")
        return rgb, alpha, feat

    def render_batch(self, cams, H, W, K, *, t_stop=1e-4, tile=16, path=PATH_AUTO, flags=0, out=None,
                     want_feat=True, stream=None):
        V = len(cams)
        nf = (self.c_f or self.mlp.n_feat) if want_feat else 0
        if out is None:
            rgb = torch.empty((V, H, W, 3), dtype=torch.float32, device="cuda")
            alpha = torch.empty((V, H, W), dtype=torch.float32, device="cuda")
            feat = torch.empty((V, H, W, nf), dtype=torch.float32, device="cuda") if nf else None
        else:
            rgb, alpha, feat = out
        arr = (_Camera * V)(*[_cam_struct(c) for c in cams])
        o = self._opts(K, t_stop, tile, path, flags, stream)
        self._check(_lib.ms_render_batch(self._h, arr, C.c_int32(V), C.c_int32(H), C.c_int32(W),
                                         C.byref(o), _ptr(rgb), _ptr(alpha), _ptr(feat)),
                    "ms_render_batch")
        return rgb, alpha, feat

    def render_host(self, cams, H, W, K, *, t_stop=1e-4, tile=16, path=PATH_AUTO, flags=0, out=None,
                    want_feat=True, stream=None):
        """End-to-end entry: HOST (pinned) output buffers, device->host copies inside the call."""
        V = len(cams)
        nf = (self.c_f or self.mlp.n_feat) if want_feat else 0
        if out is None:
            rgb = torch.empty((V, H, W, 3), dtype=torch.float32).pin_memory()
            alpha = torch.empty((V, H, W), dtype=torch.float32).pin_memory()
            feat = torch.empty((V, H, W, nf), dtype=torch.float32).pin_memory() if nf else None
        else:
            rgb, alpha, feat = out
        arr = (_Camera * V)(*[_cam_struct(c) for c in cams])
        o = self._opts(K, t_stop, tile, path, flags, stream)
        self._check(_lib.ms_render_host(self._h, arr, C.c_int32(V), C.c_int32(H), C.c_int32(W),
                                        C.byref(o), _ptr(rgb), _ptr(alpha), _ptr(feat)),
                    "ms_render_host")
        return rgb, alpha, feat

    def backward(self, cam, H, W, K, d_rgb, *, t_stop=1e-4, tile=16, grads=None, stream=None):
        """ms_backward: d_rgb = dL/d out_rgb, float32 CUDA [H, W, 3].  Returns (g_weights [n, P], g_center [n, 3],
        g_quat [n, 4], g_scale [n, 3]) float32 CUDA tensors; pass `grads` to accumulate into existing ones."""
        if grads is None:
            P = self.mlp.params_per_prim
            grads = (torch.zeros((self.n, P), dtype=torch.float32, device="cuda"),
                     torch.zeros((self.n, 3), dtype=torch.float32, device="cuda"),
                     torch.zeros((self.n, 4), dtype=torch.float32, device="cuda"),
                     torch.zeros((self.n, 3), dtype=torch.float32, device="cuda"))
        d_rgb = d_rgb.contiguous()
        assert d_rgb.dtype == torch.float32 and d_rgb.is_cuda and d_rgb.numel() == H * W * 3
        o = self._opts(K, t_stop, tile, PATH_FP32, 0, stream)
        c = _cam_struct(cam)
        self._check(_lib.ms_backward(self._h, C.byref(c), C.c_int32(H), C.c_int32(W), C.byref(o), _ptr(d_rgb),
                                     _ptr(grads[0]), _ptr(grads[1]), _ptr(grads[2]), _ptr(grads[3])), "ms_backward")
        return grads

    # -- introspection -------------------------------------------------------------
    def stats(self) -> Stats:
        st = _Stats()
        rc = _lib.ms_last_stats(self._h, C.byref(st))
        if rc not in (0, -5):                      # -5: a no-sync view that overflowed its scratch (st.overflow = 1)
            self._check(rc, "ms_last_stats")
        return Stats(st.n_pairs, st.n_intervals, st.n_samples, st.n_blocks, st.scratch_bytes, st.n_launches,
                     st.n_visible, st.n_samples_evaluated, st.n_dead_rays, st.n_bands, st.n_waves, st.staging_bytes,
                     st.overflow, st.no_sync)

    def stage_ms(self) -> dict[str, float]:
        ms = (C.c_float * len(STAGES))()
        self._check(_lib.ms_last_stage_ms(self._h, ms), "ms_last_stage_ms")
        return {k: float(v) for k, v in zip(STAGES, ms)}

    def stage_accum(self, reset: bool = False):
        """(sum of per-stage ms over the views rendered with FLAG_STAGE_TIMES, number of views)."""
        ms = (C.c_double * len(STAGES))()
        n = C.c_int64(0)
        self._check(_lib.ms_stage_accum(self._h, ms, C.byref(n), C.c_int32(1 if reset else 0)),
                    "ms_stage_accum")
        return {k: float(v) for k, v in zip(STAGES, ms)}, int(n.value)

    def debug_tile_lists(self, n_tiles: int):
        n = C.c_size_t(0)
        rc = _lib.ms_debug_tile_lists(self._h, None, None, None, C.c_size_t(0), C.byref(n))
        if rc not in (0, -5):
            self._check(rc, "ms_debug_tile_lists")
        off = np.zeros(n_tiles + 1, np.int64)
        prim = np.zeros(max(n.value, 1), np.int32)
        zb = np.zeros(max(n.value, 1), np.uint32)
        self._check(_lib.ms_debug_tile_lists(self._h, _ptr(off), _ptr(prim), _ptr(zb),
                                             C.c_size_t(prim.size), C.byref(n)), "ms_debug_tile_lists")
        return off, prim[:n.value], zb[:n.value]

    def debug_intervals(self, n_rays: int):
        n = C.c_size_t(0)
        rc = _lib.ms_debug_intervals(self._h, None, None, None, None, C.c_size_t(0), C.byref(n))
        if rc not in (0, -5):
            self._check(rc, "ms_debug_intervals")
        off = np.zeros(n_rays + 1, np.int64)
        prim = np.zeros(max(n.value, 1), np.int32)
        t_in = np.zeros(max(n.value, 1), np.float32)
        delta = np.zeros(max(n.value, 1), np.float32)
        self._check(_lib.ms_debug_intervals(self._h, _ptr(off), _ptr(prim), _ptr(t_in), _ptr(delta),
                                            C.c_size_t(prim.size), C.byref(n)), "ms_debug_intervals")
        return off, prim[:n.value], t_in[:n.value], delta[:n.value]

    def debug_sample_order(self, ray: int):
        n = C.c_size_t(0)
        rc = _lib.ms_debug_sample_order(self._h, C.c_int32(ray), None, None, None, C.c_size_t(0),
                                        C.byref(n))
        if rc not in (0, -5):
            self._check(rc, "ms_debug_sample_order")
        prim = np.zeros(max(n.value, 1), np.int32)
        k = np.zeros(max(n.value, 1), np.int32)
        t = np.zeros(max(n.value, 1), np.float32)
        self._check(_lib.ms_debug_sample_order(self._h, C.c_int32(ray), _ptr(prim), _ptr(k), _ptr(t),
                                               C.c_size_t(prim.size), C.byref(n)),
                    "ms_debug_sample_order")
        return prim[:n.value], k[:n.value], t[:n.value]

    def debug_sample_order_all(self):
        """(prim, k) of every sample in the order stage (e) composited it, rays in pixel order (FLAG_KEEP_ORDER)."""
        n = C.c_size_t(0)
        rc = _lib.ms_debug_sample_order_all(self._h, None, None, C.c_size_t(0), C.byref(n))
        if rc not in (0, -5):
            self._check(rc, "ms_debug_sample_order_all")
        prim = np.zeros(max(n.value, 1), np.int32)
        k = np.zeros(max(n.value, 1), np.int32)
        self._check(_lib.ms_debug_sample_order_all(self._h, _ptr(prim), _ptr(k), C.c_size_t(prim.size), C.byref(n)),
                    "ms_debug_sample_order_all")
        return prim[:n.value], k[:n.value]

    def debug_prim_frames(self):
        A = np.zeros((self.n, 3, 3), np.float32)
        M = np.zeros((self.n, 3, 3), np.float32)
        self._check(_lib.ms_debug_prim_frames(self._h, _ptr(A), _ptr(M)), "ms_debug_prim_frames")
        return A, M
