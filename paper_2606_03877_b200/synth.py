"""Seeded synthetic scenes and cameras for MLP-Splatting (arxiv/paper_2606_03877).

This module is the ONLY code shared by the CUDA path and the CPU oracle.  It
draws random numbers and lays them out; it holds none of the method's
arithmetic (no ray casting, no MLP evaluation, no compositing).  It imports
neither `oracle/` nor the CUDA binding.

The scenes stand in for the paper's trained Replica / ScanNet scenes
(Table 2: 0.9-2.6 k primitives per scene, one
compact MLP per primitive PAPER.md:148), with the shapes BASELINE.json
`configs` prescribes.  Recipe (DESIGN.md §"Input recipe"):

  rng = numpy default_rng(seed); fixed draw order
    centres      U(-box, box)^3
    quaternions  N(0,1)^4, normalised, order (w,x,y,z)
    semi-axes    exp(U(ln s_min, ln s_max))^3
    per layer    W ~ U(-sqrt(6/fan_in), +sqrt(6/fan_in))   ("Kaiming-uniform")
    biases       0, except the density output (channel 3 of the head) = 0.5
  everything cast to float32; for bf16 configs the weight matrices AND biases
  are then rounded to bf16 (round-to-nearest-even) and stored back as float32
  values, so oracle and GPU receive bit-identical numbers.

Per-primitive weight blob layout (float32 values), documented once here and in
include/mlpsplat.h:   for each layer l = 0..n_hidden:  W_l[in_l][out_l]
row-major (input index slowest), then b_l[out_l].
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np


MODE_LOCAL, MODE_CONTACT = 0, 1


@dataclass(frozen=True)
class MLPSpec:
    n_freq: int          # L of Eq.5
    use_viewdir: int     # 0/1: raw world-frame unit d appended after the encoding
    n_hidden: int        # hidden Linear+ReLU layers
    width: int           # hidden width
    n_feat: int          # extra linear output channels after [r,g,b,sigma]
    bf16: bool           # weights are bf16-representable values
    mode: int = 0        # 0: north-star input (local coords, K samples); 1: the paper's contact-point input (S:§8(f) NEXT-1)
    falloff: float = 4.5 # contact mode: g = exp(-falloff |p*-mu|^2_Lambda) (Q29; a parameter, default 9/2)

    @property
    def in_dim(self) -> int:
        if self.mode == MODE_CONTACT:
            return 12 * self.n_freq            # gamma([d; delta]) of Eq.4-5: 6 scalars x 2L, no identity
        return 3 + 6 * self.n_freq + (3 if self.use_viewdir else 0)

    @property
    def out_dim(self) -> int:
        return 4 + self.n_feat

    @property
    def layer_dims(self) -> list[tuple[int, int]]:
        dims = [self.in_dim] + [self.width] * self.n_hidden + [self.out_dim]
        return list(zip(dims[:-1], dims[1:]))

    @property
    def params_per_prim(self) -> int:
        return sum(i * o + o for i, o in self.layer_dims)

    @property
    def flop_per_sample(self) -> int:
        """Algorithmic (unpadded) 2*MAC per MLP evaluation."""
        return sum(2 * i * o for i, o in self.layer_dims)


@dataclass(frozen=True)
class SceneConfig:
    name: str
    seed: int
    n_prims: int
    box: float
    s_min: float
    s_max: float
    mlp: MLPSpec
    width: int           # image W
    height: int          # image H
    fov_deg: float       # horizontal FOV
    radius: float        # eye distance from origin
    K: int               # midpoint samples per interval
    n_views: int = 1
    pose_seed: int = 5
    sigma_bias: float = 0.5
    t_stop: float = 1e-4
    tile: int = 16
    c_f: int = 0         # C_f of Eq.7: four slot embeddings of this width per primitive (0 = none)


CONFIGS: dict[str, SceneConfig] = {
    # BASELINE.json configs[0..4]; seeds / eye radii per SURVEY.md §8(d), Q19.
    "cfg1": SceneConfig("cfg1", 0, 16, 1.0, 0.1, 0.4,
                        MLPSpec(4, 0, 2, 32, 0, False), 64, 64, 50.0, 3.0, 8),
    "cfg2": SceneConfig("cfg2", 1, 256, 1.0, 0.05, 0.3,
                        MLPSpec(4, 0, 3, 64, 0, True), 800, 800, 40.0, 4.0, 16),
    "cfg3": SceneConfig("cfg3", 2, 1024, 2.0, 0.05, 0.5,
                        MLPSpec(4, 1, 3, 64, 0, True), 1264, 832, 60.0, 3.0, 16),
    "cfg4": SceneConfig("cfg4", 3, 4096, 3.0, 0.03, 0.4,
                        MLPSpec(6, 0, 3, 128, 0, True), 1920, 1080, 60.0, 5.0, 24),
    "cfg5": SceneConfig("cfg5", 2, 1024, 2.0, 0.05, 0.5,
                        MLPSpec(4, 1, 3, 64, 32, True), 1920, 1080, 60.0, 5.0, 16,
                        n_views=8),
    # S:§8(f) NEXT-1, the paper's own variant: one evaluation per (ray, primitive) at
    # the contact point, 72-32-32-4 fp32 MLPs on gamma([d; delta]); N in the paper's range (Table 6).
    "next1": SceneConfig("next1", 6, 2048, 2.0, 0.05, 0.5,
                         MLPSpec(6, 0, 2, 32, 0, False, MODE_CONTACT), 1280, 720, 60.0, 5.0, 1),
    # S:§8(f) NEXT-2: the same scene with the paper's feature model (Eq.7): 4 slot embeddings of
    # C_f = 512 per primitive, gated by a tetrahedral frame, composited with the colour weights.
    # next1 with bf16 weights: the same mode on the tcgen05 path (32-wide MLPs), at the bf16 parity bar
    "next1b": SceneConfig("next1b", 6, 2048, 2.0, 0.05, 0.5,
                          MLPSpec(6, 0, 2, 32, 0, True, MODE_CONTACT), 1280, 720, 60.0, 5.0, 1),
    "next2b": SceneConfig("next2b", 6, 2048, 2.0, 0.05, 0.5,
                          MLPSpec(6, 0, 2, 32, 0, True, MODE_CONTACT), 1280, 720, 60.0, 5.0, 1, c_f=512),
    "next2": SceneConfig("next2", 6, 2048, 2.0, 0.05, 0.5,
                         MLPSpec(6, 0, 2, 32, 0, False, MODE_CONTACT), 1280, 720, 60.0, 5.0, 1, c_f=512),
    # S:§8(f) NEXT-3: CFG4's shape with an opaque medium (density bias 8, as in the early-termination pin P9): the
    # paper's trained scenes are opaque surfaces ("early t[ermination]"), CFG1-5 never terminate a ray
    "cfg4_opaque": SceneConfig("cfg4_opaque", 3, 4096, 3.0, 0.03, 0.4,
                               MLPSpec(6, 0, 3, 128, 0, True), 1920, 1080, 60.0, 5.0, 24, sigma_bias=8.0),
    # CFG4's scene seen from INSIDE the primitive cloud (the paper's Replica / ScanNet rooms): supports
    # around and behind the eye, long tile lists
    "cfg4_inside": SceneConfig("cfg4_inside", 3, 4096, 3.0, 0.03, 0.4,
                               MLPSpec(6, 0, 3, 128, 0, True), 1920, 1080, 60.0, 0.5, 24),
}


def shrink(cfg: SceneConfig, width: int, height: int, **kw) -> SceneConfig:
    """Same scene and camera pose at a smaller image (for oracle-sized parity)."""
    return replace(cfg, width=width, height=height, **kw)


def round_to_bf16(a: np.ndarray) -> np.ndarray:
    """float32 -> nearest bf16 (ties to even) -> float32.  Input formatting only."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """float32 array holding bf16-representable values -> uint16 bf16 bit patterns."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32)
    assert np.all((u & 0xFFFF) == 0), "values are not bf16-representable"
    return (u >> 16).astype(np.uint16)


@dataclass
class Scene:
    center: np.ndarray   # [N,3] f32
    quat: np.ndarray     # [N,4] f32, (w,x,y,z)
    scale: np.ndarray    # [N,3] f32 semi-axes
    weights: np.ndarray  # [N, params_per_prim] f32 values
    mlp: MLPSpec
    slots: np.ndarray | None = None   # [N, 4, C_f] f32 slot embeddings e_ik of Eq.7, contact mode only

    @property
    def n(self) -> int:
        return int(self.center.shape[0])


@dataclass
class Camera:
    fx: float
    fy: float
    cx: float
    cy: float
    c2w: np.ndarray      # [12] f32, 3x4 row-major, x right / y down / z forward
    t_near: float = 0.0
    width: int = 0
    height: int = 0


def draw_weights(rng: np.random.Generator, n: int, mlp: MLPSpec, sigma_bias: float) -> np.ndarray:
    blobs = []
    n_layers = len(mlp.layer_dims)
    for li, (fan_in, fan_out) in enumerate(mlp.layer_dims):
        bound = math.sqrt(6.0 / fan_in)
        W = rng.uniform(-bound, bound, size=(n, fan_in, fan_out))
        b = np.zeros((n, fan_out))
        if li == n_layers - 1:
            b[:, 3] = sigma_bias
        blobs.append(W.reshape(n, -1))
        blobs.append(b)
    w = np.concatenate(blobs, axis=1).astype(np.float32)
    if mlp.bf16:
        w = round_to_bf16(w)
    assert w.shape[1] == mlp.params_per_prim
    return np.ascontiguousarray(w)


def make_scene(cfg: SceneConfig) -> Scene:
    rng = np.random.default_rng(cfg.seed)
    n = cfg.n_prims
    center = rng.uniform(-cfg.box, cfg.box, size=(n, 3))
    q = rng.normal(size=(n, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    log_s = rng.uniform(math.log(cfg.s_min), math.log(cfg.s_max), size=(n, 3))
    scale = np.exp(log_s)
    weights = draw_weights(rng, n, cfg.mlp, cfg.sigma_bias)
    slots = rng.normal(size=(n, 4, cfg.c_f)).astype(np.float32) if cfg.c_f else None   # drawn last: earlier draws unchanged
    return Scene(np.ascontiguousarray(center, dtype=np.float32),
                 np.ascontiguousarray(q, dtype=np.float32),
                 np.ascontiguousarray(scale, dtype=np.float32),
                 weights, cfg.mlp, slots)


def look_at(eye, target=(0.0, 0.0, 0.0), up=(0.0, 1.0, 0.0)) -> np.ndarray:
    """3x4 row-major camera-to-world, OpenCV frame (x right, y down, z forward)."""
    eye = np.asarray(eye, dtype=np.float64)
    f = np.asarray(target, dtype=np.float64) - eye
    f /= np.linalg.norm(f)
    r = np.cross(f, np.asarray(up, dtype=np.float64))
    r /= np.linalg.norm(r)
    d = np.cross(f, r)
    m = np.stack([r, d, f, eye], axis=1)          # columns: right, down, forward, position
    return np.ascontiguousarray(m.reshape(-1), dtype=np.float32)


def eye_from_angles(radius: float, az_deg: float, el_deg: float) -> np.ndarray:
    az, el = math.radians(az_deg), math.radians(el_deg)
    return np.array([radius * math.cos(el) * math.sin(az),
                     radius * math.sin(el),
                     radius * math.cos(el) * math.cos(az)])


def pinhole(width: int, height: int, fov_deg: float, c2w: np.ndarray, t_near: float = 0.0) -> Camera:
    f = 0.5 * width / math.tan(0.5 * math.radians(fov_deg))   # horizontal FOV, fx = fy (Q14)
    f32 = float(np.float32(f))
    return Camera(f32, f32, float(np.float32(width / 2)), float(np.float32(height / 2)),
                  np.ascontiguousarray(c2w, dtype=np.float32), t_near, width, height)


def make_cameras(cfg: SceneConfig) -> list[Camera]:
    """One camera for cfg1-4 (azimuth 35, elevation 20); cfg5: 8 seeded orbit poses."""
    if cfg.n_views == 1:
        eye = eye_from_angles(cfg.radius, 35.0, 20.0)
        return [pinhole(cfg.width, cfg.height, cfg.fov_deg, look_at(eye))]
    rng = np.random.default_rng(cfg.pose_seed)
    cams = []
    for j in range(cfg.n_views):
        az = 45.0 * (j + rng.uniform())
        el = rng.uniform(-10.0, 30.0)
        cams.append(pinhole(cfg.width, cfg.height, cfg.fov_deg,
                            look_at(eye_from_angles(cfg.radius, az, el))))
    return cams


# ---------------------------------------------------------------------------
# Hand-built scenes used by pins and edge-case tests (inputs only).
# ---------------------------------------------------------------------------

def constant_mlp_weights(mlp: MLPSpec, raw_out: np.ndarray) -> np.ndarray:
    """Weights whose last layer has W = 0 and bias = raw_out: the MLP output is constant."""
    blob = []
    layers = mlp.layer_dims
    rng = np.random.default_rng(12345)
    for li, (i, o) in enumerate(layers):
        if li == len(layers) - 1:
            blob.append(np.zeros(i * o))
            blob.append(np.asarray(raw_out, dtype=np.float64).reshape(o))
        else:
            bound = math.sqrt(6.0 / i)
            blob.append(rng.uniform(-bound, bound, size=i * o))
            blob.append(np.zeros(o))
    return np.concatenate(blob).astype(np.float32)


def custom_scene(center, quat, scale, weights, mlp: MLPSpec, slots=None) -> Scene:
    return Scene(np.ascontiguousarray(center, dtype=np.float32).reshape(-1, 3),
                 np.ascontiguousarray(quat, dtype=np.float32).reshape(-1, 4),
                 np.ascontiguousarray(scale, dtype=np.float32).reshape(-1, 3),
                 np.ascontiguousarray(weights, dtype=np.float32).reshape(
                     -1, mlp.params_per_prim), mlp,
                 None if slots is None else np.ascontiguousarray(slots, dtype=np.float32))


def dense_scene(seed: int = 7, n: int = 48, sigma_bias: float = 8.0) -> tuple[Scene, SceneConfig]:
    """Opaque scene that triggers early termination (SURVEY.md pin P9): none of
    cfg1-5 ever reaches T < 1e-4, so this scene covers that branch."""
    cfg = SceneConfig("dense", seed, n, 1.0, 0.3, 0.8, MLPSpec(4, 0, 2, 32, 0, False),
                      96, 80, 50.0, 3.0, 8, sigma_bias=sigma_bias)
    return make_scene(cfg), cfg


def random_tiny_scene(seed: int, n: int = 12, *, straddle: bool = True,
                      mlp: MLPSpec | None = None) -> tuple[Scene, Camera, SceneConfig]:
    """Random small scene with a camera INSIDE the primitive cloud: exercises
    supports behind / around / straddling the camera plane and the image border."""
    mlp = mlp or MLPSpec(2, 0, 1, 8, 0, False)
    cfg = SceneConfig(f"tiny{seed}", seed, n, 1.5, 0.1, 0.9, mlp, 40, 24, 70.0, 1.0, 4)
    sc = make_scene(cfg)
    rng = np.random.default_rng(seed + 1000)
    eye = rng.uniform(-0.8, 0.8, size=3) if straddle else eye_from_angles(4.0, 20.0, 10.0)
    tgt = rng.uniform(-0.5, 0.5, size=3)
    cam = pinhole(cfg.width, cfg.height, cfg.fov_deg, look_at(eye, tgt))
    return sc, cam, cfg
