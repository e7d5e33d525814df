"""Seeded synthetic inputs for the neural-intersection-query hot path.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA path
(`paper_2604_24666_b200/`).  It holds none of the method's arithmetic: no deformation,
no intersection, no encoding, no network evaluation.  It only draws seeded random
numbers and lays them out as the arrays both sides consume ("Input recipe").

Anything that depends on the *deformed* object (camera placement, ray targets) takes the
deformed bounding box as an argument; the caller obtains it from whichever side it is
exercising.

The five configurations follow BASELINE.json `configs[0..4]` (B:7-11) with the details
SURVEY.md section 8(d).1 fixes.  The paper's own objects (cat, dragon)
are not available; these shapes stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np

N_HEAD_OUT = 12  # occlusion 1, distance 1, normal 3, albedo 3, material 4 (B:7)


@dataclass(frozen=True)
class NetShape:
    """Encoding + MLP shape.  Symbols as in SURVEY.md section 0."""
    pe_bands: int      # B: positional-encoding bands (paper's "F")
    levels: int        # L
    log2_T: int        # table entries per level = 2**log2_T
    feat: int          # F: features per table entry
    base_res: int
    growth: float
    hidden_layers: int  # H
    width: int          # W
    dtype: str          # "f32" | "f16"  (parameter storage / MMA operand type)
    enc_mode: str = "compose"   # "compose": psi = phi(gamma(x)) (Eq. 1, R1); "concat": psi = [gamma(x), phi(x)]

    @property
    def samples(self) -> int:          # S = 1 + 2B three-vectors per endpoint
        return 1 + 2 * self.pe_bands

    @property
    def d_in(self) -> int:             # 2 endpoints * S * L * F  (concat: 2 * (3 + 6B + L * F))
        if self.enc_mode == "concat":
            return 2 * (3 + 6 * self.pe_bands + self.levels * self.feat)
        return 2 * self.samples * self.levels * self.feat

    @property
    def table_entries(self) -> int:
        return 1 << self.log2_T

    def level_res(self) -> np.ndarray:
        """N_l = floor(base * growth**l), evaluated once in fp64 and handed to both sides
        as an integer table."""
        return np.array([int(math.floor(self.base_res * (self.growth ** l)))
                         for l in range(self.levels)], dtype=np.int32)

    def layer_dims(self):
        """[(fan_out, fan_in)] for the H hidden layers and the output layer."""
        dims = [(self.width, self.d_in)]
        dims += [(self.width, self.width)] * (self.hidden_layers - 1)
        dims += [(N_HEAD_OUT, self.width)]
        return dims


@dataclass(frozen=True)
class Config:
    cfg_id: int
    name: str
    nv: int
    net: NetShape
    n_poses: int
    rays_per_pose: int
    ray_kind: str            # "sphere_to_cube" | "camera" | "sphere_to_aabb" | "inside_random"
    occlusion_only: bool = False
    image_wh: tuple = (0, 0)
    geom_seed: int = 0
    pose_seed: int = 0
    net_seed: int = 0
    ray_seed: int = 0
    extra: dict = field(default_factory=dict)


_NET0 = NetShape(pe_bands=4, levels=4, log2_T=12, feat=2, base_res=4, growth=2.0,
                 hidden_layers=2, width=32, dtype="f32")
_NET1 = NetShape(pe_bands=6, levels=16, log2_T=19, feat=2, base_res=16, growth=1.38,
                 hidden_layers=3, width=64, dtype="f16")
_NET4 = NetShape(pe_bands=6, levels=16, log2_T=22, feat=4, base_res=16, growth=1.38,
                 hidden_layers=4, width=128, dtype="f16")

# The paper's own experimental shape: "voxel resolution 32^3, a two-level hash grid (base 64,
# feature dim 3), and F=3 positional encoding bands".  Table size, growth and the MLP are not stated:
# T = 2^19, growth 2 (levels 64 dense, 128 hashed) and config 1's 3x64 fp16 MLP are assumed (R26).
_NET5 = NetShape(pe_bands=3, levels=2, log2_T=19, feat=3, base_res=64, growth=2.0,
                 hidden_layers=3, width=64, dtype="f16")

CONFIGS = {
    0: Config(0, "tiny", 16, _NET0, 1, 4096, "sphere_to_cube",
              geom_seed=0, net_seed=0, ray_seed=0),
    1: Config(1, "primary_1080p", 64, _NET1, 1, 1920 * 1080, "camera",
              image_wh=(1920, 1080), geom_seed=1, net_seed=11, ray_seed=1),
    2: Config(2, "multi_pose", 128, _NET1, 8, 1 << 20, "sphere_to_aabb",
              geom_seed=2, pose_seed=1, net_seed=11, ray_seed=2),
    3: Config(3, "incoherent_occlusion", 128, _NET1, 8, 1 << 21, "inside_random",
              occlusion_only=True, geom_seed=2, pose_seed=1, net_seed=11, ray_seed=3),
    4: Config(4, "large_4k", 256, _NET4, 1, 3840 * 2160, "camera",
              image_wh=(3840, 2160), geom_seed=4, net_seed=14, ray_seed=4),
    # not a BASELINE.json config: the paper's shape on config 1's kind of object and camera
    5: Config(5, "paper_shape_32", 32, _NET5, 1, 1920 * 1080, "camera",
              image_wh=(1920, 1080), geom_seed=1, net_seed=15, ray_seed=5),
}


def get_config(cfg_id: int) -> Config:
    return CONFIGS[cfg_id]


def scaled(cfg: Config, **kw) -> Config:
    """A copy with some fields replaced (tests use reduced ray counts / image sizes)."""
    return replace(cfg, **kw)


# --------------------------------------------------------------------------------------
# geometry: occupancy on the Nv^3 rest lattice, x fastest.  Voxel centre of index i is
# (i + 0.5) * 2 / Nv - 1.
# --------------------------------------------------------------------------------------
def _centres(nv: int) -> np.ndarray:
    return (np.arange(nv, dtype=np.float64) + 0.5) * (2.0 / nv) - 1.0


def occupancy(cfg: Config) -> np.ndarray:
    """uint8 array of nv^3 entries, index ix + nv*(iy + nv*iz)."""
    nv = cfg.nv
    c = _centres(nv)
    if cfg.cfg_id == 0:                                   # ball of radius 0.8 (B:7)
        z, y, x = np.meshgrid(c, c, c, indexing="ij")
        occ = (x * x + y * y + z * z) <= 0.8 * 0.8
    elif cfg.cfg_id in (1, 5):                            # 8 Gaussian blobs, threshold 0.5 (B:8)
        rng = np.random.default_rng(cfg.geom_seed)
        ctr = rng.uniform(-0.5, 0.5, size=(8, 3))
        sig = rng.uniform(0.12, 0.25, size=8)
        z, y, x = np.meshgrid(c, c, c, indexing="ij")
        s = np.zeros_like(x)
        for b in range(8):
            r2 = (x - ctr[b, 0]) ** 2 + (y - ctr[b, 1]) ** 2 + (z - ctr[b, 2]) ** 2
            s += np.exp(-r2 / (2.0 * sig[b] ** 2))
        occ = s >= 0.5
    elif cfg.cfg_id in (2, 3):                            # torus, axis z, R=0.6 r=0.25 (B:9)
        z, y, x = np.meshgrid(c, c, c, indexing="ij")
        q = np.sqrt(x * x + y * y) - 0.6
        occ = (q * q + z * z) <= 0.25 * 0.25
    elif cfg.cfg_id == 4:                                 # 64 axis-aligned ellipsoids (B:11)
        rng = np.random.default_rng(cfg.geom_seed)
        ctr = rng.uniform(-0.6, 0.6, size=(64, 3))
        axes = rng.uniform(0.05, 0.18, size=(64, 3))
        occ = np.zeros((nv, nv, nv), dtype=bool)          # [z, y, x]
        for e in range(64):
            lo = np.searchsorted(c, ctr[e] - axes[e], side="left")
            hi = np.searchsorted(c, ctr[e] + axes[e], side="right")
            xs, ys, zs = (c[lo[a]:hi[a]] for a in range(3))
            zz, yy, xx = np.meshgrid(zs, ys, xs, indexing="ij")
            inside = (((xx - ctr[e, 0]) / axes[e, 0]) ** 2 +
                      ((yy - ctr[e, 1]) / axes[e, 1]) ** 2 +
                      ((zz - ctr[e, 2]) / axes[e, 2]) ** 2) <= 1.0
            occ[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] |= inside
    else:
        raise ValueError(cfg.cfg_id)
    return np.ascontiguousarray(occ.reshape(-1).astype(np.uint8))


def random_occupancy(nv: int, fill: float, seed: int) -> np.ndarray:
    """Random sparse grid for brute-force-vs-BVH tests."""
    rng = np.random.default_rng(seed)
    return (rng.random(nv ** 3) < fill).astype(np.uint8)


# --------------------------------------------------------------------------------------
# poses: (twist theta_max, bend k).  Composite = bend(twist(p)) (B:9, B:11).
# --------------------------------------------------------------------------------------
def poses(cfg: Config) -> np.ndarray:
    """float32 array [n_poses, 2] of (theta_max, k)."""
    if cfg.cfg_id == 0:
        p = [[1.0, 0.0]]                                  # theta(y) = 0.5 (y+1)  (B:7)
    elif cfg.cfg_id == 1:
        p = [[0.0, 0.8]]                                  # bend k = 0.8 (B:8)
    elif cfg.cfg_id in (2, 3):
        rng = np.random.default_rng(cfg.pose_seed)
        p = [[rng.uniform(0.0, math.pi / 2), rng.uniform(0.0, 1.0)]
             for _ in range(cfg.n_poses)]
    elif cfg.cfg_id == 4:
        p = [[math.pi, 1.2]]                              # B:11
    elif cfg.cfg_id == 5:
        p = [[0.6, 0.5]]                                  # a twist followed by a bend (paper shape, not in BASELINE)
    else:
        raise ValueError(cfg.cfg_id)
    return np.asarray(p, dtype=np.float32)


# --------------------------------------------------------------------------------------
# network parameters.  Draw order: table, then W1..W_{H+1}.  fp16 configs are rounded to
# fp16 ONCE here; both sides consume the rounded values.
# --------------------------------------------------------------------------------------
@dataclass
class NetParams:
    shape: NetShape
    level_res: np.ndarray          # int32 [L]
    table: np.ndarray              # float32 [L, T, F]   (fp16-representable if dtype f16)
    weights: list                  # float32 [(fan_out, fan_in)] row-major
    variant: str

    def table_storage(self) -> np.ndarray:
        return self.table.astype(np.float16) if self.shape.dtype == "f16" else self.table

    def weights_storage(self) -> list:
        if self.shape.dtype == "f16":
            return [w.astype(np.float16) for w in self.weights]
        return self.weights


def net_params(cfg_or_shape, variant: str = "uniform0.1", seed: int | None = None) -> NetParams:
    """variant "uniform0.1": everything U(-0.1, 0.1) (B:7).
    variant "varpres": weights U(+-sqrt(6/fan_in)), table U(+-1), so head outputs are O(1)
    (SURVEY 8(c).2 row 19)."""
    if isinstance(cfg_or_shape, Config):
        shape = cfg_or_shape.net
        seed = cfg_or_shape.net_seed if seed is None else seed
    else:
        shape = cfg_or_shape
        seed = 0 if seed is None else seed
    rng = np.random.default_rng(seed + (1000 if variant == "varpres" else 0))
    L, T, F = shape.levels, shape.table_entries, shape.feat
    if variant == "uniform0.1":
        table = rng.uniform(-0.1, 0.1, size=(L, T, F))
        ws = [rng.uniform(-0.1, 0.1, size=d) for d in shape.layer_dims()]
    elif variant == "varpres":
        table = rng.uniform(-1.0, 1.0, size=(L, T, F))
        ws = [rng.uniform(-1.0, 1.0, size=d) * math.sqrt(6.0 / d[1]) for d in shape.layer_dims()]
    else:
        raise ValueError(variant)
    table = table.astype(np.float32)
    ws = [np.ascontiguousarray(w.astype(np.float32)) for w in ws]
    if shape.dtype == "f16":
        table = table.astype(np.float16).astype(np.float32)
        ws = [w.astype(np.float16).astype(np.float32) for w in ws]
    return NetParams(shape, shape.level_res(), np.ascontiguousarray(table), ws, variant)


# --------------------------------------------------------------------------------------
# rays: float32 origin [n,3] and unit direction [n,3].
# --------------------------------------------------------------------------------------
def _normalize(v: np.ndarray) -> np.ndarray:
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def _finish(o: np.ndarray, d: np.ndarray):
    d = _normalize(d.astype(np.float64))
    return (np.ascontiguousarray(o.astype(np.float32)),
            np.ascontiguousarray(d.astype(np.float32)))


def camera_rays(width: int, height: int, centre, distance: float = 3.0,
                vfov_deg: float = 45.0):
    """Pinhole camera at centre + (0,0,distance) looking down -z, up +y, one ray per pixel
    centre, row-major (y down the image) (B:8)."""
    t = math.tan(math.radians(vfov_deg) / 2.0)
    px = ((np.arange(width, dtype=np.float64) + 0.5) / width * 2.0 - 1.0) * t * (width / height)
    py = (1.0 - (np.arange(height, dtype=np.float64) + 0.5) / height * 2.0) * t
    dx, dy = np.meshgrid(px, py, indexing="xy")
    d = np.stack([dx, dy, -np.ones_like(dx)], axis=-1).reshape(-1, 3)
    eye = np.asarray(centre, dtype=np.float64) + np.array([0.0, 0.0, distance])
    o = np.broadcast_to(eye, d.shape)
    return _finish(o, d)


def rays(cfg: Config, pose_index: int = 0, aabb_lo=None, aabb_hi=None, n: int | None = None):
    """Ray batch for one pose.  `aabb_lo/hi`: deformed bounding box of the posed object
    (needed by every kind except "sphere_to_cube")."""
    n = cfg.rays_per_pose if n is None else n
    rng = np.random.default_rng([cfg.ray_seed, pose_index])
    if cfg.ray_kind == "sphere_to_cube":                  # B:7
        o = 3.0 * _normalize(rng.standard_normal((n, 3)))
        tgt = rng.uniform(-0.5, 0.5, size=(n, 3))
        return _finish(o, tgt - o)
    lo = np.asarray(aabb_lo, dtype=np.float64)
    hi = np.asarray(aabb_hi, dtype=np.float64)
    if cfg.ray_kind == "camera":                          # B:8, B:11
        w, h = cfg.image_wh
        if n != cfg.rays_per_pose:                        # reduced image, same aspect
            s = math.sqrt(n / (w * h))
            w, h = max(1, int(round(w * s))), max(1, int(round(h * s)))
        return camera_rays(w, h, 0.5 * (lo + hi))
    if cfg.ray_kind == "sphere_to_aabb":                  # B:9
        o = 3.0 * _normalize(rng.standard_normal((n, 3)))
        tgt = rng.uniform(lo, hi, size=(n, 3))
        return _finish(o, tgt - o)
    if cfg.ray_kind == "inside_random":                   # B:10
        o = rng.uniform(lo, hi, size=(n, 3))
        d = rng.standard_normal((n, 3))
        return _finish(o, d)
    raise ValueError(cfg.ray_kind)


def shard_range(n: int, rank: int, world: int):
    """Contiguous ray range [begin, end) of `rank` among `world` ranks (rays are independent:
    data-parallel sharding, no exchange step)."""
    base, rem = divmod(n, world)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def wavy_lattice(nv: int, seed: int, amplitude_voxels: float = 0.35) -> np.ndarray:
    """A "user-specified deformation" that has no closed-form inverse: the rest corner
    lattice [(nv+1)^3, 3] (point (i,j,k) at index i + (nv+1)(j + (nv+1)k), coordinates (2i - nv)/nv)
    displaced by a seeded sum of three smooth sine waves per axis, amplitude `amplitude_voxels` voxel
    sizes in total (small enough that no voxel folds over).  float32."""
    rng = np.random.default_rng(seed)
    g = (2.0 * np.arange(nv + 1, dtype=np.float64) - nv) / nv
    z, y, x = np.meshgrid(g, g, g, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    h = 2.0 / nv
    disp = np.zeros_like(p)
    for _ in range(3):
        k = rng.uniform(1.0, 3.0, size=(3, 3))            # wave vectors (rad per unit length), one per displaced axis
        ph = rng.uniform(0.0, 2.0 * math.pi, size=3)
        amp = rng.uniform(0.5, 1.0, size=3) * amplitude_voxels * h / 3.0
        disp += amp * np.sin(p @ k.T + ph)
    return np.ascontiguousarray((p + disp).astype(np.float32))
