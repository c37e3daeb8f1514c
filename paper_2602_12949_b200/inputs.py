"""Seeded synthetic inputs for the Neural Irradiance Volume (NIV) inference path.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_2602_12949_b200/csrc`).  It holds none of the method's arithmetic
(no hash, no interpolation, no SH, no MLP): it only produces arrays -- model
parameters (hash-grid table, MLP weights) and queries (positions, normals,
G-buffers) -- that are then handed, as the same bytes, to both sides.

Everything is drawn from one counter-based generator (splitmix64 of
(seed, stream, index)), so streams never depend on a library version.

Workload recipes follow BASELINE.json `configs` and SURVEY.md section 8(d); the
paper's own scenes (Sponza/Bistro/...) are not available, so
the procedural G-buffer below *stands in* for them.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Tuple

import numpy as np

# ----------------------------------------------------------------------------
# counter-based RNG
# ----------------------------------------------------------------------------
_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> _U64(30))) * _U64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U64(27))) * _U64(0x94D049BB133111EB)
        z = z ^ (z >> _U64(31))
    return z


def random_u64(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """n 64-bit words; word i depends only on (seed, stream, offset + i)."""
    with np.errstate(over="ignore"):
        key = _mix64(np.array([(seed * 0x100000001B3 + stream) & 0xFFFFFFFFFFFFFFFF], dtype=_U64) + _GOLDEN)
        ctr = np.arange(offset, offset + n, dtype=_U64)
        return _mix64(key + (ctr + _U64(1)) * _GOLDEN)


def uniform01(seed: int, stream: int, n: int, offset: int = 0) -> np.ndarray:
    """float64 uniforms in [0,1) on a 2^-24 lattice (exactly representable in fp32)."""
    return (random_u64(seed, stream, n, offset) >> _U64(40)).astype(np.float64) * (1.0 / 16777216.0)


def standard_normal(seed: int, stream: int, n: int) -> np.ndarray:
    """Box-Muller from two uniform streams; float64."""
    u1 = uniform01(seed, stream * 2 + 0x1000, n)
    u2 = uniform01(seed, stream * 2 + 0x1001, n)
    r = np.sqrt(-2.0 * np.log(1.0 - u1))          # 1-u1 in (0,1]
    return r * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------
# model description (hyper-parameters only; no derived method quantities)
# ----------------------------------------------------------------------------
OUT_LINEAR = 0
OUT_SIGMOID = 1


@dataclasses.dataclass(frozen=True)
class ModelSpec:
    """Hyper-parameters of one NIV model (BASELINE.json configs / PAPER.md:314-318)."""
    n_levels: int                 # L
    n_features: int               # F  (fp16 features per table entry)
    log2_table_size: int          # T = 2^k entries per level
    base_resolution: int          # N0
    per_level_scale: float        # b
    aabb_min: Tuple[float, float, float]
    aabb_max: Tuple[float, float, float]
    hidden_width: int
    n_hidden_layers: int
    out_activation: int = OUT_SIGMOID
    n_params: int = 0             # per-call scalar scene parameters
    n_frequencies: int = 8        # sin/cos bands per parameter
    sh_degree: int = 4            # 4 => 16 SH coefficients (BASELINE.json); 0 => the raw direction, 3 values (paper)
    resolutions: Optional[Tuple[int, ...]] = None   # explicit N_l override
    dir_frequencies: int = 0      # sh_degree 0 only: sin/cos bands per axis appended to the raw direction

    @property
    def table_size(self) -> int:
        return 1 << self.log2_table_size

    @property
    def dir_dim(self) -> int:
        return 3 + 6 * self.dir_frequencies if self.sh_degree == 0 else self.sh_degree ** 2

    @property
    def pos_dim(self) -> int:
        """Grid latents, or (n_levels == 0) the 8-band positional encoding of the position."""
        return self.n_levels * self.n_features if self.n_levels else 6 * self.n_frequencies

    @property
    def in_dim(self) -> int:
        return self.pos_dim + self.dir_dim + 2 * self.n_frequencies * self.n_params

    @property
    def layer_shapes(self) -> List[Tuple[int, int]]:
        """[(out, in), ...] for W1..Wk, Wk being the 3-row output layer."""
        dims = [self.in_dim] + [self.hidden_width] * self.n_hidden_layers + [3]
        return [(dims[i + 1], dims[i]) for i in range(len(dims) - 1)]


UNIT_AABB = ((0.0, 0.0, 0.0), (1.0, 1.0, 1.0))
ROOM_AABB = ((0.0, 0.0, 0.0), (10.0, 4.0, 10.0))


def spec_tiny() -> ModelSpec:
    """BASELINE.json configs[0]: 64x64, L=8, F=2, T=2^12, N0=4, b=1.5, MLP 32->32->3, sigmoid."""
    return ModelSpec(8, 2, 12, 4, 1.5, *UNIT_AABB, hidden_width=32, n_hidden_layers=1)


def spec_fullhd(log2_T: int = 17, width: int = 64, n_hidden: int = 2) -> ModelSpec:
    """BASELINE.json configs[1]/[2]/[4]: L=16, F=2, T=2^17, N0=16, b=1.5, MLP 48->64->64->3."""
    return ModelSpec(16, 2, log2_T, 16, 1.5, *ROOM_AABB, hidden_width=width, n_hidden_layers=n_hidden)


def spec_param() -> ModelSpec:
    """BASELINE.json configs[3]: T=2^18, one scalar t (8 sin/cos bands), MLP 64->64->64->3."""
    return ModelSpec(16, 2, 18, 16, 1.5, *ROOM_AABB, hidden_width=64, n_hidden_layers=2, n_params=1)


PAPER_RESOLUTIONS = (16, 22, 32, 45, 64, 90, 128, 181)     # floor(16 * sqrt(2)^l), l = 0..7 (exact: 16 * 2^(l/2))


def spec_paper(n_levels: int = 8, width: int = 64) -> ModelSpec:
    """The paper's own model family (Table 1 382-389): T = 2^17, latent dimension 4, scale
    sqrt(2) between levels, coarsest side 16, 2..8 levels; "four-layer" ReLU MLP = 4 weight matrices (3 hidden
    layers); position + direction in, no basis functions on the direction, no activation on the final layer.
    Resolutions are passed explicitly so that no pow() rounding decides an integer."""
    return ModelSpec(n_levels, 4, 17, 16, 2.0 ** 0.5, *ROOM_AABB, hidden_width=width, n_hidden_layers=3,
                     out_activation=OUT_LINEAR, sh_degree=0, resolutions=PAPER_RESOLUTIONS[:n_levels])


def spec_paper_dirfreq(n_levels: int = 8, width: int = 64, bands: int = 4) -> ModelSpec:
    """The paper's family with the direction frequency-encoded on top of the raw vector ("raw 3-vector (plus
    optional frequency)"): 3 + 6 * bands direction inputs."""
    return ModelSpec(n_levels, 4, 17, 16, 2.0 ** 0.5, *ROOM_AABB, hidden_width=width, n_hidden_layers=3,
                     out_activation=OUT_LINEAR, sh_degree=0, resolutions=PAPER_RESOLUTIONS[:n_levels],
                     dir_frequencies=bands)


def spec_paper_pe(width: int = 64) -> ModelSpec:
    """The paper's grid-less models (Table 1 rows "-": widths 16 / 32 / 64): eight-band positional encoding of the
    position (48 values) + the direction (3), four weight matrices, linear output; no table."""
    return ModelSpec(0, 4, 17, 16, 2.0 ** 0.5, *ROOM_AABB, hidden_width=width, n_hidden_layers=3,
                     out_activation=OUT_LINEAR, sh_degree=0)


# ----------------------------------------------------------------------------
# parameters
# ----------------------------------------------------------------------------
def make_table(spec: ModelSpec, seed: int, lo: float = -1e-2, hi: float = 1e-2) -> np.ndarray:
    """Hash-grid table [L][T][F] fp16, uniform[lo,hi] then round-to-nearest-even to fp16.

    The fp16 bits ARE the model."""
    n = spec.n_levels * spec.table_size * spec.n_features
    u = uniform01(seed, 11, n)
    return (lo + (hi - lo) * u).astype(np.float16).reshape(spec.n_levels, spec.table_size, spec.n_features)


def make_mlp(spec: ModelSpec, seed: int, bias_scale: float = 0.0):
    """He-normal weights W ~ N(0, 2/fan_in) rounded to fp16, layer k stored [out][in] row-major;
    fp32 biases uniform[-bias_scale, bias_scale] (zero by default)."""
    weights, biases = [], []
    for k, (n_out, n_in) in enumerate(spec.layer_shapes):
        w = standard_normal(seed, 100 + k, n_out * n_in) * math.sqrt(2.0 / n_in)
        weights.append(w.astype(np.float16).reshape(n_out, n_in))
        b = (2.0 * uniform01(seed, 200 + k, n_out) - 1.0) * bias_scale
        biases.append(b.astype(np.float32))
    return weights, biases


def pack_weights(weights: List[np.ndarray]) -> np.ndarray:
    """W1|W2|... as one flat fp16 blob (layer-major, row-major)."""
    return np.concatenate([w.reshape(-1) for w in weights]).astype(np.float16)


def pack_biases(biases: List[np.ndarray]) -> np.ndarray:
    return np.concatenate([b.reshape(-1) for b in biases]).astype(np.float32)


# ----------------------------------------------------------------------------
# queries
# ----------------------------------------------------------------------------
def positions_uniform(n: int, aabb, seed: int) -> np.ndarray:
    """[n][3] fp32, i.i.d. uniform in the AABB (configs[0] and configs[2])."""
    lo = np.asarray(aabb[0], dtype=np.float64)
    hi = np.asarray(aabb[1], dtype=np.float64)
    u = uniform01(seed, 21, 3 * n).reshape(n, 3)
    return (lo + (hi - lo) * u).astype(np.float32)


def normals_uniform(n: int, seed: int) -> np.ndarray:
    """[n][3] fp32, uniform on the unit sphere (normalised 3-Gaussian)."""
    g = np.stack([standard_normal(seed, 31 + d, n) for d in range(3)], axis=1)
    g /= np.maximum(np.linalg.norm(g, axis=1, keepdims=True), 1e-30)
    return g.astype(np.float32)


# ----------------------------------------------------------------------------
# procedural G-buffer (stands in for the paper's rasterised scenes)
# ----------------------------------------------------------------------------
@dataclasses.dataclass
class Scene:
    sph_c: np.ndarray   # [16][3]
    sph_r: np.ndarray   # [16]
    box_c: np.ndarray   # [16][3]
    box_h: np.ndarray   # [16][3]
    window: Tuple[float, float, float, float]   # on wall x = room max: (y0, y1, z0, z1)


def make_scene(seed: int) -> Scene:
    """Box room 10x4x10 m with 16 spheres (r~U[0.2,0.8]) and 16 axis-aligned boxes
    (half extents ~U[0.2,0.8]^3), centres uniform in the room shrunk by 1 m."""
    lo = np.asarray(ROOM_AABB[0]) + 1.0
    hi = np.asarray(ROOM_AABB[1]) - 1.0
    sph_c = lo + (hi - lo) * uniform01(seed, 41, 48).reshape(16, 3)
    sph_r = 0.2 + 0.6 * uniform01(seed, 42, 16)
    box_c = lo + (hi - lo) * uniform01(seed, 43, 48).reshape(16, 3)
    box_h = 0.2 + 0.6 * uniform01(seed, 44, 48).reshape(16, 3)
    return Scene(sph_c, sph_r, box_c, box_h, window=(0.75, 3.5, 1.0, 9.0))


def _camera(scene: Scene, seed: int, sub_seed: int):
    """Camera uniform in the room shrunk by 1.5 m, outside all objects; look-at uniform in the room."""
    lo = np.asarray(ROOM_AABB[0]) + 1.5
    hi = np.asarray(ROOM_AABB[1]) - 1.5
    k = 0
    while True:
        u = uniform01(seed, 51, 6, offset=6 * (sub_seed * 64 + k))
        eye = lo + (hi - lo) * u[:3]
        in_s = np.any(np.linalg.norm(scene.sph_c - eye, axis=1) < scene.sph_r + 0.05)
        in_b = np.any(np.all(np.abs(scene.box_c - eye) < scene.box_h + 0.05, axis=1))
        if not (in_s or in_b) or k >= 63:
            break
        k += 1
    rl, rh = np.asarray(ROOM_AABB[0]), np.asarray(ROOM_AABB[1])
    target = rl + (rh - rl) * u[3:]
    return eye, target


def _raycast(scene: Scene, eye, target, width: int, height: int):
    """Primary rays (pinhole, vertical FOV 60 deg, pixel centres) -> pos, nrm (float64) and background mask."""
    fwd = target - eye
    fwd /= np.linalg.norm(fwd)
    up0 = np.array([0.0, 1.0, 0.0])
    if abs(fwd[1]) > 0.99:
        up0 = np.array([1.0, 0.0, 0.0])
    right = np.cross(fwd, up0)
    right /= np.linalg.norm(right)
    up = np.cross(right, fwd)
    tan_half = math.tan(math.radians(30.0))
    px = ((np.arange(width) + 0.5) / width * 2.0 - 1.0) * tan_half * (width / height)
    py = (1.0 - (np.arange(height) + 0.5) / height * 2.0) * tan_half
    d = (fwd[None, None, :] + px[None, :, None] * right[None, None, :] + py[:, None, None] * up[None, None, :])
    d = d.reshape(-1, 3)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    n_px = d.shape[0]

    # room: the ray leaves the box through the nearest exit face
    rl, rh = np.asarray(ROOM_AABB[0]), np.asarray(ROOM_AABB[1])
    with np.errstate(divide="ignore", invalid="ignore"):
        t_exit_ax = np.where(d > 0, (rh - eye) / d, np.where(d < 0, (rl - eye) / d, np.inf))
    ax = np.argmin(t_exit_ax, axis=1)
    t_best = t_exit_ax[np.arange(n_px), ax]
    nrm = np.zeros((n_px, 3))
    nrm[np.arange(n_px), ax] = -np.sign(d[np.arange(n_px), ax])
    wall_hit = eye + t_best[:, None] * d
    y0, y1, z0, z1 = scene.window
    background = (ax == 0) & (d[:, 0] > 0) & (wall_hit[:, 1] > y0) & (wall_hit[:, 1] < y1) \
        & (wall_hit[:, 2] > z0) & (wall_hit[:, 2] < z1)

    # spheres
    for c, r in zip(scene.sph_c, scene.sph_r):
        oc = eye - c
        b = d @ oc
        disc = b * b - (oc @ oc - r * r)
        ok = disc > 0
        t = -b - np.sqrt(np.where(ok, disc, 0.0))
        hit = ok & (t > 1e-4) & (t < t_best)
        if np.any(hit):
            t_best = np.where(hit, t, t_best)
            p = eye + t[hit, None] * d[hit]
            nrm[hit] = (p - c) / r
            background &= ~hit
    # boxes (slab test; the entry axis gives the normal)
    for c, h in zip(scene.box_c, scene.box_h):
        with np.errstate(divide="ignore", invalid="ignore"):
            inv = 1.0 / d
            t0 = (c - h - eye) * inv
            t1 = (c + h - eye) * inv
        tn = np.minimum(t0, t1)
        tf = np.maximum(t0, t1)
        t_in_ax = np.argmax(tn, axis=1)
        t_in = tn[np.arange(n_px), t_in_ax]
        t_out = np.min(tf, axis=1)
        hit = (t_in < t_out) & (t_in > 1e-4) & (t_in < t_best)
        if np.any(hit):
            t_best = np.where(hit, t_in, t_best)
            nb = np.zeros((int(hit.sum()), 3))
            nb[np.arange(nb.shape[0]), t_in_ax[hit]] = -np.sign(d[hit, t_in_ax[hit]])
            nrm[hit] = nb
            background &= ~hit
    pos = eye + t_best[:, None] * d
    # normals face the camera (outward geometric normal flipped toward the eye)
    flip = np.sum(nrm * d, axis=1) > 0
    nrm[flip] = -nrm[flip]
    pos[background] = 0.0
    nrm[background] = 0.0
    return pos, nrm, background


def make_gbuffer(width: int, height: int, seed: int, frame: int = 0) -> Dict[str, object]:
    """Seeded G-buffer: pos [n][3] fp32 world-space hit points, nrm [n][3] fp32 unit normals facing the
    camera; background texels (window) have pos = nrm = 0.  A deterministic sub-seed is advanced until
    the background fraction lies in [12 %, 18 %] (BASELINE.json configs[1]: "~15% background")."""
    scene = make_scene(seed)
    sub = frame * 1000
    lw, lh = max(width // 8, 32), max(height // 8, 18)
    for _ in range(1000):
        eye, target = _camera(scene, seed, sub)
        _, _, bg = _raycast(scene, eye, target, lw, lh)
        if 0.125 <= bg.mean() <= 0.175:
            pos, nrm, bg = _raycast(scene, eye, target, width, height)
            if 0.12 <= bg.mean() <= 0.18:
                return {"pos": np.ascontiguousarray(pos, dtype=np.float32),
                        "nrm": np.ascontiguousarray(nrm, dtype=np.float32),
                        "masked_fraction": float(bg.mean()), "sub_seed": sub,
                        "eye": eye, "target": target, "width": width, "height": height}
        sub += 1
    raise RuntimeError("no camera with 12-18 % background found")


# ----------------------------------------------------------------------------
# a synthetic probe grid (stands in for a baked DDGI-like grid)
# ----------------------------------------------------------------------------
PROBE_STREAM = 0x7000


def make_probe_grid(dims: Tuple[int, int, int], seed: int, scale: float = 1.0) -> np.ndarray:
    """-> coefficients [nz][ny][nx][9][3] fp16: 27 values per probe, x fastest.  A baked grid is not
    available (no scenes, no path tracer), so the values are seeded noise with the magnitudes of an irradiance field:
    a positive band-0 term of order one, bands 1 and 2 a half and a quarter of it, both signs."""
    nx, ny, nz = (int(v) for v in dims)
    n = nx * ny * nz
    r = uniform01(seed, PROBE_STREAM, n * 27).reshape(nz, ny, nx, 9, 3)
    band = np.array([1.0] + [0.5] * 3 + [0.25] * 5)[None, None, None, :, None]
    c = (2.0 * r - 1.0) * band
    c[..., 0, :] = 1.0 + 2.0 * r[..., 0, :]                      # band 0 in [1, 3)
    return (scale * c).astype(np.float16)


def probe_grid_dims_for_spacing(aabb_min, aabb_max, spacing: float) -> Tuple[int, int, int]:
    """Probes on a regular lattice over the box, faces included, about `spacing` apart."""
    return tuple(int(max(2, round((float(hi) - float(lo)) / spacing) + 1)) for lo, hi in zip(aabb_min, aabb_max))


# ----------------------------------------------------------------------------
# Compact G-buffer layouts (include/niv.h NIV_GBUF_*).  This is the PRODUCER side -- what a renderer would
# write -- so it lives with the input generators; the decode (the method's side) exists twice, in oracle/ and in csrc/.
GBUF_F32X3, GBUF_F32X4, GBUF_P32_OCT16, GBUF_P16_OCT8 = 0, 1, 2, 3
OUTFMT_F32X3, OUTFMT_F16X4, OUTFMT_RGB9E5 = 0, 1, 2


def _oct_encode(nrm: np.ndarray) -> np.ndarray:
    """unit vectors [n][3] -> octahedral coordinates [n][2] in [-1, 1] (float64)"""
    n = nrm.astype(np.float64)
    s = np.abs(n).sum(axis=1, keepdims=True)
    s[s == 0] = 1.0
    n = n / s
    x, y, z = n[:, 0], n[:, 1], n[:, 2]
    neg = z < 0
    fx = np.where(neg, (1.0 - np.abs(y)) * np.where(x >= 0, 1.0, -1.0), x)
    fy = np.where(neg, (1.0 - np.abs(x)) * np.where(y >= 0, 1.0, -1.0), y)
    return np.stack([fx, fy], axis=1)


def pack_gbuffer(fmt: int, pos: np.ndarray, nrm: np.ndarray, aabb=None):
    """-> (a, b): the arrays the *_packed entry points take (b is None for the single-array formats).  Background texels
    (nrm == 0) get the reserved normal code; positions of format 3 are quantised to unorm16 of `aabb` (clipped)."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    nrm = np.ascontiguousarray(nrm, dtype=np.float32)
    n = pos.shape[0]
    if fmt == GBUF_F32X3:
        return pos, nrm
    if fmt == GBUF_F32X4:
        a = np.zeros((n, 4), dtype=np.float32)
        b = np.zeros((n, 4), dtype=np.float32)
        a[:, :3], b[:, :3] = pos, nrm
        a[:, 3], b[:, 3] = 1.0, 0.0
        return a, b
    bg = np.all(nrm == 0, axis=1)
    o = _oct_encode(nrm)
    if fmt == GBUF_P32_OCT16:
        q = np.clip(np.rint(o * 32767.0), -32767, 32767).astype(np.int16)
        q[bg] = -32768
        rec = np.zeros((n, 4), dtype=np.uint32)
        rec[:, :3] = pos.view(np.uint32)
        rec[:, 3] = q[:, 0].view(np.uint16).astype(np.uint32) | (q[:, 1].view(np.uint16).astype(np.uint32) << 16)
        return rec, None
    if fmt == GBUF_P16_OCT8:
        lo, hi = np.asarray(aabb[0], dtype=np.float64), np.asarray(aabb[1], dtype=np.float64)
        u = np.clip((pos.astype(np.float64) - lo) / (hi - lo), 0.0, 1.0)
        qp = np.rint(u * 65535.0).astype(np.uint16)
        q = np.clip(np.rint(o * 127.0), -127, 127).astype(np.int8)
        q[bg] = -128
        rec = np.zeros((n, 8), dtype=np.uint8)
        rec[:, :6] = qp.view(np.uint8).reshape(n, 6)
        rec[:, 6:] = q.view(np.uint8)
        return rec, None
    raise ValueError("unknown G-buffer format")
