"""ctypes wrapper around oracle/niv_oracle.c (TEST INFRASTRUCTURE -- see the C header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It neither imports nor is imported by the CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "niv_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "niv_oracle_ext.c")]
_LIB = os.path.join(_HERE, "libniv_oracle.so")


class OracleConfig(C.Structure):
    _fields_ = [
        ("n_levels", C.c_uint32), ("n_features", C.c_uint32), ("log2_table_size", C.c_uint32),
        ("base_resolution", C.c_uint32), ("per_level_scale", C.c_double),
        ("resolutions", C.c_uint32 * 16),
        ("aabb_min", C.c_float * 3), ("aabb_max", C.c_float * 3),
        ("sh_degree", C.c_uint32), ("n_params", C.c_uint32), ("n_frequencies", C.c_uint32),
        ("n_hidden_layers", C.c_uint32), ("hidden_width", C.c_uint32), ("out_activation", C.c_uint32),
        ("dir_frequencies", C.c_uint32),
    ]


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp (no -ffast-math): the fp32 index path must not be contracted."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", _LIB] + _SRCS + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.niv_oracle_half_to_double.restype = C.c_double
        _lib.niv_oracle_half_to_double.argtypes = [C.c_uint16]
        _lib.niv_oracle_hash.restype = C.c_uint32
        _lib.niv_oracle_hash.argtypes = [C.c_uint32] * 4
        _lib.niv_oracle_in_dim.restype = C.c_uint32
        _lib.niv_oracle_max_threads.restype = C.c_int
    return _lib


def make_config(spec) -> OracleConfig:
    """spec: any object with the ModelSpec attribute names (paper_2602_12949_b200.inputs.ModelSpec)."""
    cfg = OracleConfig()
    cfg.n_levels = spec.n_levels
    cfg.n_features = spec.n_features
    cfg.log2_table_size = spec.log2_table_size
    cfg.base_resolution = spec.base_resolution
    cfg.per_level_scale = spec.per_level_scale
    res = getattr(spec, "resolutions", None)
    if res:
        for i, r in enumerate(res):
            cfg.resolutions[i] = int(r)
    for d in range(3):
        cfg.aabb_min[d] = spec.aabb_min[d]
        cfg.aabb_max[d] = spec.aabb_max[d]
    cfg.sh_degree = spec.sh_degree
    cfg.n_params = spec.n_params
    cfg.n_frequencies = spec.n_frequencies
    cfg.n_hidden_layers = spec.n_hidden_layers
    cfg.hidden_width = spec.hidden_width
    cfg.out_activation = spec.out_activation
    cfg.dir_frequencies = getattr(spec, "dir_frequencies", 0)
    return cfg


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _chk(a: np.ndarray, dtype, name: str) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=dtype)
    if not a.flags.c_contiguous:
        raise ValueError(name)
    return a


def level_table(spec):
    cfg = make_config(spec)
    N = np.zeros(spec.n_levels, dtype=np.uint32)
    dense = np.zeros(spec.n_levels, dtype=np.uint32)
    rc = lib().niv_oracle_level_table(C.byref(cfg), _p(N), _p(dense))
    if rc:
        raise ValueError("niv_oracle_level_table failed")
    return N, dense.astype(bool)


def hash_index(vx: int, vy: int, vz: int, log2_T: int) -> int:
    return int(lib().niv_oracle_hash(vx & 0xFFFFFFFF, vy & 0xFFFFFFFF, vz & 0xFFFFFFFF, log2_T))


def half_to_double(bits: int) -> float:
    return float(lib().niv_oracle_half_to_double(bits))


def sh16(n) -> np.ndarray:
    v = np.ascontiguousarray(n, dtype=np.float64)
    out = np.zeros(16, dtype=np.float64)
    lib().niv_oracle_sh16(_p(v), _p(out))
    return out


def param_encode(t: float, n_frequencies: int) -> np.ndarray:
    out = np.zeros(2 * n_frequencies, dtype=np.float64)
    lib().niv_oracle_param_encode(C.c_double(t), C.c_uint32(n_frequencies), _p(out))
    return out


def mlp(spec, weights_blob, biases_blob, x) -> np.ndarray:
    cfg = make_config(spec)
    w = _chk(weights_blob, np.float16, "weights")
    b = None if biases_blob is None else _chk(biases_blob, np.float32, "biases")
    xx = _chk(x, np.float64, "x")
    y = np.zeros(3, dtype=np.float64)
    lib().niv_oracle_mlp(C.byref(cfg), _p(w), _p(b), _p(xx), _p(y))
    return y


def encode(spec, table, pos, nrm, param=None, want_features=True, n_threads: int = 0):
    """-> dict(idx [n][L][8] u32, cell [n][L][3] i32, frac [n][L][3] f32, features [n][in_dim] f64)."""
    cfg = make_config(spec)
    table = _chk(table, np.float16, "table")
    pos = _chk(pos, np.float32, "pos")
    nrm = _chk(nrm, np.float32, "nrm")
    n = pos.shape[0]
    L = spec.n_levels
    prm = None if param is None else _chk(param, np.float32, "param")
    if spec.n_params and prm is None:
        raise ValueError("param required")
    idx = np.zeros((n, L, 8), dtype=np.uint32)
    cell = np.zeros((n, L, 3), dtype=np.int32)
    frac = np.zeros((n, L, 3), dtype=np.float32)
    feat = np.zeros((n, spec.in_dim), dtype=np.float64) if want_features else None
    rc = lib().niv_oracle_encode(C.byref(cfg), _p(table), _p(pos), _p(nrm), _p(prm), C.c_size_t(n),
                                 _p(idx), _p(cell), _p(frac), _p(feat), C.c_int(n_threads))
    if rc:
        raise ValueError("niv_oracle_encode failed")
    return {"idx": idx, "cell": cell, "frac": frac, "features": feat}


def infer(spec, table, weights_blob, biases_blob, pos, nrm, param=None, n_threads: int = 0,
          want_f64: bool = False):
    """Full path O0..O9 -> out [n][3] fp32 (and fp64 if want_f64)."""
    cfg = make_config(spec)
    table = _chk(table, np.float16, "table")
    w = _chk(weights_blob, np.float16, "weights")
    b = None if biases_blob is None else _chk(biases_blob, np.float32, "biases")
    pos = _chk(pos, np.float32, "pos")
    nrm = _chk(nrm, np.float32, "nrm")
    prm = None if param is None else _chk(param, np.float32, "param")
    if spec.n_params and prm is None:
        raise ValueError("param required")
    n = pos.shape[0]
    out32 = np.zeros((n, 3), dtype=np.float32)
    out64 = np.zeros((n, 3), dtype=np.float64) if want_f64 else None
    rc = lib().niv_oracle_infer(C.byref(cfg), _p(table), _p(w), _p(b), _p(pos), _p(nrm), _p(prm),
                                _p(out32), _p(out64), C.c_size_t(n), C.c_int(n_threads))
    if rc:
        raise ValueError("niv_oracle_infer failed")
    return (out32, out64) if want_f64 else out32


def infer_texel_params(spec, table, weights_blob, biases_blob, pos, nrm, tparam, n_threads: int = 0,
                       want_f64: bool = False):
    """as infer(), every texel with its own scene parameters tparam [n][n_params]."""
    cfg = make_config(spec)
    table = _chk(table, np.float16, "table")
    w = _chk(weights_blob, np.float16, "weights")
    b = None if biases_blob is None else _chk(biases_blob, np.float32, "biases")
    pos = _chk(pos, np.float32, "pos")
    nrm = _chk(nrm, np.float32, "nrm")
    tp = _chk(tparam, np.float32, "tparam")
    n = pos.shape[0]
    if spec.n_params == 0 or tp.size != n * spec.n_params:
        raise ValueError("tparam must hold n * n_params values")
    out32 = np.zeros((n, 3), dtype=np.float32)
    out64 = np.zeros((n, 3), dtype=np.float64) if want_f64 else None
    rc = lib().niv_oracle_infer_texel_params(C.byref(cfg), _p(table), _p(w), _p(b), _p(pos), _p(nrm), _p(tp),
                                             _p(out32), _p(out64), C.c_size_t(n), C.c_int(n_threads))
    if rc:
        raise ValueError("niv_oracle_infer_texel_params failed")
    return (out32, out64) if want_f64 else out32


def max_threads() -> int:
    return int(lib().niv_oracle_max_threads())


def compose(E, albedo, direct=None, emission=None) -> np.ndarray:
    """L = albedo / pi * E + direct + emission; E [eh][ew][3] at full or half resolution (bilinear upsample).
    -> [h][w][3] fp64."""
    E = _chk(E, np.float32, "E")
    albedo = _chk(albedo, np.float32, "albedo")
    d = None if direct is None else _chk(direct, np.float32, "direct")
    em = None if emission is None else _chk(emission, np.float32, "emission")
    h, w = albedo.shape[:2]
    out = np.zeros((h, w, 3), dtype=np.float64)
    rc = lib().niv_oracle_compose(_p(E), C.c_uint32(E.shape[1]), C.c_uint32(E.shape[0]), _p(albedo), _p(d), _p(em),
                                  _p(out), C.c_uint32(w), C.c_uint32(h))
    if rc:
        raise ValueError("niv_oracle_compose failed (resolutions must be equal or exactly 2x)")
    return out


# ---------------------------------------------------------------------------------------------------------------------
# the paper's probe baseline (niv_oracle_ext.c)
def probe_query(dims, bbox_min, bbox_max, coeffs, pos, nrm, cosine_falloff=True, n_threads: int = 0, debug=False):
    """coeffs [nz][ny][nx][9][3] fp16 (27 per probe, x fastest) -> E [n][3] fp32
    (debug: also fp64 E, the 8 normalised weights and the 8 probe indices per texel)."""
    d = (C.c_uint32 * 3)(*[int(v) for v in dims])
    lo = (C.c_float * 3)(*[float(v) for v in bbox_min])
    hi = (C.c_float * 3)(*[float(v) for v in bbox_max])
    coeffs = _chk(coeffs, np.float16, "coeffs")
    if coeffs.size != int(dims[0]) * int(dims[1]) * int(dims[2]) * 27:
        raise ValueError("coeffs must hold 27 values per probe")
    pos = _chk(pos, np.float32, "pos")
    nrm = _chk(nrm, np.float32, "nrm")
    n = pos.shape[0]
    out32 = np.zeros((n, 3), dtype=np.float32)
    out64 = np.zeros((n, 3), dtype=np.float64) if debug else None
    w = np.zeros((n, 8), dtype=np.float64) if debug else None
    pi = np.zeros((n, 8), dtype=np.uint32) if debug else None
    rc = lib().niv_oracle_probe_query(d, lo, hi, C.c_int(1 if cosine_falloff else 0), _p(coeffs), _p(pos), _p(nrm),
                                      C.c_size_t(n), _p(out32), _p(out64), _p(w), _p(pi), C.c_int(n_threads))
    if rc:
        raise ValueError("niv_oracle_probe_query failed")
    return (out32, out64, w, pi) if debug else out32


# ---------------------------------------------------------------------------------------------------------------------
# compact G-buffer formats and fp16 output (niv_oracle_ext.c)
def decode_gbuffer(fmt: int, bbox_min, bbox_max, a, b=None):
    """-> (pos [n][3] fp32, nrm [n][3] fp32) of a G-buffer in format 0..3."""
    a = np.ascontiguousarray(a)
    rec = {0: 12, 1: 16, 2: 16, 3: 8}[int(fmt)]
    n = a.nbytes // rec
    if b is not None:
        b = np.ascontiguousarray(b)
    lo = (C.c_float * 3)(*[float(v) for v in bbox_min])
    hi = (C.c_float * 3)(*[float(v) for v in bbox_max])
    pos = np.zeros((n, 3), dtype=np.float32)
    nrm = np.zeros((n, 3), dtype=np.float32)
    rc = lib().niv_oracle_decode_gbuffer(C.c_int(int(fmt)), lo, hi, _p(a), _p(b), C.c_size_t(n), _p(pos), _p(nrm))
    if rc:
        raise ValueError("niv_oracle_decode_gbuffer failed")
    return pos, nrm


def quantise_f16x4(e) -> np.ndarray:
    """[n][3] fp32 -> [n][4] uint16: (r, g, b, 0) as binary16 bit patterns, round to nearest even."""
    e = _chk(e, np.float32, "e")
    out = np.zeros((e.shape[0], 4), dtype=np.uint16)
    if lib().niv_oracle_quantise_f16x4(_p(e), C.c_size_t(e.shape[0]), _p(out)):
        raise ValueError("niv_oracle_quantise_f16x4 failed")
    return out


def quantise_rgb9e5(e) -> np.ndarray:
    """[n][3] fp32 -> [n] uint32: shared-exponent RGB9E5 words (steps Q1-Q4 of niv_oracle_ext.c)."""
    e = _chk(e, np.float32, "e")
    out = np.zeros((e.shape[0],), dtype=np.uint32)
    if lib().niv_oracle_quantise_rgb9e5(_p(e), C.c_size_t(e.shape[0]), _p(out)):
        raise ValueError("niv_oracle_quantise_rgb9e5 failed")
    return out


def decode_rgb9e5(w) -> np.ndarray:
    """[n] uint32 RGB9E5 words -> [n][3] fp64 values."""
    w = _chk(w, np.uint32, "w")
    out = np.zeros((w.shape[0], 3), dtype=np.float64)
    if lib().niv_oracle_decode_rgb9e5(_p(w), C.c_size_t(w.shape[0]), _p(out)):
        raise ValueError("niv_oracle_decode_rgb9e5 failed")
    return out


def compose_jb(E, pos_half, nrm_half, pos, nrm, albedo, sigma, power, direct=None, emission=None) -> np.ndarray:
    """Deferred compose with joint-bilateral upsampling of half-resolution E (niv_oracle_ext.c niv_oracle_compose_jb).
    E, pos_half, nrm_half [eh][ew][3]; pos, nrm, albedo (, direct, emission) [h][w][3] with (h, w) = (2 eh, 2 ew) -> fp64."""
    E, pos_half, nrm_half = (_chk(a, np.float32, "half") for a in (E, pos_half, nrm_half))
    pos, nrm, albedo = (_chk(a, np.float32, "full") for a in (pos, nrm, albedo))
    direct = None if direct is None else _chk(direct, np.float32, "direct")
    emission = None if emission is None else _chk(emission, np.float32, "emission")
    h, w = albedo.shape[:2]
    eh, ew = E.shape[:2]
    out = np.zeros((h, w, 3), dtype=np.float64)
    rc = lib().niv_oracle_compose_jb(_p(E), _p(pos_half), _p(nrm_half), C.c_uint32(ew), C.c_uint32(eh), _p(pos), _p(nrm),
                                     _p(albedo), _p(direct), _p(emission), C.c_double(sigma), C.c_double(power), _p(out),
                                     C.c_uint32(w), C.c_uint32(h))
    if rc:
        raise ValueError("niv_oracle_compose_jb failed (E must be at exactly half the resolution; sigma > 0, power >= 0)")
    return out


# ---------------------------------------------------------------------------------------------------------------------
# compact table storage (dense levels hold (N + 1)^3 entries)
def compact_entries(spec) -> int:
    cfg = make_config(spec)
    lib().niv_oracle_table_compact.restype = C.c_longlong
    n = lib().niv_oracle_table_compact(C.byref(cfg), None, None)
    if n < 0:
        raise ValueError("niv_oracle_table_compact failed")
    return int(n)


def table_compact(spec, table) -> np.ndarray:
    """[L][T][F] fp16 -> the compact table (flat fp16, compact_entries(spec) * F values)."""
    cfg = make_config(spec)
    table = _chk(table, np.float16, "table")
    out = np.zeros(compact_entries(spec) * spec.n_features, dtype=np.float16)
    lib().niv_oracle_table_compact.restype = C.c_longlong
    if lib().niv_oracle_table_compact(C.byref(cfg), _p(table), _p(out)) < 0:
        raise ValueError("niv_oracle_table_compact failed")
    return out


def table_expand(spec, compact) -> np.ndarray:
    cfg = make_config(spec)
    compact = _chk(compact, np.float16, "compact")
    out = np.zeros((spec.n_levels, spec.table_size, spec.n_features), dtype=np.float16)
    lib().niv_oracle_table_expand.restype = C.c_longlong
    if lib().niv_oracle_table_expand(C.byref(cfg), _p(compact), _p(out)) < 0:
        raise ValueError("niv_oracle_table_expand failed")
    return out
