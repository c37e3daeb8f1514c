"""ctypes binding of libniv.so (include/niv.h).  Argument marshalling only: every step of the path runs in
the CUDA kernels behind the C ABI.  PyTorch is used for device memory and streams, nothing else.

There is NO CPU fallback: if libniv.so is missing or no CUDA device is present, the calls raise.
This module never imports anything under oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("NIV_LIB") or os.path.join(_HERE, "libniv.so")   # NIV_LIB: an experimental build

NIV_API_VERSION = 1
NIV_OK = 0
NIV_ERR_INVALID_ARG = -1
NIV_ERR_UNSUPPORTED = -2
NIV_ERR_NOT_LOADED = -3
NIV_ERR_CUDA = -4
NIV_ERR_ALLOC = -5
NIV_ERR_TOO_LARGE = -6
NIV_STATIC_MAX_TEXELS = 262144        # niv_infer_host_static
NIV_OUT_LINEAR = 0
NIV_OUT_SIGMOID = 1
NIV_CENSUS_COUNTS = 49      # niv_probe_sectors: [0,16) sectors, [16,32) lines, [32] active texels, [33,49) touched

# every symbol include/niv.h declares (tests check that the library exports all of them)
NIV_GBUF_F32X3, NIV_GBUF_F32X4, NIV_GBUF_P32_OCT16, NIV_GBUF_P16_OCT8 = 0, 1, 2, 3
NIV_OUTFMT_F32X3, NIV_OUTFMT_F16X4, NIV_OUTFMT_RGB9E5 = 0, 1, 2
_GBUF_BYTES = {0: (12, 12), 1: (16, 16), 2: (16, 0), 3: (8, 0)}      # bytes per texel of gbuf_a, gbuf_b
_OUT_BYTES = {0: 12, 1: 8, 2: 4}

EXPORTS = ("niv_create", "niv_get_info", "niv_load_params", "niv_load_params_compact", "niv_infer", "niv_infer_image", "niv_infer_texel_params",
           "niv_infer_host", "niv_probe_sectors_image",
           "niv_infer_host_static",
           "niv_infer_packed", "niv_infer_image_packed", "niv_infer_host_packed", "niv_decode_gbuffer", "niv_debug_arow",
           "niv_infer_shade", "niv_infer_image_shade",
           "niv_encode",
           "niv_debug_encode", "niv_compose", "niv_compose_jb", "niv_destroy", "niv_error_string", "niv_last_cuda_error", "niv_probe_gather",
           "niv_probe_sectors",
           "niv_probes_create", "niv_probes_load", "niv_probes_query", "niv_probes_census", "niv_probes_destroy")


class NivConfig(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("api_version", C.c_uint32),
        ("n_levels", C.c_uint32), ("n_features", C.c_uint32), ("log2_table_size", C.c_uint32),
        ("base_resolution", C.c_uint32), ("per_level_scale", C.c_double),
        ("resolutions", C.c_uint32 * 16),
        ("aabb_min", C.c_float * 3), ("aabb_max", C.c_float * 3),
        ("sh_degree", C.c_uint32), ("n_params", C.c_uint32), ("n_frequencies", C.c_uint32),
        ("n_hidden_layers", C.c_uint32), ("hidden_width", C.c_uint32), ("out_activation", C.c_uint32),
        ("device", C.c_int32), ("dir_frequencies", C.c_uint32),
    ]


class NivInfo(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("in_dim", C.c_uint32),
        ("resolution", C.c_uint32 * 16), ("is_dense", C.c_uint32 * 16),
        ("table_bytes", C.c_uint64), ("weight_bytes", C.c_uint64), ("bias_bytes", C.c_uint64),
        ("num_sms", C.c_uint32), ("ctas_per_sm", C.c_uint32), ("tile_texels", C.c_uint32),
        ("smem_bytes", C.c_uint32), ("image_tiled", C.c_uint32), ("texel_params", C.c_uint32),
        ("cell_levels", C.c_uint32), ("kernel_levels", C.c_uint32), ("cell_bytes", C.c_uint64),
        ("table_bytes_compact", C.c_uint64), ("table_bytes_device", C.c_uint64),
    ]


class NivProbeConfig(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("dims", C.c_uint32 * 3), ("bbox_min", C.c_float * 3),
                ("bbox_max", C.c_float * 3), ("cosine_falloff", C.c_uint32), ("device", C.c_int32)]


class NivError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        msg = lib().niv_error_string(code).decode()
        if code == NIV_ERR_CUDA:
            msg += " [cudaError %d]" % lib().niv_last_cuda_error()
        super().__init__("%s: %s (%d)" % (what, msg, code))


_lib = None


def lib():
    """Load libniv.so (built in-tree by paper_2602_12949_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError("libniv.so not built: run `python -m paper_2602_12949_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        vp, sz = C.c_void_p, C.c_size_t
        L.niv_create.argtypes = [C.POINTER(NivConfig), C.POINTER(vp)]
        L.niv_get_info.argtypes = [vp, C.POINTER(NivInfo)]
        L.niv_load_params.argtypes = [vp, vp, sz, vp, sz, vp, sz, C.c_int, vp]
        L.niv_load_params_compact.argtypes = [vp, vp, sz, vp, sz, vp, sz, C.c_int, vp]
        L.niv_infer.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, sz, vp]
        L.niv_infer_host.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, sz, vp]
        L.niv_infer_host_static.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, sz, vp]
        L.niv_infer_texel_params.argtypes = [vp, vp, vp, vp, vp, sz, vp]
        L.niv_infer_image.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, C.c_uint32, C.c_uint32, vp]
        L.niv_probe_sectors_image.argtypes = [vp, vp, vp, C.c_uint32, C.c_uint32, vp, vp]
        L.niv_encode.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, sz, vp]
        L.niv_infer_packed.argtypes = [vp, C.c_int, vp, vp, C.POINTER(C.c_float), C.c_int, vp, sz, vp]
        L.niv_infer_shade.argtypes = [vp, C.c_int, vp, vp, C.POINTER(C.c_float), vp, vp, vp, C.c_int, vp, sz, vp]
        L.niv_infer_image_shade.argtypes = [vp, C.c_int, vp, vp, C.POINTER(C.c_float), vp, vp, vp, C.c_int, vp,
                                            C.c_uint32, C.c_uint32, vp]
        L.niv_infer_image_packed.argtypes = [vp, C.c_int, vp, vp, C.POINTER(C.c_float), C.c_int, vp, C.c_uint32, C.c_uint32, vp]
        L.niv_infer_host_packed.argtypes = [vp, C.c_int, vp, vp, C.POINTER(C.c_float), C.c_int, vp, sz, vp]
        L.niv_decode_gbuffer.argtypes = [vp, C.c_int, vp, vp, vp, vp, sz, vp]
        L.niv_debug_arow.argtypes = [vp, vp, vp, C.POINTER(C.c_float), vp, vp, C.c_uint32, sz, vp]
        L.niv_debug_encode.argtypes = [vp, vp, vp, C.POINTER(C.c_float), sz, vp, vp, vp, vp, vp]
        L.niv_compose.argtypes = [vp, C.c_uint32, C.c_uint32, vp, vp, vp, vp, C.c_uint32, C.c_uint32, vp]
        L.niv_compose_jb.argtypes = [vp, vp, vp, C.c_uint32, C.c_uint32, vp, vp, vp, vp, vp, C.c_float, C.c_float, vp,
                                     C.c_uint32, C.c_uint32, vp]
        L.niv_destroy.argtypes = [vp]
        L.niv_error_string.argtypes = [C.c_int]
        L.niv_error_string.restype = C.c_char_p
        L.niv_last_cuda_error.argtypes = []
        L.niv_probe_gather.argtypes = [vp, sz, C.c_int, C.c_uint32, C.c_uint32, C.c_uint32, vp, vp]
        L.niv_probe_sectors.argtypes = [vp, vp, vp, sz, vp, vp]
        L.niv_probes_create.argtypes = [C.POINTER(NivProbeConfig), C.POINTER(vp)]
        L.niv_probes_load.argtypes = [vp, vp, sz, C.c_int, vp]
        L.niv_probes_query.argtypes = [vp, vp, vp, vp, sz, vp]
        L.niv_probes_census.argtypes = [vp, vp, vp, sz, vp, vp]
        L.niv_probes_destroy.argtypes = [vp]
        for name in EXPORTS:
            if name != "niv_error_string":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def make_config(spec, device: int = 0) -> NivConfig:
    """spec: any object with the ModelSpec attribute names (paper_2602_12949_b200.inputs.ModelSpec)."""
    cfg = NivConfig()
    cfg.struct_size = C.sizeof(NivConfig)
    cfg.api_version = NIV_API_VERSION
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
    cfg.device = device
    return cfg


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream or None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


def _dev(t, dtype, name: str, cols: Optional[int] = None):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be a contiguous CUDA tensor of %s" % (name, dtype))
    if cols is not None and (t.dim() != 2 or t.shape[1] != cols):
        raise TypeError("%s must have shape [n][%d]" % (name, cols))
    return t.data_ptr()


def _same_rows(n: int, **bufs):
    """Every per-texel buffer of a call must hold n rows (a shorter one would be read or written out of bounds)."""
    for name, t in bufs.items():
        if t.shape[0] != n:
            raise ValueError("%s holds %d rows, pos holds %d" % (name, t.shape[0], n))


def _params(param: Optional[Sequence[float]], n_params: int):
    if n_params == 0:
        if param is not None and len(param):
            raise ValueError("model takes no scene parameter")
        return None
    if param is None or len(param) != n_params:
        raise ValueError("model takes %d scene parameter(s)" % n_params)
    return (C.c_float * n_params)(*[float(v) for v in param])


class NivModel:
    """Handle on a niv_model.  Methods mirror the C ABI one to one."""

    def __init__(self, spec, device: int = 0):
        self.spec = spec
        self._h = C.c_void_p()
        cfg = make_config(spec, device)
        rc = lib().niv_create(C.byref(cfg), C.byref(self._h))
        if rc != NIV_OK:
            self._h = C.c_void_p()
            raise NivError(rc, "niv_create")
        self.info = NivInfo()
        rc = lib().niv_get_info(self._h, C.byref(self.info))
        if rc != NIV_OK:
            raise NivError(rc, "niv_get_info")

    # ---- parameters -------------------------------------------------------------------------------
    def load_params(self, table, weights, biases=None, stream=None, compact=False):
        """table [L][T][F] fp16, weights flat fp16 blob W1|W2|.., biases flat fp32 blob or None.
        Each is a numpy array (host) or a CUDA tensor (device); all three must live on the same side."""
        import numpy as np
        on_dev = not isinstance(table, np.ndarray)
        if on_dev:
            import torch
            tp, tb = _dev(table, torch.float16, "table"), table.numel() * 2
            wp, wb = _dev(weights, torch.float16, "weights"), weights.numel() * 2
            bp, bb = (None, 0) if biases is None else (_dev(biases, torch.float32, "biases"), biases.numel() * 4)
        else:
            table = np.ascontiguousarray(table, dtype=np.float16)
            weights = np.ascontiguousarray(weights, dtype=np.float16)
            tp, tb = table.ctypes.data, table.nbytes
            wp, wb = weights.ctypes.data, weights.nbytes
            if biases is None:
                bp, bb = None, 0
            else:
                biases = np.ascontiguousarray(biases, dtype=np.float32)
                bp, bb = biases.ctypes.data, biases.nbytes
        fn = lib().niv_load_params_compact if compact else lib().niv_load_params     # compact: the table of
        rc = fn(self._h, tp, tb, wp, wb, bp, bb, int(on_dev), _stream_ptr(stream))      # niv_info.table_bytes_compact
        if rc != NIV_OK:
            raise NivError(rc, "niv_load_params_compact" if compact else "niv_load_params")

    # ---- the hot path -----------------------------------------------------------------------------
    def infer(self, pos, nrm, out, param=None, stream=None):
        """out[i] = E_theta(pos[i], nrm[i][, param]); device tensors [n][3] fp32; asynchronous."""
        import torch
        n = pos.shape[0]
        _same_rows(n, nrm=nrm, out=out)
        rc = lib().niv_infer(self._h, _dev(pos, torch.float32, "pos", 3) if n else None,
                             _dev(nrm, torch.float32, "nrm", 3) if n else None,
                             _params(param, self.spec.n_params),
                             _dev(out, torch.float32, "out", 3) if n else None, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer")
        return out

    def infer_image(self, pos, nrm, out, width, height, param=None, stream=None):
        """As infer() for a row-major height x width G-buffer ([h*w][3] tensors): warps take 8 x 4 pixel blocks."""
        import torch
        n = int(width) * int(height)
        if pos.shape[0] != n or nrm.shape[0] != n or out.shape[0] != n:
            raise ValueError("buffers must hold width * height texels")
        rc = lib().niv_infer_image(self._h, _dev(pos, torch.float32, "pos", 3) if n else None,
                                   _dev(nrm, torch.float32, "nrm", 3) if n else None,
                                   _params(param, self.spec.n_params),
                                   _dev(out, torch.float32, "out", 3) if n else None, int(width), int(height),
                                   _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_image")
        return out

    def infer_texel_params(self, pos, nrm, tparam, out, stream=None):
        """as infer(), every texel with its own scene parameters; tparam device [n][n_params] fp32."""
        import torch
        n = pos.shape[0]
        _same_rows(n, nrm=nrm, tparam=tparam, out=out)
        rc = lib().niv_infer_texel_params(self._h, _dev(pos, torch.float32, "pos", 3) if n else None,
                                          _dev(nrm, torch.float32, "nrm", 3) if n else None,
                                          _dev(tparam, torch.float32, "tparam", self.spec.n_params) if n else None,
                                          _dev(out, torch.float32, "out", 3) if n else None, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_texel_params")
        return out

    def infer_host(self, pos, nrm, out, param=None, stream=None):
        """Same, with HOST buffers (numpy arrays or pinned CPU tensors, [n][3] fp32): the library stages
        them through its own device buffers (H2D, kernel, D2H) and synchronises the stream."""
        n = pos.shape[0]
        _same_rows(n, nrm=nrm, out=out)
        rc = lib().niv_infer_host(self._h, _host_ptr(pos, "pos"), _host_ptr(nrm, "nrm"),
                                  _params(param, self.spec.n_params), _host_ptr(out, "out"), n,
                                  _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_host")
        return out

    # ---- compact G-buffer formats / fp16 output (include/niv.h: *_packed).  Buffers are taken by byte size: any dtype.
    @staticmethod
    def _raw(t, name, nbytes, cuda):
        """pointer of a contiguous buffer (CUDA tensor, or host numpy array / CPU tensor) holding exactly nbytes"""
        import numpy as np
        if t is None:
            if nbytes:
                raise TypeError("%s is required for this format" % name)
            return None
        if isinstance(t, np.ndarray):
            if cuda or not t.flags.c_contiguous:
                raise TypeError("%s must be a contiguous %s buffer" % (name, "CUDA" if cuda else "host"))
            have, ptr = t.nbytes, t.ctypes.data
        else:
            import torch
            if not isinstance(t, torch.Tensor) or t.is_cuda != cuda or not t.is_contiguous():
                raise TypeError("%s must be a contiguous %s buffer" % (name, "CUDA" if cuda else "host"))
            have, ptr = t.numel() * t.element_size(), t.data_ptr()
        if nbytes and have != nbytes:
            raise ValueError("%s holds %d bytes, the call needs %d" % (name, have, nbytes))
        return ptr

    def _packed_args(self, gbuf_format, a, b, out_format, out, n, cuda):
        ab, bb = _GBUF_BYTES[int(gbuf_format)]
        return (self._raw(a, "gbuf_a", ab * n, cuda), self._raw(b, "gbuf_b", bb * n, cuda) if bb else None,
                self._raw(out, "out", _OUT_BYTES[int(out_format)] * n, cuda))

    def infer_packed(self, gbuf_format, a, b, out, n, out_format=NIV_OUTFMT_F32X3, param=None, stream=None):
        pa, pb, po = self._packed_args(gbuf_format, a, b, out_format, out, n, True)
        rc = lib().niv_infer_packed(self._h, int(gbuf_format), pa, pb, _params(param, self.spec.n_params),
                                    int(out_format), po, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_packed")
        return out

    def infer_shade(self, a, b, albedo, out, n, direct=None, emission=None, gbuf_format=NIV_GBUF_F32X3,
                    out_format=NIV_OUTFMT_F32X3, param=None, stream=None, image=None):
        """niv_infer_shade (include/niv.h): out = albedo / pi * E + direct + emission in the inference kernel's epilogue;
        a, b, out as infer_packed, albedo / direct / emission CUDA float32 [n][3] (the last two optional).
        image = (width, height): niv_infer_image_shade on row-major buffers of width * height == n texels."""
        pa, pb, po = self._packed_args(gbuf_format, a, b, out_format, out, n, True)
        import torch
        sh = [None if t is None else _dev(t, torch.float32, name, 3) for name, t in
              (("albedo", albedo), ("direct", direct), ("emission", emission))]
        _same_rows(n, **{k: v for k, v in (("albedo", albedo), ("direct", direct), ("emission", emission)) if v is not None})
        if image is not None:
            w, h = int(image[0]), int(image[1])
            if w * h != n:
                raise ValueError("image is %d x %d, the buffers hold %d texels" % (w, h, n))
            rc = lib().niv_infer_image_shade(self._h, int(gbuf_format), pa, pb, _params(param, self.spec.n_params),
                                             sh[0], sh[1], sh[2], int(out_format), po, w, h, _stream_ptr(stream))
        else:
            rc = lib().niv_infer_shade(self._h, int(gbuf_format), pa, pb, _params(param, self.spec.n_params),
                                       sh[0], sh[1], sh[2], int(out_format), po, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_shade")
        return out

    def infer_image_packed(self, gbuf_format, a, b, out, width, height, out_format=NIV_OUTFMT_F32X3, param=None, stream=None):
        n = int(width) * int(height)
        pa, pb, po = self._packed_args(gbuf_format, a, b, out_format, out, n, True)
        rc = lib().niv_infer_image_packed(self._h, int(gbuf_format), pa, pb, _params(param, self.spec.n_params),
                                          int(out_format), po, int(width), int(height), _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_image_packed")
        return out

    def infer_host_packed(self, gbuf_format, a, b, out, n, out_format=NIV_OUTFMT_F32X3, param=None, stream=None):
        pa, pb, po = self._packed_args(gbuf_format, a, b, out_format, out, n, False)
        rc = lib().niv_infer_host_packed(self._h, int(gbuf_format), pa, pb, _params(param, self.spec.n_params),
                                         int(out_format), po, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_host_packed")
        return out

    def arow_words(self) -> int:
        """32-bit words of one layer-1 A row of the fused kernel (include/niv.h niv_debug_arow)."""
        hw = self.info.kernel_levels * self.spec.n_features // 2 if self.spec.n_levels else 24
        return (hw + (8 if self.spec.sh_degree else (3 + 6 * getattr(self.spec, "dir_frequencies", 0) + 1) // 2) + 7) // 8 * 8

    def debug_arow(self, pos, nrm, out, arow, param=None, stream=None):
        """niv_infer + the fused kernel's layer-1 A rows: arow device int32 [n][arow_words()]."""
        import torch
        n = pos.shape[0]
        _same_rows(n, nrm=nrm, out=out, arow=arow)
        rc = lib().niv_debug_arow(self._h, _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3),
                                  _params(param, self.spec.n_params), _dev(out, torch.float32, "out", 3),
                                  _dev(arow, torch.int32, "arow", self.arow_words()), self.arow_words(), n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_debug_arow")

    def decode_gbuffer(self, gbuf_format, a, b, pos, nrm, n, stream=None):
        """pos, nrm: device [n][3] fp32 outputs = what the fused kernels decode from the compact G-buffer."""
        import torch
        ab, bb = _GBUF_BYTES[int(gbuf_format)]
        rc = lib().niv_decode_gbuffer(self._h, int(gbuf_format), self._raw(a, "gbuf_a", ab * n, True),
                                      self._raw(b, "gbuf_b", bb * n, True) if bb else None,
                                      _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3), n,
                                      _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_decode_gbuffer")

    def infer_host_static(self, pos, nrm, out, param=None, stream=None):
        """infer_host without any allocation: staged through the library's static device array; at most
        NIV_STATIC_MAX_TEXELS texels per call (include/niv.h niv_infer_host_static)."""
        n = pos.shape[0]
        _same_rows(n, nrm=nrm, out=out)
        rc = lib().niv_infer_host_static(self._h, _host_ptr(pos, "pos"), _host_ptr(nrm, "nrm"),
                                         _params(param, self.spec.n_params), _host_ptr(out, "out"), n,
                                         _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_infer_host_static")
        return out

    def encode(self, pos, nrm, features, param=None, stream=None):
        """features: device [n][in_dim] fp16."""
        import torch
        n = pos.shape[0]
        rc = lib().niv_encode(self._h, _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3),
                              _params(param, self.spec.n_params),
                              _dev(features, torch.float16, "features", self.info.in_dim), n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_encode")
        return features

    def debug_encode(self, pos, nrm, param=None, idx=None, cell=None, frac=None, features=None, stream=None):
        import torch
        n = pos.shape[0]
        rc = lib().niv_debug_encode(
            self._h, _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3),
            _params(param, self.spec.n_params), n,
            None if idx is None else _dev(idx, torch.int32, "idx"),
            None if cell is None else _dev(cell, torch.int32, "cell"),
            None if frac is None else _dev(frac, torch.float32, "frac"),
            None if features is None else _dev(features, torch.float32, "features", self.info.in_dim),
            _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_debug_encode")

    def probe_sectors(self, pos, nrm, counts, stream=None):
        """counts: device int64[NIV_CENSUS_COUNTS] (include/niv.h niv_probe_sectors)."""
        import torch
        rc = lib().niv_probe_sectors(self._h, _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3),
                                     pos.shape[0], _dev(counts, torch.int64, "counts"), _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_probe_sectors")

    def probe_sectors_image(self, pos, nrm, width, height, counts, stream=None):
        """The census for infer_image's warps (include/niv.h niv_probe_sectors_image)."""
        import torch
        rc = lib().niv_probe_sectors_image(self._h, _dev(pos, torch.float32, "pos", 3),
                                           _dev(nrm, torch.float32, "nrm", 3), int(width), int(height),
                                           _dev(counts, torch.int64, "counts"), _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_probe_sectors_image")

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().niv_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _host_ptr(a, name: str):
    import numpy as np
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags.c_contiguous:
            raise TypeError("%s must be a contiguous float32 array" % name)
        return a.ctypes.data
    import torch
    if isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == torch.float32 and a.is_contiguous():
        return a.data_ptr()
    raise TypeError("%s must be a host float32 buffer" % name)


def probe_gather(buf, pattern: int, n_ctas: int, loads_per_lane: int, seed: int, sink, stream=None):
    """Launch the gather micro-benchmark (include/niv.h niv_probe_gather) on `buf` (CUDA uint8/int32 tensor)."""
    rc = lib().niv_probe_gather(buf.data_ptr(), buf.numel() * buf.element_size(), pattern, n_ctas,
                                loads_per_lane, seed, sink.data_ptr(), _stream_ptr(stream))
    if rc != NIV_OK:
        raise NivError(rc, "niv_probe_gather")


def compose_jb(E, pos_half, nrm_half, pos, nrm, albedo, out, sigma, power, direct=None, emission=None, stream=None):
    """niv_compose_jb (include/niv.h): the compose with joint-bilateral upsampling of half-resolution E; CUDA fp32 tensors,
    E / pos_half / nrm_half [eh][ew][3], the rest [2 eh][2 ew][3].  Asynchronous."""
    import torch
    h, w = albedo.shape[:2]
    eh, ew = E.shape[:2]
    for name, t, shape in (("E", E, (eh, ew, 3)), ("pos_half", pos_half, (eh, ew, 3)), ("nrm_half", nrm_half, (eh, ew, 3)),
                           ("pos", pos, (h, w, 3)), ("nrm", nrm, (h, w, 3)), ("albedo", albedo, (h, w, 3)),
                           ("out", out, (h, w, 3)), ("direct", direct, (h, w, 3)), ("emission", emission, (h, w, 3))):
        if t is None:
            continue
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() \
                or tuple(t.shape) != shape:
            raise TypeError("%s must be a contiguous CUDA float32 tensor of shape %s" % (name, (shape,)))
    rc = lib().niv_compose_jb(E.data_ptr(), pos_half.data_ptr(), nrm_half.data_ptr(), ew, eh, pos.data_ptr(), nrm.data_ptr(),
                              albedo.data_ptr(), None if direct is None else direct.data_ptr(),
                              None if emission is None else emission.data_ptr(), float(sigma), float(power),
                              out.data_ptr(), w, h, _stream_ptr(stream))
    if rc != NIV_OK:
        raise NivError(rc, "niv_compose_jb")
    return out


def compose(E, albedo, out, direct=None, emission=None, stream=None):
    """niv_compose (include/niv.h): out = albedo / pi * E + direct + emission; CUDA fp32 tensors, E [eh][ew][3] at the
    resolution of albedo [h][w][3] or at half of it.  Asynchronous."""
    import torch
    for name, t in (("E", E), ("albedo", albedo), ("out", out), ("direct", direct), ("emission", emission)):
        if t is None:
            continue
        if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() \
                or t.dim() != 3 or t.shape[2] != 3:
            raise TypeError("%s must be a contiguous CUDA float32 tensor [h][w][3]" % name)
    h, w = albedo.shape[:2]
    for name, t in (("out", out), ("direct", direct), ("emission", emission)):
        if t is not None and tuple(t.shape) != (h, w, 3):
            raise TypeError("%s must have the shape of albedo" % name)
    rc = lib().niv_compose(E.data_ptr(), E.shape[1], E.shape[0], albedo.data_ptr(),
                           None if direct is None else direct.data_ptr(),
                           None if emission is None else emission.data_ptr(), out.data_ptr(), w, h, _stream_ptr(stream))
    if rc != NIV_OK:
        raise NivError(rc, "niv_compose")


class NivProbeGrid:
    """Handle on a niv_probe_grid (the paper's probe baseline).  Methods mirror the C ABI one to one."""

    def __init__(self, dims, bbox_min, bbox_max, cosine_falloff: bool = True, device: int = 0):
        cfg = NivProbeConfig()
        cfg.struct_size = C.sizeof(NivProbeConfig)
        for d in range(3):
            cfg.dims[d] = int(dims[d])
            cfg.bbox_min[d] = float(bbox_min[d])
            cfg.bbox_max[d] = float(bbox_max[d])
        cfg.cosine_falloff = 1 if cosine_falloff else 0
        cfg.device = device
        self.dims = tuple(int(v) for v in dims)
        self._h = C.c_void_p()
        rc = lib().niv_probes_create(C.byref(cfg), C.byref(self._h))
        if rc != NIV_OK:
            self._h = C.c_void_p()
            raise NivError(rc, "niv_probes_create")

    def load(self, coeffs, stream=None):
        """coeffs [nz][ny][nx][9][3] fp16: numpy array (host) or CUDA tensor."""
        import numpy as np
        if isinstance(coeffs, np.ndarray):
            coeffs = np.ascontiguousarray(coeffs, dtype=np.float16)
            ptr, nbytes, dev = coeffs.ctypes.data, coeffs.nbytes, 0
        else:
            import torch
            ptr, nbytes, dev = _dev(coeffs, torch.float16, "coeffs"), coeffs.numel() * 2, 1
        rc = lib().niv_probes_load(self._h, ptr, nbytes, dev, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_probes_load")

    def query(self, pos, nrm, out, stream=None):
        import torch
        n = pos.shape[0]
        if nrm.shape[0] != n or out.shape[0] != n:
            raise ValueError("pos, nrm and out must hold the same number of texels")
        rc = lib().niv_probes_query(self._h, _dev(pos, torch.float32, "pos", 3) if n else None,
                                    _dev(nrm, torch.float32, "nrm", 3) if n else None,
                                    _dev(out, torch.float32, "out", 3) if n else None, n, _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_probes_query")
        return out

    def census(self, pos, nrm, counts, stream=None):
        """counts: device int64[2] = (distinct probe sectors per warp, summed; active texels)."""
        import torch
        rc = lib().niv_probes_census(self._h, _dev(pos, torch.float32, "pos", 3), _dev(nrm, torch.float32, "nrm", 3),
                                     pos.shape[0], _dev(counts, torch.int64, "counts"), _stream_ptr(stream))
        if rc != NIV_OK:
            raise NivError(rc, "niv_probes_census")

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().niv_probes_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
