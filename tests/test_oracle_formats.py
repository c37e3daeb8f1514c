"""Pins of the oracle's compact G-buffer decode and fp16 output quantiser, CPU only.
Each check is against something other than the oracle itself: numpy's own binary16 conversion, exact special cases
(axis directions, end points of the box), a numpy float32 restatement of the pinned position sequence, and error bounds
that follow from the quantisation step."""
import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I


def test_f16_quantiser_is_round_to_nearest_even(oracle):
    rng = np.random.default_rng(5)
    x = np.concatenate([
        rng.standard_normal(200000).astype(np.float32) * np.float32(3.0),
        (rng.random(100000).astype(np.float32) * np.float32(2e-4)),                      # fp16 subnormal range
        np.float32([0.0, -0.0, 1.0, 65504.0, 65519.996, 65520.0, 1e30, -1e30, np.inf, -np.inf, 5.9604645e-8, 2.9802322e-8,
                    2.9802326e-8, 8.940697e-8, 6.1035156e-5, 6.0975552e-5, 1.00048828125, 1.0009765625, 1.00146484375]),
    ]).astype(np.float32)
    x = np.resize(x, (x.size // 3) * 3).reshape(-1, 3)
    got = oracle.quantise_f16x4(x)
    with np.errstate(over="ignore"):
        want = x.astype(np.float16).view(np.uint16)
    assert np.array_equal(got[:, :3], want)
    assert np.all(got[:, 3] == 0)
    # every finite binary16 value is a fixed point, and the midpoint between neighbours goes to the even one
    h = np.arange(0, 0x7C00, dtype=np.uint16)
    f = h.view(np.float16).astype(np.float32)
    back = oracle.quantise_f16x4(np.stack([f, -f, f], axis=1))
    assert np.array_equal(back[:, 0], h) and np.array_equal(back[:, 1], h | 0x8000)
    mid = ((f[:-1].astype(np.float64) + f[1:].astype(np.float64)) / 2).astype(np.float32)   # exact in fp32
    m = oracle.quantise_f16x4(np.stack([mid, mid, mid], axis=1))[:, 0]
    even = np.where(h[:-1] % 2 == 0, h[:-1], h[1:])
    assert np.array_equal(m, even)


def test_format_f32x4_is_the_same_buffer_with_a_stride(oracle):
    pos, nrm = I.positions_uniform(5000, I.ROOM_AABB, 3), I.normals_uniform(5000, 4)
    a, b = I.pack_gbuffer(I.GBUF_F32X4, pos, nrm)
    p, n = oracle.decode_gbuffer(I.GBUF_F32X4, *I.ROOM_AABB, a, b)
    assert np.array_equal(p, pos) and np.array_equal(n, nrm)
    p0, n0 = oracle.decode_gbuffer(I.GBUF_F32X3, *I.ROOM_AABB, pos, nrm)
    assert np.array_equal(p0, pos) and np.array_equal(n0, nrm)


@pytest.mark.parametrize("fmt,max_deg", [(I.GBUF_P32_OCT16, 0.004), (I.GBUF_P16_OCT8, 1.0)])
def test_octahedral_normals(oracle, fmt, max_deg):
    # the six axis directions are representable and decode exactly
    axes = np.float32([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]])
    pos = np.tile(np.float32([[1.0, 2.0, 3.0]]), (6, 1))
    a, _ = I.pack_gbuffer(fmt, pos, axes, I.ROOM_AABB)
    _, n = oracle.decode_gbuffer(fmt, *I.ROOM_AABB, a)
    assert np.array_equal(np.abs(n), np.abs(axes)) and np.array_equal(n[np.abs(axes) == 1], axes[np.abs(axes) == 1])
    # unit length to fp32 rounding, round trip within the quantisation step, background code -> exactly zero
    nrm = I.normals_uniform(200000, 9)
    nrm[17] = 0.0
    pos = I.positions_uniform(200000, I.ROOM_AABB, 2)
    a, _ = I.pack_gbuffer(fmt, pos, nrm, I.ROOM_AABB)
    _, n = oracle.decode_gbuffer(fmt, *I.ROOM_AABB, a)
    assert np.all(n[17] == 0.0)
    keep = np.arange(nrm.shape[0]) != 17
    length = np.linalg.norm(n[keep].astype(np.float64), axis=1)
    assert np.abs(length - 1.0).max() < 1.2e-7
    cross = np.linalg.norm(np.cross(n[keep].astype(np.float64), nrm[keep].astype(np.float64)), axis=1)
    assert np.degrees(np.arcsin(np.clip(cross, 0, 1))).max() < max_deg
    # every code decodes to a unit vector (or to the background): sweep all snorm8 pairs / a grid of snorm16 pairs
    if fmt == I.GBUF_P16_OCT8:
        v = np.arange(-127, 128, dtype=np.int8)
        ox, oy = np.meshgrid(v, v, indexing="ij")
        rec = np.zeros((ox.size, 8), dtype=np.uint8)
        rec[:, 6], rec[:, 7] = ox.reshape(-1).view(np.uint8), oy.reshape(-1).view(np.uint8)
        _, n = oracle.decode_gbuffer(fmt, *I.ROOM_AABB, rec)
        assert np.abs(np.linalg.norm(n.astype(np.float64), axis=1) - 1.0).max() < 1.2e-7
        # numpy restatement of the map on the same codes
        fx, fy = ox.reshape(-1) / 127.0, oy.reshape(-1) / 127.0
        z = 1 - np.abs(fx) - np.abs(fy)
        x = np.where(z < 0, (1 - np.abs(fy)) * np.where(np.signbit(fx), -1.0, 1.0), fx)
        y = np.where(z < 0, (1 - np.abs(fx)) * np.where(np.signbit(fy), -1.0, 1.0), fy)
        w = np.stack([x, y, z], axis=1)
        w /= np.linalg.norm(w, axis=1, keepdims=True)
        assert np.abs(n - w).max() < 1e-7


def test_unorm16_positions_follow_the_pinned_fp32_sequence(oracle):
    aabb = ((-3.0, 0.5, 2.0), (7.25, 4.75, 12.5))
    rng = np.random.default_rng(11)
    q = rng.integers(0, 65536, size=(100000, 3)).astype(np.uint16)
    q[0], q[1] = 0, 65535
    rec = np.zeros((q.shape[0], 8), dtype=np.uint8)
    rec[:, :6] = q.view(np.uint8).reshape(-1, 6)
    p, _ = oracle.decode_gbuffer(I.GBUF_P16_OCT8, aabb[0], aabb[1], rec)
    lo, hi = np.float32(aabb[0]), np.float32(aabb[1])
    ext = (hi - lo).astype(np.float32)
    k = np.float32(1.0) / np.float32(65535.0)
    u = (q.astype(np.float32) * k).astype(np.float32)
    want = ((u * ext).astype(np.float32) + lo).astype(np.float32)
    assert np.array_equal(p, want)
    assert np.array_equal(p[0], lo)                                   # q = 0 is the box's corner exactly
    assert np.abs(p[1].astype(np.float64) - hi).max() <= 1e-6         # q = 65535 is the far corner to fp32 rounding
    # the encoder's quantisation error is at most half a step (+ fp32 rounding)
    pos = I.positions_uniform(100000, aabb, 8)
    a, _ = I.pack_gbuffer(I.GBUF_P16_OCT8, pos, I.normals_uniform(100000, 1), aabb)
    p2, _ = oracle.decode_gbuffer(I.GBUF_P16_OCT8, aabb[0], aabb[1], a)
    step = (np.float64(hi) - np.float64(lo)) / 65535.0
    assert np.all(np.abs(p2.astype(np.float64) - pos.astype(np.float64)) <= 0.5 * step + 2e-6)


def test_decoded_buffers_feed_the_standard_path(oracle):
    """E on a compact G-buffer == E on its decoded fp32 buffers (the definition), and background codes stay background."""
    spec = I.spec_tiny()
    table = I.make_table(spec, 2)
    w, b = I.make_mlp(spec, 2)
    wb, bb = I.pack_weights(w), I.pack_biases(b)
    pos, nrm = I.positions_uniform(600, (spec.aabb_min, spec.aabb_max), 1), I.normals_uniform(600, 2)
    nrm[::7] = 0.0
    for fmt in (I.GBUF_F32X4, I.GBUF_P32_OCT16, I.GBUF_P16_OCT8):
        a, bbuf = I.pack_gbuffer(fmt, pos, nrm, (spec.aabb_min, spec.aabb_max))
        p, n = oracle.decode_gbuffer(fmt, spec.aabb_min, spec.aabb_max, a, bbuf)
        e = oracle.infer(spec, table, wb, bb, p, n)
        assert np.all(e[::7] == 0.0) and np.all(e[1::7] > 0.0)
        if fmt == I.GBUF_P32_OCT16:                                   # fp32 positions: only the normal is quantised
            e0 = oracle.infer(spec, table, wb, bb, pos, nrm)
            assert np.abs(e - e0).max() < 1e-3


def _rgb9e5_brute(c):
    """The definition by search: the SMALLEST exponent E in 0..31 for which every component, rounded to the nearest multiple
    of 2^(E-24) (ties up), fits nine bits -- no logarithm, no frexp."""
    c = [min(max(float(v), 0.0), 65408.0) if v == v else 0.0 for v in c]
    for E in range(32):
        step = 2.0 ** (E - 24)
        m = [int(np.floor(v / step + 0.5)) for v in c]
        if max(m) <= 511:
            return m[0] | (m[1] << 9) | (m[2] << 18) | (E << 27), [mm * step for mm in m]
    raise AssertionError("unreachable: 65408 fits E = 31")


def test_rgb9e5_quantiser(oracle):
    """Shared-exponent output.  Pins: hand-worked words ((1, 1, 1) = three mantissas 256 at
    E = 16; zero; the largest value; the rounding carry just below a power of two), the definition by exhaustive search over the
    exponent on 20,000 random triples of every magnitude, exact round trip of representable values, the error bound
    |c - dec| <= max_c / 511 / 2 ... 2^(E-25), clamping of negatives / NaN / values beyond the range."""
    q = lambda rows: oracle.quantise_rgb9e5(np.float32(rows))
    assert q([[1, 1, 1]])[0] == (256 | 256 << 9 | 256 << 18 | 16 << 27) == 0x84020100
    assert q([[0, 0, 0]])[0] == 0
    assert q([[65408, 0, 65408]])[0] == (511 | 511 << 18 | 31 << 27)
    assert q([[1e9, -3, float("nan")]])[0] == (511 | 31 << 27)                       # clamped high; negative and NaN -> 0
    assert q([[0.99999, 0.5, 0.25]])[0] == (256 | 128 << 9 | 64 << 18 | 16 << 27)    # 511.99 rounds to 512: the carry
    assert q([[0.5, 0.25, 0.125]])[0] == (256 | 128 << 9 | 64 << 18 | 15 << 27)
    assert q([[2.0 ** -20, 0, 0]])[0] == (16 | 0 << 27)                              # below 2^-16: E stays 0, 2^-20 / 2^-24 = 16
    assert q([[2.0 ** -26, 0, 0]])[0] == 0                                           # under half a step of E = 0
    rng = np.random.default_rng(11)
    mag = 2.0 ** rng.uniform(-27, 17, (20000, 1))
    x = (mag * rng.uniform(0, 1, (20000, 3))).astype(np.float32)
    x[::97, 1] *= -1
    got = q(x)
    dec = oracle.decode_rgb9e5(got)
    for i in range(0, 20000, 1):
        w, vals = _rgb9e5_brute(x[i])
        assert got[i] == w, (i, x[i], hex(got[i]), hex(w))
    xc = np.clip(x.astype(np.float64), 0.0, 65408.0)
    step = 2.0 ** ((got >> 27).astype(np.float64) - 24)
    assert np.all(np.abs(dec - xc) <= step[:, None] / 2)
    top = (got & 0x1FF) | ((got >> 9) & 0x1FF) | ((got >> 18) & 0x1FF)
    assert np.all((top >= 256) | ((got >> 27) == 0))                                 # normalised: the top mantissa bit is in use
    # representable values survive exactly
    words = (rng.integers(0, 512, 5000) | (rng.integers(0, 512, 5000) << 9) | (rng.integers(256, 512, 5000) << 18)
             | (rng.integers(0, 32, 5000) << 27)).astype(np.uint32)
    v = oracle.decode_rgb9e5(words)
    assert np.array_equal(q(v.astype(np.float32)), words)
