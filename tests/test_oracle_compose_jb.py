"""Pins of the oracle's joint-bilateral compose, CPU only: the cases where it
must reduce to something already pinned (the bilinear compose, itself pinned to torch's interpolate), closed forms, and a
numpy restatement written from the step list J1..J5."""
import numpy as np

from paper_2602_12949_b200 import inputs as I


def _rand(shape, seed, lo=0.0, hi=1.0):
    n = int(np.prod(shape))
    return (lo + (hi - lo) * I.uniform01(seed, 0x6000, n)).astype(np.float32).reshape(shape)


def _unit(shape, seed):
    v = I.normals_uniform(int(np.prod(shape[:-1])), seed)
    return v.reshape(shape).astype(np.float32)


def test_uniform_guides_reduce_to_the_bilinear_compose(oracle):
    """Every pixel and texel at the same position with the same normal: g_q is the same for all four neighbours, the
    weights are the bilinear ones, so the result is niv_oracle_compose's half-resolution path."""
    eh, ew = 9, 13
    h, w = 2 * eh, 2 * ew
    E, alb, dr, em = _rand((eh, ew, 3), 1, 0, 2), _rand((h, w, 3), 2), _rand((h, w, 3), 3), _rand((h, w, 3), 4)
    pos_h, pos_f = np.tile(np.float32([1, 2, 3]), (eh, ew, 1)), np.tile(np.float32([1, 2, 3]), (h, w, 1))
    nrm_h, nrm_f = np.tile(np.float32([0, 0, 1]), (eh, ew, 1)), np.tile(np.float32([0, 0, 1]), (h, w, 1))
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, 0.3, 8.0, dr, em)
    want = oracle.compose(E, alb, dr, em)
    assert np.abs(got - want).max() < 1e-12


def test_constant_irradiance_and_zero_albedo(oracle):
    eh, ew = 6, 8
    h, w = 12, 16
    pos_h, pos_f = _rand((eh, ew, 3), 5, 0, 4), _rand((h, w, 3), 6, 0, 4)
    nrm_h, nrm_f = _unit((eh, ew, 3), 7), _unit((h, w, 3), 8)
    alb, dr, em = _rand((h, w, 3), 9), _rand((h, w, 3), 10), _rand((h, w, 3), 11)
    E = np.tile(np.float32([0.5, 1.5, 2.5]), (eh, ew, 1))
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, 0.5, 4.0, dr, em)          # weights sum out
    want = alb.astype(np.float64) / np.pi * np.float64([0.5, 1.5, 2.5]) + dr + em
    assert np.abs(got - want).max() < 1e-12
    got0 = oracle.compose_jb(_rand((eh, ew, 3), 12), pos_h, nrm_h, pos_f, nrm_f, np.zeros_like(alb), 0.5, 4.0, dr, em)
    assert np.array_equal(got0, dr.astype(np.float64) + em.astype(np.float64))


def test_edges_stop_the_blend(oracle):
    """Two surfaces meeting at a vertical edge (left: normal +x, right: normal +y; E = 1 left, 3 right).  The plain
    bilinear upsample bleeds across the edge; with the normal term the other side's texels weigh <= 1e-6 of this side's."""
    eh, ew = 4, 8
    h, w = 8, 16
    nrm_h = np.zeros((eh, ew, 3), np.float32); nrm_h[:, :4, 0] = 1; nrm_h[:, 4:, 1] = 1
    nrm_f = np.zeros((h, w, 3), np.float32); nrm_f[:, :8, 0] = 1; nrm_f[:, 8:, 1] = 1
    E = np.zeros((eh, ew, 3), np.float32); E[:, :4] = 1.0; E[:, 4:] = 3.0
    pos_h, pos_f = np.zeros((eh, ew, 3), np.float32), np.zeros((h, w, 3), np.float32)
    alb = np.full((h, w, 3), np.pi, np.float32)                                            # albedo / pi = 1 (to fp32)
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, 1.0, 8.0) / (np.float64(np.float32(np.pi)) / np.pi)
    assert np.abs(got[:, :8] - 1.0).max() < 1e-5 and np.abs(got[:, 8:] - 3.0).max() < 1e-5
    bil = oracle.compose(E, alb) / (np.float64(np.float32(np.pi)) / np.pi)
    assert np.abs(bil[:, 7] - 1.0).max() > 0.2                                             # the bilinear one does bleed
    # the position term does the same for a depth discontinuity with equal normals
    nrm_h[:], nrm_f[:] = [0, 0, 1], [0, 0, 1]
    pos_h[:, 4:, 2], pos_f[:, 8:, 2] = 5.0, 5.0
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, 0.25, 0.0) / (np.float64(np.float32(np.pi)) / np.pi)
    assert np.abs(got[:, :8] - 1.0).max() < 1e-5 and np.abs(got[:, 8:] - 3.0).max() < 1e-5


def test_no_resembling_neighbour_falls_back_to_bilinear(oracle):
    """All four neighbours face away (n_p . n_q <= 0): g = 0 everywhere, the 1e-6 floor leaves the bilinear weights."""
    eh, ew = 5, 7
    h, w = 10, 14
    E, alb = _rand((eh, ew, 3), 20, 0, 2), _rand((h, w, 3), 21)
    nrm_h, nrm_f = np.tile(np.float32([0, 0, 1]), (eh, ew, 1)), np.tile(np.float32([0, 0, -1]), (h, w, 1))
    pos_h, pos_f = _rand((eh, ew, 3), 22), _rand((h, w, 3), 23)
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, 0.4, 2.0)
    assert np.abs(got - oracle.compose(E, alb)).max() < 1e-12


def test_numpy_restatement_on_random_guides(oracle):
    eh, ew = 5, 6
    h, w = 10, 12
    E, alb, dr = _rand((eh, ew, 3), 30, 0, 2), _rand((h, w, 3), 31), _rand((h, w, 3), 32)
    pos_h, pos_f = _rand((eh, ew, 3), 33, 0, 1), _rand((h, w, 3), 34, 0, 1)
    nrm_h, nrm_f = _unit((eh, ew, 3), 35), _unit((h, w, 3), 36)
    sigma, power = 0.6, 3.0
    got = oracle.compose_jb(E, pos_h, nrm_h, pos_f, nrm_f, alb, sigma, power, dr)
    want = np.zeros((h, w, 3))
    for y in range(h):
        for x in range(w):
            fx, fy = x / 2 - 0.25, y / 2 - 0.25
            x0, y0 = int(np.floor(fx)), int(np.floor(fy))
            num, den = np.zeros(3), 0.0
            for (qx, bx) in ((x0, 1 - (fx - x0)), (x0 + 1, fx - x0)):
                for (qy, by) in ((y0, 1 - (fy - y0)), (y0 + 1, fy - y0)):
                    cx, cy = min(max(qx, 0), ew - 1), min(max(qy, 0), eh - 1)
                    d = pos_f[y, x].astype(np.float64) - pos_h[cy, cx]
                    g = np.exp(-(d @ d) / (2 * sigma ** 2)) * max(0.0, float(nrm_f[y, x].astype(np.float64) @ nrm_h[cy, cx])) ** power
                    wq = bx * by * (g + 1e-6)
                    num += wq * E[cy, cx]
                    den += wq
            want[y, x] = alb[y, x].astype(np.float64) / np.pi * (num / den) + dr[y, x]
    assert np.abs(got - want).max() < 1e-12


def test_shape_errors(oracle):
    import pytest
    a = np.zeros((4, 4, 3), np.float32)
    b = np.zeros((8, 8, 3), np.float32)
    with pytest.raises(ValueError):
        oracle.compose_jb(b, b, b, b, b, b, 0.5, 1.0)             # E at full resolution
    with pytest.raises(ValueError):
        oracle.compose_jb(a, a, a, b, b, b, 0.0, 1.0)             # sigma must be positive
