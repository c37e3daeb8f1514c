"""Pins for the probe-grid oracle (oracle/niv_oracle_ext.c niv_oracle_probe_query): the paper's probe
baseline as PAPER.md:907-915 (App. A) lists it, checked against SPEC.md's examples, closed forms, scipy's spherical
harmonics and a numpy brute force written from the same four bullet points.  CPU only."""
import math

import numpy as np

from paper_2602_12949_b200 import inputs as I

BOX = ((-1.0, 0.5, 2.0), (3.0, 2.5, 4.0))


def _y9(n):
    """Real SH bands 0..2 from scipy's complex harmonics, in SPEC.md:341-345's convention: index l(l+1)+m, positive
    signs (no Condon-Shortley phase), band-1 order (y, z, x)."""
    from scipy.special import sph_harm_y
    x, y, z = n
    theta, phi = math.acos(max(-1.0, min(1.0, z / math.sqrt(x * x + y * y + z * z)))), math.atan2(y, x)
    out = []
    for l in range(3):
        for m in range(-l, l + 1):
            Y = sph_harm_y(l, abs(m), theta, phi)
            if m == 0:
                v = Y.real
            elif m > 0:
                v = math.sqrt(2.0) * (-1) ** m * Y.real
            else:
                v = math.sqrt(2.0) * (-1) ** m * Y.imag
            out.append(v)
    return np.array(out)


def _brute(dims, lo, hi, coeffs, x, n, falloff=True):
    """App. A's four bullet points in numpy fp64 (tent-function weights, scipy harmonics)."""
    dims = np.array(dims)
    lo, hi = np.array(lo, dtype=np.float64), np.array(hi, dtype=np.float64)
    xc = np.clip(np.asarray(x, dtype=np.float64), lo, hi)
    p = (xc - lo) / (hi - lo) * (dims - 1)
    c = coeffs.astype(np.float64).reshape(dims[2], dims[1], dims[0], 9, 3)
    Y = _y9(np.asarray(n, dtype=np.float64))
    # the 8 probes of the enclosing cell; their trilinear weights written as tent functions of the lattice distance
    cell = np.minimum(np.floor(p).astype(int), dims - 2)
    tot, acc = 0.0, np.zeros(3)
    for j in range(8):
        v = cell + np.array([(j >> d) & 1 for d in range(3)])
        w = np.prod(np.maximum(0.0, 1.0 - np.abs(p - v)))
        q = lo + v * (hi - lo) / (dims - 1)
        d = q - xc
        ln = np.linalg.norm(d)
        if falloff and ln > 0:
            w *= max(0.0, float(d @ np.asarray(n, dtype=np.float64)) / ln)
        w = max(w, 1e-6)
        tot += w
        acc += w * (Y @ c[v[2], v[1], v[0]])
    return acc / tot


def test_sh9_is_the_spec_basis(oracle):
    """Y00 = 0.282095, band-1 scale 0.488603 in order (y, z, x), band-2 scales 1.092548 / 0.315392 /
    0.546274; and scipy's harmonics in that convention for random directions."""
    Y = oracle.sh16(np.array([0.0, 0.0, 1.0]))[:9]
    assert abs(Y[0] - 0.282095) < 5e-7
    assert np.allclose(Y[1:4], [0.0, 0.488603, 0.0], atol=5e-7)
    assert abs(Y[6] - 0.630783) < 1e-6                 # 0.315392 * (3 - 1)
    nrm = I.normals_uniform(50, 9).astype(np.float64)
    for n in nrm:
        n = n / np.linalg.norm(n)
        assert np.allclose(oracle.sh16(n)[:9], _y9(n), atol=1e-12)


def test_probe_query_on_a_probe_returns_that_probe(oracle):
    """x exactly at a probe position, heuristics off -> that probe's SH reconstruction at n; with the
    fall-off on the probe at x keeps its weight (reading P-d), the other seven hold the 1e-6 floor."""
    dims = (5, 3, 3)
    lo, hi = BOX
    c = I.make_probe_grid(dims, 4)
    nrm = I.normals_uniform(8, 2)
    for k, v in enumerate([(0, 0, 0), (4, 2, 2), (2, 1, 1), (1, 2, 0)]):
        x = np.array([[lo[d] + v[d] * (hi[d] - lo[d]) / (dims[d] - 1) for d in range(3)]], dtype=np.float32)
        n = nrm[k:k + 1]
        want = _y9(n[0].astype(np.float64)) @ c[v[2], v[1], v[0]].astype(np.float64)
        got = oracle.probe_query(dims, lo, hi, c, x, n, cosine_falloff=False)
        assert np.allclose(got[0], want, atol=3e-5)        # the other seven probes hold the 1e-6 floor (App. A)
        _, e64, w, pi = oracle.probe_query(dims, lo, hi, c, x, n, cosine_falloff=True, debug=True)
        me = v[0] + dims[0] * (v[1] + dims[1] * v[2])
        assert w[0][list(pi[0]).index(me)] > 1.0 - 1e-5
        assert np.allclose(e64[0], want, atol=2e-5)


def test_identical_probes_make_the_result_independent_of_x(oracle):
    """all probes hold identical coefficients -> the result does not depend on x (convex weights)."""
    dims = (4, 4, 3)
    lo, hi = BOX
    one = I.make_probe_grid((2, 2, 2), 8)[0, 0, 0]
    c = np.broadcast_to(one, (3, 4, 4, 9, 3)).copy()
    pos = I.positions_uniform(300, (lo, hi), 5)
    n = np.tile(I.normals_uniform(1, 6), (300, 1))
    for falloff in (False, True):
        got = oracle.probe_query(dims, lo, hi, c, pos, n, cosine_falloff=falloff)
        want = _y9(n[0].astype(np.float64)) @ one.astype(np.float64)
        assert np.abs(got - want[None, :]).max() < 2e-6


def test_probe_weights_are_positive_and_sum_to_one(oracle):
    """after clamping and renormalisation the weights are positive and sum to 1; every one at least the
    1e-6 floor over the largest possible sum (8)."""
    dims = (6, 4, 5)
    lo, hi = BOX
    c = I.make_probe_grid(dims, 1)
    pos = I.positions_uniform(2000, (lo, hi), 7)
    nrm = I.normals_uniform(2000, 8)
    _, _, w, pi = oracle.probe_query(dims, lo, hi, c, pos, nrm, debug=True)
    assert np.all(w >= 1e-6 / 8.0) and np.abs(w.sum(axis=1) - 1.0).max() < 1e-12
    assert pi.max() < dims[0] * dims[1] * dims[2]
    # probes behind the normal hold the floor only: their weight is at most 1e-6 / (sum >= 1e-6 * 8)
    d = np.array(dims)
    lo64, hi64 = np.array(lo), np.array(hi)
    for i in range(0, 2000, 97):
        for j in range(8):
            v = np.array([pi[i, j] % d[0], (pi[i, j] // d[0]) % d[1], pi[i, j] // (d[0] * d[1])])
            q = lo64 + v * (hi64 - lo64) / (d - 1)
            if (q - pos[i]) @ nrm[i] < -1e-6:
                assert w[i, j] <= 1e-6 / w[i].max() * 2 or w[i, j] < 1e-3


def test_probe_query_matches_numpy_brute_force(oracle):
    """The four bullet points of App. A written out in numpy on a 2x2x2 and a 4x3x5 grid, positions inside, on the
    faces and outside the box (clamped), fall-off on and off."""
    for dims, seed in (((2, 2, 2), 3), ((4, 3, 5), 4)):
        lo, hi = BOX
        c = I.make_probe_grid(dims, seed)
        pos = I.positions_uniform(60, ((lo[0] - 0.5, lo[1] - 0.5, lo[2] - 0.5), (hi[0] + 0.5, hi[1] + 0.5, hi[2] + 0.5)), seed)
        pos[0] = lo
        pos[1] = hi
        pos[2] = (lo[0], hi[1], 0.5 * (lo[2] + hi[2]))
        nrm = I.normals_uniform(60, seed + 1)
        for falloff in (False, True):
            got, e64, _, _ = oracle.probe_query(dims, lo, hi, c, pos, nrm, cosine_falloff=falloff, debug=True)
            for i in range(60):
                want = _brute(dims, lo, hi, c, pos[i], nrm[i], falloff)
                assert np.allclose(e64[i], want, rtol=0, atol=1e-5), (dims, falloff, i)    # (fp32 probe offsets, P-e)
            assert np.abs(got - e64).max() < 1e-6


def test_probe_query_masks_like_the_model(oracle):
    dims = (3, 3, 3)
    lo, hi = BOX
    c = I.make_probe_grid(dims, 2)
    pos = I.positions_uniform(4, (lo, hi), 1)
    nrm = I.normals_uniform(4, 1)
    nrm[1] = 0.0
    pos[2, 1] = np.nan
    nrm[3, 0] = np.inf
    got = oracle.probe_query(dims, lo, hi, c, pos, nrm)
    assert np.all(got[1:] == 0.0) and np.any(got[0] != 0.0)
