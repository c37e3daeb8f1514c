"""Pins for the CPU oracle (oracle/niv_oracle.c): each test checks the oracle against something
other than itself -- values fixed by the paper / SURVEY (tests/golden/), closed forms, invariants,
library routines (numpy float16, torch grid_sample, scipy sph_harm, numpy matmul) and brute force.
CPU only (-m "not gpu")."""
import dataclasses
import math
import os

import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_lines(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [ln.strip() for ln in f if ln.strip() and not ln.startswith("#")]


# ------------------------------------------------------------------ level table, D/H pattern
def test_level_tables_match_golden(oracle):
    for ln in _golden_lines("level_tables.txt"):
        head, vals = ln.split(":")
        toks = head.split()
        kv = dict(t.split("=") for t in toks[1:])
        spec = I.ModelSpec(int(kv["L"]), 2, int(kv.get("log2T", 17)), int(kv["N0"]), 1.5, *I.UNIT_AABB,
                           hidden_width=32, n_hidden_layers=1)
        N, dense = oracle.level_table(spec)
        if toks[0] == "N":
            assert list(N) == [int(v) for v in vals.split()]
            # exact integer form of floor(N0 * 1.5^l): (N0 * 3^l) >> l
            assert list(N) == [(spec.base_resolution * 3 ** l) >> l for l in range(spec.n_levels)]
        else:
            assert ["D" if d else "H" for d in dense] == vals.split()


def test_paper_grid_family_memory_matches_table1(oracle):
    """with F=4, b=sqrt(2), N0=16, T=2^17 and dense levels storing (N+1)^3 entries,
    grid + four-matrix width-64 fp16 MLP reproduces the memory column (pins the dense rule, reading #4)."""
    for ln in _golden_lines("paper_table1_memory.txt"):
        L, mb = int(ln.split()[0]), float(ln.split()[1])
        spec = I.ModelSpec(L, 4, 17, 16, math.sqrt(2.0), *I.UNIT_AABB, hidden_width=64, n_hidden_layers=3)
        N, dense = oracle.level_table(spec)
        assert list(N) == [16, 22, 32, 45, 64, 90, 128, 181][:L]
        entries = sum((int(n) + 1) ** 3 if d else spec.table_size for n, d in zip(N, dense))
        grid_bytes = entries * 4 * 2
        in_dim = 4 * L + 3                      # latents + raw direction
        mlp_bytes = (in_dim * 64 + 64 * 64 * 2 + 64 * 3) * 2
        assert abs((grid_bytes + mlp_bytes) / 1e6 - mb) / mb < 0.04


def test_compact_table_is_the_paper_memory_and_changes_nothing(oracle):
    """the compact table (dense levels with (N+1)^3 entries) is what Table 1's memory column counts
    (PAPER.md:386-389), and a model evaluated on the expanded compact table is the model, bit for bit."""
    for ln in _golden_lines("paper_table1_memory.txt"):
        L, mb = int(ln.split()[0]), float(ln.split()[1])
        spec = I.spec_paper(L, 64)
        mlp_bytes = ((4 * L + 3) * 64 + 64 * 64 * 2 + 64 * 3) * 2
        assert abs((oracle.compact_entries(spec) * 4 * 2 + mlp_bytes) / 1e6 - mb) / mb < 0.04
    spec = I.spec_tiny()                                                   # D D D D H H H H, N = 4 6 9 13 ...
    assert oracle.compact_entries(spec) == 5 ** 3 + 7 ** 3 + 10 ** 3 + 14 ** 3 + 4 * 4096
    table = I.make_table(spec, 3, -1.0, 1.0)
    comp = oracle.table_compact(spec, table)
    assert comp.size == oracle.compact_entries(spec) * 2
    back = oracle.table_expand(spec, comp)
    N, dense = oracle.level_table(spec)
    for l in range(spec.n_levels):
        cnt = (int(N[l]) + 1) ** 3 if dense[l] else spec.table_size
        assert np.array_equal(back[l, :cnt], table.reshape(spec.n_levels, spec.table_size, 2)[l, :cnt])
        assert np.all(back[l, cnt:] == 0)
    assert np.array_equal(comp[:5 ** 3 * 2].view(np.uint16), table.reshape(-1)[:5 ** 3 * 2].view(np.uint16))   # level 0 first
    w, b = I.make_mlp(spec, 3)
    wb, bb = I.pack_weights(w), I.pack_biases(b)
    pos, nrm = I.positions_uniform(3000, (spec.aabb_min, spec.aabb_max), 1), I.normals_uniform(3000, 2)
    assert np.array_equal(oracle.infer(spec, back, wb, bb, pos, nrm), oracle.infer(spec, table, wb, bb, pos, nrm))


def test_explicit_resolutions_override(oracle):
    spec = dataclasses.replace(I.spec_tiny(), resolutions=(5, 7, 11, 13, 17, 19, 23, 29))
    N, _ = oracle.level_table(spec)
    assert list(N) == [5, 7, 11, 13, 17, 19, 23, 29]


# ------------------------------------------------------------------ hash
def test_hash_worked_values(oracle):
    for ln in _golden_lines("hash_values.txt"):
        vx, vy, vz, h12, h17, h18 = (int(t) for t in ln.split())
        assert oracle.hash_index(vx, vy, vz, 12) == h12
        assert oracle.hash_index(vx, vy, vz, 17) == h17
        assert oracle.hash_index(vx, vy, vz, 18) == h18


def test_hash_x_neighbour_property(oracle):
    """The x prime is 1, so for even vx the two x-corners differ only in bit 0."""
    rng = np.random.default_rng(0)
    for vx, vy, vz in rng.integers(0, 7007, size=(200, 3)):
        a = oracle.hash_index(int(vx), int(vy), int(vz), 17)
        b = oracle.hash_index(int(vx) ^ 1, int(vy), int(vz), 17)
        assert a ^ b == 1


def test_hash_matches_bigint_formula(oracle):
    rng = np.random.default_rng(1)
    for vx, vy, vz in rng.integers(0, 2 ** 31, size=(200, 3)):
        vx, vy, vz = int(vx), int(vy), int(vz)
        ref = ((vx & 0xFFFFFFFF) ^ ((vy * 2654435761) & 0xFFFFFFFF) ^ ((vz * 805459861) & 0xFFFFFFFF)) % (1 << 18)
        assert oracle.hash_index(vx, vy, vz, 18) == ref


# ------------------------------------------------------------------ fp16 decode (library routine: numpy)
def test_half_to_double_all_bit_patterns(oracle):
    bits = np.arange(65536, dtype=np.uint16)
    ref = bits.view(np.float16).astype(np.float64)
    got = np.array([oracle.half_to_double(int(b)) for b in bits])
    fin = np.isfinite(ref)
    assert np.array_equal(got[fin], ref[fin])
    assert np.array_equal(np.isnan(got), np.isnan(ref))
    assert np.array_equal(np.isinf(got), np.isinf(ref))
    assert np.array_equal(np.signbit(got[fin]), np.signbit(ref[fin]))     # -0 kept


# ------------------------------------------------------------------ locate / weights / blend
def _up(n):
    return np.tile(np.array([[0.0, 0.0, 1.0]], dtype=np.float32), (n, 1))


def test_vertex_query_returns_vertex_entry(oracle):
    """north_star: 'a query exactly on a grid vertex returns that vertex's table entry'.
    Vertices whose fp32 round trip fl(fl(k/N)*N) != k are filtered."""
    spec = I.spec_tiny()
    table = I.make_table(spec, 3, -1.0, 1.0)
    N, dense = oracle.level_table(spec)
    rng = np.random.default_rng(2)
    checked = 0
    for l in range(spec.n_levels):
        n = int(N[l])
        ks = rng.integers(0, n + 1, size=(64, 3))
        u = (ks.astype(np.float32) / np.float32(n)).astype(np.float32)
        ok = np.all((u * np.float32(n)).astype(np.float32) == ks.astype(np.float32), axis=1)
        ks, u = ks[ok], u[ok]
        out = oracle.encode(spec, table, u, _up(len(u)))
        for q, k in enumerate(ks):
            if dense[l]:
                R = n + 1
                e = int(k[0]) + R * (int(k[1]) + R * int(k[2]))
            else:
                e = ((int(k[0]) ^ (int(k[1]) * 2654435761) ^ (int(k[2]) * 805459861)) & 0xFFFFFFFF) % spec.table_size
            want = table[l, e].astype(np.float64)
            assert np.array_equal(out["features"][q, l * 2:l * 2 + 2], want)
            checked += 1
    assert checked > 300


def test_voxel_centre_is_mean_of_corners(oracle):
    """SPEC.md:228.  Power-of-two resolutions make the centre exactly representable."""
    spec = dataclasses.replace(I.spec_tiny(), resolutions=(4, 8, 16, 32, 64, 128, 256, 512))
    table = I.make_table(spec, 4, -1.0, 1.0)
    N, _ = oracle.level_table(spec)
    rng = np.random.default_rng(3)
    for l in range(spec.n_levels):
        n = int(N[l])
        c = rng.integers(0, n, size=(16, 3))
        u = ((c + 0.5) / n).astype(np.float32)
        out = oracle.encode(spec, table, u, _up(16))
        assert np.array_equal(out["cell"][:, l, :], c)
        assert np.all(out["frac"][:, l, :] == 0.5)
        vals = table[l][out["idx"][:, l, :]].astype(np.float64)        # [16][8][F]
        np.testing.assert_allclose(out["features"][:, 2 * l:2 * l + 2], vals.mean(axis=1), rtol=0, atol=1e-15)


def test_zero_table_gives_zero_latents(oracle):
    spec = I.spec_tiny()
    table = np.zeros((spec.n_levels, spec.table_size, 2), dtype=np.float16)
    out = oracle.encode(spec, table, I.positions_uniform(256, I.UNIT_AABB, 0), I.normals_uniform(256, 0))
    assert np.all(out["features"][:, :16] == 0)


def test_weights_partition_of_unity_and_ranges(oracle):
    """Interpolation weights sum to 1 (north_star): a per-level constant table gives that constant for
    every x, dense or hashed; cells / fractions stay in range including u = 0, u = 1 and outside."""
    spec = I.spec_tiny()
    consts = np.linspace(-0.75, 0.75, spec.n_levels * 2).astype(np.float16).reshape(spec.n_levels, 1, 2)
    table = np.broadcast_to(consts, (spec.n_levels, spec.table_size, 2)).copy()
    pos = I.positions_uniform(2048, I.UNIT_AABB, 5)
    pos[:64] = np.round(pos[:64])                     # exact corners of the AABB: u in {0,1}
    pos[64:128] = pos[64:128] * 3.0 - 1.0             # some outside the AABB -> clamped
    out = oracle.encode(spec, table, pos, _up(len(pos)))
    want = consts.astype(np.float64).reshape(-1)
    np.testing.assert_allclose(out["features"][:, :16], np.broadcast_to(want, (len(pos), 16)), rtol=0, atol=4e-16)
    N, _ = oracle.level_table(spec)
    for l in range(spec.n_levels):
        assert out["cell"][:, l].min() >= 0 and out["cell"][:, l].max() <= int(N[l]) - 1
        assert out["frac"][:, l].min() >= 0.0 and out["frac"][:, l].max() <= 1.0
    # u = 1 lands in the last cell with weight exactly 1 (reading #6)
    one = np.ones((1, 3), dtype=np.float32)
    o1 = oracle.encode(spec, table, one, _up(1))
    for l in range(spec.n_levels):
        assert list(o1["cell"][0, l]) == [int(N[l]) - 1] * 3 and list(o1["frac"][0, l]) == [1.0] * 3


def test_out_of_aabb_is_clamped(oracle):
    """Reading #7: positions outside the AABB behave like their clamped position."""
    spec = I.spec_fullhd()
    table = I.make_table(spec, 6)
    pos = I.positions_uniform(128, I.ROOM_AABB, 7)
    far = pos.copy()
    far[:, 0] += 25.0
    far[:, 1] -= 9.0
    clamped = pos.copy()
    clamped[:, 0] = 10.0
    clamped[:, 1] = 0.0
    a = oracle.encode(spec, table, far, _up(128))
    b = oracle.encode(spec, table, clamped, _up(128))
    assert np.array_equal(a["idx"], b["idx"]) and np.array_equal(a["frac"], b["frac"])


def test_dense_levels_reproduce_affine_functions(oracle):
    """Trilinear interpolation on a vertex-aligned lattice reproduces a*px+b*py+c*pz+d exactly;
    pins the dense index order (x fastest) and the corner/weight pairing."""
    spec = I.spec_tiny()
    N, dense = oracle.level_table(spec)
    table = np.zeros((spec.n_levels, spec.table_size, 2), dtype=np.float16)
    coef = (1.0, 8.0, 64.0)          # distinct per axis, exactly representable in fp16 products below
    for l in range(spec.n_levels):
        if not dense[l]:
            continue
        R = int(N[l]) + 1
        v = np.arange(R)
        vz, vy, vx = np.meshgrid(v, v, v, indexing="ij")
        f0 = (coef[0] * vx + coef[1] * vy + coef[2] * vz).reshape(-1) / 64.0
        f1 = (coef[2] * vx + coef[0] * vy + coef[1] * vz).reshape(-1) / 64.0
        assert np.array_equal(f0.astype(np.float16).astype(np.float64), f0)
        table[l, :R ** 3, 0] = f0
        table[l, :R ** 3, 1] = f1
    pos = I.positions_uniform(512, I.UNIT_AABB, 8)
    out = oracle.encode(spec, table, pos, _up(512))
    for l in range(spec.n_levels):
        if not dense[l]:
            continue
        p = out["cell"][:, l].astype(np.float64) + out["frac"][:, l].astype(np.float64)
        w0 = (coef[0] * p[:, 0] + coef[1] * p[:, 1] + coef[2] * p[:, 2]) / 64.0
        w1 = (coef[2] * p[:, 0] + coef[0] * p[:, 1] + coef[1] * p[:, 2]) / 64.0
        np.testing.assert_allclose(out["features"][:, 2 * l], w0, rtol=0, atol=1e-12)
        np.testing.assert_allclose(out["features"][:, 2 * l + 1], w1, rtol=0, atol=1e-12)


def test_dense_levels_equal_torch_grid_sample(oracle):
    """Library routine: grid_sample(bilinear, align_corners=True, border) on CPU in fp64 is vertex-aligned
    trilinear interpolation."""
    torch = pytest.importorskip("torch")
    spec = I.spec_tiny()
    table = I.make_table(spec, 9, -1.0, 1.0)
    N, dense = oracle.level_table(spec)
    pos = I.positions_uniform(1024, I.UNIT_AABB, 10)
    pos[:8] = np.round(pos[:8])
    out = oracle.encode(spec, table, pos, _up(len(pos)))
    for l in range(spec.n_levels):
        if not dense[l]:
            continue
        R = int(N[l]) + 1
        vol = torch.from_numpy(table[l, :R ** 3].astype(np.float64)).reshape(R, R, R, 2).permute(3, 0, 1, 2)[None]
        # sample at the oracle's own fp32 lattice coordinate p = cell + frac, mapped to [-1,1]
        p = out["cell"][:, l].astype(np.float64) + out["frac"][:, l].astype(np.float64)
        g = torch.from_numpy(2.0 * p / float(N[l]) - 1.0).reshape(1, -1, 1, 1, 3)
        ref = torch.nn.functional.grid_sample(vol, g, mode="bilinear", padding_mode="border", align_corners=True)
        ref = ref.reshape(2, -1).T.numpy()
        np.testing.assert_allclose(out["features"][:, 2 * l:2 * l + 2], ref, rtol=0, atol=2e-14)


def _hash_py(vx, vy, vz, T):
    return ((vx & 0xFFFFFFFF) ^ ((vy * 2654435761) & 0xFFFFFFFF) ^ ((vz * 805459861) & 0xFFFFFFFF)) % T


def _brute_force_latents(spec, N, dense, table, u):
    """Tent-function definition: f = sum over ALL lattice vertices v of table[index(v)] * prod_d max(0,
    1-|p_d-v_d|), no corner selection, separately coded index/hash (north_star: brute-force enumeration)."""
    T = spec.table_size
    tab = table.astype(np.float64)
    F = spec.n_features
    feats = np.zeros((len(u), spec.n_levels * F))
    for l in range(spec.n_levels):
        n = int(N[l])
        R = n + 1
        v = np.arange(R)
        vz, vy, vx = np.meshgrid(v, v, v, indexing="ij")
        vx, vy, vz = vx.reshape(-1), vy.reshape(-1), vz.reshape(-1)
        if dense[l]:
            e = vx + R * (vy + R * vz)
        else:
            e = np.array([_hash_py(int(a), int(b), int(c), T) for a, b, c in zip(vx, vy, vz)])
        vals = tab[l][e]
        for q in range(len(u)):
            p = (u[q].astype(np.float32) * np.float32(n)).astype(np.float64)     # fp32 product, as in O2
            wx = np.maximum(0.0, 1.0 - np.abs(p[0] - vx))
            wy = np.maximum(0.0, 1.0 - np.abs(p[1] - vy))
            wz = np.maximum(0.0, 1.0 - np.abs(p[2] - vz))
            feats[q, F * l:F * l + F] = ((wx * wy * wz)[:, None] * vals).sum(axis=0)
    return feats


def test_brute_force_enumeration_4x4(oracle):
    """north_star: 'brute-force enumeration matches on 4x4 inputs' -- a 4x4 G-buffer (16 texels) through the
    whole path: tent-sum latents over every lattice vertex (dense and hashed levels), textbook SH via
    scipy, numpy fp64 matmul chain, sigmoid."""
    spec = I.spec_tiny()
    table = I.make_table(spec, 0, -1.0, 1.0)
    weights, biases = I.make_mlp(spec, 0, bias_scale=0.1)
    N, dense = oracle.level_table(spec)
    pos = I.positions_uniform(16, I.UNIT_AABB, 0)
    nrm = I.normals_uniform(16, 0)
    lat = _brute_force_latents(spec, N, dense, table, pos)
    enc = oracle.encode(spec, table, pos, nrm)
    np.testing.assert_allclose(enc["features"][:, :16], lat, rtol=0, atol=1e-13)
    x = np.concatenate([lat, np.stack([_sh16_scipy(n) for n in nrm.astype(np.float64)])], axis=1)
    h = x
    for k, (w, b) in enumerate(zip(weights, biases)):
        h = h @ w.astype(np.float64).T + b.astype(np.float64)
        if k + 1 < len(weights):
            h = np.maximum(h, 0.0)
    ref = 1.0 / (1.0 + np.exp(-h))
    out32, out64 = oracle.infer(spec, table, I.pack_weights(weights), I.pack_biases(biases), pos, nrm, want_f64=True)
    # fp32 normals are unit only to ~6e-8 and are used as given (reading #13) while the textbook routine
    # sees the direction only: hence 2e-7 here; test_sh16_matches_scipy holds 5e-15 on exactly-unit input
    np.testing.assert_allclose(out64, ref, rtol=0, atol=2e-7)
    assert np.array_equal(out32, out64.astype(np.float32))


def test_paper_family_brute_force_4x4(oracle):
    """The paper's own model family: latent dimension 4, scale sqrt(2), coarsest
    side 16, position + RAW direction in, four weight matrices, no output activation -- a 4x4 G-buffer through the
    whole path against the tent-sum over every lattice vertex and a numpy matmul chain.  T = 2^14 so that levels
    2..3 are hashed and the enumeration stays small."""
    spec = dataclasses.replace(I.spec_paper(4, 32), log2_table_size=14, aabb_min=I.UNIT_AABB[0], aabb_max=I.UNIT_AABB[1])
    assert spec.in_dim == 4 * 4 + 3 and spec.layer_shapes == [(32, 19), (32, 32), (32, 32), (3, 32)]
    table = I.make_table(spec, 3, -1.0, 1.0)
    weights, biases = I.make_mlp(spec, 3, bias_scale=0.1)
    N, dense = oracle.level_table(spec)
    assert list(N) == [16, 22, 32, 45] and list(dense) == [True, True, False, False]
    pos = I.positions_uniform(16, I.UNIT_AABB, 5)
    nrm = I.normals_uniform(16, 5)
    lat = _brute_force_latents(spec, N, dense, table, pos)
    enc = oracle.encode(spec, table, pos, nrm)
    np.testing.assert_allclose(enc["features"][:, :16], lat, rtol=0, atol=1e-13)
    assert np.array_equal(enc["features"][:, 16:19], nrm.astype(np.float64))          # the direction as given
    h = np.concatenate([lat, nrm.astype(np.float64)], axis=1)
    for k, (w, b) in enumerate(zip(weights, biases)):
        h = h @ w.astype(np.float64).T + b.astype(np.float64)
        if k + 1 < len(weights):
            h = np.maximum(h, 0.0)
    out32, out64 = oracle.infer(spec, table, I.pack_weights(weights), I.pack_biases(biases), pos, nrm, want_f64=True)
    np.testing.assert_allclose(out64, h, rtol=0, atol=1e-12)                            # linear output
    assert np.array_equal(out32, out64.astype(np.float32))


def test_paper_family_vertex_and_partition_of_unity(oracle):
    """F = 4: a query on a lattice vertex returns that vertex's four latents; a per-level constant table gives
    that constant for any position (dense and hashed levels of the full 8-level paper grid)."""
    spec = dataclasses.replace(I.spec_paper(8, 64), aabb_min=I.UNIT_AABB[0], aabb_max=I.UNIT_AABB[1])
    N, dense = oracle.level_table(spec)
    assert list(N) == list(I.PAPER_RESOLUTIONS) and list(dense) == [True] * 4 + [False] * 4
    table = I.make_table(spec, 7, -1.0, 1.0)
    nrm = I.normals_uniform(8, 1)
    for l in (0, 2, 4, 6):                    # power-of-two resolutions: k/N and (k/N)*N are exact in fp32
        n = int(N[l])
        k = np.array([[1, 2, 3], [n, n, n], [0, n // 2, n - 1], [5, 0, 7]], dtype=np.int64)
        pos = (k / float(n)).astype(np.float32)
        enc = oracle.encode(spec, table, pos, nrm[:4])
        for q in range(4):
            vx, vy, vz = (int(v) for v in k[q])
            e = vx + (n + 1) * (vy + (n + 1) * vz) if dense[l] else _hash_py(vx, vy, vz, spec.table_size)
            np.testing.assert_allclose(enc["features"][q, 4 * l:4 * l + 4], table[l][e].astype(np.float64), atol=1e-15)
    const = np.zeros_like(table)
    for l in range(8):
        const[l, :, :] = np.float16(0.125 * (l + 1))
    pos = I.positions_uniform(64, I.UNIT_AABB, 9)
    enc = oracle.encode(spec, const, pos, I.normals_uniform(64, 9))
    want = np.repeat(0.125 * (np.arange(8) + 1), 4)
    np.testing.assert_allclose(enc["features"][:, :32], np.broadcast_to(want, (64, 32)), atol=1e-14)


def test_paper_gridless_models_brute_force_4x4(oracle):
    """Table 1 rows without a grid: eight-band positional encoding of the position,
    raw direction, four matrices.  SPEC.md:216-219 examples pin the band order; the whole path is checked against
    numpy on a 4x4 G-buffer; the memory column of Table 1 (0.003 / 0.01 / 0.03 MB) is consistent with the input width
    48 + 3 to one unit of its last printed digit (a weak pin: the column has one significant digit)."""
    for width, mb in ((16, 0.003), (32, 0.01), (64, 0.03)):
        spec = I.spec_paper_pe(width)
        assert spec.in_dim == 51
        n_par = sum(o * i for o, i in spec.layer_shapes)
        assert abs(n_par * 2 / 1e6 - mb) <= 10 ** (-3 if mb < 0.005 else -2)     # one unit of the last printed digit
    spec = dataclasses.replace(I.spec_paper_pe(32), aabb_min=(-1.0, 0.0, 2.0), aabb_max=(3.0, 2.0, 4.0))
    weights, biases = I.make_mlp(spec, 4, bias_scale=0.1)
    table = I.make_table(spec, 0)
    assert table.size == 0
    pos = I.positions_uniform(16, (spec.aabb_min, spec.aabb_max), 6)
    nrm = I.normals_uniform(16, 6)
    enc = oracle.encode(spec, table, pos, nrm)["features"]
    ext = np.float32(spec.aabb_max) - np.float32(spec.aabb_min)
    u = ((pos - np.float32(spec.aabb_min)) * (np.float32(1.0) / ext)).astype(np.float32).astype(np.float64)
    k = 2.0 ** np.arange(8)
    want = np.empty((16, 48))
    for d in range(3):
        want[:, 16 * d:16 * d + 16:2] = np.sin(np.pi * u[:, d:d + 1] * k)
        want[:, 16 * d + 1:16 * d + 16:2] = np.cos(np.pi * u[:, d:d + 1] * k)
    np.testing.assert_allclose(enc[:, :48], want, atol=1e-12)
    assert np.array_equal(enc[:, 48:51], nrm.astype(np.float64))
    # SPEC.md:217-218 on the position path: u = 0 -> (0, 1) pairs; u = 0.5 -> first band (1, 0)
    e0 = oracle.encode(spec, table, np.float32([[-1.0, 1.0, 2.0]]), nrm[:1])["features"][0]
    np.testing.assert_allclose(e0[0:16], np.tile([0.0, 1.0], 8), atol=1e-15)
    np.testing.assert_allclose(e0[16:18], [1.0, 0.0], atol=1e-15)
    h = np.concatenate([want, nrm.astype(np.float64)], axis=1)
    for j, (w, b) in enumerate(zip(weights, biases)):
        h = h @ w.astype(np.float64).T + b.astype(np.float64)
        if j + 1 < len(weights):
            h = np.maximum(h, 0.0)
    out32, out64 = oracle.infer(spec, table, I.pack_weights(weights), I.pack_biases(biases), pos, nrm, want_f64=True)
    np.testing.assert_allclose(out64, h, rtol=0, atol=1e-11)


def test_direction_frequency_encoding(oracle):
    """SPEC.md:198 "directionEncoding: raw 3-vector (plus optional frequency)" with freq_encode of SPEC.md:211-219 per
    axis (reading 3.8): [n | s(n_x) | s(n_y) | s(n_z)], s(p) = (sin, cos)(2^k pi p), k < B.  Pins: the SPEC
    examples on the direction path (n_d = 0 -> (0, 1) pairs; n_d = 0.5 -> first band (1, 0); n_d = -0.5 -> (-1, 0): the
    input range is [-1, 1], sin is odd), numpy for the whole feature block, B = 0 reduces to the raw model bit for bit,
    one-hot first-layer weights read single features out through the MLP, and the whole path against a numpy chain."""
    B = 4
    spec = I.spec_paper_dirfreq(2, 32, B)
    raw = I.spec_paper(2, 32)
    assert spec.dir_dim == 3 + 6 * B and spec.in_dim == raw.in_dim + 6 * B == 8 + 27
    table = I.make_table(spec, 3, -1.0, 1.0)
    pos = I.positions_uniform(40, (spec.aabb_min, spec.aabb_max), 2)
    nrm = I.normals_uniform(40, 2)
    nrm[0] = (0.0, 0.5, -0.5)                      # not unit: the encoding is defined on the values as given
    nrm[1] = (1.0, 0.0, 0.0)
    enc = oracle.encode(spec, table, pos, nrm)["features"]
    enc_raw = oracle.encode(raw, table, pos, nrm)["features"]
    assert np.array_equal(enc[:, :11], enc_raw)                     # latents and the raw vector are untouched
    d0 = enc[0, 11:]
    np.testing.assert_allclose(d0[0:2 * B], np.tile([0.0, 1.0], B), atol=1e-15)              # n_x = 0
    np.testing.assert_allclose(d0[2 * B:2 * B + 2], [1.0, 0.0], atol=1e-15)                  # n_y = 0.5, band 0
    np.testing.assert_allclose(d0[4 * B:4 * B + 2], [-1.0, 0.0], atol=1e-15)                 # n_z = -0.5, band 0
    np.testing.assert_allclose(enc[1, 11:13], [0.0, -1.0], atol=2e-16)                       # n_x = 1: (sin pi, cos pi)
    k = 2.0 ** np.arange(B)
    want = np.empty((40, 6 * B))
    n64 = nrm.astype(np.float64)
    for d in range(3):
        want[:, 2 * B * d:2 * B * (d + 1):2] = np.sin(np.pi * n64[:, d:d + 1] * k)
        want[:, 2 * B * d + 1:2 * B * (d + 1):2] = np.cos(np.pi * n64[:, d:d + 1] * k)
    np.testing.assert_allclose(enc[:, 11:], want, atol=1e-12)
    # dir_frequencies = 0 is the raw model
    zero = dataclasses.replace(spec, dir_frequencies=0)
    assert zero.in_dim == raw.in_dim and np.array_equal(oracle.encode(zero, table, pos, nrm)["features"], enc_raw)
    # through the MLP: a one-layer-deep probe of single input columns (hidden unit j = +feature c, unit j+1 = -feature c)
    one = dataclasses.replace(spec, n_hidden_layers=1)
    for c in (8, 10, 11, 12, 11 + 2 * B, 11 + 6 * B - 1):
        w1 = np.zeros((32, one.in_dim), np.float16)
        w1[0, c], w1[1, c] = 1.0, -1.0
        w2 = np.zeros((3, 32), np.float16)
        w2[0, 0], w2[0, 1] = 1.0, -1.0                               # relu(f) - relu(-f) = f
        out32, out64 = oracle.infer(one, table, I.pack_weights([w1, w2]), None, pos, nrm, want_f64=True)
        np.testing.assert_allclose(out64[:, 0], enc[:, c], atol=1e-15)
    weights, biases = I.make_mlp(spec, 4, bias_scale=0.1)
    h = enc.copy()
    for j, (w, b) in enumerate(zip(weights, biases)):
        h = h @ w.astype(np.float64).T + b.astype(np.float64)
        if j + 1 < len(weights):
            h = np.maximum(h, 0.0)
    out32, out64 = oracle.infer(spec, table, I.pack_weights(weights), I.pack_biases(biases), pos, nrm, want_f64=True)
    np.testing.assert_allclose(out64, h, rtol=0, atol=1e-11)


# ------------------------------------------------------------------ SH-16
def _sh16_scipy(n):
    """Real orthonormal SH, bands 0..3, index l(l+1)+m, no Condon-Shortley sign, from scipy's complex Y_l^m."""
    sp = pytest.importorskip("scipy.special")
    x, y, z = n
    r = math.sqrt(x * x + y * y + z * z)
    theta = math.acos(max(-1.0, min(1.0, z / r)))      # polar
    phi = math.atan2(y, x)                             # azimuth
    out = np.zeros(16)
    for l in range(4):
        for m in range(-l, l + 1):
            if hasattr(sp, "sph_harm_y"):
                Y = sp.sph_harm_y(l, abs(m), theta, phi)
            else:
                Y = sp.sph_harm(abs(m), l, phi, theta)
            if m == 0:
                v = Y.real
            elif m > 0:
                v = math.sqrt(2.0) * (-1) ** m * Y.real
            else:
                v = math.sqrt(2.0) * (-1) ** m * Y.imag
            out[l * (l + 1) + m] = v
    return out


def test_sh16_matches_scipy(oracle):
    nrm = I.normals_uniform(200, 11).astype(np.float64)
    for n in nrm:
        n = n / np.linalg.norm(n)
        np.testing.assert_allclose(oracle.sh16(n), _sh16_scipy(n), rtol=0, atol=5e-15)


def test_sh16_golden_constants_and_zonal_values(oracle):
    g = {ln.split()[0]: [float(v) for v in ln.split()[1:]] for ln in _golden_lines("sh_values.txt")}
    z = oracle.sh16([0.0, 0.0, 1.0])
    assert abs(z[0] - g["Y00"][0]) < 5e-7
    for l, want in enumerate(g["zonal_at_plus_z"]):
        assert abs(z[l * (l + 1)] - want) < 5e-7
    nz = [i for i in range(16) if i not in (0, 2, 6, 12)]
    assert np.all(z[nz] == 0.0)
    # band-1 order (y, z, x) with positive signs
    assert abs(oracle.sh16([1, 0, 0])[3] - g["band1"][0]) < 5e-7
    assert abs(oracle.sh16([0, 1, 0])[1] - g["band1"][0]) < 5e-7
    s = 1.0 / math.sqrt(2.0)
    assert abs(oracle.sh16([s, s, 0])[4] - g["band2"][0] * 0.5) < 5e-7       # c2a*x*y
    assert abs(oracle.sh16([0, 0, 1])[6] - g["band2"][1] * 2.0) < 1e-6       # c2b*(3z^2-1)
    assert abs(oracle.sh16([1, 0, 0])[8] - g["band2"][2]) < 5e-7             # c2c*(x^2-y^2)


def test_sh16_addition_theorem(oracle):
    """sum_m Y_lm^2 = (2l+1)/(4 pi) per band and sum over 16 = 4/pi for every unit n."""
    for n in I.normals_uniform(200, 12).astype(np.float64):
        n = n / np.linalg.norm(n)
        y = oracle.sh16(n)
        for l in range(4):
            assert abs(np.sum(y[l * l:(l + 1) ** 2] ** 2) - (2 * l + 1) / (4 * math.pi)) < 1e-14
        assert abs(np.sum(y * y) - 4.0 / math.pi) < 1e-14


def test_sh16_orthonormal_by_quadrature(oracle):
    """Gauss-Legendre in cos(theta) x uniform phi integrates degree-6 polynomials exactly."""
    xs, ws = np.polynomial.legendre.leggauss(8)
    nphi = 16
    G = np.zeros((16, 16))
    for ct, w in zip(xs, ws):
        st = math.sqrt(1 - ct * ct)
        for k in range(nphi):
            ph = 2 * math.pi * (k + 0.5) / nphi
            y = oracle.sh16([st * math.cos(ph), st * math.sin(ph), ct])
            G += w * (2 * math.pi / nphi) * np.outer(y, y)
    np.testing.assert_allclose(G, np.eye(16), rtol=0, atol=1e-13)


# ------------------------------------------------------------------ parameter encoding
def test_param_encode_examples(oracle):
    """p=0,B=2 -> [0,1,0,1]; p=0.5,B=1 -> [1,0]; order sin,cos per band, argument 2^k pi p."""
    np.testing.assert_allclose(oracle.param_encode(0.0, 2), [0, 1, 0, 1], atol=0)
    np.testing.assert_allclose(oracle.param_encode(0.5, 1), [1, 0], atol=1e-16)
    e = oracle.param_encode(0.3, 8)
    assert len(e) == 16
    np.testing.assert_allclose(e[0::2] ** 2 + e[1::2] ** 2, np.ones(8), atol=1e-15)
    np.testing.assert_allclose(e[:4], [math.sin(0.3 * math.pi), math.cos(0.3 * math.pi),
                                       math.sin(0.6 * math.pi), math.cos(0.6 * math.pi)], atol=1e-15)
    # t = 0.25: band k=2 has argument pi -> (sin, cos) = (0, -1)
    np.testing.assert_allclose(oracle.param_encode(0.25, 3)[4:6], [0.0, -1.0], atol=2e-16)


# ------------------------------------------------------------------ MLP
def _blob(ws):
    return np.concatenate([np.asarray(w, dtype=np.float16).reshape(-1) for w in ws])


def test_mlp_zero_weights_give_activation_of_bias(oracle):
    spec = I.spec_tiny()
    ws = [np.zeros(s) for s in spec.layer_shapes]
    b = np.concatenate([np.zeros(32), [0.25, -1.0, 2.0]]).astype(np.float32)
    x = np.linspace(-1, 1, 32)
    np.testing.assert_array_equal(oracle.mlp(spec, _blob(ws), b, x), [0.25, -1.0, 2.0])
    table = I.make_table(spec, 0)
    pos, nrm = I.positions_uniform(8, I.UNIT_AABB, 1), I.normals_uniform(8, 1)
    out = oracle.infer(spec, table, _blob(ws), None, pos, nrm)
    assert np.all(out == np.float32(0.5))                                  # sigmoid(0)
    lin = dataclasses.replace(spec, out_activation=I.OUT_LINEAR)
    assert np.all(oracle.infer(lin, table, _blob(ws), None, pos, nrm) == 0.0)


def test_mlp_identity_and_sign_split(oracle):
    """W1 = I (32x32), W2 selects rows 0..2 -> out = ReLU(x_0..2); [I;-I] then [I,-I] passes signed inputs
    through the ReLU exactly."""
    spec = dataclasses.replace(I.spec_tiny(), out_activation=I.OUT_LINEAR)
    x = np.linspace(-1.0, 1.0, 32)
    x[:3] = [-0.5, 0.25, 0.75]
    w1 = np.eye(32)
    w2 = np.zeros((3, 32))
    w2[[0, 1, 2], [0, 1, 2]] = 1.0
    np.testing.assert_array_equal(oracle.mlp(spec, _blob([w1, w2]), None, x), [0.0, 0.25, 0.75])
    # sign split on the first 16 inputs: hidden = [x_0..15 ; -x_0..15], out_c = h_c - h_{16+c} = x_c
    w1 = np.zeros((32, 32))
    w1[:16, :16] = np.eye(16)
    w1[16:, :16] = -np.eye(16)
    w2 = np.zeros((3, 32))
    for c in range(3):
        w2[c, c], w2[c, 16 + c] = 1.0, -1.0
    np.testing.assert_array_equal(oracle.mlp(spec, _blob([w1, w2]), None, x), x[:3])


def test_mlp_matches_numpy_matmul_chain(oracle):
    """Library routine: fp64 X @ W.T chain on every BASELINE MLP shape; also pins layer
    order, [out][in] orientation and where ReLU is (not) applied."""
    rng = np.random.default_rng(4)
    for spec in (I.spec_tiny(), I.spec_fullhd(), I.spec_param(), I.spec_fullhd(width=128), I.spec_fullhd(width=32),
                 dataclasses.replace(I.spec_fullhd(), n_hidden_layers=3, out_activation=I.OUT_LINEAR)):
        weights, biases = I.make_mlp(spec, 5, bias_scale=0.2)
        for _ in range(4):
            x = rng.uniform(-1, 1, spec.in_dim)
            h = x
            for k, (w, b) in enumerate(zip(weights, biases)):
                h = w.astype(np.float64) @ h + b.astype(np.float64)
                if k + 1 < len(weights):
                    h = np.maximum(h, 0)
            y = oracle.mlp(spec, I.pack_weights(weights), I.pack_biases(biases), x)
            np.testing.assert_allclose(y, h, rtol=0, atol=1e-13)


# ------------------------------------------------------------------ composition, mask, determinism
def test_infer_is_composition_of_parts_and_masks(oracle):
    spec = I.spec_param()
    table = I.make_table(spec, 1)
    weights, biases = I.make_mlp(spec, 1, bias_scale=0.1)
    wb, bb = I.pack_weights(weights), I.pack_biases(biases)
    pos = I.positions_uniform(64, I.ROOM_AABB, 2)
    nrm = I.normals_uniform(64, 2)
    nrm[5] = 0.0                       # background texel
    pos[6, 1] = np.nan                 # non-finite inputs are masked, never fault (reading #9)
    nrm[7, 0] = np.inf
    t = np.array([0.37], dtype=np.float32)
    enc = oracle.encode(spec, table, pos, nrm, t)
    out32, out64 = oracle.infer(spec, table, wb, bb, pos, nrm, t, want_f64=True)
    for i in range(64):
        if i in (5, 6, 7):
            assert np.all(out32[i] == 0) and np.all(enc["features"][i] == 0) and np.all(enc["idx"][i] == 0)
            continue
        y = oracle.mlp(spec, wb, bb, enc["features"][i])
        np.testing.assert_allclose(out64[i], 1.0 / (1.0 + np.exp(-y)), rtol=0, atol=3e-16)   # libm vs numpy exp
    # layout of the input vector: latents | SH-16 | param encoding (reading #12)
    np.testing.assert_array_equal(enc["features"][0, 32:48], oracle.sh16(nrm[0].astype(np.float64)))
    np.testing.assert_array_equal(enc["features"][0, 48:64], oracle.param_encode(float(t[0]), 8))
    # determinism and thread-count independence
    again = oracle.infer(spec, table, wb, bb, pos, nrm, t, n_threads=1)
    assert np.array_equal(out32, again)


def test_texel_params_are_the_per_call_function_row_by_row(oracle):
    """with per-texel parameters, texel i is the per-call function (pinned above)
    evaluated at t = tparam[i]; a constant buffer reproduces the per-call result bit for bit; two parameters keep their
    order (reading #12: parameter q at input columns enc_dim + 16 q .. + 16), checked through the MLP composition."""
    for n_params in (1, 2):
        spec = dataclasses.replace(I.spec_param(), n_params=n_params)
        table = I.make_table(spec, 4)
        weights, biases = I.make_mlp(spec, 4, bias_scale=0.1)
        wb, bb = I.pack_weights(weights), I.pack_biases(biases)
        n = 48
        pos = I.positions_uniform(n, I.ROOM_AABB, 5)
        nrm = I.normals_uniform(n, 5)
        nrm[3] = 0.0                                   # a background texel stays zero whatever its parameter
        tp = I.uniform01(17, 3, n * n_params).astype(np.float32).reshape(n, n_params)
        out = oracle.infer_texel_params(spec, table, wb, bb, pos, nrm, tp, want_f64=True)[1]
        for i in range(n):
            row = oracle.infer(spec, table, wb, bb, pos[i:i + 1], nrm[i:i + 1], tp[i], want_f64=True)[1]
            assert np.array_equal(out[i], row[0])
        assert np.all(out[3] == 0)
        const = np.tile(tp[7], (n, 1))
        a = oracle.infer_texel_params(spec, table, wb, bb, pos, nrm, const)
        b = oracle.infer(spec, table, wb, bb, pos, nrm, tp[7])
        assert np.array_equal(a, b)
        # composition of parts: features of texel 0 with ITS parameters through the MLP
        enc = oracle.encode(spec, table, pos[:1], nrm[:1], tp[0])
        x = enc["features"][0]
        for q in range(n_params):
            np.testing.assert_array_equal(x[48 + 16 * q:64 + 16 * q], oracle.param_encode(float(tp[0, q]), 8))
        y = oracle.mlp(spec, wb, bb, x)
        np.testing.assert_allclose(out[0], 1.0 / (1.0 + np.exp(-y)), rtol=0, atol=3e-16)
    # the parameter really enters: two different t give different irradiance
    assert not np.array_equal(out[0], oracle.infer(spec, table, wb, bb, pos[:1], nrm[:1], tp[1], want_f64=True)[1][0])


def test_locate_uses_fp32_op_sequence(oracle):
    """Reading #10: the cell is decided by fl32(fl32(fl32(x-min)*inv)*N) -- compare with the same sequence in
    numpy float32 (an all-fp64 evaluation flips cells on ~1e-3 of full-HD texels)."""
    spec = I.spec_fullhd()
    table = np.zeros((spec.n_levels, spec.table_size, 2), dtype=np.float16)
    N, _ = oracle.level_table(spec)
    pos = I.positions_uniform(200000, I.ROOM_AABB, 13)
    out = oracle.encode(spec, table, pos, _up(len(pos)), want_features=False)
    lo = np.asarray(spec.aabb_min, dtype=np.float32)
    hi = np.asarray(spec.aabb_max, dtype=np.float32)
    inv = (np.float32(1.0) / (hi - lo)).astype(np.float32)
    u = np.clip(((pos - lo).astype(np.float32) * inv).astype(np.float32), np.float32(0), np.float32(1))
    n_flip64 = 0
    for l in range(spec.n_levels):
        p = (u * np.float32(N[l])).astype(np.float32)
        c = np.minimum(np.floor(p).astype(np.int32), int(N[l]) - 1)
        assert np.array_equal(out["cell"][:, l], c)
        assert np.array_equal(out["frac"][:, l], (p - c.astype(np.float32)).astype(np.float32))
        p64 = (pos.astype(np.float64) - lo.astype(np.float64)) / (hi.astype(np.float64) - lo.astype(np.float64)) * float(N[l])
        n_flip64 += int(np.any(np.minimum(np.floor(p64).astype(np.int32), int(N[l]) - 1) != c, axis=1).sum())
    assert n_flip64 > 0          # the fp64 sequence is a different function: the pin above is not vacuous


# ------------------------------------------------------------------ f2: compose + half-resolution upsample
def test_compose_closed_forms_and_torch_interpolate(oracle):
    """PAPER.md:269 (Eq. 2), 405-406 (half resolution with the full-size albedo buffer).  Pins: zero albedo ->
    D + L_e exactly; constant E -> half-res path == full-res path; Eq. 2 by hand on one pixel; the
    upsample equals torch's bilinear interpolate (align_corners=False), a library routine."""
    import torch
    rng = np.random.default_rng(3)
    h, w = 12, 20
    alb = rng.uniform(0, 1, (h, w, 3)).astype(np.float32)
    D = rng.uniform(0, 2, (h, w, 3)).astype(np.float32)
    Le = rng.uniform(0, 1, (h, w, 3)).astype(np.float32)
    Eh = rng.uniform(0, 3, (h // 2, w // 2, 3)).astype(np.float32)
    Ef = rng.uniform(0, 3, (h, w, 3)).astype(np.float32)
    out = oracle.compose(Ef, np.zeros_like(alb), D, Le)
    assert np.array_equal(out, D.astype(np.float64) + Le.astype(np.float64))
    out = oracle.compose(Ef, alb, D, Le)
    y, x, c = 5, 7, 1
    assert abs(out[y, x, c] - (float(alb[y, x, c]) / math.pi * float(Ef[y, x, c]) + float(D[y, x, c]) + float(Le[y, x, c]))) < 1e-15
    const = np.full((h // 2, w // 2, 3), 1.75, dtype=np.float32)
    np.testing.assert_allclose(oracle.compose(const, alb, D, Le),
                               oracle.compose(np.full((h, w, 3), 1.75, dtype=np.float32), alb, D, Le), atol=1e-15)
    up = torch.nn.functional.interpolate(torch.from_numpy(Eh.astype(np.float64)).permute(2, 0, 1)[None], scale_factor=2,
                                         mode="bilinear", align_corners=False)[0].permute(1, 2, 0).numpy()
    want = alb.astype(np.float64) / math.pi * up
    np.testing.assert_allclose(oracle.compose(Eh, alb), want, atol=1e-14)
    with pytest.raises(ValueError):
        oracle.compose(Eh[:, :-1], alb)
