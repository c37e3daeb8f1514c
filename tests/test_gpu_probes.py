"""GPU parity of the probe-grid query (niv_probes_query through the C ABI) against the oracle
(oracle/niv_oracle_ext.c niv_oracle_probe_query), element by element on the same seeded inputs.

Tolerance: the cell is bit-exact by construction (same fp32 op sequence); weights, basis and the
27 x 8 multiply-adds run in fp32 on fp16-exact coefficients, so |error| <= ~100 fp32 roundings of terms bounded by
S = sum_k max|c_k| max|Y_k| -> 2e-5 * S is a generous bound that still fails on any wrong probe, weight or sign."""
import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I

pytestmark = pytest.mark.gpu

ROOM = ((0.0, 0.0, 0.0), (10.0, 4.0, 10.0))


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def niv():
    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv as N
    B.build()
    N.lib()
    return N


def _scale(coeffs):
    ymax = np.array([0.2821, 0.4886, 0.4886, 0.4886, 0.5463, 0.5463, 0.6308, 0.5463, 0.5463])
    return float((np.abs(coeffs.astype(np.float64)).max(axis=(0, 1, 2, 4)) * ymax).sum())


def _run(torch, niv, dims, box, coeffs, pos, nrm, falloff=True):
    g = niv.NivProbeGrid(dims, box[0], box[1], cosine_falloff=falloff)
    g.load(coeffs)
    n = pos.shape[0]
    out = torch.full((n + 3, 3), float("nan"), dtype=torch.float32, device="cuda")     # 3 guard rows
    g.query(torch.from_numpy(pos).cuda(), torch.from_numpy(nrm).cuda(), out[:n])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.all(np.isnan(got[n:])), "wrote past the end of out"
    g.close()
    return got[:n]


@pytest.mark.parametrize("dims,n,falloff", [((2, 2, 2), 1000, True), ((7, 5, 9), 256 * 37 + 11, True),
                                            ((7, 5, 9), 4099, False), ((65, 27, 65), 50000, True)])
def test_probe_query_parity(torch_cuda, niv, oracle, dims, n, falloff):
    coeffs = I.make_probe_grid(dims, 11)
    lo, hi = ROOM
    pos = I.positions_uniform(n, ((lo[0] - 0.3, lo[1] - 0.3, lo[2] - 0.3), (hi[0] + 0.3, hi[1] + 0.3, hi[2] + 0.3)), 5)
    nrm = I.normals_uniform(n, 6)
    pos[0], pos[1] = lo, hi                                  # box corners: the clamp of the last cell
    nrm[7] = 0.0                                             # background
    pos[9, 2] = np.nan
    got = _run(torch_cuda, niv, dims, ROOM, coeffs, pos, nrm, falloff)
    want = oracle.probe_query(dims, lo, hi, coeffs, pos, nrm, cosine_falloff=falloff)
    assert np.all(got[7] == 0.0) and np.all(got[9] == 0.0)
    err = np.abs(got.astype(np.float64) - want.astype(np.float64))
    assert err.max() <= 2e-5 * _scale(coeffs), err.max()


def test_probe_query_on_probes_and_identical_probes(torch_cuda, niv, oracle):
    """SPEC.md:371-372 on the GPU: a query on a probe returns that probe; identical probes -> independent of x."""
    dims = (6, 4, 5)
    lo, hi = ROOM
    coeffs = I.make_probe_grid(dims, 3)
    v = np.array([(0, 0, 0), (5, 3, 4), (2, 1, 3), (4, 0, 2)])
    pos = np.array([[lo[d] + a[d] * (hi[d] - lo[d]) / (dims[d] - 1) for d in range(3)] for a in v], dtype=np.float32)
    nrm = I.normals_uniform(4, 2)
    got = _run(torch_cuda, niv, dims, ROOM, coeffs, pos, nrm, falloff=False)
    for k in range(4):
        Y = oracle.sh16(nrm[k].astype(np.float64))[:9]
        want = Y @ coeffs[v[k][2], v[k][1], v[k][0]].astype(np.float64)
        assert np.abs(got[k] - want).max() <= 5e-5
    one = coeffs[0, 0, 0]
    same = np.broadcast_to(one, coeffs.shape).copy()
    pos = I.positions_uniform(2000, ROOM, 8)
    nrm = np.tile(I.normals_uniform(1, 9), (2000, 1))
    got = _run(torch_cuda, niv, dims, ROOM, same, pos, nrm)
    want = oracle.sh16(nrm[0].astype(np.float64))[:9] @ one.astype(np.float64)
    assert np.abs(got - want[None, :]).max() <= 2e-5 * _scale(same)


def test_probe_query_full_hd_frame(torch_cuda, niv, oracle):
    """The launch bench.py --workload probes times: the configs[1] G-buffer against a 65 x 27 x 65 grid, the WHOLE frame
    against the oracle; census sanity (at most 16 sectors per texel, at least 2 per warp)."""
    torch = torch_cuda
    g = I.make_gbuffer(1920, 1080, 0)
    pos, nrm = g["pos"], g["nrm"]
    dims = I.probe_grid_dims_for_spacing(*ROOM, 10.0 / 64)
    coeffs = I.make_probe_grid(dims, 0)
    got = _run(torch, niv, dims, ROOM, coeffs, pos, nrm)
    want = oracle.probe_query(dims, ROOM[0], ROOM[1], coeffs, pos, nrm)
    masked = np.all(nrm == 0, axis=1)
    assert np.all(got[masked] == 0.0)
    assert np.abs(got.astype(np.float64) - want.astype(np.float64)).max() <= 2e-5 * _scale(coeffs)
    grid = niv.NivProbeGrid(dims, ROOM[0], ROOM[1])
    grid.load(coeffs)
    counts = torch.zeros(2, dtype=torch.int64, device="cuda")
    grid.census(torch.from_numpy(pos).cuda(), torch.from_numpy(nrm).cuda(), counts)
    torch.cuda.synchronize()
    sectors, active = (int(v) for v in counts.cpu().numpy())
    assert active == int((~masked).sum())
    assert 2 * active / 32 <= sectors <= 16 * active
    grid.close()


def test_probe_api_errors(torch_cuda, niv):
    with pytest.raises(niv.NivError):
        niv.NivProbeGrid((1, 2, 2), ROOM[0], ROOM[1])
    with pytest.raises(niv.NivError):
        niv.NivProbeGrid((2, 2, 2), ROOM[1], ROOM[0])
    g = niv.NivProbeGrid((2, 2, 2), ROOM[0], ROOM[1])
    torch = torch_cuda
    p = torch.zeros((4, 3), device="cuda")
    with pytest.raises(niv.NivError):                        # query before load
        g.query(p, p, torch.zeros((4, 3), device="cuda"))
    with pytest.raises(niv.NivError):                        # wrong byte count
        g.load(np.zeros(26, dtype=np.float16))
    g.load(I.make_probe_grid((2, 2, 2), 1))
    g.query(p[:0], p[:0], torch.zeros((0, 3), device="cuda"))  # empty: a no-op
    g.close()
