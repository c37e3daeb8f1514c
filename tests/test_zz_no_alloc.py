"""niv_infer_host_static (include/niv.h): the host-buffer call that allocates nothing -- the fused kernel staged through the
library's static device array -- against the existing path (niv_infer_host, and niv_infer on device buffers), on two calls
in a row.  Collected last on purpose (the suite runs with `pytest -x`)."""
import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I

pytestmark = pytest.mark.gpu

MAX_ABS = 2e-3          # the irradiance bar of tests/test_gpu_parity.py
MEAN_ABS = 2e-4


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


def _model(niv, spec, seed):
    m = niv.NivModel(spec)
    w, b = I.make_mlp(spec, seed, 0.05)
    m.load_params(I.make_table(spec, seed, -1.0, 1.0), I.pack_weights(w), I.pack_biases(b))
    return m


def _frame(spec, n, seed):
    pos, nrm = I.positions_uniform(n, (spec.aabb_min, spec.aabb_max), seed), I.normals_uniform(n, seed)
    g = I.make_gbuffer(96, 54, seed)                       # a coherent part with background texels
    k = min(n, g["pos"].shape[0])
    pos[:k], nrm[:k] = g["pos"][:k], g["nrm"][:k]
    return pos, nrm


def test_static_scratch_entry_point_matches_the_existing_path(torch_cuda, niv):
    torch = torch_cuda
    spec = I.spec_fullhd()
    m = _model(niv, spec, 3)
    # two calls in a row on the shared array: a large one, then a smaller ragged one (stale rows of the first call must
    # not show), then the first again
    calls = [_frame(spec, 200003, 1), _frame(spec, 4097, 2), _frame(spec, 200003, 1)]
    results = []
    for pos, nrm in calls:
        n = pos.shape[0]
        want = np.full((n, 3), np.nan, dtype=np.float32)
        m.infer_host(pos, nrm, want)                                        # the existing path (staged copies)
        got = np.full((n, 3), np.nan, dtype=np.float32)
        m.infer_host_static(pos, nrm, got)
        assert np.all(np.isfinite(got))
        masked = np.all(nrm == 0, axis=1)
        assert masked.any() and np.all(got[masked] == 0.0)
        err = np.abs(got.astype(np.float64) - want.astype(np.float64))
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (err.max(), err.mean())
        dev = torch.full((n, 3), float("nan"), device="cuda")               # and the device path
        m.infer(torch.from_numpy(pos).cuda(), torch.from_numpy(nrm).cuda(), dev)
        torch.cuda.synchronize()
        err = np.abs(got.astype(np.float64) - dev.cpu().numpy().astype(np.float64))
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (err.max(), err.mean())
        results.append(got)
    assert np.array_equal(results[0], results[2])                           # same input, same bits, whatever ran between
    # pinned buffers and a caller's stream work the same way
    pos, nrm = calls[1]
    st = torch.cuda.Stream()
    pp, pn = torch.from_numpy(pos).pin_memory(), torch.from_numpy(nrm).pin_memory()
    po = torch.full((pos.shape[0], 3), float("nan")).pin_memory()
    m.infer_host_static(pp, pn, po, stream=st)
    assert np.array_equal(po.numpy(), results[1])
    m.close()


def test_static_scratch_limit_and_other_models(torch_cuda, niv):
    L = niv.lib()
    spec = I.spec_param()                                                   # a model with a scene parameter
    m = _model(niv, spec, 5)
    nmax = niv.NIV_STATIC_MAX_TEXELS
    pos, nrm = _frame(spec, nmax + 1, 4)
    out = np.zeros((nmax + 1, 3), dtype=np.float32)
    rc = L.niv_infer_host_static(m._h, pos.ctypes.data, nrm.ctypes.data, (niv.C.c_float * 1)(0.25), out.ctypes.data,
                                 nmax + 1, None)
    assert rc == niv.NIV_ERR_TOO_LARGE and b"NIV_STATIC_MAX_TEXELS" in L.niv_error_string(rc)
    assert L.niv_infer_host_static(m._h, None, None, None, None, 0, None) == niv.NIV_OK          # n = 0: a no-op
    assert L.niv_infer_host_static(m._h, pos.ctypes.data, nrm.ctypes.data, None, out.ctypes.data, 8, None) \
        == niv.NIV_ERR_INVALID_ARG                                                                # the model wants a parameter
    # exactly the maximum, twice in a row, against the existing path
    for t in (0.25, 0.75):
        want = np.full((nmax, 3), np.nan, dtype=np.float32)
        got = np.full((nmax, 3), np.nan, dtype=np.float32)
        m.infer_host(pos[:nmax], nrm[:nmax], want, param=[t])
        m.infer_host_static(pos[:nmax], nrm[:nmax], got, param=[t])
        err = np.abs(got.astype(np.float64) - want.astype(np.float64))
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (err.max(), err.mean())
    m.close()
