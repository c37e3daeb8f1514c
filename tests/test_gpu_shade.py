"""GPU parity of niv_infer_shade (include/niv.h): the deferred compose L = albedo / pi * E + direct + emission
(Eq. 2, 403) as the epilogue of the inference kernel, against the oracle's infer followed by the oracle's
compose, through the C ABI."""
import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I

from .test_gpu_parity import Case, MAX_ABS, MEAN_ABS, niv, torch_cuda  # noqa: F401  (fixtures)
from .test_gpu_formats import _dev_bytes, _frame

pytestmark = pytest.mark.gpu


def _shading_inputs(n, seed):
    rng = np.random.default_rng(seed)
    albedo = rng.uniform(0.0, 1.0, (n, 3)).astype(np.float32)
    direct = rng.uniform(0.0, 2.0, (n, 3)).astype(np.float32)
    emission = np.where(rng.uniform(size=(n, 1)) < 0.1, rng.uniform(0.0, 5.0, (n, 3)), 0.0).astype(np.float32)
    return albedo, direct, emission


@pytest.mark.parametrize("which,n", [("tiny", 4100), ("fullhd", 30012), ("paper", 20004), ("param", 12004)])
def test_shade_matches_oracle_infer_then_compose(torch_cuda, niv, oracle, which, n):
    torch = torch_cuda
    spec = {"tiny": I.spec_tiny, "fullhd": I.spec_fullhd, "paper": lambda: I.spec_paper(8, 64), "param": I.spec_param}[which]()
    case = Case(spec, 11, table_amp=0.1 if which == "paper" else 1.0, bias_scale=0.05)
    m = case.gpu_model(niv)
    pos, nrm = _frame(spec, n, 5)
    nrm[5::101] = 0.0                                                      # background texels in every tile
    param = [0.371] if spec.n_params else None
    albedo, direct, emission = _shading_inputs(n, 9)
    e = oracle.infer(spec, case.table, case.wblob, case.bblob, pos, nrm, param=param)
    masked = np.all(nrm == 0, axis=1)
    assert masked.any()
    dp, dn = _dev_bytes(torch, pos), _dev_bytes(torch, nrm)
    da, dd, de = (_dev_bytes(torch, x) for x in (albedo, direct, emission))
    e_gpu = torch.full((n, 3), float("nan"), device="cuda")
    m.infer(dp, dn, e_gpu, param=param)
    for use_d, use_e in ((True, True), (True, False), (False, False)):
        want = oracle.compose(e.reshape(1, n, 3), albedo.reshape(1, n, 3), direct.reshape(1, n, 3) if use_d else None,
                              emission.reshape(1, n, 3) if use_e else None).reshape(n, 3)
        out = torch.full((n + 8, 3), float("nan"), device="cuda")          # guard rows behind the output
        m.infer_shade(dp, dn, da, out[:n], n, direct=dd if use_d else None, emission=de if use_e else None, param=param)
        # the two-pass path of the library: niv_infer, then niv_compose (its 128-bit path: n % 4 == 0) -- the same
        # arithmetic, hence the same bits
        two = torch.full((1, n, 3), float("nan"), device="cuda")
        niv.compose(e_gpu.reshape(1, n, 3), da.reshape(1, n, 3), two, dd.reshape(1, n, 3) if use_d else None,
                    de.reshape(1, n, 3) if use_e else None)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        assert np.isnan(got[n:]).all()
        got = got[:n]
        assert np.array_equal(got.view(np.uint32), two.cpu().numpy().reshape(n, 3).view(np.uint32))
        # against the oracle: E's tolerance scaled by albedo / pi <= 1 / pi, plus the fp32 rounding of the sum
        scale = 1.0 if spec.out_activation == I.OUT_SIGMOID else max(1.0, float(e.max() - e.min()))
        err = np.abs(got.astype(np.float64) - want)
        assert err.max() <= MAX_ABS * scale / np.pi + 1e-6 * max(1.0, float(np.abs(want).max()))
        assert err.mean() <= MEAN_ABS * scale / np.pi + 1e-6
        # background: no irradiance, the sky's direct + emission pass through exactly
        bg = (direct if use_d else 0.0) + (emission if use_e else 0.0) + np.zeros((n, 3), np.float32)
        assert np.array_equal(got[masked], bg[masked].astype(np.float32))
    m.close()


def test_shade_with_compact_formats_and_fp16_output(torch_cuda, niv, oracle):
    torch = torch_cuda
    spec = I.spec_fullhd()
    case = Case(spec, 3)
    m = case.gpu_model(niv)
    n = 25013
    pos, nrm = _frame(spec, n, 8)
    albedo, direct, emission = _shading_inputs(n, 2)
    da, dd, de = (_dev_bytes(torch, x) for x in (albedo, direct, emission))
    for fmt in (I.GBUF_P32_OCT16, I.GBUF_P16_OCT8):
        a, b = I.pack_gbuffer(fmt, pos, nrm, (spec.aabb_min, spec.aabb_max))
        dec_p, dec_n = oracle.decode_gbuffer(fmt, spec.aabb_min, spec.aabb_max, a, b)
        e = oracle.infer(spec, case.table, case.wblob, case.bblob, dec_p, dec_n)
        want = oracle.compose(e.reshape(1, n, 3), albedo.reshape(1, n, 3), direct.reshape(1, n, 3),
                              emission.reshape(1, n, 3)).reshape(n, 3)
        ga = _dev_bytes(torch, a)
        o32 = torch.full((n, 3), float("nan"), device="cuda")
        m.infer_shade(ga, None, da, o32, n, direct=dd, emission=de, gbuf_format=fmt)
        o16 = torch.full((n, 4), -1, dtype=torch.int16, device="cuda")
        m.infer_shade(ga, None, da, o16, n, direct=dd, emission=de, gbuf_format=fmt, out_format=I.OUTFMT_F16X4)
        torch.cuda.synchronize()
        got = o32.cpu().numpy()
        err = np.abs(got.astype(np.float64) - want)
        assert err.max() <= MAX_ABS / np.pi + 1e-6 * float(np.abs(want).max()) and err.mean() <= MEAN_ABS / np.pi + 1e-6
        assert np.array_equal(o16.cpu().numpy().view(np.uint16), oracle.quantise_f16x4(got))
    m.close()


def test_shade_error_codes(torch_cuda, niv):
    torch = torch_cuda
    L = niv.lib()
    z = torch.zeros(4096, dtype=torch.float32, device="cuda")
    p = z.data_ptr()
    m = Case(I.spec_fullhd(), 2).gpu_model(niv)
    assert L.niv_infer_shade(m._h, 0, p, p, None, None, None, None, 0, p + 2048, 8, None) == niv.NIV_ERR_INVALID_ARG   # no albedo
    assert L.niv_infer_shade(m._h, 9, p, p, None, p, None, None, 0, p + 2048, 8, None) == niv.NIV_ERR_INVALID_ARG
    assert L.niv_infer_shade(m._h, 0, p, p, None, p, None, None, 0, p + 2048, 0, None) == niv.NIV_OK                   # n = 0
    assert L.niv_infer_shade(m._h, 0, p, p, None, p, None, None, 0, p + 2048, 8, None) == niv.NIV_OK
    assert L.niv_infer_shade(None, 0, p, p, None, p, None, None, 0, p + 2048, 8, None) == niv.NIV_ERR_INVALID_ARG
    torch.cuda.synchronize()
    m.close()
    wide = Case(I.spec_fullhd(17, 128, 2), 2).gpu_model(niv)
    assert L.niv_infer_shade(wide._h, 0, p, p, None, p, None, None, 0, p + 2048, 8, None) == niv.NIV_ERR_UNSUPPORTED
    wide.close()


def test_shade_image_tiling_and_gridless(torch_cuda, niv, oracle):
    """niv_infer_image_shade: the same bits as niv_infer_shade (8 x 4 pixel blocks per warp, partial edge tiles); the
    grid-less models shade too (against the oracle)."""
    torch = torch_cuda
    w, h = 212, 67
    n = w * h
    g = I.make_gbuffer(w, h, 4)
    albedo, direct, emission = _shading_inputs(n, 4)
    da, dd, de = (_dev_bytes(torch, x) for x in (albedo, direct, emission))
    for spec, amp in ((I.spec_fullhd(), 1.0), (I.spec_paper(8, 64), 0.1), (I.spec_paper_pe(32), 0.1)):
        case = Case(spec, 6, table_amp=amp, bias_scale=0.05)
        m = case.gpu_model(niv)
        dp, dn = _dev_bytes(torch, g["pos"]), _dev_bytes(torch, g["nrm"])
        lin = torch.full((n, 3), float("nan"), device="cuda")
        img = torch.full((n, 3), float("nan"), device="cuda")
        m.infer_shade(dp, dn, da, lin, n, direct=dd, emission=de)
        m.infer_shade(dp, dn, da, img, n, direct=dd, emission=de, image=(w, h))
        torch.cuda.synchronize()
        assert torch.equal(lin, img)
        e = oracle.infer(spec, case.table, case.wblob, case.bblob, g["pos"], g["nrm"])
        want = oracle.compose(e.reshape(h, w, 3), albedo.reshape(h, w, 3), direct.reshape(h, w, 3),
                              emission.reshape(h, w, 3)).reshape(n, 3)
        scale = 1.0 if spec.out_activation == I.OUT_SIGMOID else max(1.0, float(e.max() - e.min()))
        err = np.abs(lin.cpu().numpy().astype(np.float64) - want)
        assert err.max() <= MAX_ABS * scale / np.pi + 1e-6 * max(1.0, float(np.abs(want).max()))
        assert err.mean() <= MEAN_ABS * scale / np.pi + 1e-6
        m.close()


def test_shade_back_to_back_on_rotating_and_aliased_buffers(torch_cuda, niv):
    """launch overlap with the three shading inputs in the records: a chain of calls where each call's `direct` is the
    previous call's output, beside calls on disjoint buffers -- the result of serial execution (NIV_OVERLAP=0 semantics:
    computed here by synchronising after every call)."""
    torch = torch_cuda
    spec = I.spec_fullhd()
    m = Case(spec, 8).gpu_model(niv)
    w, h = 320, 180
    n = w * h
    g = I.make_gbuffer(w, h, 2)
    dp, dn = _dev_bytes(torch, g["pos"]), _dev_bytes(torch, g["nrm"])
    albedo, direct, _ = _shading_inputs(n, 6)
    da, d0 = _dev_bytes(torch, albedo), _dev_bytes(torch, direct)

    def chain(sync):
        bufs = [torch.zeros((n, 3), device="cuda") for _ in range(4)]
        prev = d0
        for k in range(12):
            out = bufs[k % 4]
            m.infer_shade(dp, dn, da, out, n, direct=prev, image=(w, h))
            if sync:
                torch.cuda.synchronize()
            prev = out
        torch.cuda.synchronize()
        return prev.clone()

    assert torch.equal(chain(False), chain(True))
    m.close()


def test_shade_full_hd_frame(torch_cuda, niv, oracle):
    """BASELINE.json configs[1] at full size through the launch `bench.py --shade` times (niv_infer_image_shade): every texel
    bit-equal to niv_infer_image + niv_compose, 100,000 sampled texels against the oracle's infer + compose, RGB9E5 words of
    the whole frame against the oracle's quantiser."""
    torch = torch_cuda
    spec = I.spec_fullhd()
    case = Case(spec, 0)
    m = case.gpu_model(niv)
    w, h = 1920, 1080
    n = w * h
    g = I.make_gbuffer(w, h, 0)
    pos, nrm = g["pos"], g["nrm"]
    rng = np.random.default_rng(5)
    albedo = rng.uniform(0, 1, (n, 3)).astype(np.float32)
    direct = rng.uniform(0, 2, (n, 3)).astype(np.float32)
    dp, dn, da, dd = (_dev_bytes(torch, x) for x in (pos, nrm, albedo, direct))
    out = torch.full((n, 3), float("nan"), device="cuda")
    m.infer_shade(dp, dn, da, out, n, direct=dd, image=(w, h))
    e = torch.full((n, 3), float("nan"), device="cuda")
    m.infer_image(dp, dn, e, w, h)
    two = torch.full((h, w, 3), float("nan"), device="cuda")
    niv.compose(e.view(h, w, 3), da.view(h, w, 3), two, dd.view(h, w, 3))
    words = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    m.infer_shade(dp, dn, da, words, n, direct=dd, image=(w, h), out_format=I.OUTFMT_RGB9E5)
    torch.cuda.synchronize()
    assert torch.equal(out, two.view(n, 3))
    got = out.cpu().numpy()
    assert np.array_equal(words.cpu().numpy().view(np.uint32), oracle.quantise_rgb9e5(got))
    sel = np.unique((I.random_u64(91, 1, 100000) % np.uint64(n)).astype(np.int64))
    eo = oracle.infer(spec, case.table, case.wblob, case.bblob, pos[sel], nrm[sel])
    k = sel.shape[0]
    want = oracle.compose(eo.reshape(1, k, 3), albedo[sel].reshape(1, k, 3), direct[sel].reshape(1, k, 3)).reshape(k, 3)
    err = np.abs(got[sel].astype(np.float64) - want)
    assert err.max() <= MAX_ABS / np.pi + 1e-6 * float(np.abs(want).max()) and err.mean() <= MEAN_ABS / np.pi + 1e-6
    m.close()
