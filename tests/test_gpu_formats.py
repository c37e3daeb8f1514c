"""GPU parity of the compact G-buffer formats and the fp16 output (include/niv.h *_packed): the CUDA
path against the oracle's decode + the standard oracle path, through the C ABI."""
import numpy as np
import pytest

from paper_2602_12949_b200 import inputs as I

from .test_gpu_parity import Case, MAX_ABS, MEAN_ABS, _check_irradiance, niv, torch_cuda  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu


def _dev_bytes(torch, arr):
    return None if arr is None else torch.from_numpy(np.ascontiguousarray(arr)).cuda()


def _frame(spec, n, seed):
    g = I.make_gbuffer(160, 90, seed)
    pos, nrm = I.positions_uniform(n, (spec.aabb_min, spec.aabb_max), seed), I.normals_uniform(n, seed)
    k = min(n, g["pos"].shape[0])
    pos[:k], nrm[:k] = g["pos"][:k], g["nrm"][:k]                   # coherent part with background texels
    pos[k - 1] = np.float32(spec.aabb_max)                          # u = 1 on every axis
    return pos, nrm


@pytest.mark.parametrize("fmt", [I.GBUF_F32X4, I.GBUF_P32_OCT16, I.GBUF_P16_OCT8])
def test_decode_matches_the_oracle_bit_for_bit_in_position(torch_cuda, niv, oracle, fmt):
    torch = torch_cuda
    spec = I.spec_fullhd()
    m = Case(spec, 1).gpu_model(niv)
    n = 50021
    pos, nrm = _frame(spec, n, 3)
    a, b = I.pack_gbuffer(fmt, pos, nrm, (spec.aabb_min, spec.aabb_max))
    want_p, want_n = oracle.decode_gbuffer(fmt, spec.aabb_min, spec.aabb_max, a, b)
    dp = torch.full((n, 3), float("nan"), device="cuda")
    dn = torch.full((n, 3), float("nan"), device="cuda")
    m.decode_gbuffer(fmt, _dev_bytes(torch, a), _dev_bytes(torch, b), dp, dn, n)
    torch.cuda.synchronize()
    assert np.array_equal(dp.cpu().numpy().view(np.uint32), want_p.view(np.uint32))      # positions decide cells: exact
    gn = dn.cpu().numpy()
    assert np.abs(gn - want_n).max() <= 3e-7
    bg = np.all(want_n == 0, axis=1)
    assert bg.any() and np.all(gn[bg] == 0)
    # hence the indices: the debug dump on the GPU-decoded positions equals the oracle's on its own decode
    idx = torch.zeros((n, spec.n_levels, 8), dtype=torch.int32, device="cuda")
    m.debug_encode(dp, dn, idx=idx)
    torch.cuda.synchronize()
    enc = oracle.encode(spec, Case(spec, 1).table, want_p, want_n, want_features=False)
    assert np.array_equal(idx.cpu().numpy().astype(np.uint32), enc["idx"])
    m.close()


@pytest.mark.parametrize("which", ["fullhd", "paper"])
@pytest.mark.parametrize("fmt", [I.GBUF_F32X4, I.GBUF_P32_OCT16, I.GBUF_P16_OCT8])
@pytest.mark.parametrize("ofmt", [I.OUTFMT_F32X3, I.OUTFMT_F16X4])
def test_packed_inference_matches_the_oracle(torch_cuda, niv, oracle, which, fmt, ofmt):
    torch = torch_cuda
    spec = I.spec_fullhd() if which == "fullhd" else I.spec_paper(8, 64)
    case = Case(spec, 5, table_amp=1.0 if which == "fullhd" else 0.1, bias_scale=0.05)
    m = case.gpu_model(niv)
    n = 30011
    pos, nrm = _frame(spec, n, 7)
    a, b = I.pack_gbuffer(fmt, pos, nrm, (spec.aabb_min, spec.aabb_max))
    dec_p, dec_n = oracle.decode_gbuffer(fmt, spec.aabb_min, spec.aabb_max, a, b)
    want = oracle.infer(spec, case.table, case.wblob, case.bblob, dec_p, dec_n)
    scale = 1.0 if spec.out_activation == I.OUT_SIGMOID else max(1.0, float(want.max() - want.min()))
    da, db = _dev_bytes(torch, a), _dev_bytes(torch, b)
    ref32 = torch.full((n, 3), float("nan"), device="cuda")
    m.infer_packed(fmt, da, db, ref32, n)
    if ofmt == I.OUTFMT_F32X3:
        torch.cuda.synchronize()
        _check_irradiance(ref32.cpu().numpy(), want, dec_n, dec_p, scale)
    else:
        out = torch.full((n, 4), -1, dtype=torch.int16, device="cuda")
        m.infer_packed(fmt, da, db, out, n, out_format=ofmt)
        torch.cuda.synchronize()
        bits = out.cpu().numpy().view(np.uint16)
        # the conversion itself: bit-exact against the oracle's quantiser fed the GPU's own fp32 result
        assert np.array_equal(bits, oracle.quantise_f16x4(ref32.cpu().numpy()))
        # and the value: the oracle's irradiance within the bar plus half an fp16 step of the output range
        got = bits[:, :3].view(np.float16).astype(np.float32)
        masked = np.all(dec_n == 0, axis=1)
        assert np.all(got[masked] == 0)
        err = np.abs(got[~masked].astype(np.float64) - want[~masked])
        assert err.max() <= (MAX_ABS + 2.0 ** -11 * max(1.0, float(np.abs(want).max()))) * scale
        assert err.mean() <= (MEAN_ABS + 2.0 ** -12 * max(1.0, float(np.abs(want).max()))) * scale
    m.close()


@pytest.mark.parametrize("which", ["fullhd", "paper"])
def test_rgb9e5_output_matches_the_oracle(torch_cuda, niv, oracle, which):
    """NIV_OUTFMT_RGB9E5: the words are bit-exact against the oracle's quantiser fed the GPU's own
    fp32 result, and the decoded values are the oracle's irradiance within the bar plus half a quantisation step; negative
    irradiance of a linear output layer clamps to 0; every entry point (device, image, host pageable / pinned) and the shading
    epilogue write the same words."""
    torch = torch_cuda
    spec = I.spec_fullhd() if which == "fullhd" else I.spec_paper(8, 64)
    case = Case(spec, 5, table_amp=1.0 if which == "fullhd" else 0.1, bias_scale=0.05)
    m = case.gpu_model(niv)
    w, h = 212, 67
    n = w * h
    g = I.make_gbuffer(w, h, 4)
    pos, nrm = g["pos"], g["nrm"]
    want = oracle.infer(spec, case.table, case.wblob, case.bblob, pos, nrm)
    dp, dn = _dev_bytes(torch, pos), _dev_bytes(torch, nrm)
    ref32 = torch.full((n, 3), float("nan"), device="cuda")
    m.infer(dp, dn, ref32)
    out = torch.full((n + 5,), -1, dtype=torch.int32, device="cuda")
    m.infer_packed(I.GBUF_F32X3, dp, dn, out[:n], n, out_format=I.OUTFMT_RGB9E5)
    img = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    m.infer_image_packed(I.GBUF_F32X3, dp, dn, img, w, h, out_format=I.OUTFMT_RGB9E5)
    torch.cuda.synchronize()
    words = out.cpu().numpy().view(np.uint32)
    assert np.all(words[n:] == 0xFFFFFFFF)                                      # guard entries behind the output
    words = words[:n]
    e32 = ref32.cpu().numpy()
    assert np.array_equal(words, oracle.quantise_rgb9e5(e32))
    assert np.array_equal(img.cpu().numpy().view(np.uint32), words)
    dec = oracle.decode_rgb9e5(words)
    masked = np.all(nrm == 0, axis=1)
    assert masked.any() and np.all(words[masked] == 0)
    wc = np.clip(want.astype(np.float64), 0.0, 65408.0)
    if which == "paper":
        assert (want < 0).any()                                                 # the linear output does go negative: clamped
    scale = 1.0 if spec.out_activation == I.OUT_SIGMOID else max(1.0, float(want.max() - want.min()))
    step = 2.0 ** ((words >> 27).astype(np.float64) - 24)
    err = np.abs(dec - wc)[~masked]
    assert np.all(err <= MAX_ABS * scale + step[~masked, None] / 2)
    assert err.mean() <= MEAN_ABS * scale + float(step[~masked].mean()) / 2
    host = np.zeros((n,), dtype=np.uint32)                                       # pageable: staged copies
    m.infer_host_packed(I.GBUF_F32X3, pos, nrm, host, n, out_format=I.OUTFMT_RGB9E5)
    assert np.array_equal(host, words)
    pp, pn = torch.from_numpy(pos).pin_memory(), torch.from_numpy(nrm).pin_memory()   # pinned: zero copy
    po = torch.zeros((n,), dtype=torch.int32).pin_memory()
    m.infer_host_packed(I.GBUF_F32X3, pp, pn, po, n, out_format=I.OUTFMT_RGB9E5)
    assert np.array_equal(po.numpy().view(np.uint32), words)
    # the shading epilogue into RGB9E5: the quantiser of its own fp32 result
    rng = np.random.default_rng(1)
    alb, dr = (torch.from_numpy(rng.uniform(0, 1, (n, 3)).astype(np.float32)).cuda() for _ in range(2))
    s32 = torch.full((n, 3), float("nan"), device="cuda")
    s9 = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    m.infer_shade(dp, dn, alb, s32, n, direct=dr, image=(w, h))
    m.infer_shade(dp, dn, alb, s9, n, direct=dr, image=(w, h), out_format=I.OUTFMT_RGB9E5)
    torch.cuda.synchronize()
    assert np.array_equal(s9.cpu().numpy().view(np.uint32), oracle.quantise_rgb9e5(s32.cpu().numpy()))
    # misaligned output -> INVALID_ARG
    L = niv.lib()
    assert L.niv_infer_packed(m._h, 0, dp.data_ptr(), dn.data_ptr(), None, 2, out.data_ptr() + 2, 8, None) == niv.NIV_ERR_INVALID_ARG
    m.close()


def test_packed_entry_points_agree_with_each_other(torch_cuda, niv):
    """image tiling, the host entry point (pinned and pageable buffers) and the linear device path: the same bits."""
    torch = torch_cuda
    spec = I.spec_fullhd()
    m = Case(spec, 2).gpu_model(niv)
    w, h = 212, 67
    g = I.make_gbuffer(w, h, 4)
    n = w * h
    for fmt in (I.GBUF_F32X4, I.GBUF_P32_OCT16, I.GBUF_P16_OCT8):
        a, b = I.pack_gbuffer(fmt, g["pos"], g["nrm"], (spec.aabb_min, spec.aabb_max))
        da, db = _dev_bytes(torch, a), _dev_bytes(torch, b)
        for ofmt, shape, dt, npdt in ((I.OUTFMT_F32X3, (n, 3), torch.float32, np.float32), (I.OUTFMT_F16X4, (n, 4), torch.int16, np.int16)):
            lin = torch.zeros(shape, dtype=dt, device="cuda")
            img = torch.zeros(shape, dtype=dt, device="cuda")
            m.infer_packed(fmt, da, db, lin, n, out_format=ofmt)
            m.infer_image_packed(fmt, da, db, img, w, h, out_format=ofmt)
            torch.cuda.synchronize()
            assert torch.equal(lin, img)
            host_out = np.zeros(shape, dtype=npdt)                                        # pageable: staged copies
            m.infer_host_packed(fmt, a, b, host_out, n, out_format=ofmt)
            assert np.array_equal(host_out, lin.cpu().numpy())
            pa = torch.from_numpy(a).pin_memory()                                         # pinned: zero copy
            pb = None if b is None else torch.from_numpy(b).pin_memory()
            po = torch.zeros(shape, dtype=dt).pin_memory()
            m.infer_host_packed(fmt, pa, pb, po, n, out_format=ofmt)
            assert torch.equal(po, lin.cpu())
    m.close()


def test_packed_error_codes(torch_cuda, niv):
    torch = torch_cuda
    spec = I.spec_fullhd()
    m = Case(spec, 2).gpu_model(niv)
    L = niv.lib()
    z = torch.zeros(1024, dtype=torch.float32, device="cuda")
    p = z.data_ptr()
    assert L.niv_infer_packed(m._h, 7, p, p, None, 0, p, 8, None) == niv.NIV_ERR_INVALID_ARG             # unknown format
    assert L.niv_infer_packed(m._h, 0, p, p, None, 5, p, 8, None) == niv.NIV_ERR_INVALID_ARG
    assert L.niv_infer_packed(m._h, 2, p + 4, None, None, 0, p, 8, None) == niv.NIV_ERR_INVALID_ARG      # 16-byte records
    assert L.niv_infer_packed(m._h, 3, p + 4, None, None, 0, p, 8, None) == niv.NIV_ERR_INVALID_ARG
    assert L.niv_infer_packed(m._h, 0, p, p, None, 1, p + 4, 8, None) == niv.NIV_ERR_INVALID_ARG         # fp16 x 4 output
    assert L.niv_infer_packed(m._h, 1, p, None, None, 0, p, 8, None) == niv.NIV_ERR_INVALID_ARG          # two arrays needed
    assert L.niv_infer_packed(m._h, 2, p, None, None, 0, p, 0, None) == niv.NIV_OK                       # n = 0
    assert L.niv_infer_packed(m._h, 2, p, None, None, 1, p, 8, None) == niv.NIV_OK
    torch.cuda.synchronize()
    m.close()
    wide = Case(I.spec_fullhd(17, 128, 2), 2).gpu_model(niv)                                            # width 128: fp32 x 3 only
    assert L.niv_infer_packed(wide._h, 2, p, None, None, 0, p, 8, None) == niv.NIV_ERR_UNSUPPORTED
    assert L.niv_infer_packed(wide._h, 0, p, p, None, 0, p, 8, None) == niv.NIV_OK
    torch.cuda.synchronize()
    wide.close()
