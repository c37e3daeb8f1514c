#!/usr/bin/env python
"""bench.py -- throughput of the fused NIV inference path (BASELINE.json metric) on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload fullhd|incoherent|param] [--impl ours|reference]

One "step" = one pass of the whole hot path (niv_infer: one fused kernel, rows a0..a12 of DESIGN.md) over one
1920x1080 G-buffer per GPU.  Prints ONE JSON line on rank 0 (contract in the task statement / DESIGN.md sec. 7).

  value / ms_per_step   device-resident inputs, CUDA events on the launching stream, max over ranks
  e2e                   niv_infer_host: pinned HOST buffers in, HOST buffer out, copies inside the timed region
  roofline              gather roofline (measured random-sector rate, sector census of this very frame), with the
                        tensor and HBM rooflines beside it; frac = slowest roofline time / measured time
  cpu_baseline          the oracle, as it stands, on this box's host cores over a bounded sample (rank 0, N=1)

--impl reference times the CPU oracle instead (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2602_12949_b200 import dist as D  # noqa: E402
from paper_2602_12949_b200 import inputs as I  # noqa: E402

W_PX, H_PX = 1920, 1080
N_TEXELS = W_PX * H_PX
METRIC = "NIV fused inference throughput on a 1920x1080 G-buffer (ms_per_step = ms per frame)"
UNIT = "Gqueries/s"
PROBES_METRIC = "probe-grid query throughput on a 1920x1080 G-buffer (SURVEY 8 f4; ms_per_step = ms per frame)"
RING = 8                      # distinct input/output buffer sets rotated between steps (8 x 74.6 MB > 126 MB L2)


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


PAPER_LEVELS, PAPER_WIDTH = 8, 64        # --paper-levels / --paper-width (workload "paper")
PAPER_DIR_BANDS = 0                      # --paper-dir-bands: frequency bands on the direction, 0 or 4
# PAPER.md:383-389 (Table 1, RTX 4090, full HD): ms per frame by (grid levels, width)
PAPER_TABLE1_MS = {(0, 16): 0.19, (0, 32): 0.20, (0, 64): 0.25, (2, 64): 0.31, (4, 64): 0.67, (6, 64): 1.06, (8, 64): 1.35}
PAPER_TABLE1_HALF_MS = {(0, 16): 0.029, (0, 32): 0.031, (0, 64): 0.069, (2, 64): 0.088, (4, 64): 0.18, (6, 64): 0.26, (8, 64): 0.37}


def make_workload(name: str, frame: int, with_params: bool = True):
    """-> spec, table, wblob, bblob, pos, nrm, param, description  (with_params False: table and blobs are None -- a rank
    that receives the parameters by broadcast does not generate them)"""
    paper_levels, paper_width = PAPER_LEVELS, PAPER_WIDTH
    if name == "param":
        spec, param = I.spec_param(), [0.625]
    elif name == "paper":
        spec = I.spec_paper(paper_levels, paper_width) if paper_levels else I.spec_paper_pe(paper_width)
        if PAPER_DIR_BANDS:
            spec = I.spec_paper_dirfreq(paper_levels, paper_width, PAPER_DIR_BANDS)
        param = None
    else:
        spec, param = I.spec_fullhd(), None
    table = I.make_table(spec, 0) if with_params else None
    w, b = I.make_mlp(spec, 0) if with_params else (None, None)
    if name == "incoherent":
        pos = I.positions_uniform(N_TEXELS, (spec.aabb_min, spec.aabb_max), frame)
        nrm = I.normals_uniform(N_TEXELS, frame)
        desc = "configs[2]: 2,073,600 i.i.d. queries in the room AABB, normals uniform on S^2"
        masked = 0.0
    else:
        g = I.make_gbuffer(W_PX, H_PX, 0, frame=frame)
        pos, nrm, masked = g["pos"], g["nrm"], g["masked_fraction"]
        desc = ("configs[%d]: 1920x1080 G-buffer ray-cast from the seeded procedural room (16 spheres + 16 boxes), "
                "%.1f%% background texels" % (3 if name == "param" else 1, 100 * masked))
        if name == "paper":
            desc = ("the paper's own model (PAPER.md Table 1 row 'width %d, %s grid levels': %s, four weight matrices) on "
                    "the configs[1] G-buffer, %.1f%% background texels"
                    % (paper_width, paper_levels or "-", "F=4, scale sqrt 2, T=2^17" if paper_levels else
                       "eight-band positional encoding", 100 * masked))
            if PAPER_DIR_BANDS:
                desc += "; direction = raw vector + %d frequency bands per axis" % PAPER_DIR_BANDS
    return (spec, table, I.pack_weights(w) if with_params else None, I.pack_biases(b) if with_params else None, pos, nrm,
            param, desc, masked)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "tflops_burst": float(d["bf16_tflops"]),
                "tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "50"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0]))
                mx.append(float(c[1]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(pos, nrm, n_sample):
    """Every k-th 128-texel tile of the frame, so the sample has the frame's mix of coherent / masked texels."""
    n = pos.shape[0]
    tiles = n // 128
    want_tiles = max(1, min(tiles, n_sample // 128))
    sel_t = np.linspace(0, tiles - 1, want_tiles).astype(np.int64)
    sel = (sel_t[:, None] * 128 + np.arange(128)[None, :]).reshape(-1)
    return np.ascontiguousarray(pos[sel]), np.ascontiguousarray(nrm[sel]), sel.size


def time_oracle(spec, table, wb, bb, pos, nrm, param, budget_s):
    """The oracle as it stands on all host cores, on a sample sized for ~budget_s seconds."""
    from oracle import niv_oracle
    niv_oracle.build()
    prm = None if param is None else np.float32(param)
    cal_p, cal_n, cal = oracle_sample(pos, nrm, 32768)
    t0 = time.perf_counter()
    niv_oracle.infer(spec, table, wb, bb, cal_p, cal_n, param=prm)
    rate = cal / (time.perf_counter() - t0)
    n_s = int(min(pos.shape[0], max(32768, rate * budget_s)))
    sp, sn, n_s = oracle_sample(pos, nrm, n_s)
    t0 = time.perf_counter()
    niv_oracle.infer(spec, table, wb, bb, sp, sn, param=prm)
    dt = time.perf_counter() - t0
    cores = niv_oracle.max_threads()
    # ... and on ONE thread (SURVEY 8(d) "(a) 1 thread and (b) all cores"), on a 1/16 sample
    s1p, s1n, n_1 = oracle_sample(pos, nrm, max(4096, n_s // 16))
    t0 = time.perf_counter()
    niv_oracle.infer(spec, table, wb, bb, s1p, s1n, param=prm, n_threads=1)
    dt1 = time.perf_counter() - t0
    return n_s, dt, cores, n_1, dt1


def run_reference(args):
    """Reference arm of this tier = the CPU oracle, timed on this box's host cores (rank 0 only)."""
    if _env_int("RANK", 0) != 0:
        return
    from oracle import niv_oracle
    niv_oracle.build()
    if args.workload == "probes":
        aabb = I.ROOM_AABB
        dims = I.probe_grid_dims_for_spacing(aabb[0], aabb[1], args.probe_spacing)
        coeffs = I.make_probe_grid(dims, 0)
        g = I.make_gbuffer(W_PX, H_PX, 0, frame=0)
        pos, nrm = g["pos"], g["nrm"]
        desc = "configs[1] G-buffer queried in a %dx%dx%d grid of SH-2 probes" % dims

        spec = None

        def once(sp, sn):
            niv_oracle.probe_query(dims, aabb[0], aabb[1], coeffs, sp, sn)
    else:
        spec, table, wb, bb, pos, nrm, param, desc, masked = make_workload(args.workload, 0)
        prm = None if param is None else np.float32(param)

        def once(sp, sn):
            niv_oracle.infer(spec, table, wb, bb, sp, sn, param=prm)
    sp, sn, n_s = oracle_sample(pos, nrm, args.ref_sample)
    for _ in range(args.warmup):
        once(sp, sn)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        once(sp, sn)
    dt = (time.perf_counter() - t0) / args.steps
    val = n_s / dt / 1e9
    cores = niv_oracle.max_threads()
    sample = "%d of %d texels per step (every k-th 128-texel tile of the frame)" % (n_s, N_TEXELS)
    print(json.dumps({
        "impl": "reference", "metric": PROBES_METRIC if args.workload == "probes" else METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "ms_per_frame_extrapolated":
        dt * 1e3 * N_TEXELS / n_s, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "description": desc,
                   "model": _model_str(spec) if spec is not None else "SH-2 probe grid, 27 fp16 per probe"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def _model_str(spec):
    dims = [spec.in_dim] + [spec.hidden_width] * spec.n_hidden_layers + [3]
    grid = ("hash grid L=%d F=%d T=2^%d N0=%d b=%g" % (spec.n_levels, spec.n_features, spec.log2_table_size,
                                                        spec.base_resolution, spec.per_level_scale)
            if spec.n_levels else "no grid: 8-band positional encoding")
    return "%s; %s%s; MLP %s fp16 weights / fp32 accumulate; %s output" % (
        grid,
        "raw direction" if spec.sh_degree == 0 else "SH-16",
        "; %d param(s) x 8 sin/cos" % spec.n_params if spec.n_params else "", "->".join(map(str, dims)),
        "sigmoid" if spec.out_activation == I.OUT_SIGMOID else "linear")


def measure_gather_peak(torch, niv, table_bytes, num_sms):
    """Random 32-byte-sector gather rate from a resident buffer of the tables' size (SURVEY.md 8(d) BW_L2g),
    and the same with 8 lanes sharing a sector.  Returns GB/s of sector traffic."""
    nbytes = 1 << int(np.ceil(np.log2(max(table_bytes, 8 << 20))))
    buf = torch.zeros(nbytes // 4, dtype=torch.int32, device="cuda")
    sink = torch.zeros(4, dtype=torch.int32, device="cuda")
    res = {}
    n_ctas, lpl = num_sms * 8, 256
    for name, pattern, sectors_per_load in (("random_sector", 0, 1.0), ("shared_sector_x8", 3, 1.0 / 8)):
        for _ in range(3):
            niv.probe_gather(buf, pattern, n_ctas, lpl, 1, sink)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 10
        e0.record()
        for r in range(reps):
            niv.probe_gather(buf, pattern, n_ctas, lpl, 100 + r, sink)
        e1.record()
        torch.cuda.synchronize()
        dt = e0.elapsed_time(e1) * 1e-3 / reps
        loads = n_ctas * 256 * lpl
        res[name] = {"gloads_per_s": loads / dt / 1e9, "sector_gbs": loads * sectors_per_load * 32 / dt / 1e9}
    del buf
    return res, nbytes


def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    rank, world, local = D.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        B.build()
    if world > 1:
        dist.barrier()
    niv.lib()

    # weak scaling: each rank owns one full frame per step; strong scaling: the ranks share ONE frame, each a block of
    # rows.  The model is replicated: rank 0 builds the parameters, one broadcast per blob hands them out.
    strong = args.scaling == "strong" and world > 1
    frame = 0 if strong else D.frame_of_rank(rank, world)[0]
    spec, table, wb, bb, pos, nrm, param, desc, masked = make_workload(args.workload, frame, with_params=(rank == 0))
    img_w, img_h = W_PX, H_PX
    n_job = pos.shape[0] * (1 if strong else world)                 # texels all ranks process per step
    if strong:
        if args.workload == "incoherent":
            lo, hi = D.texel_range_of_rank(pos.shape[0], rank, world)
        else:
            r0, r1 = D.row_range_of_rank(H_PX, rank, world)
            lo, hi, img_h = r0 * W_PX, r1 * W_PX, r1 - r0
        pos, nrm = np.ascontiguousarray(pos[lo:hi]), np.ascontiguousarray(nrm[lo:hi])
        masked = float(np.mean(np.all(nrm == 0, axis=1)))
    n = pos.shape[0]
    model = niv.NivModel(spec, local)
    if world > 1:
        wl = sum(a * b_ for a, b_ in zip([spec.in_dim] + [spec.hidden_width] * spec.n_hidden_layers,
                                         [spec.hidden_width] * spec.n_hidden_layers + [3]))
        bl = spec.hidden_width * spec.n_hidden_layers + 3
        shapes = [((spec.n_levels * spec.table_size * spec.n_features,), torch.float16), ((wl,), torch.float16),
                  ((bl,), torch.float32)]
        t_table, t_w, t_b = D.broadcast_params([table, wb, bb] if rank == 0 else None, shapes, torch.device("cuda", local))
        model.load_params(t_table, t_w, t_b)
        del t_table, t_w, t_b
    else:
        model.load_params(table, wb, bb)
    info = model.info

    d_pos = [torch.from_numpy(pos).cuda() for _ in range(RING)]
    d_nrm = [torch.from_numpy(nrm).cuda() for _ in range(RING)]
    d_out = [torch.empty((n, 3), dtype=torch.float32, device="cuda") for _ in range(RING)]
    stream = torch.cuda.current_stream()
    d_tp = None
    if args.texel_params:                            # the parameter varies over the image, one value per texel
        if not spec.n_params:
            raise SystemExit("--texel-params needs a model with scene parameters (--workload param)")
        tp = (np.float32(param)[None, :] + np.float32(0.25) * (np.arange(n, dtype=np.float32) / np.float32(n))[:, None])
        d_tp = torch.from_numpy(np.ascontiguousarray(tp, dtype=np.float32)).cuda()

    # the G-buffer workloads are images: niv_infer_image (8 x 4 pixel blocks per warp); the incoherent set has no
    # image structure and goes through niv_infer (32 consecutive texels per warp), as does --tiling linear
    image = args.tiling == "image" and args.workload != "incoherent" and d_tp is None and bool(info.image_tiled)

    def infer_dev(k):
        if d_tp is not None:
            model.infer_texel_params(d_pos[k], d_nrm[k], d_tp, d_out[k])
        elif image:
            model.infer_image(d_pos[k], d_nrm[k], d_out[k], img_w, img_h, param=param)
        else:
            model.infer(d_pos[k], d_nrm[k], d_out[k], param=param)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ---------------------------------------------------------------------
    for s in range(args.warmup):
        infer_dev(s % RING)
    # the timed region: K launches back to back between two events (an event record after every launch costs 2.5 us
    # per step, profiles/r01_v2.md); the per-launch spread comes from a second, instrumented pass of the same K steps
    ev_a, ev_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clocks = ClockSampler(local) if rank == 0 else None
    ev_a.record(stream)
    for s in range(args.steps):
        infer_dev(s % RING)
    ev_b.record(stream)
    barrier()
    total_ms = ev_a.elapsed_time(ev_b)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for s in range(args.steps):
        infer_dev(s % RING)
        ev[s + 1].record(stream)
    torch.cuda.synchronize()
    per = np.array([ev[s].elapsed_time(ev[s + 1]) for s in range(args.steps)])
    kernel_ms_timed = total_ms / args.steps            # this rank's average launch duration over the timed region
    # cold variant (SURVEY 8(d) timing protocol): the table evicted from L2 before every launch by streaming a 512 MB
    # buffer, one event pair per launch; the tables then come from HBM once per frame
    cold = None
    if args.cold_steps > 0 and rank == 0:
        evict = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
        c_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.cold_steps)]
        for s in range(args.cold_steps):
            evict.fill_(s & 0xFF)
            c_ev[s][0].record(stream)
            infer_dev(s % RING)
            c_ev[s][1].record(stream)
        torch.cuda.synchronize()
        c = np.array([a.elapsed_time(b) for a, b in c_ev])
        cold = {"ms_median": float(np.median(c)), "ms_min": float(np.min(c)), "launches": int(args.cold_steps),
                "note": "a 512 MB buffer is overwritten before every launch: tables, cell blocks and weights come from HBM"}
        del evict
    # clocks keep sampling a little longer so that short runs still get a few samples under load
    t_end = time.time() + 0.3
    while time.time() < t_end:
        infer_dev(0)
        torch.cuda.synchronize()
    clk = clocks.stop() if clocks else None
    total_ms = D.reduce_max(total_ms, "cuda")
    ms_step = total_ms / args.steps
    value = n_job / (ms_step * 1e-3) / 1e9               # whole job: all ranks' texels over the slowest rank's time

    # ---- end to end: pinned host buffers through niv_infer_host ------------------------------------
    e2e_steps = max(3, min(args.steps, 20))
    h_pos = [torch.from_numpy(pos).pin_memory() for _ in range(2)]
    h_nrm = [torch.from_numpy(nrm).pin_memory() for _ in range(2)]
    h_out = [torch.empty((n, 3), dtype=torch.float32).pin_memory() for _ in range(2)]
    for s in range(3):
        model.infer_host(h_pos[s % 2], h_nrm[s % 2], h_out[s % 2], param=param)
    barrier()
    t0 = time.perf_counter()
    for s in range(e2e_steps):
        model.infer_host(h_pos[s % 2], h_nrm[s % 2], h_out[s % 2], param=param)   # synchronises: out has landed
    torch.cuda.synchronize()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    e2e_ms = D.reduce_max(e2e_ms, "cuda")
    e2e_value = n_job / (e2e_ms * 1e-3) / 1e9
    checksum = float(h_out[0].sum())

    # ---- the same end-to-end call on the compact G-buffer formats / fp16 output: fewer bytes per
    #      texel over PCIe.  Formats of include/niv.h; the packing is the producer's job and is not timed.
    e2e_compact = []
    if spec.hidden_width <= 64 and spec.n_levels and not args.no_compact_e2e:
        aabb = (spec.aabb_min, spec.aabb_max)
        for gf, of, name in ((I.GBUF_P32_OCT16, I.OUTFMT_F16X4, "pos fp32 x 3 + oct16 normal (16 B) -> fp16 x 4 (8 B)"),
                             (I.GBUF_P16_OCT8, I.OUTFMT_F16X4, "pos unorm16 x 3 + oct8 normal (8 B) -> fp16 x 4 (8 B)"),
                             (I.GBUF_P16_OCT8, I.OUTFMT_RGB9E5, "pos unorm16 x 3 + oct8 normal (8 B) -> RGB9E5 (4 B)")):
            a, b = I.pack_gbuffer(gf, pos, nrm, aabb)
            ha = [torch.from_numpy(a).pin_memory() for _ in range(2)]
            ho = [(torch.empty((n,), dtype=torch.int32) if of == I.OUTFMT_RGB9E5 else torch.empty((n, 4), dtype=torch.int16)).pin_memory()
                  for _ in range(2)]
            for s in range(3):
                model.infer_host_packed(gf, ha[s % 2], None, ho[s % 2], n, out_format=of, param=param)
            barrier()
            t0 = time.perf_counter()
            for s in range(e2e_steps):
                model.infer_host_packed(gf, ha[s % 2], None, ho[s % 2], n, out_format=of, param=param)
            torch.cuda.synchronize()
            ms = D.reduce_max((time.perf_counter() - t0) * 1e3 / e2e_steps, "cuda")
            e2e_compact.append({"formats": name, "gbuf_format": gf, "out_format": of, "value": n_job / (ms * 1e-3) / 1e9,
                                "unit": UNIT, "ms_per_step": ms, "h2d_bytes_per_step": int(a.nbytes),
                                "d2h_bytes_per_step": int(ho[0].numel() * ho[0].element_size()),
                                "api": "niv_infer_host_packed (pinned host buffers, zero copy)"})
            del ha, ho

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rooflines (rank 0) -------------------------------------------------------------------------
    peaks = load_peaks()
    counts = torch.zeros(niv.NIV_CENSUS_COUNTS, dtype=torch.int64, device="cuda")
    if image:
        model.probe_sectors_image(d_pos[0], d_nrm[0], img_w, img_h, counts)    # the census of the warps that ran
    else:
        model.probe_sectors(d_pos[0], d_nrm[0], counts)
    torch.cuda.synchronize()
    c = counts.cpu().numpy()
    L = spec.n_levels
    sectors, lines, n_active = int(c[:L].sum()), int(c[16:16 + L].sum()), int(c[32])
    touched = int(c[33:33 + L].sum())                   # sectors the kernel's own layout touches (cell-block levels)
    gpeak, probe_bytes = measure_gather_peak(torch, niv, info.table_bytes, info.num_sms)
    kernel_s = kernel_ms_timed * 1e-3                   # one fused kernel per step: timed region / K (gaps included)
    dims = [spec.in_dim] + [spec.hidden_width] * spec.n_hidden_layers + [3]
    flop_texel = 2 * sum(dims[i] * dims[i + 1] for i in range(len(dims) - 1))
    hbm_bytes = 36 * n
    t_gather = sectors * 32 / (gpeak["random_sector"]["sector_gbs"] * 1e9)
    t_tensor = flop_texel * n / (peaks["tflops_sustained"] * 1e12)
    t_hbm = hbm_bytes / (peaks["hbm_gbs"] * 1e9)
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")             # ncu DRAM bytes per launch (profiles/traffic.md)
    if os.path.exists(tp):
        with open(tp) as f:
            for ln in f.read().splitlines()[1:]:
                k, _, v = ln.partition(",")
                if k == args.workload and v.strip().isdigit():
                    traffic = int(v)
    t_all = {"l2-gather": t_gather, "tensor": t_tensor, "hbm": t_hbm}
    bound = max(t_all, key=t_all.get)                # the slowest roofline bounds the kernel (north_star)
    roofline = {
        "bound": bound, "kernel": "niv_fused_kernel" if spec.hidden_width <= 64 else "niv_fused_w128_kernel",
        "achieved": {"l2-gather": sectors * 32 / kernel_s / 1e9, "tensor": flop_texel * n / kernel_s / 1e12,
                     "hbm": hbm_bytes / kernel_s / 1e9}[bound],
        "peak": {"l2-gather": gpeak["random_sector"]["sector_gbs"], "tensor": peaks["tflops_sustained"],
                 "hbm": peaks["hbm_gbs"]}[bound],
        "unit": "TFLOP/s" if bound == "tensor" else "GB/s",
        "frac": t_all[bound] / kernel_s, "traffic": traffic,
        "l2_gather": {"achieved": sectors * 32 / kernel_s / 1e9, "peak": gpeak["random_sector"]["sector_gbs"],
                      "unit": "GB/s", "frac": t_gather / kernel_s},
        "peak_source": "measured in this run: niv_probe_gather, random 32 B sectors of a resident %d MiB buffer"
                       % (probe_bytes >> 20),
        "algorithmic": {"sectors_per_launch": sectors, "sectors_per_active_texel": sectors / max(n_active, 1),
                        "lines_per_active_texel": lines / max(n_active, 1), "active_texels": n_active,
                        "gathers_per_active_texel": 8 * L, "sectors_per_level": [int(v) for v in c[:L]],
                        "definition": "distinct 32 B sectors per (warp, level) among the corner addresses of the [L][T] "
                                      "table as loaded (SURVEY.md 8(d)); independent of the library's internal layout"},
        "touched": {"sectors_per_launch": touched, "sectors_per_active_texel": touched / max(n_active, 1),
                    "sectors_per_level": [int(v) for v in c[33:33 + L]], "cell_block_levels": int(info.cell_levels),
                    "cell_block_bytes": int(info.cell_bytes), "achieved_gbs": touched * 32 / kernel_s / 1e9,
                    "frac_of_probe_peak": touched * 32 / kernel_s / 1e9 / gpeak["random_sector"]["sector_gbs"],
                    "note": "what the kernel's own layout reads: levels held as cell blocks cost one sector per "
                            "distinct cell instead of the 8 corners' sectors"},
        "gather_rate_ggathers_per_s": 8 * L * n_active / kernel_s / 1e9,
        "frac_note": ("frac is the ALGORITHMIC census (sectors of the [L][T] table the frame needs) over the probe's random-sector "
                      "rate; on levels held as cell blocks one sector serves the 8 corners the census counts up to 8 sectors for, so "
                      "on scattered queries it can exceed 1 -- `touched` is the same ratio for what is really read"),
        "probe": gpeak,
        "t_roofline_us": {"l2_gather": t_gather * 1e6, "tensor": t_tensor * 1e6, "hbm": t_hbm * 1e6},
        "tensor": {"achieved": flop_texel * n / kernel_s / 1e12, "peak": peaks["tflops_sustained"],
                   "unit": "TFLOP/s", "frac": t_tensor / kernel_s, "peak_source": peaks["source"] + " bf16 sustained (fp16 = same rate)"},
        "hbm": {"achieved": hbm_bytes / kernel_s / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": t_hbm / kernel_s, "peak_source": peaks["source"]},
        "kernel_ms": {"timed_region_mean": kernel_ms_timed,
                      "instrumented_pass": {"mean": float(np.mean(per)), "median": float(np.median(per)),
                                            "min": float(np.min(per)),
                                            "note": "same K steps again with an event after every launch"}},
    }

    cpu = None
    if world == 1 and not args.no_cpu_baseline and d_tp is None:
        n_s, dt, cores, n_1, dt1 = time_oracle(spec, table, wb, bb, pos, nrm, param, args.cpu_budget)
        cpu = {"value": n_s / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%d of %d texels (every k-th 128-texel tile of the frame), %.1f s" % (n_s, n, dt),
               "ms_per_frame_extrapolated": dt * 1e3 * n / n_s,
               "one_thread": {"value": n_1 / dt1 / 1e9, "unit": UNIT, "cores": 1,
                              "sample": "%d texels, %.1f s" % (n_1, dt1), "ms_per_frame_extrapolated": dt1 * 1e3 * n / n_1}}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step,
        # the same K steps again with an event after every launch (which costs ~2.5 us per step and keeps consecutive
        # launches from overlapping): per-launch median and minimum
        "ms_per_launch_instrumented": {"median": float(np.median(per)), "min": float(np.min(per))},
        "higher_is_better": True, "scaling": "strong" if strong else "weak",
        # BASELINE.md holds a paper number only for the paper's own model: 1.35 ms per full-HD frame on an RTX 4090
        # = 1.536 Gqueries/s -- another machine's, context not target
        "vs_baseline": (value / (N_TEXELS / ((PAPER_TABLE1_HALF_MS if args.half else PAPER_TABLE1_MS)[(PAPER_LEVELS, PAPER_WIDTH)]
                                             * 1e-3) / 1e9))
        if (args.workload == "paper" and world == 1 and (PAPER_LEVELS, PAPER_WIDTH) in PAPER_TABLE1_MS and not PAPER_DIR_BANDS) else None,
        "dtype": "f16 operands / f32 accumulate (index path: f32 + u32)", "data": "synthetic",
        "config": {"workload": args.workload, "description": desc, "model": _model_str(spec),
                   "texels_per_gpu_per_step": n, "masked_fraction": masked, "parallelism": "dp%d (model replicated by one "
                   "broadcast per blob, %s, no data-path collective)" % (world, "row blocks of ONE frame per rank" if strong
                                                                         else "one frame per rank"),
                   "l2": "inputs/outputs rotate over %d distinct buffer sets (%.0f MB > 126 MB L2) so G-buffer reads "
                         "come from HBM; the %.0f MiB table stays L2-resident by design" %
                         (RING, RING * 36 * n / 1e6, info.table_bytes / 2 ** 20),
                   "grid": "%d CTAs = %d SMs x %d, %d texels per tile" % (info.num_sms * info.ctas_per_sm,
                                                                         info.num_sms, info.ctas_per_sm,
                                                                         info.tile_texels),
                   "tiling": ("niv_infer_image: a warp = an 8 x 4 pixel block, a tile = 32 x 4 pixels" if image else
                              "niv_infer: a warp = 32 consecutive texels, a tile = 128"),
                   **({"texel_params": "device timing through niv_infer_texel_params, t = %s + 0.25 i/n per texel; "
                                       "e2e stays the per-call entry point; no cpu_baseline on this line" % list(param)}
                      if d_tp is not None else {})},
        "active_gqueries_per_s": value * (1.0 - masked),
        "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                "h2d_bytes_per_step": 24 * n, "d2h_bytes_per_step": 12 * n,
                "api": "niv_infer_host (pinned host buffers, zero copy: the fused kernel reads the G-buffer and writes the irradiance over PCIe itself)",
                "checksum": checksum},
        "gpu_launches": args.steps, "clocks": clk, "roofline": roofline,
    }
    if e2e_compact:
        out["e2e_compact"] = e2e_compact
    if cold:
        out["cold_l2"] = cold
    if cpu:
        out["cpu_baseline"] = cpu
    print(json.dumps(out))
    model.close()
    if world > 1:
        dist.destroy_process_group()


def run_probes(args):
    """the paper's probe-grid baseline as a second workload over the configs[1] G-buffer:
    a regular SH-2 probe grid at the memory budget the paper compares at ("5.4 MB budget": 54 B per probe
    -> ~100 k probes, 0.16 m apart in the 10 x 4 x 10 m room), queried once per texel.  Same JSON contract."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if _env_int("WORLD_SIZE", 1) != 1:
        raise SystemExit("--workload probes is a one-GPU line")
    torch.cuda.set_device(0)
    B.build()
    niv.lib()
    aabb = I.ROOM_AABB
    dims = I.probe_grid_dims_for_spacing(aabb[0], aabb[1], args.probe_spacing)
    coeffs = I.make_probe_grid(dims, 0)
    g = I.make_gbuffer(W_PX, H_PX, 0, frame=0)
    pos, nrm, masked = g["pos"], g["nrm"], g["masked_fraction"]
    n = pos.shape[0]
    grid = niv.NivProbeGrid(dims, aabb[0], aabb[1], cosine_falloff=True)
    grid.load(coeffs)
    d_pos = [torch.from_numpy(pos).cuda() for _ in range(RING)]
    d_nrm = [torch.from_numpy(nrm).cuda() for _ in range(RING)]
    d_out = [torch.empty((n, 3), dtype=torch.float32, device="cuda") for _ in range(RING)]
    stream = torch.cuda.current_stream()
    for s in range(args.warmup):
        grid.query(d_pos[s % RING], d_nrm[s % RING], d_out[s % RING])
    ev_a, ev_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    clocks = ClockSampler(0)
    ev_a.record(stream)
    for s in range(args.steps):
        grid.query(d_pos[s % RING], d_nrm[s % RING], d_out[s % RING])
    ev_b.record(stream)
    torch.cuda.synchronize()
    ms_step = ev_a.elapsed_time(ev_b) / args.steps
    t_end = time.time() + 0.3
    while time.time() < t_end:
        grid.query(d_pos[0], d_nrm[0], d_out[0])
        torch.cuda.synchronize()
    clk = clocks.stop()
    # end to end: pinned host buffers, copies inside the timed region (the probe query has no host entry point of its own)
    h_pos, h_nrm = torch.from_numpy(pos).pin_memory(), torch.from_numpy(nrm).pin_memory()
    h_out = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))

    def e2e_once():
        d_pos[0].copy_(h_pos, non_blocking=True)
        d_nrm[0].copy_(h_nrm, non_blocking=True)
        grid.query(d_pos[0], d_nrm[0], d_out[0])
        h_out.copy_(d_out[0], non_blocking=True)
        torch.cuda.synchronize()

    for _ in range(2):
        e2e_once()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_once()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps

    peaks = load_peaks()
    counts = torch.zeros(2, dtype=torch.int64, device="cuda")
    grid.census(d_pos[0], d_nrm[0], counts)
    torch.cuda.synchronize()
    sectors, n_active = int(counts[0].item()), int(counts[1].item())
    grid_bytes = 64 * dims[0] * dims[1] * dims[2]
    info_sms = torch.cuda.get_device_properties(0).multi_processor_count
    gpeak, probe_bytes = measure_gather_peak(torch, niv, grid_bytes, info_sms)
    kernel_s = ms_step * 1e-3
    hbm_bytes = 36 * n
    t_gather = sectors * 32 / (gpeak["random_sector"]["sector_gbs"] * 1e9)
    t_hbm = hbm_bytes / (peaks["hbm_gbs"] * 1e9)
    t_all = {"l2-gather": t_gather, "hbm": t_hbm}
    bound = max(t_all, key=t_all.get)
    roofline = {
        "bound": bound, "kernel": "niv_probes_query_kernel",
        "achieved": {"l2-gather": sectors * 32 / kernel_s / 1e9, "hbm": hbm_bytes / kernel_s / 1e9}[bound],
        "peak": {"l2-gather": gpeak["random_sector"]["sector_gbs"], "hbm": peaks["hbm_gbs"]}[bound], "unit": "GB/s",
        "frac": t_all[bound] / kernel_s, "traffic": None,
        "peak_source": ("measured in this run: niv_probe_gather, random 32 B sectors of a resident %d MiB buffer" % (probe_bytes >> 20))
        if bound == "l2-gather" else peaks["source"],
        "algorithmic": {"sectors_per_launch": sectors, "sectors_per_active_texel": sectors / max(n_active, 1),
                        "active_texels": n_active, "probes_per_texel": 8, "bytes_per_probe_record": 64,
                        "hbm_bytes_per_texel": 36},
        "t_roofline_us": {"l2_gather": t_gather * 1e6, "hbm": t_hbm * 1e6},
        "hbm": {"achieved": hbm_bytes / kernel_s / 1e9, "peak": peaks["hbm_gbs"], "frac": t_hbm / kernel_s},
        "l2_gather": {"achieved": sectors * 32 / kernel_s / 1e9, "peak": gpeak["random_sector"]["sector_gbs"],
                      "frac": t_gather / kernel_s},
    }
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import niv_oracle
        niv_oracle.build()
        sp, sn, n_s = oracle_sample(pos, nrm, 262144)
        t0 = time.perf_counter()
        niv_oracle.probe_query(dims, aabb[0], aabb[1], coeffs, sp, sn)
        rate = n_s / (time.perf_counter() - t0)
        sp, sn, n_s = oracle_sample(pos, nrm, int(min(n, max(262144, rate * args.cpu_budget))))
        t0 = time.perf_counter()
        niv_oracle.probe_query(dims, aabb[0], aabb[1], coeffs, sp, sn)
        dt = time.perf_counter() - t0
        cpu = {"value": n_s / dt / 1e9, "unit": UNIT, "cores": niv_oracle.max_threads(), "kind": "oracle",
               "sample": "%d of %d texels (every k-th 128-texel tile of the frame), %.1f s" % (n_s, n, dt)}
    out = {
        "metric": PROBES_METRIC,
        "value": n / kernel_s / 1e9, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16 probes / f32 arithmetic (cell: f32 + u32)", "data": "synthetic",
        "config": {"workload": "probes", "description": "configs[1] G-buffer (%.1f%% background) queried in a %dx%dx%d grid of "
                   "SH-2 probes, %.2f m apart (%.2f MB at the paper's 54 B per probe; 64 B records on the device), cosine "
                   "fall-off on" % (100 * masked, dims[0], dims[1], dims[2], args.probe_spacing,
                                    54 * dims[0] * dims[1] * dims[2] / 1e6),
                   "texels_per_gpu_per_step": n, "masked_fraction": masked,
                   "l2": "inputs/outputs rotate over %d distinct buffer sets (%.0f MB > 126 MB L2)" % (RING, RING * 36 * n / 1e6)},
        "e2e": {"value": n / (e2e_ms * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": e2e_ms, "steps": e2e_steps,
                "h2d_bytes_per_step": 24 * n, "d2h_bytes_per_step": 12 * n,
                "api": "pinned host buffers -> cudaMemcpyAsync -> niv_probes_query -> cudaMemcpyAsync, synchronised per step"},
        "gpu_launches": args.steps, "clocks": clk, "roofline": roofline,
    }
    if cpu:
        out["cpu_baseline"] = cpu
    print(json.dumps(out))
    grid.close()


def run_probe_patterns(args):
    """The gather micro-benchmark in all its access patterns (include/niv.h niv_probe_gather) on an L1-resident, a
    borderline and an L2-resident buffer: clocks per warp-wide load instruction.  A table for profiles/, not the
    contract line."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    B.build()
    niv.lib()
    torch.cuda.set_device(0)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    mhz = 1965.0
    sink = torch.zeros(4, dtype=torch.int32, device="cuda")
    for kb in (32, 64, 8192):
        buf = torch.zeros(kb * 256, dtype=torch.int32, device="cuda")
        for pat in range(10):
            n_ctas, lpl = sms * 8, 256
            for _ in range(3):
                niv.probe_gather(buf, pat, n_ctas, lpl, 1, sink)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for r in range(10):
                niv.probe_gather(buf, pat, n_ctas, lpl, 100 + r, sink)
            e1.record()
            torch.cuda.synchronize()
            dt = e0.elapsed_time(e1) * 1e-3 / 10
            loads = n_ctas * 256 * lpl
            per_clk = loads / 32 / dt / sms / (mhz * 1e6)
            print(json.dumps({"buffer_KB": kb, "pattern": pat, "gloads_per_s": loads / dt / 1e9,
                              "clocks_per_warp_load_at_1965MHz": 1.0 / per_clk}), flush=True)


def run_encode(args):
    """north_star (2): the stand-alone encoding kernel (niv_encode: rows a1..a9, fp16 feature rows to HBM) on the
    configs[1] frame: ms, the gather census GB/s and its fraction of the measured random-sector rate, HBM GB/s (24 B in,
    2 * in_dim B out per texel).  One JSON line (not the contract line); ncu counters: profiles/r02_encode.md."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    B.build()
    niv.lib()
    torch.cuda.set_device(0)
    spec, table, wb, bb, pos, nrm, param, desc, masked = make_workload("fullhd", 0)
    n = pos.shape[0]
    model = niv.NivModel(spec, 0)
    model.load_params(table, wb, bb)
    ring = 4
    d_pos = [torch.from_numpy(pos).cuda() for _ in range(ring)]
    d_nrm = [torch.from_numpy(nrm).cuda() for _ in range(ring)]
    d_f = [torch.empty((n, spec.in_dim), dtype=torch.float16, device="cuda") for _ in range(ring)]
    steps = args.steps or 100
    for k in range(5):
        model.encode(d_pos[k % ring], d_nrm[k % ring], d_f[k % ring])
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for k in range(steps):
        model.encode(d_pos[k % ring], d_nrm[k % ring], d_f[k % ring])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    counts = torch.zeros(niv.NIV_CENSUS_COUNTS, dtype=torch.int64, device="cuda")
    model.probe_sectors(d_pos[0], d_nrm[0], counts)
    torch.cuda.synchronize()
    c = counts.cpu().numpy()
    sectors = int(c[:spec.n_levels].sum())
    gpeak, _ = measure_gather_peak(torch, niv, model.info.table_bytes, model.info.num_sms)
    peaks = load_peaks()
    hbm_bytes = (24 + 2 * spec.in_dim) * n
    print(json.dumps({"op": "niv_encode", "workload": "fullhd", "ms": ms, "gqueries_per_s": n / ms / 1e6,
                      "gather": {"sectors": sectors, "achieved_gbs": sectors * 32 / ms / 1e6,
                                 "peak_gbs": gpeak["random_sector"]["sector_gbs"],
                                 "frac": sectors * 32 / ms / 1e6 / gpeak["random_sector"]["sector_gbs"]},
                      "hbm": {"bytes": hbm_bytes, "achieved_gbs": hbm_bytes / ms / 1e6, "peak_gbs": peaks["hbm_gbs"],
                              "frac": hbm_bytes / ms / 1e6 / peaks["hbm_gbs"]},
                      "cell_levels": int(model.info.cell_levels)}))
    model.close()


def run_sweep(args):
    """BASELINE.json configs[4]: table size x MLP width at full HD, and resolution x frames per call.  One JSON line
    per case on stdout (NOT the contract line: a table for profiles/)."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    B.build()
    niv.lib()
    torch.cuda.set_device(0)
    gb_cache = {}

    def gbuf(w, h, frames):
        key = (w, h, frames)
        if key not in gb_cache:
            gs = [I.make_gbuffer(w, h, 0, frame=f) for f in range(frames)]
            gb_cache[key] = (np.concatenate([g["pos"] for g in gs]), np.concatenate([g["nrm"] for g in gs]),
                             float(np.mean([g["masked_fraction"] for g in gs])))
        return gb_cache[key]

    def one(log2_T, width, w, h, frames):
        spec = I.spec_fullhd(log2_T, width, 2)
        pos, nrm, masked = gbuf(w, h, frames)
        n = pos.shape[0]
        model = niv.NivModel(spec, 0)
        wts, bs = I.make_mlp(spec, 0)
        model.load_params(I.make_table(spec, 0), I.pack_weights(wts), I.pack_biases(bs))
        ring = max(2, min(8, int(np.ceil(200e6 / (36.0 * n)))))
        d_pos = [torch.from_numpy(pos).cuda() for _ in range(ring)]
        d_nrm = [torch.from_numpy(nrm).cuda() for _ in range(ring)]
        d_out = [torch.empty((n, 3), dtype=torch.float32, device="cuda") for _ in range(ring)]
        # frames stacked in one call form one taller image (every height here is a multiple of the 4-row tile)
        image = args.tiling == "image" and bool(model.info.image_tiled)

        def call(k):
            if image:
                model.infer_image(d_pos[k % ring], d_nrm[k % ring], d_out[k % ring], w, h * frames)
            else:
                model.infer(d_pos[k % ring], d_nrm[k % ring], d_out[k % ring])

        for k in range(5):
            call(k)
        steps = 30
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for k in range(steps):
            call(k)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        counts = torch.zeros(niv.NIV_CENSUS_COUNTS, dtype=torch.int64, device="cuda")
        if image:
            model.probe_sectors_image(d_pos[0], d_nrm[0], w, h * frames, counts)
        else:
            model.probe_sectors(d_pos[0], d_nrm[0], counts)
        torch.cuda.synchronize()
        sectors = int(counts[:16].sum().item())
        info = model.info
        row = {"log2_T": log2_T, "table_MiB": info.table_bytes / 2 ** 20, "width": width, "res": "%dx%d" % (w, h),
               "frames_per_call": frames, "tiling": "image" if image else "linear", "texels": n, "masked": masked, "ms_per_call": ms, "ms_per_frame": ms / frames,
               "gqueries_per_s": n / ms / 1e6, "gather_sector_GBs": sectors * 32 / ms / 1e6,
               "hbm_io_GBs": 36.0 * n / ms / 1e6, "ctas_per_sm": info.ctas_per_sm, "smem_bytes": info.smem_bytes}
        print(json.dumps(row), flush=True)
        model.close()
        del d_pos, d_nrm, d_out
        torch.cuda.empty_cache()

    for log2_T in (14, 16, 18, 20):
        for width in (32, 64, 128):
            one(log2_T, width, W_PX, H_PX, 1)
    for (w, h) in ((1280, 720), (1920, 1080), (2560, 1440), (3840, 2160)):
        for frames in (1, 2, 4):
            one(17, 64, w, h, frames)


def graph_ms(launch, steps):
    """ms per launch of `steps` launches (launch(k), k = 0..steps-1) recorded into ONE CUDA graph and replayed between two
    events: a 25 us kernel is shorter than one call through the Python binding, so a loop of calls would time the host."""
    import torch

    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for k in range(steps):
                launch(k)
        g.replay()                                       # warm-up of the instantiated graph
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        side.synchronize()
        e0.record(side)
        g.replay()
        e1.record(side)
        side.synchronize()
    return e0.elapsed_time(e1) / steps


def run_compose(args):
    """the compose kernel alone (HBM-bound) at full HD, E at full and at half resolution.  One JSON line
    per case: ms, algorithmic GB/s and its fraction of the measured HBM copy bandwidth."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    B.build()
    niv.lib()
    torch.cuda.set_device(0)
    peaks = load_peaks()
    for (h, w) in ((H_PX, W_PX), (2 * H_PX, 2 * W_PX)):
        ring = 6 if h == H_PX else 2                     # 6 x 100 MB / 2 x 400 MB > L2
        for half in (False, True):
            eh, ew = (h // 2, w // 2) if half else (h, w)
            bufs = [[torch.rand((h, w, 3), device="cuda") for _ in range(3)] + [torch.rand((eh, ew, 3), device="cuda"),
                    torch.empty((h, w, 3), device="cuda")] for _ in range(ring)]
            for k in range(5):
                a, d, le, e, o = bufs[k % ring]
                niv.compose(e, a, o, d, le)
            steps = args.steps or 100

            def one(k):
                a, d, le, e, o = bufs[k % ring]
                niv.compose(e, a, o, d, le)
            ms = graph_ms(one, steps)
            nbytes = (48 + (3 if half else 12)) * h * w
            print(json.dumps({"op": "niv_compose", "E_resolution": "%dx%d" % (ew, eh), "frame": "%dx%d" % (w, h),
                              "ms": ms, "algorithmic_bytes": nbytes,
                              "roofline": {"bound": "hbm", "achieved": nbytes / ms / 1e6, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                           "frac": nbytes / ms / 1e6 / peaks["hbm_gbs"], "peak_source": peaks["source"]}}), flush=True)
        # joint-bilateral upsample (niv_compose_jb): + the full-resolution position and normal (24 B per pixel) and the
        # half-resolution guides (6 B per pixel)
        eh, ew = h // 2, w // 2
        gf, gh = I.make_gbuffer(w, h, 0), I.make_gbuffer(ew, eh, 0)
        c = lambda a, sh: torch.from_numpy(np.ascontiguousarray(a.reshape(sh))).cuda()
        sets = [[c(gf["pos"], (h, w, 3)), c(gf["nrm"], (h, w, 3)), torch.rand((h, w, 3), device="cuda"),
                 torch.rand((h, w, 3), device="cuda"), torch.rand((h, w, 3), device="cuda"), torch.empty((h, w, 3), device="cuda")]
                for _ in range(ring)]
        e_h, p_h, n_h = torch.rand((eh, ew, 3), device="cuda"), c(gh["pos"], (eh, ew, 3)), c(gh["nrm"], (eh, ew, 3))

        def jb(k):
            p, n_, a, d, le, o = sets[k % ring]
            niv.compose_jb(e_h, p_h, n_h, p, n_, a, o, 0.15, 8.0, d, le)
        for k in range(5):
            jb(k)
        steps = args.steps or 100
        ms = graph_ms(jb, steps)
        nbytes = (72 + 9) * h * w
        print(json.dumps({"op": "niv_compose_jb", "E_resolution": "%dx%d" % (ew, eh), "frame": "%dx%d" % (w, h), "ms": ms,
                          "algorithmic_bytes": nbytes,
                          "roofline": {"bound": "hbm", "achieved": nbytes / ms / 1e6, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                       "frac": nbytes / ms / 1e6 / peaks["hbm_gbs"], "peak_source": peaks["source"]}}), flush=True)
        del sets


def run_shade(args):
    """full-resolution shading of the configs[1] frame, two ways -- niv_infer_image then niv_compose (the
    irradiance goes to HBM and comes back), niv_infer (linear tiles) then niv_compose, and niv_infer_shade (the compose as
    the inference kernel's epilogue).  One JSON line; ms per frame from `steps` launches between two events, buffers rotating
    over RING sets."""
    import torch

    from paper_2602_12949_b200 import build as B
    from paper_2602_12949_b200 import niv

    B.build()
    niv.lib()
    torch.cuda.set_device(0)
    spec, table, wb, bb, pos, nrm, param, desc, masked = make_workload(args.workload, 0)
    n = pos.shape[0]
    model = niv.NivModel(spec, 0)
    model.load_params(table, wb, bb)
    ring = 4
    d_pos = [torch.from_numpy(pos).cuda() for _ in range(ring)]
    d_nrm = [torch.from_numpy(nrm).cuda() for _ in range(ring)]
    d_alb, d_dir, d_emi = ([torch.rand((n, 3), device="cuda") for _ in range(ring)] for _ in range(3))
    d_e = [torch.empty((n, 3), device="cuda") for _ in range(ring)]
    d_out = [torch.empty((n, 3), device="cuda") for _ in range(ring)]
    img = lambda t: t.view(H_PX, W_PX, 3)

    def two_pass_image(k):
        model.infer_image(d_pos[k], d_nrm[k], d_e[k], W_PX, H_PX, param=param)
        niv.compose(img(d_e[k]), img(d_alb[k]), img(d_out[k]), img(d_dir[k]), img(d_emi[k]))

    def two_pass_linear(k):
        model.infer(d_pos[k], d_nrm[k], d_e[k], param=param)
        niv.compose(img(d_e[k]), img(d_alb[k]), img(d_out[k]), img(d_dir[k]), img(d_emi[k]))

    def fused(k):
        model.infer_shade(d_pos[k], d_nrm[k], d_alb[k], d_out[k], n, direct=d_dir[k], emission=d_emi[k], param=param)

    def fused_image(k):
        model.infer_shade(d_pos[k], d_nrm[k], d_alb[k], d_out[k], n, direct=d_dir[k], emission=d_emi[k], param=param,
                          image=(W_PX, H_PX))

    def infer_only(k):
        model.infer(d_pos[k], d_nrm[k], d_e[k], param=param)

    steps, warm = args.steps or 100, max(3, args.warmup or 5)
    res = {}
    for name, fn in (("niv_infer_image + niv_compose", two_pass_image), ("niv_infer + niv_compose", two_pass_linear),
                     ("niv_infer_shade", fused), ("niv_infer_image_shade", fused_image), ("niv_infer", infer_only)):
        for k in range(warm):
            fn(k % ring)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for k in range(steps):
            fn(k % ring)
        e1.record()
        torch.cuda.synchronize()
        res[name] = e0.elapsed_time(e1) / steps
    # same bits from both paths (fp32 output)
    two_pass_linear(0)
    ref = d_out[0].clone()
    fused(0)
    torch.cuda.synchronize()
    same = bool(torch.equal(ref, d_out[0]))
    fused_image(0)
    torch.cuda.synchronize()
    same = same and bool(torch.equal(ref, d_out[0]))
    print(json.dumps({"op": "shade", "workload": desc, "frame": "%dx%d" % (W_PX, H_PX), "steps": steps, "ms_per_frame": res,
                      "fused_equals_two_pass_bitwise": same,
                      "hbm_bytes_per_texel": {"two_pass": 24 + 12 + 12 + 36 + 12, "fused": 24 + 36 + 12}}), flush=True)
    model.close()


def run_dry(args):
    """--dry: the multi-rank plumbing of run_ours WITHOUT a GPU (gloo): self-launch, one broadcast per parameter blob from
    rank 0, the weak / strong split, max-over-ranks timing, one JSON line from rank 0.  The "step" is a checksum of the
    rank's slice and of the received parameters (no kernel, no oracle): for the world-size-2 CPU test of the launcher."""
    import torch
    import torch.distributed as dist
    rank, world, local = D.env_rank_world()
    if world > 1:
        dist.init_process_group("gloo")
    spec = I.spec_tiny()
    strong = args.scaling == "strong" and world > 1
    w_px, h_px = 64, 64
    g = I.make_gbuffer(w_px, h_px, 0, frame=0 if strong else D.frame_of_rank(rank, world)[0])
    pos, nrm = g["pos"], g["nrm"]
    n_job = pos.shape[0] * (1 if strong else world)
    if strong:
        r0, r1 = D.row_range_of_rank(h_px, rank, world)
        pos, nrm = pos[r0 * w_px:r1 * w_px], nrm[r0 * w_px:r1 * w_px]
    table = wb = bb = None
    if rank == 0:
        table = I.make_table(spec, 0)
        w, b = I.make_mlp(spec, 0)
        wb, bb = I.pack_weights(w), I.pack_biases(b)
    wl = spec.in_dim * spec.hidden_width + 3 * spec.hidden_width
    shapes = [((spec.n_levels * spec.table_size * spec.n_features,), torch.float16), ((wl,), torch.float16),
              ((spec.hidden_width + 3,), torch.float32)]
    t_table, t_w, t_b = D.broadcast_params([table, wb, bb] if rank == 0 else None, shapes, "cpu")
    check = float(t_table.double().sum() + t_w.double().sum() + t_b.double().sum())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        local_sum = float(np.abs(pos).sum() + np.abs(nrm).sum())
    ms = (time.perf_counter() - t0) * 1e3 / max(args.steps, 1) + 1e-6
    ms_max = D.reduce_max(ms)
    checks = [None] * world
    if world > 1:
        dist.all_gather_object(checks, (check, pos.shape[0], local_sum))
    else:
        checks = [(check, pos.shape[0], local_sum)]
    if rank == 0:
        print(json.dumps({"dry": True, "metric": METRIC, "value": n_job / (ms_max * 1e-3) / 1e9, "unit": UNIT, "n_gpus": world,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max, "higher_is_better": True,
                          "scaling": "strong" if strong else "weak", "texels_per_rank": [c[1] for c in checks],
                          "param_checksums": [c[0] for c in checks], "texels_per_step": n_job}))
    if world > 1:
        dist.destroy_process_group()


def self_launch(args):
    """python bench.py --gpus N (N > 1) outside torchrun: start N ranks of this script on this node, one per GPU."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = D.launcher_command(args.gpus, port, os.path.abspath(__file__), sys.argv[1:])
    raise SystemExit(subprocess.run(cmd).returncode)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: one frame per rank (weak) or the row blocks of ONE frame (strong, SURVEY 8(e))")
    ap.add_argument("--dry", action="store_true", help="multi-rank plumbing only, on the CPU over gloo (for the launcher test)")
    ap.add_argument("--workload", default="fullhd", choices=["fullhd", "incoherent", "param", "paper", "probes"])
    ap.add_argument("--probe-spacing", type=float, default=0.16, help="workload probes: probe spacing in metres (0.16 m = "
                    "the 5.4 MB budget of PAPER.md:462 in the 10 x 4 x 10 m room)")
    ap.add_argument("--paper-levels", type=int, default=8, choices=[0, 2, 4, 6, 8], help="workload paper: grid levels (0 = none)")
    ap.add_argument("--paper-width", type=int, default=64, choices=[16, 32, 64])
    ap.add_argument("--paper-dir-bands", type=int, default=0, choices=[0, 4],
                    help="workload paper: frequency bands per axis on top of the raw direction (grid models, width 64)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cold-steps", type=int, default=10, help="launches of the cold-L2 variant (0 = skip)")
    ap.add_argument("--no-compact-e2e", action="store_true", help="skip the end-to-end legs on the compact G-buffer formats")
    ap.add_argument("--shade", action="store_true", help="SURVEY 8(f2): niv_infer_shade against niv_infer + niv_compose")
    ap.add_argument("--compose", action="store_true", help="SURVEY 8(f2): time the compose kernel (HBM roofline)")
    ap.add_argument("--tiling", default="image", choices=["image", "linear"],
                    help="device path of the G-buffer workloads: niv_infer_image (default) or niv_infer")
    ap.add_argument("--texel-params", action="store_true",
                    help="--workload param only: time niv_infer_texel_params (one scene parameter value per texel, SURVEY 8 f3)")
    ap.add_argument("--half", action="store_true", help="quarter pixel count: a 960x540 G-buffer (PAPER.md:405, Table 1 'half')")
    ap.add_argument("--encode", action="store_true", help="time the stand-alone encoding kernel (north_star (2))")
    ap.add_argument("--probe-patterns", action="store_true", help="niv_probe_gather in all patterns x three buffer sizes")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json configs[4]: table-size / width / resolution sweep")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle wall time for cpu_baseline")
    ap.add_argument("--ref-sample", type=int, default=131072, help="texels per step of the reference arm")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:           # not under torchrun: start the ranks ourselves
        self_launch(args)
    if args.dry:
        args.steps = 3 if args.steps is None else args.steps
        args.warmup = 0 if args.warmup is None else args.warmup
        run_dry(args)
        return
    global PAPER_LEVELS, PAPER_WIDTH, PAPER_DIR_BANDS
    PAPER_LEVELS, PAPER_WIDTH, PAPER_DIR_BANDS = args.paper_levels, args.paper_width, args.paper_dir_bands
    if args.probe_patterns:
        run_probe_patterns(args)
        return
    if args.encode:
        run_encode(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.shade:
        run_shade(args)
        return
    if args.compose:
        run_compose(args)
        return
    if args.half:
        global W_PX, H_PX, N_TEXELS, METRIC
        W_PX, H_PX = 960, 540
        N_TEXELS = W_PX * H_PX
        METRIC = "NIV fused inference throughput on a 960x540 (half-resolution) G-buffer (ms_per_step = ms per frame)"
    if args.impl == "reference":
        args.steps = 5 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 200 if args.steps is None else args.steps
        args.warmup = 20 if args.warmup is None else max(args.warmup, 3)
        if args.workload == "probes":
            run_probes(args)
        else:
            run_ours(args)


if __name__ == "__main__":
    main()
