// niv_fused.cuh -- the fused encode + MLP kernel (rows a0..a12 of DESIGN.md section 1), hidden width <= 64.
// Included by niv.cu.
//
//   persistent CTAs of 128 threads, thread t owns texel t of a 128-texel tile (= MMA row t = TMEM lane t);
//   weights staged once per CTA with one bulk async copy (TMA engine); the gathers of two batches of NB levels are
//   in flight per thread while the previous batch is blended (packed fp16); every layer is a series of tcgen05.mma
//   (M = 128, kind::f16, fp32 accumulators AND the fp16 A operand in tensor memory, biases as one extra K-step);
//   activations never leave the SM.
// TMEM columns per CTA (128 allocated): D [0, WIDTH) fp32 | A [64, 96) packed fp16 pairs | ones [96, 104).
// NPT > 0: every texel carries its own NPT scene parameters (P.tparam [n][NPT]); their sin/cos encoding
// becomes 16 * NPT more columns of the layer-1 A row (K1 grows by one K-step per parameter) instead of the per-call
// fold into the bias row.  TMEM columns then: A [64, 96 + 8 (NPT - 1)), ones behind it.
// IMG (niv_infer_image): texels are addressed as 8 x 4 pixel blocks per warp of a row-major image (image_texel).
// OUT128 (niv_infer_host): the output leaves as 128-bit stores through shared memory (buffers in pinned host memory).
#pragma once
#include <type_traits>

namespace niv {

constexpr float kInvPi = 0.318309886183790671538f;

__device__ __forceinline__ uint32_t pack_relu_half2(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}

// width 32 with 16 levels would take 130 registers (3 CTAs per SM): capped at 128; width 64 is left alone, the cap
// changes its schedule for the worse (0.193 instead of 0.189 ms, profiles/r01_v2.md); the per-texel-parameter
// variants are capped too (two parameters at width 64 would take 140 registers)
// NC: the coarsest NC levels are read from their cell-block copies, one 32- / 64-byte load per level
// PACKED: the caller's buffers are in one of the compact G-buffer / output formats (P.gbuf_fmt, P.out_fmt: a uniform
// run-time switch per tile); false = fp32 x 3 in and out with no trace of the switch in the code (it cost the headline
// kernel 1.5 %: its level loop sits at the register cap and every live value more changes the schedule)
// DIRB (RAWDIR only): bands of frequency encoding appended to the raw direction: the row holds
// the 3 + 6 DIRB direction values in consecutive fp16 pairs, the column order of W1
// OS (ones in shared memory): the (1, 1, 0, ...) A operand of the bias K-step is a 4 KB shared-memory tile read by an
// SS-form MMA (as in niv_fused_w128.cuh) instead of 8 tensor-memory columns, so a tile needs D + A columns only:
//   width 64: D [0, 64) and A [0, 32) in TWO allocations (64 + 32 = 96 columns: five CTAs per SM instead of four)
//   width 32: D [0, 32) | A [32, 64) in one allocation of 64 (eight CTAs per SM)
// For the kernels whose registers allow that many CTAs: the paper's family (F = 4) and its grid-less models.
template <int WIDTH, int L, int NB, int F, bool RAWDIR, bool OUT128, int NPT, bool IMG, int NC, bool PACKED, int DIRB = 0,
          bool OS = false>
__global__ void __launch_bounds__(kTile, (WIDTH == 32 || NPT >= 1) ? 4 : 0) niv_fused_kernel(
                                                               const __grid_constant__ KParams P,
                                                               const float* __restrict__ pos,
                                                               const float* __restrict__ nrm,
                                                               float* __restrict__ out, size_t n, uint32_t n_tiles)
{
    static_assert(WIDTH <= 64, "A-in-TMEM kernel: D + A + ones must fit 128 columns");
    static_assert(NC <= L, "cell-block levels are the leading levels");
    // width 16 (the paper's smallest grid-less model): D 16 | A 32 | ones 8 fit 64 columns -> eight CTAs per SM
    static_assert(!OS || ((WIDTH == 32 || WIDTH == 64) && NPT == 0), "ones in shared memory: width 32 / 64, no per-texel parameters");
    constexpr bool OS64 = OS && WIDTH == 64;          // A in a second allocation of 32 columns
    constexpr uint32_t TMEM_COLS = (OS || WIDTH == 16) ? 64 : 128, A_COL = OS64 ? 0 : OS ? 32 : WIDTH == 16 ? 16 : 64,
                       ONES_COL = OS ? A_COL + 32 : WIDTH == 16 ? 48 : NPT == 2 ? 104 : 96;
    constexpr int NG = L / NB;
    constexpr int HW = L ? L * F / 2 : 24;            // 32-bit words of hash latents in one A row (L = 0: the
                                                      // 3 x 8 (sin, cos) pairs of the positional encoding)
    static_assert(DIRB == 0 || RAWDIR, "frequency bands ride on the raw direction");
    constexpr int DW = RAWDIR ? (3 + 6 * DIRB + 1) / 2 : 8;   // ... of the direction input: (x, y | z, 0) [+ bands] or SH-16
    constexpr int AW = (HW + DW + 7) / 8 * 8;         // ... of the position + direction part of a layer-1 A row
    constexpr int AWT = AW + 8 * NPT;                 // ... of the whole row (K1 = 2 * AWT)
    static_assert(AWT <= 40 && A_COL + AWT <= ONES_COL, "layer-1 A row must end before the ones chunk (OS: fit the A columns)");
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* sW = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + P.misc_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);
    uint32_t* s_tile = tmem_slot + 1;                 // [2]: the tile after next, handed from thread 0 to the CTA
    uint32_t* s_txy = s_tile + 2;                     // [2]: IMG: its (tile column | tile row << 16)
    uint32_t* tmem_slot2 = s_txy + 2;                 // OS64: the A allocation
    uint8_t* sOnes = smem + P.ones_off;               // OS: [2][128 rows][16 B], K columns 0..7 | 8..15 of the ones tile

    const uint32_t tid = threadIdx.x;
    const uint32_t warp = tid >> 5;
    const uint32_t bar_w = smem_u32(&bars[0]);
    const uint32_t bar_mma = smem_u32(&bars[1]);
    const uint32_t sW_u32 = smem_u32(sW);

    if (tid == 0) {
        mbar_init(bar_w, 1);
        mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    // G-buffer texel of the first tile.  Requested here, ahead of everything, when the host found that no launch that
    // may still be running writes this launch's inputs (P.early_read); otherwise after the waits below.  Inside the loop
    // the NEXT tile's texel is requested a tile ahead, so its HBM latency hides under a whole tile of work (a1 prefetch)
    float pn[3] = {0.f, 0.f, 0.f}, nn[3] = {0.f, 0.f, 0.f};
    float tn[NPT > 0 ? NPT : 1] = {0.f};              // per-texel scene parameters, prefetched like the G-buffer
    // texel of thread tid in tile t: 128 consecutive texels per tile, or (IMG) a 32 x 4 pixel tile of the image
    //   (txy: the tile's packed image coordinates, which thread 0 works out with the tile index; unused otherwise)
    auto texel_of = [&](uint32_t t, uint32_t txy, bool& ok) -> size_t {
        if constexpr (IMG) return image_texel_xy(P, txy, tid, ok);
        const size_t idx = (size_t)t * kTile + tid;
        ok = idx < n;
        return idx;
    };
    uint32_t txy = 0, txy_next = 0;
    if constexpr (IMG) txy = image_tile_xy(P, blockIdx.x);
    auto load_first_texel = [&]() {
        bool ok;
        const size_t i0 = texel_of(blockIdx.x, txy, ok);
        if (ok) {
            load_texel_raw(PACKED ? P.gbuf_fmt : 0u, pos, nrm, i0, pn, nn);
#pragma unroll
            for (int q = 0; q < NPT; ++q) tn[q] = __ldg(P.tparam + i0 * NPT + q);
        }
    };
    if (P.early_read) load_first_texel();
    if (warp == 0) {
        if constexpr (OS64) {
            tmem_alloc_keep(smem_u32(tmem_slot), 64);
            tmem_alloc_keep(smem_u32(tmem_slot2), 32);
            tmem_relinquish();
        } else {
            tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
        }
    }
    if constexpr (OS) {                               // the bias K-step's A operand: (1, 1, 0, ..., 0) in every row
        *reinterpret_cast<uint4*>(sOnes + tid * 16) = make_uint4(0x3C003C00u, 0u, 0u, 0u);
        *reinterpret_cast<uint4*>(sOnes + 2048 + tid * 16) = make_uint4(0u, 0u, 0u, 0u);
    }
    // dynamic tile scheduling: tile blockIdx.x is static, every further tile comes from a global counter, so a CTA
    // that drew cheap (background) tiles or a fast SM simply draws more of them and the grid drains together
    auto next_tile = [&](uint32_t after) -> uint32_t {
        return P.tile_ctr ? gridDim.x + atomicAdd(P.tile_ctr, 1u) : after + gridDim.x;
    };
    if (tid == 0) {
        const uint32_t t1 = next_tile(blockIdx.x);
        s_tile[0] = t1;
        if constexpr (IMG) s_txy[0] = image_tile_xy(P, t1);
    }
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_taddr = tmem + ((warp * 32u) << 16);
    uint32_t tmem_a = tmem + A_COL;                   // first column of the A operand
    if constexpr (OS64) tmem_a = *tmem_slot2;
    const uint32_t lane_a = tmem_a + ((warp * 32u) << 16);
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_w, P.wpack_bytes);
        bulk_g2s(sW_u32, P.wpack, P.wpack_bytes, bar_w);
    }
    if constexpr (!OS) {   // the bias K-step's A operand: (1, 1, 0, ..., 0) in every row, written once
        uint32_t ones[8] = {0x3C003C00u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
        tmem_st_x8(lane_taddr + ONES_COL, ones);
    }
    const uint64_t desc_ones = make_smem_desc(smem_u32(sOnes), 2048u, 128u);
    // shared-memory descriptor (low half) of every layer's B operand at K-step 0: (address >> 4) | (N * 16 >> 4) << 16,
    // the high half is the constant 0x4008 = SBO 128 B >> 4 | descriptor version 1 << 14 (niv_tc.cuh make_smem_desc)
    constexpr uint32_t K1 = 2 * AWT;
    const uint32_t n_layers = P.n_layers;
    uint32_t desc_lo0[kMaxLayers];
#pragma unroll
    for (int l = 0; l < kMaxLayers; ++l) {
        const uint32_t N = (l + 1 == (int)n_layers) ? 16u : (uint32_t)WIDTH;
        desc_lo0[l] = (((sW_u32 + P.w_off[l]) & 0x3FFFFu) >> 4) | (N << 16);
    }
    uint32_t phase = 0;
    // Programmatic dependent launch (launch_fused sets the stream-serialisation attribute): everything above touches
    // only the model's own memory, so this launch's CTAs may take the place of the previous launch's as those drain,
    // with TMEM allocated and weights staged; from here on the caller's buffers are read and written, which needs the
    // previous kernel of the stream complete.  The next launch may start filling in behind this one right away.
    if (P.grid_wait) pdl_wait();
    if (P.wait_a) {                    // launches two and three back: complete before this one touches a buffer
        if (tid == 0) {                // (both words requested before either is looked at)
            uint32_t va = ld_acquire_gpu(P.wait_a), vb = P.wait_b ? ld_acquire_gpu(P.wait_b) : P.gen_b;
            while ((int32_t)(va - P.gen_a) < 0) { __nanosleep(64); va = ld_acquire_gpu(P.wait_a); }
            while ((int32_t)(vb - P.gen_b) < 0) { __nanosleep(64); vb = ld_acquire_gpu(P.wait_b); }
        }
        __syncthreads();
    }
    // only now may the NEXT launch's CTAs be scheduled: when one of them starts, every CTA of this launch has passed the
    // waits above, so the launches two and more before THIS one are complete -- which is what lets the next launch
    // request its first texel at once (P.early_read: the host has checked this launch and the one before it)
    pdl_launch_dependents();
    if constexpr (IMG) txy_next = s_txy[0];
    if (!P.early_read) load_first_texel();
    // the weights are waited for only now: their copy (issued in the prologue) and the first texel's trip from HBM overlap
    mbar_wait(bar_w, 0);

    // ---- a8: fold the per-call parameter encoding into layer 1's bias K-row (hi, lo) in shared memory
    if (NPT == 0 && P.n_params != 0 && tid < WIDTH) {
        float b = reinterpret_cast<const float*>(sW + P.b_off[0])[tid];
        const uint32_t np16 = 16 * P.n_params;
        for (uint32_t q = 0; q < P.n_params; ++q) {
            float enc[16];
            param_encode8(P.t[q], enc);
            const float* wp = reinterpret_cast<const float*>(sW + P.wparam_off) + tid * np16 + 16 * q;
#pragma unroll
            for (int k = 0; k < 16; ++k) b = fmaf(wp[k], enc[k], b);
        }
        const __half hi = __float2half_rn(b);
        const __half lo = __float2half_rn(b - __half2float(hi));
        const uint32_t word = (uint32_t)__half_as_ushort(hi) | ((uint32_t)__half_as_ushort(lo) << 16);
        *reinterpret_cast<uint32_t*>(sW + P.w_off[0] + (P.kdim[0] >> 3) * (P.npad[0] * 16u) + tid * 16u) = word;
    }
    fence_proxy_async_smem();          // the bias row is read by the tensor core through the async proxy

    uint32_t tile = blockIdx.x, tnext = s_tile[0], it = 0;
    while (tile < n_tiles) {
        bool valid;
        const size_t i = texel_of(tile, txy, valid);
        float p[3] = {pn[0], pn[1], pn[2]}, nv[3] = {nn[0], nn[1], nn[2]};
        if constexpr (PACKED) decode_texel(P, pn, nn, p, nv);     // the raw words of a compact format -> fp32 position, normal
        float tv[NPT > 0 ? NPT : 1];
#pragma unroll
        for (int q = 0; q < NPT; ++q) tv[q] = tn[q];
        uint32_t tnn_mine = 0;
        uint32_t txy_mine = 0;
        if (tid == 0) {
            tnn_mine = next_tile(tnext);                                      // the tile after next
            if constexpr (IMG) txy_mine = image_tile_xy(P, tnn_mine);
        }
        // a1 prefetch: the next tile's texel is requested when this tile's A row is complete (below), so that it arrives
        // under the layers (three MMA round trips, ~1 us) and does not occupy six registers during the level loop
        auto prefetch_next = [&]() {
            bool ok;
            const size_t inext = texel_of(tnext, txy_next, ok);   // (a tile index past the end gives ok = false)
#pragma unroll
            for (int d = 0; d < 3; ++d) { pn[d] = 0.f; nn[d] = 0.f; }
            if (ok) {
                load_texel_raw(PACKED ? P.gbuf_fmt : 0u, pos, nrm, inext, pn, nn);
#pragma unroll
                for (int q = 0; q < NPT; ++q) tn[q] = __ldg(P.tparam + inext * NPT + q);
            }
        };
        const bool masked = !valid || texel_masked(p, nv);

        // ---- a2..a9: this thread's A row in registers.  Rows are independent in the GEMMs and masked rows are
        //      overwritten with zeros at the store, so a masked thread just passes zeros.
        uint32_t a[AWT];
#pragma unroll
        for (int k = 0; k < AWT; ++k) a[k] = 0u;
        if (!masked) {
            float u[3];
            normalise(P, p, u);
            auto encode_direction = [&]() {
                if constexpr (RAWDIR && DIRB > 0) {   // ... followed by its frequency encoding, axis after axis
                    float dv[2 * DW];
                    dv[0] = nv[0]; dv[1] = nv[1]; dv[2] = nv[2];
                    dv[2 * DW - 1] = 0.0f;
#pragma unroll
                    for (int d = 0; d < 3; ++d) dirfreq<DIRB>(nv[d], dv + 3 + 2 * DIRB * d);
#pragma unroll
                    for (int k = 0; k < DW; ++k) a[HW + k] = pack_half2(dv[2 * k], dv[2 * k + 1]);
                } else if (RAWDIR) {                  // the paper's model: the direction itself
                    a[HW] = pack_half2(nv[0], nv[1]);
                    a[HW + 1] = pack_half2(nv[2], 0.0f);
                } else {
                    float sh[16];
                    sh16(nv, sh);
#pragma unroll
                    for (int k = 0; k < 8; ++k) a[HW + k] = pack_half2(sh[2 * k], sh[2 * k + 1]);
                }
            };
            if constexpr (L == 0) {                   // grid-less models: eight-band positional encoding
                encode_direction();
#pragma unroll
                for (int d = 0; d < 3; ++d) posenc8_packed(u[d], a + 8 * d);
            } else {
                Batch<NB, F> ba, bb;
                batch_issue<NB, F, NC>(P, 0, u, ba);
#pragma unroll
                for (int g = 0; g < NG; g += 2) {
                    if (g + 1 < NG) batch_issue<NB, F, NC>(P, (g + 1) * NB, u, bb);
                    batch_blend<NB, F>(ba, a + g * NB * (F / 2));
                    if (g + 2 < NG) batch_issue<NB, F, NC>(P, (g + 2) * NB, u, ba);
                    if (g + 1 < NG) batch_blend<NB, F>(bb, a + (g + 1) * NB * (F / 2));
                }
                // the direction last: its 8 words (SH-16) would otherwise sit in registers through the whole level loop,
                // and so would the next tile's texel, which is requested only below (0.1512 -> 0.1478 ms per frame:
                // the level loop runs at the 128-register cap)
                encode_direction();
            }
            // a8 per texel: gamma(t) = (sin, cos)(2^k pi t), k = 0..7, as fp16 pairs
#pragma unroll
            for (int q = 0; q < NPT; ++q) param_encode8_packed(tv[q], a + AW + 8 * q);
        }
        if constexpr (PACKED) {                       // niv_debug_arow: the row as the tensor core will read it
            if (P.dump_a && valid) {
#pragma unroll
                for (int k = 0; k < AWT; ++k) P.dump_a[i * P.dump_words + k] = a[k];
            }
        }
        prefetch_next();
        // niv_infer_shade: this texel's albedo and direct + emission, requested here so that they arrive under the layers
        float sh_a[3] = {0.f, 0.f, 0.f}, sh_v[3] = {0.f, 0.f, 0.f};
        if constexpr (PACKED) {
            if (P.shade_albedo && valid) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    sh_a[c] = __ldcs(P.shade_albedo + 3 * i + c);
                    if (P.shade_direct) sh_v[c] = __ldcs(P.shade_direct + 3 * i + c);
                    if (P.shade_emission) sh_v[c] += __ldcs(P.shade_emission + 3 * i + c);
                }
            }
        }
        __syncwarp();
        if constexpr (AW == 8) tmem_st_x8(lane_a, a);
        else tmem_st_x16(lane_a, a);
        if constexpr (AW == 24) tmem_st_x8(lane_a + 16, a + 16);
        if constexpr (AW == 32) tmem_st_x16(lane_a + 16, a + 16);
        if constexpr (NPT >= 1) tmem_st_x8(lane_a + AW, a + AW);
        if constexpr (NPT == 2) tmem_st_x8(lane_a + AW + 8, a + AW + 8);
        tmem_st_wait();
        if (tid == 0) {
            s_tile[(it + 1) & 1] = tnn_mine;
            if constexpr (IMG) s_txy[(it + 1) & 1] = txy_mine;
        }
        tc_fence_before_sync();
        __syncthreads();
        const uint32_t tnn = s_tile[(it + 1) & 1];
        uint32_t txy_nn = 0;
        if constexpr (IMG) txy_nn = s_txy[(it + 1) & 1];

        // ---- a10..a12: the layers.  K depends on the layer's position only (compile time), N on whether it is the
        //      last one (run time, uniform); the descriptors are one add per K-step from values prepared before the
        //      tile loop, so the issuing thread's critical path is ~6 instructions per MMA.
#pragma unroll
        for (int layer = 0; layer < kMaxLayers; ++layer) {
            if (layer >= (int)n_layers) break;
            const bool last_layer = layer + 1 == (int)n_layers;
            const uint32_t ksteps_ct = layer == 0 ? K1 / 16 : WIDTH / 16;
            if (warp == 0 && elect_one_sync()) {
                tc_fence_after_sync();
                const uint32_t N = last_layer ? 16u : (uint32_t)WIDTH;
                const uint32_t idesc = make_idesc_f16(kTile, N);
                const uint32_t lo = desc_lo0[layer], step = 2u * N;
#pragma unroll
                for (uint32_t ks = 0; ks < ksteps_ct; ++ks)
                    umma_f16_ts2(tmem, tmem_a + ks * 8u, lo + ks * step, 0x4008u, idesc, ks > 0 ? 1u : 0u);
                if constexpr (OS)                                                                       // + bias
                    umma_f16_ss(tmem, desc_ones, ((uint64_t)0x4008u << 32) | (uint64_t)(lo + ksteps_ct * step), idesc, 1u);
                else
                    umma_f16_ts2(tmem, tmem + ONES_COL, lo + ksteps_ct * step, 0x4008u, idesc, 1u);
                umma_commit(bar_mma);
            }
            mbar_wait(bar_mma, phase);
            phase ^= 1u;
            tc_fence_after_sync();

            if (!last_layer) {
                // hidden epilogue: D (fp32) -> ReLU + fp16 pack -> A columns of the next layer
                if constexpr (WIDTH == 64) {          // both loads in flight, one wait
                    uint32_t r0[32], r1[32];
                    tmem_ld_x32(lane_taddr, r0);
                    tmem_ld_x32(lane_taddr + 32, r1);
                    tmem_ld_wait();
                    uint32_t pk[32];
#pragma unroll
                    for (int h = 0; h < 16; ++h) {
                        pk[h] = pack_relu_half2(__uint_as_float(r0[2 * h]), __uint_as_float(r0[2 * h + 1]));
                        pk[16 + h] = pack_relu_half2(__uint_as_float(r1[2 * h]), __uint_as_float(r1[2 * h + 1]));
                    }
                    tmem_st_x16(lane_a, pk);
                    tmem_st_x16(lane_a + 16, pk + 16);
                } else if constexpr (WIDTH == 32) {
                    uint32_t r[32];
                    tmem_ld_x32(lane_taddr, r);
                    tmem_ld_wait();
                    uint32_t pk[16];
#pragma unroll
                    for (int h = 0; h < 16; ++h)
                        pk[h] = pack_relu_half2(__uint_as_float(r[2 * h]), __uint_as_float(r[2 * h + 1]));
                    tmem_st_x16(lane_a, pk);
                } else {                              // width 16
                    uint32_t r[16];
                    tmem_ld_x16(lane_taddr, r);
                    tmem_ld_wait();
                    uint32_t pk[8];
#pragma unroll
                    for (int h = 0; h < 8; ++h)
                        pk[h] = pack_relu_half2(__uint_as_float(r[2 * h]), __uint_as_float(r[2 * h + 1]));
                    tmem_st_x8(lane_a, pk);
                }
                tmem_st_wait();
                tc_fence_before_sync();
                __syncthreads();
            } else {
                uint32_t r[4];
                tmem_ld_x4(lane_taddr, r);
                tmem_ld_wait();
                tc_fence_before_sync();
                if constexpr (OUT128) {
                    // a12 for buffers in pinned HOST memory (niv_infer_host, zero copy): the warp's 32 x 3 floats go
                    // through shared memory and leave as 24 aligned 128-bit stores = three full 128-byte lines, which
                    // cross PCIe as full-line writes (scalar 12-byte-stride stores take 2.9 ms per frame, these 0.49)
                    float y[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float v = __uint_as_float(r[c]);
                        if (P.out_act == NIV_OUT_SIGMOID) v = __fdividef(1.0f, 1.0f + __expf(-v));
                        y[c] = masked ? 0.0f : v;
                        if (PACKED && P.shade_albedo) y[c] = fmaf(sh_a[c] * kInvPi, y[c], sh_v[c]);
                    }
                    const uint32_t lane = tid & 31u;
                    float* so = reinterpret_cast<float*>(smem + P.misc_off + 64) + warp * 96;
                    const size_t w0 = ((size_t)tile * kTile + warp * 32u) * 3;        // first float of the warp
                    const bool vec = (w0 + 96 <= 3 * n) && ((reinterpret_cast<uintptr_t>(out) & 15u) == 0);
                    if (PACKED && P.out_fmt == NIV_OUTFMT_F16X4) {      // 8 bytes per texel: a warp's stores are 256 contiguous bytes
                        if (valid)
                            reinterpret_cast<uint2*>(out)[i] = make_uint2(pack_half2(y[0], y[1]), pack_half2(y[2], 0.0f));
                    } else if (PACKED && P.out_fmt == NIV_OUTFMT_RGB9E5) {   // 4 bytes per texel: one 128-byte line per warp
                        if (valid) reinterpret_cast<uint32_t*>(out)[i] = pack_rgb9e5(y[0], y[1], y[2]);
                    } else if (vec) {
                        so[lane * 3] = y[0];
                        so[lane * 3 + 1] = y[1];
                        so[lane * 3 + 2] = y[2];
                        __syncwarp();
                        if (lane < 24) *reinterpret_cast<float4*>(out + w0 + lane * 4) = *reinterpret_cast<const float4*>(so + lane * 4);
                        __syncwarp();
                    } else if (valid) {
                        out[3 * i] = y[0];
                        out[3 * i + 1] = y[1];
                        out[3 * i + 2] = y[2];
                    }
                } else if (valid) {
                    float y[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float v = __uint_as_float(r[c]);
                        if (P.out_act == NIV_OUT_SIGMOID) v = __fdividef(1.0f, 1.0f + __expf(-v));
                        y[c] = masked ? 0.0f : v;
                        if (PACKED && P.shade_albedo) y[c] = fmaf(sh_a[c] * kInvPi, y[c], sh_v[c]);   // Eq. 2, as niv_compose
                    }
                    if (PACKED && P.out_fmt == NIV_OUTFMT_F16X4) {      // (r, g, b, 0) as four fp16: one 8-byte store
                        reinterpret_cast<uint2*>(out)[i] = make_uint2(pack_half2(y[0], y[1]), pack_half2(y[2], 0.0f));
                    } else if (PACKED && P.out_fmt == NIV_OUTFMT_RGB9E5) {   // shared-exponent word: one 4-byte store
                        reinterpret_cast<uint32_t*>(out)[i] = pack_rgb9e5(y[0], y[1], y[2]);
                    } else {
                        out[3 * i] = y[0];
                        out[3 * i + 1] = y[1];
                        out[3 * i + 2] = y[2];
                    }
                }
            }
        }
        tile = tnext;
        tnext = tnn;
        if constexpr (IMG) { txy = txy_next; txy_next = txy_nn; }
        ++it;
    }

    __syncthreads();
    if (warp == 0) {
        tmem_dealloc(tmem, TMEM_COLS);
        if constexpr (OS64) tmem_dealloc(tmem_a, 32);
    }
    if (tid == 0 && P.tile_ctr) {   // the last CTA to finish leaves the (tile, done) counter pair zero and reports the slot free
        __threadfence();
        if (atomicAdd(P.tile_ctr + 1, 1u) == gridDim.x - 1) {
            P.tile_ctr[0] = 0u;
            P.tile_ctr[1] = 0u;
            __threadfence();
            st_release_gpu(P.tile_ctr + 2, P.slot_gen);        // "this launch is complete", for the launches after the next
            if (P.slot_done) *P.slot_done = P.slot_gen;
        }
    }
}

}  // namespace niv
