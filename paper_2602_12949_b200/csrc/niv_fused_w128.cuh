// niv_fused_w128.cuh -- fused encode + MLP for hidden width 128 (BASELINE.json configs[4] sweep), A operand in TMEM.
// Included by niv.cu after the v2 kernel, whose structure it follows (dynamic tiles, G-buffer prefetch, batched
// gathers, packed-fp16 blend, biases in the MMA, prepared descriptors).
//
// Width 128 does not fit the v2 column plan (D 128 + A 64 + ones 8 = 200 -> 256 columns -> two CTAs per SM).  Here a
// hidden layer is computed as TWO N = 64 halves into the same 64 accumulator columns:
//     TMEM (128 columns per CTA):  D [0, 64) fp32  |  A [64, 128) = K up to 128 packed fp16 pairs
//     half h: MMAs over all K-steps with the B rows [64h, 64h + 64) -> D; epilogue keeps the 32 packed words in
//     registers; after the second half (which still reads A) the 64 words go to the A columns.
// The "ones" A operand of the bias K-step lives in shared memory (4 KB, SS-form MMA).  128 columns and 62 KB of
// shared memory per CTA -> three CTAs (12 warps) per SM instead of two with the A tile in shared memory.
#pragma once
#include <type_traits>

namespace niv {

template <int L, int NB>
__global__ void __launch_bounds__(kTile, 3) niv_fused_w128_kernel(const __grid_constant__ KParams P,
                                                               const float* __restrict__ pos,
                                                               const float* __restrict__ nrm,
                                                               float* __restrict__ out, size_t n, uint32_t n_tiles)
{
    constexpr int WIDTH = 128, F = 2;
    constexpr uint32_t TMEM_COLS = 128, A_COL = 64;
    constexpr int NG = L / NB;
    constexpr int HW = L * F / 2;
    constexpr int AW = (HW + 8 + 7) / 8 * 8;          // 32-bit words of one layer-1 A row (K1 = 2 * AW)
    constexpr uint32_t K1 = 2 * AW;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* sW = smem;
    uint8_t* sOnes = smem + P.ones_off;               // [2][128 rows][16 B]
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + P.misc_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);
    uint32_t* s_tile = tmem_slot + 1;

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
    if (warp == 0) tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
    auto next_tile = [&](uint32_t after) -> uint32_t {     // NULL counter = static striding (niv_fused.cuh)
        return P.tile_ctr ? gridDim.x + atomicAdd(P.tile_ctr, 1u) : after + gridDim.x;
    };
    if (tid == 0) s_tile[0] = next_tile(blockIdx.x);
    *reinterpret_cast<uint4*>(sOnes + tid * 16) = make_uint4(0x3C003C00u, 0u, 0u, 0u);      // fp16 (1, 1, 0, ...)
    *reinterpret_cast<uint4*>(sOnes + 2048 + tid * 16) = make_uint4(0u, 0u, 0u, 0u);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_taddr = tmem + ((warp * 32u) << 16);
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_w, P.wpack_bytes);
        bulk_g2s(sW_u32, P.wpack, P.wpack_bytes, bar_w);
    }
    mbar_wait(bar_w, 0);

    // ---- a8: fold the per-call parameter encoding into layer 1's bias K-row (hi, lo) in shared memory
    if (P.n_params != 0 && tid < WIDTH) {
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
        *reinterpret_cast<uint32_t*>(sW + P.w_off[0] + (K1 >> 3) * (WIDTH * 16u) + tid * 16u) = word;
    }
    fence_proxy_async_smem();          // ones chunk and bias row are read by the tensor core through the async proxy

    // B descriptors (low half) at K-step 0, row 0; LBO = N * 16 bytes.  A descriptor of the ones chunk.
    const uint32_t n_layers = P.n_layers;
    uint32_t desc_lo0[kMaxLayers];
#pragma unroll
    for (int l = 0; l < kMaxLayers; ++l) {
        const uint32_t N = (l + 1 == (int)n_layers) ? 16u : (uint32_t)WIDTH;
        desc_lo0[l] = (((sW_u32 + P.w_off[l]) & 0x3FFFFu) >> 4) | (N << 16);
    }
    const uint64_t desc_ones = make_smem_desc(smem_u32(sOnes), 2048u, 128u);

    // MMAs of one layer (or of one 64-column half of a hidden layer) into D; issued by one elected lane of warp 0
    // after a CTA barrier.  KSTEPS is a compile-time constant so that the K loop unrolls into back-to-back UTCHMMAs.
    auto issue = [&](int layer, auto ksteps_c, uint32_t n_mma, uint32_t row0) {
        constexpr uint32_t KSTEPS = decltype(ksteps_c)::value;
        if (warp == 0 && elect_one_sync()) {
            tc_fence_after_sync();
            const uint32_t N = (layer + 1 == (int)n_layers) ? 16u : (uint32_t)WIDTH;   // rows of the packed B
            const uint32_t idesc = make_idesc_f16(kTile, n_mma);
            const uint32_t lo = desc_lo0[layer] + row0, step = 2u * N;                // row0 rows x 16 B >> 4
#pragma unroll
            for (uint32_t ks = 0; ks < KSTEPS; ++ks)
                umma_f16_ts2(tmem, tmem + A_COL + ks * 8u, lo + ks * step, 0x4008u, idesc, ks > 0 ? 1u : 0u);
            const uint64_t db = ((uint64_t)0x4008u << 32) | (uint64_t)(lo + KSTEPS * step);
            umma_f16_ss(tmem, desc_ones, db, idesc, 1u);                               // + bias
            umma_commit(bar_mma);
        }
    };
    using KS1 = std::integral_constant<uint32_t, K1 / 16>;
    using KSH = std::integral_constant<uint32_t, WIDTH / 16>;

    uint32_t phase = 0;
    float pn[3] = {0.f, 0.f, 0.f}, nn[3] = {0.f, 0.f, 0.f};
    if ((size_t)blockIdx.x * kTile + tid < n) {
        load3(pos, (size_t)blockIdx.x * kTile + tid, pn);
        load3(nrm, (size_t)blockIdx.x * kTile + tid, nn);
    }
    uint32_t tile = blockIdx.x, tnext = s_tile[0], it = 0;
    while (tile < n_tiles) {
        const size_t i = (size_t)tile * kTile + tid;
        const bool valid = i < n;
        const float p[3] = {pn[0], pn[1], pn[2]}, nv[3] = {nn[0], nn[1], nn[2]};
        uint32_t tnn_mine = 0;
        if (tid == 0) tnn_mine = next_tile(tnext);
        {
            const size_t inext = (size_t)tnext * kTile + tid;
#pragma unroll
            for (int d = 0; d < 3; ++d) { pn[d] = 0.f; nn[d] = 0.f; }
            if (inext < n) {
                load3(pos, inext, pn);
                load3(nrm, inext, nn);
            }
        }
        const bool masked = !valid || texel_masked(p, nv);

        uint32_t a[AW];
#pragma unroll
        for (int k = 0; k < AW; ++k) a[k] = 0u;
        if (!masked) {
            float u[3];
            normalise(P, p, u);
            Batch<NB, F> ba, bb;
            batch_issue<NB, F>(P, 0, u, ba);
            float sh[16];
            sh16(nv, sh);
#pragma unroll
            for (int k = 0; k < 8; ++k) a[HW + k] = pack_half2(sh[2 * k], sh[2 * k + 1]);
#pragma unroll
            for (int g = 0; g < NG; g += 2) {
                if (g + 1 < NG) batch_issue<NB, F>(P, (g + 1) * NB, u, bb);
                batch_blend<NB, F>(ba, a + g * NB);
                if (g + 2 < NG) batch_issue<NB, F>(P, (g + 2) * NB, u, ba);
                if (g + 1 < NG) batch_blend<NB, F>(bb, a + (g + 1) * NB);
            }
        }
        __syncwarp();
        tmem_st_x16(lane_taddr + A_COL, a);
        if constexpr (AW == 24) tmem_st_x8(lane_taddr + A_COL + 16, a + 16);
        tmem_st_wait();
        if (tid == 0) s_tile[(it + 1) & 1] = tnn_mine;
        tc_fence_before_sync();
        __syncthreads();
        const uint32_t tnn = s_tile[(it + 1) & 1];

#pragma unroll
        for (int layer = 0; layer < kMaxLayers; ++layer) {
            if (layer >= (int)n_layers) break;
            if (layer + 1 < (int)n_layers) {
                uint32_t pk[64];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (layer == 0) issue(layer, KS1{}, 64u, 64u * h);
                    else issue(layer, KSH{}, 64u, 64u * h);
                    mbar_wait(bar_mma, phase);
                    phase ^= 1u;
                    tc_fence_after_sync();
                    uint32_t r0[32], r1[32];
                    tmem_ld_x32(lane_taddr, r0);
                    tmem_ld_x32(lane_taddr + 32, r1);
                    tmem_ld_wait();
#pragma unroll
                    for (int q = 0; q < 16; ++q) {
                        pk[h * 32 + q] = pack_relu_half2(__uint_as_float(r0[2 * q]), __uint_as_float(r0[2 * q + 1]));
                        pk[h * 32 + 16 + q] = pack_relu_half2(__uint_as_float(r1[2 * q]), __uint_as_float(r1[2 * q + 1]));
                    }
                    if (h == 0) {                     // D is about to be overwritten by the second half
                        tc_fence_before_sync();
                        __syncthreads();
                    }
                }
                // both halves done: the MMAs no longer read A
#pragma unroll
                for (int c4 = 0; c4 < 4; ++c4) tmem_st_x16(lane_taddr + A_COL + c4 * 16, pk + c4 * 16);
                tmem_st_wait();
                tc_fence_before_sync();
                __syncthreads();
            } else {
                if (layer == 0) issue(layer, KS1{}, 16u, 0u);
                else issue(layer, KSH{}, 16u, 0u);
                mbar_wait(bar_mma, phase);
                phase ^= 1u;
                tc_fence_after_sync();
                uint32_t r[4];
                tmem_ld_x4(lane_taddr, r);
                tmem_ld_wait();
                tc_fence_before_sync();
                if (valid) {
                    float y[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float v = __uint_as_float(r[c]);
                        if (P.out_act == NIV_OUT_SIGMOID) v = __fdividef(1.0f, 1.0f + __expf(-v));
                        y[c] = masked ? 0.0f : v;
                    }
                    out[3 * i] = y[0];
                    out[3 * i + 1] = y[1];
                    out[3 * i + 2] = y[2];
                }
            }
        }
        tile = tnext;
        tnext = tnn;
        ++it;
    }

    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, TMEM_COLS);
    if (tid == 0 && P.tile_ctr) {   // the last CTA to finish leaves the (tile, done) counter pair zero and reports the slot free
        __threadfence();
        if (atomicAdd(P.tile_ctr + 1, 1u) == gridDim.x - 1) {
            P.tile_ctr[0] = 0u;
            P.tile_ctr[1] = 0u;
            if (P.slot_done) *P.slot_done = P.slot_gen;
        }
    }
}

}  // namespace niv
