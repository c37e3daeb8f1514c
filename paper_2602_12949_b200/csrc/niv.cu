// niv.cu -- libniv: kernels and the C ABI declared in include/niv.h.
//
// Kernels (all sm_100a, hand-written):
//   niv_fused_tmem_kernel<WIDTH, L, NB>  rows a0..a12 of DESIGN.md section 1 (the default, WIDTH <= 64):
//                            persistent CTAs of 128 threads, one texel per thread, 128-texel tiles; weights
//                            staged once per CTA with a bulk async copy; gathers from the L2-resident table run
//                            NB levels ahead of the packed-fp16 blend; every layer is a tcgen05.mma (M = 128,
//                            kind::f16, fp32 accumulators AND the fp16 A operand in tensor memory, biases as
//                            one extra K-step); activations never leave the SM.
//   niv_fused_kernel<WIDTH, L, NB>       the same with the A operand in shared memory (WIDTH = 128, and A/B runs).
//   niv_encode_kernel        rows a1..a9 only (stand-alone encoding, fp16 features to global memory).
//   niv_debug_kernel         index / cell / fraction / fp32 feature dump through the same device functions.
//   niv_probe_gather_kernel  random-sector gather micro-benchmark (the measured L2-gather roofline).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <atomic>
#include <cmath>
#include <new>
#include <vector>

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "../../include/niv.h"
#include "niv_device.cuh"
#include "niv_tc.cuh"

namespace niv {

// =====================================================================================================
// fused encode + MLP, v1: specialised on <WIDTH, L>, level loop fully unrolled and software-pipelined
// =====================================================================================================
// Differences from the first kernel (v0, profiles/r01_v0_baseline.md: 2435 instructions per texel, a runtime
// level loop, fp32 blend, fp32 bias + ReLU epilogue):
//   * the level loop is unrolled (level constants become immediate constant-bank operands) and the gathers run
//     NB levels ahead of the blend, two batches in flight per thread;
//   * blend on packed half2 (blend8_h2): the result is directly the fp16 pair of the A operand;
//   * biases ride in the MMA: every layer gets one extra K-step whose A operand is a constant "ones" chunk
//     ([1, 1, 0, ...] per row, written once per CTA) and whose B rows are (bias_hi, bias_lo, 0, ...) in fp16,
//     bias_hi + bias_lo = the fp32 bias to 2^-22 relative; the hidden epilogue is then one
//     cvt.rn.relu.f16x2.f32 per two activations;
//   * the per-call parameter fold (a8) is written into layer 1's bias row in shared memory.
__device__ __forceinline__ uint32_t pack_relu_half2(float lo, float hi) {
    uint32_t d;
    asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}

template <int WIDTH, int L, int NB>
__global__ void __launch_bounds__(kTile) niv_fused_kernel(const __grid_constant__ KParams P,
                                                          const float* __restrict__ pos,
                                                          const float* __restrict__ nrm,
                                                          float* __restrict__ out, size_t n, uint32_t n_tiles)
{
    constexpr uint32_t TMEM_COLS = WIDTH < 32 ? 32 : WIDTH;
    constexpr int NG = L / NB;                        // gather batches per texel
    constexpr int HC = L / 4;                         // 16-byte chunks of hash latents
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* sW = smem;                                              // packed weights (+ bias K-rows)
    uint8_t* sA = smem + P.a_off;                                    // A operand: [K/8][128 rows][16 B]
    uint8_t* sOnes = smem + P.ones_off;                              // [2][128 rows][16 B]: the bias K-step's A
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + P.misc_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);

    const uint32_t tid = threadIdx.x;
    const uint32_t warp = tid >> 5;
    const uint32_t bar_w = smem_u32(&bars[0]);
    const uint32_t bar_mma = smem_u32(&bars[1]);
    const uint32_t sA_u32 = smem_u32(sA);
    const uint32_t sW_u32 = smem_u32(sW);
    const uint32_t sOnes_u32 = smem_u32(sOnes);

    // ---- a0: one-time setup: barriers, TMEM columns, weights, ones chunk
    if (tid == 0) {
        mbar_init(bar_w, 1);
        mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(smem_u32(tmem_slot), TMEM_COLS);
    *reinterpret_cast<uint4*>(sOnes + tid * 16) = make_uint4(0x3C003C00u, 0u, 0u, 0u);      // fp16 (1, 1, 0, ...)
    *reinterpret_cast<uint4*>(sOnes + 2048 + tid * 16) = make_uint4(0u, 0u, 0u, 0u);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_w, P.wpack_bytes);
        bulk_g2s(sW_u32, P.wpack, P.wpack_bytes, bar_w);
    }
    mbar_wait(bar_w, 0);

    // ---- a8: the parameter encoding is constant over the call: b1' = b1 + W1[:, enc_dim:] * enc(t), written as
    //      (hi, lo) fp16 into layer 1's bias K-row
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
        *reinterpret_cast<uint32_t*>(sW + P.w_off[0] + (P.kdim[0] >> 3) * (P.npad[0] * 16u) + tid * 16u) = word;
    }
    // (the first tile's fence + barrier below also publish the ones chunk and the bias row to the async proxy)

    const uint32_t lane_taddr = tmem + ((warp * 32u) << 16);
    const uint32_t k1_chunks = P.kdim[0] >> 3;
    uint32_t phase = 0;

    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const size_t i = (size_t)tile * kTile + tid;
        const bool valid = i < n;
        float p[3] = {0.f, 0.f, 0.f}, nv[3] = {0.f, 0.f, 0.f};
        if (valid) {
            load3(pos, i, p);
            load3(nrm, i, nv);
        }
        const bool masked = !valid || texel_masked(p, nv);

        // ---- a2..a9: encode this thread's texel into row `tid` of the A tile
        uint8_t* rowp = sA + tid * 16;
        if (!masked) {
            float u[3];
            normalise(P, p, u);
            uint32_t f[L];
            Batch<NB, 2> ba, bb;
            batch_issue<NB, 2>(P, 0, u, ba);
#pragma unroll
            for (int g = 0; g < NG; g += 2) {
                if (g + 1 < NG) batch_issue<NB, 2>(P, (g + 1) * NB, u, bb);
                batch_blend<NB, 2>(ba, f + g * NB);
                if (g + 2 < NG) batch_issue<NB, 2>(P, (g + 2) * NB, u, ba);
                if (g + 1 < NG) batch_blend<NB, 2>(bb, f + (g + 1) * NB);
            }
#pragma unroll
            for (int c = 0; c < HC; ++c)
                *reinterpret_cast<uint4*>(rowp + c * 2048) = make_uint4(f[4 * c], f[4 * c + 1], f[4 * c + 2], f[4 * c + 3]);
            float sh[16];
            sh16(nv, sh);
            *reinterpret_cast<uint4*>(rowp + (HC + 0) * 2048) =
                make_uint4(pack_half2(sh[0], sh[1]), pack_half2(sh[2], sh[3]), pack_half2(sh[4], sh[5]), pack_half2(sh[6], sh[7]));
            *reinterpret_cast<uint4*>(rowp + (HC + 1) * 2048) =
                make_uint4(pack_half2(sh[8], sh[9]), pack_half2(sh[10], sh[11]), pack_half2(sh[12], sh[13]), pack_half2(sh[14], sh[15]));
            if ((HC + 2) & 1)                                            // K padding up to a multiple of 16
                *reinterpret_cast<uint4*>(rowp + (HC + 2) * 2048) = make_uint4(0, 0, 0, 0);
        } else {
            for (uint32_t kc = 0; kc < k1_chunks; ++kc)
                *reinterpret_cast<uint4*>(rowp + kc * 2048) = make_uint4(0, 0, 0, 0);
        }
        fence_proxy_async_smem();
        tc_fence_before_sync();
        __syncthreads();

        // ---- a10..a11: layers on the tensor cores
        for (uint32_t layer = 0; layer < P.n_layers; ++layer) {
            const uint32_t K = P.kdim[layer], N = P.npad[layer];
            if (tid == 0) {
                tc_fence_after_sync();
                const uint32_t idesc = make_idesc_f16(kTile, N);
                const uint32_t b_base = sW_u32 + P.w_off[layer];
                const uint32_t ksteps = K >> 4;
                for (uint32_t ks = 0; ks < ksteps; ++ks) {
                    const uint64_t da = make_smem_desc(sA_u32 + ks * 4096u, 2048u, 128u);
                    const uint64_t db = make_smem_desc(b_base + ks * (N * 32u), N * 16u, 128u);
                    umma_f16_ss(tmem, da, db, idesc, ks > 0 ? 1u : 0u);
                }
                {   // + bias: ones chunk x (bias_hi, bias_lo) rows
                    const uint64_t da = make_smem_desc(sOnes_u32, 2048u, 128u);
                    const uint64_t db = make_smem_desc(b_base + ksteps * (N * 32u), N * 16u, 128u);
                    umma_f16_ss(tmem, da, db, idesc, 1u);
                }
                umma_commit(bar_mma);
            }
            mbar_wait(bar_mma, phase);
            phase ^= 1u;
            tc_fence_after_sync();

            if (layer + 1 < P.n_layers) {
                // hidden epilogue: ReLU + fp16 pack in one conversion -> next layer's A operand (same buffer)
#pragma unroll
                for (int cc = 0; cc < WIDTH / 32; ++cc) {
                    uint32_t r[32];
                    tmem_ld_x32(lane_taddr + cc * 32, r);
                    tmem_ld_wait();
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        uint32_t pk[4];
#pragma unroll
                        for (int h = 0; h < 4; ++h)
                            pk[h] = pack_relu_half2(__uint_as_float(r[g * 8 + h * 2]), __uint_as_float(r[g * 8 + h * 2 + 1]));
                        *reinterpret_cast<uint4*>(rowp + (cc * 4 + g) * 2048) = make_uint4(pk[0], pk[1], pk[2], pk[3]);
                    }
                }
                fence_proxy_async_smem();
                tc_fence_before_sync();
                __syncthreads();
            } else {
                // ---- a11..a12: output layer: 3 useful columns (bias already in), activation, store
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
    }

    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, TMEM_COLS);
}

// =====================================================================================================
// fused encode + MLP, v2: as v1, with the A operand of every layer in TENSOR MEMORY (WIDTH <= 64)
// =====================================================================================================
// profiles/r01_v1_nb4.md: v1 is bound by the L1TEX data pipe (69 % busy: 220 K gather wavefronts, 46 K
// shared-store wavefronts per SM) and its 43 KB of shared memory per CTA leave only ~50 KB of L1 per SM.
// Here thread t keeps row t of the A operand in TMEM lane t: tcgen05.st instead of STS (no L1TEX wavefronts,
// no generic->async proxy fence), tcgen05.mma reads A from TMEM, and shared memory holds the weights only.
// TMEM columns per CTA (128 allocated): D [0, WIDTH) fp32 | A [64, 96) packed fp16 pairs | ones [96, 104).
// NPT > 0: every texel carries its own NPT scene parameters (P.tparam [n][NPT]); their sin/cos encoding
// becomes 16 * NPT more columns of the layer-1 A row (K1 grows by one K-step per parameter) instead of the per-call
// fold into the bias row.  TMEM columns then: A [64, 96 + 8 (NPT - 1)), ones behind it.
// IMG (niv_infer_image): texels are addressed as 8 x 4 pixel blocks per warp of a row-major image (image_texel).
template <int WIDTH, int L, int NB, int F, bool RAWDIR, bool OUT128 = false, int NPT = 0, bool IMG = false>
#ifdef NIV_EXPERIMENT_V2_MINB          // timing experiment only: another register budget for the v2 kernel
__global__ void __launch_bounds__(kTile, NIV_EXPERIMENT_V2_MINB) niv_fused_tmem_kernel(
#else
// width 32 with 16 levels would take 130 registers (3 CTAs per SM): capped at 128; width 64 is left alone, the cap
// changes its schedule for the worse (0.193 instead of 0.189 ms, profiles/r01_v2.md); the per-texel-parameter
// variants are capped too (two parameters at width 64 would take 140 registers; with one the capped schedule is the
// faster one, 0.162 against 0.177 ms)
__global__ void __launch_bounds__(kTile, (WIDTH == 32 || NPT >= 1) ? 4 : 0) niv_fused_tmem_kernel(
#endif
                                                               const __grid_constant__ KParams P,
                                                               const float* __restrict__ pos,
                                                               const float* __restrict__ nrm,
                                                               float* __restrict__ out, size_t n, uint32_t n_tiles)
{
    static_assert(WIDTH <= 64, "A-in-TMEM kernel: D + A + ones must fit 128 columns");
    constexpr uint32_t TMEM_COLS = 128, A_COL = 64, ONES_COL = NPT == 2 ? 104 : 96;
    constexpr int NG = L / NB;
    constexpr int HW = L ? L * F / 2 : 24;            // 32-bit words of hash latents in one A row (L = 0: the
                                                      // 3 x 8 (sin, cos) pairs of the positional encoding)
    constexpr int DW = RAWDIR ? 2 : 8;                // ... of the direction input: (x, y | z, 0) or SH-16
    constexpr int AW = (HW + DW + 7) / 8 * 8;         // ... of the position + direction part of a layer-1 A row
    constexpr int AWT = AW + 8 * NPT;                 // ... of the whole row (K1 = 2 * AWT)
    static_assert(AWT <= 40 && A_COL + AWT <= ONES_COL, "layer-1 A row must end before the ones chunk");
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* sW = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + P.misc_off);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);
    uint32_t* s_tile = tmem_slot + 1;                 // [2]: the tile after next, handed from thread 0 to the CTA
    uint32_t* s_txy = s_tile + 2;                     // [2]: IMG: its (tile column | tile row << 16)

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
    // dynamic tile scheduling: tile blockIdx.x is static, every further tile comes from a global counter, so a CTA
    // that drew cheap (background) tiles or a fast SM simply draws more of them and the grid drains together
    if (tid == 0) {
        const uint32_t t1 = gridDim.x + atomicAdd(P.tile_ctr, 1u);
        s_tile[0] = t1;
        if constexpr (IMG) s_txy[0] = image_tile_xy(P, t1);
    }
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_taddr = tmem + ((warp * 32u) << 16);
    if (tid == 0) {
        mbar_arrive_expect_tx(bar_w, P.wpack_bytes);
        bulk_g2s(sW_u32, P.wpack, P.wpack_bytes, bar_w);
    }
    {   // the bias K-step's A operand: (1, 1, 0, ..., 0) in every row, written once
        uint32_t ones[8] = {0x3C003C00u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};
        tmem_st_x8(lane_taddr + ONES_COL, ones);
    }
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
    pdl_launch_dependents();
    pdl_wait();
    // G-buffer texel of the first tile; inside the loop the NEXT tile's texel is requested before the current
    // one is encoded, so its HBM latency hides under a whole tile of work (a1 prefetch)
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
    if constexpr (IMG) { txy = image_tile_xy(P, blockIdx.x); txy_next = s_txy[0]; }
    {
        bool ok;
        const size_t i0 = texel_of(blockIdx.x, txy, ok);
        if (ok) {
            load3(pos, i0, pn);
            load3(nrm, i0, nn);
#pragma unroll
            for (int q = 0; q < NPT; ++q) tn[q] = __ldg(P.tparam + i0 * NPT + q);
        }
    }
    uint32_t tile = blockIdx.x, tnext = s_tile[0], it = 0;
#ifdef NIV_EXPERIMENT_TIMING
    unsigned long long tacc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long tprev = clock64();
#define NIV_TICK(slot) do { const long long tn__ = clock64(); tacc[slot] += (unsigned long long)(tn__ - tprev); tprev = tn__; } while (0)
#else
#define NIV_TICK(slot) do { } while (0)
#endif
    while (tile < n_tiles) {
        bool valid;
        const size_t i = texel_of(tile, txy, valid);
        const float p[3] = {pn[0], pn[1], pn[2]}, nv[3] = {nn[0], nn[1], nn[2]};
        float tv[NPT > 0 ? NPT : 1];
#pragma unroll
        for (int q = 0; q < NPT; ++q) tv[q] = tn[q];
        uint32_t tnn_mine = 0;
        uint32_t txy_mine = 0;
        if (tid == 0) {
            tnn_mine = gridDim.x + atomicAdd(P.tile_ctr, 1u);                 // the tile after next
            if constexpr (IMG) txy_mine = image_tile_xy(P, tnn_mine);
        }
        {
            bool ok;
            const size_t inext = texel_of(tnext, txy_next, ok);   // (a tile index past the end gives ok = false)
#pragma unroll
            for (int d = 0; d < 3; ++d) { pn[d] = 0.f; nn[d] = 0.f; }
            if (ok) {
                load3(pos, inext, pn);
                load3(nrm, inext, nn);
#pragma unroll
                for (int q = 0; q < NPT; ++q) tn[q] = __ldg(P.tparam + inext * NPT + q);
            }
        }
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
                if (RAWDIR) {                         // the paper's model: the direction itself
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
                batch_issue<NB, F>(P, 0, u, ba);
                encode_direction();                   // arithmetic under the first batch's latency
#pragma unroll
                for (int g = 0; g < NG; g += 2) {
                    if (g + 1 < NG) batch_issue<NB, F>(P, (g + 1) * NB, u, bb);
                    batch_blend<NB, F>(ba, a + g * NB * (F / 2));
                    if (g + 2 < NG) batch_issue<NB, F>(P, (g + 2) * NB, u, ba);
                    if (g + 1 < NG) batch_blend<NB, F>(bb, a + (g + 1) * NB * (F / 2));
                }
            }
            // a8 per texel: gamma(t) = (sin, cos)(2^k pi t), k = 0..7, as fp16 pairs
#pragma unroll
            for (int q = 0; q < NPT; ++q) param_encode8_packed(tv[q], a + AW + 8 * q);
        }
        NIV_TICK(0);                                  // encode
        __syncwarp();
        if constexpr (AW == 8) tmem_st_x8(lane_taddr + A_COL, a);
        else tmem_st_x16(lane_taddr + A_COL, a);
        if constexpr (AW == 24) tmem_st_x8(lane_taddr + A_COL + 16, a + 16);
        if constexpr (AW == 32) tmem_st_x16(lane_taddr + A_COL + 16, a + 16);
        if constexpr (NPT >= 1) tmem_st_x8(lane_taddr + A_COL + AW, a + AW);
        if constexpr (NPT == 2) tmem_st_x8(lane_taddr + A_COL + AW + 8, a + AW + 8);
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
        NIV_TICK(1);                                  // A store + tile barrier

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
                    umma_f16_ts2(tmem, tmem + A_COL + ks * 8u, lo + ks * step, 0x4008u, idesc, ks > 0 ? 1u : 0u);
                umma_f16_ts2(tmem, tmem + ONES_COL, lo + ksteps_ct * step, 0x4008u, idesc, 1u);        // + bias
                umma_commit(bar_mma);
            }
            NIV_TICK(2);                              // MMA issue (thread 0)
            mbar_wait(bar_mma, phase);
            phase ^= 1u;
            tc_fence_after_sync();
            NIV_TICK(3);                              // MMA wait

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
                    tmem_st_x16(lane_taddr + A_COL, pk);
                    tmem_st_x16(lane_taddr + A_COL + 16, pk + 16);
                } else if constexpr (WIDTH == 32) {
                    uint32_t r[32];
                    tmem_ld_x32(lane_taddr, r);
                    tmem_ld_wait();
                    uint32_t pk[16];
#pragma unroll
                    for (int h = 0; h < 16; ++h)
                        pk[h] = pack_relu_half2(__uint_as_float(r[2 * h]), __uint_as_float(r[2 * h + 1]));
                    tmem_st_x16(lane_taddr + A_COL, pk);
                } else {                              // width 16
                    uint32_t r[16];
                    tmem_ld_x16(lane_taddr, r);
                    tmem_ld_wait();
                    uint32_t pk[8];
#pragma unroll
                    for (int h = 0; h < 8; ++h)
                        pk[h] = pack_relu_half2(__uint_as_float(r[2 * h]), __uint_as_float(r[2 * h + 1]));
                    tmem_st_x8(lane_taddr + A_COL, pk);
                }
                tmem_st_wait();
                NIV_TICK(4);                          // hidden epilogue
                tc_fence_before_sync();
                __syncthreads();
                NIV_TICK(5);                          // layer barrier
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
                    }
                    const uint32_t lane = tid & 31u;
                    float* so = reinterpret_cast<float*>(smem + P.misc_off + 64) + warp * 96;
                    const size_t w0 = ((size_t)tile * kTile + warp * 32u) * 3;        // first float of the warp
                    const bool vec = (w0 + 96 <= 3 * n) && ((reinterpret_cast<uintptr_t>(out) & 15u) == 0);
                    if (vec) {
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
                    }
                    out[3 * i] = y[0];
                    out[3 * i + 1] = y[1];
                    out[3 * i + 2] = y[2];
                }
            }
        }
        NIV_TICK(6);                                  // output layer epilogue + store
        tile = tnext;
        tnext = tnn;
        if constexpr (IMG) { txy = txy_next; txy_next = txy_nn; }
        ++it;
    }
#ifdef NIV_EXPERIMENT_TIMING
    if (tid == 0 && P.dbg) {
        for (int q = 0; q < 7; ++q) atomicAdd(P.dbg + q, tacc[q]);
        atomicAdd(P.dbg + 7, (unsigned long long)it);
    }
#endif
#undef NIV_TICK

    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, TMEM_COLS);
    if (tid == 0) {       // the last CTA to finish leaves the (tile, done) counter pair zero for the slot's next launch
        __threadfence();
        if (atomicAdd(P.tile_ctr + 1, 1u) == gridDim.x - 1) {
            P.tile_ctr[0] = 0u;
            P.tile_ctr[1] = 0u;
        }
    }
}

}  // namespace niv
#include "niv_fused_w128.cuh"
#include "niv_fused_mma.cuh"
#include "niv_compose.cuh"
namespace niv {

// =====================================================================================================
// stand-alone encode (fp16 features to global) and debug dump
// =====================================================================================================
__global__ void __launch_bounds__(128) niv_encode_kernel(const __grid_constant__ KParams P,
                                                         const float* __restrict__ pos,
                                                         const float* __restrict__ nrm,
                                                         uint4* __restrict__ feat, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t chunks = P.in_dim >> 3;
    uint4* row = feat + i * chunks;
    float p[3], nv[3];
    load3(pos, i, p);
    load3(nrm, i, nv);
    if (texel_masked(p, nv)) {
        for (uint32_t c = 0; c < chunks; ++c) row[c] = make_uint4(0, 0, 0, 0);
        return;
    }
    float u[3];
    normalise(P, p, u);
    const uint32_t n_groups = P.L >> 2;
    for (uint32_t g = 0; g < n_groups; ++g) row[g] = encode_group4(P, (int)(g * 4), u);
    float sh[16];
    sh16(nv, sh);
    row[n_groups] = make_uint4(pack_half2(sh[0], sh[1]), pack_half2(sh[2], sh[3]),
                               pack_half2(sh[4], sh[5]), pack_half2(sh[6], sh[7]));
    row[n_groups + 1] = make_uint4(pack_half2(sh[8], sh[9]), pack_half2(sh[10], sh[11]),
                                   pack_half2(sh[12], sh[13]), pack_half2(sh[14], sh[15]));
    for (uint32_t q = 0; q < P.n_params; ++q) {
        float e[16];
        param_encode8(P.t[q], e);
        row[n_groups + 2 + 2 * q] = make_uint4(pack_half2(e[0], e[1]), pack_half2(e[2], e[3]),
                                               pack_half2(e[4], e[5]), pack_half2(e[6], e[7]));
        row[n_groups + 3 + 2 * q] = make_uint4(pack_half2(e[8], e[9]), pack_half2(e[10], e[11]),
                                               pack_half2(e[12], e[13]), pack_half2(e[14], e[15]));
    }
}

__global__ void __launch_bounds__(128) niv_debug_kernel(const __grid_constant__ KParams P,
                                                        const float* __restrict__ pos,
                                                        const float* __restrict__ nrm, size_t n,
                                                        uint32_t* __restrict__ idx, int32_t* __restrict__ cell,
                                                        float* __restrict__ frac, float* __restrict__ feat)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t L = P.L;
    float p[3], nv[3];
    load3(pos, i, p);
    load3(nrm, i, nv);
    const bool masked = texel_masked(p, nv);
    float u[3] = {0.f, 0.f, 0.f};
    if (!masked) normalise(P, p, u);
    for (uint32_t l = 0; l < L; ++l) {
        int c[3] = {0, 0, 0};
        float w[3] = {0.f, 0.f, 0.f};
        uint32_t e[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        float f[4] = {0.f, 0.f, 0.f, 0.f};
        const uint32_t FW = P.n_features >> 1;               // 32-bit words per entry
        if (!masked) {
            locate(P.lv[l], u, c, w);
            corner_entries(P.lv[l], P.tmask, c, e);
            if (feat) {
                for (uint32_t h = 0; h < FW; ++h) {
                    uint32_t v[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) v[j] = __ldg(P.lv[l].tb + (size_t)e[j] * FW + h);
                    const float2 t = blend8(v, w);
                    f[2 * h] = t.x;
                    f[2 * h + 1] = t.y;
                }
            }
        }
        if (idx)
            for (int j = 0; j < 8; ++j) idx[(i * L + l) * 8 + j] = e[j];
        if (cell)
            for (int d = 0; d < 3; ++d) cell[(i * L + l) * 3 + d] = c[d];
        if (frac)
            for (int d = 0; d < 3; ++d) frac[(i * L + l) * 3 + d] = w[d];
        if (feat)
            for (uint32_t k = 0; k < P.n_features; ++k) feat[i * P.in_dim + P.n_features * l + k] = f[k];
    }
    if (feat && L == 0) {                            // grid-less: accurate per-band sincospi (the fused path doubles angles)
        for (int d = 0; d < 3; ++d) {
            float e[16];
            param_encode8(u[d], e);
            for (int k = 0; k < 16; ++k) feat[i * P.in_dim + 16 * d + k] = masked ? 0.f : e[k];
        }
    }
    if (feat) {
        const uint32_t o = L ? P.n_features * L : 48u;
        uint32_t dd;
        if (P.raw_dir) {
            dd = 3;
            for (int k = 0; k < 3; ++k) feat[i * P.in_dim + o + k] = masked ? 0.f : nv[k];
        } else {
            dd = 16;
            float sh[16];
            sh16(nv, sh);
            for (int k = 0; k < 16; ++k) feat[i * P.in_dim + o + k] = masked ? 0.f : sh[k];
        }
        for (uint32_t q = 0; q < P.n_params; ++q) {
            float e[16];
            param_encode8(P.t[q], e);
            for (int k = 0; k < 16; ++k) feat[i * P.in_dim + o + dd + 16 * q + k] = masked ? 0.f : e[k];
        }
    }
}

// =====================================================================================================
// gather micro-benchmark
// =====================================================================================================
__device__ __forceinline__ uint32_t mix32(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

// One random address stream per lane (patterns 0, 2, 4, 5, 6, 7), per warp (1) or per group of 8 lanes (3);
// 8 independent loads are in flight per thread.  PATTERN is a template parameter so that every variant is a
// tight loop of its own load instruction.
template <int PATTERN>
__global__ void __launch_bounds__(256) niv_probe_gather_kernel(const uint32_t* __restrict__ buf, uint32_t word_mask,
                                                               uint32_t loads_per_lane, uint32_t seed,
                                                               uint32_t* __restrict__ sink)
{
    const uint32_t gid = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t wid = gid >> 5;
    uint32_t acc = 0;
    for (uint32_t it = 0; it < loads_per_lane; it += 8) {
        uint32_t v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint32_t salt = ((it + k) * 0x85EBCA6Bu) ^ seed;
            if (PATTERN == 0) {                 // every lane: its own random 4-byte word (random 32 B sector)
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                v[k] = __ldg(buf + a);
            } else if (PATTERN == 1) {          // random 128 B line per warp, lanes consecutive (coalesced)
                const uint32_t a = (mix32((wid * 0x9E3779B9u) ^ salt) & word_mask & ~31u) + lane;
                v[k] = __ldg(buf + a);
            } else if (PATTERN == 2) {          // every lane: random aligned 8-byte pair, one 64-bit load
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask & ~1u;
                const uint2 t = __ldg(reinterpret_cast<const uint2*>(buf + a));
                v[k] = t.x ^ t.y;
            } else if (PATTERN == 3) {          // groups of 8 lanes share one random 32 B sector (one word each)
                const uint32_t a = (mix32(((gid >> 3) * 0x9E3779B9u) ^ salt) & word_mask & ~7u) + (lane & 7u);
                v[k] = __ldg(buf + a);
            } else if (PATTERN == 4) {          // every lane: random aligned 16-byte quad, one 128-bit load
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask & ~3u;
                const uint4 t = __ldg(reinterpret_cast<const uint4*>(buf + a));
                v[k] = t.x ^ t.y ^ t.z ^ t.w;
            } else if (PATTERN == 5) {          // every lane: one whole random 32 B sector, one 256-bit load
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask & ~7u;
                uint32_t r[8];
                asm volatile("ld.global.nc.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                             : "l"(buf + a));
                v[k] = r[0] ^ r[1] ^ r[2] ^ r[3] ^ r[4] ^ r[5] ^ r[6] ^ r[7];
            } else if (PATTERN == 6) {          // every lane: TWO 4-byte loads (two instructions) from one random sector
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                v[k] = __ldg(buf + a) ^ __ldg(buf + (a ^ 1u));
            } else {                            // 7: as 0 but L1 no-allocate
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                asm volatile("ld.global.nc.L1::no_allocate.b32 %0, [%1];" : "=r"(v[k]) : "l"(buf + a));
            }
        }
#pragma unroll
        for (int k = 0; k < 8; ++k) acc ^= v[k];
    }
    if (acc == 0x12345678u) sink[0] = acc;      // keep the loads alive
}

// =====================================================================================================
// sector census: the S of the gather roofline
// =====================================================================================================
// One warp per group of 32 consecutive texels (the fused kernel's own texel -> warp map).  For every level the
// warp's <= 256 corner addresses are reduced to the number of DISTINCT 32-byte sectors (and distinct 128-byte
// lines); the per-level counts are summed over the grid.  counts[0..L) = sectors, counts[16..16+L) = lines,
// counts[32] = active texels.
__global__ void __launch_bounds__(128) niv_sector_census_kernel(const __grid_constant__ KParams P,
                                                                const float* __restrict__ pos,
                                                                const float* __restrict__ nrm, size_t n,
                                                                unsigned long long* __restrict__ counts)
{
    __shared__ uint32_t s_sec[4][256];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    float p[3] = {0.f, 0.f, 0.f}, nv[3] = {0.f, 0.f, 0.f};
    bool valid = i < n;
    if (P.tiles_x) i = image_texel(P, blockIdx.x, threadIdx.x, valid);      // the warps of niv_infer_image
    if (valid) { load3(pos, i, p); load3(nrm, i, nv); }
    const bool masked = !valid || texel_masked(p, nv);
    float u[3] = {0.f, 0.f, 0.f};
    if (!masked) normalise(P, p, u);
    const uint32_t n_act = __popc(__ballot_sync(0xffffffffu, !masked));
    if (lane == 0 && n_act) atomicAdd(&counts[32], (unsigned long long)n_act);
    for (uint32_t l = 0; l < P.L; ++l) {
        uint32_t e[8];
        if (!masked) {
            int c[3]; float w[3];
            locate(P.lv[l], u, c, w);
            corner_entries(P.lv[l], P.tmask, c, e);
        }
#pragma unroll
        for (int j = 0; j < 8; ++j)                                           // 8 (F = 2) or 4 (F = 4) entries per 32-byte sector
            s_sec[warp][lane * 8 + j] = masked ? 0xFFFFFFFFu : ((P.lv[l].base + e[j]) >> (P.n_features == 4 ? 2 : 3));
        __syncwarp();
        uint32_t sec = 0, lin = 0;
        for (int q = 0; q < 8; ++q) {
            const uint32_t me = lane * 8 + q;
            const uint32_t v = s_sec[warp][me];
            if (v == 0xFFFFFFFFu) continue;
            bool first_s = true, first_l = true;
            for (uint32_t k = 0; k < me; ++k) {
                const uint32_t o = s_sec[warp][k];
                if (o == 0xFFFFFFFFu) continue;
                first_s &= (o != v);
                first_l &= ((o >> 2) != (v >> 2));
            }
            sec += first_s; lin += first_l;
        }
        for (int o = 16; o; o >>= 1) {
            sec += __shfl_xor_sync(0xffffffffu, sec, o);
            lin += __shfl_xor_sync(0xffffffffu, lin, o);
        }
        if (lane == 0 && sec) {
            atomicAdd(&counts[l], (unsigned long long)sec);
            atomicAdd(&counts[16 + l], (unsigned long long)lin);
        }
        __syncwarp();
    }
}

}  // namespace niv

// =====================================================================================================
// host side: the C ABI
// =====================================================================================================
using namespace niv;

constexpr uint32_t kCtrSlots = 64;      // launches of one model that may be in flight at once (different streams)

struct niv_model {
    niv_config cfg;
    niv_info info;
    KParams kp;
    uint32_t* d_table = nullptr;
    uint8_t* d_wpack = nullptr;
    std::vector<uint32_t> layer_out, layer_in;     // true (unpadded) shapes
    bool loaded = false;
    uint32_t grid_fused = 0;
    uint32_t smem_fused = 0;
    void (*fused)(KParams, const float*, const float*, float*, size_t, uint32_t) = nullptr;
    void (*fused_host)(KParams, const float*, const float*, float*, size_t, uint32_t) = nullptr;   // 128-bit output stores
    uint32_t grid_host = 0;
    // per-texel scene parameters (niv_infer_texel_params): a kernel whose layer 1 has the parameter columns as K-steps,
    // with its own packed weights and shared-memory layout
    void (*fused_tp)(KParams, const float*, const float*, float*, size_t, uint32_t) = nullptr;
    KParams kp_tp;
    uint8_t* d_wpack_tp = nullptr;
    uint32_t grid_tp = 0, smem_tp = 0;
    // niv_infer_image: the same kernel with 8 x 4 pixel blocks per warp
    void (*fused_img)(KParams, const float*, const float*, float*, size_t, uint32_t) = nullptr;
    uint32_t grid_img = 0;
    bool mma_kernel = false;                       // NIV_KERNEL=6: the per-warp mma.sync A/B kernel (32-texel tiles)
    uint32_t* d_wmma = nullptr;
    uint32_t* d_ctr = nullptr;                     // kCtrSlots tile counters, 128 B apart; one per launch in flight
    mutable std::atomic<uint32_t> ctr_next{0};
    bool pdl = true;                               // NIV_PDL=0: launch without programmatic stream serialisation (A/B knob)
    mutable std::atomic<uint32_t> ctr_next_captured{0};   // launches recorded into a CUDA graph draw from their own pool
    // niv_infer_host staging (grown on demand)
    float* d_stage = nullptr;          // [pos | nrm | out], each 3*stage_cap floats
    size_t stage_cap = 0;
    cudaStream_t hs[2] = {nullptr, nullptr};
    cudaEvent_t hev = nullptr;
};

static thread_local int g_last_cuda_error = 0;

#define NIV_CUDA(call)                                   \
    do {                                                 \
        cudaError_t e__ = (call);                        \
        if (e__ != cudaSuccess) {                        \
            g_last_cuda_error = (int)e__;                \
            (void)cudaGetLastError();                    \
            return NIV_ERR_CUDA;                         \
        }                                                \
    } while (0)

static uint32_t round_up(uint32_t v, uint32_t m) { return (v + m - 1) / m * m; }

// Resident CTAs per SM from the kernel's own resource use.  (cudaOccupancyMaxActiveBlocksPerMultiprocessor
// answers 1 for these kernels on sm_100a with driver 580 -- measured, see DESIGN.md section 6 -- so it is not used.)
template <typename K>
static int setup_kernel(niv_model* m, K kernel, int tmem_cols, const char* name, uint32_t* grid_out = nullptr,
                        uint32_t smem_override = 0) {
    const uint32_t smem_dyn = smem_override ? smem_override : m->smem_fused;
    NIV_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_dyn));
    cudaFuncAttributes fa;
    NIV_CUDA(cudaFuncGetAttributes(&fa, kernel));
    cudaDeviceProp prop;
    NIV_CUDA(cudaGetDeviceProperties(&prop, m->cfg.device));
    const int regs_per_cta = ((fa.numRegs + 7) / 8 * 8) * kTile;
    const int smem_per_cta = (int)round_up(smem_dyn + (uint32_t)fa.sharedSizeBytes + (uint32_t)prop.reservedSharedMemPerBlock, 128);
    int blocks = prop.regsPerMultiprocessor / regs_per_cta;
    blocks = std::min(blocks, (int)prop.sharedMemPerMultiprocessor / smem_per_cta);
    blocks = std::min(blocks, prop.maxThreadsPerMultiProcessor / kTile);
    blocks = std::min(blocks, 512 / tmem_cols);                // TMEM: 512 columns per SM
    blocks = std::min(blocks, 32);
    if (const char* s = getenv("NIV_CTAS_PER_SM")) { int v = atoi(s); if (v > 0) blocks = std::min(blocks, v); }   // tuning knob
    if (getenv("NIV_DEBUG"))
        fprintf(stderr, "[niv] %s: %d regs, %d B smem/CTA, %d TMEM cols -> %d CTAs/SM\n", name, fa.numRegs,
                smem_per_cta, tmem_cols, blocks);
    if (blocks < 1) return NIV_ERR_UNSUPPORTED;
    {   // the gathers live on L1 hits: ask for the smallest shared-memory carve-out that still holds `blocks` CTAs,
        // the rest of the 228 KB becomes L1
        int pct = (blocks * smem_per_cta * 100 + (int)prop.sharedMemPerMultiprocessor - 1) / (int)prop.sharedMemPerMultiprocessor;
        if (const char* s = getenv("NIV_CARVEOUT")) { int v = atoi(s); if (v >= 0) pct = v; }
        pct = std::min(100, std::max(0, pct));
        NIV_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pct));
        if (getenv("NIV_DEBUG")) fprintf(stderr, "[niv] %s: shared-memory carve-out %d %%\n", name, pct);
    }
    if (grid_out) { *grid_out = (uint32_t)blocks * m->info.num_sms; return NIV_OK; }
    m->info.ctas_per_sm = (uint32_t)blocks;
    m->grid_fused = (uint32_t)blocks * m->info.num_sms;
    return NIV_OK;
}

typedef void (*fused_fn)(KParams, const float*, const float*, float*, size_t, uint32_t);

template <int W, int L>
static fused_fn pick_nb(int nb) { return nb == 4 ? niv_fused_kernel<W, L, 4> : niv_fused_kernel<W, L, 2>; }
template <int W>
static fused_fn pick_l(uint32_t L, int nb) {
    switch (L) {
        case 4:  return niv_fused_kernel<W, 4, 4>;
        case 8:  return pick_nb<W, 8>(nb);
        case 12: return niv_fused_kernel<W, 12, 4>;
        case 16: return pick_nb<W, 16>(nb);
        default: return nullptr;
    }
}
static fused_fn pick_fused(uint32_t W, uint32_t L, int nb) {
    if (W == 32) return pick_l<32>(L, nb);
    if (W == 64) return pick_l<64>(L, nb);
    return pick_l<128>(L, nb);
}
template <int W, int L, bool O>
static fused_fn pick_tmem_nb(int nb) {
    if (O) return niv_fused_tmem_kernel<W, L, 4, 2, false, O>;          // host-buffer variant: one batch size
    return nb == 4 ? niv_fused_tmem_kernel<W, L, 4, 2, false, O> : niv_fused_tmem_kernel<W, L, 2, 2, false, false>;
}
template <int W, bool O>
static fused_fn pick_tmem_l(uint32_t L, int nb) {
    switch (L) {
        case 4:  return niv_fused_tmem_kernel<W, 4, 4, 2, false, O>;
        case 8:  return pick_tmem_nb<W, 8, O>(nb);
        case 12: return niv_fused_tmem_kernel<W, 12, 4, 2, false, O>;
        case 16: return pick_tmem_nb<W, 16, O>(nb);
        default: return nullptr;
    }
}
// the paper's own family: F = 4, raw direction, 2..8 levels, 2 levels (16 x 8-byte gathers) per batch
template <int W, bool O>
static fused_fn pick_tmem_paper(uint32_t L) {
    switch (L) {
        case 2: return niv_fused_tmem_kernel<W, 2, 2, 4, true, O>;
        case 4: return niv_fused_tmem_kernel<W, 4, 2, 4, true, O>;
        case 6: return niv_fused_tmem_kernel<W, 6, 2, 4, true, O>;
        case 8: return niv_fused_tmem_kernel<W, 8, 2, 4, true, O>;
        default: return nullptr;
    }
}
// O = true: the variant whose output leaves as 128-bit stores (buffers in pinned host memory)
template <bool O>
static fused_fn pick_tmem(uint32_t W, uint32_t L, int nb, uint32_t F) {
    if (L == 0)                                     // grid-less: positional encoding, no gathers
        return W == 16 ? niv_fused_tmem_kernel<16, 0, 1, 2, true, O> : W == 32 ? niv_fused_tmem_kernel<32, 0, 1, 2, true, O>
             : W == 64 ? niv_fused_tmem_kernel<64, 0, 1, 2, true, O> : nullptr;
    if (F == 4) return W == 32 ? pick_tmem_paper<32, O>(L) : W == 64 ? pick_tmem_paper<64, O>(L) : nullptr;
    if (W == 32) return pick_tmem_l<32, O>(L, nb);
    if (W == 64) return pick_tmem_l<64, O>(L, nb);
    return nullptr;
}

// image tiling (niv_infer_image): BASELINE.json's family (F = 2, 8..16 levels reach cells smaller than a warp's strip).
// The paper's own family (F = 4, <= 8 levels, finest cell 5.5 cm) measured SLOWER with it (0.1098 against 0.1049 ms,
// profiles/r01_v2.md): its cells are larger than a 32-pixel strip anyway; it keeps the linear kernel, as do the
// grid-less models, which gather nothing.
template <int W>
static fused_fn pick_tmem_img_w(uint32_t L) {
    switch (L) {
        case 4:  return niv_fused_tmem_kernel<W, 4, 4, 2, false, false, 0, true>;
        case 8:  return niv_fused_tmem_kernel<W, 8, 4, 2, false, false, 0, true>;
        case 12: return niv_fused_tmem_kernel<W, 12, 4, 2, false, false, 0, true>;
        case 16: return niv_fused_tmem_kernel<W, 16, 4, 2, false, false, 0, true>;
        default: return nullptr;
    }
}
static fused_fn pick_tmem_img(uint32_t W, uint32_t L, uint32_t F) {
    if (L == 0 || F != 2) return nullptr;
    return W == 32 ? pick_tmem_img_w<32>(L) : W == 64 ? pick_tmem_img_w<64>(L) : nullptr;
}

// per-texel scene parameters: BASELINE.json's family (F = 2, SH-16), 8 or 16 levels, width 32 / 64, 1 or 2 parameters
template <int W, int NPT>
static fused_fn pick_tmem_tp_l(uint32_t L) {
    switch (L) {
        case 8:  return niv_fused_tmem_kernel<W, 8, 4, 2, false, false, NPT>;
        case 16: return niv_fused_tmem_kernel<W, 16, 4, 2, false, false, NPT>;
        default: return nullptr;
    }
}
static fused_fn pick_tmem_tp(uint32_t W, uint32_t L, uint32_t F, uint32_t sh_degree, uint32_t n_params) {
    if (F != 2 || sh_degree != 4) return nullptr;
    if (n_params == 1) return W == 32 ? pick_tmem_tp_l<32, 1>(L) : W == 64 ? pick_tmem_tp_l<64, 1>(L) : nullptr;
    if (n_params == 2) return W == 32 ? pick_tmem_tp_l<32, 2>(L) : W == 64 ? pick_tmem_tp_l<64, 2>(L) : nullptr;
    return nullptr;
}

extern "C" int niv_create(const niv_config* cfg, niv_model** out)
{
    if (!cfg || !out) return NIV_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->struct_size != sizeof(niv_config) || cfg->api_version != NIV_API_VERSION) return NIV_ERR_INVALID_ARG;
    if (cfg->n_levels > NIV_MAX_LEVELS || cfg->n_features == 0) return NIV_ERR_INVALID_ARG;
    if (cfg->log2_table_size < 4 || cfg->log2_table_size > 24) return NIV_ERR_INVALID_ARG;
    if (cfg->n_hidden_layers == 0 || cfg->hidden_width == 0) return NIV_ERR_INVALID_ARG;
    if (cfg->out_activation > NIV_OUT_SIGMOID) return NIV_ERR_INVALID_ARG;
    for (int d = 0; d < 3; ++d) {
        if (!std::isfinite(cfg->aabb_min[d]) || !std::isfinite(cfg->aabb_max[d])) return NIV_ERR_INVALID_ARG;
        if (!(cfg->aabb_max[d] > cfg->aabb_min[d])) return NIV_ERR_INVALID_ARG;
    }
    bool explicit_res = false;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) explicit_res |= cfg->resolutions[l] != 0;
    if (cfg->n_levels && !explicit_res && (cfg->base_resolution == 0 || !(cfg->per_level_scale >= 1.0) || !std::isfinite(cfg->per_level_scale)))
        return NIV_ERR_INVALID_ARG;
    // shapes this build has kernels for
    // two model families: BASELINE.json's (F = 2, SH-16 direction, L in {4, 8, 12, 16}) and the paper's own
    // (F = 4, raw direction, L in {2, 4, 6, 8}, width <= 64)
    // and the paper's grid-less models (n_levels = 0: eight-band positional encoding, raw direction, width 16/32/64)
    if (cfg->n_levels == 0) {
        if (cfg->sh_degree != 0 || cfg->n_frequencies != 8) return NIV_ERR_UNSUPPORTED;
        if (cfg->hidden_width != 16 && cfg->hidden_width != 32 && cfg->hidden_width != 64) return NIV_ERR_UNSUPPORTED;
    } else if (cfg->n_features == 2) {
        if (cfg->sh_degree != 4 || cfg->n_levels % 4 != 0) return NIV_ERR_UNSUPPORTED;
    } else if (cfg->n_features == 4) {
        if (cfg->sh_degree != 0 || cfg->n_levels % 2 != 0 || cfg->n_levels > 8 || cfg->hidden_width > 64) return NIV_ERR_UNSUPPORTED;
    } else return NIV_ERR_UNSUPPORTED;
    if (cfg->n_params > 2 || (cfg->n_params && cfg->n_frequencies != 8)) return NIV_ERR_UNSUPPORTED;
    if (cfg->n_hidden_layers > 3) return NIV_ERR_UNSUPPORTED;
    if (cfg->hidden_width != 32 && cfg->hidden_width != 64 && cfg->hidden_width != 128 &&
        !(cfg->n_levels == 0 && cfg->hidden_width == 16)) return NIV_ERR_UNSUPPORTED;

    niv_model* m = new (std::nothrow) niv_model();
    if (!m) return NIV_ERR_ALLOC;
    m->cfg = *cfg;
    niv_info& I = m->info;
    memset(&I, 0, sizeof(I));
    I.struct_size = sizeof(niv_info);
    KParams& P = m->kp;
    memset(&P, 0, sizeof(P));

    // level table (readings #2, #4)
    const uint64_t T = (uint64_t)1 << cfg->log2_table_size;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        uint64_t N;
        if (explicit_res) N = cfg->resolutions[l];
        else N = (uint64_t)std::floor((double)cfg->base_resolution * std::pow(cfg->per_level_scale, (double)l));
        if (N == 0 || N >= (1u << 24)) { delete m; return NIV_ERR_INVALID_ARG; }
        const uint64_t R = N + 1;
        const bool dense = R * R * R <= T;
        I.resolution[l] = (uint32_t)N;
        I.is_dense[l] = dense ? 1u : 0u;
        P.lv[l].Nf = (float)N;
        P.lv[l].Nm1 = (int32_t)N - 1;
        P.lv[l].R = (uint32_t)R;
        P.lv[l].R2 = dense ? (uint32_t)(R * R) : 0u;
        P.lv[l].base = (uint32_t)(l * T);
        P.lv[l].dense = dense ? 1u : 0u;
    }
    for (int d = 0; d < 3; ++d) {
        P.amin[d] = cfg->aabb_min[d];
        volatile float ext = cfg->aabb_max[d] - cfg->aabb_min[d];
        volatile float inv = 1.0f / ext;
        P.ainv[d] = inv;
    }
    P.L = cfg->n_levels;
    P.tmask = (uint32_t)(T - 1);
    P.n_features = cfg->n_features;
    P.raw_dir = cfg->sh_degree == 0 ? 1u : 0u;
    P.enc_dim = (cfg->n_levels ? cfg->n_levels * cfg->n_features : 6u * cfg->n_frequencies) + (P.raw_dir ? 3u : 16u);
    P.in_dim = P.enc_dim + 2 * cfg->n_frequencies * cfg->n_params;
    P.n_params = cfg->n_params;
    P.n_layers = cfg->n_hidden_layers + 1;
    P.out_act = cfg->out_activation;
    I.in_dim = P.in_dim;
    I.table_bytes = (uint64_t)cfg->n_levels * T * cfg->n_features * 2;      // 0 for the grid-less models
    I.tile_texels = kTile;

    // layer shapes and the packed weight blob layout
    const uint32_t W = cfg->hidden_width;
    uint32_t off = 0;
    uint32_t in = P.in_dim;
    for (uint32_t k = 0; k < P.n_layers; ++k) {
        const uint32_t o = (k + 1 == P.n_layers) ? 3u : W;
        m->layer_out.push_back(o);
        m->layer_in.push_back(in);
        I.weight_bytes += (uint64_t)o * in * 2;
        I.bias_bytes += (uint64_t)o * 4;
        P.kdim[k] = (k == 0) ? round_up(P.enc_dim, 16) : in;      // layer 1 consumes the encoded part only
        P.npad[k] = round_up(o, 16);
        P.w_off[k] = off;
        off += (P.kdim[k] + 16) * P.npad[k] * 2;                 // + the bias K-step: rows (bias_hi, bias_lo, 0, ..)
        in = o;
    }
    for (uint32_t k = 0; k < P.n_layers; ++k) { P.b_off[k] = off; off += P.npad[k] * 4; }
    P.wparam_off = off;
    off += W * 16 * cfg->n_params * 4;
    P.wpack_bytes = round_up(off, 16);
    uint32_t kmax = P.kdim[0];
    for (uint32_t k = 1; k < P.n_layers; ++k) kmax = kmax > P.kdim[k] ? kmax : P.kdim[k];
    P.a_off = round_up(P.wpack_bytes, 128);
    P.ones_off = P.a_off + kTile * kmax * 2;
    P.misc_off = P.ones_off + 2 * kTile * 16;
    m->smem_fused = P.misc_off + W * 4 + 2 * 8 + 16;
    I.smem_bytes = m->smem_fused;

    // device side
    g_last_cuda_error = 0;
    int rc = NIV_OK;
    cudaError_t e = cudaSetDevice(cfg->device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cfg->device);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); delete m; return NIV_ERR_CUDA; }
    if (prop.major != 10) { delete m; return NIV_ERR_UNSUPPORTED; }           // sm_100a only; no fallback
    I.num_sms = (uint32_t)prop.multiProcessorCount;
    {
        if (const char* pv = getenv("NIV_PDL")) m->pdl = atoi(pv) != 0;
        const char* kv = getenv("NIV_KERNEL");          // A-B knob: 1 = v1 (A operand in shared memory), 2 = v2 (A in TMEM)
        const char* nbv = getenv("NIV_NB");             // levels per gather batch: 2 or 4
        const int nb = nbv ? atoi(nbv) : 4;
        int kind = kv ? atoi(kv) : 2;
        if (kind != 1 && kind != 2 && kind != 6) kind = 2;
        if (cfg->n_levels == 0 || cfg->n_features == 4) kind = 2;   // the paper's families exist as v2 only
        int tmem_cols = W < 32 ? 32 : (int)W;
        if (kind == 1) m->fused = pick_fused(W, cfg->n_levels, nb);
        else if (kind == 6 && W == 64 && cfg->n_levels == 16 && cfg->n_features == 2 && cfg->n_hidden_layers == 2 &&
                 cfg->n_params == 0) {
            m->fused = niv_fused_mma_kernel<4, 4>;       // 4 levels per gather batch, 128 registers, 4 CTAs per SM
            m->mma_kernel = true;
            tmem_cols = 32;                              // no tensor memory: do not let it limit the occupancy
            m->smem_fused = (kMmaWords + 4 * kMmaStage) * 4;
            I.smem_bytes = m->smem_fused;
        } else if (W == 128) {                            // two N = 64 halves per hidden layer (niv_fused_w128.cuh)
            switch (cfg->n_levels) {
                case 4:  m->fused = niv_fused_w128_kernel<4, 4>; break;
                case 8:  m->fused = niv_fused_w128_kernel<8, 4>; break;
                case 12: m->fused = niv_fused_w128_kernel<12, 4>; break;
                case 16: m->fused = niv_fused_w128_kernel<16, 4>; break;
                default: m->fused = nullptr;
            }
            tmem_cols = 128;
            P.ones_off = P.a_off;                        // weights | ones chunk | barriers
            P.misc_off = P.a_off + 2 * kTile * 16;
            m->smem_fused = P.misc_off + 2 * 8 + 16;
            I.smem_bytes = m->smem_fused;
        } else {
            m->fused = pick_tmem<false>(W, cfg->n_levels, nb, cfg->n_features);
            m->fused_host = pick_tmem<true>(W, cfg->n_levels, nb, cfg->n_features);
            tmem_cols = 128;
            m->smem_fused = P.a_off + 64 + 4 * 384;      // weights | barriers, TMEM slot, tile slots | output staging
            P.misc_off = P.a_off;
            I.smem_bytes = m->smem_fused;
        }
        if (!m->fused) { delete m; return NIV_ERR_UNSUPPORTED; }
        rc = setup_kernel(m, m->fused, tmem_cols, kind == 1 ? "fused_v1" : m->mma_kernel ? "fused_mma" : W == 128 ? "fused_w128" : "fused_v2");
        if (rc == NIV_OK && m->fused_host && kind == 2 && W != 128 && !m->mma_kernel)
            rc = setup_kernel(m, m->fused_host, tmem_cols, "fused_v2_host", &m->grid_host);
        else m->fused_host = nullptr;
        if (rc == NIV_OK && kind == 2 && W != 128 && !m->mma_kernel) {
            m->fused_img = pick_tmem_img(W, cfg->n_levels, cfg->n_features);
            if (m->fused_img) rc = setup_kernel(m, m->fused_img, 128, "fused_v2_image", &m->grid_img);
        }
        if (rc == NIV_OK && cfg->n_params && kind == 2 && W != 128)
            m->fused_tp = pick_tmem_tp(W, cfg->n_levels, cfg->n_features, cfg->sh_degree, cfg->n_params);
        if (m->fused_tp) {
            // layout of the per-texel-parameter variant: layer 1 with K = round16(enc_dim) + 16 n_params, no fold blob
            KParams& T = m->kp_tp;
            T = P;
            uint32_t o2 = 0;
            for (uint32_t k = 0; k < P.n_layers; ++k) {
                if (k == 0) T.kdim[0] = round_up(P.enc_dim, 16) + 16 * cfg->n_params;
                T.w_off[k] = o2;
                o2 += (T.kdim[k] + 16) * T.npad[k] * 2;
            }
            for (uint32_t k = 0; k < P.n_layers; ++k) { T.b_off[k] = o2; o2 += T.npad[k] * 4; }
            T.wparam_off = o2;
            T.wpack_bytes = round_up(o2, 16);
            T.a_off = round_up(T.wpack_bytes, 128);
            T.misc_off = T.a_off;
            m->smem_tp = T.a_off + 64 + 4 * 384;
            rc = setup_kernel(m, m->fused_tp, 128, "fused_v2_texel_params", &m->grid_tp, m->smem_tp);
        }
    }
    if (rc != NIV_OK) { delete m; return rc; }
    I.image_tiled = m->fused_img ? 1u : 0u;
    I.texel_params = m->fused_tp ? 1u : 0u;
    e = cudaMalloc(&m->d_table, I.table_bytes ? I.table_bytes : 16);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_wpack, P.wpack_bytes);
    if (e == cudaSuccess && m->fused_tp) e = cudaMalloc(&m->d_wpack_tp, m->kp_tp.wpack_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_ctr, 2 * kCtrSlots * 128);
    if (e == cudaSuccess) e = cudaMemset(m->d_ctr, 0, 2 * kCtrSlots * 128);
    if (e != cudaSuccess) {
        g_last_cuda_error = (int)e; (void)cudaGetLastError();
        cudaFree(m->d_table); cudaFree(m->d_wpack); cudaFree(m->d_wpack_tp); cudaFree(m->d_ctr); delete m;
        return NIV_ERR_ALLOC;
    }
    P.table = m->d_table;
    P.wpack = m->d_wpack;
    m->kp_tp.table = m->d_table;
    m->kp_tp.wpack = m->d_wpack_tp;
#ifdef NIV_EXPERIMENT_TIMING
    cudaMalloc(&P.dbg, 8 * sizeof(unsigned long long));
    cudaMemset(P.dbg, 0, 8 * sizeof(unsigned long long));
#endif
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        P.lv[l].tb = m->d_table + (size_t)P.lv[l].base * (cfg->n_features / 2);
        m->kp_tp.lv[l].tb = P.lv[l].tb;
    }
    *out = m;
    return NIV_OK;
}

extern "C" int niv_get_info(const niv_model* m, niv_info* info)
{
    if (!m || !info) return NIV_ERR_INVALID_ARG;
    *info = m->info;
    return NIV_OK;
}

extern "C" int niv_load_params(niv_model* m, const void* table_fp16, size_t table_bytes,
                               const void* weights_fp16, size_t weight_bytes,
                               const float* biases_f32, size_t bias_bytes, int src_on_device, void* stream)
{
    if (!m || (!table_fp16 && m->info.table_bytes) || !weights_fp16) return NIV_ERR_INVALID_ARG;
    if (table_bytes != m->info.table_bytes || weight_bytes != m->info.weight_bytes) return NIV_ERR_INVALID_ARG;
    if (biases_f32 ? bias_bytes != m->info.bias_bytes : bias_bytes != 0) return NIV_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    NIV_CUDA(cudaSetDevice(m->cfg.device));
    const KParams& P = m->kp;

    // host copies of the small blobs
    std::vector<uint16_t> w(weight_bytes / 2);
    std::vector<float> b(m->info.bias_bytes / 4, 0.0f);
    if (src_on_device) {
        NIV_CUDA(cudaMemcpyAsync(w.data(), weights_fp16, weight_bytes, cudaMemcpyDeviceToHost, st));
        if (biases_f32) NIV_CUDA(cudaMemcpyAsync(b.data(), biases_f32, bias_bytes, cudaMemcpyDeviceToHost, st));
        NIV_CUDA(cudaStreamSynchronize(st));
    } else {
        memcpy(w.data(), weights_fp16, weight_bytes);
        if (biases_f32) memcpy(b.data(), biases_f32, bias_bytes);
    }

    // pack: per layer, the UMMA K-major no-swizzle layout of B = W[out][in]:
    //   element (n, k) at  (k/8) * (Npad*16) + n*16 + (k%8)*2  bytes; rows n >= out and columns k >= in are zero.
    //   texel_params: layer 1 keeps its parameter columns, as K rows round16(enc_dim) .. + 16 n_params (kp_tp layout)
    auto pack_blob = [&](const KParams& P, bool texel_params) {
    std::vector<uint8_t> pack(P.wpack_bytes, 0);
    size_t wsrc = 0, bsrc = 0;
    for (uint32_t k = 0; k < P.n_layers; ++k) {
        const uint32_t o = m->layer_out[k], in = m->layer_in[k];
        const uint32_t kuse = (k == 0) ? P.enc_dim : in;
        uint16_t* dst = reinterpret_cast<uint16_t*>(pack.data() + P.w_off[k]);
        for (uint32_t r = 0; r < o; ++r)
            for (uint32_t c = 0; c < kuse; ++c)
                dst[(size_t)(c >> 3) * (P.npad[k] * 8) + r * 8 + (c & 7)] = w[wsrc + (size_t)r * in + c];
        if (k == 0 && texel_params) {
            const uint32_t k0 = round_up(P.enc_dim, 16);
            for (uint32_t r = 0; r < o; ++r)
                for (uint32_t c = 0; c < 16 * P.n_params; ++c)
                    dst[(size_t)((k0 + c) >> 3) * (P.npad[k] * 8) + r * 8 + ((k0 + c) & 7)] = w[wsrc + (size_t)r * in + P.enc_dim + c];
        } else if (k == 0 && P.n_params) {
            float* wp = reinterpret_cast<float*>(pack.data() + P.wparam_off);
            const uint32_t np16 = 16 * P.n_params;
            for (uint32_t r = 0; r < o; ++r)
                for (uint32_t c = 0; c < np16; ++c) {
                    __half_raw hr; hr.x = w[wsrc + (size_t)r * in + P.enc_dim + c];
                    wp[r * np16 + c] = __half2float(__half(hr));
                }
        }
        float* bd = reinterpret_cast<float*>(pack.data() + P.b_off[k]);
        for (uint32_t r = 0; r < o; ++r) {
            bd[r] = b[bsrc + r];
            // bias K-step rows: K index kdim -> bias_hi, kdim + 1 -> bias_lo (hi + lo = bias to 2^-22 relative)
            const __half hi = __float2half_rn(b[bsrc + r]);
            const __half lo = __float2half_rn(b[bsrc + r] - __half2float(hi));
            uint16_t* brow = dst + (size_t)(P.kdim[k] >> 3) * (P.npad[k] * 8) + r * 8;
            brow[0] = __half_as_ushort(hi);
            brow[1] = __half_as_ushort(lo);
        }
        wsrc += (size_t)o * in;
        bsrc += o;
    }
    return pack;
    };
    const std::vector<uint8_t> pack = pack_blob(P, false);
    NIV_CUDA(cudaMemcpyAsync(m->d_wpack, pack.data(), P.wpack_bytes, cudaMemcpyHostToDevice, st));
    std::vector<uint8_t> pack_tp;                       // (alive until the stream is synchronised below)
    if (m->fused_tp) {
        pack_tp = pack_blob(m->kp_tp, true);
        NIV_CUDA(cudaMemcpyAsync(m->d_wpack_tp, pack_tp.data(), m->kp_tp.wpack_bytes, cudaMemcpyHostToDevice, st));
    }
    std::vector<uint32_t> wm;
    if (m->mma_kernel) {                                // row-major padded weights + fp32 biases (niv_fused_mma.cuh)
        wm.assign(kMmaWords, 0u);
        uint16_t* h = reinterpret_cast<uint16_t*>(wm.data());
        const size_t o2 = (size_t)64 * P.in_dim, o3 = o2 + 64 * 64;
        for (uint32_t r = 0; r < 64; ++r) {
            for (uint32_t c2 = 0; c2 < 48; ++c2) h[(kMmaW1 + r * kMmaS1) * 2 + c2] = w[(size_t)r * P.in_dim + c2];
            for (uint32_t c2 = 0; c2 < 64; ++c2) h[(kMmaW2 + r * kMmaS2) * 2 + c2] = w[o2 + (size_t)r * 64 + c2];
        }
        for (uint32_t r = 0; r < 3; ++r)
            for (uint32_t c2 = 0; c2 < 64; ++c2) h[(kMmaW3 + r * kMmaS2) * 2 + c2] = w[o3 + (size_t)r * 64 + c2];
        float* bf = reinterpret_cast<float*>(wm.data() + kMmaB1);
        for (uint32_t r = 0; r < 64; ++r) { bf[r] = b[r]; bf[64 + r] = b[64 + r]; }
        for (uint32_t r = 0; r < 3; ++r) bf[128 + r] = b[128 + r];
        if (!m->d_wmma) NIV_CUDA(cudaMalloc(&m->d_wmma, kMmaWords * 4));
        NIV_CUDA(cudaMemcpyAsync(m->d_wmma, wm.data(), kMmaWords * 4, cudaMemcpyHostToDevice, st));
        m->kp.wmma = m->d_wmma;
    }
    if (table_bytes) NIV_CUDA(cudaMemcpyAsync(m->d_table, table_fp16, table_bytes,
                             src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    NIV_CUDA(cudaStreamSynchronize(st));
    m->loaded = true;
    return NIV_OK;
}

static int fill_params(const niv_model* m, const float* param, KParams& P)
{
    P = m->kp;
    if (m->cfg.n_params) {
        if (!param) return NIV_ERR_INVALID_ARG;
        for (uint32_t q = 0; q < m->cfg.n_params; ++q) P.t[q] = param[q];
    } else if (param) {
        return NIV_ERR_INVALID_ARG;
    }
    return NIV_OK;
}

// The tile counter of one launch.  A launch recorded into a CUDA graph keeps its slot for every replay, so captured
// launches take theirs from a second pool of kCtrSlots that live launches never touch: a replay cannot meet a live
// launch on the same counter.
static uint32_t* draw_tile_counter(const niv_model* m, cudaStream_t st)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
    const uint32_t slot = cs == cudaStreamCaptureStatusActive
                              ? kCtrSlots + m->ctr_next_captured.fetch_add(1u) % kCtrSlots
                              : m->ctr_next.fetch_add(1u) % kCtrSlots;
    return m->d_ctr + (size_t)slot * 32;
}

// One launch of a fused kernel; `pdl`: with the programmatic-stream-serialisation attribute (v2 kernels, which hold
// their griddepcontrol.wait before the first access to a caller's buffer).
static int launch_v2(fused_fn fn, uint32_t grid, uint32_t smem, cudaStream_t st, bool pdl, const KParams& P,
                     const float* pos, const float* nrm, float* out, size_t n, uint32_t n_tiles)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kTile);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    NIV_CUDA(cudaLaunchKernelEx(&cfg, fn, P, pos, nrm, out, n, n_tiles));
    return NIV_OK;
}

static int launch_fused(const niv_model* m, const KParams& Pin, const float* pos, const float* nrm, float* out,
                        size_t n, cudaStream_t st, bool host_variant = false)
{
    KParams P = Pin;
    P.tile_ctr = draw_tile_counter(m, st);
    // (no memset: the kernels leave their counter pair zero, see the end of niv_fused_tmem_kernel)
    if (m->mma_kernel) {                                // warp-granular 32-texel tiles, four per CTA
        const uint32_t nt32 = (uint32_t)((n + 31) / 32), ctas = (nt32 + 3) / 4;
        m->fused<<<ctas < m->grid_fused ? ctas : m->grid_fused, kTile, m->smem_fused, st>>>(P, pos, nrm, out, n, nt32);
        NIV_CUDA(cudaGetLastError());
        return NIV_OK;
    }
    const uint32_t n_tiles = (uint32_t)((n + kTile - 1) / kTile);
    const uint32_t cap = host_variant ? m->grid_host : m->grid_fused;
    const uint32_t grid = n_tiles < cap ? n_tiles : cap;
    return launch_v2(host_variant ? m->fused_host : m->fused, grid, m->smem_fused, st, m->pdl && m->fused_host, P, pos,
                     nrm, out, n, n_tiles);
}

extern "C" int niv_infer(niv_model* m, const float* pos, const float* nrm, const float* param,
                         float* out, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !out) return NIV_ERR_INVALID_ARG;
    if (n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    return launch_fused(m, P, pos, nrm, out, n, (cudaStream_t)stream);
}

extern "C" int niv_infer_image(niv_model* m, const float* pos, const float* nrm, const float* param,
                               float* out, uint32_t width, uint32_t height, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    const size_t n = (size_t)width * height;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !out) return NIV_ERR_INVALID_ARG;
    if (n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    // models without an image-tiled kernel (and images beyond the packed tile coordinates): same result, linear tiles
    if (!m->fused_img || width > (1u << 20) || height > (1u << 17) || getenv("NIV_IMAGE_LINEAR"))
        return launch_fused(m, P, pos, nrm, out, n, (cudaStream_t)stream);
    P.img_w = width;
    P.img_h = height;
    P.tiles_x = (width + 31u) / 32u;
    const uint32_t n_tiles = P.tiles_x * ((height + 3u) / 4u);
    P.tile_ctr = draw_tile_counter(m, (cudaStream_t)stream);
    const uint32_t grid = n_tiles < m->grid_img ? n_tiles : m->grid_img;
    return launch_v2(m->fused_img, grid, m->smem_fused, (cudaStream_t)stream, m->pdl, P, pos, nrm, out, n, n_tiles);
}

extern "C" int niv_infer_texel_params(niv_model* m, const float* pos, const float* nrm, const float* tparam,
                                      float* out, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (m->cfg.n_params == 0) return NIV_ERR_INVALID_ARG;
    if (!m->fused_tp) return NIV_ERR_UNSUPPORTED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !tparam || !out) return NIV_ERR_INVALID_ARG;
    if (n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    KParams P = m->kp_tp;
    P.tparam = tparam;
    P.tile_ctr = draw_tile_counter(m, (cudaStream_t)stream);
    const uint32_t n_tiles = (uint32_t)((n + kTile - 1) / kTile);
    const uint32_t grid = n_tiles < m->grid_tp ? n_tiles : m->grid_tp;
    return launch_v2(m->fused_tp, grid, m->smem_tp, (cudaStream_t)stream, m->pdl, P, pos, nrm, out, n, n_tiles);
}

extern "C" int niv_infer_host(niv_model* m, const float* pos, const float* nrm, const float* param,
                              float* out, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !out) return NIV_ERR_INVALID_ARG;
    if (n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    NIV_CUDA(cudaSetDevice(m->cfg.device));
    // Zero copy: if all three buffers are pinned (or registered) host memory the fused kernel reads the G-buffer and
    // writes the irradiance over PCIe itself -- the texel of the next tile is requested a tile ahead, the output
    // leaves as full 128-byte lines -- so transfer and compute overlap tile by tile in ONE launch with no staging
    // (1.04 ms per full-HD frame against 1.21 ms with chunked copies; 0.91 ms is the copy time of the input alone).
    if (m->fused_host && !getenv("NIV_HOST_STAGED")) {
        cudaPointerAttributes ap, an, ao;
        if (cudaPointerGetAttributes(&ap, pos) == cudaSuccess && cudaPointerGetAttributes(&an, nrm) == cudaSuccess &&
            cudaPointerGetAttributes(&ao, out) == cudaSuccess && ap.type == cudaMemoryTypeHost &&
            an.type == cudaMemoryTypeHost && ao.type == cudaMemoryTypeHost && ap.devicePointer && an.devicePointer &&
            ao.devicePointer && ((uintptr_t)ao.devicePointer & 15u) == 0) {
            rc = launch_fused(m, P, (const float*)ap.devicePointer, (const float*)an.devicePointer,
                              (float*)ao.devicePointer, n, (cudaStream_t)stream, true);
            if (rc != NIV_OK) return rc;
            NIV_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
            return NIV_OK;
        }
        (void)cudaGetLastError();                    // pageable memory: cudaPointerGetAttributes may have set an error
    }
    if (!m->hs[0]) {
        NIV_CUDA(cudaStreamCreateWithFlags(&m->hs[0], cudaStreamNonBlocking));
        NIV_CUDA(cudaStreamCreateWithFlags(&m->hs[1], cudaStreamNonBlocking));
        NIV_CUDA(cudaEventCreateWithFlags(&m->hev, cudaEventDisableTiming));
    }
    if (n > m->stage_cap) {
        if (m->d_stage) { NIV_CUDA(cudaFree(m->d_stage)); m->d_stage = nullptr; m->stage_cap = 0; }
        const size_t cap = (n + 1023) / 1024 * 1024;
        cudaError_t e = cudaMalloc(&m->d_stage, cap * 9 * sizeof(float));
        if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); return NIV_ERR_ALLOC; }
        m->stage_cap = cap;
    }
    float* d_pos = m->d_stage;
    float* d_nrm = m->d_stage + 3 * m->stage_cap;
    float* d_out = m->d_stage + 6 * m->stage_cap;
    // order after the caller's stream
    NIV_CUDA(cudaEventRecord(m->hev, (cudaStream_t)stream));
    NIV_CUDA(cudaStreamWaitEvent(m->hs[0], m->hev, 0));
    NIV_CUDA(cudaStreamWaitEvent(m->hs[1], m->hev, 0));
    // chunks of whole tiles; >= 4 chunks on a full frame so H2D, kernel and D2H of different chunks overlap
    size_t chunk = (n / 8 + kTile - 1) / kTile * kTile;
    if (chunk < 32768) chunk = 32768;
    int k = 0;
    for (size_t o = 0; o < n; o += chunk, ++k) {
        const size_t c = (n - o < chunk) ? n - o : chunk;
        cudaStream_t st = m->hs[k & 1];
        NIV_CUDA(cudaMemcpyAsync(d_pos + 3 * o, pos + 3 * o, c * 12, cudaMemcpyHostToDevice, st));
        NIV_CUDA(cudaMemcpyAsync(d_nrm + 3 * o, nrm + 3 * o, c * 12, cudaMemcpyHostToDevice, st));
        rc = launch_fused(m, P, d_pos + 3 * o, d_nrm + 3 * o, d_out + 3 * o, c, st);
        if (rc != NIV_OK) return rc;
        NIV_CUDA(cudaMemcpyAsync(out + 3 * o, d_out + 3 * o, c * 12, cudaMemcpyDeviceToHost, st));
    }
    NIV_CUDA(cudaStreamSynchronize(m->hs[0]));
    NIV_CUDA(cudaStreamSynchronize(m->hs[1]));
    return NIV_OK;
}

extern "C" int niv_encode(niv_model* m, const float* pos, const float* nrm, const float* param,
                          void* features_fp16, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !features_fp16 || ((uintptr_t)features_fp16 & 15)) return NIV_ERR_INVALID_ARG;
    if (m->cfg.n_features != 2) return NIV_ERR_UNSUPPORTED;      // the stand-alone kernel serves the F = 2 / SH-16 family
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    const unsigned grid = (unsigned)((n + 127) / 128);
    niv_encode_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (uint4*)features_fp16, n);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_debug_encode(niv_model* m, const float* pos, const float* nrm, const float* param, size_t n,
                                uint32_t* idx, int32_t* cell, float* frac, float* features, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm) return NIV_ERR_INVALID_ARG;
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    const unsigned grid = (unsigned)((n + 127) / 128);
    niv_debug_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, n, idx, cell, frac, features);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_probe_sectors(niv_model* m, const float* pos, const float* nrm, size_t n,
                                 uint64_t* counts, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (!pos || !nrm || !counts || n == 0) return NIV_ERR_INVALID_ARG;
    NIV_CUDA(cudaMemsetAsync(counts, 0, 33 * sizeof(uint64_t), (cudaStream_t)stream));
    const unsigned grid = (unsigned)((n + 127) / 128);
    niv_sector_census_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(m->kp, pos, nrm, n, (unsigned long long*)counts);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_probe_sectors_image(const niv_model* m, const float* pos, const float* nrm, uint32_t width,
                                       uint32_t height, uint64_t* counts, void* stream)
{
    if (!m || !pos || !nrm || !counts || width == 0 || height == 0) return NIV_ERR_INVALID_ARG;
    NIV_CUDA(cudaMemsetAsync(counts, 0, 33 * sizeof(uint64_t), (cudaStream_t)stream));
    KParams P = m->kp;
    P.img_w = width;
    P.img_h = height;
    P.tiles_x = (width + 31u) / 32u;
    const unsigned grid = P.tiles_x * ((height + 3u) / 4u);
    niv_sector_census_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (size_t)width * height,
                                                                     (unsigned long long*)counts);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_compose(const float* E, uint32_t ew, uint32_t eh, const float* albedo, const float* direct,
                           const float* emission, float* out, uint32_t w, uint32_t h, void* stream)
{
    if (!E || !albedo || !out) return NIV_ERR_INVALID_ARG;
    if (w == 0 || h == 0) return NIV_OK;
    int half;
    if (ew == w && eh == h) half = 0;
    else if (2ull * ew == w && 2ull * eh == h) half = 1;
    else return NIV_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    NIV_CUDA(cudaGetDevice(&dev));
    NIV_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t st = (cudaStream_t)stream;
    const uintptr_t align = (uintptr_t)albedo | (uintptr_t)out | (uintptr_t)(direct ? direct : albedo) |
                            (uintptr_t)(emission ? emission : albedo) | (half ? 0 : (uintptr_t)E);
    const size_t n = (size_t)w * h;
    if ((w & 3u) == 0 && (align & 15u) == 0) {
        const size_t groups = n / 4;
        const unsigned grid = (unsigned)std::min<size_t>((groups + 255) / 256, (size_t)sms * 8);   // 8 x 256 threads per SM
        if (half) niv_compose_kernel<true><<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h);
        else niv_compose_kernel<false><<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h);
    } else {
        const unsigned grid = (unsigned)std::min<size_t>((n + 255) / 256, (size_t)sms * 8);
        niv_compose_scalar_kernel<<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h, half);
    }
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_destroy(niv_model* m)
{
    if (!m) return NIV_OK;
    cudaSetDevice(m->cfg.device);
#ifdef NIV_EXPERIMENT_TIMING
    {
        unsigned long long h[8];
        cudaDeviceSynchronize();
        cudaMemcpy(h, m->kp.dbg, sizeof(h), cudaMemcpyDeviceToHost);
        const char* nm[7] = {"encode", "A store + tile barrier", "MMA issue", "MMA wait", "hidden epilogue", "layer barrier", "output"};
        if (h[7]) for (int q = 0; q < 7; ++q) fprintf(stderr, "[niv timing] %-24s %10.0f cycles per tile (thread 0)\n", nm[q], (double)h[q] / (double)h[7]);
        cudaFree(m->kp.dbg);
    }
#endif
    cudaFree(m->d_table);
    cudaFree(m->d_wpack);
    cudaFree(m->d_wpack_tp);
    cudaFree(m->d_ctr);
    cudaFree(m->d_wmma);
    cudaFree(m->d_stage);
    if (m->hs[0]) cudaStreamDestroy(m->hs[0]);
    if (m->hs[1]) cudaStreamDestroy(m->hs[1]);
    if (m->hev) cudaEventDestroy(m->hev);
    delete m;
    return NIV_OK;
}

extern "C" const char* niv_error_string(int code)
{
    switch (code) {
        case NIV_OK: return "ok";
        case NIV_ERR_INVALID_ARG: return "invalid argument";
        case NIV_ERR_UNSUPPORTED: return "configuration not supported by this build (sm_100a kernels only)";
        case NIV_ERR_NOT_LOADED: return "parameters not loaded";
        case NIV_ERR_CUDA: return "CUDA runtime error (see niv_last_cuda_error)";
        case NIV_ERR_ALLOC: return "allocation failed";
        default: return "unknown error code";
    }
}

extern "C" int niv_last_cuda_error(void) { return g_last_cuda_error; }

extern "C" int niv_probe_gather(const void* buf, size_t buf_bytes, int pattern, uint32_t n_ctas,
                                uint32_t loads_per_lane, uint32_t seed, void* sink, void* stream)
{
    if (!buf || !sink || buf_bytes < 4096 || (buf_bytes & (buf_bytes - 1)) || buf_bytes > ((size_t)1 << 33))
        return NIV_ERR_INVALID_ARG;
    if (pattern < 0 || pattern > 7 || n_ctas == 0 || loads_per_lane == 0 || (loads_per_lane & 7)) return NIV_ERR_INVALID_ARG;
    if (((uintptr_t)buf & 31) != 0) return NIV_ERR_INVALID_ARG;
    const uint32_t word_mask = (uint32_t)(buf_bytes / 4 - 1);
    const uint32_t* b = (const uint32_t*)buf;
    uint32_t* sk = (uint32_t*)sink;
    cudaStream_t st = (cudaStream_t)stream;
    switch (pattern) {
        case 0: niv_probe_gather_kernel<0><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 1: niv_probe_gather_kernel<1><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 2: niv_probe_gather_kernel<2><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 3: niv_probe_gather_kernel<3><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 4: niv_probe_gather_kernel<4><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 5: niv_probe_gather_kernel<5><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        case 6: niv_probe_gather_kernel<6><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
        default: niv_probe_gather_kernel<7><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk); break;
    }
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}
