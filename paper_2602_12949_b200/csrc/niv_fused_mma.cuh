// niv_fused_mma.cuh -- the fused encode + MLP with per-warp mma.sync (legacy HMMA) instead of tcgen05 / TMEM.
// Included by niv.cu.  An A/B kernel (NIV_MMA_SYNC=1 at niv_create) for the question north_star (3) leaves to the measurements:
// "tcgen05/TMEM or mma.sync, whichever ncu shows is faster".  BASELINE.json configs[1] shape only: L = 16, F = 2, SH-16,
// 48 -> 64 -> 64 -> 3, no scene parameter.
//
// Every warp is on its own: it draws a 32-texel tile, encodes it (same device functions as the v2 kernel, one texel
// per thread), turns the 32 rows into mma.m16n8k16 A fragments through a private 3.5 KB shared-memory patch, and runs
// the three layers with its own HMMAs: B fragments straight from the (row-major, padded) weights in shared memory,
// fp32 accumulators in registers, bias as accumulator initial value, ReLU + fp16 pack turns the accumulator
// fragments directly into the next layer's A fragments (the D and A fragment layouts coincide).  No CTA barrier, no
// mbarrier, no tensor memory after the prologue.
#pragma once

namespace niv {

__device__ __forceinline__ void mma_16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// shared-memory layout of the weights for this kernel (32-bit words; built on the host by pack_mma_weights):
constexpr uint32_t kMmaS1 = 28, kMmaS2 = 36;                       // row strides: K/2 words + 4 words of padding
constexpr uint32_t kMmaW1 = 0;                                     // [64][28]   W1[n][k < 48]
constexpr uint32_t kMmaW2 = kMmaW1 + 64 * kMmaS1;                  // [64][36]   W2[n][k < 64]
constexpr uint32_t kMmaW3 = kMmaW2 + 64 * kMmaS2;                  // [8][36]    W3[n < 3][k < 64], rows 3..7 zero
constexpr uint32_t kMmaB1 = kMmaW3 + 8 * kMmaS2;                   // fp32 b1[64] | b2[64] | b3[8]
constexpr uint32_t kMmaWords = kMmaB1 + 64 + 64 + 8;
constexpr uint32_t kMmaStage = 32 * kMmaS1;                        // per-warp A staging patch, words

template <int NB, int MINB>
__global__ void __launch_bounds__(kTile, MINB) niv_fused_mma_kernel(const __grid_constant__ KParams P,
                                                              const float* __restrict__ pos,
                                                              const float* __restrict__ nrm,
                                                              float* __restrict__ out, size_t n, uint32_t n_tiles32)
{
    const uint32_t* __restrict__ wmma = P.wmma;
    constexpr int L = 16, F = 2, NG = L / NB, HW = 16, AW = 24;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint32_t* sWm = reinterpret_cast<uint32_t*>(smem);
    const float* sBias = reinterpret_cast<const float*>(sWm + kMmaB1);
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31u;
    uint32_t* sA = sWm + kMmaWords + warp * kMmaStage;
    const uint32_t g = lane >> 2, c = lane & 3u;

    for (uint32_t k = tid; k < kMmaWords; k += kTile) sWm[k] = __ldg(wmma + k);
    __syncthreads();

    // warp-granular dynamic tiles: the first one is static, the rest come from the launch's counter
    uint32_t tile = blockIdx.x * 4u + warp;
    while (tile < n_tiles32) {
        uint32_t tnext = 0;
        if (lane == 0) tnext = P.tile_ctr ? gridDim.x * 4u + atomicAdd(P.tile_ctr, 1u) : tile + gridDim.x * 4u;   // NULL: static striding
        tnext = __shfl_sync(0xffffffffu, tnext, 0);
        const size_t i = (size_t)tile * 32u + lane;
        const bool valid = i < n;
        float p[3] = {0.f, 0.f, 0.f}, nv[3] = {0.f, 0.f, 0.f};
        if (valid) { load3(pos, i, p); load3(nrm, i, nv); }
        const bool masked = !valid || texel_masked(p, nv);
        const uint32_t live = __ballot_sync(0xffffffffu, !masked);

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
            for (int gg = 0; gg < NG; gg += 2) {
                if (gg + 1 < NG) batch_issue<NB, F>(P, (gg + 1) * NB, u, bb);
                batch_blend<NB, F>(ba, a + gg * NB);
                if (gg + 2 < NG) batch_issue<NB, F>(P, (gg + 2) * NB, u, ba);
                if (gg + 1 < NG) batch_blend<NB, F>(bb, a + (gg + 1) * NB);
            }
        }
        if (live != 0u) {                                 // a warp of background texels only: straight to the zeros
            // ---- rows -> A fragments through the warp's shared-memory patch (stride 28 words: conflict-free both ways)
            __syncwarp();
#pragma unroll
            for (int q = 0; q < 6; ++q)
                *reinterpret_cast<uint4*>(sA + lane * kMmaS1 + 4 * q) = make_uint4(a[4 * q], a[4 * q + 1], a[4 * q + 2], a[4 * q + 3]);
            __syncwarp();

            float acc[2][8][4];
            // ---- layer 1: K = 48 (3 k-steps), N = 64
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const float2 b = *reinterpret_cast<const float2*>(sBias + nt * 8 + 2 * c);
                    acc[mt][nt][0] = b.x; acc[mt][nt][1] = b.y; acc[mt][nt][2] = b.x; acc[mt][nt][3] = b.y;
                }
#pragma unroll
            for (int s = 0; s < 3; ++s) {
                uint32_t af[2][4];
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) {
                    const uint32_t* r0 = sA + (mt * 16 + g) * kMmaS1 + 8 * s + c;
                    af[mt][0] = r0[0]; af[mt][1] = r0[8 * kMmaS1]; af[mt][2] = r0[4]; af[mt][3] = r0[8 * kMmaS1 + 4];
                }
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const uint32_t* wr = sWm + kMmaW1 + (nt * 8 + g) * kMmaS1 + 8 * s + c;
                    const uint32_t b0 = wr[0], b1 = wr[4];
                    mma_16816(acc[0][nt], af[0], b0, b1);
                    mma_16816(acc[1][nt], af[1], b0, b1);
                }
            }
            // ---- ReLU + pack: accumulator fragments ARE the next layer's A fragments
            uint32_t hf[2][4][4];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    hf[mt][s][0] = pack_relu_half2(acc[mt][2 * s][0], acc[mt][2 * s][1]);
                    hf[mt][s][1] = pack_relu_half2(acc[mt][2 * s][2], acc[mt][2 * s][3]);
                    hf[mt][s][2] = pack_relu_half2(acc[mt][2 * s + 1][0], acc[mt][2 * s + 1][1]);
                    hf[mt][s][3] = pack_relu_half2(acc[mt][2 * s + 1][2], acc[mt][2 * s + 1][3]);
                }
            // ---- layer 2: K = 64, N = 64
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const float2 b = *reinterpret_cast<const float2*>(sBias + 64 + nt * 8 + 2 * c);
                    acc[mt][nt][0] = b.x; acc[mt][nt][1] = b.y; acc[mt][nt][2] = b.x; acc[mt][nt][3] = b.y;
                }
#pragma unroll
            for (int s = 0; s < 4; ++s)
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) {
                    const uint32_t* wr = sWm + kMmaW2 + (nt * 8 + g) * kMmaS2 + 8 * s + c;
                    const uint32_t b0 = wr[0], b1 = wr[4];
                    mma_16816(acc[0][nt], hf[0][s], b0, b1);
                    mma_16816(acc[1][nt], hf[1][s], b0, b1);
                }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    hf[mt][s][0] = pack_relu_half2(acc[mt][2 * s][0], acc[mt][2 * s][1]);
                    hf[mt][s][1] = pack_relu_half2(acc[mt][2 * s][2], acc[mt][2 * s][3]);
                    hf[mt][s][2] = pack_relu_half2(acc[mt][2 * s + 1][0], acc[mt][2 * s + 1][1]);
                    hf[mt][s][3] = pack_relu_half2(acc[mt][2 * s + 1][2], acc[mt][2 * s + 1][3]);
                }
            // ---- output layer: K = 64, N = 8 (3 real columns)
            float o3[2][4];
            {
                const float2 b = *reinterpret_cast<const float2*>(sBias + 128 + 2 * c);
#pragma unroll
                for (int mt = 0; mt < 2; ++mt) { o3[mt][0] = b.x; o3[mt][1] = b.y; o3[mt][2] = b.x; o3[mt][3] = b.y; }
            }
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const uint32_t* wr = sWm + kMmaW3 + g * kMmaS2 + 8 * s + c;
                const uint32_t b0 = wr[0], b1 = wr[4];
                mma_16816(o3[0], hf[0][s], b0, b1);
                mma_16816(o3[1], hf[1][s], b0, b1);
            }
            // ---- activation + store: lane (g, c) holds columns 2c, 2c+1 of rows g and g+8 of both m-tiles
            if (c < 2) {
#pragma unroll
                for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                    for (int hh = 0; hh < 2; ++hh) {
                        const uint32_t r = mt * 16 + g + 8 * hh;
                        const size_t ir = (size_t)tile * 32u + r;
                        if (ir < n) {
                            const bool dead = ((live >> r) & 1u) == 0u;
                            float v0 = o3[mt][2 * hh], v1 = o3[mt][2 * hh + 1];
                            if (P.out_act == NIV_OUT_SIGMOID) {
                                v0 = __fdividef(1.0f, 1.0f + __expf(-v0));
                                v1 = __fdividef(1.0f, 1.0f + __expf(-v1));
                            }
                            if (dead) { v0 = 0.0f; v1 = 0.0f; }
                            out[3 * ir + 2 * c] = v0;
                            if (c == 0) out[3 * ir + 1] = v1;
                        }
                    }
            }
        } else if (valid) {
            out[3 * i] = 0.0f; out[3 * i + 1] = 0.0f; out[3 * i + 2] = 0.0f;
        }
        tile = tnext;
    }
    // leave the (tile, done) counter pair zero for the slot's next launch
    __syncthreads();
    if (tid == 0 && P.tile_ctr) {
        __threadfence();
        if (atomicAdd(P.tile_ctr + 1, 1u) == gridDim.x - 1) {
            P.tile_ctr[0] = 0u;
            P.tile_ctr[1] = 0u;
            if (P.slot_done) *P.slot_done = P.slot_gen;
        }
    }
}

}  // namespace niv
