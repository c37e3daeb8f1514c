// niv_device.cuh -- kernel parameter block and the per-texel device functions shared by the fused kernel,
// the stand-alone encode kernel and the debug dump (steps O0..O7).
// The integer path O0..O3 exists ONCE, here; parity of indices is checked on the debug dump that calls it.
#pragma once
#include <cstdint>
#include <cuda_fp16.h>
#include <cuda_runtime.h>

namespace niv {

constexpr int kMaxLevels = 16;
constexpr int kMaxLayers = 4;       // up to 3 hidden + output
constexpr int kTile = 128;          // texels per CTA tile = MMA M = TMEM lanes

struct LevelP {
    float    Nf;        // (float)N_l, exact
    int32_t  Nm1;       // N_l - 1
    uint32_t R;         // N_l + 1 vertices per side (dense stride)
    uint32_t R2;        // R*R
    uint32_t base;      // first table entry of this level = l*T
    uint32_t dense;     // 1 dense, 0 hashed
};

struct KParams {
    float    amin[3];
    float    ainv[3];           // fl32(1 / fl32(max - min))
    uint32_t L;
    uint32_t tmask;             // T - 1
    uint32_t in_dim;            // L*F + 16 + 16*n_params
    uint32_t enc_dim;           // L*F + 16     (what the layer-1 MMA consumes)
    uint32_t n_params;
    uint32_t n_layers;          // hidden + 1
    uint32_t out_act;
    float    t[2];              // per-call scene parameters
    LevelP   lv[kMaxLevels];
    const uint32_t* table;      // [L][T] entries of 2 x fp16
    const uint8_t*  wpack;      // packed weights + biases (see niv.cu pack_weights)
    uint32_t wpack_bytes;
    uint32_t kdim[kMaxLayers];  // K of layer k's MMA (multiple of 16)
    uint32_t npad[kMaxLayers];  // N of layer k's MMA (multiple of 16)
    uint32_t w_off[kMaxLayers]; // byte offsets inside wpack
    uint32_t b_off[kMaxLayers];
    uint32_t wparam_off;        // fp32 [width][16*n_params] columns of W1 that multiply the parameter encoding
    uint32_t a_off;             // byte offset of the A tile in shared memory
    uint32_t misc_off;          // byte offset of folded bias / barriers
};

// ---------------------------------------------------------------- O0: background / non-finite mask
__device__ __forceinline__ bool texel_masked(const float p[3], const float n[3]) {
    bool fin = isfinite(p[0]) && isfinite(p[1]) && isfinite(p[2]) && isfinite(n[0]) && isfinite(n[1]) && isfinite(n[2]);
    bool zero = (n[0] == 0.0f) && (n[1] == 0.0f) && (n[2] == 0.0f);
    return !fin || zero;
}

// ---------------------------------------------------------------- O1: normalise (fp32, one rounded op each)
__device__ __forceinline__ void normalise(const KParams& P, const float p[3], float u[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float v = __fmul_rn(__fsub_rn(p[d], P.amin[d]), P.ainv[d]);
        u[d] = fminf(fmaxf(v, 0.0f), 1.0f);
    }
}

// ---------------------------------------------------------------- O2: locate the cell on one level
__device__ __forceinline__ void locate(const LevelP& lv, const float u[3], int c[3], float w[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float p = __fmul_rn(u[d], lv.Nf);
        int ci = min(__float2int_rd(p), lv.Nm1);
        c[d] = ci;
        w[d] = __fsub_rn(p, (float)ci);
    }
}

// ---------------------------------------------------------------- O3: the 8 corner entries (level base added)
// corner j: bit 0 -> +1 in x, bit 1 -> +1 in y, bit 2 -> +1 in z.
__device__ __forceinline__ void corner_entries(const LevelP& lv, uint32_t tmask, const int c[3], uint32_t e[8]) {
    if (lv.dense) {
        uint32_t b = lv.base + (uint32_t)c[0] + lv.R * (uint32_t)c[1] + lv.R2 * (uint32_t)c[2];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            e[j] = b + (j & 1) + ((j >> 1) & 1) * lv.R + ((j >> 2) & 1) * lv.R2;
    } else {
        uint32_t x0 = (uint32_t)c[0], x1 = x0 + 1u;
        uint32_t y0 = (uint32_t)c[1] * 2654435761u, y1 = y0 + 2654435761u;   // (c+1)*p == c*p + p  (mod 2^32)
        uint32_t z0 = (uint32_t)c[2] * 805459861u,  z1 = z0 + 805459861u;
        uint32_t yz[4] = { y0 ^ z0, y1 ^ z0, y0 ^ z1, y1 ^ z1 };
#pragma unroll
        for (int j = 0; j < 8; ++j)
            e[j] = lv.base + ((((j & 1) ? x1 : x0) ^ yz[j >> 1]) & tmask);
    }
}

// ---------------------------------------------------------------- O4: trilinear blend of 8 (fp16 x 2) entries
__device__ __forceinline__ float2 blend8(const uint32_t v[8], const float w[3]) {
    const float wx1 = w[0], wx0 = 1.0f - w[0];
    const float wy1 = w[1], wy0 = 1.0f - w[1];
    const float wz1 = w[2], wz0 = 1.0f - w[2];
    const float wyz[4] = { wy0 * wz0, wy1 * wz0, wy0 * wz1, wy1 * wz1 };
    float2 acc = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float om = ((j & 1) ? wx1 : wx0) * wyz[j >> 1];
        __half2 h = *reinterpret_cast<const __half2*>(&v[j]);
        float2 f = __half22float2(h);          // exact, fp16 subnormals included
        acc.x = fmaf(om, f.x, acc.x);
        acc.y = fmaf(om, f.y, acc.y);
    }
    return acc;
}

__device__ __forceinline__ uint32_t pack_half2(float a, float b) {
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
}

// One group of 4 levels (8 latents = one 16-byte fp16 chunk of the A operand): all 32 gathers are issued
// before the first use so that they are in flight together.
__device__ __forceinline__ void encode_group4(const KParams& P, int l0, const float u[3], float2 f[4]) {
    uint32_t e[4][8];
    float w[4][3];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        int c[3];
        locate(P.lv[l0 + q], u, c, w[q]);
        corner_entries(P.lv[l0 + q], P.tmask, c, e[q]);
    }
    uint32_t v[4][8];
#pragma unroll
    for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int j = 0; j < 8; ++j) v[q][j] = __ldg(P.table + e[q][j]);
#pragma unroll
    for (int q = 0; q < 4; ++q) f[q] = blend8(v[q], w[q]);
}

// ---------------------------------------------------------------- O5: real SH, bands 0..3 (reading #13)
__device__ __forceinline__ void sh16(const float n[3], float o[16]) {
    const float x = n[0], y = n[1], z = n[2];
    const float xx = x * x, yy = y * y, zz = z * z;
    o[0]  = 0.28209479177387814f;
    o[1]  = 0.4886025119029199f * y;
    o[2]  = 0.4886025119029199f * z;
    o[3]  = 0.4886025119029199f * x;
    o[4]  = 1.0925484305920792f * x * y;
    o[5]  = 1.0925484305920792f * y * z;
    o[6]  = 0.31539156525252005f * (3.0f * zz - 1.0f);
    o[7]  = 1.0925484305920792f * x * z;
    o[8]  = 0.5462742152960396f * (xx - yy);
    o[9]  = 0.5900435899266435f * y * (3.0f * xx - yy);
    o[10] = 2.890611442640554f * x * y * z;
    o[11] = 0.4570457994644658f * y * (5.0f * zz - 1.0f);
    o[12] = 0.3731763325901154f * z * (5.0f * zz - 3.0f);
    o[13] = 0.4570457994644658f * x * (5.0f * zz - 1.0f);
    o[14] = 1.445305721320277f * z * (xx - yy);
    o[15] = 0.5900435899266435f * x * (xx - 3.0f * yy);
}

// ---------------------------------------------------------------- O6: sin/cos(2^k pi t), k = 0..7
__device__ __forceinline__ void param_encode8(float t, float o[16]) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        float s, c;
        sincospif(t * (float)(1 << k), &s, &c);      // 2^k * t is exact in fp32
        o[2 * k] = s;
        o[2 * k + 1] = c;
    }
}

__device__ __forceinline__ void load3(const float* __restrict__ p, size_t i, float v[3]) {
    v[0] = __ldg(p + 3 * i);
    v[1] = __ldg(p + 3 * i + 1);
    v[2] = __ldg(p + 3 * i + 2);
}

}  // namespace niv
