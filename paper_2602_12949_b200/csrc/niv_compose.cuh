// niv_compose.cuh -- SURVEY 8(f2): the deferred compose L = rho/pi * E + D + L_e (Eq. 2, Fig. 3) with the
// irradiance at full or at half resolution ("run at reduced resolution ... while still using the
// full size albedo buffer"), half-resolution E upsampled bilinearly with pixel-centre alignment (full-res pixel x at
// half-res coordinate x/2 - 1/4, edge texels clamped).  Included by niv.cu.
//
// HBM-bound: 48 B of full-resolution streams per pixel (albedo, direct, emission in, radiance out) + 12 B (full) or
// 3 B (half) of E.  One thread owns four consecutive pixels of a row = three 128-bit words per stream, read with
// streaming loads (ld.global.cs) and written with streaming stores; the half-resolution E (6 MB per full-HD frame,
// every texel used by ~8 threads) goes through L1/L2 with ordinary loads.
#pragma once

namespace niv {

__device__ __forceinline__ float4 ldcs4(const float* p) { return __ldcs(reinterpret_cast<const float4*>(p)); }

// E of the four pixels (x0..x0+3, y), x0 % 4 == 0, from the half-resolution buffer: 12 floats, channel-interleaved
__device__ __forceinline__ void upsample4(const float* __restrict__ E, uint32_t ew, uint32_t eh, uint32_t x0, uint32_t y,
                                          float e[12]) {
    const int k = (int)(x0 >> 1), j = (int)(y >> 1);
    int j0, j1;
    float ty;
    if (y & 1u) { j0 = j; j1 = min(j + 1, (int)eh - 1); ty = 0.25f; }
    else        { j0 = max(j - 1, 0); j1 = j; ty = 0.75f; }
    const int c[4] = { max(k - 1, 0), k, min(k + 1, (int)ew - 1), min(k + 2, (int)ew - 1) };
    float r[4][3];                                       // the two rows blended, half-res columns k-1 .. k+2
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const float* a = E + ((size_t)j0 * ew + c[q]) * 3;
        const float* b = E + ((size_t)j1 * ew + c[q]) * 3;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            const float va = __ldg(a + ch), vb = __ldg(b + ch);
            r[q][ch] = fmaf(ty, vb - va, va);
        }
    }
    // pixel x0: 0.25 (k-1) + 0.75 k;  x0+1: 0.75 k + 0.25 (k+1);  x0+2: 0.25 k + 0.75 (k+1);  x0+3: 0.75 (k+1) + 0.25 (k+2)
#pragma unroll
    for (int ch = 0; ch < 3; ++ch) {
        e[0 + ch] = fmaf(0.75f, r[1][ch] - r[0][ch], r[0][ch]);
        e[3 + ch] = fmaf(0.25f, r[2][ch] - r[1][ch], r[1][ch]);
        e[6 + ch] = fmaf(0.75f, r[2][ch] - r[1][ch], r[1][ch]);
        e[9 + ch] = fmaf(0.25f, r[3][ch] - r[2][ch], r[2][ch]);
    }
}

// Vector path: w % 4 == 0, all full-resolution pointers 16-byte aligned.  HALF: E is [h/2][w/2][3].
template <bool HALF>
__global__ void __launch_bounds__(256) niv_compose_kernel(const float* __restrict__ E, uint32_t ew, uint32_t eh,
                                                          const float* __restrict__ albedo,
                                                          const float* __restrict__ direct,
                                                          const float* __restrict__ emission,
                                                          float* __restrict__ out, uint32_t w, uint32_t h)
{
    const uint32_t groups_per_row = w >> 2;
    const size_t n_groups = (size_t)groups_per_row * h;
    const float inv_pi = 0.318309886183790671538f;
    for (size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x; g < n_groups; g += (size_t)gridDim.x * blockDim.x) {
        const uint32_t y = (uint32_t)(g / groups_per_row);
        const uint32_t x0 = (uint32_t)(g - (size_t)y * groups_per_row) << 2;
        const size_t o = ((size_t)y * w + x0) * 3;       // first float of the group: a multiple of 12 floats
        float a[12], v[12], e[12];
        *reinterpret_cast<float4*>(a + 0) = ldcs4(albedo + o);
        *reinterpret_cast<float4*>(a + 4) = ldcs4(albedo + o + 4);
        *reinterpret_cast<float4*>(a + 8) = ldcs4(albedo + o + 8);
#pragma unroll
        for (int q = 0; q < 12; ++q) v[q] = 0.0f;
        if (direct) {
            *reinterpret_cast<float4*>(v + 0) = ldcs4(direct + o);
            *reinterpret_cast<float4*>(v + 4) = ldcs4(direct + o + 4);
            *reinterpret_cast<float4*>(v + 8) = ldcs4(direct + o + 8);
        }
        if (emission) {
            float t[12];
            *reinterpret_cast<float4*>(t + 0) = ldcs4(emission + o);
            *reinterpret_cast<float4*>(t + 4) = ldcs4(emission + o + 4);
            *reinterpret_cast<float4*>(t + 8) = ldcs4(emission + o + 8);
#pragma unroll
            for (int q = 0; q < 12; ++q) v[q] += t[q];
        }
        if (HALF) {
            upsample4(E, ew, eh, x0, y, e);
        } else {
            *reinterpret_cast<float4*>(e + 0) = ldcs4(E + o);
            *reinterpret_cast<float4*>(e + 4) = ldcs4(E + o + 4);
            *reinterpret_cast<float4*>(e + 8) = ldcs4(E + o + 8);
        }
#pragma unroll
        for (int q = 0; q < 12; ++q) v[q] = fmaf(a[q] * inv_pi, e[q], v[q]);
        __stcs(reinterpret_cast<float4*>(out + o), *reinterpret_cast<float4*>(v + 0));
        __stcs(reinterpret_cast<float4*>(out + o + 4), *reinterpret_cast<float4*>(v + 4));
        __stcs(reinterpret_cast<float4*>(out + o + 8), *reinterpret_cast<float4*>(v + 8));
    }
}

// Scalar path for any width / alignment: one thread per pixel.
__global__ void __launch_bounds__(256) niv_compose_scalar_kernel(const float* __restrict__ E, uint32_t ew, uint32_t eh,
                                                                 const float* __restrict__ albedo,
                                                                 const float* __restrict__ direct,
                                                                 const float* __restrict__ emission,
                                                                 float* __restrict__ out, uint32_t w, uint32_t h, int half)
{
    const size_t n = (size_t)w * h;
    const float inv_pi = 0.318309886183790671538f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const uint32_t y = (uint32_t)(i / w), x = (uint32_t)(i - (size_t)y * w);
        float e[3];
        if (!half) {
            for (int ch = 0; ch < 3; ++ch) e[ch] = E[i * 3 + ch];
        } else {
            const int k = (int)(x >> 1), j = (int)(y >> 1);
            int c0, c1, j0, j1;
            float tx, ty;
            if (x & 1u) { c0 = k; c1 = min(k + 1, (int)ew - 1); tx = 0.25f; } else { c0 = max(k - 1, 0); c1 = k; tx = 0.75f; }
            if (y & 1u) { j0 = j; j1 = min(j + 1, (int)eh - 1); ty = 0.25f; } else { j0 = max(j - 1, 0); j1 = j; ty = 0.75f; }
            for (int ch = 0; ch < 3; ++ch) {
                const float e00 = E[((size_t)j0 * ew + c0) * 3 + ch], e10 = E[((size_t)j0 * ew + c1) * 3 + ch];
                const float e01 = E[((size_t)j1 * ew + c0) * 3 + ch], e11 = E[((size_t)j1 * ew + c1) * 3 + ch];
                const float r0 = fmaf(ty, e01 - e00, e00), r1 = fmaf(ty, e11 - e10, e10);
                e[ch] = fmaf(tx, r1 - r0, r0);
            }
        }
        for (int ch = 0; ch < 3; ++ch) {
            float v = albedo[i * 3 + ch] * inv_pi * e[ch];
            if (direct) v += direct[i * 3 + ch];
            if (emission) v += emission[i * 3 + ch];
            out[i * 3 + ch] = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// niv_compose_jb: the compose with JOINT-BILATERAL upsampling of half-resolution E ("industry practice
// upsampling methods"; steps J1..J5 of DESIGN.md 3.7): the four half-res texels of the bilinear footprint, each weighted
// by its bilinear weight x (exp(-|x_p - x_q|^2 / 2 sigma^2) max(0, n_p . n_q)^k + 1e-6), renormalised.
// One thread per full-resolution pixel (grid-stride): 72 B of full-resolution streams per pixel (position, normal, albedo,
// direct, emission in, radiance out) + the half-resolution E, position and normal (9 x 4 B per texel, each texel used by
// ~9 pixels: L1 / L2).  inv2s2 = 1 / (2 sigma^2).
__global__ void __launch_bounds__(256) niv_compose_jb_kernel(const float* __restrict__ E, const float* __restrict__ pos_h,
                                                             const float* __restrict__ nrm_h, uint32_t ew, uint32_t eh,
                                                             const float* __restrict__ pos, const float* __restrict__ nrm,
                                                             const float* __restrict__ albedo,
                                                             const float* __restrict__ direct,
                                                             const float* __restrict__ emission, float inv2s2, float power,
                                                             float* __restrict__ out, uint32_t w, uint32_t h)
{
    const size_t n = (size_t)w * h;
    const float inv_pi = 0.318309886183790671538f;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (size_t)gridDim.x * blockDim.x) {
        const uint32_t y = (uint32_t)(p / w), x = (uint32_t)(p - (size_t)y * w);
        const int k = (int)(x >> 1), j = (int)(y >> 1);
        int xs[2], ys[2];
        float tx, ty;                                                       // J1: the bilinear footprint of pixel (x, y)
        if (x & 1u) { xs[0] = k; xs[1] = min(k + 1, (int)ew - 1); tx = 0.25f; } else { xs[0] = max(k - 1, 0); xs[1] = k; tx = 0.75f; }
        if (y & 1u) { ys[0] = j; ys[1] = min(j + 1, (int)eh - 1); ty = 0.25f; } else { ys[0] = max(j - 1, 0); ys[1] = j; ty = 0.75f; }
        float xp[3], np_[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) { xp[d] = __ldcs(pos + 3 * p + d); np_[d] = __ldcs(nrm + 3 * p + d); }
        float acc[3] = {0.f, 0.f, 0.f}, wsum = 0.f;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const size_t t = ((size_t)ys[q >> 1] * ew + (size_t)xs[q & 1]) * 3;
            const float b = ((q & 1) ? tx : 1.0f - tx) * ((q >> 1) ? ty : 1.0f - ty);
            float d2 = 0.f, dot = 0.f;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const float dv = xp[d] - __ldg(pos_h + t + d);
                d2 = fmaf(dv, dv, d2);
                dot = fmaf(np_[d], __ldg(nrm_h + t + d), dot);
            }
            const float g = expf(-d2 * inv2s2) * powf(fmaxf(dot, 0.0f), power);          // J2 (powf(0, 0) = 1, as pow)
            const float wq = b * (g + 1e-6f);                                            // J3
            wsum += wq;
#pragma unroll
            for (int c = 0; c < 3; ++c) acc[c] = fmaf(wq, __ldg(E + t + c), acc[c]);
        }
        const float inv = 1.0f / wsum;
#pragma unroll
        for (int c = 0; c < 3; ++c) {                                                    // J4, J5
            float v = __ldcs(albedo + 3 * p + c) * inv_pi * (acc[c] * inv);
            if (direct) v += __ldcs(direct + 3 * p + c);
            if (emission) v += __ldcs(emission + 3 * p + c);
            __stcs(out + 3 * p + c, v);
        }
    }
}

}  // namespace niv
