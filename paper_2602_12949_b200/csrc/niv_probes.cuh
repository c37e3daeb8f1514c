// niv_probes.cuh -- SURVEY 8(f4): query of a regular grid of SH-2 irradiance probes, the paper's baseline
// (App. A: 9 coefficients x 3 channels in half precision, trilinear weights x cosine fall-off,
// weights clamped to 1e-6, renormalised; SPEC.md:341-346 basis, 365-368 query, 396 storage order).  Included by niv.cu.
// Steps P0..P7 of DESIGN.md 3.6; the cell (P1-P2) uses the fp32 op sequence of O1-O2, so it is bit-exact.
//
// Device layout: one probe = 64 bytes = 27 fp16 (coefficient k, channel c at 3k + c) + 5 zeros, x fastest: a probe
// is four aligned 128-bit loads = two sectors, and the two x neighbours of a cell are one 128-byte line when the cell
// index is even.  One thread per texel; the 8 probes of a cell are fetched two at a time (8 loads in flight).
#pragma once

namespace niv {

struct ProbeParams {
    float    amin[3], amax[3];
    float    ainv[3];           // fl32(1 / fl32(max - min))
    float    nf[3];             // (float)(n_d - 1): cells per axis
    int32_t  nm2[3];            // n_d - 2: the last cell
    float    step[3];           // fl32(fl32(max - min) / (n_d - 1)): probe spacing
    uint32_t dims[3];
    uint32_t falloff;           // 1: cosine fall-off on
    const uint4* probes;        // [nz][ny][nx][4] x 16 bytes
};

__device__ __forceinline__ void sh9(const float n[3], float o[9]) {
    const float x = n[0], y = n[1], z = n[2];
    o[0] = 0.28209479177387814f;
    o[1] = 0.4886025119029199f * y;
    o[2] = 0.4886025119029199f * z;
    o[3] = 0.4886025119029199f * x;
    o[4] = 1.0925484305920792f * x * y;
    o[5] = 1.0925484305920792f * y * z;
    o[6] = 0.31539156525252005f * (3.0f * z * z - 1.0f);
    o[7] = 1.0925484305920792f * x * z;
    o[8] = 0.5462742152960396f * (x * x - y * y);
}

// P1-P2: the cell and the fractions (fp32, one rounded op each, as O1-O2)
__device__ __forceinline__ void probe_locate(const ProbeParams& G, const float p[3], int c[3], float w[3], float xc[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        float u = __fmul_rn(__fsub_rn(p[d], G.amin[d]), G.ainv[d]);
        u = fminf(fmaxf(u, 0.0f), 1.0f);
        const float pp = __fmul_rn(u, G.nf[d]);
        const int ci = min(__float2int_rd(pp), G.nm2[d]);
        c[d] = ci;
        w[d] = __fsub_rn(pp, (float)ci);
        xc[d] = fminf(fmaxf(p[d], G.amin[d]), G.amax[d]);
    }
}

// P3-P5 for corner j: probe index and its clamped (not yet normalised) weight
__device__ __forceinline__ float probe_weight(const ProbeParams& G, const int c[3], const float w[3], const float xc[3],
                                              const float n[3], int j, uint32_t& index) {
    float wt = 1.0f, dv[3], len2 = 0.0f;
    uint32_t v[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int bit = (j >> d) & 1;
        v[d] = (uint32_t)(c[d] + bit);
        wt *= bit ? w[d] : 1.0f - w[d];
        dv[d] = __fsub_rn(__fadd_rn(__fmul_rn((float)v[d], G.step[d]), G.amin[d]), xc[d]);   // pinned (reading P-e)
        len2 = fmaf(dv[d], dv[d], len2);
    }
    if (G.falloff && len2 > 0.0f) {
        const float dot = (dv[0] * n[0] + dv[1] * n[1] + dv[2] * n[2]) * rsqrtf(len2);
        wt *= fmaxf(dot, 0.0f);
    }
    index = v[0] + G.dims[0] * (v[1] + G.dims[1] * v[2]);
    return fmaxf(wt, 1e-6f);
}

__device__ __forceinline__ void probe_accumulate(const uint4 q[4], const float wy[9], float e[3]) {
    const uint32_t words[16] = {q[0].x, q[0].y, q[0].z, q[0].w, q[1].x, q[1].y, q[1].z, q[1].w,
                                q[2].x, q[2].y, q[2].z, q[2].w, q[3].x, q[3].y, q[3].z, q[3].w};
    float c[32];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&words[k]));
        c[2 * k] = f.x;
        c[2 * k + 1] = f.y;
    }
#pragma unroll
    for (int k = 0; k < 9; ++k)
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) e[ch] = fmaf(wy[k], c[3 * k + ch], e[ch]);
}

__global__ void __launch_bounds__(256) niv_probes_query_kernel(const __grid_constant__ ProbeParams G,
                                                               const float* __restrict__ pos,
                                                               const float* __restrict__ nrm,
                                                               float* __restrict__ out, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float p[3], nv[3];
    load3(pos, i, p);
    load3(nrm, i, nv);
    float e[3] = {0.f, 0.f, 0.f};
    if (!texel_masked(p, nv)) {                           // P0
        int c[3];
        float w[3], xc[3];
        probe_locate(G, p, c, w, xc);
        float wt[8], sum = 0.0f;
        uint32_t idx[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            wt[j] = probe_weight(G, c, w, xc, nv, j, idx[j]);
            sum += wt[j];
        }
        const float inv = 1.0f / sum;                     // P6
        float Y[9];
        sh9(nv, Y);
#pragma unroll
        for (int j = 0; j < 8; j += 2) {                  // P7, two probes (8 x 128 bits) in flight
            uint4 qa[4], qb[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                qa[k] = __ldg(G.probes + (size_t)idx[j] * 4 + k);
                qb[k] = __ldg(G.probes + (size_t)idx[j + 1] * 4 + k);
            }
            float wy[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) wy[k] = wt[j] * inv * Y[k];
            probe_accumulate(qa, wy, e);
#pragma unroll
            for (int k = 0; k < 9; ++k) wy[k] = wt[j + 1] * inv * Y[k];
            probe_accumulate(qb, wy, e);
        }
    }
    out[3 * i] = e[0];
    out[3 * i + 1] = e[1];
    out[3 * i + 2] = e[2];
}

// fp16 [27] per probe -> the padded 64-byte device records
__global__ void niv_probes_pack_kernel(const uint16_t* __restrict__ src, uint16_t* __restrict__ dst, size_t n_probes)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_probes * 32) return;
    const size_t pr = t >> 5;
    const uint32_t k = (uint32_t)(t & 31);
    dst[t] = k < 27 ? src[pr * 27 + k] : (uint16_t)0;
}

// Census for the gather roofline of the query: distinct 32-byte sectors (two per probe) among a warp's 8 x 32 probe
// records, summed over the grid.  counts[0] = sectors, counts[1] = active texels.
__global__ void __launch_bounds__(128) niv_probes_census_kernel(const __grid_constant__ ProbeParams G,
                                                                const float* __restrict__ pos,
                                                                const float* __restrict__ nrm, size_t n,
                                                                unsigned long long* __restrict__ counts)
{
    __shared__ uint32_t s_idx[4][256];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    float p[3] = {0.f, 0.f, 0.f}, nv[3] = {0.f, 0.f, 0.f};
    if (i < n) { load3(pos, i, p); load3(nrm, i, nv); }
    const bool masked = i >= n || texel_masked(p, nv);
    uint32_t idx[8];
    if (!masked) {
        int c[3];
        float w[3], xc[3];
        probe_locate(G, p, c, w, xc);
#pragma unroll
        for (int j = 0; j < 8; ++j) (void)probe_weight(G, c, w, xc, nv, j, idx[j]);
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) s_idx[warp][lane * 8 + j] = masked ? 0xFFFFFFFFu : idx[j];
    __syncwarp();
    uint32_t distinct = 0;
    for (int q = 0; q < 8; ++q) {
        const uint32_t me = lane * 8 + q, v = s_idx[warp][me];
        if (v == 0xFFFFFFFFu) continue;
        bool first = true;
        for (uint32_t k = 0; k < me; ++k) first &= (s_idx[warp][k] != v);
        distinct += first;
    }
    for (int o = 16; o; o >>= 1) distinct += __shfl_xor_sync(0xffffffffu, distinct, o);
    const uint32_t n_act = __popc(__ballot_sync(0xffffffffu, !masked));
    if (lane == 0 && n_act) {
        atomicAdd(&counts[0], 2ull * distinct);
        atomicAdd(&counts[1], (unsigned long long)n_act);
    }
}

}  // namespace niv
