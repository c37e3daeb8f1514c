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
    float    cmaxf;     // 2^23 + (N_l - 1) as a float: the clamp of the cell in the "floor by addition" form (locate_bits)
    int32_t  Nm1;       // N_l - 1
    uint32_t R;         // N_l + 1 vertices per side (dense stride)
    uint32_t R2;        // R*R
    uint32_t base;      // first table entry of this level = l*T
    uint32_t dense;     // 1 dense, 0 hashed
    uint32_t cs, cs2;   // cell-block levels: N_l and N_l^2 (cell (cx, cy, cz) is block cx + cs cy + cs2 cz)
    const uint32_t* tb; // this level's first entry = table + base * (F/2) words (a gather address is ONE IMAD.WIDE)
    const uint4* cells; // cell-block copy of the level: per cell its 8 corner entries, corner j at
                        // word j * F/2, i.e. 32 B (F = 2) or 64 B (F = 4) per cell; NULL = gather from tb
};

struct KParams {
    float    amin[3];
    float    ainv[3];           // fl32(1 / fl32(max - min))
    uint32_t L;
    uint32_t tmask;             // T - 1
    uint32_t in_dim;            // L*F + dir_dim + 16*n_params
    uint32_t enc_dim;           // L*F + dir_dim  (what the layer-1 MMA consumes); dir_dim = 16 (SH) or 3 (raw)
    uint32_t n_features;        // F
    uint32_t raw_dir;           // 1: the direction itself is the input (paper), 0: SH-16
    uint32_t n_params;
    uint32_t n_layers;          // hidden + 1
    uint32_t out_act;
    float    t[2];              // per-call scene parameters
    LevelP   lv[kMaxLevels];
    uint32_t* tile_ctr;         // this launch's (tile, done) counter pair, left zero by the launch's last CTA: dynamic
                                // tile scheduling; NULL = static striding (launches recorded into a CUDA graph)
    volatile uint32_t* slot_done; // host-mapped word of the counter slot: the last CTA writes slot_gen (slot free again)
    uint32_t slot_gen;          //   (tile_ctr[2] receives it too: the device-visible "launch complete" word)
    // launch overlap (niv.cu plan_overlap): grid_wait = 1: griddepcontrol.wait before the first access to a caller's
    // buffer (the previous kernel of the stream is complete); 0: the previous launch is one of this library's on
    // disjoint buffers, so this one may run beside its last tiles.  wait_a / wait_b: completion words of the two
    // launches before that one, polled until they reach gen_a / gen_b (NULL: nothing to poll)
    uint32_t grid_wait;
    uint32_t early_read;        // 1: none of this launch's INPUT buffers is written by the two launches that may still be running
                                // (grid_wait = 0 and no overlap with their outputs): the first texel may be requested at once
    uint32_t gen_a, gen_b;
    const uint32_t* wait_a;
    const uint32_t* wait_b;
    const uint32_t* table;      // [L][T] entries of 2 x fp16
    const uint8_t*  wpack;      // packed weights + biases (see niv.cu pack_weights)
    uint32_t wpack_bytes;
    uint32_t kdim[kMaxLayers];  // K of layer k's MMA (multiple of 16)
    uint32_t npad[kMaxLayers];  // N of layer k's MMA (multiple of 16)
    uint32_t w_off[kMaxLayers]; // byte offsets inside wpack
    uint32_t b_off[kMaxLayers];
    uint32_t wparam_off;        // fp32 [width][16*n_params] columns of W1 that multiply the parameter encoding
    uint32_t a_off;             // byte offset of the A tile in shared memory
    uint32_t ones_off;          // byte offset of the constant "ones" A chunk of the bias K-step
    uint32_t misc_off;          // byte offset of folded bias / barriers
    const uint32_t* wmma;       // weights in the layout of the mma.sync A/B kernel (niv_fused_mma.cuh), else NULL
    const float* tparam;        // per-texel scene parameters [n][n_params] (niv_infer_texel_params), else NULL
    uint32_t* dump_a;           // niv_debug_arow (PACKED kernels): every texel's layer-1 A row, [n][dump_words] x 32 bit
    uint32_t dump_words;
    uint32_t gbuf_fmt;          // NIV_GBUF_*: how the caller's G-buffer texels are stored (load_texel_raw / decode_texel)
    uint32_t out_fmt;           // NIV_OUTFMT_*: fp32 x 3 or fp16 x 4 per texel
    float    aext[3];           // fl32(max - min): the scale of the unorm16 position format
    uint32_t img_w, img_h;      // niv_infer_image: the buffers are a row-major img_h x img_w image ...
    uint32_t tiles_x;           // ... cut into 32 x 4 pixel tiles, tiles_x = ceil(img_w / 32) per tile row (else 0)
    // niv_infer_shade (PACKED kernels): the deferred compose as the epilogue, out = albedo / pi * E + direct + emission
    // (Eq. 2, 403); [n][3] fp32 each, shade_albedo NULL = plain inference, the other two may be NULL (zero)
    uint32_t dir_freq;          // raw_dir only: bands of frequency encoding appended to the direction (0 or 4)
    const float* shade_albedo;
    const float* shade_direct;
    const float* shade_emission;
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
// c = min(floor(p), N - 1), w = p - (float)c with p = fl32(u N) in [0, N], N <= 2^22, evaluated without a float -> int
// conversion (F2I / I2F run on the quarter-rate conversion pipe; these are five full-rate FP32 instructions per axis):
//   t  = p + 2^23 rounded toward -inf  = 2^23 + floor(p) exactly (one ulp at 2^23 is 1)
//   tc = min(t, 2^23 + N - 1)          = 2^23 + c
//   cf = tc - 2^23                     = (float)c exactly;   w = fl32(p - cf): the subtraction of step O2
// The bits of tc are 0x4B000000 + c: locate_bits hands them out as they are (the low 24 bits of 0x4B000000 are zero and
// so are those of any multiple of it, which is all the hashed and cell-block index arithmetic needs, see below);
// locate() masks them to the integer cell.
constexpr float kTwo23 = 8388608.0f;
__device__ __forceinline__ void locate_bits(const LevelP& lv, const float u[3], uint32_t cb[3], float w[3]) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const float p = __fmul_rn(u[d], lv.Nf);
        const float tc = fminf(__fadd_rd(p, kTwo23), lv.cmaxf);
        cb[d] = __float_as_uint(tc);
        w[d] = __fsub_rn(p, __fsub_rn(tc, kTwo23));
    }
}
__device__ __forceinline__ void locate(const LevelP& lv, const float u[3], int c[3], float w[3]) {
    uint32_t cb[3];
    locate_bits(lv, u, cb, w);
#pragma unroll
    for (int d = 0; d < 3; ++d) c[d] = (int)(cb[d] & 0x007FFFFFu);
}

// ---------------------------------------------------------------- O3: the 8 corner entries, relative to the level's first entry
// corner j: bit 0 -> +1 in x, bit 1 -> +1 in y, bit 2 -> +1 in z.
// (a ^ b) & c as ONE LOP3 (immLut 0x28); inline PTX so that the optimiser cannot re-associate the XORs into
// a 3-input XOR followed by a separate AND (16 instead of 12 logic ops per level).
__device__ __forceinline__ uint32_t xor_and(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x28;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ void corner_entries_dense(const LevelP& lv, const int c[3], uint32_t e[8]) {
    uint32_t b = (uint32_t)c[0] + lv.R * (uint32_t)c[1] + lv.R2 * (uint32_t)c[2];
#pragma unroll
    for (int j = 0; j < 8; ++j)
        e[j] = b + (j & 1) + ((j >> 1) & 1) * lv.R + ((j >> 2) & 1) * lv.R2;
}
// (c may carry the 0x4B000000 of locate_bits: every term then changes by a multiple of 2^24, which `& tmask` removes,
//  tmask < 2^24)
__device__ __forceinline__ void corner_entries_hashed(uint32_t tmask, const int c[3], uint32_t e[8]) {
    uint32_t x0 = (uint32_t)c[0], x1 = x0 + 1u;
    uint32_t y0 = (uint32_t)c[1] * 2654435761u, y1 = y0 + 2654435761u;   // (c+1)*p == c*p + p  (mod 2^32)
    uint32_t z0 = (uint32_t)c[2] * 805459861u,  z1 = z0 + 805459861u;
    uint32_t yz[4] = { y0 ^ z0, y1 ^ z0, y0 ^ z1, y1 ^ z1 };
#pragma unroll
    for (int j = 0; j < 8; ++j)
        e[j] = xor_and((j & 1) ? x1 : x0, yz[j >> 1], tmask);
}
__device__ __forceinline__ void corner_entries(const LevelP& lv, uint32_t tmask, const int c[3], uint32_t e[8]) {
    if (lv.dense) corner_entries_dense(lv, c, e);
    else corner_entries_hashed(tmask, c, e);
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

// ---------------------------------------------------------------- O4 on the fused path: half2 lerp tree
// F = 2: one table entry IS one half2, so the blend runs on packed fp16 pairs: lerp in x (4), y (2), z (1),
// each lerp = HADD2 (b - a) + HFMA2 (w * d + a) -> 14 instructions per level instead of 16 conversions +
// 16 FFMA + 15 weight ops, and the result is already the packed fp16 pair the A operand wants.
// Error: <= 15 * 2^-11 * max|table| worst case, ~2e-4 * max|table| rms.
// The three fractions of a level travel as fp16 in 1.5 registers: (w_x, w_y) in one word, w_z of two levels in
// another; the lerps read them through the .H0_H0 / .H1_H1 operand selectors of HFMA2 (no unpacking instruction).
__device__ __forceinline__ __half2 u2h(uint32_t v) { return *reinterpret_cast<__half2*>(&v); }
__device__ __forceinline__ uint32_t h2u(__half2 v) { return *reinterpret_cast<uint32_t*>(&v); }
__device__ __forceinline__ __half2 lerp2(__half2 a, __half2 b, __half2 w) { return __hfma2(w, __hsub2(b, a), a); }
__device__ __forceinline__ uint32_t blend8_h2(const uint32_t v[8], __half2 wx, __half2 wy, __half2 wz) {
    const __half2 a0 = lerp2(u2h(v[0]), u2h(v[1]), wx), a1 = lerp2(u2h(v[2]), u2h(v[3]), wx);
    const __half2 a2 = lerp2(u2h(v[4]), u2h(v[5]), wx), a3 = lerp2(u2h(v[6]), u2h(v[7]), wx);
    const __half2 b0 = lerp2(a0, a1, wy), b1 = lerp2(a2, a3, wy);
    return h2u(lerp2(b0, b1, wz));
}

// A batch of NB levels in flight: the 8*NB gathers are issued by batch_issue and consumed by batch_blend, so
// the caller can issue the next batch before blending the current one (software pipelining inside a thread).
// F = fp16 latents per entry: 2 (one 32-bit word per entry, BASELINE.json) or 4 (one 64-bit word, the paper).
template <int NB, int F>
struct Batch {
    uint32_t v[NB][8][F / 2];   // gathered entries (F/2 x half2 each)
    uint32_t wxy[NB];           // (w_x, w_y) of a level as one fp16 pair
    uint32_t wz[(NB + 1) / 2];  // w_z of levels 2k (low half) and 2k + 1 (high half)
};
// The per-level dense / hashed branch is uniform; it also keeps ptxas from sinking a batch's gathers down to their
// first use (measured: with the split known at compile time ptxas interleaves loads and blends, 72 registers, and
// the frame takes 0.208 instead of 0.193 ms even with a warp-level fence between issue and blend).
// 256-bit load (sm_100: one LDG.E.256): a whole F = 2 cell block, or half of an F = 4 one
__device__ __forceinline__ void ldg256(const void* p, uint32_t* r0, uint32_t* r1, uint32_t* r2, uint32_t* r3,
                                       uint32_t* r4, uint32_t* r5, uint32_t* r6, uint32_t* r7) {
    const uint4 a = __ldg(reinterpret_cast<const uint4*>(p)), b = __ldg(reinterpret_cast<const uint4*>(p) + 1);
    *r0 = a.x; *r1 = a.y; *r2 = a.z; *r3 = a.w; *r4 = b.x; *r5 = b.y; *r6 = b.z; *r7 = b.w;
}
// NC: levels 0 .. NC-1 are read from their cell-block copies (known at compile time: a run-time test per level costs
// ten predicated-off instructions on every level and measured 0.198 instead of 0.167 ms per frame; the dense / hashed
// test of the other levels stays a run-time uniform branch, see above)
template <int NB, int F, int NC = 0>
__device__ __forceinline__ void batch_issue(const KParams& P, int l0, const float u[3], Batch<NB, F>& b) {
    static_assert(F == 2 || F == 4, "F = 2 or 4");
    float wzf[NB + 1];
    wzf[NB] = 0.0f;
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const LevelP& lv = P.lv[l0 + q];
        uint32_t cb[3];
        float w[3];
        locate_bits(lv, u, cb, w);
        if (l0 + q < NC) {
            // cell-block level: the 8 corner entries of the cell are one 32-byte (F = 2) / 64-byte (F = 4) block, no
            // corner indices at all.  (the 0x4B000000 of locate_bits leaves the low 24 bits of the sum alone)
            const uint32_t ci = (cb[0] + lv.cs * cb[1] + lv.cs2 * cb[2]) & 0x00FFFFFFu;
            const uint4* blk = lv.cells + (size_t)ci * F;
            if (F == 2) {
                ldg256(blk, &b.v[q][0][0], &b.v[q][1][0], &b.v[q][2][0], &b.v[q][3][0],
                       &b.v[q][4][0], &b.v[q][5][0], &b.v[q][6][0], &b.v[q][7][0]);
            } else {
                ldg256(blk, &b.v[q][0][0], &b.v[q][0][F / 2 - 1], &b.v[q][1][0], &b.v[q][1][F / 2 - 1],
                       &b.v[q][2][0], &b.v[q][2][F / 2 - 1], &b.v[q][3][0], &b.v[q][3][F / 2 - 1]);
                ldg256(blk + 2, &b.v[q][4][0], &b.v[q][4][F / 2 - 1], &b.v[q][5][0], &b.v[q][5][F / 2 - 1],
                       &b.v[q][6][0], &b.v[q][6][F / 2 - 1], &b.v[q][7][0], &b.v[q][7][F / 2 - 1]);
            }
        } else {
            uint32_t e[8];
            if (lv.dense) {
                const int c[3] = {(int)(cb[0] & 0x007FFFFFu), (int)(cb[1] & 0x007FFFFFu), (int)(cb[2] & 0x007FFFFFu)};
                corner_entries_dense(lv, c, e);
            } else {
                const int c[3] = {(int)cb[0], (int)cb[1], (int)cb[2]};
                corner_entries_hashed(P.tmask, c, e);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if (F == 2) {
                    b.v[q][j][0] = __ldg(lv.tb + e[j]);
                } else {
                    const uint2 t = __ldg(reinterpret_cast<const uint2*>(lv.tb) + e[j]);
                    b.v[q][j][0] = t.x;
                    b.v[q][j][F / 2 - 1] = t.y;
                }
            }
        }
        b.wxy[q] = pack_half2(w[0], w[1]);
        wzf[q] = w[2];
    }
#pragma unroll
    for (int q = 0; q < NB; q += 2) b.wz[q / 2] = pack_half2(wzf[q], wzf[q + 1]);
}
template <int NB, int F>
__device__ __forceinline__ void batch_blend(const Batch<NB, F>& b, uint32_t* f) {
#pragma unroll
    for (int q = 0; q < NB; ++q) {
        const __half2 wxy = u2h(b.wxy[q]), wzz = u2h(b.wz[q / 2]);
        const __half2 wx = __low2half2(wxy), wy = __high2half2(wxy);
        const __half2 wz = (q & 1) ? __high2half2(wzz) : __low2half2(wzz);
#pragma unroll
        for (int h = 0; h < F / 2; ++h) {
            uint32_t v[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) v[j] = b.v[q][j][h];
            f[q * (F / 2) + h] = blend8_h2(v, wx, wy, wz);
        }
    }
}

// One group of 4 levels (8 latents = one 16-byte fp16 chunk of the A operand), gathers issued together (F = 2).
template <int NC = 0>
__device__ __forceinline__ uint4 encode_group4(const KParams& P, int l0, const float u[3]) {
    Batch<4, 2> b;
    batch_issue<4, 2, NC>(P, l0, u, b);
    uint32_t f[4];
    batch_blend<4, 2>(b, f);
    return make_uint4(f[0], f[1], f[2], f[3]);
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

// ---------------------------------------------------------------- positional encoding of u in [0, 1] (grid-less models)
// 8 bands, packed (sin, cos) fp16 pairs.  One sincospi and seven angle doublings (sin 2a = 2 sin a cos a,
// cos 2a = 1 - 2 sin^2 a): the error doubles per band, 128 x 6e-8 at the last one, far below the fp16 rounding.
__device__ __forceinline__ void posenc8_packed(float uu, uint32_t o[8]) {
    float s, c;
    sincospif(uu, &s, &c);
    o[0] = pack_half2(s, c);
#pragma unroll
    for (int k = 1; k < 8; ++k) {
        const float s2 = 2.0f * s * c;
        const float c2 = fmaf(-2.0f * s, s, 1.0f);
        s = s2;
        c = c2;
        o[k] = pack_half2(s, c);
    }
}

// frequency encoding of one direction component v in [-1, 1], B bands, as floats (sin, cos per band): one sincospi and
// B - 1 angle doublings (error <= 2^(B-1) * 6e-8, far below the fp16 rounding of the A operand)
template <int B>
__device__ __forceinline__ void dirfreq(float v, float* o) {
    float s, c;
    sincospif(v, &s, &c);
    o[0] = s;
    o[1] = c;
#pragma unroll
    for (int k = 1; k < B; ++k) {
        const float s2 = 2.0f * s * c;
        const float c2 = fmaf(-2.0f * s, s, 1.0f);
        s = s2;
        c = c2;
        o[2 * k] = s;
        o[2 * k + 1] = c;
    }
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

// the same values as fp16 pairs (sin, cos) per band: one A-row chunk of 8 words (per-texel parameters)
// One sincospif and seven angle doublings (as the positional encoding above): the doubling error, < 2^7 * 2^-23 = 1.5e-5,
// is far below the fp16 rounding of the stored value (2.4e-4 at |v| ~ 1); 22 instead of ~90 instructions per parameter.
__device__ __forceinline__ void param_encode8_packed(float t, uint32_t o[8]) { posenc8_packed(t, o); }

// niv_infer_image: tile = 32 x 4 pixels, warp w of the CTA = columns 8w .. 8w+7 of it (an 8 x 4 pixel block, lane =
// 8 * row + column).  A warp's 32 texels then lie in a compact patch of the surface instead of a 32-pixel strip, so
// they share more grid cells: 14 % fewer distinct sectors per warp on the full-HD frame (profiles/r01_v2.md).
// (tile column | tile row << 16) of a tile index: the one division, done by one thread per tile in the fused kernel
__device__ __forceinline__ uint32_t image_tile_xy(const KParams& P, uint32_t tile) {
    const uint32_t ty = tile / P.tiles_x, tx = tile - ty * P.tiles_x;
    return tx | (min(ty, 0xFFFFu) << 16);
           // rows past the image (tile indices past the end) stay invalid
}
__device__ __forceinline__ size_t image_texel_xy(const KParams& P, uint32_t txy, uint32_t tid, bool& valid) {
    const uint32_t x = (txy & 0xFFFFu) * 32u + (tid >> 5) * 8u + (tid & 7u), y = (txy >> 16) * 4u + ((tid >> 3) & 3u);
    valid = x < P.img_w && y < P.img_h;
    return (size_t)y * P.img_w + x;
}
__device__ __forceinline__ size_t image_texel(const KParams& P, uint32_t tile, uint32_t tid, bool& valid) {
    return image_texel_xy(P, image_tile_xy(P, tile), tid, valid);
}

__device__ __forceinline__ void load3(const float* __restrict__ p, size_t i, float v[3]) {
    v[0] = __ldg(p + 3 * i);
    v[1] = __ldg(p + 3 * i + 1);
    v[2] = __ldg(p + 3 * i + 2);
}

// ---------------------------------------------------------------- a12 for NIV_OUTFMT_RGB9E5 (steps Q1..Q4)
// Exact in fp32: the scalings are by powers of two and the sums v + 1/2 stay below 2^10 with integers representable.
__device__ __forceinline__ uint32_t pack_rgb9e5(float r, float g, float b) {
    r = fminf(fmaxf(r, 0.0f), 65408.0f);               // fmaxf(NaN, 0) = 0
    g = fminf(fmaxf(g, 0.0f), 65408.0f);
    b = fminf(fmaxf(b, 0.0f), 65408.0f);
    const float maxc = fmaxf(r, fmaxf(g, b));
    int E = max(-16, (int)(__float_as_uint(maxc) >> 23) - 127) + 16;      // floor(log2 maxc) from the exponent field (zero and subnormals: below -16)
    float scale = __uint_as_float((uint32_t)(127 + 24 - E) << 23);        // 2^(24 - E)
    if (floorf(fmaf(maxc, scale, 0.5f)) == 512.0f) { E += 1; scale *= 0.5f; }
    const uint32_t mr = (uint32_t)floorf(fmaf(r, scale, 0.5f)), mg = (uint32_t)floorf(fmaf(g, scale, 0.5f)),
                   mb = (uint32_t)floorf(fmaf(b, scale, 0.5f));
    return mr | (mg << 9) | (mb << 18) | ((uint32_t)E << 27);
}

// ---------------------------------------------------------------- a1 for the compact G-buffer formats
// DESIGN.md 3.4.  The raw words of texel i travel in the six registers the fp32 texel takes (they are requested a tile
// ahead); decode_texel turns them into the fp32 position and normal the rest of the path is defined on.
//   NIV_GBUF_F32X3      pos[i] = 3 floats, nrm[i] = 3 floats (two arrays)
//   NIV_GBUF_F32X4      the same with a stride of 16 bytes (xyzw, w ignored): one 128-bit load per array
//   NIV_GBUF_P32_OCT16  one array, 16 bytes per texel: x, y, z fp32 | octahedral normal, 2 x snorm16: one 128-bit load
//   NIV_GBUF_P16_OCT8   one array, 8 bytes per texel: position 3 x unorm16 of the model's box | octahedral normal,
//                       2 x snorm8: one 64-bit load
// The position decode is a pinned fp32 sequence (it decides cells): x = fl32(fl32(fl32((float)q * fl32(1/65535)) * ext) + min).
__device__ __forceinline__ void load_texel_raw(uint32_t fmt, const float* __restrict__ a, const float* __restrict__ b,
                                               size_t i, float pr[3], float nr[3]) {
    if (fmt == 0) {
        load3(a, i, pr);
        load3(b, i, nr);
    } else if (fmt == 1) {
        const float4 p4 = __ldg(reinterpret_cast<const float4*>(a) + i), n4 = __ldg(reinterpret_cast<const float4*>(b) + i);
        pr[0] = p4.x; pr[1] = p4.y; pr[2] = p4.z;
        nr[0] = n4.x; nr[1] = n4.y; nr[2] = n4.z;
    } else if (fmt == 2) {
        const uint4 t = __ldg(reinterpret_cast<const uint4*>(a) + i);
        pr[0] = __uint_as_float(t.x); pr[1] = __uint_as_float(t.y); pr[2] = __uint_as_float(t.z);
        nr[0] = __uint_as_float(t.w);
    } else {
        const uint2 t = __ldg(reinterpret_cast<const uint2*>(a) + i);
        pr[0] = __uint_as_float(t.x); pr[1] = __uint_as_float(t.y);
    }
}
// octahedral direction: (fx, fy) in [-1, 1]^2 -> unit vector
__device__ __forceinline__ void oct_decode(float fx, float fy, float n[3]) {
    float z = 1.0f - fabsf(fx) - fabsf(fy), x = fx, y = fy;
    if (z < 0.0f) {
        x = copysignf(1.0f - fabsf(fy), fx);
        y = copysignf(1.0f - fabsf(fx), fy);
    }
    const float r = rsqrtf(x * x + y * y + z * z);
    n[0] = x * r; n[1] = y * r; n[2] = z * r;
}
__device__ __forceinline__ void decode_texel(const KParams& P, const float pr[3], const float nr[3], float p[3], float n[3]) {
    if (P.gbuf_fmt <= 1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { p[d] = pr[d]; n[d] = nr[d]; }
    } else if (P.gbuf_fmt == 2) {
#pragma unroll
        for (int d = 0; d < 3; ++d) p[d] = pr[d];
        const uint32_t o = __float_as_uint(nr[0]);
        const int ox = (int)(short)(o & 0xFFFFu), oy = (int)(short)(o >> 16);
        if (ox == -32768 && oy == -32768) { n[0] = n[1] = n[2] = 0.0f; }           // background
        else oct_decode((float)ox * (1.0f / 32767.0f), (float)oy * (1.0f / 32767.0f), n);
    } else {
        const uint32_t w0 = __float_as_uint(pr[0]), w1 = __float_as_uint(pr[1]);
        const uint32_t q[3] = {w0 & 0xFFFFu, w0 >> 16, w1 & 0xFFFFu};
#pragma unroll
        for (int d = 0; d < 3; ++d)
            p[d] = __fadd_rn(__fmul_rn(__fmul_rn((float)q[d], 1.0f / 65535.0f), P.aext[d]), P.amin[d]);
        const int ox = (int)(signed char)((w1 >> 16) & 0xFFu), oy = (int)(signed char)(w1 >> 24);
        if (ox == -128 && oy == -128) { n[0] = n[1] = n[2] = 0.0f; }
        else oct_decode((float)ox * (1.0f / 127.0f), (float)oy * (1.0f / 127.0f), n);
    }
}

}  // namespace niv
