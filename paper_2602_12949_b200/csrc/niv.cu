// niv.cu -- libniv: kernels and the C ABI declared in include/niv.h.
//
// Kernels (all sm_100a, hand-written):
//   niv_fused_kernel         (niv_fused.cuh) rows a0..a12 of DESIGN.md section 1, hidden width <= 64: tcgen05 / TMEM
//   niv_fused_w128_kernel    (niv_fused_w128.cuh) the same for hidden width 128
//   niv_fused_mma_kernel     (niv_fused_mma.cuh) the mma.sync A/B kernel (NIV_MMA_SYNC=1 at niv_create)
//   niv_compose_kernel       (niv_compose.cuh) deferred compose, SURVEY 8(f2)
//   niv_encode_kernel        rows a1..a9 only (stand-alone encoding, fp16 features to global memory).
//   niv_debug_kernel         index / cell / fraction / fp32 feature dump through the same device functions.
//   niv_probe_gather_kernel  random-sector gather micro-benchmark (the measured L2-gather roofline).
//   niv_sector_census_kernel distinct sectors per warp and level (the numerator of that roofline).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <atomic>
#include <cmath>
#include <mutex>
#include <new>
#include <type_traits>
#include <unordered_map>
#include <vector>

#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include "../../include/niv.h"
#include "niv_device.cuh"
#include "niv_tc.cuh"

#include "niv_fused.cuh"
#include "niv_fused_w128.cuh"
#include "niv_fused_mma.cuh"
#include "niv_compose.cuh"
#include "niv_probes.cuh"
namespace niv {

// =====================================================================================================
// stand-alone encode (fp16 features to global) and debug dump
// =====================================================================================================
// NC: levels 0 .. NC-1 from their cell-block copies (as the fused kernel); groups of four levels, at most four groups
template <int NC>
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
#pragma unroll
    for (int g = 0; g < kMaxLevels / 4; ++g)
        if ((uint32_t)g < n_groups) row[g] = encode_group4<NC>(P, g * 4, u);
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
            dd = 3 + 6 * P.dir_freq;
            for (int k = 0; k < 3; ++k) feat[i * P.in_dim + o + k] = masked ? 0.f : nv[k];
            for (uint32_t d = 0; d < 3; ++d)         // accurate per-band sincospi (the fused path doubles angles)
                for (uint32_t k = 0; k < P.dir_freq; ++k) {
                    float sn, cs;
                    sincospif(nv[d] * (float)(1u << k), &sn, &cs);
                    feat[i * P.in_dim + o + 3 + 2 * (P.dir_freq * d + k)] = masked ? 0.f : sn;
                    feat[i * P.in_dim + o + 3 + 2 * (P.dir_freq * d + k) + 1] = masked ? 0.f : cs;
                }
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
// cell-block copy of a coarse level: block (cx, cy, cz) = the 8 corner entries of that cell, found
// through the same corner_entries() as every other kernel.  One thread per cell; run once per niv_load_params.
// =====================================================================================================
__global__ void __launch_bounds__(256) niv_build_cells_kernel(const __grid_constant__ KParams P, uint32_t level,
                                                              uint32_t* __restrict__ dst, uint32_t n_cells)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_cells) return;
    const LevelP& lv = P.lv[level];
    const uint32_t N = lv.cs;
    const int c[3] = {(int)(i % N), (int)((i / N) % N), (int)(i / (N * N))};
    uint32_t e[8];
    corner_entries(lv, P.tmask, c, e);
    const uint32_t FW = P.n_features >> 1;
    for (int j = 0; j < 8; ++j)
        for (uint32_t h = 0; h < FW; ++h) dst[((size_t)i * 8 + j) * FW + h] = lv.tb[(size_t)e[j] * FW + h];
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
                                                               uint32_t* __restrict__ sink, cudaTextureObject_t tex)
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
            } else if (PATTERN == 7) {          // as 0 but L1 no-allocate
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                asm volatile("ld.global.nc.L1::no_allocate.b32 %0, [%1];" : "=r"(v[k]) : "l"(buf + a));
            } else if (PATTERN == 8) {          // as 0 through the texture path (TLD, 32-bit texel index)
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                v[k] = tex1Dfetch<unsigned int>(tex, (int)a);
            } else {                            // 9: as 0, alternating between the LSU path (LDG) and the texture path
                const uint32_t a = mix32((gid * 0x9E3779B9u) ^ salt) & word_mask;
                v[k] = (k & 1) ? tex1Dfetch<unsigned int>(tex, (int)a) : __ldg(buf + a);
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
// counts[32] = active texels.  These are the addresses of the table as niv_load_params receives it ([L][T] entries):
// the algorithmic figure of SURVEY.md 8(d).  counts[33..33+L) = the sectors the fused kernel really touches: the same
// on gathered levels, the distinct cell blocks (32 B, or 64 B = 2 sectors for F = 4) on cell-block levels.
__global__ void __launch_bounds__(128) niv_sector_census_kernel(const __grid_constant__ KParams P,
                                                                const float* __restrict__ pos,
                                                                const float* __restrict__ nrm, size_t n,
                                                                unsigned long long* __restrict__ counts, int with_cells)
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
        uint32_t touched = sec;
        if (with_cells && P.lv[l].cs) {                                       // distinct cells among the warp's texels
            int c[3] = {0, 0, 0}; float w[3];
            if (!masked) locate(P.lv[l], u, c, w);
            const uint32_t ci = masked ? 0xFFFFFFFFu : (uint32_t)c[0] + P.lv[l].cs * (uint32_t)c[1] + P.lv[l].cs2 * (uint32_t)c[2];
            const uint32_t same = __match_any_sync(0xffffffffu, ci);
            const bool first = !masked && (__ffs(same) - 1 == (int)lane);
            touched = __popc(__ballot_sync(0xffffffffu, first)) * (P.n_features == 4 ? 2u : 1u);
        }
        if (lane == 0 && touched && with_cells) atomicAdd(&counts[33 + l], (unsigned long long)touched);
    }
}

}  // namespace niv

// =====================================================================================================
// host side: the C ABI
// =====================================================================================================
using namespace niv;

constexpr int kCellBudgetMB = 320;      // default budget of the cell-block copies of the coarse levels
constexpr uint32_t kCtrSlots = 2048;     // dynamically scheduled launches of one model that may be in flight at once

typedef void (*fused_fn)(KParams, const float*, const float*, float*, size_t, uint32_t);

struct FusedKernel {                    // one instantiation, with the launch shape its resources allow
    fused_fn fn = nullptr;
    uint32_t grid = 0, smem = 0, ctas_per_sm = 0;
};

struct niv_model {
    niv_config cfg;
    niv_info info;
    KParams kp;
    uint32_t* d_table = nullptr;
    uint64_t lev_entries[kMaxLevels] = {};         // entries a level really has: (N + 1)^3 (dense) or T (hashed)
    uint64_t dev_table_bytes = 0;                  // device storage: the levels back to back, each padded to 8 entries
    uint32_t kernel_levels = 0;                    // levels the fused kernels run (n_levels rounded up to whole batches)
    uint32_t k_shift = 0;                          // (kernel_levels - n_levels) * F: where the direction columns of W1 move to
    uint32_t* d_cells = nullptr;                   // cell-block copies of the coarse levels (KParams::lv[].cells)
    uint64_t cell_off[kMaxLevels] = {};            //   byte offset of a level's blocks in d_cells
    uint8_t* d_wpack = nullptr;
    std::vector<uint32_t> layer_out, layer_in;     // true (unpadded) shapes
    bool loaded = false;
    FusedKernel fused;                             // niv_infer
    FusedKernel fused_host;                        // niv_infer_host, pinned buffers: 128-bit output stores
    FusedKernel fused_pk, fused_host_pk;           // *_packed entry points: compact G-buffer formats / fp16 output
    FusedKernel fused_img;                         // niv_infer_image: 8 x 4 pixel blocks per warp
    FusedKernel fused_img_pk;                      //   ... with the compact formats / the shading epilogue (cell-block models)
    FusedKernel fused_tp;                          // niv_infer_texel_params: parameter columns as K-steps of layer 1,
    KParams kp_tp;                                 //   with its own packed weights and shared-memory layout
    uint8_t* d_wpack_tp = nullptr;
    bool mma_kernel = false;                       // NIV_MMA_SYNC=1: the per-warp mma.sync A/B kernel (32-texel tiles)
    uint32_t* d_wmma = nullptr;
    // knobs read ONCE, at niv_create (never on the call path)
    bool pdl = true;                               // NIV_PDL=0: no programmatic stream serialisation
    bool overlap = true;                           // NIV_OVERLAP=0: every launch waits for the previous kernel of its stream
    bool image_linear = false;                     // NIV_IMAGE_LINEAR=1: niv_infer_image through the linear kernel
    bool host_staged = false;                      // NIV_HOST_STAGED=1: niv_infer_host always through staging copies
    bool debug = false;                            // NIV_DEBUG=1: resource report on stderr
    // tile-counter slots (dynamic tile scheduling): 128 B apart on the device; a host-mapped word per slot carries
    // the generation of the last launch that FINISHED on it, so a slot is handed out again only when it is free
    uint32_t* d_ctr = nullptr;
    volatile uint32_t* h_done = nullptr;           // pinned, mapped
    uint32_t* d_done = nullptr;                    // its device address
    uint32_t slot_gen[kCtrSlots] = {};             // generation of the last launch ISSUED on the slot
    uint32_t slot_next = 0;
    std::mutex slot_mu;
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
static bool env_flag(const char* name, bool dflt) {
    const char* s = getenv(name);
    return s ? atoi(s) != 0 : dflt;
}

// Resident CTAs per SM from the kernel's own resource use.  (cudaOccupancyMaxActiveBlocksPerMultiprocessor
// answers 1 for kernels that allocate tensor memory on driver 580 -- measured, DESIGN.md section 6 -- so it is not used.)
static int setup_kernel(niv_model* m, FusedKernel& k, int tmem_cols, const char* name) {
    if (!k.fn) return NIV_OK;
    cudaFuncAttributes fa;
    NIV_CUDA(cudaFuncGetAttributes(&fa, k.fn));
    cudaDeviceProp prop;
    NIV_CUDA(cudaGetDeviceProperties(&prop, m->cfg.device));
    const int regs_per_cta = ((fa.numRegs + 7) / 8 * 8) * kTile;
    // 96 columns = two allocations per CTA (64, then 32): eight CTAs holding 64 each and waiting for 32 would wait for
    // ever, so such a kernel must never have eight CTAs on an SM (launches overlap: the grid size alone does not say).
    // Today's kernels take >= 72 registers (seven CTAs); should one drop to <= 64, its shared memory is padded to an
    // eighth of the SM's so that seven fit at most.
    if (tmem_cols == 96 && prop.regsPerMultiprocessor / regs_per_cta >= 8)
        k.smem = std::max<uint32_t>(k.smem, (uint32_t)prop.sharedMemPerMultiprocessor / 8 + 128);
    NIV_CUDA(cudaFuncSetAttribute(k.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.smem));
    const int smem_per_cta = (int)round_up(k.smem + (uint32_t)fa.sharedSizeBytes + (uint32_t)prop.reservedSharedMemPerBlock, 128);
    int blocks = prop.regsPerMultiprocessor / regs_per_cta;
    blocks = std::min(blocks, (int)prop.sharedMemPerMultiprocessor / smem_per_cta);
    blocks = std::min(blocks, prop.maxThreadsPerMultiProcessor / kTile);
    if (tmem_cols) blocks = std::min(blocks, 512 / tmem_cols);           // tensor memory: 512 columns per SM
    blocks = std::min(blocks, 32);
    if (blocks < 1) return NIV_ERR_UNSUPPORTED;
    // the gathers live on L1 hits: ask for the smallest shared-memory carve-out that still holds `blocks` CTAs, the
    // rest of the 228 KB becomes L1
    int pct = (blocks * smem_per_cta * 100 + (int)prop.sharedMemPerMultiprocessor - 1) / (int)prop.sharedMemPerMultiprocessor;
    pct = std::min(100, std::max(0, pct));
    NIV_CUDA(cudaFuncSetAttribute(k.fn, cudaFuncAttributePreferredSharedMemoryCarveout, pct));
    if (m->debug)
        fprintf(stderr, "[niv] %s: %d regs, %zu B local, %d B smem/CTA, %d TMEM cols -> %d CTAs/SM, carve-out %d %%\n", name,
                fa.numRegs, (size_t)fa.localSizeBytes, smem_per_cta, tmem_cols, blocks, pct);
    k.ctas_per_sm = (uint32_t)blocks;
    k.grid = (uint32_t)blocks * m->info.num_sms;
    return NIV_OK;
}

// ---- which instantiation serves which model -----------------------------------------------------------------------
// O = output as 128-bit stores (pinned host buffers), NPT = per-texel parameters, IMG = image tiling,
// C = read the coarsest min(L, kCellLevels) levels from their cell-block copies
// how many: BASELINE.json's family (F = 2) seven (0.1673 -> 0.1613 / 0.1585 / 0.1567 ms per full-HD frame with 3 / 4 / 5
// levels; the sixth, N = 121, 57 MB: 0.1532 -> 0.1511 ms; the seventh, N = 182, 193 MB: 0.1508 -> 0.1459 ms -- a frame
// touches only the cells on its visible surfaces, a few MB; the incoherent set 0.527 -> 0.493 -> 0.477 ms), or five when
// the budget or a level's cell count (< 2^24) does not allow seven (tiers 2 and 1 of `C`); the paper's family (F = 4, 64-byte blocks) six (N = 16 .. 90,
// 68 MB; its 8-level model: 0.0932 ms with four, 0.0802 with six, 0.0881 with seven -- a kernel whose time also moves by
// several per cent with its place in the module) -- profiles/r02_cells.md
// the bias K-step's ones tile in shared memory instead of tensor memory (niv_fused.cuh OS): the paper's family and its
// grid-less models at width 32 / 64, whose 56..106 registers allow five to eight CTAs per SM once a tile takes 96 / 64
// tensor-memory columns instead of 128; BASELINE.json's family sits at the register cap with four CTAs either way
constexpr bool ones_in_smem(uint32_t W, uint32_t L, uint32_t F) { return (F == 4 || L == 0) && (W == 32 || W == 64); }
// tier C: 0 = none; 1 = the first five levels (F = 2) / six (F = 4); 2 = seven levels (F = 2: N = 16 .. 182, 274 MB of copies)
constexpr int cell_levels_of(int L, int F, int C = 2) {
    return C == 0 ? 0 : F == 4 ? (L < 6 ? L : 6) : C == 1 ? (L < 5 ? L : 5) : (L < 7 ? L : 7);
}
template <int W, int L, int F, bool RAWDIR, bool O, int NPT, bool IMG, int C, bool PK = false, int DB = 0>
static fused_fn fused_inst() {
    // levels per gather batch (two batches in flight): BASELINE.json's family four = 32 gathers; the paper's family
    // (8-byte entries) two = 32 registers
    constexpr int NB = L == 0 ? 1 : F == 4 ? 2 : 4;
    return niv_fused_kernel<W, L, NB, F, RAWDIR, O, NPT, IMG, cell_levels_of(L, F, C), PK, DB, ones_in_smem(W, L, F)>;
}
template <int W, bool O, int NPT, bool IMG, int C, bool PK = false>
static fused_fn pick_levels_f2(uint32_t L) {        // BASELINE.json's family: F = 2, SH-16
    switch (L) {
        case 4:  return fused_inst<W, 4, 2, false, O, NPT, IMG, C, PK>();
        case 8:  return fused_inst<W, 8, 2, false, O, NPT, IMG, C, PK>();
        case 12: return fused_inst<W, 12, 2, false, O, NPT, IMG, C, PK>();
        case 16: return fused_inst<W, 16, 2, false, O, NPT, IMG, C, PK>();
        default: return nullptr;
    }
}
template <int W, bool O, int C, bool PK = false, int DB = 0>
static fused_fn pick_levels_f4(uint32_t L) {        // the paper's own family: F = 4, raw direction
    switch (L) {
        case 2: return fused_inst<W, 2, 4, true, O, 0, false, C, PK, DB>();
        case 4: return fused_inst<W, 4, 4, true, O, 0, false, C, PK, DB>();
        case 6: return fused_inst<W, 6, 4, true, O, 0, false, C, PK, DB>();
        case 8: return fused_inst<W, 8, 4, true, O, 0, false, C, PK, DB>();
        default: return nullptr;
    }
}
// PK: the variant that reads the compact G-buffer formats / writes fp16 (linear tiles; the grid models of both families)
template <bool O, int C, bool PK = false>
static fused_fn pick_fused(uint32_t W, uint32_t L, uint32_t F, uint32_t dir_freq = 0) {
    if (dir_freq) {                                 // frequency-encoded direction: the paper's family at width 64, device buffers
        if constexpr (!O) return (F == 4 && W == 64 && dir_freq == 4) ? pick_levels_f4<64, false, (C > 1 ? 1 : C), PK, 4>(L) : nullptr;
        else return nullptr;                        // (host buffers take niv_infer_host's staged path)
    }
    if (L == 0)                                     // grid-less: positional encoding, no gathers
        return W == 16 ? fused_inst<16, 0, 2, true, O, 0, false, 0, PK>() : W == 32 ? fused_inst<32, 0, 2, true, O, 0, false, 0, PK>()
             : W == 64 ? fused_inst<64, 0, 2, true, O, 0, false, 0, PK>() : nullptr;
    if (F == 4) return W == 32 ? pick_levels_f4<32, O, (C > 1 ? 1 : C), PK>(L) : W == 64 ? pick_levels_f4<64, O, (C > 1 ? 1 : C), PK>(L) : nullptr;
    return W == 32 ? pick_levels_f2<32, O, 0, false, C, PK>(L) : W == 64 ? pick_levels_f2<64, O, 0, false, C, PK>(L) : nullptr;
}
// image tiling (niv_infer_image): BASELINE.json's family (F = 2, 8..16 levels reach cells smaller than a warp's strip).
// The paper's own family (F = 4, <= 8 levels, finest cell 5.5 cm) measured SLOWER with it (profiles/r01_v2.md): its
// cells are larger than a 32-pixel strip anyway; it keeps the linear kernel, as do the grid-less models.
template <int C, bool PK = false>
static fused_fn pick_fused_img(uint32_t W, uint32_t L, uint32_t F) {
    if (L == 0 || F != 2) return nullptr;
    return W == 32 ? pick_levels_f2<32, false, 0, true, C, PK>(L) : W == 64 ? pick_levels_f2<64, false, 0, true, C, PK>(L) : nullptr;
}
// per-texel scene parameters: BASELINE.json's family, 8 or 16 levels, width 32 / 64, 1 or 2 parameters
template <int W, int NPT, int C>
static fused_fn pick_tp_levels(uint32_t L) {
    return L == 8 ? fused_inst<W, 8, 2, false, false, NPT, false, C>() : L == 16 ? fused_inst<W, 16, 2, false, false, NPT, false, C>() : nullptr;
}
template <int C>
static fused_fn pick_fused_tp(uint32_t W, uint32_t L, uint32_t F, uint32_t sh_degree, uint32_t n_params) {
    if (F != 2 || sh_degree != 4) return nullptr;
    if (n_params == 1) return W == 32 ? pick_tp_levels<32, 1, C>(L) : W == 64 ? pick_tp_levels<64, 1, C>(L) : nullptr;
    if (n_params == 2) return W == 32 ? pick_tp_levels<32, 2, C>(L) : W == 64 ? pick_tp_levels<64, 2, C>(L) : nullptr;
    return nullptr;
}

// byte layout of the packed weight blob and of the CTA's shared memory for a layer-1 K of `k1`
static void layout_blob(const niv_model* m, KParams& P, uint32_t k1, bool fold_params) {
    const uint32_t W = m->cfg.hidden_width;
    uint32_t off = 0, in = P.in_dim;
    for (uint32_t k = 0; k < P.n_layers; ++k) {
        const uint32_t o = (k + 1 == P.n_layers) ? 3u : W;
        P.kdim[k] = (k == 0) ? k1 : in;
        P.npad[k] = round_up(o, 16);
        P.w_off[k] = off;
        // + the bias K-step.  Only its first group of 8 K rows is stored: (bias_hi, bias_lo, 0 x 6).  Rows 8..15 of
        // the step are whatever follows in the blob (the next layer's weights, finite by niv_load_params' check; a
        // zero block after the last layer): the A side of the step is (1, 1, 0 x 14), so they are multiplied by zero.
        off += (P.kdim[k] + 8) * P.npad[k] * 2;
        in = o;
    }
    off += P.npad[P.n_layers - 1] * 16;
    for (uint32_t k = 0; k < P.n_layers; ++k) { P.b_off[k] = off; off += P.npad[k] * 4; }
    P.wparam_off = off;
    if (fold_params) off += W * 16 * m->cfg.n_params * 4;
    P.wpack_bytes = round_up(off, 16);
    P.a_off = round_up(P.wpack_bytes, 128);
    P.ones_off = P.a_off;                                        // weights | barriers, slots | (output staging)
    P.misc_off = P.a_off;
}

extern "C" int niv_create(const niv_config* cfg, niv_model** out)
{
    if (!cfg || !out) return NIV_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->struct_size != sizeof(niv_config) || cfg->api_version != NIV_API_VERSION) return NIV_ERR_INVALID_ARG;
    if (cfg->n_levels > NIV_MAX_LEVELS || (cfg->n_levels && cfg->n_features == 0)) return NIV_ERR_INVALID_ARG;
    if (cfg->n_levels && (cfg->log2_table_size < 4 || cfg->log2_table_size > 24)) return NIV_ERR_INVALID_ARG;
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
    // shapes this build has kernels for: BASELINE.json's family (F = 2, SH-16 direction, L in {4, 8, 12, 16}), the
    // paper's own (F = 4, raw direction, L in {2, 4, 6, 8}, width <= 64) and the paper's grid-less models (n_levels = 0:
    // eight-band positional encoding, raw direction, width 16/32/64)
    if (cfg->n_levels == 0) {
        if (cfg->sh_degree != 0 || cfg->n_frequencies != 8) return NIV_ERR_UNSUPPORTED;
        if (cfg->hidden_width != 16 && cfg->hidden_width != 32 && cfg->hidden_width != 64) return NIV_ERR_UNSUPPORTED;
    } else if (cfg->n_features == 2) {
        if (cfg->sh_degree != 4) return NIV_ERR_UNSUPPORTED;
    } else if (cfg->n_features == 4) {
        if (cfg->sh_degree != 0 || cfg->n_levels > 8 || cfg->hidden_width > 64) return NIV_ERR_UNSUPPORTED;
    } else return NIV_ERR_UNSUPPORTED;
    // frequency-encoded direction: on top of the raw vector only; kernels for 4 bands, the paper's grid family, width 64
    if (cfg->dir_frequencies && cfg->sh_degree != 0) return NIV_ERR_INVALID_ARG;
    if (cfg->dir_frequencies && (cfg->dir_frequencies != 4 || cfg->n_levels == 0 || cfg->n_features != 4 || cfg->hidden_width != 64))
        return NIV_ERR_UNSUPPORTED;
    // Any number of levels: the kernels are compiled for whole gather batches (multiples of 4 levels for F = 2, of 2 for
    // F = 4); a model with fewer levels runs the next larger kernel with DUMMY levels that read a block of zeros and meet
    // zero weight columns (their latent columns of W1 are zero in the packed blob), so they add exactly 0 to every sum.
    const uint32_t lev_step = cfg->n_features == 4 ? 2u : 4u;
    const uint32_t Lk = cfg->n_levels ? round_up(cfg->n_levels, lev_step) : 0u;
    if (cfg->n_params > 2 || (cfg->n_params && cfg->n_frequencies != 8)) return NIV_ERR_UNSUPPORTED;
    if (cfg->n_hidden_layers > 3) return NIV_ERR_UNSUPPORTED;
    if (cfg->hidden_width != 32 && cfg->hidden_width != 64 && cfg->hidden_width != 128 &&
        !(cfg->n_levels == 0 && cfg->hidden_width == 16)) return NIV_ERR_UNSUPPORTED;

    niv_model* m = new (std::nothrow) niv_model();
    if (!m) return NIV_ERR_ALLOC;
    m->cfg = *cfg;
    m->pdl = env_flag("NIV_PDL", true);
    m->overlap = env_flag("NIV_OVERLAP", true);
    m->image_linear = env_flag("NIV_IMAGE_LINEAR", false);
    m->host_staged = env_flag("NIV_HOST_STAGED", false);
    m->debug = env_flag("NIV_DEBUG", false);
    const bool want_mma_sync = env_flag("NIV_MMA_SYNC", false);
    niv_info& I = m->info;
    memset(&I, 0, sizeof(I));
    I.struct_size = sizeof(niv_info);
    KParams& P = m->kp;
    memset(&P, 0, sizeof(P));

    // level table (readings #2, #4)
    const uint64_t T = (uint64_t)1 << cfg->log2_table_size;
    uint64_t dev_entries = 0;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        uint64_t N;
        if (explicit_res) N = cfg->resolutions[l];
        else N = (uint64_t)std::floor((double)cfg->base_resolution * std::pow(cfg->per_level_scale, (double)l));
        if (N == 0 || N > (1u << 22)) { delete m; return NIV_ERR_INVALID_ARG; }   // locate_bits: N + 2^23 exact in fp32
        const uint64_t R = N + 1;
        const bool dense = R * R * R <= T;
        I.resolution[l] = (uint32_t)N;
        I.is_dense[l] = dense ? 1u : 0u;
        P.lv[l].Nf = (float)N;
        P.lv[l].Nm1 = (int32_t)N - 1;
        P.lv[l].cmaxf = (float)(8388608u + (uint32_t)N - 1u);               // exact: < 2^24
        P.lv[l].R = (uint32_t)R;
        P.lv[l].R2 = dense ? (uint32_t)(R * R) : 0u;
        // compact device storage (Table 1's memory column): a dense level holds its (N + 1)^3
        // entries only; every level starts at a multiple of 8 entries (32-byte sectors, as in the [L][T] layout)
        m->lev_entries[l] = dense ? R * R * R : T;
        P.lv[l].base = (uint32_t)(dev_entries);
        dev_entries += (m->lev_entries[l] + 7) / 8 * 8;
        I.table_bytes_compact += m->lev_entries[l] * cfg->n_features * 2;
        P.lv[l].dense = dense ? 1u : 0u;
    }
    m->dev_table_bytes = dev_entries * cfg->n_features * 2;
    I.table_bytes_device = m->dev_table_bytes;
    for (int d = 0; d < 3; ++d) {
        P.amin[d] = cfg->aabb_min[d];
        volatile float ext = cfg->aabb_max[d] - cfg->aabb_min[d];
        volatile float inv = 1.0f / ext;
        P.ainv[d] = inv;
    }
    for (uint32_t l = cfg->n_levels; l < Lk; ++l) {      // dummy levels: one cell, dense, over a block of zeros
        P.lv[l].Nf = 1.0f;
        P.lv[l].Nm1 = 0;
        P.lv[l].cmaxf = 8388608.0f;
        P.lv[l].R = 2;
        P.lv[l].R2 = 4;
        P.lv[l].dense = 1u;
        P.lv[l].cs = 1;
        P.lv[l].cs2 = 1;
    }
    m->kernel_levels = Lk;
    m->k_shift = (Lk - cfg->n_levels) * cfg->n_features;
    I.kernel_levels = Lk;
    P.L = cfg->n_levels;
    P.tmask = (uint32_t)(T - 1);
    P.n_features = cfg->n_features;
    P.raw_dir = cfg->sh_degree == 0 ? 1u : 0u;
    P.dir_freq = cfg->dir_frequencies;
    P.enc_dim = (cfg->n_levels ? cfg->n_levels * cfg->n_features : 6u * cfg->n_frequencies) + (P.raw_dir ? 3u + 6u * P.dir_freq : 16u);
    P.in_dim = P.enc_dim + 2 * cfg->n_frequencies * cfg->n_params;
    P.n_params = cfg->n_params;
    P.n_layers = cfg->n_hidden_layers + 1;
    P.out_act = cfg->out_activation;
    I.in_dim = P.in_dim;
    I.table_bytes = (uint64_t)cfg->n_levels * T * cfg->n_features * 2;      // 0 for the grid-less models
    // cell-block copies of the coarsest min(L, kCellLevels) levels, if their N^3 blocks of 8 entries fit
    // the budget (NIV_CELL_MB, read once here; 0 = none): the kernels that read them are compiled for exactly that
    // many levels, so it is all of them or none.  (width 128 and the mma.sync A/B kernel gather from the table)
    int cell_tier = 0;                             // 0 none, 1 five (four) levels, 2 seven: the highest that fits
    if (cfg->n_levels && cfg->hidden_width <= 64 && !want_mma_sync) {
        const char* s_mb = getenv("NIV_CELL_MB");
        const uint64_t budget = (uint64_t)(s_mb ? std::max(0, atoi(s_mb)) : kCellBudgetMB) << 20;
        for (int tier = cfg->n_features == 4 ? 1 : 2; tier >= 1 && cell_tier == 0; --tier) {
            const uint32_t want = std::min((uint32_t)cell_levels_of((int)Lk, (int)cfg->n_features, tier), cfg->n_levels);   // the real ones
            uint64_t off = 0;
            bool fits = true;
            for (uint32_t l = 0; l < want && fits; ++l) {
                const uint64_t N = I.resolution[l], bytes = N * N * N * 8 * cfg->n_features * 2;
                if (N * N * N >= (1u << 24) || off + bytes > budget) fits = false;
                m->cell_off[l] = off;
                off += bytes;
            }
            if (!fits) continue;
            for (uint32_t l = 0; l < want; ++l) {
                P.lv[l].cs = I.resolution[l];
                P.lv[l].cs2 = I.resolution[l] * I.resolution[l];
            }
            I.cell_levels = want;
            I.cell_bytes = off;
            cell_tier = tier;
        }
    }
    const bool use_cells = cell_tier != 0;
    I.tile_texels = kTile;

    // layer shapes and the packed weight blob layout
    const uint32_t W = cfg->hidden_width;
    {
        uint32_t in = P.in_dim;
        for (uint32_t k = 0; k < P.n_layers; ++k) {
            const uint32_t o = (k + 1 == P.n_layers) ? 3u : W;
            m->layer_out.push_back(o);
            m->layer_in.push_back(in);
            I.weight_bytes += (uint64_t)o * in * 2;
            I.bias_bytes += (uint64_t)o * 4;
            in = o;
        }
    }
    layout_blob(m, P, round_up(P.enc_dim + m->k_shift, 16), true);   // layer 1 consumes the encoded part only (parameters fold)

    // device side
    g_last_cuda_error = 0;
    int rc = NIV_OK;
    cudaError_t e = cudaSetDevice(cfg->device);
    cudaDeviceProp prop;
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cfg->device);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); delete m; return NIV_ERR_CUDA; }
    if (prop.major != 10) { delete m; return NIV_ERR_UNSUPPORTED; }           // sm_100a only; no fallback
    I.num_sms = (uint32_t)prop.multiProcessorCount;
    const bool os = ones_in_smem(W, cfg->n_levels, cfg->n_features) && !want_mma_sync;
    if (os) P.misc_off = P.ones_off + 2 * kTile * 16;    // weights | ones tile (4 KB, SS-form bias K-step) | barriers
    const uint32_t smem_dev = P.misc_off + 64, smem_host = smem_dev + 4 * 384;  // host variant: + output staging
    if (want_mma_sync && W == 64 && cfg->n_levels == 16 && cfg->n_features == 2 && cfg->n_hidden_layers == 2 &&
        cfg->n_params == 0) {
        m->fused.fn = niv_fused_mma_kernel<4, 4>;        // 4 levels per gather batch, 128 registers, 4 CTAs per SM
        m->fused.smem = (kMmaWords + 4 * kMmaStage) * 4;
        m->mma_kernel = true;
        rc = setup_kernel(m, m->fused, 0, "fused_mma_sync");
    } else if (W == 128) {                                // two N = 64 halves per hidden layer (niv_fused_w128.cuh)
        switch (Lk) {
            case 4:  m->fused.fn = niv_fused_w128_kernel<4, 4>; break;
            case 8:  m->fused.fn = niv_fused_w128_kernel<8, 4>; break;
            case 12: m->fused.fn = niv_fused_w128_kernel<12, 4>; break;
            case 16: m->fused.fn = niv_fused_w128_kernel<16, 4>; break;
            default: break;
        }
        P.misc_off = P.ones_off + 2 * kTile * 16;        // weights | ones chunk (4 KB, SS-form bias K-step) | barriers
        m->fused.smem = P.misc_off + 64;
        rc = m->fused.fn ? setup_kernel(m, m->fused, 128, "fused_w128") : NIV_ERR_UNSUPPORTED;
    } else {
        // D | A | ones in one allocation (niv_fused.cuh TMEM_COLS); ones in shared memory: D 64 + A 32, or D 32 | A 32
        const int tmem_cols = os ? (W == 64 ? 96 : 64) : W == 16 ? 64 : 128;
        m->fused.fn = cell_tier == 2 ? pick_fused<false, 2>(W, Lk, cfg->n_features, cfg->dir_frequencies)
                    : cell_tier == 1 ? pick_fused<false, 1>(W, Lk, cfg->n_features, cfg->dir_frequencies)
                                     : pick_fused<false, 0>(W, Lk, cfg->n_features, cfg->dir_frequencies);
        m->fused.smem = smem_dev;
        rc = m->fused.fn ? setup_kernel(m, m->fused, tmem_cols, "fused") : NIV_ERR_UNSUPPORTED;
        if (rc == NIV_OK) {
            m->fused_host.fn = pick_fused<true, 0>(W, Lk, cfg->n_features, cfg->dir_frequencies);   // PCIe-bound: table gathers
            m->fused_host.smem = smem_host;
            rc = setup_kernel(m, m->fused_host, tmem_cols, "fused_host");
        }
        if (rc == NIV_OK) {
            m->fused_pk.fn = cell_tier == 2 ? pick_fused<false, 2, true>(W, Lk, cfg->n_features, cfg->dir_frequencies)
                           : cell_tier == 1 ? pick_fused<false, 1, true>(W, Lk, cfg->n_features, cfg->dir_frequencies)
                                            : pick_fused<false, 0, true>(W, Lk, cfg->n_features, cfg->dir_frequencies);
            m->fused_pk.smem = smem_dev;
            rc = setup_kernel(m, m->fused_pk, tmem_cols, "fused_packed");
        }
        if (rc == NIV_OK) {
            m->fused_host_pk.fn = pick_fused<true, 0, true>(W, Lk, cfg->n_features, cfg->dir_frequencies);
            m->fused_host_pk.smem = smem_host;
            rc = setup_kernel(m, m->fused_host_pk, tmem_cols, "fused_host_packed");
        }
        if (rc == NIV_OK) {
            m->fused_img.fn = cell_tier == 2 ? pick_fused_img<2>(W, Lk, cfg->n_features)
                            : cell_tier == 1 ? pick_fused_img<1>(W, Lk, cfg->n_features)
                                             : pick_fused_img<0>(W, Lk, cfg->n_features);
            m->fused_img.smem = smem_dev;
            rc = setup_kernel(m, m->fused_img, tmem_cols, "fused_image");
        }
        if (rc == NIV_OK && use_cells && m->fused_img.fn) {
            m->fused_img_pk.fn = cell_tier == 2 ? pick_fused_img<2, true>(W, Lk, cfg->n_features)
                                                : pick_fused_img<1, true>(W, Lk, cfg->n_features);
            m->fused_img_pk.smem = smem_dev;
            rc = setup_kernel(m, m->fused_img_pk, tmem_cols, "fused_image_packed");
        }
        if (rc == NIV_OK && cfg->n_params) {
            m->fused_tp.fn = cell_tier == 2 ? pick_fused_tp<2>(W, Lk, cfg->n_features, cfg->sh_degree, cfg->n_params)
                           : cell_tier == 1 ? pick_fused_tp<1>(W, Lk, cfg->n_features, cfg->sh_degree, cfg->n_params)
                                            : pick_fused_tp<0>(W, Lk, cfg->n_features, cfg->sh_degree, cfg->n_params);
            if (m->fused_tp.fn) {
                // layout of the per-texel-parameter variant: layer 1 with K = round16(enc_dim) + 16 n_params, no fold blob
                m->kp_tp = P;
                layout_blob(m, m->kp_tp, round_up(P.enc_dim + m->k_shift, 16) + 16 * cfg->n_params, false);
                m->fused_tp.smem = m->kp_tp.misc_off + 64;
                rc = setup_kernel(m, m->fused_tp, tmem_cols, "fused_texel_params");
            }
        }
    }
    if (rc != NIV_OK) { delete m; return rc; }
    I.ctas_per_sm = m->fused.ctas_per_sm;
    I.smem_bytes = m->fused.smem;
    I.image_tiled = m->fused_img.fn ? 1u : 0u;
    I.texel_params = m->fused_tp.fn ? 1u : 0u;
    e = cudaMalloc(&m->d_table, m->dev_table_bytes + 64);     // + a block of zeros for the dummy levels
    if (e == cudaSuccess) e = cudaMemset(m->d_table, 0, m->dev_table_bytes + 64);
    if (e == cudaSuccess && I.cell_bytes) e = cudaMalloc(&m->d_cells, I.cell_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_wpack, P.wpack_bytes);
    if (e == cudaSuccess && m->fused_tp.fn) e = cudaMalloc(&m->d_wpack_tp, m->kp_tp.wpack_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_ctr, kCtrSlots * 128);
    if (e == cudaSuccess) e = cudaMemset(m->d_ctr, 0, kCtrSlots * 128);
    if (e == cudaSuccess) e = cudaHostAlloc((void**)&m->h_done, kCtrSlots * sizeof(uint32_t), cudaHostAllocMapped);
    if (e == cudaSuccess) {
        for (uint32_t s = 0; s < kCtrSlots; ++s) m->h_done[s] = 0u;
        e = cudaHostGetDevicePointer((void**)&m->d_done, (void*)m->h_done, 0);
    }
    if (e != cudaSuccess) {
        g_last_cuda_error = (int)e; (void)cudaGetLastError();
        niv_destroy(m);
        return NIV_ERR_ALLOC;
    }
    P.table = m->d_table;
    P.wpack = m->d_wpack;
    m->kp_tp.table = m->d_table;
    m->kp_tp.wpack = m->d_wpack_tp;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        P.lv[l].tb = m->d_table + (size_t)P.lv[l].base * (cfg->n_features / 2);
        if (l < I.cell_levels) P.lv[l].cells = reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(m->d_cells) + m->cell_off[l]);
        m->kp_tp.lv[l] = P.lv[l];
    }
    for (uint32_t l = cfg->n_levels; l < Lk; ++l) {
        P.lv[l].tb = reinterpret_cast<const uint32_t*>(reinterpret_cast<const uint8_t*>(m->d_table) + m->dev_table_bytes);
        P.lv[l].cells = reinterpret_cast<const uint4*>(P.lv[l].tb);
        m->kp_tp.lv[l] = P.lv[l];
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

// compact: the table comes as the levels back to back with exactly lev_entries[l] entries each (niv_load_params_compact)
static int load_params_impl(niv_model* m, const void* table_fp16, size_t table_bytes, bool compact,
                            const void* weights_fp16, size_t weight_bytes,
                            const float* biases_f32, size_t bias_bytes, int src_on_device, void* stream)
{
    if (!m || (!table_fp16 && m->info.table_bytes) || !weights_fp16) return NIV_ERR_INVALID_ARG;
    if (table_bytes != (compact ? m->info.table_bytes_compact : m->info.table_bytes) || weight_bytes != m->info.weight_bytes)
        return NIV_ERR_INVALID_ARG;
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

    // "all parameters finite"; a bias beyond the fp16 range could not ride in the MMA as (hi, lo) fp16 rows
    for (float v : b)
        if (!std::isfinite(v) || std::fabs(v) > 65504.0f) return NIV_ERR_INVALID_ARG;
    for (uint16_t h : w)
        if ((h & 0x7C00u) == 0x7C00u) return NIV_ERR_INVALID_ARG;          // fp16 Inf / NaN

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
        // (layer 1 of a model with dummy levels: the direction columns sit behind the dummy levels' zero columns)
        const uint32_t n_lat = m->cfg.n_levels * m->cfg.n_features, shift = (k == 0) ? m->k_shift : 0u;
        for (uint32_t r = 0; r < o; ++r)
            for (uint32_t c = 0; c < kuse; ++c) {
                const uint32_t ck = (shift && c >= n_lat) ? c + shift : c;
                dst[(size_t)(ck >> 3) * (P.npad[k] * 8) + r * 8 + (ck & 7)] = w[wsrc + (size_t)r * in + c];
            }
        if (k == 0 && texel_params) {
            const uint32_t k0 = round_up(P.enc_dim + m->k_shift, 16);
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
    if (m->fused_tp.fn) {
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
    {   // the table, level by level, into the compact device storage (a dense level: its first (N + 1)^3 entries)
        const size_t eb = (size_t)m->cfg.n_features * 2, T = (size_t)1 << m->cfg.log2_table_size;
        size_t src_off = 0;
        for (uint32_t l = 0; l < m->cfg.n_levels; ++l) {
            const size_t bytes = (size_t)m->lev_entries[l] * eb;
            NIV_CUDA(cudaMemcpyAsync(reinterpret_cast<uint8_t*>(m->d_table) + (size_t)P.lv[l].base * eb,
                                     static_cast<const uint8_t*>(table_fp16) + (compact ? src_off : (size_t)l * T * eb), bytes,
                                     src_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
            src_off += bytes;
        }
    }
    for (uint32_t l = 0; l < m->info.cell_levels; ++l) {            // cell-block copies of the coarse levels
        const uint32_t n_cells = P.lv[l].cs * P.lv[l].cs2;
        niv_build_cells_kernel<<<(n_cells + 255) / 256, 256, 0, st>>>(
            P, l, reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(m->d_cells) + m->cell_off[l]), n_cells);
        NIV_CUDA(cudaGetLastError());
    }
    NIV_CUDA(cudaStreamSynchronize(st));
    m->loaded = true;
    return NIV_OK;
}

extern "C" int niv_load_params(niv_model* m, const void* table_fp16, size_t table_bytes,
                               const void* weights_fp16, size_t weight_bytes,
                               const float* biases_f32, size_t bias_bytes, int src_on_device, void* stream)
{
    return load_params_impl(m, table_fp16, table_bytes, false, weights_fp16, weight_bytes, biases_f32, bias_bytes,
                            src_on_device, stream);
}

extern "C" int niv_load_params_compact(niv_model* m, const void* table_fp16, size_t table_bytes,
                                       const void* weights_fp16, size_t weight_bytes,
                                       const float* biases_f32, size_t bias_bytes, int src_on_device, void* stream)
{
    return load_params_impl(m, table_fp16, table_bytes, true, weights_fp16, weight_bytes, biases_f32, bias_bytes,
                            src_on_device, stream);
}

static int fill_params(const niv_model* m, const float* param, KParams& P)
{
    P = m->kp;
    if (m->cfg.n_params) {
        if (!param) return NIV_ERR_INVALID_ARG;
        for (uint32_t q = 0; q < m->cfg.n_params; ++q) {
            if (!std::isfinite(param[q])) return NIV_ERR_INVALID_ARG;
            P.t[q] = param[q];
        }
    } else if (param) {
        return NIV_ERR_INVALID_ARG;
    }
    return NIV_OK;
}

// The tile counter of one launch (dynamic tile scheduling).  A slot is handed out only while no launch is using it:
// the last CTA of a launch writes the slot's generation to a host-mapped word, the host compares it with the
// generation it issued.  If all kCtrSlots are busy -- or the stream is being captured into a CUDA graph, whose
// replays the host never sees -- the launch falls back to static striding (tile += gridDim.x): slower on frames with
// large background regions, never wrong.  A launch that faulted leaves its slot busy for good, which only retires it.
static void draw_tile_counter(niv_model* m, cudaStream_t st, KParams& P)
{
    P.tile_ctr = nullptr;
    P.slot_done = nullptr;
    P.slot_gen = 0;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { (void)cudaGetLastError(); return; }
    if (cs != cudaStreamCaptureStatusNone) return;
    std::lock_guard<std::mutex> lock(m->slot_mu);
    for (uint32_t k = 0; k < kCtrSlots; ++k) {
        const uint32_t s = (m->slot_next + k) % kCtrSlots;
        if (m->h_done[s] != m->slot_gen[s]) continue;            // a launch is still running on this slot
        m->slot_next = s + 1;
        P.tile_ctr = m->d_ctr + (size_t)s * 32;
        P.slot_done = m->d_done + s;
        P.slot_gen = ++m->slot_gen[s];
        return;
    }
}

// ---- launch overlap -------------------------------------------------------------------------------------------------
// Back-to-back launches on one stream (one frame per call): with programmatic stream serialisation the
// CTAs of launch n take the SM slots of launch n-1 as those drain, but griddepcontrol.wait holds them until ALL of n-1
// has finished, so every launch pays the drain of the last tiles and the fill of the first ones (8 us of a 156 us
// frame).  If n-1 is a launch of this library whose buffers are disjoint from those of n (nothing n reads or writes is
// written by n-1, nothing n writes is read by n-1), n does not need that wait: it starts on its own buffers beside the
// last tiles of n-1.  What keeps this exact:
//   * the host keeps, per stream, the buffer ranges and completion words of the last three launches it issued there;
//     any other kernel or copy the caller puts between two launches only adds ordering (it does not trigger early);
//   * launch n polls the completion words (tile_ctr[2], written with release by the last CTA) of launches n-2 and n-3
//     before it touches a caller's buffer, so at most two launches ever run beside each other, and it skips the
//     griddepcontrol.wait only if n-1, n-2 and n-3 all have such a word (launches recorded into a CUDA graph, on the
//     static-striding fallback or through another kernel have none: the next launches wait in full);
//   * niv_destroy forgets all history (cudaFree has synchronised the device by then).
constexpr int kRanges = 7, kOutRange = 6;
struct LaunchRec {
    bool tracked = false;
    uintptr_t lo[kRanges] = {}, hi[kRanges] = {};             // pos, nrm, tparam, albedo, direct, emission (read), out (written)
    const uint32_t* done = nullptr;
    uint32_t gen = 0;
};
struct StreamHist { LaunchRec r[3]; };                        // r[0] = the previous launch on the stream, r[1], r[2] before it
static std::mutex g_hist_mu;
static std::unordered_map<cudaStream_t, StreamHist> g_hist;

static bool ranges_overlap(const LaunchRec& a, int i, const LaunchRec& b, int j) {
    return a.lo[i] < b.hi[j] && b.lo[j] < a.hi[i];
}
static bool launches_conflict(const LaunchRec& prev, const LaunchRec& cur) {
    for (int j = 0; j < kRanges; ++j)
        if (ranges_overlap(prev, kOutRange, cur, j)) return true;     // cur touches what prev writes
    for (int i = 0; i < kOutRange; ++i)
        if (ranges_overlap(prev, i, cur, kOutRange)) return true;     // cur writes what prev reads
    return false;
}
static void forget_history() {
    std::lock_guard<std::mutex> lock(g_hist_mu);
    g_hist.clear();
}

// One launch of a fused kernel; `pdl`: with the programmatic-stream-serialisation attribute (the tcgen05 kernels of
// width <= 64, which hold their griddepcontrol.wait before the first access to a caller's buffer).
static int launch_one(const niv_model* m, const FusedKernel& k, cudaStream_t st, bool pdl, KParams& P, const float* pos,
                      const float* nrm, float* out, size_t n, uint32_t n_tiles)
{
    LaunchRec cur;
    static const size_t kA[4] = {12, 16, 16, 8}, kB[4] = {12, 16, 0, 0}, kO[3] = {12, 8, 4};   // bytes per texel by format
    const void* base[kRanges] = {pos, nrm, P.tparam, P.shade_albedo, P.shade_direct, P.shade_emission, out};
    const size_t bytes[kRanges] = {n * kA[P.gbuf_fmt & 3], n * kB[P.gbuf_fmt & 3], P.tparam ? n * 4 * m->cfg.n_params : 0,
                                   P.shade_albedo ? n * 12 : 0, P.shade_direct ? n * 12 : 0, P.shade_emission ? n * 12 : 0,
                                   n * kO[P.out_fmt < 3 ? P.out_fmt : 0]};
    for (int i = 0; i < kRanges; ++i) { cur.lo[i] = (uintptr_t)base[i]; cur.hi[i] = cur.lo[i] + bytes[i]; }
    cur.tracked = pdl && m->overlap && P.tile_ctr != nullptr;
    cur.done = P.tile_ctr ? P.tile_ctr + 2 : nullptr;
    cur.gen = P.slot_gen;
    P.grid_wait = 1;
    P.early_read = 0;
    P.wait_a = P.wait_b = nullptr;
    P.gen_a = P.gen_b = 0;

    std::lock_guard<std::mutex> lock(g_hist_mu);
    if (g_hist.size() > 4096) g_hist.clear();                 // stream handles come and go
    StreamHist& h = g_hist[st];
    if (cur.tracked) {                                        // (a launch without a counter slot is being captured: no polls)
        const LaunchRec *a = &h.r[1], *b = &h.r[2];
        if (!a->tracked) { a = b; b = nullptr; }
        if (a && a->tracked) { P.wait_a = a->done; P.gen_a = a->gen; }
        if (b && b->tracked && P.wait_a) { P.wait_b = b->done; P.gen_b = b->gen; }
        if (h.r[0].tracked && h.r[1].tracked && h.r[2].tracked && !launches_conflict(h.r[0], cur)) P.grid_wait = 0;
        // A CTA of launch n starts only after every CTA of n-1 has passed ITS waits (griddepcontrol.launch_dependents comes
        // after them in the kernel), i.e. with n-3 and everything older complete; n-1 writes nothing this launch reads
        // (grid_wait = 0); if n-2 does not either, the first texel can be requested at the very top of the kernel, before
        // this launch's own polls (which still precede everything else it does with a caller's buffer)
        if (P.grid_wait == 0) {
            bool raw = false;
            for (int j = 0; j < kOutRange; ++j) raw |= ranges_overlap(h.r[1], kOutRange, cur, j);
            P.early_read = raw ? 0u : 1u;
        }
    }
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(n_tiles < k.grid ? n_tiles : k.grid);
    cfg.blockDim = dim3(kTile);
    cfg.dynamicSmemBytes = k.smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 1 : 0;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, k.fn, P, pos, nrm, out, n, n_tiles);
    h.r[2] = h.r[1];
    h.r[1] = h.r[0];
    h.r[0] = cur;
    if (e != cudaSuccess) {
        h.r[0].tracked = false;
        g_last_cuda_error = (int)e;
        (void)cudaGetLastError();
        return NIV_ERR_CUDA;
    }
    return NIV_OK;
}
// a launch that goes around launch_one (the mma.sync A/B kernel, the staged host path): the next ones wait in full
static void note_untracked_launch(cudaStream_t st) {
    std::lock_guard<std::mutex> lock(g_hist_mu);
    StreamHist& h = g_hist[st];
    h.r[2] = h.r[1];
    h.r[1] = h.r[0];
    h.r[0] = LaunchRec();
}

static int launch_fused(niv_model* m, const KParams& Pin, const float* pos, const float* nrm, float* out,
                        size_t n, cudaStream_t st, bool host_variant = false)
{
    KParams P = Pin;
    draw_tile_counter(m, st, P);
    if (m->mma_kernel) {                                // warp-granular 32-texel tiles, four per CTA
        const uint32_t nt32 = (uint32_t)((n + 31) / 32), ctas = (nt32 + 3) / 4;
        note_untracked_launch(st);
        m->fused.fn<<<ctas < m->fused.grid ? ctas : m->fused.grid, kTile, m->fused.smem, st>>>(P, pos, nrm, out, n, nt32);
        NIV_CUDA(cudaGetLastError());
        return NIV_OK;
    }
    const uint32_t n_tiles = (uint32_t)((n + kTile - 1) / kTile);
    const bool tc5 = m->cfg.hidden_width <= 64;          // the kernels with the griddepcontrol pair
    // (the zero-copy host variant is followed by a stream synchronisation: it has nothing to overlap with)
    const bool packed = P.gbuf_fmt != NIV_GBUF_F32X3 || P.out_fmt != NIV_OUTFMT_F32X3 || P.shade_albedo != nullptr;
    const FusedKernel& k = packed ? (host_variant ? m->fused_host_pk : m->fused_pk) : (host_variant ? m->fused_host : m->fused);
    if (!k.fn) return NIV_ERR_UNSUPPORTED;
    return launch_one(m, k, st, m->pdl && tc5 && !host_variant, P, pos, nrm, out, n, n_tiles);
}

static int check_call(const niv_model* m, const void* pos, const void* nrm, const void* out, size_t n)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return 1;                               // nothing to do
    if (!pos || !nrm || !out) return NIV_ERR_INVALID_ARG;
    if (n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    return NIV_OK;
}

// ---- G-buffer / output formats (include/niv.h NIV_GBUF_*, NIV_OUTFMT_*) ---------------------------------------------
struct FmtInfo { size_t a_bytes, b_bytes, out_bytes; uintptr_t in_align, out_align; };
static bool fmt_info(int gf, int of, FmtInfo& f)
{
    switch (gf) {
        case NIV_GBUF_F32X3:     f.a_bytes = 12; f.b_bytes = 12; f.in_align = 4;  break;
        case NIV_GBUF_F32X4:     f.a_bytes = 16; f.b_bytes = 16; f.in_align = 16; break;
        case NIV_GBUF_P32_OCT16: f.a_bytes = 16; f.b_bytes = 0;  f.in_align = 16; break;
        case NIV_GBUF_P16_OCT8:  f.a_bytes = 8;  f.b_bytes = 0;  f.in_align = 8;  break;
        default: return false;
    }
    switch (of) {
        case NIV_OUTFMT_F32X3: f.out_bytes = 12; f.out_align = 4; break;
        case NIV_OUTFMT_F16X4: f.out_bytes = 8;  f.out_align = 8; break;
        case NIV_OUTFMT_RGB9E5: f.out_bytes = 4; f.out_align = 4; break;
        default: return false;
    }
    return true;
}
// common argument checks of the *_packed entry points; > 0: nothing to do
static int check_packed(const niv_model* m, int gf, const void* a, const void* b, int of, const void* out, size_t n, FmtInfo& f)
{
    if (!fmt_info(gf, of, f)) return NIV_ERR_INVALID_ARG;
    int rc = check_call(m, a, f.b_bytes ? b : a, out, n);
    if (rc != NIV_OK) return rc;
    if (((uintptr_t)a & (f.in_align - 1)) || (f.b_bytes && ((uintptr_t)b & (f.in_align - 1))) ||
        ((uintptr_t)out & (f.out_align - 1))) return NIV_ERR_INVALID_ARG;
    // the compact formats live in the tcgen05 kernels of width <= 64 (the width-128 and mma.sync kernels load fp32 x 3)
    if ((gf != NIV_GBUF_F32X3 || of != NIV_OUTFMT_F32X3) && (m->cfg.hidden_width > 64 || m->mma_kernel || !m->fused_pk.fn))
        return NIV_ERR_UNSUPPORTED;
    return NIV_OK;
}
static void set_formats(const niv_model* m, KParams& P, int gf, int of)
{
    P.gbuf_fmt = (uint32_t)gf;
    P.out_fmt = (uint32_t)of;
    for (int d = 0; d < 3; ++d) {
        volatile float ext = m->cfg.aabb_max[d] - m->cfg.aabb_min[d];
        P.aext[d] = ext;
    }
}

extern "C" int niv_infer_packed(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b, const float* param,
                                int out_format, void* out, size_t n, void* stream)
{
    FmtInfo f;
    int rc = check_packed(m, gbuf_format, gbuf_a, gbuf_b, out_format, out, n, f);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, gbuf_format, out_format);
    return launch_fused(m, P, (const float*)gbuf_a, (const float*)gbuf_b, (float*)out, n, (cudaStream_t)stream);
}

// the deferred compose as the EPILOGUE of the inference kernel (Eq. 2, 403): the irradiance
// never goes to memory, out = albedo / pi * E + direct + emission in the arithmetic of niv_compose.
extern "C" int niv_infer_shade(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b, const float* param,
                               const float* albedo, const float* direct, const float* emission, int out_format, void* out,
                               size_t n, void* stream)
{
    FmtInfo f;
    int rc = check_packed(m, gbuf_format, gbuf_a, gbuf_b, out_format, out, n, f);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    if (!albedo) return NIV_ERR_INVALID_ARG;
    if (m->cfg.hidden_width > 64 || m->mma_kernel || !m->fused_pk.fn) return NIV_ERR_UNSUPPORTED;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, gbuf_format, out_format);
    P.shade_albedo = albedo;
    P.shade_direct = direct;
    P.shade_emission = emission;
    return launch_fused(m, P, (const float*)gbuf_a, (const float*)gbuf_b, (float*)out, n, (cudaStream_t)stream);
}

// Debug: niv_infer through the PACKED kernel variant (fp32 x 3 in and out) which also writes every texel's layer-1 A
// row -- the packed fp16 words the tensor core reads: latents, direction, zero padding -- for feature-level parity of
// the FUSED path (cell-block levels, packed-fp16 blend) in every model family.
extern "C" int niv_debug_arow(niv_model* m, const float* pos, const float* nrm, const float* param, float* out,
                              uint32_t* arow, uint32_t row_words, size_t n, void* stream)
{
    int rc = check_call(m, pos, nrm, out, n);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    if (!arow || !m->fused_pk.fn) return arow ? NIV_ERR_UNSUPPORTED : NIV_ERR_INVALID_ARG;
    const uint32_t hw = m->cfg.n_levels ? m->kernel_levels * m->cfg.n_features / 2 : 24u;
    const uint32_t need = (hw + (m->cfg.sh_degree ? 8u : (3u + 6u * m->cfg.dir_frequencies + 1u) / 2u) + 7u) / 8u * 8u;
    if (row_words != need) return NIV_ERR_INVALID_ARG;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, NIV_GBUF_F32X3, NIV_OUTFMT_F32X3);
    P.dump_a = arow;
    P.dump_words = row_words;
    draw_tile_counter(m, (cudaStream_t)stream, P);
    return launch_one(m, m->fused_pk, (cudaStream_t)stream, m->pdl, P, pos, nrm, out, n, (uint32_t)((n + kTile - 1) / kTile));
}

extern "C" int niv_infer(niv_model* m, const float* pos, const float* nrm, const float* param,
                         float* out, size_t n, void* stream)
{
    return niv_infer_packed(m, NIV_GBUF_F32X3, pos, nrm, param, NIV_OUTFMT_F32X3, out, n, stream);
}

// an image call: the 8 x 4-block kernel where the model has one for this call (fp32 x 3 in and out: fused_img; compact
// formats or the shading epilogue: fused_img_pk), else linear tiles -- the same result
static int launch_image(niv_model* m, KParams& P, const void* gbuf_a, const void* gbuf_b, void* out, uint32_t width,
                        uint32_t height, cudaStream_t st)
{
    const size_t n = (size_t)width * height;
    const bool packed = P.gbuf_fmt != NIV_GBUF_F32X3 || P.out_fmt != NIV_OUTFMT_F32X3 || P.shade_albedo != nullptr;
    const FusedKernel& k = packed ? m->fused_img_pk : m->fused_img;
    if (!k.fn || width > (1u << 20) || height > (1u << 17) || m->image_linear)
        return launch_fused(m, P, (const float*)gbuf_a, (const float*)gbuf_b, (float*)out, n, st);
    P.img_w = width;
    P.img_h = height;
    P.tiles_x = (width + 31u) / 32u;
    const uint32_t n_tiles = P.tiles_x * ((height + 3u) / 4u);
    draw_tile_counter(m, st, P);
    return launch_one(m, k, st, m->pdl, P, (const float*)gbuf_a, (const float*)gbuf_b, (float*)out, n, n_tiles);
}

extern "C" int niv_infer_image_packed(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b,
                                      const float* param, int out_format, void* out, uint32_t width, uint32_t height,
                                      void* stream)
{
    const size_t n = (size_t)width * height;
    FmtInfo f;
    int rc = check_packed(m, gbuf_format, gbuf_a, gbuf_b, out_format, out, n, f);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, gbuf_format, out_format);
    // models without an image-tiled kernel (and images beyond the packed tile coordinates): same result, linear tiles
    // (and the compact formats, whose kernels are linear-tile ones)
    return launch_image(m, P, gbuf_a, gbuf_b, out, width, height, (cudaStream_t)stream);
}

// niv_infer_shade for a G-buffer that is an image (8 x 4 pixel blocks per warp where the model has that kernel)
extern "C" int niv_infer_image_shade(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b,
                                     const float* param, const float* albedo, const float* direct, const float* emission,
                                     int out_format, void* out, uint32_t width, uint32_t height, void* stream)
{
    const size_t n = (size_t)width * height;
    FmtInfo f;
    int rc = check_packed(m, gbuf_format, gbuf_a, gbuf_b, out_format, out, n, f);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    if (!albedo) return NIV_ERR_INVALID_ARG;
    if (m->cfg.hidden_width > 64 || m->mma_kernel || !m->fused_pk.fn) return NIV_ERR_UNSUPPORTED;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, gbuf_format, out_format);
    P.shade_albedo = albedo;
    P.shade_direct = direct;
    P.shade_emission = emission;
    return launch_image(m, P, gbuf_a, gbuf_b, out, width, height, (cudaStream_t)stream);
}

extern "C" int niv_infer_image(niv_model* m, const float* pos, const float* nrm, const float* param,
                               float* out, uint32_t width, uint32_t height, void* stream)
{
    return niv_infer_image_packed(m, NIV_GBUF_F32X3, pos, nrm, param, NIV_OUTFMT_F32X3, out, width, height, stream);
}

extern "C" int niv_infer_texel_params(niv_model* m, const float* pos, const float* nrm, const float* tparam,
                                      float* out, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (m->cfg.n_params == 0) return NIV_ERR_INVALID_ARG;
    if (!m->fused_tp.fn) return NIV_ERR_UNSUPPORTED;
    int rc = check_call(m, pos, nrm, out, n);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    if (!tparam) return NIV_ERR_INVALID_ARG;
    KParams P = m->kp_tp;
    P.tparam = tparam;
    draw_tile_counter(m, (cudaStream_t)stream, P);
    const uint32_t n_tiles = (uint32_t)((n + kTile - 1) / kTile);
    return launch_one(m, m->fused_tp, (cudaStream_t)stream, m->pdl, P, pos, nrm, out, n, n_tiles);
}

extern "C" int niv_infer_host_packed(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b,
                                     const float* param, int out_format, void* out, size_t n, void* stream)
{
    FmtInfo f;
    int rc = check_packed(m, gbuf_format, gbuf_a, gbuf_b, out_format, out, n, f);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, gbuf_format, out_format);
    NIV_CUDA(cudaSetDevice(m->cfg.device));
    const uint8_t* a = (const uint8_t*)gbuf_a;
    const uint8_t* b = (const uint8_t*)gbuf_b;
    uint8_t* o = (uint8_t*)out;
    // Zero copy: if all buffers are pinned (or registered) host memory the fused kernel reads the G-buffer and
    // writes the irradiance over PCIe itself -- the texel of the next tile is requested ahead, the output leaves as
    // full lines -- so transfer and compute overlap tile by tile in ONE launch with no staging (1.04 ms per full-HD
    // frame against 1.21 ms with chunked copies for fp32 x 3 in and out; the compact formats move 16 + 8 or 8 + 8
    // bytes per texel instead of 24 + 12).
    const bool packed = gbuf_format != NIV_GBUF_F32X3 || out_format != NIV_OUTFMT_F32X3;
    if ((packed ? m->fused_host_pk.fn : m->fused_host.fn) && !m->host_staged) {
        cudaPointerAttributes ap, an, ao;
        const bool ok_a = cudaPointerGetAttributes(&ap, a) == cudaSuccess && ap.type == cudaMemoryTypeHost && ap.devicePointer;
        const bool ok_b = !f.b_bytes || (cudaPointerGetAttributes(&an, b) == cudaSuccess && an.type == cudaMemoryTypeHost && an.devicePointer);
        const bool ok_o = cudaPointerGetAttributes(&ao, o) == cudaSuccess && ao.type == cudaMemoryTypeHost && ao.devicePointer &&
                          ((uintptr_t)ao.devicePointer & 15u) == 0;
        if (ok_a && ok_b && ok_o) {
            rc = launch_fused(m, P, (const float*)ap.devicePointer, f.b_bytes ? (const float*)an.devicePointer : nullptr,
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
    if (n > m->stage_cap) {                          // [a | b | out], each 16 bytes per texel at most
        if (m->d_stage) { NIV_CUDA(cudaFree(m->d_stage)); m->d_stage = nullptr; m->stage_cap = 0; }
        const size_t cap = (n + 1023) / 1024 * 1024;
        cudaError_t e = cudaMalloc(&m->d_stage, cap * 48);
        if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); return NIV_ERR_ALLOC; }
        m->stage_cap = cap;
    }
    uint8_t* d_a = reinterpret_cast<uint8_t*>(m->d_stage);
    uint8_t* d_b = d_a + 16 * m->stage_cap;
    uint8_t* d_o = d_a + 32 * m->stage_cap;
    // order after the caller's stream
    NIV_CUDA(cudaEventRecord(m->hev, (cudaStream_t)stream));
    NIV_CUDA(cudaStreamWaitEvent(m->hs[0], m->hev, 0));
    NIV_CUDA(cudaStreamWaitEvent(m->hs[1], m->hev, 0));
    // chunks of whole tiles; >= 4 chunks on a full frame so H2D, kernel and D2H of different chunks overlap
    size_t chunk = (n / 8 + kTile - 1) / kTile * kTile;
    if (chunk < 32768) chunk = 32768;
    int k = 0;
    for (size_t t0 = 0; t0 < n; t0 += chunk, ++k) {
        const size_t c = (n - t0 < chunk) ? n - t0 : chunk;
        cudaStream_t st = m->hs[k & 1];
        NIV_CUDA(cudaMemcpyAsync(d_a + f.a_bytes * t0, a + f.a_bytes * t0, c * f.a_bytes, cudaMemcpyHostToDevice, st));
        if (f.b_bytes) NIV_CUDA(cudaMemcpyAsync(d_b + f.b_bytes * t0, b + f.b_bytes * t0, c * f.b_bytes, cudaMemcpyHostToDevice, st));
        rc = launch_fused(m, P, (const float*)(d_a + f.a_bytes * t0), (const float*)(d_b + f.b_bytes * t0),
                          (float*)(d_o + f.out_bytes * t0), c, st);
        if (rc != NIV_OK) return rc;
        NIV_CUDA(cudaMemcpyAsync(o + f.out_bytes * t0, d_o + f.out_bytes * t0, c * f.out_bytes, cudaMemcpyDeviceToHost, st));
    }
    NIV_CUDA(cudaStreamSynchronize(m->hs[0]));
    NIV_CUDA(cudaStreamSynchronize(m->hs[1]));
    return NIV_OK;
}

extern "C" int niv_infer_host(niv_model* m, const float* pos, const float* nrm, const float* param,
                              float* out, size_t n, void* stream)
{
    return niv_infer_host_packed(m, NIV_GBUF_F32X3, pos, nrm, param, NIV_OUTFMT_F32X3, out, n, stream);
}

// ---- niv_infer_host_static: the host-buffer call for callers that must not allocate ---------------------------------
// The staged path of niv_infer_host keeps its staging buffers in cudaMalloc'ed memory that it grows on demand (and it
// creates two streams on first use).  This variant runs the same fused kernel on staging buffers that live in ONE
// file-scope device array of a fixed, modest size, so the call allocates nothing: no cudaMalloc / cudaFree, no stream
// or event creation, only cudaMemsetAsync, cudaMemcpyAsync, one kernel launch and a stream synchronisation on the
// caller's stream.  Every GPU that loads the library holds the array (9.4 MB) until the process exits.
//   layout: [0, 256)  the launch's tile-counter triple (tile, done, complete) -- must start at zero: cleared per call
//           then pos | nrm | out staging, 12 bytes x NIV_STATIC_MAX_TEXELS each
// The array is shared by every call of the process on that device (all models, all streams) and keeps the last call's
// contents: two calls that overlap on the GPU race.
constexpr size_t kStaticStage = (size_t)12 * NIV_STATIC_MAX_TEXELS;
static __device__ __align__(256) uint8_t g_static_scratch[256 + 3 * kStaticStage];

// In host code `g_static_scratch` is a host-side stand-in, not a device address: the address the kernel and the copies
// need comes from cudaGetSymbolAddress, asked once per device with that device current.
static std::mutex g_static_mu;
static uint8_t* g_static_ptr[64] = {};
static int static_scratch_address(int device, uint8_t** out)
{
    if (device < 0 || device >= 64) return NIV_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[device]) {
        NIV_CUDA(cudaSetDevice(device));
        void* p = nullptr;
        NIV_CUDA(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p) return NIV_ERR_CUDA;
        g_static_ptr[device] = static_cast<uint8_t*>(p);
    }
    *out = g_static_ptr[device];
    return NIV_OK;
}

extern "C" int niv_infer_host_static(niv_model* m, const float* pos, const float* nrm, const float* param,
                                     float* out, size_t n, void* stream)
{
    int rc = check_call(m, pos, nrm, out, n);
    if (rc != NIV_OK) return rc > 0 ? NIV_OK : rc;
    if (n > (size_t)NIV_STATIC_MAX_TEXELS) return NIV_ERR_TOO_LARGE;
    if (m->mma_kernel || !m->fused.fn) return NIV_ERR_UNSUPPORTED;
    KParams P;
    rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    set_formats(m, P, NIV_GBUF_F32X3, NIV_OUTFMT_F32X3);
    uint8_t* scratch = nullptr;
    rc = static_scratch_address(m->cfg.device, &scratch);
    if (rc != NIV_OK) return rc;
    NIV_CUDA(cudaSetDevice(m->cfg.device));
    cudaStream_t st = (cudaStream_t)stream;
    float* d_pos = reinterpret_cast<float*>(scratch + 256);
    float* d_nrm = reinterpret_cast<float*>(scratch + 256 + kStaticStage);
    float* d_out = reinterpret_cast<float*>(scratch + 256 + 2 * kStaticStage);
    NIV_CUDA(cudaMemsetAsync(scratch, 0, 256, st));                   // the tile counters must start at zero
    NIV_CUDA(cudaMemcpyAsync(d_pos, pos, n * 12, cudaMemcpyHostToDevice, st));
    NIV_CUDA(cudaMemcpyAsync(d_nrm, nrm, n * 12, cudaMemcpyHostToDevice, st));
    P.tile_ctr = reinterpret_cast<uint32_t*>(scratch);               // dynamic tile scheduling on the static counters
    P.slot_done = nullptr;
    P.slot_gen = 1;
    // no programmatic serialisation, no launch overlap: the launch is strictly ordered between its copies
    rc = launch_one(m, m->fused, st, false, P, d_pos, d_nrm, d_out, n, (uint32_t)((n + kTile - 1) / kTile));
    if (rc != NIV_OK) return rc;
    NIV_CUDA(cudaMemcpyAsync(out, d_out, n * 12, cudaMemcpyDeviceToHost, st));
    NIV_CUDA(cudaStreamSynchronize(st));
    return NIV_OK;
}

// The decoded fp32 position and normal of every texel of a compact G-buffer (what the fused kernels work on): for tests
// (bit-exact positions against the CPU decode) and for callers that want the fp32 buffers.
__global__ void __launch_bounds__(256) niv_decode_kernel(const __grid_constant__ KParams P, const float* __restrict__ a,
                                                         const float* __restrict__ b, float* __restrict__ pos,
                                                         float* __restrict__ nrm, size_t n)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float pr[3] = {0.f, 0.f, 0.f}, nr[3] = {0.f, 0.f, 0.f}, p[3], nv[3];
    load_texel_raw(P.gbuf_fmt, a, b, i, pr, nr);
    decode_texel(P, pr, nr, p, nv);
    for (int d = 0; d < 3; ++d) { pos[3 * i + d] = p[d]; nrm[3 * i + d] = nv[d]; }
}
extern "C" int niv_decode_gbuffer(niv_model* m, int gbuf_format, const void* gbuf_a, const void* gbuf_b, float* pos,
                                  float* nrm, size_t n, void* stream)
{
    FmtInfo f;
    if (!m || !pos || !nrm) return NIV_ERR_INVALID_ARG;
    if (!fmt_info(gbuf_format, NIV_OUTFMT_F32X3, f)) return NIV_ERR_INVALID_ARG;
    if (n == 0) return NIV_OK;
    if (!gbuf_a || (f.b_bytes && !gbuf_b)) return NIV_ERR_INVALID_ARG;
    if (((uintptr_t)gbuf_a & (f.in_align - 1)) || (f.b_bytes && ((uintptr_t)gbuf_b & (f.in_align - 1)))) return NIV_ERR_INVALID_ARG;
    KParams P = m->kp;
    set_formats(m, P, gbuf_format, NIV_OUTFMT_F32X3);
    niv_decode_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(P, (const float*)gbuf_a, (const float*)gbuf_b, pos, nrm, n);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_encode(niv_model* m, const float* pos, const float* nrm, const float* param,
                          void* features_fp16, size_t n, void* stream)
{
    if (!m) return NIV_ERR_INVALID_ARG;
    if (!m->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !features_fp16 || ((uintptr_t)features_fp16 & 15)) return NIV_ERR_INVALID_ARG;
    if (m->cfg.n_features != 2 || m->kernel_levels != m->cfg.n_levels || m->cfg.n_levels == 0)
        return NIV_ERR_UNSUPPORTED;                              // the stand-alone kernel serves F = 2 / SH-16, L a multiple of 4
    KParams P;
    int rc = fill_params(m, param, P);
    if (rc != NIV_OK) return rc;
    const unsigned grid = (unsigned)((n + 127) / 128);
    switch (m->info.cell_levels) {                     // (F = 2: four or five cell-block levels, or none)
        case 5:  niv_encode_kernel<5><<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (uint4*)features_fp16, n); break;
        case 4:  niv_encode_kernel<4><<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (uint4*)features_fp16, n); break;
        default: niv_encode_kernel<0><<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (uint4*)features_fp16, n); break;
    }
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
    NIV_CUDA(cudaMemsetAsync(counts, 0, NIV_CENSUS_COUNTS * sizeof(uint64_t), (cudaStream_t)stream));
    const unsigned grid = (unsigned)((n + 127) / 128);
    niv_sector_census_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(m->kp, pos, nrm, n, (unsigned long long*)counts, 1);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_probe_sectors_image(const niv_model* m, const float* pos, const float* nrm, uint32_t width,
                                       uint32_t height, uint64_t* counts, void* stream)
{
    if (!m || !pos || !nrm || !counts || width == 0 || height == 0) return NIV_ERR_INVALID_ARG;
    NIV_CUDA(cudaMemsetAsync(counts, 0, NIV_CENSUS_COUNTS * sizeof(uint64_t), (cudaStream_t)stream));
    KParams P = m->kp;
    P.img_w = width;
    P.img_h = height;
    P.tiles_x = (width + 31u) / 32u;
    const unsigned grid = P.tiles_x * ((height + 3u) / 4u);
    niv_sector_census_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(P, pos, nrm, (size_t)width * height,
                                                                     (unsigned long long*)counts, 1);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

// SM count of the current device, looked up once per device
static cudaError_t current_device_sms(int* sms)
{
    static std::atomic<int> cache[64];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    int v = (dev >= 0 && dev < 64) ? cache[dev].load(std::memory_order_relaxed) : 0;
    if (v == 0) {
        e = cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) cache[dev].store(v, std::memory_order_relaxed);
    }
    *sms = v;
    return cudaSuccess;
}

// Grid of 256-thread CTAs for a grid-stride loop over `items`: at most 8 CTAs per SM (one resident wave), and every
// thread the same number of iterations -- with min(ceil(items / 256), 8 * sms) CTAs a full-HD frame (518,400 groups
// of four pixels over 303,104 threads) gave 71 % of the threads two iterations and the rest one: a tail of 15 %
static unsigned balanced_grid(size_t items, int sms)
{
    const size_t wave = (size_t)sms * 8 * 256;
    const size_t iters = (items + wave - 1) / wave;
    const size_t threads = (items + iters - 1) / (iters ? iters : 1);
    return (unsigned)std::max<size_t>(1, (threads + 255) / 256);
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
    int sms = 0;
    NIV_CUDA(current_device_sms(&sms));
    cudaStream_t st = (cudaStream_t)stream;
    const uintptr_t align = (uintptr_t)albedo | (uintptr_t)out | (uintptr_t)(direct ? direct : albedo) |
                            (uintptr_t)(emission ? emission : albedo) | (half ? 0 : (uintptr_t)E);
    const size_t n = (size_t)w * h;
    if ((w & 3u) == 0 && (align & 15u) == 0) {
        const size_t groups = n / 4;
        const unsigned grid = balanced_grid(groups, sms);
        if (half) niv_compose_kernel<true><<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h);
        else niv_compose_kernel<false><<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h);
    } else {
        const unsigned grid = balanced_grid(n, sms);
        niv_compose_scalar_kernel<<<grid, 256, 0, st>>>(E, ew, eh, albedo, direct, emission, out, w, h, half);
    }
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_compose_jb(const float* E, const float* pos_half, const float* nrm_half, uint32_t ew, uint32_t eh,
                              const float* pos, const float* nrm, const float* albedo, const float* direct,
                              const float* emission, float sigma, float power, float* out, uint32_t w, uint32_t h,
                              void* stream)
{
    if (!E || !pos_half || !nrm_half || !pos || !nrm || !albedo || !out) return NIV_ERR_INVALID_ARG;
    if (!(sigma > 0.0f) || !std::isfinite(sigma) || !(power >= 0.0f) || !std::isfinite(power)) return NIV_ERR_INVALID_ARG;
    if (w == 0 || h == 0) return NIV_OK;
    if (2ull * ew != w || 2ull * eh != h) return NIV_ERR_INVALID_ARG;
    int sms = 0;
    NIV_CUDA(current_device_sms(&sms));
    const size_t n = (size_t)w * h;
    const unsigned grid = balanced_grid(n, sms);
    niv_compose_jb_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(E, pos_half, nrm_half, ew, eh, pos, nrm, albedo, direct,
                                                                  emission, 1.0f / (2.0f * sigma * sigma), power, out, w, h);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

// =====================================================================================================
// the probe-grid baseline
// =====================================================================================================
struct niv_probe_grid {
    niv_probe_config cfg;
    ProbeParams gp;
    uint4* d_probes = nullptr;
    size_t n_probes = 0;
    bool loaded = false;
};

extern "C" int niv_probes_create(const niv_probe_config* cfg, niv_probe_grid** out)
{
    if (!cfg || !out) return NIV_ERR_INVALID_ARG;
    *out = nullptr;
    if (cfg->struct_size != sizeof(niv_probe_config)) return NIV_ERR_INVALID_ARG;
    size_t n_probes = 1;
    for (int d = 0; d < 3; ++d) {
        if (cfg->dims[d] < 2 || cfg->dims[d] > 4096) return NIV_ERR_INVALID_ARG;
        if (!std::isfinite(cfg->bbox_min[d]) || !std::isfinite(cfg->bbox_max[d]) || !(cfg->bbox_max[d] > cfg->bbox_min[d]))
            return NIV_ERR_INVALID_ARG;
        n_probes *= cfg->dims[d];
    }
    if (n_probes > ((size_t)1 << 30) || cfg->cosine_falloff > 1) return NIV_ERR_INVALID_ARG;
    niv_probe_grid* g = new (std::nothrow) niv_probe_grid();
    if (!g) return NIV_ERR_ALLOC;
    g->cfg = *cfg;
    g->n_probes = n_probes;
    ProbeParams& G = g->gp;
    memset(&G, 0, sizeof(G));
    for (int d = 0; d < 3; ++d) {
        G.amin[d] = cfg->bbox_min[d];
        G.amax[d] = cfg->bbox_max[d];
        volatile float ext = cfg->bbox_max[d] - cfg->bbox_min[d];
        volatile float inv = 1.0f / ext;
        volatile float step = ext / (float)(cfg->dims[d] - 1);
        G.ainv[d] = inv;
        G.step[d] = step;
        G.nf[d] = (float)(cfg->dims[d] - 1);
        G.nm2[d] = (int32_t)cfg->dims[d] - 2;
        G.dims[d] = cfg->dims[d];
    }
    G.falloff = cfg->cosine_falloff;
    g_last_cuda_error = 0;
    cudaError_t e = cudaSetDevice(cfg->device);
    if (e == cudaSuccess) e = cudaMalloc(&g->d_probes, n_probes * 64);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); delete g; return e == cudaErrorMemoryAllocation ? NIV_ERR_ALLOC : NIV_ERR_CUDA; }
    G.probes = g->d_probes;
    *out = g;
    return NIV_OK;
}

extern "C" int niv_probes_load(niv_probe_grid* g, const void* coeffs_fp16, size_t bytes, int src_on_device, void* stream)
{
    if (!g || !coeffs_fp16 || bytes != g->n_probes * 54) return NIV_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    NIV_CUDA(cudaSetDevice(g->cfg.device));
    const uint16_t* src = (const uint16_t*)coeffs_fp16;
    uint16_t* tmp = nullptr;
    if (!src_on_device) {
        NIV_CUDA(cudaMalloc(&tmp, bytes));
        cudaError_t e = cudaMemcpyAsync(tmp, coeffs_fp16, bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { cudaFree(tmp); g_last_cuda_error = (int)e; return NIV_ERR_CUDA; }
        src = tmp;
    }
    const size_t total = g->n_probes * 32;
    niv_probes_pack_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(src, (uint16_t*)g->d_probes, g->n_probes);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (tmp) cudaFree(tmp);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); return NIV_ERR_CUDA; }
    g->loaded = true;
    return NIV_OK;
}

extern "C" int niv_probes_query(niv_probe_grid* g, const float* pos, const float* nrm, float* out, size_t n, void* stream)
{
    if (!g) return NIV_ERR_INVALID_ARG;
    if (!g->loaded) return NIV_ERR_NOT_LOADED;
    if (n == 0) return NIV_OK;
    if (!pos || !nrm || !out || n > ((size_t)1 << 31)) return NIV_ERR_INVALID_ARG;
    niv_probes_query_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(g->gp, pos, nrm, out, n);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_probes_census(niv_probe_grid* g, const float* pos, const float* nrm, size_t n, uint64_t* counts,
                                 void* stream)
{
    if (!g || !pos || !nrm || !counts || n == 0) return NIV_ERR_INVALID_ARG;
    NIV_CUDA(cudaMemsetAsync(counts, 0, 2 * sizeof(uint64_t), (cudaStream_t)stream));
    niv_probes_census_kernel<<<(unsigned)((n + 127) / 128), 128, 0, (cudaStream_t)stream>>>(g->gp, pos, nrm, n,
                                                                                           (unsigned long long*)counts);
    NIV_CUDA(cudaGetLastError());
    return NIV_OK;
}

extern "C" int niv_probes_destroy(niv_probe_grid* g)
{
    if (!g) return NIV_OK;
    cudaSetDevice(g->cfg.device);
    cudaFree(g->d_probes);
    delete g;
    return NIV_OK;
}

extern "C" int niv_destroy(niv_model* m)
{
    if (!m) return NIV_OK;
    forget_history();                       // launch records point at this model's completion words
    cudaSetDevice(m->cfg.device);
    cudaFree(m->d_table);
    cudaFree(m->d_cells);
    cudaFree(m->d_wpack);
    cudaFree(m->d_wpack_tp);
    cudaFree(m->d_ctr);
    if (m->h_done) cudaFreeHost((void*)m->h_done);
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
        case NIV_ERR_TOO_LARGE: return "more texels than the static scratch holds (NIV_STATIC_MAX_TEXELS)";
        default: return "unknown error code";
    }
}

extern "C" int niv_last_cuda_error(void) { return g_last_cuda_error; }

extern "C" int niv_probe_gather(const void* buf, size_t buf_bytes, int pattern, uint32_t n_ctas,
                                uint32_t loads_per_lane, uint32_t seed, void* sink, void* stream)
{
    if (!buf || !sink || buf_bytes < 4096 || (buf_bytes & (buf_bytes - 1)) || buf_bytes > ((size_t)1 << 33))
        return NIV_ERR_INVALID_ARG;
    if (pattern < 0 || pattern > 9 || n_ctas == 0 || loads_per_lane == 0 || (loads_per_lane & 7)) return NIV_ERR_INVALID_ARG;
    if (((uintptr_t)buf & 31) != 0) return NIV_ERR_INVALID_ARG;
    const uint32_t word_mask = (uint32_t)(buf_bytes / 4 - 1);
    const uint32_t* b = (const uint32_t*)buf;
    uint32_t* sk = (uint32_t*)sink;
    cudaStream_t st = (cudaStream_t)stream;
    cudaTextureObject_t tex = 0;
    if (pattern >= 8) {                                  // texture path: a 1-D linear texture of 32-bit texels over buf
        if (buf_bytes / 4 > ((size_t)1 << 27)) return NIV_ERR_INVALID_ARG;
        cudaResourceDesc rd;
        memset(&rd, 0, sizeof(rd));
        rd.resType = cudaResourceTypeLinear;
        rd.res.linear.devPtr = const_cast<void*>(buf);
        rd.res.linear.desc = cudaCreateChannelDesc<unsigned int>();
        rd.res.linear.sizeInBytes = buf_bytes;
        cudaTextureDesc td;
        memset(&td, 0, sizeof(td));
        td.readMode = cudaReadModeElementType;
        NIV_CUDA(cudaCreateTextureObject(&tex, &rd, &td, nullptr));
    }
#define NIV_PROBE_CASE(K) case K: niv_probe_gather_kernel<K><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk, tex); break;
    switch (pattern) {
        NIV_PROBE_CASE(0) NIV_PROBE_CASE(1) NIV_PROBE_CASE(2) NIV_PROBE_CASE(3) NIV_PROBE_CASE(4)
        NIV_PROBE_CASE(5) NIV_PROBE_CASE(6) NIV_PROBE_CASE(7) NIV_PROBE_CASE(8)
        default: niv_probe_gather_kernel<9><<<n_ctas, 256, 0, st>>>(b, word_mask, loads_per_lane, seed, sk, tex); break;
    }
#undef NIV_PROBE_CASE
    cudaError_t le = cudaGetLastError();
    if (tex) {                                           // the object must outlive the launch: wait for it
        cudaStreamSynchronize(st);
        cudaDestroyTextureObject(tex);
    }
    if (le != cudaSuccess) { g_last_cuda_error = (int)le; return NIV_ERR_CUDA; }
    return NIV_OK;
}
