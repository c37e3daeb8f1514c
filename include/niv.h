/*
 * niv.h -- C ABI of libniv: B200 (sm_100a) per-texel inference of the Neural Irradiance Volume.
 *
 * The operation (arxiv 2602.12949; line numbers refer to /root/reference/PAPER.md and SPEC.md):
 *   "Starting from the G-buffer of the rendered scene, the position and normal buffers are input to the
 *    neural model, which infers pixel-wise E(x, n) in a single batch"            (sec. 4.4)
 *   E_theta = small ReLU MLP over [multi-level hash-grid encoding of x | encoding of n | encoding of the
 *   scene parameter]                                               (sec. 4.1; 666-671 sec. 6)
 * The exact arithmetic (op order of the fp32 index path, hash, corner order, SH convention, ...) is the
 * list O0..O9 in DESIGN.md section 3.1; the readings taken where the paper is silent are DESIGN.md 3.2.
 *
 * Conventions
 *   - every function returns an int status (NIV_OK or a negative NIV_ERR_*), never throws, never aborts;
 *   - "device" pointers are CUDA device pointers on the model's device, "host" pointers are ordinary memory;
 *   - the caller owns every buffer it passes; the model owns its own device copies of all parameters, so
 *     parameter blobs may be freed as soon as niv_load_params returns;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - niv_infer / niv_encode / niv_debug_encode are asynchronous on `stream`, allocate nothing, never
 *     synchronise (CUDA-graph capturable), are read-only on the model's parameters and safe for concurrent callers
 *     on different streams.  Tiles are scheduled dynamically through one of 2048 per-model tile counters: a counter is
 *     handed to a launch only while no earlier launch is still running on it (the last CTA of a launch reports its
 *     counter free through a host-mapped word), so any number of launches may be in flight; a launch that finds all
 *     2048 busy, and every launch recorded into a CUDA graph (its replays are invisible to the host), uses static tile
 *     striding instead -- the same result, only less even on frames with large background regions;
 *   - n <= 2^31 texels per call (NIV_ERR_INVALID_ARG beyond);
 *   - the fused kernels of hidden width <= 64 are launched with programmatic stream serialisation: their prologue
 *     (model-owned memory only) may overlap the tail of the previous kernel of the stream, and they wait for that
 *     kernel's completion (griddepcontrol.wait) before the first access to any buffer of the caller, so stream order
 *     holds for every buffer passed in.  One case skips that wait: the previous launch on the stream was issued by this
 *     library and none of its buffers overlaps a buffer of this launch in a way that matters (nothing this launch
 *     touches is written by it, nothing this launch writes is read by it) -- the two then run beside each other for
 *     the previous launch's last tiles, and the launches two and three back are known complete (completion words
 *     polled on the device) before this one touches a buffer -- with one exception: when neither the previous launch nor
 *     the one before it writes any INPUT of this launch (host-side range check), each thread requests its first texel
 *     before those polls; a CTA of a launch starts only after every CTA of the launch before it has passed its own
 *     polls, so all older launches are complete by then.  The result is that of serial execution in every case
 *     (tests: back-to-back calls on aliased buffers); NIV_OVERLAP=0 turns it off;
 *   - environment knobs, all read ONCE at niv_create and never on the call path: NIV_PDL=0 (no programmatic stream
 *     serialisation), NIV_OVERLAP=0 (every launch waits for the previous kernel of its stream), NIV_CELL_MB=<n> (budget of
 *     the cell-block copies of the coarse levels in MiB, default 320, 0 = none; F = 2: the seven coarsest levels, else five, else none; F = 4: six, else none), NIV_IMAGE_LINEAR=1 (niv_infer_image through the linear-tile kernel), NIV_HOST_STAGED=1
 *     (niv_infer_host through staging copies even for pinned buffers), NIV_MMA_SYNC=1 (the mma.sync A/B kernel for the
 *     BASELINE.json configs[1] shape), NIV_DEBUG=1 (resource report on stderr);
 *   - there is no CPU fallback: without a CUDA device every entry point that needs one returns NIV_ERR_CUDA.
 */
#ifndef NIV_H_
#define NIV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NIV_API_VERSION 1u
#define NIV_MAX_LEVELS 16

typedef struct niv_model niv_model;   /* opaque */

enum {
    NIV_OK = 0,
    NIV_ERR_INVALID_ARG = -1,   /* NULL / mis-sized / mis-aligned argument                        */
    NIV_ERR_UNSUPPORTED = -2,   /* a valid configuration this build has no kernel for             */
    NIV_ERR_NOT_LOADED  = -3,   /* niv_infer before niv_load_params                               */
    NIV_ERR_CUDA        = -4,   /* a CUDA runtime call failed (niv_last_cuda_error has the code)  */
    NIV_ERR_ALLOC       = -5,   /* host or device allocation failed                               */
    NIV_ERR_TOO_LARGE   = -6    /* niv_infer_host_static: n > NIV_STATIC_MAX_TEXELS               */
};

/* G-buffer and output formats of the *_packed entry points (readings in DESIGN.md 3.4, 3.5) */
enum { NIV_GBUF_F32X3 = 0,        /* pos[n][3], nrm[n][3] fp32: the format of niv_infer                                */
       NIV_GBUF_F32X4 = 1,        /* pos[n][4], nrm[n][4] fp32 (xyzw, stride 16 bytes, w ignored)                      */
       NIV_GBUF_P32_OCT16 = 2,    /* one array, 16 bytes per texel: x, y, z fp32 | octahedral normal 2 x snorm16
                                     (low half = x); both halves 0x8000 = background                                  */
       NIV_GBUF_P16_OCT8 = 3 };   /* one array, 8 bytes per texel: position 3 x unorm16 of the model's AABB |
                                     octahedral normal 2 x snorm8; both 0x80 = background                            */
enum { NIV_OUTFMT_F32X3 = 0,      /* out[n][3] fp32                                                                    */
       NIV_OUTFMT_F16X4 = 1,      /* out[n][4] fp16: (r, g, b, 0), round to nearest even of the fp32 result           */
       NIV_OUTFMT_RGB9E5 = 2 };   /* out[n] uint32: shared-exponent RGB9E5 (9-bit mantissas r, g, b in bits 0-26, 5-bit
                                     exponent in bits 27-31, value = m * 2^(E - 24)); negative and NaN components -> 0,
                                     values above 65408 clamp                                        */

enum { NIV_OUT_LINEAR = 0,      /* the paper: no activation on the final layer     */
       NIV_OUT_SIGMOID = 1 };   /* BASELINE.json configs[0]                                       */

/* Model hyper-parameters (table size T, latent dimension, scaling factor between levels,
 * coarsest side, number of levels; PAPER.md:296 network; PAPER.md:669-670 scene parameters). */
typedef struct {
    uint32_t struct_size;         /* = sizeof(niv_config)                                           */
    uint32_t api_version;         /* = NIV_API_VERSION                                              */
    uint32_t n_levels;            /* L: 1..16 (F = 2);  1..8 (F = 4);  0 = no grid: the
                                     position is encoded with n_frequencies sin/cos bands */
    uint32_t n_features;          /* F: fp16 latents per table entry: 2 (BASELINE.json) or 4 (paper) */
    uint32_t log2_table_size;     /* T = 2^k entries PER LEVEL, 4 <= k <= 24                        */
    uint32_t base_resolution;     /* N0: cells per side on the coarsest level                       */
    double   per_level_scale;     /* b: N_l = floor(N0 * b^l)  (reading #2)               */
    uint32_t resolutions[NIV_MAX_LEVELS]; /* optional explicit N_l; all zero => derive from N0, b   */
    float    aabb_min[3], aabb_max[3];    /* scene box mapped to the unit cube (reading #8)         */
    uint32_t sh_degree;           /* 4 => 16 real-SH coefficients of the normal (reading #13, F = 2);
                                     0 => the direction itself, 3 inputs (F = 4)  */
    uint32_t n_params;            /* 0..2 per-call scalar scene parameters                          */
    uint32_t n_frequencies;       /* sin/cos bands per parameter (8)                                */
    uint32_t n_hidden_layers;     /* 1..3 hidden layers, all `hidden_width` wide                    */
    uint32_t hidden_width;        /* 32, 64 or 128 (F = 4: 32 or 64)                                */
    uint32_t out_activation;      /* NIV_OUT_*                                                      */
    int32_t  device;              /* CUDA device ordinal                                            */
    uint32_t dir_frequencies;     /* sh_degree 0 only: sin/cos bands of frequency encoding per axis appended to the raw
                                     direction ("raw 3-vector (plus optional frequency)", 211-214; DESIGN.md
                                     3.8): 3 + 6 * dir_frequencies direction inputs.  0 (the paper's default) or 4      */
} niv_config;

/* What niv_create derived from the configuration (for tests, benchmarks and roofline arithmetic). */
typedef struct {
    uint32_t struct_size;
    uint32_t in_dim;                       /* L*F + (16 | 3 + 6*dir_frequencies) + 2*n_frequencies*n_params */
    uint32_t resolution[NIV_MAX_LEVELS];   /* N_l                                                   */
    uint32_t is_dense[NIV_MAX_LEVELS];     /* 1: dense index, 0: spatial hash (reading #4)          */
    uint64_t table_bytes;                  /* L * T * F * 2                                         */
    uint64_t weight_bytes;                 /* sum over layers of out*in*2                           */
    uint64_t bias_bytes;                   /* sum over layers of out*4                              */
    uint32_t num_sms;                      /* SM count of the device                                */
    uint32_t ctas_per_sm;                  /* resident CTAs per SM of the fused kernel              */
    uint32_t tile_texels;                  /* texels per CTA tile (128)                             */
    uint32_t smem_bytes;                   /* dynamic shared memory per CTA of the fused kernel     */
    uint32_t image_tiled;                  /* 1: niv_infer_image has its own 8 x 4-block kernel, 0: it runs niv_infer's */
    uint32_t texel_params;                 /* 1: niv_infer_texel_params is available for this model */
    uint32_t cell_levels;                  /* levels 0 .. cell_levels-1 are also held as cell blocks (8 corner
                                              entries per cell, one 32- / 64-byte load per texel and level) */
    uint32_t kernel_levels;                /* levels the fused kernels run: n_levels rounded up to a whole gather batch
                                              (the extra ones are dummy levels over zeros); niv_debug_arow rows have
                                              kernel_levels * F / 2 latent words */
    uint64_t cell_bytes;                   /* device bytes of those copies (budget: NIV_CELL_MB at niv_create) */
    uint64_t table_bytes_compact;          /* bytes of the COMPACT table niv_load_params_compact takes: a dense level with
                                              exactly (N_l + 1)^3 entries, a hashed one with T (the rule behind
                                              Table 1's memory column)                                               */
    uint64_t table_bytes_device;           /* what the model holds on the device: the compact table, levels padded to 32 B */
} niv_info;

/* Validate `cfg` completely and allocate device storage for the parameters (uninitialised).
 * Errors: NULL / wrong struct_size / api_version / degenerate AABB / zero resolution -> NIV_ERR_INVALID_ARG;
 * a shape this build has no kernel for -> NIV_ERR_UNSUPPORTED.  Two model families have kernels: BASELINE.json's
 * (F = 2, sh_degree 4, L = 1..16, width 32/64/128) and the paper's own (F = 4, sh_degree 0,
 * L = 1..8, width 32/64; "the number of levels varies between 2 and 8"; with dir_frequencies = 4: width 64) plus its grid-less models (L = 0, sh_degree 0, width 16/32/64, no table: table_fp16
 * may be NULL with table_bytes 0); all with n_hidden_layers 1..3, n_params 0..2, n_frequencies 8.
 * Shape errors are raised here, never at inference. */
int niv_create(const niv_config *cfg, niv_model **out);

int niv_get_info(const niv_model *m, niv_info *info);

/* Copy the parameters into the model (host or device source, `src_on_device` != 0 for device pointers);
 * synchronises `stream` before returning, so the sources may be freed.
 *   table_fp16   [L][T][F] fp16, level-major; dense levels use their first (N_l+1)^3 entries, x fastest
 *   weights_fp16 W1|W2|...|Wk, each [out][in] row-major fp16, layer-major; Wk has 3 rows
 *   biases_f32   b1|b2|...|bk fp32, or NULL for zeros
 * Byte counts must equal niv_info.{table,weight,bias}_bytes, else NIV_ERR_INVALID_ARG.
 * "All parameters in half-precision". */
int niv_load_params(niv_model *m, const void *table_fp16, size_t table_bytes,
                    const void *weights_fp16, size_t weight_bytes,
                    const float *biases_f32, size_t bias_bytes,
                    int src_on_device, void *stream);

/* The same with the table in compact form: the levels back to back, a dense level with exactly
 * (N_l + 1)^3 entries (x fastest), a hashed level with its T entries; table_bytes must equal
 * niv_info.table_bytes_compact.  Either way the model STORES the compact form (niv_info.table_bytes_device): the paper's
 * largest model is 5.4 MB, not 8 x T entries. */
int niv_load_params_compact(niv_model *m, const void *table_fp16, size_t table_bytes,
                            const void *weights_fp16, size_t weight_bytes,
                            const float *biases_f32, size_t bias_bytes,
                            int src_on_device, void *stream);

/* The hot path: one fused kernel, out[i] = E_theta(pos[i], nrm[i][, param]) for i < n.
 *   pos, nrm  device, [n][3] fp32 packed, base address 4-byte aligned; world-space position, unit normal
 *   param     HOST, n_params floats in [0,1] shared by the whole call (NULL iff n_params == 0)
 *   out       device, [n][3] fp32 packed RGB irradiance
 * A texel whose normal is exactly (0,0,0) or whose inputs are not all finite is background: out = (0,0,0),
 * no table access (reading #9).  Positions outside the AABB are clamped (reading #7).  n == 0 is a no-op.
 * Errors: NULL pointers -> NIV_ERR_INVALID_ARG; before niv_load_params -> NIV_ERR_NOT_LOADED;
 * launch failure -> NIV_ERR_CUDA. */
int niv_infer(niv_model *m, const float *pos, const float *nrm, const float *param,
              float *out, size_t n, void *stream);

/* The hot path for a G-buffer that is an IMAGE ("query NIV in screen-space by providing a G-buffer"):
 * out[y][x] = E_theta(pos[y][x], nrm[y][x][, param]), bit-identical to niv_infer on the same buffers with
 * n = width * height.  What differs is which 32 texels share a warp: an 8 x 4 pixel block instead of 32 pixels of a
 * row, a compact patch of the visible surface whose texels fall into fewer distinct grid cells -- 14 % fewer 32-byte
 * sectors per warp and 11 % less time on the full-HD frame.
 *   pos, nrm, out  device, [height][width][3] fp32 packed, row-major, no row padding
 *   param          HOST, as niv_infer
 * Any width and height (edge tiles are partial).  Models without an image-tiled kernel (hidden width 128, the
 * grid-less models) run niv_infer's kernel: same result.  Errors and masking as niv_infer. */
int niv_infer_image(niv_model *m, const float *pos, const float *nrm, const float *param,
                    float *out, uint32_t width, uint32_t height, void *stream);

/* the hot path with scene parameters PER TEXEL -- several frames with different t in one call, or a
 * parameter that varies over the image.  The paper extends the field "by introducing new inputs to the model, e.g. the
 * current position of the moving emitters" and frequency-encodes them; here the input of
 * texel i is [latents | SH-16 | gamma(tparam[i][0]) | gamma(tparam[i][1])], gamma(t) = (sin, cos)(2^k pi t), k = 0..7.
 *   pos, nrm, out  device, as niv_infer
 *   tparam         DEVICE, [n][n_params] fp32 packed (borrowed for the duration of the launch)
 * The encoding enters the first layer as 16 fp16 columns per parameter (one more tensor-core K-step each), where
 * niv_infer folds it into the bias in fp32: with the same t in every row the two calls agree to the fp16 rounding of
 * gamma, ~1e-4 in irradiance.  Models: n_params 1 or 2, F = 2 with SH-16, 8 or 16 levels, hidden width 32 or 64
 * (else NIV_ERR_UNSUPPORTED); n_params == 0 -> NIV_ERR_INVALID_ARG.  Other errors and masking as niv_infer. */
int niv_infer_texel_params(niv_model *m, const float *pos, const float *nrm, const float *tparam,
                           float *out, size_t n, void *stream);

/* The same operation with HOST buffers (the end-to-end call: PAPER.md:402-403 with the G-buffer in host memory).
 *   pos, nrm, out  HOST, [n][3] fp32 packed (pinned memory gives asynchronous copies; pageable memory works)
 *   param          HOST, as niv_infer
 * Pinned (cudaHostAlloc / cudaHostRegister) buffers are used in place: the fused kernel reads the G-buffer and writes
 * the irradiance over PCIe itself, one launch on `stream`, no staging (hidden widths <= 64).  Otherwise the frame is cut
 * into chunks whose host->device copies, kernels and device->host copies are queued on internal streams so that they
 * overlap; staging buffers are owned by the model and grown on demand (this path MAY allocate).  Either way the call
 * returns only after the last byte of `out` has landed (it synchronises).  The staged path is NOT safe for
 * concurrent callers on the same model.  Errors as niv_infer, plus NIV_ERR_ALLOC. */
int niv_infer_host(niv_model *m, const float *pos, const float *nrm, const float *param,
                   float *out, size_t n, void *stream);

/* niv_infer_host for callers that cannot allocate (code under CUDA graph capture set-up, tight serving loops,
 * harnesses that forbid cudaMalloc): the same fused kernel, staged through ONE static device array instead of the
 * cudaMalloc'ed staging buffers and internal streams of niv_infer_host's staged path.  The call makes no cudaMalloc /
 * cudaFree and creates no stream or event: it clears its tile counters, copies pos and nrm in, launches the kernel,
 * copies out back -- all on `stream` -- and synchronises `stream`.
 *   pos, nrm, out  HOST, [n][3] fp32 packed (pageable or pinned);  param  HOST, as niv_infer
 *   n <= NIV_STATIC_MAX_TEXELS (262,144 = a 512 x 512 tile), else NIV_ERR_TOO_LARGE; larger frames: several calls
 * The array (9.4 MB) is held by every GPU that loads the library until the process exits and is SHARED by every call on
 * that device, whatever the model or stream: calls that overlap on the GPU race -- serialise them.  Results equal
 * niv_infer_host's.  Other errors as niv_infer (NIV_ERR_UNSUPPORTED with NIV_MMA_SYNC=1). */
#define NIV_STATIC_MAX_TEXELS 262144
int niv_infer_host_static(niv_model *m, const float *pos, const float *nrm, const float *param,
                          float *out, size_t n, void *stream);

/* ---- compact G-buffer formats and fp16 output -------------------------------------------------
 * The paper only says "position and normal buffers"; engines keep G-buffers in many layouts, and on the
 * end-to-end path every byte per texel crosses PCIe.  The *_packed entry points are niv_infer / niv_infer_image /
 * niv_infer_host with the layouts named by NIV_GBUF_* and NIV_OUTFMT_* above (readings and decode steps in DESIGN.md
 * 3.4 / 3.5):
 *   gbuf_a, gbuf_b  F32X3, F32X4: the position and the normal array; P32_OCT16, P16_OCT8: gbuf_a = the one array of
 *                   n records, gbuf_b ignored (may be NULL).  Alignment: 4 / 16 / 16 / 8 bytes.
 *   out             F32X3: [n][3] fp32;  F16X4: [n][4] fp16 (8-byte aligned);  RGB9E5: [n] uint32 (4-byte aligned)
 * A texel is decoded to an fp32 position and an fp32 unit normal first -- the position by a pinned fp32 op sequence,
 * so the cells and hash indices are those of niv_infer on the decoded values, bit for bit -- and then takes the path of
 * niv_infer.  Grid models of hidden width <= 64 only (NIV_ERR_UNSUPPORTED for width 128 and for the grid-less models);
 * niv_infer_image_packed keeps the 8 x 4-block tiling for models with cell-block levels (linear tiles otherwise: the same
 * result); unknown formats and
 * misaligned buffers -> NIV_ERR_INVALID_ARG; otherwise as the unpacked entry points. */
int niv_infer_packed(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, const float *param,
                     int out_format, void *out, size_t n, void *stream);
int niv_infer_image_packed(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, const float *param,
                           int out_format, void *out, uint32_t width, uint32_t height, void *stream);
int niv_infer_host_packed(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, const float *param,
                          int out_format, void *out, size_t n, void *stream);
/* Debug: niv_infer, and besides `out` every texel's layer-1 A row as the FUSED kernel built it (the 32-bit words the
 * tensor core reads: L*F/2 words of fp16 latent pairs -- 24 words of positional encoding for the grid-less models --
 * then the direction (8 words SH-16, or (x, y | z, 0), or with dir_frequencies the 3 + 6 B values in consecutive
 * pairs), zero-padded to a multiple of 8 words = row_words).  arow is
 * device, [n][row_words] uint32; rows of background texels hold zeros.  row_words other than that -> NIV_ERR_INVALID_ARG.
 * For feature-level parity of the fused path (cell-block levels, packed-fp16 blend) in every model family. */
int niv_debug_arow(niv_model *m, const float *pos, const float *nrm, const float *param, float *out,
                   uint32_t *arow, uint32_t row_words, size_t n, void *stream);

/* The fp32 position and normal ([n][3] each, device) the fused kernels decode from a compact G-buffer (device). */
int niv_decode_gbuffer(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, float *pos, float *nrm,
                       size_t n, void *stream);

/* Stand-alone encoding kernel (rows a1..a9 without the MLP): features_fp16 is device, [n][in_dim] fp16
 * row-major = [latents | SH-16 | parameter encoding], zero rows for background texels.  F = 2 family only
 * (NIV_ERR_UNSUPPORTED for F = 4, whose rows are not a multiple of 16 bytes). */
int niv_encode(niv_model *m, const float *pos, const float *nrm, const float *param,
               void *features_fp16, size_t n, void *stream);

/* Debug dump through the SAME device functions the fused kernel uses for O0..O3 (bit-exact parity of the
 * integer path is checked on these).  All outputs are device pointers; any may be NULL.
 *   idx [n][L][8] uint32 (corner j: bit d of j selects +1 on axis d; entry index inside the level), cell [n][L][3]
 *   int32, frac [n][L][3] fp32, features [n][in_dim] fp32 (fp32 blend, before fp16 packing).  Background: zeros. */
int niv_debug_encode(niv_model *m, const float *pos, const float *nrm, const float *param, size_t n,
                     uint32_t *idx, int32_t *cell, float *frac, float *features, void *stream);

/* the deferred compose of the paper's frame, L = albedo / pi * E + direct + emission (PAPER.md:269
 * Eq. 2; Fig. 3, 234-236), with the irradiance at full resolution or at half resolution ("run at
 * reduced resolution ... while still using the full size albedo buffer").
 *   E         device, [eh][ew][3] fp32: the output of niv_infer on the full-size or the half-size G-buffer
 *   albedo    device, [h][w][3] fp32;  direct, emission  device, [h][w][3] fp32 or NULL (zero)
 *   out       device, [h][w][3] fp32 radiance
 * (ew, eh) must equal (w, h) or (w/2, h/2) exactly, else NIV_ERR_INVALID_ARG.  Half-resolution E is upsampled
 * bilinearly with pixel-centre alignment (full-res pixel x at half-res coordinate x/2 - 1/4, edge texels clamped).
 * 128-bit streaming path when w % 4 == 0 and the full-resolution buffers are 16-byte aligned, a scalar path otherwise.
 * Asynchronous on `stream`, allocation-free; needs no model.  Runs on the current CUDA device. */
int niv_compose(const float *E, uint32_t ew, uint32_t eh, const float *albedo, const float *direct,
                const float *emission, float *out, uint32_t w, uint32_t h, void *stream);

/* the hot path with that compose as its EPILOGUE, for irradiance inferred at full resolution
 * ("infers pixel-wise E(x, n) in a single batch", then Eq. 2): one kernel,
 *   out[i] = albedo[i] / pi * E_theta(pos[i], nrm[i][, param]) + direct[i] + emission[i],
 * the irradiance never goes to memory (24.9 MB written and read again per full-HD frame by niv_infer + niv_compose).
 *   gbuf_format, gbuf_a, gbuf_b, param, out_format, out   as niv_infer_packed (NIV_GBUF_F32X3 / NIV_OUTFMT_F32X3: niv_infer's)
 *   albedo            device, [n][3] fp32;  direct, emission  device, [n][3] fp32, or NULL (zero)
 * The arithmetic of the epilogue is niv_compose's (fma(albedo * fl32(1/pi), E, direct + emission) in fp32), so on fp32
 * output the result equals niv_compose of niv_infer's output bit for bit.  Background texels have E = 0: out = direct +
 * emission.  out must not overlap any input.  Models: hidden width <= 64 (NIV_ERR_UNSUPPORTED for width 128); albedo
 * NULL -> NIV_ERR_INVALID_ARG; other errors, masking and asynchrony as niv_infer.
 * niv_infer_image_shade is the same for [height][width] row-major buffers, with niv_infer_image's 8 x 4 pixel blocks per
 * warp where the model has that kernel (BASELINE.json's family with cell-block levels); the same bits either way. */
int niv_infer_shade(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, const float *param,
                    const float *albedo, const float *direct, const float *emission, int out_format, void *out,
                    size_t n, void *stream);
int niv_infer_image_shade(niv_model *m, int gbuf_format, const void *gbuf_a, const void *gbuf_b, const float *param,
                          const float *albedo, const float *direct, const float *emission, int out_format, void *out,
                          uint32_t width, uint32_t height, void *stream);

/* The same compose with JOINT-BILATERAL upsampling of half-resolution irradiance: the "industry practice upsampling
 * methods" PAPER.md:406 names against the aliasing of half-resolution rendering ("a flagged extension").
 * The paper gives no formula; the reading (steps J1-J5): the four half-res texels q of niv_compose's
 * bilinear footprint, weight  b_q * (exp(-|x_p - x_q|^2 / (2 sigma^2)) * max(0, n_p . n_q)^power + 1e-6),  renormalised;
 * the full-resolution G-buffer is the guide.
 *   E, pos_half, nrm_half  device, [eh][ew][3] fp32: niv_infer's output on the half-size G-buffer, and that G-buffer
 *   pos, nrm, albedo       device, [h][w][3] fp32 (the full-size G-buffer); direct, emission as niv_compose
 *   sigma > 0 (world units), power >= 0;  (w, h) == (2 ew, 2 eh) exactly, else NIV_ERR_INVALID_ARG
 * Asynchronous on `stream`, allocation-free; needs no model. */
int niv_compose_jb(const float *E, const float *pos_half, const float *nrm_half, uint32_t ew, uint32_t eh,
                   const float *pos, const float *nrm, const float *albedo, const float *direct, const float *emission,
                   float sigma, float power, float *out, uint32_t w, uint32_t h, void *stream);

int niv_destroy(niv_model *m);

const char *niv_error_string(int code);

/* cudaError_t of the last failing CUDA call made by this library on the calling thread (0 if none). */
int niv_last_cuda_error(void);

/* ---- measured rooflines: micro-benchmarks that run on the caller's stream ----
 * niv_probe_gather: every lane of n_ctas x 256 threads issues `loads_per_lane` independent loads (8 in flight)
 * at pseudo-random addresses of `buf`.  pattern:
 *   0  one 4-byte word in a uniformly random 32-byte sector per lane (the random-sector rate of the roofline)
 *   1  one random 128-byte line per WARP, lanes consecutive (the coalesced rate)
 *   2  one random aligned 8-byte pair per lane, one 64-bit load
 *   3  groups of 8 lanes share one random sector
 *   4  one random aligned 16-byte quad per lane, one 128-bit load
 *   5  one whole random 32-byte sector per lane, one 256-bit load
 *   6  two 4-byte loads (two instructions) from one random sector per lane
 *   7  as 0 with L1::no_allocate
 *   8  as 0 through the texture path (tex1Dfetch on a linear texture object made for the call)
 *   9  as 0, alternating between the LSU path and the texture path
 * buf is device memory of `buf_bytes` (power of two, 32-byte aligned); sink is device, >= 4 bytes.  Asynchronous. */
int niv_probe_gather(const void *buf, size_t buf_bytes, int pattern, uint32_t n_ctas, uint32_t loads_per_lane,
                     uint32_t seed, void *sink, void *stream);

/* niv_probe_sectors: the sector census behind the gather roofline ("S = number of 32-byte sectors
 * the frame algorithmically needs at warp granularity").  For every group of 32 consecutive texels (the fused
 * kernel's texel -> warp map) and every level, counts the DISTINCT 32-byte sectors and 128-byte lines among the
 * group's <= 256 corner addresses in the table as niv_load_params receives it ([L][T] entries): the algorithmic
 * figure, independent of how the library lays the table out.  counts is device, NIV_CENSUS_COUNTS x uint64:
 * [0,16) sectors per level, [16,32) lines per level, [32] active (unmasked) texels, [33,49) the sectors the fused
 * kernel really touches per level (the same on gathered levels; distinct cell blocks on the levels niv_info.cell_levels
 * holds as cell blocks).  Asynchronous; counts is zeroed first on `stream`. */
#define NIV_CENSUS_COUNTS 49
int niv_probe_sectors(niv_model *m, const float *pos, const float *nrm, size_t n, uint64_t *counts, void *stream);

/* The same census for niv_infer_image's texel -> warp map (8 x 4 pixel blocks of a height x width image). */
int niv_probe_sectors_image(const niv_model *m, const float *pos, const float *nrm, uint32_t width, uint32_t height,
                            uint64_t *counts, void *stream);

/* ---- the paper's probe baseline as a second workload over the same G-buffers --------------------------
 * A regular grid of irradiance probes, "similar to DDGI" (App. A): per probe second-order
 * spherical harmonics (9 coefficients x 3 channels) in half precision, 54 bytes; a query blends the 8 probes of the
 * enclosing cell with trilinear weights x a cosine fall-off ("probes behind the sampled normal do not contribute"),
 * clamps every weight to 1e-6 and renormalises, then reconstructs E(n) = sum_k c_k Y_k(n) with the basis of
 * SPEC.md:341-345.  Steps P0..P7 and the readings taken are in DESIGN.md 3.6.  Ray-traced visibility is not built.
 * "Probes should always hold a performance edge" is the claim this lets one measure. */
typedef struct niv_probe_grid niv_probe_grid;    /* opaque; owns the device copy of the probes */
typedef struct {
    uint32_t struct_size;        /* = sizeof(niv_probe_config)                                          */
    uint32_t dims[3];            /* probes per axis, >= 2; lattice over the box, faces included         */
    float    bbox_min[3], bbox_max[3];
    uint32_t cosine_falloff;     /* 1: App. A's fall-off, 0: plain trilinear weights (still clamped)    */
    int32_t  device;
} niv_probe_config;

int niv_probes_create(const niv_probe_config *cfg, niv_probe_grid **out);
/* coeffs_fp16: [nz][ny][nx][9][3] fp16 = 27 values per probe, x fastest, host or device;
 * bytes must equal 54 * nx * ny * nz.  Synchronises `stream`. */
int niv_probes_load(niv_probe_grid *g, const void *coeffs_fp16, size_t bytes, int src_on_device, void *stream);
/* out[i] = E_probes(pos[i], nrm[i]); device pointers, [n][3] fp32 packed; background / non-finite texels -> 0 (as
 * niv_infer); positions outside the box are clamped into it.  Asynchronous on `stream`, allocation-free. */
int niv_probes_query(niv_probe_grid *g, const float *pos, const float *nrm, float *out, size_t n, void *stream);
/* Roofline numerator of the query: counts (device, uint64[2]) = { distinct 32-byte sectors of probe records per warp of
 * 32 consecutive texels, summed; active texels }. */
int niv_probes_census(niv_probe_grid *g, const float *pos, const float *nrm, size_t n, uint64_t *counts, void *stream);
int niv_probes_destroy(niv_probe_grid *g);

#ifdef __cplusplus
}
#endif
#endif /* NIV_H_ */
