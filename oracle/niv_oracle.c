/*
 * niv_oracle.c -- CPU oracle for Neural Irradiance Volume (NIV) per-texel inference.
 *
 * TEST INFRASTRUCTURE.  Plain, slow, obviously-correct restatement of what the hot
 * path computes, written from the paper (arxiv 2602.12949, /root/reference/PAPER.md)
 * and the readings listed in DESIGN.md.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or constant generator with paper_2602_12949_b200/csrc (the CUDA path).
 *
 * What E_theta is (sec. 4.1; 402-403 sec. 4.4; 666-671 sec. 6):
 *   position x  --multi-level hash-grid encoding-->  L*F latents
 *   normal   n  --real spherical harmonics, bands 0..3--> 16 values  (BASELINE.json configs),
 *                 or the direction itself, 3 values (the paper's own model)
 *   scalar   t  --sin/cos frequency encoding-->  2*B values per parameter
 *   concat --> fully connected ReLU network, no activation on the final layer
 *    --> optional output activation --> RGB irradiance.
 *
 * Steps O0..O9 follow SURVEY.md sec. 8(c.3) / DESIGN.md "The algorithm":
 *   O0 mask, O1 normalise (fp32, pinned op order), O2 locate (fp32, pinned),
 *   O3 corner indices (integer), O4 trilinear blend (fp64), O5 SH-16 (fp64),
 *   O6 parameter encoding (fp64), O7 concat, O8 MLP (fp64 on fp16-valued weights),
 *   O9 output activation, cast to fp32.
 * Floating point is fp64 everywhere except O1/O2, whose fp32 op sequence decides an
 * integer (the cell) and is therefore part of the definition; build with
 * -ffp-contract=off so no fused multiply-add is formed.
 *
 * Parity pins (tests/test_oracle_pins.py): level tables, hash worked values, vertex /
 * voxel-centre queries, partition of unity, affine reproduction, torch grid_sample on
 * dense levels, brute-force tent-function sum on hashed levels, SH closed forms and
 * addition theorem, sin/cos examples, MLP closed forms and an fp64 matmul chain.
 * End-to-end E_theta has no printed value in the paper: "parity unpinned" by the paper
 * for the composition; it is pinned only through its parts.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NIV_ORACLE_MAX_LEVELS 16
#define NIV_ORACLE_MAX_DIM 512

typedef struct {
    uint32_t n_levels;          /* L */
    uint32_t n_features;        /* F, fp16 values per table entry */
    uint32_t log2_table_size;   /* T = 2^k entries per level */
    uint32_t base_resolution;   /* N0, cells per side at level 0 */
    double   per_level_scale;   /* b */
    uint32_t resolutions[NIV_ORACLE_MAX_LEVELS]; /* explicit N_l; all zero => derive */
    float    aabb_min[3], aabb_max[3];
    uint32_t sh_degree;         /* 4 => 16 coefficients */
    uint32_t n_params;          /* per-call scalars */
    uint32_t n_frequencies;     /* bands per scalar */
    uint32_t n_hidden_layers;
    uint32_t hidden_width;
    uint32_t out_activation;    /* 0 linear, 1 sigmoid */
    uint32_t dir_frequencies;   /* sh_degree 0 only: bands of frequency encoding appended to the raw direction (0 = none) */
} niv_oracle_config;

/* ---- fp16 -> fp64, exact, subnormals included (no flush to zero) ---- */
double niv_oracle_half_to_double(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1f;
    int m = h & 0x3ff;
    double v;
    if (e == 0)       v = ldexp((double)m, -24);                 /* subnormal: m * 2^-24 */
    else if (e == 31) v = m ? NAN : INFINITY;
    else              v = ldexp((double)(m + 1024), e - 25);     /* (1 + m/1024) * 2^(e-15) */
    return sign ? -v : v;
}

/* ---- level table: N_l = floor(N0 * b^l) cells per side (reading #2) ----
 * dense iff (N_l + 1)^3 <= T (reading #4; "latents of the finer levels are
 * stored in a hash table"). */
int niv_oracle_level_table(const niv_oracle_config *cfg, uint32_t *N, uint32_t *is_dense)
{
    if (!cfg || cfg->n_levels > NIV_ORACLE_MAX_LEVELS) return -1;
    int explicit_res = 0;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) if (cfg->resolutions[l]) explicit_res = 1;
    uint64_t T = (uint64_t)1 << cfg->log2_table_size;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        uint32_t n;
        if (explicit_res) n = cfg->resolutions[l];
        else              n = (uint32_t)floor((double)cfg->base_resolution * pow(cfg->per_level_scale, (double)l));
        if (n == 0) return -1;
        N[l] = n;
        uint64_t R = (uint64_t)n + 1;
        if (is_dense) is_dense[l] = (R * R * R <= T) ? 1u : 0u;
    }
    return 0;
}

/* ---- O3 spatial hash (reading #1): uint32 wrap-around products ---- */
uint32_t niv_oracle_hash(uint32_t vx, uint32_t vy, uint32_t vz, uint32_t log2_T)
{
    uint32_t h = (vx * 1u) ^ (vy * 2654435761u) ^ (vz * 805459861u);
    return h & (uint32_t)(((uint64_t)1 << log2_T) - 1);
}

void niv_oracle_param_encode(double t, uint32_t n_frequencies, double *out);

static int texel_masked(const float *p, const float *n)
{
    for (int d = 0; d < 3; ++d) if (!isfinite(p[d]) || !isfinite(n[d])) return 1;
    return n[0] == 0.0f && n[1] == 0.0f && n[2] == 0.0f;
}

/* ---- O1..O4 for one texel.  Any output pointer may be NULL. ---- */
static void encode_one(const niv_oracle_config *cfg, const uint32_t *N, const uint32_t *dense,
                       const uint16_t *table, const float *pos,
                       uint32_t *idx /*[L][8]*/, int32_t *cell /*[L][3]*/, float *frac /*[L][3]*/,
                       double *feat /*[L*F]*/)
{
    const uint32_t L = cfg->n_levels, F = cfg->n_features;
    const uint64_t T = (uint64_t)1 << cfg->log2_table_size;
    float u[3];
    /* O1 (fp32, one IEEE op per line) */
    for (int d = 0; d < 3; ++d) {
        float ext = cfg->aabb_max[d] - cfg->aabb_min[d];
        float inv = 1.0f / ext;
        float s = pos[d] - cfg->aabb_min[d];
        float v = s * inv;
        v = fmaxf(v, 0.0f);
        v = fminf(v, 1.0f);
        u[d] = v;
    }
    if (L == 0 && feat) {                                          /* grid-less: positional encoding of u */
        for (int d = 0; d < 3; ++d)
            niv_oracle_param_encode((double)u[d], cfg->n_frequencies, feat + 2 * cfg->n_frequencies * d);
    }
    for (uint32_t l = 0; l < L; ++l) {
        int32_t c[3];
        float w[3];
        const float Nf = (float)N[l];
        /* O2 (fp32) */
        for (int d = 0; d < 3; ++d) {
            float p = u[d] * Nf;
            int32_t ci = (int32_t)floorf(p);
            if (ci > (int32_t)N[l] - 1) ci = (int32_t)N[l] - 1;
            c[d] = ci;
            w[d] = p - (float)ci;
        }
        if (cell) for (int d = 0; d < 3; ++d) cell[l * 3 + d] = c[d];
        if (frac) for (int d = 0; d < 3; ++d) frac[l * 3 + d] = w[d];
        double acc[16];
        for (uint32_t k = 0; k < F; ++k) acc[k] = 0.0;
        for (int j = 0; j < 8; ++j) {
            /* O3: bit d of j selects the +1 corner on axis d (bit 0 = x) */
            uint32_t v[3];
            double omega = 1.0;
            for (int d = 0; d < 3; ++d) {
                int up = (j >> d) & 1;
                v[d] = (uint32_t)(c[d] + up);
                omega *= up ? (double)w[d] : 1.0 - (double)w[d];
            }
            uint32_t id;
            if (dense[l]) {
                uint32_t R = N[l] + 1;
                id = v[0] + R * (v[1] + R * v[2]);          /* x fastest (reading #5) */
            } else {
                id = niv_oracle_hash(v[0], v[1], v[2], cfg->log2_table_size);
            }
            if (idx) idx[l * 8 + j] = id;
            /* O4 */
            if (feat) {
                const uint16_t *e = table + ((uint64_t)l * T + id) * F;
                for (uint32_t k = 0; k < F; ++k) acc[k] += omega * niv_oracle_half_to_double(e[k]);
            }
        }
        if (feat) for (uint32_t k = 0; k < F; ++k) feat[l * F + k] = acc[k];
    }
}

/* ---- O5: real spherical harmonics, bands 0..3, positive signs (no Condon-Shortley phase),
 * index l(l+1)+m, band-1 order (y,z,x) (reading #13).  n used as given. ---- */
void niv_oracle_sh16(const double n[3], double out[16])
{
    const double PI = 3.14159265358979323846;
    const double x = n[0], y = n[1], z = n[2];
    const double c0  = 0.5 * sqrt(1.0 / PI);
    const double c1  = sqrt(3.0 / (4.0 * PI));
    const double c2a = 0.5 * sqrt(15.0 / PI);
    const double c2b = 0.25 * sqrt(5.0 / PI);
    const double c2c = 0.25 * sqrt(15.0 / PI);
    const double c3a = 0.25 * sqrt(35.0 / (2.0 * PI));
    const double c3b = 0.5 * sqrt(105.0 / PI);
    const double c3c = 0.25 * sqrt(21.0 / (2.0 * PI));
    const double c3d = 0.25 * sqrt(7.0 / PI);
    const double c3e = 0.25 * sqrt(105.0 / PI);
    out[0]  = c0;
    out[1]  = c1 * y;
    out[2]  = c1 * z;
    out[3]  = c1 * x;
    out[4]  = c2a * x * y;
    out[5]  = c2a * y * z;
    out[6]  = c2b * (3.0 * z * z - 1.0);
    out[7]  = c2a * x * z;
    out[8]  = c2c * (x * x - y * y);
    out[9]  = c3a * y * (3.0 * x * x - y * y);
    out[10] = c3b * x * y * z;
    out[11] = c3c * y * (5.0 * z * z - 1.0);
    out[12] = c3d * z * (5.0 * z * z - 3.0);
    out[13] = c3c * x * (5.0 * z * z - 1.0);
    out[14] = c3e * z * (x * x - y * y);
    out[15] = c3a * x * (x * x - 3.0 * y * y);
}

/* ---- O6: [sin(2^0 pi t), cos(2^0 pi t), ..., sin(2^(B-1) pi t), cos(2^(B-1) pi t)]
 * ("frequency encoding") ---- */
void niv_oracle_param_encode(double t, uint32_t n_frequencies, double *out)
{
    const double PI = 3.14159265358979323846;
    for (uint32_t k = 0; k < n_frequencies; ++k) {
        double a = ldexp(1.0, (int)k) * PI * t;
        out[2 * k]     = sin(a);
        out[2 * k + 1] = cos(a);
    }
}

/* ---- direction input (O5): sh_degree 4 -> the 16 real-SH values (BASELINE.json configs);
 * sh_degree 0 -> the direction itself, (x, y, z) as given: the paper's own model feeds "the input
 * position and direction" to the network and needs no basis functions (
 * SPEC.md:306 "raw 3-vector"). ---- */
/* With dir_frequencies = B > 0 the raw direction is followed by its frequency encoding ("directionEncoding:
 * raw 3-vector (plus optional frequency)", "The paper does not specify ... whether the direction vector is
 * frequency-encoded"; freq_encode of SPEC.md:211-214 on scalars in [-1, 1], axis after axis):
 *   [n_x, n_y, n_z | s(n_x) | s(n_y) | s(n_z)],  s(p) = [sin(2^0 pi p), cos(2^0 pi p), ..., sin(2^(B-1) pi p), cos(2^(B-1) pi p)]
 * = 3 + 6 B values (reading 3.8). */
static uint32_t dir_dim_of(const niv_oracle_config *cfg)
{
    return cfg->sh_degree == 0 ? 3u + 6u * cfg->dir_frequencies : cfg->sh_degree * cfg->sh_degree;
}

static void dir_encode(const niv_oracle_config *cfg, const double n[3], double *out)
{
    if (cfg->sh_degree == 0) {
        out[0] = n[0]; out[1] = n[1]; out[2] = n[2];
        for (int d = 0; d < 3; ++d)
            niv_oracle_param_encode(n[d], cfg->dir_frequencies, out + 3 + 2 * cfg->dir_frequencies * d);
    }
    else niv_oracle_sh16(n, out);
}

/* ---- position input: L > 0 -> the L*F grid latents (O1-O4); L == 0 -> the grid-less models of Table 1
 * ("Networks without grid encoding use eight-band positional encoding"): the normalised
 * position u (O1) is frequency-encoded per axis, x then y then z, each [sin(2^0 pi u), cos(2^0 pi u), ...,
 * sin(2^(B-1) pi u), cos(2^(B-1) pi u)] with B = n_frequencies. ---- */
static uint32_t pos_dim_of(const niv_oracle_config *cfg)
{
    return cfg->n_levels ? cfg->n_levels * cfg->n_features : 6 * cfg->n_frequencies;
}

static uint32_t in_dim_of(const niv_oracle_config *cfg)
{
    return pos_dim_of(cfg) + dir_dim_of(cfg) + 2 * cfg->n_frequencies * cfg->n_params;
}

uint32_t niv_oracle_in_dim(const niv_oracle_config *cfg) { return in_dim_of(cfg); }

/* ---- O8: h = W h + b, ReLU on all but the final layer;
 * W_k stored [out][in] row-major, layers in order (reading #18). ---- */
void niv_oracle_mlp(const niv_oracle_config *cfg, const uint16_t *weights, const float *biases,
                    const double *x, double y[3])
{
    double h0[NIV_ORACLE_MAX_DIM], h1[NIV_ORACLE_MAX_DIM];
    uint32_t n_in = in_dim_of(cfg);
    memcpy(h0, x, n_in * sizeof(double));
    double *cur = h0, *nxt = h1;
    const uint32_t n_layers = cfg->n_hidden_layers + 1;
    for (uint32_t k = 0; k < n_layers; ++k) {
        uint32_t n_out = (k + 1 == n_layers) ? 3u : cfg->hidden_width;
        for (uint32_t o = 0; o < n_out; ++o) {
            double s = 0.0;
            for (uint32_t i = 0; i < n_in; ++i)
                s += niv_oracle_half_to_double(weights[(uint64_t)o * n_in + i]) * cur[i];
            s += biases ? (double)biases[o] : 0.0;
            if (k + 1 != n_layers && s < 0.0) s = 0.0;
            nxt[o] = s;
        }
        weights += (uint64_t)n_out * n_in;
        if (biases) biases += n_out;
        n_in = n_out;
        double *t = cur; cur = nxt; nxt = t;
    }
    y[0] = cur[0]; y[1] = cur[1]; y[2] = cur[2];
}

static int check_cfg(const niv_oracle_config *cfg)
{
    if (!cfg) return -1;
    if (cfg->n_levels > NIV_ORACLE_MAX_LEVELS) return -1;
    if (cfg->n_levels == 0 && cfg->n_frequencies == 0) return -1;
    if (cfg->n_features == 0 || cfg->n_features > 16) return -1;
    if (cfg->log2_table_size == 0 || cfg->log2_table_size > 30) return -1;
    if (cfg->sh_degree != 4 && cfg->sh_degree != 0) return -1;
    if (cfg->dir_frequencies > 16 || (cfg->sh_degree != 0 && cfg->dir_frequencies != 0)) return -1;
    if (in_dim_of(cfg) > NIV_ORACLE_MAX_DIM || cfg->hidden_width > NIV_ORACLE_MAX_DIM) return -1;
    return 0;
}

/* ---- debug dump: idx [n][L][8] u32, cell [n][L][3] i32, frac [n][L][3] f32,
 * features [n][in_dim] f64 (hash latents | SH-16 | param encoding), zero for masked texels. ---- */
int niv_oracle_encode(const niv_oracle_config *cfg, const uint16_t *table,
                      const float *pos, const float *nrm, const float *param, size_t n,
                      uint32_t *idx, int32_t *cell, float *frac, double *features, int n_threads)
{
    if (check_cfg(cfg)) return -1;
    uint32_t N[NIV_ORACLE_MAX_LEVELS], dense[NIV_ORACLE_MAX_LEVELS];
    if (niv_oracle_level_table(cfg, N, dense)) return -1;
    const uint32_t L = cfg->n_levels, D = in_dim_of(cfg);
    (void)n_threads;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    #pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        uint32_t *ii = idx ? idx + (size_t)i * L * 8 : NULL;
        int32_t *cc = cell ? cell + (size_t)i * L * 3 : NULL;
        float *ff = frac ? frac + (size_t)i * L * 3 : NULL;
        double *xx = features ? features + (size_t)i * D : NULL;
        if (texel_masked(pos + 3 * i, nrm + 3 * i)) {               /* O0 */
            if (ii) memset(ii, 0, sizeof(uint32_t) * L * 8);
            if (cc) memset(cc, 0, sizeof(int32_t) * L * 3);
            if (ff) memset(ff, 0, sizeof(float) * L * 3);
            if (xx) memset(xx, 0, sizeof(double) * D);
            continue;
        }
        encode_one(cfg, N, dense, table, pos + 3 * i, ii, cc, ff, xx);
        if (xx) {
            double nn[3] = { (double)nrm[3 * i], (double)nrm[3 * i + 1], (double)nrm[3 * i + 2] };
            dir_encode(cfg, nn, xx + pos_dim_of(cfg));                         /* O5 */
            for (uint32_t q = 0; q < cfg->n_params; ++q)             /* O6 */
                niv_oracle_param_encode((double)param[q], cfg->n_frequencies,
                                        xx + pos_dim_of(cfg) + dir_dim_of(cfg) + 2 * cfg->n_frequencies * q);
        }
    }
    return 0;
}

/* ---- full path O0..O9.  out_f32 [n][3] and/or out_f64 [n][3] (either may be NULL). ---- */
static int infer_impl(const niv_oracle_config *cfg, const uint16_t *table,
                      const uint16_t *weights, const float *biases,
                      const float *pos, const float *nrm, const float *param_base, size_t param_stride,
                      float *out_f32, double *out_f64, size_t n, int n_threads)
{
    if (check_cfg(cfg)) return -1;
    uint32_t N[NIV_ORACLE_MAX_LEVELS], dense[NIV_ORACLE_MAX_LEVELS];
    if (niv_oracle_level_table(cfg, N, dense)) return -1;
    (void)n_threads;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    #pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        double y[3] = { 0.0, 0.0, 0.0 };
        const float *param = param_base ? param_base + (size_t)i * param_stride : NULL;   /* this texel's scalars */
        if (!texel_masked(pos + 3 * i, nrm + 3 * i)) {               /* O0 */
            double x[NIV_ORACLE_MAX_DIM];
            encode_one(cfg, N, dense, table, pos + 3 * i, NULL, NULL, NULL, x);   /* O1-O4 */
            double nn[3] = { (double)nrm[3 * i], (double)nrm[3 * i + 1], (double)nrm[3 * i + 2] };
            dir_encode(cfg, nn, x + pos_dim_of(cfg));                          /* O5, O7 */
            for (uint32_t q = 0; q < cfg->n_params; ++q)             /* O6, O7 */
                niv_oracle_param_encode((double)param[q], cfg->n_frequencies,
                                        x + pos_dim_of(cfg) + dir_dim_of(cfg) + 2 * cfg->n_frequencies * q);
            niv_oracle_mlp(cfg, weights, biases, x, y);              /* O8 */
            if (cfg->out_activation == 1)                            /* O9 */
                for (int c = 0; c < 3; ++c) y[c] = 1.0 / (1.0 + exp(-y[c]));
        }
        for (int c = 0; c < 3; ++c) {
            if (out_f32) out_f32[3 * i + c] = (float)y[c];
            if (out_f64) out_f64[3 * i + c] = y[c];
        }
    }
    return 0;
}

/* the scene parameters are the same for every texel of the call (one frame, one time of day: PAPER.md:669-671) */
int niv_oracle_infer(const niv_oracle_config *cfg, const uint16_t *table,
                     const uint16_t *weights, const float *biases,
                     const float *pos, const float *nrm, const float *param,
                     float *out_f32, double *out_f64, size_t n, int n_threads)
{
    return infer_impl(cfg, table, weights, biases, pos, nrm, param, 0, out_f32, out_f64, n, n_threads);
}

/* ---- f3: every texel carries its own scene parameters, tparam [n][n_params] f32 (several frames with different
 * t in one call, or a parameter that varies over the image).  The network input of texel i is O7 with
 * gamma(tparam[i][q]) in place of gamma(t[q]) -- the paper's "new inputs to the model" evaluated per
 * shading point; nothing else changes. ---- */
int niv_oracle_infer_texel_params(const niv_oracle_config *cfg, const uint16_t *table,
                                  const uint16_t *weights, const float *biases,
                                  const float *pos, const float *nrm, const float *tparam,
                                  float *out_f32, double *out_f64, size_t n, int n_threads)
{
    if (!cfg || cfg->n_params == 0 || !tparam) return -1;
    return infer_impl(cfg, table, weights, biases, pos, nrm, tparam, cfg->n_params, out_f32, out_f64, n, n_threads);
}

int niv_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- f2: deferred compose with optional half-resolution irradiance (Eq. 2 and Fig. 3 234-236:
 * L = rho/pi * E + D + L_e; "run at reduced resolution ... while still using the full size albedo
 * buffer"; "E bilinearly upsampled; multiplied by FULL-res albedo; D, emission at full res").
 * E is [eh][ew][3]; albedo, direct, emission, out are [h][w][3]; direct / emission may be NULL (zero).
 * (ew, eh) == (w, h): E is used per pixel.  (2 ew, 2 eh) == (w, h): E is upsampled bilinearly with pixel-centre
 * alignment -- full-res pixel x sits at half-res coordinate x/2 - 1/4, neighbours clamped to the edge (the paper
 * names no filter beyond "upsampling"; this is the plain bilinear one, identical to
 * torch.nn.functional.interpolate(scale_factor=2, mode="bilinear", align_corners=False)).  Returns -1 otherwise. ---- */
int niv_oracle_compose(const float *E, uint32_t ew, uint32_t eh, const float *albedo, const float *direct,
                       const float *emission, double *out, uint32_t w, uint32_t h)
{
    const double PI = 3.14159265358979323846;
    int half;
    if (!E || !albedo || !out || w == 0 || h == 0) return -1;
    if (ew == w && eh == h) half = 0;
    else if (2 * ew == w && 2 * eh == h) half = 1;
    else return -1;
    for (uint32_t y = 0; y < h; ++y)
        for (uint32_t x = 0; x < w; ++x)
            for (int c = 0; c < 3; ++c) {
                double e;
                if (!half) {
                    e = (double)E[((size_t)y * ew + x) * 3 + c];
                } else {
                    double fx = 0.5 * (double)x - 0.25, fy = 0.5 * (double)y - 0.25;
                    double x0f = floor(fx), y0f = floor(fy);
                    double tx = fx - x0f, ty = fy - y0f;
                    long x0 = (long)x0f, y0 = (long)y0f, x1 = x0 + 1, y1 = y0 + 1;
                    if (x0 < 0) x0 = 0;
                    if (y0 < 0) y0 = 0;
                    if (x1 > (long)ew - 1) x1 = (long)ew - 1;
                    if (y1 > (long)eh - 1) y1 = (long)eh - 1;
                    double e00 = (double)E[((size_t)y0 * ew + x0) * 3 + c], e10 = (double)E[((size_t)y0 * ew + x1) * 3 + c];
                    double e01 = (double)E[((size_t)y1 * ew + x0) * 3 + c], e11 = (double)E[((size_t)y1 * ew + x1) * 3 + c];
                    e = (1.0 - ty) * ((1.0 - tx) * e00 + tx * e10) + ty * ((1.0 - tx) * e01 + tx * e11);
                }
                size_t o = ((size_t)y * w + x) * 3 + c;
                double v = (double)albedo[o] / PI * e;
                if (direct) v += (double)direct[o];
                if (emission) v += (double)emission[o];
                out[o] = v;
            }
    return 0;
}

/* ---- f1: compact table storage.  PAPER.md:303 "latents of the finer levels are stored in a hash table": the coarse
 * (dense) levels need (N_l + 1)^3 entries only, which is the rule that reproduces Table 1's memory column (
 * reading #4).  The compact table is the levels back to back, a dense level with exactly (N_l + 1)^3 entries (x fastest,
 * as in the [L][T] layout), a hashed level with its T entries.  niv_oracle_table_compact copies [L][T] -> compact,
 * niv_oracle_table_expand the other way (unused entries zero); both return the compact size in ENTRIES, and may be
 * called with NULL buffers to get it. ---- */
static long long compact_walk(const niv_oracle_config *cfg, const uint16_t *src, uint16_t *dst, int to_compact)
{
    uint32_t N[NIV_ORACLE_MAX_LEVELS], dense[NIV_ORACLE_MAX_LEVELS];
    if (niv_oracle_level_table(cfg, N, dense)) return -1;
    const uint64_t T = (uint64_t)1 << cfg->log2_table_size, F = cfg->n_features;
    uint64_t off = 0;
    for (uint32_t l = 0; l < cfg->n_levels; ++l) {
        const uint64_t R = (uint64_t)N[l] + 1, cnt = dense[l] ? R * R * R : T;
        if (src && dst) {
            if (to_compact) memcpy(dst + off * F, src + (uint64_t)l * T * F, cnt * F * sizeof(uint16_t));
            else {
                memset(dst + (uint64_t)l * T * F, 0, T * F * sizeof(uint16_t));
                memcpy(dst + (uint64_t)l * T * F, src + off * F, cnt * F * sizeof(uint16_t));
            }
        }
        off += cnt;
    }
    return (long long)off;
}
long long niv_oracle_table_compact(const niv_oracle_config *cfg, const uint16_t *table, uint16_t *compact)
{
    return compact_walk(cfg, table, compact, 1);
}
long long niv_oracle_table_expand(const niv_oracle_config *cfg, const uint16_t *compact, uint16_t *table)
{
    return compact_walk(cfg, compact, table, 0);
}
