/*
 * niv_oracle_ext.c -- CPU oracle, second file: the operations around E_theta that SURVEY.md 8(f) lists as "next".
 *
 * TEST INFRASTRUCTURE, like niv_oracle.c (same rules: only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it; nothing is shared with paper_2602_12949_b200/csrc).
 * fp64 everywhere except the fp32 op sequences that decide an integer (a cell, a quantised code), which are part of
 * the definition and are written one IEEE operation per line; build with -ffp-contract=off.
 *
 *   niv_oracle_probe_query   SURVEY 8(f4): the paper's probe baseline (App. A)
 *   niv_oracle_decode_*      compact G-buffer formats (readings in DESIGN.md 3.4; PAPER.md:402-403 only
 *                            says "position and normal buffers")
 *   niv_oracle_quantise_*    fp16 / RGB9E5 output formats
 *   niv_oracle_upsample_jb   SURVEY 8(f2): joint-bilateral upsample of half-resolution irradiance
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

double niv_oracle_half_to_double(uint16_t h);            /* niv_oracle.c */
void niv_oracle_sh16(const double n[3], double out[16]); /* niv_oracle.c: bands 0..2 are its first 9 values */

static int masked6(const float *p, const float *n)
{
    for (int d = 0; d < 3; ++d)
        if (!isfinite(p[d]) || !isfinite(n[d])) return 1;
    return n[0] == 0.0f && n[1] == 0.0f && n[2] == 0.0f;
}

/* =====================================================================================================
 * Probe-grid query (the paper's DDGI-like baseline):
 *   "the directional indirect irradiance is represented using second-order spherical harmonics (9 coefficients)
 *    ... quantized to half-precision ... (54 bytes / probe)"
 *   "a cosine fall-off is applied such that probes behind the sampled normal do not contribute to trilinear
 *    interpolation"; "the interpolation weights are clamped to a small number (1e-6)"; "interpolation weights are
 *    re-normalized after the above heuristics".                       Ray-traced visibility is out of scope.
 * Steps (SPEC.md:365-368 `query` post-condition; readings P-a..P-f in DESIGN.md 3.6):
 *   P0 mask        as O0: nrm == 0 exactly or any input non-finite -> 0
 *   P1 normalise   u_d = clamp(fl32(fl32(x_d - min_d) * inv_d), 0, 1), inv_d = fl32(1 / fl32(max_d - min_d))   (fp32, as O1)
 *   P2 locate      p_d = fl32(u_d * (float)(n_d - 1)); c_d = min(floor(p_d), n_d - 2); w_d = fl32(p_d - c_d)    (fp32, as O2)
 *   P3 trilinear   probe j (bit d of j = +1 on axis d) at lattice point c + bits, weight prod_d (bit ? w_d : 1 - w_d);
 *                  probes stored x fastest: index vx + nx (vy + ny vz)
 *   P4 fall-off    weight *= max(0, dot(normalize(q_j - xc), n)), q_j the probe position, xc = x clamped into the box;
 *                  a probe AT xc (zero vector) keeps its weight (factor 1).  The vector q_j - xc is evaluated in fp32
 *                  with a pinned op sequence (step_d = fl32(fl32(max_d - min_d) / (float)(n_d - 1)),
 *                  q = fl32(fl32((float)v * step_d) + min_d), d = fl32(q - xc)): next to a probe the direction is
 *                  ill-conditioned in the probe position, and where its cosine crosses zero the weights are not
 *                  Lipschitz in it, so the precision of this one vector is part of the definition (reading P-e)
 *   P5 clamp       weight = max(weight, 1e-6);  P6 renormalise to sum 1
 *   P7 reconstruct E = sum_j weight_j sum_k c_jk Y_k(n), Y the real SH of bands 0..2 in the order and with the
 *                  constants of SPEC.md:341-345 (= the first nine of niv_oracle_sh16); coefficients [9][3] fp16 per probe
 * ===================================================================================================== */
int niv_oracle_probe_query(const uint32_t dims[3], const float bmin[3], const float bmax[3], int cosine_falloff,
                           const uint16_t *coeffs, const float *pos, const float *nrm, size_t n,
                           float *out32, double *out64, double *weights, uint32_t *probe_idx, int n_threads)
{
    if (!dims || !bmin || !bmax || !coeffs || !pos || !nrm) return -1;
    for (int d = 0; d < 3; ++d)
        if (dims[d] < 2 || !(bmax[d] > bmin[d])) return -1;
    float inv[3], step[3];
    for (int d = 0; d < 3; ++d) {
        volatile float ext = bmax[d] - bmin[d];
        volatile float iv = 1.0f / ext;
        volatile float st = ext / (float)(dims[d] - 1);
        inv[d] = iv;
        step[d] = st;
    }
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
#pragma omp parallel for schedule(static)
    for (long long ii = 0; ii < (long long)n; ++ii) {
        const size_t i = (size_t)ii;
        const float *p = pos + 3 * i, *nv = nrm + 3 * i;
        double E[3] = {0.0, 0.0, 0.0};
        double wj[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        uint32_t pj[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        if (!masked6(p, nv)) {
            int c[3];
            float w[3], xc[3];
            for (int d = 0; d < 3; ++d) {
                volatile float t0 = p[d] - bmin[d];                       /* P1 */
                volatile float t1 = t0 * inv[d];
                float u = t1;
                u = fminf(fmaxf(u, 0.0f), 1.0f);
                volatile float pp = u * (float)(dims[d] - 1);             /* P2 */
                int ci = (int)floorf(pp);
                if (ci > (int)dims[d] - 2) ci = (int)dims[d] - 2;
                volatile float ww = pp - (float)ci;
                c[d] = ci;
                w[d] = ww;
                xc[d] = fminf(fmaxf(p[d], bmin[d]), bmax[d]);
            }
            const double nd[3] = {(double)nv[0], (double)nv[1], (double)nv[2]};
            double sum = 0.0;
            for (int j = 0; j < 8; ++j) {
                double wt = 1.0, dvec[3], len2 = 0.0;
                uint32_t v[3];
                for (int d = 0; d < 3; ++d) {
                    const int bit = (j >> d) & 1;
                    v[d] = (uint32_t)(c[d] + bit);
                    wt *= bit ? (double)w[d] : 1.0 - (double)w[d];        /* P3 */
                    volatile float q0 = (float)v[d] * step[d];            /* P4: pinned fp32 sequence */
                    volatile float q1 = q0 + bmin[d];
                    volatile float dd = q1 - xc[d];
                    dvec[d] = (double)dd;
                    len2 += dvec[d] * dvec[d];
                }
                if (cosine_falloff && len2 > 0.0) {                       /* P4 */
                    const double len = sqrt(len2);
                    double dot = (dvec[0] * nd[0] + dvec[1] * nd[1] + dvec[2] * nd[2]) / len;
                    wt *= dot > 0.0 ? dot : 0.0;
                }
                if (wt < 1e-6) wt = 1e-6;                                 /* P5 */
                wj[j] = wt;
                pj[j] = v[0] + dims[0] * (v[1] + dims[1] * v[2]);
                sum += wt;
            }
            double Y[16];
            niv_oracle_sh16(nd, Y);
            for (int j = 0; j < 8; ++j) {
                wj[j] /= sum;                                             /* P6 */
                const uint16_t *cf = coeffs + (size_t)pj[j] * 27;
                for (int k = 0; k < 9; ++k)                               /* P7 */
                    for (int ch = 0; ch < 3; ++ch) E[ch] += wj[j] * niv_oracle_half_to_double(cf[3 * k + ch]) * Y[k];
            }
        }
        for (int ch = 0; ch < 3; ++ch) {
            if (out32) out32[3 * i + ch] = (float)E[ch];
            if (out64) out64[3 * i + ch] = E[ch];
        }
        if (weights) memcpy(weights + 8 * i, wj, sizeof(wj));
        if (probe_idx) memcpy(probe_idx + 8 * i, pj, sizeof(pj));
    }
    return 0;
}

/* =====================================================================================================
 * Compact G-buffer formats.  PAPER.md:402-403 says "position and normal buffers" and nothing about
 * their layout; the formats are this build's readings.  A texel is DECODED to an fp32 position and
 * an fp32 normal, and everything downstream (O0..O9) is defined on the decoded values.
 *   format 0  pos[n][3], nrm[n][3] fp32                                   (the layout of niv_oracle_infer)
 *   format 1  pos[n][4], nrm[n][4] fp32, w ignored
 *   format 2  one array of 16-byte records: x, y, z fp32 | oct, 2 x snorm16 (low half = first component)
 *   format 3  one array of 8-byte records: qx, qy, qz unorm16 of the box | oct, 2 x snorm8
 * D1 position, format 3 (fp32, one rounded operation per line -- it decides cells):
 *        u = fl32((float)q * fl32(1 / 65535));  t = fl32(u * fl32(max - min));  x = fl32(t + min)
 * D2 normal, formats 2 / 3: components v in [-32767, 32767] / [-127, 127] -> f = v / 32767 (/ 127); the reserved code
 *        (-32768, -32768) / (-128, -128) is "background": normal (0, 0, 0), which O0 masks.  Octahedral map:
 *        z = 1 - |fx| - |fy|;  if z < 0: (x, y) = ((1 - |fy|) sgn fx, (1 - |fx|) sgn fy) with sgn 0 = +1, else (fx, fy);
 *        n = (x, y, z) / |(x, y, z)|   in fp64, rounded to fp32 at the end.
 * ===================================================================================================== */
static void oct_decode(double fx, double fy, double n[3])
{
    double z = 1.0 - fabs(fx) - fabs(fy), x = fx, y = fy;
    if (z < 0.0) {
        x = copysign(1.0 - fabs(fy), fx);
        y = copysign(1.0 - fabs(fx), fy);
    }
    const double r = sqrt(x * x + y * y + z * z);
    n[0] = x / r; n[1] = y / r; n[2] = z / r;
}

int niv_oracle_decode_gbuffer(int format, const float bmin[3], const float bmax[3], const void *a, const void *b,
                              size_t n, float *pos, float *nrm)
{
    if (!a || !pos || !nrm || format < 0 || format > 3) return -1;
    if (format <= 1 && !b) return -1;
    if (format == 3 && (!bmin || !bmax)) return -1;
    for (size_t i = 0; i < n; ++i) {
        if (format <= 1) {
            const size_t s = format == 0 ? 3 : 4;
            for (int d = 0; d < 3; ++d) {
                pos[3 * i + d] = ((const float *)a)[s * i + d];
                nrm[3 * i + d] = ((const float *)b)[s * i + d];
            }
        } else if (format == 2) {
            const uint8_t *r = (const uint8_t *)a + 16 * i;
            uint32_t o;
            memcpy(pos + 3 * i, r, 12);
            memcpy(&o, r + 12, 4);
            const int ox = (int16_t)(o & 0xFFFFu), oy = (int16_t)(o >> 16);
            if (ox == -32768 && oy == -32768) {
                nrm[3 * i] = nrm[3 * i + 1] = nrm[3 * i + 2] = 0.0f;
            } else {
                double v[3];
                oct_decode(ox / 32767.0, oy / 32767.0, v);
                for (int d = 0; d < 3; ++d) nrm[3 * i + d] = (float)v[d];
            }
        } else {
            const uint8_t *r = (const uint8_t *)a + 8 * i;
            uint16_t q[3];
            memcpy(q, r, 6);
            const float k = 1.0f / 65535.0f;
            for (int d = 0; d < 3; ++d) {                        /* D1 */
                const float ext = bmax[d] - bmin[d];
                const float u = (float)q[d] * k;
                const float t = u * ext;
                pos[3 * i + d] = t + bmin[d];
            }
            const int ox = (int8_t)r[6], oy = (int8_t)r[7];
            if (ox == -128 && oy == -128) {
                nrm[3 * i] = nrm[3 * i + 1] = nrm[3 * i + 2] = 0.0f;
            } else {
                double v[3];
                oct_decode(ox / 127.0, oy / 127.0, v);
                for (int d = 0; d < 3; ++d) nrm[3 * i + d] = (float)v[d];
            }
        }
    }
    return 0;
}

/* =====================================================================================================
 * fp16 output ("fp16 / packed output formats"): out[i] = (r, g, b, 0) as four IEEE
 * binary16 values, each the round-to-nearest-even of the fp32 result (overflow -> infinity, subnormals kept).
 * ===================================================================================================== */
static uint16_t float_to_half_rne(float f)
{
    uint32_t x;
    memcpy(&x, &f, 4);
    const uint32_t sign = (x >> 16) & 0x8000u;
    const uint32_t mag = x & 0x7FFFFFFFu;
    if (mag >= 0x7F800000u) return (uint16_t)(sign | 0x7C00u | ((mag > 0x7F800000u) ? 0x200u : 0u));   /* inf / nan */
    if (mag >= 0x477FF000u) return (uint16_t)(sign | 0x7C00u);            /* >= 65520 rounds to infinity */
    if (mag < 0x33000001u) return (uint16_t)sign;                         /* <= 2^-25: rounds to zero (ties to even) */
    int e = (int)(mag >> 23) - 127;
    uint32_t m = (mag & 0x7FFFFFu) | 0x800000u;                           /* 24-bit significand */
    int shift = (e < -14) ? (13 + (-14 - e)) : 13;                        /* bits dropped */
    uint32_t half = m >> shift;
    const uint32_t rem = m & ((1u << shift) - 1u), halfway = 1u << (shift - 1);
    if (rem > halfway || (rem == halfway && (half & 1u))) ++half;
    if (e < -14) return (uint16_t)(sign | half);                          /* subnormal (a carry makes it the smallest normal) */
    /* normal: half holds 1.mantissa (11 bits); a carry out of the mantissa bumps the exponent by itself */
    return (uint16_t)(sign | ((uint32_t)((e + 15) << 10) + (half - 0x400u)));
}

int niv_oracle_quantise_f16x4(const float *e, size_t n, uint16_t *out)
{
    if (!e || !out) return -1;
    for (size_t i = 0; i < n; ++i) {
        for (int c = 0; c < 3; ++c) out[4 * i + c] = float_to_half_rne(e[3 * i + c]);
        out[4 * i + 3] = 0;
    }
    return 0;
}

/* ---- SURVEY 8 f2 "fp16 / packed output formats": the shared-exponent format RGB9E5 (DESIGN.md 3.5 reading) -------------
 * One 32-bit word per texel: three 9-bit mantissas r, g, b (bits 0-8, 9-17, 18-26) and one 5-bit exponent E (bits 27-31),
 * value_c = m_c * 2^(E - 15 - 9) -- the HDR colour format of the graphics APIs, restated here:
 *   Q1  c' = min(max(c, 0), 65408) per component (NaN -> 0; irradiance is not negative, a linear output layer may be);
 *       65408 = 511/512 * 2^16 is the largest representable value
 *   Q2  E' = max(-16, floor(log2 max_c c')) + 16                     (so that the largest mantissa has its top bit set)
 *   Q3  if floor(max_c c' / 2^(E' - 24) + 1/2) = 512 (the rounding carried): E = E' + 1, else E = E'
 *   Q4  m_c = floor(c' / 2^(E - 24) + 1/2)
 * All of it is exact in fp64 for fp32 inputs (scalings by powers of two, one addition of 1/2 to a number below 2^9). ---- */
int niv_oracle_quantise_rgb9e5(const float *e, size_t n, uint32_t *out)
{
    if (!e || !out) return -1;
    for (size_t i = 0; i < n; ++i) {
        double c[3], maxc = 0.0;
        for (int k = 0; k < 3; ++k) {
            double v = (double)e[3 * i + k];
            if (!(v > 0.0)) v = 0.0;                       /* negative, -0, NaN */
            if (v > 65408.0) v = 65408.0;
            c[k] = v;
            if (v > maxc) maxc = v;
        }
        int ex = -16;
        if (maxc > 0.0) {
            int fe;
            (void)frexp(maxc, &fe);                        /* maxc = f * 2^fe, f in [0.5, 1): floor(log2 maxc) = fe - 1 */
            if (fe - 1 > ex) ex = fe - 1;
        }
        int E = ex + 16;
        if (floor(ldexp(maxc, 24 - E) + 0.5) == 512.0) E += 1;
        uint32_t word = (uint32_t)E << 27;
        for (int k = 0; k < 3; ++k) word |= (uint32_t)floor(ldexp(c[k], 24 - E) + 0.5) << (9 * k);
        out[i] = word;
    }
    return 0;
}

/* the value an RGB9E5 word stands for (exact in fp64) */
int niv_oracle_decode_rgb9e5(const uint32_t *w, size_t n, double *out)
{
    if (!w || !out) return -1;
    for (size_t i = 0; i < n; ++i)
        for (int k = 0; k < 3; ++k) out[3 * i + k] = ldexp((double)((w[i] >> (9 * k)) & 0x1FFu), (int)(w[i] >> 27) - 24);
    return 0;
}

/* =====================================================================================================
 * Deferred compose with JOINT-BILATERAL upsampling of half-resolution irradiance.
 * half-resolution rendering "introduces aliasing artifacts which could be partly resolved by using
 * industry practice upsampling methods" (joint bilateral upsampling); SPEC.md:490 leaves it "a flagged extension".
 * The paper gives no formula; the reading is the classic one with the full-resolution G-buffer as guide:
 *   J1 footprint   the four half-res texels q of the bilinear upsample of niv_oracle_compose (full-res pixel x at
 *                  half-res coordinate x/2 - 1/4, neighbours clamped to the edge) with its bilinear weights b_q
 *   J2 range       g_q = exp(-|x_p - x_q|^2 / (2 sigma^2)) * max(0, n_p . n_q)^k     (world positions, normals as given)
 *   J3 floor       w_q = b_q (g_q + 1e-6): a pixel none of whose neighbours resembles it falls back, continuously, to
 *                  the plain bilinear blend (the floor of the paper's probe interpolation, reused)
 *   J4 blend       E_p = sum_q w_q E_q / sum_q w_q;      J5 compose  L = albedo / pi * E_p + direct + emission  (Eq. 2)
 * A clamped neighbour that coincides with another one simply appears twice (as in the bilinear blend).  fp64.
 * ===================================================================================================== */
int niv_oracle_compose_jb(const float *E, const float *pos_half, const float *nrm_half, uint32_t ew, uint32_t eh,
                          const float *pos, const float *nrm, const float *albedo, const float *direct,
                          const float *emission, double sigma, double power, double *out, uint32_t w, uint32_t h)
{
    const double PI = 3.14159265358979323846;
    if (!E || !pos_half || !nrm_half || !pos || !nrm || !albedo || !out || w == 0 || h == 0) return -1;
    if (2 * ew != w || 2 * eh != h || !(sigma > 0.0) || !(power >= 0.0)) return -1;
    for (uint32_t y = 0; y < h; ++y)
        for (uint32_t x = 0; x < w; ++x) {
            const size_t p = (size_t)y * w + x;
            const double fx = 0.5 * (double)x - 0.25, fy = 0.5 * (double)y - 0.25;
            const double x0f = floor(fx), y0f = floor(fy);
            const double tx = fx - x0f, ty = fy - y0f;
            long xs[2] = {(long)x0f, (long)x0f + 1}, ys[2] = {(long)y0f, (long)y0f + 1};
            for (int k = 0; k < 2; ++k) {
                if (xs[k] < 0) xs[k] = 0;
                if (ys[k] < 0) ys[k] = 0;
                if (xs[k] > (long)ew - 1) xs[k] = (long)ew - 1;
                if (ys[k] > (long)eh - 1) ys[k] = (long)eh - 1;
            }
            double acc[3] = {0.0, 0.0, 0.0}, wsum = 0.0;
            for (int j = 0; j < 4; ++j) {                                              /* J1 */
                const size_t q = (size_t)ys[j >> 1] * ew + (size_t)xs[j & 1];
                const double b = ((j & 1) ? tx : 1.0 - tx) * ((j >> 1) ? ty : 1.0 - ty);
                double d2 = 0.0, dot = 0.0;
                for (int d = 0; d < 3; ++d) {
                    const double dv = (double)pos[3 * p + d] - (double)pos_half[3 * q + d];
                    d2 += dv * dv;
                    dot += (double)nrm[3 * p + d] * (double)nrm_half[3 * q + d];
                }
                const double g = exp(-d2 / (2.0 * sigma * sigma)) * pow(dot > 0.0 ? dot : 0.0, power);   /* J2 */
                const double wq = b * (g + 1e-6);                                                       /* J3 */
                wsum += wq;
                for (int c = 0; c < 3; ++c) acc[c] += wq * (double)E[3 * q + c];
            }
            for (int c = 0; c < 3; ++c) {                                              /* J4, J5 */
                double v = (double)albedo[3 * p + c] / PI * (acc[c] / wsum);
                if (direct) v += (double)direct[3 * p + c];
                if (emission) v += (double)emission[3 * p + c];
                out[3 * p + c] = v;
            }
        }
    return 0;
}
