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
