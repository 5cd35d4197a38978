/*
 * lacosmic_oracle.c -- CPU ORACLE for the L.A.Cosmic iteration.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct definition that the CUDA path is
 * checked against.  It is NOT part of the product: only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or helper with paper_2602_17938_b200/csrc/.
 *
 * What it follows
 *   step list : PAPER.md:53-62 (section Methods/Algorithm, items 1-7)
 *   formulas  : BASELINE.json north_star (1)-(7)
 *   readings  : SURVEY.md section 8(c), O0-O7 and R1-R20 (restated in DESIGN.md section 3);
 *               R21 (gain estimation, PAPER.md:74,43 -- SURVEY.md 8(f)-2) in DESIGN.md section 3
 *
 * Precision: north_star fixes fp32 ("4000x6500 fp32 L.A.Cosmic", "fp32 L+, N, S and S'"),
 * so every arithmetic step is ONE fp32 round-to-nearest operation, in the order written
 * (compile with -ffp-contract=off, never -ffast-math).  Every median is a full sort of the
 * gathered window (insertion sort) followed by picking the middle element.  No blocking,
 * fusion, or reordering: each step materialises its whole plane before the next starts.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): closed forms for constant and
 * single-spike frames, scipy.ndimage median_filter / binary_dilation equivalence, brute
 * force on tiny tiles, hand-computed replacement cases (tests/golden/), 180-degree rotation
 * and flip invariance, fixed-point behaviour of the iteration.  No function here is
 * "parity unpinned".
 *
 * Notation: X<y,x> = X[clamp(y,0,h-1)][clamp(x,0,w-1)]  (edge-replicate read of a stored
 * plane, R3).  OpenMP only splits independent output rows between threads.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_MEM (-2)

/* R1: Laplacian kernel [0 -1 0; -1 4 -1; 0 -1 0], no 1/4 normalisation. */

typedef struct {
    int iter;          /* which iteration (0-based) to dump */
    float *Lp, *N, *S, *Sp, *m3, *F;       /* fp32 [h][w], nullable */
    uint8_t *G1, *G2, *M1, *M2, *M3, *C;   /* 0/1 [h][w], nullable; C = cumulative mask AFTER the iteration */
    float *work_in;                        /* the iteration's input image, nullable */
} orc_debug;

static inline int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

static inline float rd(const float *X, int h, int w, int y, int x) {
    return X[(size_t)clampi(y, 0, h - 1) * (size_t)w + (size_t)clampi(x, 0, w - 1)];
}

static void sort_ascending(float *v, int n) { /* insertion sort */
    for (int i = 1; i < n; ++i) {
        float t = v[i];
        int j = i - 1;
        while (j >= 0 && v[j] > t) { v[j + 1] = v[j]; --j; }
        v[j + 1] = t;
    }
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_get_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* O1 -- north_star (1).  2x block-replicate, 3x3 Laplacian, clip, 2x2 block-average.
 * Sub-pixel (2y+i, 2x+j) of the replicated grid has value c; two of its four 4-neighbours lie in
 * its own block (value c), one is the vertical neighbour V in {U,D} and one the horizontal
 * neighbour H in {Lf,R}:  4c - c - c - V - H = 2c - (V + H).  Clamping on the 2h x 2w grid and on
 * the h x w grid select the same neighbours. */
void orc_lplus(const float *work, float *Lp, int h, int w) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            float c = work[(size_t)y * w + x];
            float U = rd(work, h, w, y - 1, x), D = rd(work, h, w, y + 1, x);
            float Lf = rd(work, h, w, y, x - 1), R = rd(work, h, w, y, x + 1);
            float two = 2.0f * c;
            float a = two - (U + Lf);
            float b = two - (U + R);
            float g = two - (D + Lf);
            float d = two - (D + R);
            a = a > 0.0f ? a : 0.0f;
            b = b > 0.0f ? b : 0.0f;
            g = g > 0.0f ? g : 0.0f;
            d = d > 0.0f ? d : 0.0f;
            Lp[(size_t)y * w + x] = ((a + b) + (g + d)) * 0.25f;
        }
}

/* True (non-separable) k x k median; edge-replicate (R3).  k in {3,5,7}. */
int orc_medfilt(const float *X, float *out, int h, int w, int k) {
    if (!(k == 3 || k == 5 || k == 7) || h < 1 || w < 1) return ORC_ERR_ARG;
    int r = (k - 1) / 2, n = k * k;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y) {
        float v[49];
        for (int x = 0; x < w; ++x) {
            int m = 0;
            for (int dy = -r; dy <= r; ++dy)
                for (int dx = -r; dx <= r; ++dx) v[m++] = rd(X, h, w, y + dy, x + dx);
            sort_ascending(v, n);
            out[(size_t)y * w + x] = v[(n - 1) / 2];
        }
    }
    return ORC_OK;
}

/* 3x3 binary dilation, 8-connected, out-of-frame = 0 (O6, R10). */
void orc_dilate3(const uint8_t *in, uint8_t *out, int h, int w) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            uint8_t o = 0;
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    int yy = y + dy, xx = x + dx;
                    if (yy >= 0 && yy < h && xx >= 0 && xx < w && in[(size_t)yy * w + xx]) o = 1;
                }
            out[(size_t)y * w + x] = o;
        }
}

/* O7 -- north_star (7), R13-R16.  out = img where mask == 0; where mask != 0 the
 * median of the 5x5 edge-replicated taps of img whose (clamped) pixel is unmasked; duplicated
 * taps count with multiplicity; even count -> mean of the two middle values; no donor -> plain
 * median of all 25 taps. */
void orc_masked_median(const float *img, const uint8_t *mask, float *out, int h, int w) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y) {
        float v[25];
        for (int x = 0; x < w; ++x) {
            size_t p = (size_t)y * w + x;
            if (!mask[p]) { out[p] = img[p]; continue; }
            int k = 0;
            for (int dy = -2; dy <= 2; ++dy)
                for (int dx = -2; dx <= 2; ++dx) {
                    size_t q = (size_t)clampi(y + dy, 0, h - 1) * w + (size_t)clampi(x + dx, 0, w - 1);
                    if (!mask[q]) v[k++] = img[q];
                }
            if (k == 0)
                for (int dy = -2; dy <= 2; ++dy)
                    for (int dx = -2; dx <= 2; ++dx) v[k++] = rd(img, h, w, y + dy, x + dx);
            sort_ascending(v, k);
            out[p] = (k & 1) ? v[k / 2] : (v[k / 2 - 1] + v[k / 2]) * 0.5f;
        }
    }
}

/* ---- R21: gain estimation ("If a gain is not supplied, then it will be estimated at each
 * iteration"; PAPER.md:43 sigma_clip).  The paper gives no formula; R21 is the reading:
 * for Poisson-dominated noise var(work) = signal/gain, so r = (work - med5(work)) / sqrt(med5(work)) has
 * standard deviation 1/sqrt(gain).  sigma is estimated robustly and ORDER-INDEPENDENTLY (selection
 * only, no sums): three rounds of { c = median of r over the kept set, d = median of |r - c| over the
 * kept set, s = 1.4826 d, keep c - 5 s <= r <= c + 5 s (intersected with the previous interval) },
 * "median" = the element of 0-based rank (n-1)/2 of the ascending sort.  The gain then follows from s and
 * the read noise through the noise model itself (orc_estimate_gain below). */
static int cmp_float(const void *a, const void *b) {
    float x = *(const float *)a, y = *(const float *)b;
    return (x > y) - (x < y);
}

/* rank-(n-1)/2 element of v[0..n-1] by a full sort (v is reordered) */
static float lower_median(float *v, size_t n) {
    qsort(v, n, sizeof(float), cmp_float);
    return v[(n - 1) / 2];
}

/* sigma clipping of r[0..n-1] as defined above.  stats (nullable) receives, for the LAST round,
 * {c, s, lo, hi, kept count} where lo/hi is the interval the round started from.  Returns s. */
float orc_sigma_clip(const float *r, size_t n, int rounds, float *stats) {
    float lo = -INFINITY, hi = INFINITY, c = 0.0f, s = 0.0f;
    float *v = malloc((n ? n : 1) * sizeof(float));
    if (!v) return NAN;
    for (int j = 0; j < rounds; ++j) {
        size_t m = 0;
        for (size_t p = 0; p < n; ++p)
            if (r[p] >= lo && r[p] <= hi) v[m++] = r[p];
        if (m == 0) break;
        float lo0 = lo, hi0 = hi;
        c = lower_median(v, m);
        m = 0;
        for (size_t p = 0; p < n; ++p)
            if (r[p] >= lo0 && r[p] <= hi0) v[m++] = fabsf(r[p] - c);
        float d = lower_median(v, m);
        s = 1.4826f * d;
        float five_s = 5.0f * s;
        float nlo = c - five_s, nhi = c + five_s;
        if (stats) { stats[0] = c; stats[1] = s; stats[2] = lo0; stats[3] = hi0; stats[4] = (float)m; }
        lo = nlo > lo0 ? nlo : lo0;
        hi = nhi < hi0 ? nhi : hi0;
    }
    free(v);
    return s;
}

/* gain estimate of one image (the `work` plane of an iteration).  stats: nullable float[6] = the sigma-clip
 * statistics above plus stats[5] = mt.  The noise model of O2 is var(work) = signal/gain + (rn/gain)^2, so
 * with sigma^2 = var(r) = var(work)/signal:  sigma^2 gain^2 - gain - rn^2/mt = 0, mt = the typical signal =
 * rank-(n-1)/2 element of max(med5, 1e-4) over the pixels the last clipping round kept.  The positive root,
 * in this operation order (fp32):  s2 = s*s;  a = ((4*s2)*rn2)/mt;  gain = (1 + sqrt(1 + a)) / (2*s2).
 * rn = 0 gives gain = 1/s2 exactly.  gain = 1 if s is 0 or the result is not finite and positive. */
int orc_estimate_gain(const float *work, int h, int w, float readnoise, float *gain_out, float *stats) {
    if (!work || !gain_out || h < 1 || w < 1 || !(readnoise >= 0.0f)) return ORC_ERR_ARG;
    size_t P = (size_t)h * (size_t)w;
    float *m5 = malloc(P * 4), *r = malloc(P * 4), *v = malloc(P * 4);
    if (!m5 || !r || !v) { free(m5); free(r); free(v); return ORC_ERR_MEM; }
    orc_medfilt(work, m5, h, w, 5);
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < P; ++p) {
        float m = m5[p] > 1e-4f ? m5[p] : 1e-4f;
        float dev = work[p] - m5[p];
        r[p] = dev / sqrtf(m);
    }
    float st[5];
    float s = orc_sigma_clip(r, P, 3, st);
    /* typical signal over the set the last round kept: st[2] <= r <= st[3] */
    size_t m = 0;
    for (size_t p = 0; p < P; ++p)
        if (r[p] >= st[2] && r[p] <= st[3]) v[m++] = m5[p] > 1e-4f ? m5[p] : 1e-4f;
    float mt = m ? lower_median(v, m) : 1.0f;
    const float rn2 = readnoise * readnoise;
    float s2 = s * s;
    float a = ((4.0f * s2) * rn2) / mt;
    float g = (1.0f + sqrtf(1.0f + a)) / (2.0f * s2);
    *gain_out = (s > 0.0f && isfinite(s) && isfinite(g) && g > 0.0f) ? g : 1.0f;
    if (stats) { memcpy(stats, st, sizeof st); stats[5] = mt; }
    free(m5); free(r); free(v);
    return ORC_OK;
}

#define COPY_IF(dst, src, bytes) do { if (dst) memcpy((dst), (src), (bytes)); } while (0)

/* The whole path: O0-O7 of SURVEY.md 8(c).  Returns 0, or <0 on bad arguments / out of memory.
 * iter_counts (nullable) receives new_t for t = 0..niter-1; dbg (nullable) receives the planes
 * of iteration dbg->iter; iter_gains (nullable) the gain used in each iteration (gain == 0: R21).  All niter iterations are always executed (R17: stopping at new_t = 0
 * would give the identical result; the oracle does not take the shortcut). */
int orc_run(const float *img, int h, int w, float gain, float readnoise, float sigclip,
            float sigfrac, float objlim, int niter, float satlevel, uint8_t *mask_out,
            float *clean_out, int32_t *iter_counts, orc_debug *dbg, float *iter_gains) {
    if (!img || !mask_out || !clean_out || h < 1 || w < 1 || niter < 0) return ORC_ERR_ARG;
    const int estimate = (gain == 0.0f);   /* R21: gain 0 = "not supplied" */
    if (!(gain >= 0.0f) || !(readnoise >= 0.0f) || !(sigclip > 0.0f) || !(sigfrac > 0.0f) ||
        !(objlim >= 0.0f))
        return ORC_ERR_ARG;
    size_t P = (size_t)h * (size_t)w;
    float *work = clean_out;
    float *Lp = malloc(P * 4), *m5 = malloc(P * 4), *N = malloc(P * 4), *S = malloc(P * 4);
    float *mS = malloc(P * 4), *Sp = malloc(P * 4), *m3 = malloc(P * 4), *m7 = malloc(P * 4);
    float *F = malloc(P * 4);
    uint8_t *G1 = malloc(P), *G2 = malloc(P), *M1 = malloc(P), *D = malloc(P), *M2 = malloc(P);
    uint8_t *M3 = malloc(P), *C = mask_out;
    int rc = ORC_OK;
    if (!Lp || !m5 || !N || !S || !mS || !Sp || !m3 || !m7 || !F || !G1 || !G2 || !M1 || !D ||
        !M2 || !M3) {
        rc = ORC_ERR_MEM;
        goto done;
    }
    /* O0 */
    memset(C, 0, P);
    memcpy(work, img, P * 4);
    const float siglow = sigfrac * sigclip;   /* R9: one fp32 multiply */
    const float rn2 = readnoise * readnoise;

    for (int t = 0; t < niter; ++t) {
        if (dbg && dbg->iter == t) COPY_IF(dbg->work_in, work, P * 4);
        if (estimate) {   /* R21: estimated at each iteration, from the iteration's input image */
            rc = orc_estimate_gain(work, h, w, readnoise, &gain, NULL);
            if (rc) goto done;
        }
        if (iter_gains) iter_gains[t] = gain;
        /* O1 */
        orc_lplus(work, Lp, h, w);
        /* O2 -- north_star (2): N = sqrt(gain*med5(img) + rn^2)/gain, med5 floored at 1e-4 (R5) */
        orc_medfilt(work, m5, h, w, 5);
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {
            float m = m5[p] > 1e-4f ? m5[p] : 1e-4f;
            float gm = gain * m;
            float var = gm + rn2;
            N[p] = sqrtf(var) / gain;
        }
        /* O3 -- north_star (3): S = L+/(2N); S' = S - med5(S) */
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {
            float twoN = 2.0f * N[p];
            S[p] = Lp[p] / twoN;
        }
        orc_medfilt(S, mS, h, w, 5);
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) Sp[p] = S[p] - mS[p];
        /* O4 -- north_star (4): F = med3(img) - med7(med3(img)), floored at 0.01; med7 replicates
         * the stored m3 plane's edges (R4) */
        orc_medfilt(work, m3, h, w, 3);
        orc_medfilt(m3, m7, h, w, 7);
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {
            float f = m3[p] - m7[p];
            F[p] = f > 0.01f ? f : 0.01f;
        }
        /* O5 -- north_star (5), R8 (strict >, IEEE division then compare), R12 (satlevel) */
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {
            int ok = work[p] < satlevel;
            G1[p] = (uint8_t)(ok && (Sp[p] > sigclip));
            G2[p] = (uint8_t)(ok && (Sp[p] > siglow));
            float ratio = Lp[p] / F[p];
            M1[p] = (uint8_t)(G1[p] && (ratio > objlim));
        }
        /* O6 -- north_star (6), R10, R11 */
        orc_dilate3(M1, D, h, w);
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) M2[p] = (uint8_t)(D[p] && G1[p]);
        orc_dilate3(M2, D, h, w);
        int64_t newc = 0;
#pragma omp parallel for schedule(static) reduction(+ : newc)
        for (size_t p = 0; p < P; ++p) {
            M3[p] = (uint8_t)(D[p] && G2[p]);
            if (M3[p] && !C[p]) ++newc;
            C[p] = (uint8_t)(C[p] || M3[p]);
        }
        if (iter_counts) iter_counts[t] = (int32_t)newc;
        /* O7 -- donors from img_in, cumulative mask (R13) */
        orc_masked_median(img, C, work, h, w);

        if (dbg && dbg->iter == t) {
            COPY_IF(dbg->Lp, Lp, P * 4); COPY_IF(dbg->N, N, P * 4); COPY_IF(dbg->S, S, P * 4);
            COPY_IF(dbg->Sp, Sp, P * 4); COPY_IF(dbg->m3, m3, P * 4); COPY_IF(dbg->F, F, P * 4);
            COPY_IF(dbg->G1, G1, P); COPY_IF(dbg->G2, G2, P); COPY_IF(dbg->M1, M1, P);
            COPY_IF(dbg->M2, M2, P); COPY_IF(dbg->M3, M3, P); COPY_IF(dbg->C, C, P);
        }
    }
done:
    free(Lp); free(m5); free(N); free(S); free(mS); free(Sp); free(m3); free(m7); free(F);
    free(G1); free(G2); free(M1); free(D); free(M2); free(M3);
    return rc;
}

/* ======================================================================================================
 * SURVEY.md 8(f)-3 / 8(f)-4 variants (readings R22-R26).  Everything above is untouched: orc_run
 * stays the definition of the north-star path; orc_run_ex below restates the same loop with the variant
 * branches written in, and a pin checks that with no variant selected it equals orc_run bit for bit.
 * ====================================================================================================== */

/* R26: separable k x k median (the approximation PAPER.md:29,37 argues AGAINST; comparison only):
 * T[y][x] = middle element of the k values X<y, x+dx>, |dx| <= (k-1)/2 (row pass);
 * out[y][x] = middle element of the k values T<y+dy, x>, |dy| <= (k-1)/2 (column pass on the stored T plane). */
int orc_sepmedfilt(const float *X, float *out, int h, int w, int k) {
    if (!(k == 3 || k == 5 || k == 7) || h < 1 || w < 1) return ORC_ERR_ARG;
    int r = (k - 1) / 2;
    float *T = malloc((size_t)h * w * 4);
    if (!T) return ORC_ERR_MEM;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y) {
        float v[7];
        for (int x = 0; x < w; ++x) {
            for (int dx = -r; dx <= r; ++dx) v[dx + r] = rd(X, h, w, y, x + dx);
            sort_ascending(v, k);
            T[(size_t)y * w + x] = v[r];
        }
    }
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y) {
        float v[7];
        for (int x = 0; x < w; ++x) {
            for (int dy = -r; dy <= r; ++dy) v[dy + r] = rd(T, h, w, y + dy, x);
            sort_ascending(v, k);
            out[(size_t)y * w + x] = v[r];
        }
    }
    free(T);
    return ORC_OK;
}

/* R25: extended saturated-star mask.  core = (med5(img) >= satlevel): the pixels whose 5x5 edge-replicated
 * neighbourhood is saturated in its majority (an isolated saturated pixel, e.g. a strong cosmic-ray hit, is not a
 * core); out = core dilated `grow` times by the 3x3 square (grow = 0: the core itself). */
int orc_satstar_mask(const float *img, int h, int w, float satlevel, int grow, uint8_t *out) {
    if (!img || !out || h < 1 || w < 1 || grow < 0) return ORC_ERR_ARG;
    size_t P = (size_t)h * w;
    float *m5 = malloc(P * 4);
    uint8_t *tmp = malloc(P);
    if (!m5 || !tmp) { free(m5); free(tmp); return ORC_ERR_MEM; }
    orc_medfilt(img, m5, h, w, 5);
    for (size_t p = 0; p < P; ++p) out[p] = (uint8_t)(m5[p] >= satlevel);
    for (int j = 0; j < grow; ++j) {
        orc_dilate3(out, tmp, h, w);
        memcpy(out, tmp, P);
    }
    free(m5); free(tmp);
    return ORC_OK;
}

/* O7 with an input bad-pixel mask (R23): as orc_masked_median, but a tap is a donor iff its (clamped) pixel is
 * neither in `mask` nor in `bpm`; no donor -> plain median of all 25 taps (R15).  bpm == NULL: orc_masked_median. */
void orc_masked_median_bpm(const float *img, const uint8_t *mask, const uint8_t *bpm, float *out, int h, int w) {
#pragma omp parallel for schedule(static)
    for (int y = 0; y < h; ++y) {
        float v[25];
        for (int x = 0; x < w; ++x) {
            size_t p = (size_t)y * w + x;
            if (!mask[p]) { out[p] = img[p]; continue; }
            int k = 0;
            for (int dy = -2; dy <= 2; ++dy)
                for (int dx = -2; dx <= 2; ++dx) {
                    size_t q = (size_t)clampi(y + dy, 0, h - 1) * w + (size_t)clampi(x + dx, 0, w - 1);
                    if (!mask[q] && !(bpm && bpm[q])) v[k++] = img[q];
                }
            if (k == 0)
                for (int dy = -2; dy <= 2; ++dy)
                    for (int dx = -2; dx <= 2; ++dx) v[k++] = rd(img, h, w, y + dy, x + dx);
            sort_ascending(v, k);
            out[p] = (k & 1) ? v[k / 2] : (v[k / 2 - 1] + v[k / 2]) * 0.5f;
        }
    }
}

typedef struct {
    int fsmode;          /* 0: R7, the north-star test L+/F > objlim with F in ADU;
                            1: R22, noise-normalised fine structure: Fn = max((m3 - m7)/N, 0.01), test S'/Fn > objlim */
    int satgrow;         /* < 0: off; k >= 0: R25, pixels of orc_satstar_mask(img_in, satlevel, k) are never flagged */
    int sepmed;          /* 0: true medians; 1: R26, every median of O2-O4 replaced by orc_sepmedfilt (comparison) */
    const uint8_t *bpm;  /* nullable [h][w], R23: != 0 = bad pixel: never flagged, never a donor */
    const float *var;    /* nullable [h][w], R24: variance plane [ADU^2]: N = sqrt(max(var, 1e-8)), replaces O2 */
} orc_variant;

static int medfilt_v(const float *X, float *out, int h, int w, int k, int sepmed) {
    return sepmed ? orc_sepmedfilt(X, out, h, w, k) : orc_medfilt(X, out, h, w, k);
}

/* The whole path with the variants of R22-R26.  v == NULL or all-default: identical to orc_run.
 * R23/R25: nok = bpm OR satstar; O5's `ok` becomes (work < satlevel) AND NOT nok, so such pixels are never candidates
 * and never added by growth (hence never in C, never replaced).  R23 also removes bad pixels from the donors of O7.
 * R24: with a variance plane O2 is replaced by N = sqrt(max(var, 1e-8)); the gain is then not used (never estimated).
 * The dumped F plane is Fn when fsmode == 1. */
int orc_run_ex(const float *img, int h, int w, float gain, float readnoise, float sigclip, float sigfrac,
               float objlim, int niter, float satlevel, const orc_variant *v, uint8_t *mask_out, float *clean_out,
               int32_t *iter_counts, orc_debug *dbg, float *iter_gains) {
    static const orc_variant none = {0, -1, 0, NULL, NULL};
    if (!v) v = &none;
    if (!img || !mask_out || !clean_out || h < 1 || w < 1 || niter < 0) return ORC_ERR_ARG;
    if (!(v->fsmode == 0 || v->fsmode == 1) || !(v->sepmed == 0 || v->sepmed == 1)) return ORC_ERR_ARG;
    const int estimate = (gain == 0.0f) && !v->var;
    if (!(gain >= 0.0f) || !(readnoise >= 0.0f) || !(sigclip > 0.0f) || !(sigfrac > 0.0f) || !(objlim >= 0.0f))
        return ORC_ERR_ARG;
    size_t P = (size_t)h * (size_t)w;
    float *work = clean_out;
    float *Lp = malloc(P * 4), *m5 = malloc(P * 4), *N = malloc(P * 4), *S = malloc(P * 4);
    float *mS = malloc(P * 4), *Sp = malloc(P * 4), *m3 = malloc(P * 4), *m7 = malloc(P * 4);
    float *F = malloc(P * 4);
    uint8_t *G1 = malloc(P), *G2 = malloc(P), *M1 = malloc(P), *D = malloc(P), *M2 = malloc(P);
    uint8_t *M3 = malloc(P), *nok = malloc(P), *C = mask_out;
    int rc = ORC_OK;
    if (!Lp || !m5 || !N || !S || !mS || !Sp || !m3 || !m7 || !F || !G1 || !G2 || !M1 || !D || !M2 || !M3 || !nok) {
        rc = ORC_ERR_MEM;
        goto done;
    }
    memset(C, 0, P);
    memcpy(work, img, P * 4);
    const float siglow = sigfrac * sigclip;
    const float rn2 = readnoise * readnoise;
    /* R23 / R25: the pixels that may never be flagged, fixed for the frame (from img_in) */
    memset(nok, 0, P);
    if (v->satgrow >= 0) {
        rc = orc_satstar_mask(img, h, w, satlevel, v->satgrow, nok);
        if (rc) goto done;
    }
    if (v->bpm)
        for (size_t p = 0; p < P; ++p) nok[p] = (uint8_t)(nok[p] || v->bpm[p]);

    for (int t = 0; t < niter; ++t) {
        if (dbg && dbg->iter == t) COPY_IF(dbg->work_in, work, P * 4);
        if (estimate) {
            rc = orc_estimate_gain(work, h, w, readnoise, &gain, NULL);
            if (rc) goto done;
        }
        if (iter_gains) iter_gains[t] = gain;
        orc_lplus(work, Lp, h, w);                                                /* O1 */
        if (v->var) {                                                             /* R24 */
#pragma omp parallel for schedule(static)
            for (size_t p = 0; p < P; ++p) {
                float vv = v->var[p] > 1e-8f ? v->var[p] : 1e-8f;
                N[p] = sqrtf(vv);
            }
        } else {                                                                  /* O2 */
            rc = medfilt_v(work, m5, h, w, 5, v->sepmed);
            if (rc) goto done;
#pragma omp parallel for schedule(static)
            for (size_t p = 0; p < P; ++p) {
                float m = m5[p] > 1e-4f ? m5[p] : 1e-4f;
                float gm = gain * m;
                float var = gm + rn2;
                N[p] = sqrtf(var) / gain;
            }
        }
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {                                          /* O3 */
            float twoN = 2.0f * N[p];
            S[p] = Lp[p] / twoN;
        }
        rc = medfilt_v(S, mS, h, w, 5, v->sepmed);
        if (rc) goto done;
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) Sp[p] = S[p] - mS[p];
        rc = medfilt_v(work, m3, h, w, 3, v->sepmed);                             /* O4 */
        if (rc) goto done;
        rc = medfilt_v(m3, m7, h, w, 7, v->sepmed);
        if (rc) goto done;
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {
            float f = m3[p] - m7[p];
            if (v->fsmode == 1) f = f / N[p];                                     /* R22: in units of the noise */
            F[p] = f > 0.01f ? f : 0.01f;
        }
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) {                                          /* O5, R12, R23, R25 */
            int ok = (work[p] < satlevel) && !nok[p];
            G1[p] = (uint8_t)(ok && (Sp[p] > sigclip));
            G2[p] = (uint8_t)(ok && (Sp[p] > siglow));
            float ratio = (v->fsmode == 1 ? Sp[p] : Lp[p]) / F[p];                /* R22: S'/Fn; R7: L+/F */
            M1[p] = (uint8_t)(G1[p] && (ratio > objlim));
        }
        orc_dilate3(M1, D, h, w);                                                 /* O6 */
#pragma omp parallel for schedule(static)
        for (size_t p = 0; p < P; ++p) M2[p] = (uint8_t)(D[p] && G1[p]);
        orc_dilate3(M2, D, h, w);
        int64_t newc = 0;
#pragma omp parallel for schedule(static) reduction(+ : newc)
        for (size_t p = 0; p < P; ++p) {
            M3[p] = (uint8_t)(D[p] && G2[p]);
            if (M3[p] && !C[p]) ++newc;
            C[p] = (uint8_t)(C[p] || M3[p]);
        }
        if (iter_counts) iter_counts[t] = (int32_t)newc;
        orc_masked_median_bpm(img, C, v->bpm, work, h, w);                        /* O7, R23 */

        if (dbg && dbg->iter == t) {
            COPY_IF(dbg->Lp, Lp, P * 4); COPY_IF(dbg->N, N, P * 4); COPY_IF(dbg->S, S, P * 4);
            COPY_IF(dbg->Sp, Sp, P * 4); COPY_IF(dbg->m3, m3, P * 4); COPY_IF(dbg->F, F, P * 4);
            COPY_IF(dbg->G1, G1, P); COPY_IF(dbg->G2, G2, P); COPY_IF(dbg->M1, M1, P);
            COPY_IF(dbg->M2, M2, P); COPY_IF(dbg->M3, M3, P); COPY_IF(dbg->C, C, P);
        }
    }
done:
    free(Lp); free(m5); free(N); free(S); free(mS); free(Sp); free(m3); free(m7); free(F);
    free(G1); free(G2); free(M1); free(D); free(M2); free(M3); free(nok);
    return rc;
}
