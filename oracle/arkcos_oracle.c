/*
 * arkcos_oracle.c - TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, FP64 CPU brute-force evaluation of the real-space spherical convolution that the
 * CUDA library (include/arkcos.h) computes.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code, header,
 * table or helper with the CUDA path (paper_1211_3556_b200/csrc/).
 *
 * What it computes ("convolving a ... map with a radial kernel"; PAPER.md:L44 the
 * "real-space portion ... truncated"; BASELINE.json north_star "plain, slow FP64 CPU brute-force
 * direct sum over all input pixels within theta_cut"; SURVEY.md §8 "Definition of the result"):
 *
 *     out[p] = sum over input pixels q with gamma(p,q) <= theta_cut of  K(gamma(p,q)) * A_q * in[q]
 *
 * on the ECP grid of BASELINE.json configs[0]: ring centres theta_i = (i + 1/2) pi / N_theta,
 * phi_k = 2 pi k / N_phi; A_q is the exact area of a ring-j pixel,
 * A_j = dphi * (cos(j dtheta) - cos((j+1) dtheta))  (north_star: "folds in the exact ring pixel area");
 * K is the linear interpolant of the radial table T[m] = K(m * theta_cut / (n_table - 1))
 * ("interpolate this kernel").
 *
 * The oracle is the definition written out, in the order stated there:
 *   1. pixel-centre unit vectors n = (sin t cos p, sin t sin p, cos t);
 *   2. angle from the chord and co-chord: gamma = 2 atan2(|n_p - n_q|, |n_p + n_q|)  (equal to
 *      SURVEY's 2 asin(|n_p - n_q|/2) but also well-conditioned near gamma = pi, which the
 *      theta_cut = pi all-pairs test exercises; reading R2);
 *   3. support test gamma <= theta_cut (inclusive);
 *   4. K(gamma): t = gamma / theta_cut * (n-1), m = min(floor t, n-2), f = t - m,
 *      K = (1-f) T[m] + f T[m+1];
 *   5. out[p] = sum_q K * A_j(q) * in[q], accumulated in long double;
 *   6. level 0 visits ALL q; level 1 visits only rings |i-j| <= ceil(theta_cut/dtheta) + 1 and, per
 *      ring, a phi window padded by 2 pixels each side (or the whole ring), still applying step 3 to
 *      every visited pair and reusing no weight between output pixels.
 *
 * Two-zone ("biased") table, PAPER.md:L88 (§3): "we place half the available interpolation nodes within
 * the first 1/16th of the available support".  oracle_convolve_biased takes the node index m_split that
 * sits exactly at theta_split: nodes 0..m_split are uniform on [0, theta_split], nodes m_split..n-1 are
 * uniform on [theta_split, theta_cut]; K stays the linear interpolant between neighbouring nodes.  Step 4
 * then reads  t = gamma/theta_split*m_split  (gamma < theta_split)  or
 * t = m_split + (gamma-theta_split)/(theta_cut-theta_split)*(n-1-m_split).  m_split = 0 is the uniform
 * table.  Pinned by tests/test_biased_table.py against numpy.interp over the explicit node positions.
 *
 * Parity pins (tests/test_oracle_*.py, `-m "not gpu"`): delta-input point values against an
 * independent atan2 angle formula, total area = 4 pi, phi-shift and N/S-mirror equivariance,
 * area-weighted self-adjointness, constant-map and Y_lm closed forms (b_l of the piecewise-linear
 * table), level 1 == level 0, and an independent numpy all-pairs sum on tiny maps.  The paper prints
 * no convolution output values, so beyond those pins parity is "unpinned by the paper".
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL 1
#define ORACLE_ENOMEM 2

typedef struct {
    int n_theta, n_phi, n_table;
    double theta_cut, dtheta, dphi;
    int m_split;             /* 0: uniform table */
    double theta_split;
    double *sin_t, *cos_t;   /* per ring  */
    double *cos_p, *sin_p;   /* per phi   */
    double *area;            /* per ring  */
    const double *table;
} grid_t;

static void grid_free(grid_t *g) {
    free(g->sin_t); free(g->cos_t); free(g->cos_p); free(g->sin_p); free(g->area);
}

static int grid_init(grid_t *g, int n_theta, int n_phi, const double *table, int n_table, double theta_cut) {
    memset(g, 0, sizeof(*g));
    if (n_theta < 1 || n_phi < 1 || n_table < 2 || !table || !(theta_cut > 0.0) || theta_cut > M_PI + 1e-15)
        return ORACLE_EINVAL;
    g->n_theta = n_theta; g->n_phi = n_phi; g->n_table = n_table; g->theta_cut = theta_cut;
    g->dtheta = M_PI / n_theta; g->dphi = 2.0 * M_PI / n_phi; g->table = table;
    g->sin_t = malloc(sizeof(double) * n_theta); g->cos_t = malloc(sizeof(double) * n_theta);
    g->area = malloc(sizeof(double) * n_theta);
    g->cos_p = malloc(sizeof(double) * n_phi); g->sin_p = malloc(sizeof(double) * n_phi);
    if (!g->sin_t || !g->cos_t || !g->area || !g->cos_p || !g->sin_p) { grid_free(g); return ORACLE_ENOMEM; }
    for (int i = 0; i < n_theta; i++) {
        double t = (i + 0.5) * g->dtheta;                 /* ring centre, configs[0] */
        g->sin_t[i] = sin(t); g->cos_t[i] = cos(t);
        g->area[i] = g->dphi * (cos(i * g->dtheta) - cos((i + 1) * g->dtheta));   /* exact ring pixel area */
    }
    for (int k = 0; k < n_phi; k++) {
        double p = k * g->dphi;
        g->cos_p[k] = cos(p); g->sin_p[k] = sin(p);
    }
    return ORACLE_OK;
}

/* steps 1-4 for one (output, input) pixel pair; returns 1 and the kernel value if inside the support */
static inline int pair_kernel(const grid_t *g, int i, int k, int j, int kk, double *kval) {
    double dx = g->sin_t[i] * g->cos_p[k] - g->sin_t[j] * g->cos_p[kk];
    double dy = g->sin_t[i] * g->sin_p[k] - g->sin_t[j] * g->sin_p[kk];
    double dz = g->cos_t[i] - g->cos_t[j];
    double sx = g->sin_t[i] * g->cos_p[k] + g->sin_t[j] * g->cos_p[kk];
    double sy = g->sin_t[i] * g->sin_p[k] + g->sin_t[j] * g->sin_p[kk];
    double sz = g->cos_t[i] + g->cos_t[j];
    double chord = sqrt(dx * dx + dy * dy + dz * dz);      /* |n_p - n_q| = 2 sin(gamma/2) */
    double cochord = sqrt(sx * sx + sy * sy + sz * sz);    /* |n_p + n_q| = 2 cos(gamma/2) */
    double gamma = 2.0 * atan2(chord, cochord);
    if (!(gamma <= g->theta_cut)) return 0;                /* support, inclusive */
    double t;
    if (g->m_split <= 0) t = gamma / g->theta_cut * (double)(g->n_table - 1);
    else if (gamma < g->theta_split) t = gamma / g->theta_split * (double)g->m_split;
    else t = (double)g->m_split + (gamma - g->theta_split) / (g->theta_cut - g->theta_split) * (double)(g->n_table - 1 - g->m_split);
    int m = (int)floor(t); if (m > g->n_table - 2) m = g->n_table - 2; if (m < 0) m = 0;
    double f = t - (double)m;
    *kval = (1.0 - f) * g->table[m] + f * g->table[m + 1];
    return 1;
}

/* level 0: every input pixel */
static long double pixel_level0(const grid_t *g, const double *in, int i, int k, unsigned long long *npairs) {
    long double acc = 0.0L; unsigned long long n = 0;
    for (int j = 0; j < g->n_theta; j++)
        for (int kk = 0; kk < g->n_phi; kk++) {
            double kv;
            if (pair_kernel(g, i, k, j, kk, &kv)) {
                acc += (long double)(kv * g->area[j]) * (long double)in[(size_t)j * g->n_phi + kk];
                n++;
            }
        }
    *npairs += n;
    return acc;
}

/* level 1: conservative ring band and phi window, every visited pair still tested */
static long double pixel_level1(const grid_t *g, const double *in, int i, int k, unsigned long long *npairs) {
    long double acc = 0.0L; unsigned long long n = 0;
    int band = (int)ceil(g->theta_cut / g->dtheta) + 1;
    double cos_cut = cos(g->theta_cut);
    for (int j = i - band; j <= i + band; j++) {
        if (j < 0 || j >= g->n_theta) continue;           /* no wrap over the pole */
        /* gamma <= theta_cut  <=>  cos(dphi) >= (cos theta_cut - cos t_i cos t_j) / (sin t_i sin t_j) */
        double c = (cos_cut - g->cos_t[i] * g->cos_t[j]) / (g->sin_t[i] * g->sin_t[j]);
        int half;                                          /* visited window: k-half .. k+half */
        if (c <= -1.0 + 1e-12) half = g->n_phi;            /* whole ring */
        else if (c >= 1.0) half = 2;                        /* nothing expected: padding only */
        else half = (int)ceil(acos(c) / g->dphi) + 2;
        if (2 * half + 1 >= g->n_phi) {
            for (int kk = 0; kk < g->n_phi; kk++) {
                double kv;
                if (pair_kernel(g, i, k, j, kk, &kv)) {
                    acc += (long double)(kv * g->area[j]) * (long double)in[(size_t)j * g->n_phi + kk];
                    n++;
                }
            }
        } else {
            for (int d = -half; d <= half; d++) {
                int kk = ((k + d) % g->n_phi + g->n_phi) % g->n_phi;
                double kv;
                if (pair_kernel(g, i, k, j, kk, &kv)) {
                    acc += (long double)(kv * g->area[j]) * (long double)in[(size_t)j * g->n_phi + kk];
                    n++;
                }
            }
        }
    }
    *npairs += n;
    return acc;
}

/*
 * Evaluate the convolution at `n_pix` output pixels.
 *   level      0 = all pairs, 1 = windowed
 *   in         [n_theta][n_phi] FP64 (an FP32 map is promoted exactly by the caller)
 *   pix        flat output pixel indices i*n_phi+k, or NULL for all pixels 0..n_theta*n_phi-1
 *   out        [n_pix] FP64 results, in the order of `pix`
 *   n_pairs    (optional) number of in-support (output,input) pairs = kernel-pixel evaluations
 *   n_threads  <= 0: OpenMP default
 * Returns ORACLE_OK / ORACLE_EINVAL / ORACLE_ENOMEM.
 */
int oracle_convolve_biased(int level, int n_theta, int n_phi, const double *table, int n_table, double theta_cut,
                           int m_split, double theta_split,
                           const double *in, const long long *pix, long long n_pix, double *out,
                           unsigned long long *n_pairs, int n_threads) {
    grid_t g;
    if (!in || !out || (level != 0 && level != 1) || n_pix < 0) return ORACLE_EINVAL;
    if (m_split < 0 || (m_split > 0 && (m_split > n_table - 2 || !(theta_split > 0.0) || !(theta_split < theta_cut))))
        return ORACLE_EINVAL;
    int rc = grid_init(&g, n_theta, n_phi, table, n_table, theta_cut);
    if (rc != ORACLE_OK) return rc;
    g.m_split = m_split; g.theta_split = theta_split;
    long long total = (long long)n_theta * n_phi;
    if (!pix) n_pix = total;
    unsigned long long pairs = 0;
    int bad = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : pairs) reduction(| : bad)
    for (long long a = 0; a < n_pix; a++) {
        long long p = pix ? pix[a] : a;
        if (p < 0 || p >= total) { bad |= 1; out[a] = NAN; continue; }
        int i = (int)(p / n_phi), k = (int)(p % n_phi);
        unsigned long long n = 0;
        long double v = level == 0 ? pixel_level0(&g, in, i, k, &n) : pixel_level1(&g, in, i, k, &n);
        out[a] = (double)v;
        pairs += n;
    }
    if (n_pairs) *n_pairs = pairs;
    grid_free(&g);
    return bad ? ORACLE_EINVAL : ORACLE_OK;
}

/* uniform table: the two-zone entry point with no inner zone */
int oracle_convolve(int level, int n_theta, int n_phi, const double *table, int n_table, double theta_cut,
                    const double *in, const long long *pix, long long n_pix, double *out,
                    unsigned long long *n_pairs, int n_threads) {
    return oracle_convolve_biased(level, n_theta, n_phi, table, n_table, theta_cut, 0, 0.0, in, pix, n_pix, out, n_pairs, n_threads);
}

/* exact ring pixel areas A_j, for the area pin (sum_j N_phi A_j = 4 pi) and the adjointness pin */
int oracle_ring_area(int n_theta, int n_phi, double *area) {
    if (n_theta < 1 || n_phi < 1 || !area) return ORACLE_EINVAL;
    double dtheta = M_PI / n_theta, dphi = 2.0 * M_PI / n_phi;
    for (int j = 0; j < n_theta; j++) area[j] = dphi * (cos(j * dtheta) - cos((j + 1) * dtheta));
    return ORACLE_OK;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
