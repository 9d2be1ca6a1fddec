/*
 * arkcos_split.h - the arithmetic of the paper's kernel split that the paper specifies (host, FP64).
 *
 * Sutter, Wandelt & Elsner, arXiv:1211.3556, §2.  SURVEY.md §8(f) N4.  These calls serve
 * the layer ABOVE the hot path (the split optimiser "scytale"): they tell a caller which theta_cut to hand to
 * arkcos_plan_create.  They run on the host, need no device and never touch the convolution kernels.
 * NOT provided, because the paper does not specify it: the fit that produces the truncated real-space kernel
 * from K_l ("our computational approach damps oscillations in l-space").  The caller supplies the
 * real-space kernel as the same radial table arkcos_plan_create takes.
 *
 * All arrays are HOST memory owned by the caller; nothing is retained.  Every call returns an arkcos_status
 * (include/arkcos.h): ARKCOS_EINVAL for NULL / out-of-range / non-finite arguments, ARKCOS_ENOMEM, else ARKCOS_OK.
 */
#ifndef ARKCOS_SPLIT_H_
#define ARKCOS_SPLIT_H_

#include "arkcos.h"

#ifdef __cplusplus
extern "C" {
#endif

/*
 * arkcos_table_legendre - the Legendre transform P_{l theta} K_theta of Eq. 2.1 for the
 * kernel exactly as the library applies it: the piecewise-linear interpolant of the radial table, zero beyond
 * theta_cut,
 *       b_l = 2 pi * integral_0^theta_cut K(theta) P_l(cos theta) sin(theta) dtheta,     l = 0 .. l_max.
 * Convolving Y_lm with the kernel multiplies it by b_l (spherical convolution theorem).
 *   k_table, n_table, theta_cut_rad       as arkcos_plan_create
 *   m_split, theta_split_rad              two-zone table as arkcos_plan_create_biased; m_split = 0: uniform
 *   l_max >= 0;  b_l  out, [l_max + 1]
 * Integrated cell by cell with Gauss-Legendre quadrature whose order follows l_max * cell width (the
 * integrand is a polynomial in cos/sin times a linear function on every cell); P_l by the three-term recurrence.
 */
arkcos_status arkcos_table_legendre(const double *k_table, int n_table, double theta_cut_rad, int m_split,
                                    double theta_split_rad, int l_max, double *b_l);

/*
 * arkcos_split_error - Eq. 2.1 and Eq. 2.2.
 *   k_l      [l_max+1] the full kernel K_l
 *   b_l      [l_max+1] Legendre transform of the truncated real-space kernel (arkcos_table_legendre)
 *   l_cut    truncation of the l-space part, -1 (no l-space part) .. l_max
 *   compensate  0: Khat_l = K_l for l <= l_cut, else 0 (plain truncation).
 *               1: Khat_l = K_l - b_l for l <= l_cut, else 0: the l-space part absorbs what the real-space part
 *                  does at low l ("percent-level adjustments in the l-space kernel"), so that
 *                  Ktilde_l = K_l exactly up to l_cut ("essentially zero error").  DESIGN.md R16.
 *   alpha    the empirical inflation of Eq. 2.2 (the paper: 5)
 *   sigma    out: alpha * sqrt( sum_l (2l+1)(Ktilde_l - K_l)^2 / sum_l (2l+1) K_l^2 ), sums over 0..l_max;
 *            sigma_rms^2 of Eq. 2.2 is read as (1/4pi) sum (2l+1)(Ktilde_l - K_l)^2 (R17)
 *   khat_l, ktilde_l  optional outs [l_max+1] (NULL to skip): Khat_l and Ktilde_l = Khat_l + b_l (Eq. 2.1)
 */
arkcos_status arkcos_split_error(const double *k_l, const double *b_l, int l_max, int l_cut, int compensate,
                                 double alpha, double *sigma, double *khat_l, double *ktilde_l);

/* Cost models of Eq. 2.3 / Eq. 2.4, generalised so that a measured curve can be used:
 *   t_gpu(theta_cut) = gpu_a2 * theta^2 + gpu_a1 * theta + gpu_c   [s], theta in ARCMINUTES
 *                      (the paper, GTX 480: a2 = 0, a1 = 0.0232, c = 2.428; this library's direct sum on
 *                       B200 is quadratic: take a2, c from `bench.py --sweep`)
 *   t_cpu(l_cut)     = cpu_full_s * l_cut^2 * l_max / cpu_l_ref^3    (the paper: 160 s, 4096)              */
typedef struct {
    double gpu_a2, gpu_a1, gpu_c;
    double cpu_full_s, cpu_l_ref;
} arkcos_cost_model;

/*
 * arkcos_split_search - the scan of PAPER.md:L74: among the candidate real-space truncations, keep the
 * (l_cut, theta_cut) pairs whose estimated error is within `bound`, and return the one that minimises the
 * time of the two halves running in parallel, max(t_gpu, t_cpu) - i.e. the pair closest to t_gpu = t_cpu.
 *   n_cand, theta_cut_arcmin[n_cand], b_l_cand[n_cand][l_max+1]   the candidates and their Legendre transforms
 *   best_cand / best_l_cut / best_time_s / best_sigma             outs; best_cand = -1 if no pair meets the bound
 *   For every candidate the smallest admissible l_cut is taken (t_cpu grows with l_cut).
 */
arkcos_status arkcos_split_search(const double *k_l, int l_max, int n_cand, const double *theta_cut_arcmin,
                                  const double *b_l_cand, int compensate, double alpha, double bound,
                                  const arkcos_cost_model *cost, int *best_cand, int *best_l_cut,
                                  double *best_time_s, double *best_sigma);

#ifdef __cplusplus
}
#endif
#endif /* ARKCOS_SPLIT_H_ */
