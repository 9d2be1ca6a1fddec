/*
 * arkcos_spectral.h - N2 of SURVEY.md §8(f): the phi-spectral ring-pair path.  The SAME operator as arkcos_convolve
 * (include/arkcos.h), evaluated per ring pair in the Fourier domain of phi: every ring pair (i, j) is a circular
 * correlation in phi, so  OUT_i[m] = sum_j What_ij[m] X_j[m]  with X_j the real FFT of input ring j and What_ij the
 * (real) spectrum of the symmetric weight vector w_ij[d] = A_j K(gamma_ij(d)) of step S2.  Its work per output ring
 * is (2R+1) n_phi/2 multiply-adds whatever the window widths, i.e. LINEAR in theta_cut - the shape of the paper's
 * fitted GPU cost t = 0.0232 s x theta_cut + 2.428 s (Eq. 2.3), where the direct banded
 * sum that north_star prescribes is quadratic.  It is a cross-check of the direct path and the cost model the
 * split optimiser (include/arkcos_split.h) can consume; the product's hot path remains arkcos_convolve.
 * Arithmetic: What in FP64 at plan time, rounded once to FP32; FFTs and the mode products in FP32.
 */
#ifndef ARKCOS_SPECTRAL_H_
#define ARKCOS_SPECTRAL_H_

#include "arkcos.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Flag of arkcos_plan_create_ex: also build the weight spectra ((n_theta+1)/2 x (2R+1) x (n_phi/2+1) floats of
 * device memory).  n_phi must be a power of two, 16 <= n_phi <= 16384, else ARKCOS_EUNSUPPORTED. */
#define ARKCOS_PLAN_SPECTRAL 16u

/* Bytes of DEVICE workspace arkcos_convolve_spectral needs for n_maps maps (the ring spectra X_j). */
arkcos_status arkcos_spectral_workspace_bytes(const arkcos_plan *plan, int n_maps, unsigned long long *bytes);

/*
 * arkcos_convolve_spectral - as arkcos_convolve_batch (same d_in / d_out rules, asynchronous on `stream`, no
 * allocation, no host synchronisation), through the spectral path.
 *   d_work, work_bytes  DEVICE scratch owned by the CALLER for the duration of the call on `stream`, 16-byte
 *                       aligned, at least arkcos_spectral_workspace_bytes(plan, n_maps); the plan itself stays
 *                       immutable, so concurrent calls on several streams need one workspace each
 * Errors: as arkcos_convolve_batch; EUNSUPPORTED if the plan was created without ARKCOS_PLAN_SPECTRAL; EINVAL for a
 * NULL / misaligned / too small workspace.
 */
arkcos_status arkcos_convolve_spectral(const arkcos_plan *plan, const float *d_in, float *d_out, int n_maps,
                                       void *d_work, unsigned long long work_bytes, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* ARKCOS_SPECTRAL_H_ */
