/*
 * arkcos.h - C ABI of arkcos-b200: real-space convolution of an ECP-pixelated spherical map with
 * the compact part K(theta <= theta_cut) of a radially symmetric kernel, on one NVIDIA B200.
 *
 * This is the GPU half of the hybrid kernel split of Sutter, Wandelt & Elsner (arXiv:1211.3556):
 * "the real-space portion, which will be applied using a GPU", computed by "the GPU
 * code ARKCoS" with a kernel that is "interpolate[d]" from nodes
 * in single precision.  The operation, per BASELINE.json north_star / SURVEY.md §8:
 *
 *     out[i,k] = sum_j sum_k'  [gamma <= theta_cut] * K(gamma) * A_j * in[j,k']
 *     cos(gamma) = cos(t_i) cos(t_j) + sin(t_i) sin(t_j) cos((k'-k) dphi)
 *
 * on the grid  t_i = (i + 1/2) pi / n_theta,  phi_k = 2 pi k / n_phi,  with the exact ring pixel
 * area A_j = dphi (cos(j dtheta) - cos((j+1) dtheta)) and K the LINEAR interpolant of `k_table`.
 *
 * Conventions
 *   - every function returns an arkcos_status and never throws, aborts or prints;
 *   - maps are row-major [n_theta][n_phi], FP32, phi fastest; "DEVICE" = CUDA device memory of the
 *     device that was current at plan creation, "HOST" = ordinary host memory;
 *   - pointers passed in stay owned by the caller; nothing is retained after the call returns
 *     except by arkcos_plan_create (which COPIES the table).
 *   - no CPU fallback exists: without a usable CUDA device every compute entry point fails with
 *     ARKCOS_ECUDA.
 */
#ifndef ARKCOS_H_
#define ARKCOS_H_

#ifdef __cplusplus
extern "C" {
#endif

#define ARKCOS_VERSION_MAJOR 0
#define ARKCOS_VERSION_MINOR 1

typedef struct arkcos_plan arkcos_plan; /* opaque; immutable after creation */

typedef enum {
    ARKCOS_OK = 0,
    ARKCOS_EINVAL = 1,       /* bad argument (range, NULL, alignment, aliasing, non-finite table) */
    ARKCOS_ENOMEM = 2,       /* host or device allocation failed                                  */
    ARKCOS_ECUDA = 3,        /* a CUDA runtime call failed (no device, launch error, ...)         */
    ARKCOS_EUNSUPPORTED = 4, /* valid request this build cannot serve (e.g. n_phi % 4 != 0)       */
    ARKCOS_EINTERNAL = 5     /* the ring-pair schedule failed its own validation (a bug in this   */
                             /* library; nothing was uploaded or launched)                        */
} arkcos_status;

/* flags of arkcos_plan_create_ex */
#define ARKCOS_PLAN_DEFAULT 0u
/* Build only the host-side ring-pair schedule (step S1): no CUDA call is made, no device is needed.
 * Introspection calls work; compute calls return ARKCOS_EUNSUPPORTED. */
#define ARKCOS_PLAN_HOST_ONLY 1u
/* Run the weight generator (step S2) once, at plan creation, and reuse its output in every
 * arkcos_convolve.  Default is to regenerate the weights on the fly inside each call
 * (north_star (b)); both give bit-identical results. */
#define ARKCOS_PLAN_CACHE_WEIGHTS 2u
/* (bits 4 and 8 are measurement hooks declared in arkcos_measure.h) */

/*
 * arkcos_plan_create - step S1 (ring-pair scheduler, host FP64) and device uploads.
 *   plan           out; set to NULL on failure
 *   n_theta,n_phi  ECP grid (BASELINE.json configs[0]); n_theta >= 1, n_phi >= 4, n_phi % 4 == 0
 *   k_table        HOST, n_table FP64 samples K(theta_m), theta_m = m * theta_cut / (n_table - 1),
 *                  both ends included; copied; must be finite
 *   n_table        >= 2
 *   theta_cut_rad  support radius, 0 < theta_cut <= pi, inclusive (K_real(theta <= theta_cut))
 * The plan owns its device memory on the device current at this call.  Before anything is uploaded the
 * schedule is validated on the host: every global range and shared-memory offset the kernels will form from
 * it is re-derived and bounds-checked (EINTERNAL if not; the kernels themselves carry no bounds checks).
 * All uploads have completed when the call returns, so the plan may be used at once on any stream.
 * Errors: EINVAL, EUNSUPPORTED (n_phi % 4 != 0), ENOMEM, ECUDA, EINTERNAL.
 */
arkcos_status arkcos_plan_create(arkcos_plan **plan, int n_theta, int n_phi, const double *k_table,
                                 int n_table, double theta_cut_rad);
arkcos_status arkcos_plan_create_ex(arkcos_plan **plan, int n_theta, int n_phi, const double *k_table,
                                    int n_table, double theta_cut_rad, unsigned flags);

/*
 * arkcos_plan_create_biased - as arkcos_plan_create_ex, for the paper's two-zone interpolation table
 * (§3: "we place half the available interpolation nodes within the first 1/16th of the
 * available support", because the split kernel oscillates fastest at small angles).
 *   k_table          HOST, n_table samples at the nodes
 *                       theta_m = m * theta_split / m_split                                  (m <= m_split)
 *                       theta_m = theta_split + (m - m_split) * (theta_cut - theta_split) / (n_table - 1 - m_split)
 *                    i.e. node m_split sits exactly at theta_split and the nodes are uniform on either side;
 *                    K is the linear interpolant between neighbouring nodes, as for the uniform table
 *   m_split          1 <= m_split <= n_table - 2   (the paper: m_split = (n_table - 1) / 2)
 *   theta_split_rad  0 < theta_split < theta_cut   (the paper: theta_cut / 16)
 * Everything else (support, ring areas, schedule, kernels) is unchanged: only step S2's table lookup differs.
 * Errors: as arkcos_plan_create_ex, plus EINVAL for an m_split / theta_split outside the ranges above.
 */
arkcos_status arkcos_plan_create_biased(arkcos_plan **plan, int n_theta, int n_phi, const double *k_table,
                                        int n_table, double theta_cut_rad, int m_split, double theta_split_rad,
                                        unsigned flags);

/*
 * arkcos_convolve - the hot path, steps S2 (weight generator) + S3/S3w (convolution kernels).
 *   d_in   DEVICE, [n_theta][n_phi] FP32, 16-byte aligned, read only
 *   d_out  DEVICE, same shape, 16-byte aligned, fully overwritten; must not overlap d_in
 *   stream cudaStream_t cast to void* (NULL = legacy default stream)
 * Asynchronous on `stream`: no allocation, no host synchronisation, no host<->device copy.
 * A plan is immutable and may be used from several streams and host threads at the same time: the only
 * plan-owned memory a call writes is the weight buffer, and step S2 is a pure function of the plan - every
 * call rewrites each weight with the bit-identical value, and each call's own S2 precedes its own S3 on its
 * stream, so concurrent calls never observe a different value (cached plans do not write at all).
 * The current device must be the plan's device.
 * The map must be finite: windows are padded to whole 2- / 4- / 16-tap steps with ZERO weights, so an Inf or NaN
 * input pixel makes the outputs within theta_cut of it - and up to 15 pixels further along its ring - NaN
 * (0 x Inf), where the definition would give NaN only inside theta_cut.  Results are deterministic: one owner per
 * output, fixed summation order (blocks of <= ~1000 taps).
 * Errors: EINVAL (NULL / misaligned / overlapping pointers, wrong current device), EUNSUPPORTED (host-only
 * plan), ECUDA.
 */
arkcos_status arkcos_convolve(const arkcos_plan *plan, const float *d_in, float *d_out, void *stream);

/*
 * arkcos_convolve_batch - n_maps independent maps with one plan (BASELINE.json configs[4]: a batch
 * of 8 maps); the weights are generated once per call and shared by all maps.
 *   d_in, d_out  DEVICE, [n_maps][n_theta][n_phi]; same rules as arkcos_convolve
 */
arkcos_status arkcos_convolve_batch(const arkcos_plan *plan, const float *d_in, float *d_out, int n_maps,
                                    void *stream);

/*
 * arkcos_convolve_host - end to end: HOST map in, HOST map out.
 * Copies h_in to plan-owned device staging, runs arkcos_convolve and copies the result back; returns after
 * the result is in h_out (synchronises `stream`).  Pinned host memory makes the copies asynchronous DMA;
 * pageable memory also works.  The staging (two maps) is allocated by arkcos_plan_reserve_host_io, which this
 * call makes itself if the caller has not; unlike arkcos_convolve it uses plan-owned staging, so one call per
 * plan at a time.
 */
arkcos_status arkcos_plan_reserve_host_io(arkcos_plan *plan);
arkcos_status arkcos_convolve_host(arkcos_plan *plan, const float *h_in, float *h_out, void *stream);

/* Releases the plan and its device memory.  NULL is a no-op. */
arkcos_status arkcos_plan_destroy(arkcos_plan *plan);

const char *arkcos_status_string(arkcos_status s);
/* Text of the last CUDA error seen by the calling thread inside this library ("" if none). */
const char *arkcos_last_cuda_error(void);

/* ---- introspection (the metric's denominators, and test hooks for steps S1 and S2) ------------- */

/*
 * Work of one arkcos_convolve (one map):
 *   pair_evals     in-support (output pixel, input pixel) pairs = kernel-pixel evaluations
 *   weights        distinct (output ring, input ring, dphi) weights inside the support
 *   ring_halfband  R = floor(theta_cut / dtheta)
 * Any out pointer may be NULL.
 */
arkcos_status arkcos_plan_work(const arkcos_plan *plan, unsigned long long *pair_evals,
                               unsigned long long *weights, int *ring_halfband);

typedef struct {
    int n_theta, n_phi, n_table;
    double theta_cut;
    int ring_halfband;                   /* R                                                     */
    unsigned long long pair_evals;       /* useful FMAs per map                                   */
    unsigned long long weights;          /* in-support weights (no symmetry reduction)            */
    unsigned long long fma_slots;        /* FMA lanes the kernels issue per map (>= pair_evals:   */
                                         /*   zero-padded taps, idle tile lanes)                  */
    unsigned long long weight_slots;     /* FP32 weights the generator writes per call            */
    int n_items;                         /* CTAs of the convolution launch (cost-sorted work list) */
    int n_gen_units;                     /* work units of the weight generator                    */
    int kernels_per_convolve;            /* kernel launches inside one arkcos_convolve            */
    int sm_count;                        /* 0 for host-only plans                                 */
    unsigned flags;
    unsigned long long device_bytes;     /* device memory owned by the plan                       */
    unsigned long long fma_slots_wide;   /* part of fma_slots issued by the WIDE work items       */
    int first_narrow_ring;               /* northern rings [first_narrow_ring, ceil(n_theta/2))   */
                                         /*   and their mirrors take the NARROW path              */
} arkcos_plan_info;
arkcos_status arkcos_plan_get_info(const arkcos_plan *plan, arkcos_plan_info *info);

/*
 * Step S1 test hook: the phi window of ring pair (output ring i, input ring j).
 *   *half_width = -1  no input pixel of ring j is inside theta_cut of ring i
 *               = D   taps d = -D..D are inside (0 <= D < n_phi/2)
 *               = n_phi  every pixel of ring j is inside (each taken exactly once)
 */
arkcos_status arkcos_plan_window(const arkcos_plan *plan, int i, int j, int *half_width);

/*
 * Step S2 test hook: run the weight generator and copy the FP32 weights w_ij[d] = A_j K(gamma_ij(d)),
 * d = 0..min(D, n_phi/2), of ring pair (i, j) to HOST h_w (capacity `cap` floats); *n = count written.
 * Synchronises the device.  EUNSUPPORTED on host-only plans.
 */
arkcos_status arkcos_plan_pair_weights(const arkcos_plan *plan, int i, int j, float *h_w, int cap, int *n);

#ifdef __cplusplus
}
#endif
#endif /* ARKCOS_H_ */
