// arkcos_spectral.cuh - N2, the phi-spectral ring-pair path: the same operator as S3,
// evaluated per ring pair in the Fourier domain of phi.  Product code; shares nothing with oracle/.
//
// Each ring pair (i, j) is a circular correlation in phi with the symmetric weight vector w_ij[d] (step S2),
//     out_i[k] = sum_j sum_d w_ij[d] in_j[(k + d) mod n],
// so with the real DFT along phi (X_j[m] = sum_k in_j[k] e^{-2 pi i m k / n}) it is one real multiply per mode:
//     OUT_i[m] = sum_j What_ij[m] X_j[m],      What_ij[m] = w_ij[0] + 2 sum_{d >= 1} w_ij[d] cos(2 pi m d / n)
// (whole-ring windows: the single tap d = -n/2 enters once).  Work per output ring is (2R+1) n/2 complex-real
// multiply-adds whatever the window widths are: LINEAR in theta_cut, the shape of the paper's fitted GPU cost
// t = 0.0232 s * theta_cut + 2.428 s (Eq. 2.3), where the direct sum is quadratic.  The price is
// FP32 FFT rounding (forward and inverse) on top of the FP32 accumulation; DESIGN.md gives the measured error.
//
//   k_spectral_weights   plan time, FP64: What_ij[m] * (2/n) for every northern ring pair, rounded once to FP32
//   k_rfft_rings         per call: X_j = real FFT of every input ring (half-length complex Stockham FFT in
//                        shared memory + the real-input split)
//   k_spectral_apply     per call, one CTA per output ring: OUT_i[m] = sum_j What_ij[m] X_j[m], inverse split,
//                        inverse half-length FFT, store
// n_phi must be a power of two, 16 <= n_phi <= kSpecMaxPhi.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "arkcos_internal.h"

namespace arkcos {

constexpr int kSpecThreads = 256;
constexpr int kSpecMaxPhi = 16384;       // two half-length complex buffers + twiddles = 10 n bytes of shared memory

// One (northern output ring, input ring) pair of the spectral path: the geometry step S2 needs (as GenUnit).
struct SpecPair {
    double a;         // sin^2((t_i - t_j)/2)
    double b;         // sin t_i sin t_j
    double area;      // A_j
    int32_t half;     // D, n_phi = whole ring, -1 = empty
    int32_t pad_;
};

struct SpecWeightParams {
    const SpecPair* pairs;   // [n_north][2R+1]
    const double* s2;        // [n_phi/2+1] sin^2(d dphi / 2)
    const double* table;     // [n_table]
    const double* costab;    // [n_phi] cos(2 pi k / n_phi), FP64
    float* wspec;            // [n_north][2R+1][n_phi/2+1]
    int n_pairs, n_phi, n_table;
    double t_scale, theta_split, t_scale2;
    int m_split;
};

// K(gamma) * A_j for tap |d| = ad of a pair: the arithmetic of step S2 (k_generate_weights), FP64, unrounded
__device__ __forceinline__ double spec_weight(const SpecWeightParams& p, const SpecPair& g, const int ad) {
    double h = fma(g.b, p.s2[ad], g.a);
    h = fmin(h, 1.0);
    const double gam = 2.0 * asin(sqrt(h));
    double t = gam * p.t_scale;
    if (p.m_split > 0 && gam >= p.theta_split) t = (double)p.m_split + (gam - p.theta_split) * p.t_scale2;
    int m = (int)t;
    m = min(m, p.n_table - 2);
    const double f = t - (double)m;
    return g.area * ((1.0 - f) * p.table[m] + f * p.table[m + 1]);
}

__global__ void __launch_bounds__(kSpecThreads) k_spectral_weights(const SpecWeightParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ double s_w[];
#else
    double* s_w = reinterpret_cast<double*>(emu::g_smem);
#endif
    const int n = p.n_phi, h = n >> 1;
    for (int pair = blockIdx.x; pair < p.n_pairs; pair += gridDim.x) {
        const SpecPair g = p.pairs[pair];
        float* dst = p.wspec + (size_t)pair * (h + 1);
        if (g.half < 0) {
            for (int m = threadIdx.x; m <= h; m += kSpecThreads) dst[m] = 0.0f;
            continue;
        }
        const bool whole = g.half == n;
        const int dm = whole ? h : g.half;                     // taps |d| = 0 .. dm are inside the support
        __syncthreads();                                        // the previous pair's weights are no longer read
        for (int d = threadIdx.x; d <= dm; d += kSpecThreads) s_w[d] = spec_weight(p, g, d);
        __syncthreads();
        const double scale = 2.0 / (double)n;                   // the inverse half-length FFT is unnormalised: fold 1/(n/2) in
        for (int m = threadIdx.x; m <= h; m += kSpecThreads) {
            double acc = s_w[0];
            int idx = 0;
            const int dlast = whole ? h - 1 : dm;               // taps that occur as +d and -d
            for (int d = 1; d <= dlast; d++) {
                idx = (idx + m) & (n - 1);
                acc = fma(2.0 * s_w[d], p.costab[idx], acc);
            }
            if (whole) acc = fma(s_w[h], (m & 1) ? -1.0 : 1.0, acc);   // d = -n/2 only: cos(pi m)
            dst[m] = (float)(acc * scale);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Complex FFT of length h (a power of two) in shared memory: Stockham autosort, radix 2, ping-pong between x and
// y; tw[k] = exp(-2 pi i k / h), k < h/2 (conjugated for the inverse).  Returns the buffer that holds the result
// in natural order.  All threads of the CTA must call it.
// ------------------------------------------------------------------------------------------------
template <bool INVERSE>
__device__ __forceinline__ float2* fft_pow2(float2* x, float2* y, const float2* tw, const int h) {
    int ncur = h, s = 1;
    while (ncur > 1) {
        const int m = ncur >> 1;
        int sh = 0;
        while ((1 << sh) < s) sh++;
        for (int t = threadIdx.x; t < (h >> 1); t += kSpecThreads) {
            const int pp = t >> sh, q = t & (s - 1);
            const float2 a = x[q + s * pp], b = x[q + s * (pp + m)];
            float2 w = tw[pp * s];
            if (INVERSE) w.y = -w.y;
            const float dx = a.x - b.x, dy = a.y - b.y;
            y[q + s * (2 * pp)] = make_float2(a.x + b.x, a.y + b.y);
            y[q + s * (2 * pp + 1)] = make_float2(dx * w.x - dy * w.y, dx * w.y + dy * w.x);
        }
        __syncthreads();
        float2* t2 = x; x = y; y = t2;
        ncur = m; s <<= 1;
    }
    return x;
}

struct SpecParams {
    const float* in;         // [n_maps][n_theta][n_phi]
    float* out;
    float2* xspec;           // workspace [n_maps][n_theta][n_phi/2+1]
    const float* wspec;      // [n_north][2R+1][n_phi/2+1]
    const PairDesc* pairs;   // [n_north][2R+1] (half < 0: empty pair)
    const float2* tw_h;      // [n_phi/4] exp(-2 pi i k / (n_phi/2))
    const float2* tw_n;      // [n_phi/2+1] exp(-2 pi i m / n_phi)
    int n_theta, n_phi, R;
};

// X_j[m], m = 0 .. n/2, of every input ring.  grid (n_theta, n_maps).
__global__ void __launch_bounds__(kSpecThreads) k_rfft_rings(const SpecParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ float2 s_f[];
#else
    float2* s_f = reinterpret_cast<float2*>(emu::g_smem);
#endif
    const int n = p.n_phi, h = n >> 1;
    float2* bx = s_f; float2* by = s_f + h; float2* tw = s_f + 2 * h;            // [h], [h], [h/2]
    const size_t ring = (size_t)blockIdx.y * p.n_theta + blockIdx.x;
    const float2* src = reinterpret_cast<const float2*>(p.in + ring * n);        // z[k] = in[2k] + i in[2k+1]
    for (int k = threadIdx.x; k < h; k += kSpecThreads) bx[k] = src[k];
    for (int k = threadIdx.x; k < (h >> 1); k += kSpecThreads) tw[k] = p.tw_h[k];
    __syncthreads();
    const float2* z = fft_pow2<false>(bx, by, tw, h);
    float2* dst = p.xspec + ring * (h + 1);
    for (int m = threadIdx.x; m <= h; m += kSpecThreads) {
        const float2 zm = z[m & (h - 1)], zc = z[(h - m) & (h - 1)];             // Z[m], Z[h-m] (indices mod h)
        const float ex = 0.5f * (zm.x + zc.x), ey = 0.5f * (zm.y - zc.y);        // (Z[m] + conj Z[h-m]) / 2
        const float ox = 0.5f * (zm.x - zc.x), oy = 0.5f * (zm.y + zc.y);        // (Z[m] - conj Z[h-m]) / 2
        const float2 w = p.tw_n[m];                                              // e^{-2 pi i m / n}
        // X = E - i w O
        const float tx = w.x * ox - w.y * oy, ty = w.x * oy + w.y * ox;          // w O
        dst[m] = make_float2(ex + ty, ey - tx);
    }
}

// out_i = inverse real FFT of sum_j What_ij X_j.  grid (n_theta, n_maps).
__global__ void __launch_bounds__(kSpecThreads) k_spectral_apply(const SpecParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ float2 s_f[];
#else
    float2* s_f = reinterpret_cast<float2*>(emu::g_smem);
#endif
    const int n = p.n_phi, h = n >> 1, W = 2 * p.R + 1;
    float2* bx = s_f; float2* by = s_f + h; float2* tw = s_f + 2 * h + 1;        // [h], [h+1] (holds Y first), [h/2]
    const int i = blockIdx.x;
    const bool mirrored = 2 * i >= p.n_theta;
    const int i_n = mirrored ? p.n_theta - 1 - i : i;
    const float2* xs = p.xspec + (size_t)blockIdx.y * p.n_theta * (h + 1);
    for (int k = threadIdx.x; k < (h >> 1); k += kSpecThreads) tw[k] = p.tw_h[k];
    // Y[m] = sum_r What[i_n][r][m] X_{j(r)}[m]
    for (int m = threadIdx.x; m <= h; m += kSpecThreads) {
        float yx = 0.f, yy = 0.f;
        for (int r = 0; r < W; r++) {
            if (p.pairs[(size_t)i_n * W + r].half < 0) continue;
            const int j = mirrored ? i - (r - p.R) : i + (r - p.R);
            const float wv = p.wspec[((size_t)i_n * W + r) * (h + 1) + m];
            const float2 x = xs[(size_t)j * (h + 1) + m];
            yx = fmaf(wv, x.x, yx); yy = fmaf(wv, x.y, yy);
        }
        by[m] = make_float2(yx, yy);
    }
    __syncthreads();
    // inverse split: Z'[k] = (Y[k] + conj Y[h-k]) / 2 + i e^{+2 pi i k / n} (Y[k] - conj Y[h-k]) / 2,  k < h
    for (int k = threadIdx.x; k < h; k += kSpecThreads) {
        const float2 yk = by[k], yc = by[h - k];
        const float ex = 0.5f * (yk.x + yc.x), ey = 0.5f * (yk.y - yc.y);
        const float ox = 0.5f * (yk.x - yc.x), oy = 0.5f * (yk.y + yc.y);
        const float2 w = p.tw_n[k];                                              // conj -> e^{+2 pi i k / n}
        const float tx = w.x * ox + w.y * oy, ty = w.x * oy - w.y * ox;          // conj(w) O
        bx[k] = make_float2(ex - ty, ey + tx);                                   // E + i conj(w) O
    }
    __syncthreads();
    const float2* z = fft_pow2<true>(bx, by, tw, h);                             // unnormalised; 2/n is folded into What
    float2* dst = reinterpret_cast<float2*>(p.out + ((size_t)blockIdx.y * p.n_theta + i) * n);
    for (int k = threadIdx.x; k < h; k += kSpecThreads) dst[k] = z[k];           // out[2k] = Re z[k], out[2k+1] = Im z[k]
}

}  // namespace arkcos
