// arkcos_kernels.cuh - the sm_100a kernels of the hot path: S2 weight generator, S3/S3w convolution.
// Product code; shares nothing with oracle/.  See DESIGN.md for the design and its evidence.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "arkcos_internal.h"

namespace arkcos {

// ================================================================================================
// S2 - weight generator (BASELINE.json north_star (b))
//   w_ij[d] = A_j * K(gamma_ij(d)),  sin^2(gamma/2) = sin^2((t_i-t_j)/2) + sin t_i sin t_j sin^2(d dphi/2)
//   (the cancellation-free form of cos(gamma) = cos t_i cos t_j + sin t_i sin t_j cos(d dphi), H3),
//   K by LINEAR interpolation in the radial table held in shared memory, FP64 throughout, rounded
//   once to FP32.  Output layout: for each northern ring pair, `ntaps` floats for taps
//   d = start .. start+ntaps-1, zero outside |d| <= D (so the convolution kernel needs no masks).
// ================================================================================================
struct GenParams {
    const PairDesc* pairs;
    const GenUnit* units;
    const double* sin_t;     // [n_theta]
    const double* area;      // [n_theta]
    const double* a_r;       // [R+1]
    const double* s2;        // [n_phi/2+1]
    const double* table;     // [n_table]
    float* weights;
    int n_units, n_theta, n_phi, n_table, R;
    double t_scale;          // (n_table-1)/theta_cut
    int table_in_smem;       // 1: the table was copied to dynamic shared memory
};

__global__ void __launch_bounds__(256) k_generate_weights(const GenParams p) {
    extern __shared__ double s_table[];
    const double* tab = p.table;
    if (p.table_in_smem) {
        for (int m = threadIdx.x; m < p.n_table; m += blockDim.x) s_table[m] = p.table[m];
        __syncthreads();
        tab = s_table;
    }
    const int W = 2 * p.R + 1;
    for (int u = blockIdx.x; u < p.n_units; u += gridDim.x) {   // persistent CTA: table loaded once
        const GenUnit gu = p.units[u];
        const PairDesc pd = p.pairs[gu.pair];
        const int i = (int)(gu.pair / (uint32_t)W);
        const int r = (int)(gu.pair % (uint32_t)W) - p.R;
        const int j = i + r;
        const double a = p.a_r[r < 0 ? -r : r];
        const double b = p.sin_t[i] * p.sin_t[j];
        const double area = p.area[j];
        const int e_end = min(pd.ntaps, (int)gu.e0 + kGenUnitTaps);
        const bool whole = (pd.half == p.n_phi);
        for (int e = (int)gu.e0 + (int)threadIdx.x; e < e_end; e += blockDim.x) {
            const int d = pd.start + e;
            const int ad = d < 0 ? -d : d;
            float w = 0.0f;
            if (whole || ad <= pd.half) {
                double h = fma(b, p.s2[ad], a);
                h = fmin(h, 1.0);
                const double g = 2.0 * asin(sqrt(h));
                const double t = g * p.t_scale;
                int m = (int)t;
                m = min(m, p.n_table - 2);
                const double f = t - (double)m;
                const double k = (1.0 - f) * tab[m] + f * tab[m + 1];
                w = (float)(area * k);
            }
            p.weights[(size_t)pd.w_off + e] = w;
        }
    }
}

// ================================================================================================
// S3 / S3w - convolution (BASELINE.json north_star (c))
//
//   out[i,k] = sum_r sum_e w_{i,i+r}[e] * in[i+r, (k + start + e) mod n_phi]
//
// One CTA = one work item = (northern ring i, phi tile of 512 F outputs).  It produces ring i AND its
// southern mirror n_theta-1-i: the two share every weight (A_j, sin t are N/S symmetric), so one
// packed FFMA2 (fma.rn.f32x2, sm_100) does both with the weight as the broadcast scalar operand and
// the (north, south) input pair as the 64-bit operand.  Input rows j and n_theta-1-j are therefore
// staged INTERLEAVED in shared memory: Z[m] = (in[j][phi0+m], in[j'][phi0+m]).
//
// Each thread owns kP = 16 consecutive outputs (x2 rings) in registers and slides a 20-pair register
// window over the taps, 4 taps per step: 2 LDS.128 (4 new pairs) + 1 broadcast LDS.128 (4 weights)
// feed 64 FFMA2 = 128 FMAs.  The 8 warps of a CTA are F phi sub-tiles x S = 8/F tap splits; tap
// splits are summed in a fixed order through shared memory (deterministic, no atomics).
// ================================================================================================
struct ConvParams {
    const float* in;
    float* out;
    const PairDesc* pairs;
    const Item* items;
    const float* weights;
    int n_theta, n_phi, R;
    long long map_stride;    // elements between consecutive maps of a batch
};

__device__ __forceinline__ uint32_t zswz(uint32_t chunk) { return chunk ^ ((chunk >> 3) & 7u); }

__device__ __forceinline__ void ffma2(uint64_t& acc, const uint64_t z, const float w) {
    uint64_t ww;
    asm("mov.b64 %0, {%1, %1};" : "=l"(ww) : "f"(w));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(z), "l"(ww));
}

// One 4-tap step at rotation phase PH: logical window slot m lives in physical register (m + 4 PH) % 20.
template <int PH>
__device__ __forceinline__ void conv_step(uint64_t (&acc)[kP], uint64_t (&z)[kP + 4], const uint4* __restrict__ zs,
                                          const float* __restrict__ ws, const uint32_t chunk_new, const int e) {
    const ulonglong2 n0 = *reinterpret_cast<const ulonglong2*>(zs + zswz(chunk_new));
    const ulonglong2 n1 = *reinterpret_cast<const ulonglong2*>(zs + zswz(chunk_new + 1));
    const float4 w = *reinterpret_cast<const float4*>(ws + e);
    z[(kP + 0 + 4 * PH) % (kP + 4)] = n0.x;
    z[(kP + 1 + 4 * PH) % (kP + 4)] = n0.y;
    z[(kP + 2 + 4 * PH) % (kP + 4)] = n1.x;
    z[(kP + 3 + 4 * PH) % (kP + 4)] = n1.y;
    const float wq[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
    for (int q = 0; q < 4; q++)
#pragma unroll
        for (int p = 0; p < kP; p++) ffma2(acc[p], z[(p + q + 4 * PH) % (kP + 4)], wq[q]);
}

__global__ void __launch_bounds__(kThreads, 2) k_convolve(const ConvParams p) {
    extern __shared__ uint4 smem[];
    const Item it = p.items[blockIdx.x];
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int L = kWarpSpan << it.f_log2;
    const int TB = tap_block(it.f_log2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int cap_pairs = (L + TB + 8 + 15) & ~15;          // Z capacity in (north,south) pairs
    uint4* zs = smem;                                        // cap_pairs/2 chunks of 16 B
    float* ws = reinterpret_cast<float*>(smem + cap_pairs / 2);
    const float* in = p.in + (long long)blockIdx.y * p.map_stride;
    float* out = p.out + (long long)blockIdx.y * p.map_stride;

    const int i = it.i_north, i_s = p.n_theta - 1 - i;
    const int W = 2 * p.R + 1;
    const int lane_pair0 = f * kWarpSpan + lane * kP;        // first output of this thread inside the tile

    uint64_t acc[kP];
#pragma unroll
    for (int q = 0; q < kP; q++) acc[q] = 0ull;

    for (int r = 0; r < W; r++) {
        const PairDesc pd = p.pairs[(size_t)i * W + r];
        if (pd.ntaps == 0) continue;
        const int j = i + r - p.R, j_s = p.n_theta - 1 - j;
        const float* row_n = in + (size_t)j * p.n_phi;
        const float* row_s = in + (size_t)j_s * p.n_phi;
        for (int e0 = 0; e0 < pd.ntaps; e0 += TB) {
            const int nt = min(TB, pd.ntaps - e0);
            // ---- stage the interleaved (north, south) segment and the weights of this tap block -----
            const int org = it.k0 + pd.start + e0;           // phi of tap e0 for output k0 (may be < 0)
            const int org4 = org & ~3;                       // float4-aligned origin (two's complement floor)
            const int delta = org - org4;                    // 0 or 2
            const int nq = (delta + L + nt - 1 + 3) >> 2;    // quads of 4 phi to stage
            int phi = org4 % p.n_phi; if (phi < 0) phi += p.n_phi;
            for (int q = threadIdx.x; q < nq; q += kThreads) {
                int ph = (int)(((long long)phi + 4ll * q) % p.n_phi);
                const float4 a = __ldg(reinterpret_cast<const float4*>(row_n + ph));
                const float4 b = __ldg(reinterpret_cast<const float4*>(row_s + ph));
                const uint32_t c = zswz(2u * (uint32_t)q);
                reinterpret_cast<float4*>(zs)[c] = make_float4(a.x, b.x, a.y, b.y);
                reinterpret_cast<float4*>(zs)[c ^ 1u] = make_float4(a.z, b.z, a.w, b.w);
            }
            const float4* wsrc = reinterpret_cast<const float4*>(p.weights + (size_t)pd.w_off + e0);
            for (int q = threadIdx.x; q < (nt >> 2); q += kThreads) reinterpret_cast<float4*>(ws)[q] = __ldg(wsrc + q);
            __syncthreads();
            // ---- compute: this warp's share of the taps -----------------------------------------------
            const int chunk_taps = (((nt >> 2) + S - 1) / S) << 2;
            int e = s * chunk_taps;
            const int e_hi = min(nt, e + chunk_taps);
            if (e < e_hi) {
                uint64_t z[kP + 4];
                uint32_t c0 = (uint32_t)(delta + lane_pair0 + e) >> 1;   // chunk of the first window pair
#pragma unroll
                for (int q = 0; q < kP / 2; q++) {
                    const ulonglong2 v = *reinterpret_cast<const ulonglong2*>(zs + zswz(c0 + q));
                    z[2 * q] = v.x; z[2 * q + 1] = v.y;
                }
                uint32_t cn = c0 + kP / 2;                               // chunk of the next 2 new pairs
                while (e + 20 <= e_hi) {
                    conv_step<0>(acc, z, zs, ws, cn, e);
                    conv_step<1>(acc, z, zs, ws, cn + 2, e + 4);
                    conv_step<2>(acc, z, zs, ws, cn + 4, e + 8);
                    conv_step<3>(acc, z, zs, ws, cn + 6, e + 12);
                    conv_step<4>(acc, z, zs, ws, cn + 8, e + 16);
                    cn += 10; e += 20;
                }
                if (e < e_hi) { conv_step<0>(acc, z, zs, ws, cn, e); e += 4;
                if (e < e_hi) { conv_step<1>(acc, z, zs, ws, cn + 2, e); e += 4;
                if (e < e_hi) { conv_step<2>(acc, z, zs, ws, cn + 4, e); e += 4;
                if (e < e_hi) { conv_step<3>(acc, z, zs, ws, cn + 6, e); e += 4; } } } }
            }
            __syncthreads();
        }
    }

    // ---- epilogue ---------------------------------------------------------------------------------
    const bool mirror_distinct = (i_s != i);
    if (S == 1) {
        const int phi0 = it.k0 + lane_pair0;
        float* on = out + (size_t)i * p.n_phi + phi0;
        float* os = out + (size_t)i_s * p.n_phi + phi0;
#pragma unroll
        for (int v = 0; v < kP / 4; v++) {
            if (phi0 + 4 * v < p.n_phi) {
                float n[4], so[4];
#pragma unroll
                for (int q = 0; q < 4; q++) asm("mov.b64 {%0, %1}, %2;" : "=f"(n[q]), "=f"(so[q]) : "l"(acc[4 * v + q]));
                *reinterpret_cast<float4*>(on + 4 * v) = make_float4(n[0], n[1], n[2], n[3]);
                if (mirror_distinct) *reinterpret_cast<float4*>(os + 4 * v) = make_float4(so[0], so[1], so[2], so[3]);
            }
        }
    } else {
        // fixed-order sum of the S tap splits through shared memory (the staging buffers are free now)
        uint64_t* red = reinterpret_cast<uint64_t*>(smem);
#pragma unroll
        for (int q = 0; q < kP; q++) red[(warp * kP + q) * 32 + lane] = acc[q];
        __syncthreads();
        const int per = kP / S;                              // outputs of this sub-tile each split warp finishes
        for (int q = s * per; q < (s + 1) * per; q++) {
            float n = 0.f, so = 0.f;
            for (int s2 = 0; s2 < S; s2++) {
                const uint64_t v = red[((s2 * F + f) * kP + q) * 32 + lane];
                float a, b;
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
                n += a; so += b;
            }
            const int phi = it.k0 + lane_pair0 + q;
            if (phi < p.n_phi) {
                out[(size_t)i * p.n_phi + phi] = n;
                if (mirror_distinct) out[(size_t)i_s * p.n_phi + phi] = so;
            }
        }
    }
}

// dynamic shared memory of k_convolve for a given F
inline size_t conv_smem_bytes(int f_log2) {
    const int L = kWarpSpan << f_log2, TB = tap_block(f_log2);
    const size_t cap_pairs = (size_t)((L + TB + 8 + 15) & ~15);
    size_t stage = cap_pairs * 8 + (size_t)TB * 4;
    size_t red = (size_t)kWarps * kP * 32 * 8;
    return stage > red ? stage : red;
}

}  // namespace arkcos
