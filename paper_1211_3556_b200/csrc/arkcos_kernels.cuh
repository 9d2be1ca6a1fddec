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
//   once to FP32; zero outside the window (so the convolution kernels need no masks).
//   Output layouts (PairDesc): plain taps for the narrow rings, (K(d), K(d+1), K(d-1), K(d)) steps
//   for the wide rings.  One warp per work unit; persistent CTAs so the table is loaded into shared
//   memory once per SM.
// ================================================================================================
struct GenParams {
    const GenUnit* units;
    const double* s2;        // [n_phi/2+1] sin^2(d dphi / 2)
    const double* table;     // [n_table]
    float* weights;
    int n_units, n_phi, n_table;
    double t_scale;          // (n_table-1)/theta_cut
    int table_in_smem;       // 1: the table was copied to dynamic shared memory
};

constexpr int kGenThreads = 512;

__device__ __forceinline__ float gen_weight(const GenParams& p, const GenUnit& g, const double* tab, const int d) {
    const int ad = d < 0 ? -d : d;
    const bool inside = (g.half == p.n_phi) ? (d >= -(p.n_phi / 2) && d < p.n_phi / 2) : (ad <= g.half);
    if (!inside) return 0.0f;
    double h = fma(g.b, p.s2[ad], g.a);
    h = fmin(h, 1.0);
    const double gam = 2.0 * asin(sqrt(h));
    const double t = gam * p.t_scale;
    int m = (int)t;
    m = min(m, p.n_table - 2);
    const double f = t - (double)m;
    const double k = (1.0 - f) * tab[m] + f * tab[m + 1];
    return (float)(g.area * k);
}

__global__ void __launch_bounds__(kGenThreads) k_generate_weights(const GenParams p) {
    extern __shared__ double s_table[];
    const double* tab = p.table;
    if (p.table_in_smem) {
        for (int m = threadIdx.x; m < p.n_table; m += blockDim.x) s_table[m] = p.table[m];
        __syncthreads();
        tab = s_table;
    }
    const int warps = kGenThreads / 32, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int u = blockIdx.x * warps + warp; u < p.n_units; u += gridDim.x * warps) {
        const GenUnit g = p.units[u];
        if (g.eo == 0) {
            for (int e = lane; e < g.count; e += 32) p.weights[(size_t)g.w_base + e] = gen_weight(p, g, tab, g.d0 + e);
        } else {
            // step t: d = d0 + 2t.  K(d-1) of a lane is K(d+1) of the lane before it.
            float carry = gen_weight(p, g, tab, g.d0 - 1);
            for (int e0 = 0; e0 < g.count; e0 += 32) {
                const int e = e0 + lane;
                const int d = g.d0 + 2 * e;
                float k0 = 0.f, k1 = 0.f;
                if (e < g.count) { k0 = gen_weight(p, g, tab, d); k1 = gen_weight(p, g, tab, d + 1); }
                float km = __shfl_up_sync(0xffffffffu, k1, 1);
                if (lane == 0) km = carry;
                carry = __shfl_sync(0xffffffffu, k1, 31);
                if (e < g.count) *reinterpret_cast<float4*>(p.weights + (size_t)g.w_base + 4 * (size_t)e) = make_float4(k0, k1, km, k0);
            }
        }
    }
}

// ================================================================================================
// S3 / S3w - convolution (BASELINE.json north_star (c))
//
//   out[i,k] = sum_r sum_e w_{i,i+r}[e] * in[i+r, (k + start + e) mod n_phi]
//
// A CTA produces northern ring(s) i AND the southern mirror(s) n_theta-1-i: the two share every weight
// (A_j and sin t are N/S symmetric), so one packed FFMA2 (fma.rn.f32x2, sm_100) does both, with the
// weight as the broadcast scalar operand and the (north, south) input pair as the 64-bit operand.
// Input rows j and n_theta-1-j are therefore staged INTERLEAVED in shared memory,
// Z[m] = (in[j][phi0+m], in[j'][phi0+m]), 16-byte chunks XOR-swizzled against bank conflicts.
//
// Each thread owns kP = 16 consecutive outputs (x2 rings) in registers and slides a 20-pair register
// window over the taps, 4 taps per step: 2 LDS.128 (4 new pairs) + 1 broadcast LDS.128 (4 weights)
// feed 64 FFMA2 = 128 FMAs.  A CTA is 8 warps = F phi sub-tiles x S; one CTA per SM.
//
//   WIDE items   (polar / high-latitude rings, windows of 64 .. n_phi taps): one ring, S tap splits
//                summed in a fixed order through shared memory; stages = (row, tap block), double
//                buffered, the next stage prefetched through registers while the current one computes.
//   NARROW items (windows inside [-32, 32)): a band of rings marches through a shared-memory ring of
//                2R+S interleaved rows, S rings per pass, so every input row is staged once per band
//                instead of once per output ring; the S new rows of the next pass are prefetched
//                through registers during the pass.
// ================================================================================================
struct ConvParams {
    const float* in;
    float* out;
    const PairDesc* pairs;
    const Item* items;
    const float* weights;
    const uint32_t* ring_w_off;
    const uint32_t* ring_slots;
    int n_theta, n_phi, R;
    int wslot;               // floats per ring in the narrow weight buffers
    long long map_stride;    // elements between consecutive maps of a batch
};

__device__ __forceinline__ uint32_t zswz(uint32_t chunk) { return chunk ^ ((chunk >> 3) & 7u); }

__device__ __forceinline__ void ffma2(uint64_t& acc, const uint64_t z, const float w) {
    uint64_t ww;
    asm("mov.b64 %0, {%1, %1};" : "=l"(ww) : "f"(w));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(z), "l"(ww));
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

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

// acc[p] += sum_{e in [e_lo, e_hi)} ws[e] * Z[pair0 + p + e]   (e_lo, e_hi multiples of 4; pair0 even)
__device__ __forceinline__ void conv_taps(uint64_t (&acc)[kP], const uint4* __restrict__ zs, const float* __restrict__ ws,
                                          const uint32_t pair0, int e, const int e_hi) {
    if (e >= e_hi) return;
    uint64_t z[kP + 4];
    const uint32_t c0 = (pair0 + (uint32_t)e) >> 1;          // 16-byte chunk of the first window pair
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
    if (e < e_hi) { conv_step<3>(acc, z, zs, ws, cn + 6, e); } } } }
}

// Interleaved staging through registers: quad q of a segment = 4 consecutive phi of the northern row
// and of its mirror row -> two 16-byte chunks (n0 s0 n1 s1)(n2 s2 n3 s3).
struct Quad { float4 n, s; };

__device__ __forceinline__ Quad quad_load(const float* __restrict__ row_n, const float* __restrict__ row_s, int phi) {
    Quad v;
    v.n = __ldg(reinterpret_cast<const float4*>(row_n + phi));
    v.s = __ldg(reinterpret_cast<const float4*>(row_s + phi));
    return v;
}
__device__ __forceinline__ void quad_store(uint4* zs, int q, const Quad& v) {
    const uint32_t c = zswz(2u * (uint32_t)q);
    reinterpret_cast<float4*>(zs)[c] = make_float4(v.n.x, v.s.x, v.n.y, v.s.y);
    reinterpret_cast<float4*>(zs)[c ^ 1u] = make_float4(v.n.z, v.s.z, v.n.w, v.s.w);
}
__device__ __forceinline__ int wrap_phi(int phi, int n_phi) {   // phi may be any int; result in [0, n_phi)
    int r = phi % n_phi;
    return r < 0 ? r + n_phi : r;
}

__device__ __forceinline__ void store_outputs(const ConvParams& p, float* out, int i, int phi0, const uint64_t (&acc)[kP]) {
    const int i_s = p.n_theta - 1 - i;
    float* on = out + (size_t)i * p.n_phi + phi0;
    float* os = out + (size_t)i_s * p.n_phi + phi0;
#pragma unroll
    for (int v = 0; v < kP / 4; v++) {
        if (phi0 + 4 * v < p.n_phi) {
            float n[4], so[4];
#pragma unroll
            for (int q = 0; q < 4; q++) asm("mov.b64 {%0, %1}, %2;" : "=f"(n[q]), "=f"(so[q]) : "l"(acc[4 * v + q]));
            *reinterpret_cast<float4*>(on + 4 * v) = make_float4(n[0], n[1], n[2], n[3]);
            if (i_s != i) *reinterpret_cast<float4*>(os + 4 * v) = make_float4(so[0], so[1], so[2], so[3]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// WIDE item: one output ring (either hemisphere), F sub-tiles of kWideSpan outputs x S tap splits.
//
// Every warp is autonomous: it streams ITS share of the ring's taps through two private stage buffers
// filled with cp.async (no CTA barrier until the final reduction of the S splits), so the warps of an
// SM drift apart and the FMA pipe never waits for a common stage hand-over.
//
// Even/odd packing: a lane owns 32 consecutive outputs k..k+31.  For the aligned input pair
// Z = (x[k+2m+d], x[k+2m+d+1]), d even, one FFMA2 with the weight pair (K(d), K(d+1)) advances the
// EVEN output k+2m by two taps, and one with (K(d-1), K(d)) advances the ODD output k+2m+1; the two
// halves of an accumulator are added at the end.  No input interleaving, no weight duplication:
// the input rows are staged as they are in memory.
//
// Stage layout: logical float m of the stage = x[(phi0 + m) mod n_phi]; 16-byte chunk c sits at
// physical chunk c + (c >> 3), i.e. lane tiles (8 chunks) have a stride of 9 chunks and LDS.128 is
// conflict free without swizzle arithmetic.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void ffma2p(uint64_t& acc, const uint64_t z, const uint64_t w) {
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(z), "l"(w));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int kZRing = 10;                // register window: 10 chunks = 20 input pairs (17 live + prefetch)

// 16-byte shared-memory load that the compiler may not sink, hoist or drop: the loads below are
// software prefetches issued one double step ahead of their first use.
__device__ __forceinline__ void lds128(uint64_t& a, uint64_t& b, const uint32_t addr) {
    asm volatile("ld.shared.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "r"(addr));
}

// One double step (4 taps) at window phase PH.  Live chunks q .. q+8 sit in ring slots (PH + c) % 10;
// chunk q+9 is fetched into the slot chunk q-1 has just left, the weights of double step q+1 into the
// other half of the weight double buffer.
template <int PH>
__device__ __forceinline__ void eo_dstep(uint64_t (&E)[16], uint64_t (&O)[16], uint64_t (&z)[2 * kZRing],
                                         uint64_t (&w)[2][4], const uint32_t zlane, const uint32_t ws, const int q) {
    constexpr int B = PH & 1;
    const int u = q + 9;
    lds128(z[(2 * (PH + 9)) % (2 * kZRing)], z[(2 * (PH + 9) + 1) % (2 * kZRing)], zlane + (uint32_t)((u + (u >> 3)) << 4));
    lds128(w[B ^ 1][0], w[B ^ 1][1], ws + (uint32_t)(32 * q + 32));
    lds128(w[B ^ 1][2], w[B ^ 1][3], ws + (uint32_t)(32 * q + 48));
#pragma unroll
    for (int m = 0; m < 16; m++) {
        ffma2p(E[m], z[(2 * PH + m) % (2 * kZRing)], w[B][0]);
        ffma2p(O[m], z[(2 * PH + m) % (2 * kZRing)], w[B][1]);
    }
#pragma unroll
    for (int m = 0; m < 16; m++) {
        ffma2p(E[m], z[(2 * PH + 1 + m) % (2 * kZRing)], w[B][2]);
        ffma2p(O[m], z[(2 * PH + 1 + m) % (2 * kZRing)], w[B][3]);
    }
}

// E[m] += sum_t Z[m+t] * ws[t].x,  O[m] += sum_t Z[m+t] * ws[t].y  over t = 0 .. 2 nq - 1
// zlane / ws: shared-memory addresses of the lane's first chunk and of the stage's weights.
__device__ __forceinline__ void eo_taps(uint64_t (&E)[16], uint64_t (&O)[16], const uint32_t zlane, const uint32_t ws,
                                        const int nq) {
    uint64_t z[2 * kZRing];
#pragma unroll
    for (int c = 0; c < 9; c++) lds128(z[2 * c], z[2 * c + 1], zlane + (uint32_t)((c + (c >> 3)) << 4));
    z[18] = 0ull; z[19] = 0ull;
    uint64_t w[2][4];
    lds128(w[0][0], w[0][1], ws);
    lds128(w[0][2], w[0][3], ws + 16);
    int q = 0;
    for (;;) {
        eo_dstep<0>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<1>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<2>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<3>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<4>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<5>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<6>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<7>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<8>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
        eo_dstep<9>(E, O, z, w, zlane, ws, q); if (++q == nq) break;
    }
}

struct WideStage {
    const float* row;    // input ring
    int phi0;            // phi of logical float 0 of the stage, in [0, n_phi), multiple of 4
    int nq;              // double steps (4 taps each), 1 .. kWideStage/2
    uint32_t w_off;      // first weight of the stage (floats)
};

__device__ void conv_wide(const ConvParams& p, const Item& it, uint4* smem, const float* in, float* out) {
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int W = 2 * p.R + 1;
    const int i = it.i0;
    const bool mirrored = 2 * i >= p.n_theta;                  // southern ring: weights of its mirror pair
    const int i_n = mirrored ? p.n_theta - 1 - i : i;
    char* wsm = reinterpret_cast<char*>(smem) + (size_t)warp * 2 * kWideStageBytes;
    const uint32_t wsm_addr = (uint32_t)__cvta_generic_to_shared(wsm);
    PairDesc* spd = reinterpret_cast<PairDesc*>(reinterpret_cast<char*>(smem) + (size_t)kWarps * 2 * kWideStageBytes);
    for (int r = threadIdx.x; r < W; r += kThreads) spd[r] = p.pairs[(size_t)i_n * W + r];
    __syncthreads();

    const int K0 = it.k0 + f * kWideSpan;                      // first output of this warp
    // this warp's share [g_lo, g_hi) of the ring's double steps (rows concatenated)
    int G = 0;
    for (int r = 0; r < W; r++) G += spd[r].ntaps >> 2;
    int g_lo = (int)(((long long)G * s) / S), g_hi = (int)(((long long)G * (s + 1)) / S);
    if (K0 >= p.n_phi) g_hi = g_lo;                            // ragged tile: no outputs here
    int r = 0, q = 0, remaining = g_hi - g_lo;
    for (int acc = 0; r < W; r++) {
        const int n = spd[r].ntaps >> 2;
        if (g_lo < acc + n) { q = g_lo - acc; break; }
        acc += n;
    }
    auto next_stage = [&](WideStage& st) -> bool {
        if (remaining <= 0) return false;
        while (q >= (spd[r].ntaps >> 2)) { r++; q = 0; }
        const PairDesc pd = spd[r];
        st.nq = min(min(kWideStage / 2, (pd.ntaps >> 2) - q), remaining);
        const int j = mirrored ? i - (r - p.R) : i + (r - p.R);
        st.row = in + (size_t)j * p.n_phi;
        st.phi0 = wrap_phi(K0 + pd.start + 4 * q, p.n_phi);
        st.w_off = pd.w_off + 8u * (uint32_t)q;
        q += st.nq; remaining -= st.nq;
        return true;
    };
    // lane-constant parts of the stage fill: chunk c = lane + 32 n sits at physical chunk
    // (lane + (lane >> 3)) + 36 n, its input at phi0 + 4 lane + 128 n (mod n_phi)
    const int lane_phi = (4 * lane) % p.n_phi, phi_step = 128 % p.n_phi;
    const int lane_dst = (lane + (lane >> 3)) << 4;
    auto issue = [&](const WideStage& st, const int b) {
        char* zb = wsm + b * kWideStageBytes;
        const int nchunks = kWideSpan / 4 + st.nq + 1;
        int phi = st.phi0 + lane_phi;
        if (phi >= p.n_phi) phi -= p.n_phi;
        char* dst = zb + lane_dst;
#pragma unroll 4
        for (int c = lane; c < nchunks; c += 32) {
            cp_async16(dst, st.row + phi);
            dst += 36 * 16;
            phi += phi_step;
            if (phi >= p.n_phi) phi -= p.n_phi;
        }
        char* wb = zb + kWideZChunks * 16;
        const float* wsrc = p.weights + st.w_off;
        for (int c = lane; c < 2 * st.nq; c += 32) cp_async16(wb + 16 * c, wsrc + 4 * c);
        cp_async_commit();
    };

    uint64_t E[16], O[16];
#pragma unroll
    for (int m = 0; m < 16; m++) { E[m] = 0ull; O[m] = 0ull; }

    WideStage cur, nxt;
    bool have = next_stage(cur);
    int b = 0;
    if (have) issue(cur, 0);
    while (have) {
        const bool more = next_stage(nxt);
        if (more) { issue(nxt, b ^ 1); cp_async_wait_group<1>(); } else { cp_async_wait_group<0>(); }
        __syncwarp();
        const uint32_t zb = wsm_addr + (uint32_t)(b * kWideStageBytes);
        eo_taps(E, O, zb + (uint32_t)(lane * 144), zb + (uint32_t)(kWideZChunks * 16), cur.nq);
        __syncwarp();                                          // buffer b is free for the stage after next
        cur = nxt; have = more; b ^= 1;
    }

    // ---- epilogue: fold the two halves, sum the S splits in a fixed order, store float4 -----------------
    float v[kWideP];
#pragma unroll
    for (int m = 0; m < 16; m++) {
        float a0, a1, b0, b1;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(a0), "=f"(a1) : "l"(E[m]));
        asm("mov.b64 {%0, %1}, %2;" : "=f"(b0), "=f"(b1) : "l"(O[m]));
        v[2 * m] = a0 + a1; v[2 * m + 1] = b0 + b1;
    }
    float* orow = out + (size_t)i * p.n_phi;
    if (S == 1) {
        const int phi = K0 + lane * kWideP;
#pragma unroll
        for (int g = 0; g < kWideP / 4; g++)
            if (phi + 4 * g < p.n_phi)
                *reinterpret_cast<float4*>(orow + phi + 4 * g) = make_float4(v[4 * g], v[4 * g + 1], v[4 * g + 2], v[4 * g + 3]);
    } else {
        __syncthreads();                                       // every warp is done with its stage buffers
        float* red = reinterpret_cast<float*>(smem);           // [warp][p][lane]
#pragma unroll
        for (int pp = 0; pp < kWideP; pp++) red[(warp * kWideP + pp) * 32 + lane] = v[pp];
        __syncthreads();
        const int per = (kWideP / 4) / S;                      // float4 groups of this lane's 32 outputs per split
        for (int g = s * per; g < (s + 1) * per; g++) {
            float o[4];
#pragma unroll
            for (int x = 0; x < 4; x++) {
                float sum = 0.f;
                for (int s2 = 0; s2 < S; s2++) sum += red[((s2 * F + f) * kWideP + 4 * g + x) * 32 + lane];
                o[x] = sum;
            }
            const int phi = K0 + lane * kWideP + 4 * g;
            if (phi < p.n_phi) *reinterpret_cast<float4*>(orow + phi) = make_float4(o[0], o[1], o[2], o[3]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// NARROW item: band marching
// ------------------------------------------------------------------------------------------------
__device__ void conv_narrow(const ConvParams& p, const Item& it, uint4* smem, const float* in, float* out) {
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int L = kWarpSpan << it.f_log2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int W = 2 * p.R + 1;
    const int nslot = 2 * p.R + S;
    const int slot_pairs = L + 2 * kHaloNarrow;
    const int slot_chunks = slot_pairs / 2;
    const int nq_row = slot_pairs / 4;                        // quads per staged row
    float* wbuf = reinterpret_cast<float*>(smem + (size_t)nslot * slot_chunks);          // [2][S][wslot]
    PairDesc* pdbuf = reinterpret_cast<PairDesc*>(wbuf + 2 * (size_t)S * p.wslot);        // [2][S][W]
    const int phi_org = wrap_phi(it.k0 - kHaloNarrow, p.n_phi);                          // phi of slot pair 0
    const uint32_t lane_pair0 = (uint32_t)(kHaloNarrow + f * kWarpSpan + lane * kP);
    const int i_end = it.i0 + it.nrings;
    const int npass = (it.nrings + S - 1) / S;

    // the (row-in-pass, quad, phi) this thread stages in every pass: fixed for the whole item
    int pf_jr[kPrefetchNarrow], pf_q[kPrefetchNarrow], pf_phi[kPrefetchNarrow];
    const int total_new = S * nq_row;
#pragma unroll
    for (int u = 0; u < kPrefetchNarrow; u++) {
        const int idx = threadIdx.x + u * kThreads;
        const int jr = idx / nq_row;
        pf_jr[u] = idx < total_new ? jr : -1;
        pf_q[u] = idx - jr * nq_row;
        pf_phi[u] = wrap_phi(phi_org + 4 * pf_q[u], p.n_phi);
    }

    // rows [j_lo, j_hi) -> their slots, directly (band prologue)
    {
        const int j_lo = it.i0 - p.R, j_hi = it.i0 + S + p.R;
        const int total = (j_hi - j_lo) * nq_row;
        for (int idx = threadIdx.x; idx < total; idx += kThreads) {
            const int jr = idx / nq_row, q = idx - jr * nq_row;
            const int j = j_lo + jr;
            if (j < 0 || j >= p.n_theta) continue;
            const float* row_n = in + (size_t)j * p.n_phi;
            const float* row_s = in + (size_t)(p.n_theta - 1 - j) * p.n_phi;
            const int slot = (j + nslot * 4) % nslot;         // j >= -R > -4 nslot
            quad_store(smem + (size_t)slot * slot_chunks, q, quad_load(row_n, row_s, wrap_phi(phi_org + 4 * q, p.n_phi)));
        }
    }
    // weights and pair descriptors of the S rings of a pass -> buffer b (cp.async)
    auto stage_ring_tables = [&](int pass, int b) {
        for (int rs = 0; rs < S; rs++) {
            const int i = it.i0 + pass * S + rs;
            if (i >= i_end) break;
            const PairDesc* psrc = p.pairs + (size_t)i * W;
            PairDesc* pdst = pdbuf + ((size_t)b * S + rs) * W;
            for (int q = threadIdx.x; q < W; q += kThreads) cp_async16(pdst + q, psrc + q);
            const float* src = p.weights + p.ring_w_off[i];
            float* dst = wbuf + ((size_t)b * S + rs) * p.wslot;
            const int n4 = (int)(p.ring_slots[i] >> 2);
            for (int q = threadIdx.x; q < n4; q += kThreads) cp_async16(dst + 4 * q, src + 4 * q);
        }
    };
    stage_ring_tables(0, 0);
    cp_async_wait_all();
    __syncthreads();

    int slot_lo = (it.i0 - p.R + nslot * 4) % nslot;          // slot of row ibase - R
    for (int pass = 0; pass < npass; pass++) {
        const int ibase = it.i0 + pass * S;
        const bool more = pass + 1 < npass;
        // ---- prefetch the S new rows of the next pass into registers ----------------------------------
        Quad pf[kPrefetchNarrow];
        const int j_new = ibase + S + p.R;                    // first new row of the next pass
        if (more) {
#pragma unroll
            for (int u = 0; u < kPrefetchNarrow; u++) {
                const int j = j_new + pf_jr[u];
                if (pf_jr[u] >= 0 && j < p.n_theta)
                    pf[u] = quad_load(in + (size_t)j * p.n_phi, in + (size_t)(p.n_theta - 1 - j) * p.n_phi, pf_phi[u]);
            }
            stage_ring_tables(pass + 1, (pass + 1) & 1);
        }
        // ---- compute ring ibase + s from the rows resident in shared memory ------------------------------
        const int i = ibase + s;
        if (i < i_end) {
            uint64_t acc[kP];
#pragma unroll
            for (int q = 0; q < kP; q++) acc[q] = 0ull;
            const float* wring = wbuf + ((size_t)(pass & 1) * S + s) * p.wslot;
            const PairDesc* spd = pdbuf + ((size_t)(pass & 1) * S + s) * W;
            uint32_t w0 = 0xFFFFFFFFu;
            int slot = slot_lo + s;                           // slot of row i - R
            if (slot >= nslot) slot -= nslot;
            PairDesc pd = spd[0];
            for (int r = 0; r < W; r++) {
                const PairDesc pd_next = spd[r + 1 < W ? r + 1 : r];
                if (pd.ntaps != 0) {
                    if (w0 == 0xFFFFFFFFu) w0 = pd.w_off;      // first stored row = start of the ring's weights
                    conv_taps(acc, smem + (size_t)slot * slot_chunks, wring + (pd.w_off - w0),
                              (uint32_t)((int)lane_pair0 + pd.start), 0, pd.ntaps);
                }
                pd = pd_next;
                if (++slot == nslot) slot = 0;
            }
            store_outputs(p, out, i, it.k0 + f * kWarpSpan + lane * kP, acc);
        }
        __syncthreads();                                      // every warp is done with the oldest S rows
        if (more) {
            int slot_new = slot_lo;                           // the new rows replace rows ibase-R .. ibase-R+S-1
#pragma unroll
            for (int u = 0; u < kPrefetchNarrow; u++) {
                const int j = j_new + pf_jr[u];
                if (pf_jr[u] >= 0 && j < p.n_theta) {
                    int sl = slot_new + pf_jr[u];
                    if (sl >= nslot) sl -= nslot;
                    quad_store(smem + (size_t)sl * slot_chunks, pf_q[u], pf[u]);
                }
            }
            cp_async_wait_all();
        }
        slot_lo += S;
        if (slot_lo >= nslot) slot_lo -= nslot;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kThreads, 1) k_convolve(const ConvParams p) {
    extern __shared__ uint4 smem[];
    const Item it = p.items[blockIdx.x];
    const float* in = p.in + (long long)blockIdx.y * p.map_stride;
    float* out = p.out + (long long)blockIdx.y * p.map_stride;
    if (it.kind == kWide) conv_wide(p, it, smem, in, out);
    else conv_narrow(p, it, smem, in, out);
}

}  // namespace arkcos
