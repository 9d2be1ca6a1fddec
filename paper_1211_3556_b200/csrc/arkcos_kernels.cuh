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
//   One warp per work unit; persistent CTAs so the table is loaded into shared memory once per SM.
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
        const bool whole = (g.half == p.n_phi);
        for (int e = lane; e < g.count; e += 32) {
            const int d = g.d0 + e;
            const int ad = d < 0 ? -d : d;
            float w = 0.0f;
            if (whole || ad <= g.half) {
                double h = fma(g.b, p.s2[ad], g.a);
                h = fmin(h, 1.0);
                const double gam = 2.0 * asin(sqrt(h));
                const double t = gam * p.t_scale;
                int m = (int)t;
                m = min(m, p.n_table - 2);
                const double f = t - (double)m;
                const double k = (1.0 - f) * tab[m] + f * tab[m + 1];
                w = (float)(g.area * k);
            }
            p.weights[(size_t)g.w_base + e] = w;
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
// WIDE item
// ------------------------------------------------------------------------------------------------
struct WideStage {       // one (row, tap block) of the item
    int r, e0, nt;       // row slot 0..2R, first tap, taps in the block; r > 2R = end
    int j;               // input ring
    int phi4;            // float4-aligned phi of segment pair 0, in [0, n_phi)
    int delta;           // 0 or 2: pair index of tap e0 for output k0
    int nq;              // quads to stage
    uint32_t w_off;      // weights of this block
};

__device__ __forceinline__ void wide_describe(const ConvParams& p, const Item& it, int L, WideStage& s, const PairDesc& pd) {
    s.nt = min(tap_block(it.f_log2), pd.ntaps - s.e0);
    s.j = it.i0 + s.r - p.R;
    const int org = it.k0 + pd.start + s.e0;
    const int org4 = org & ~3;
    s.delta = org - org4;
    s.phi4 = wrap_phi(org4, p.n_phi);
    s.nq = (s.delta + L + s.nt - 1 + 3) >> 2;
    s.w_off = pd.w_off + (uint32_t)s.e0;
}
// first stage at or after (r, e0); the ring's pair descriptors are in shared memory
__device__ __forceinline__ void wide_seek(const ConvParams& p, const Item& it, int L, WideStage& s, const PairDesc* spd) {
    const int W = 2 * p.R + 1;
    while (s.r < W) {
        const PairDesc pd = spd[s.r];
        if (s.e0 < pd.ntaps) { wide_describe(p, it, L, s, pd); return; }
        s.r++; s.e0 = 0;
    }
}

__device__ void conv_wide(const ConvParams& p, const Item& it, uint4* smem, const float* in, float* out) {
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int L = kWarpSpan << it.f_log2, TB = tap_block(it.f_log2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int W = 2 * p.R + 1;
    const int cap_pairs = (L + TB + 8 + 15) & ~15;
    const int buf_chunks = cap_pairs / 2 + TB / 4;           // one stage buffer: Z chunks then weights
    const uint32_t lane_pair0 = (uint32_t)(f * kWarpSpan + lane * kP);
    const int s_log2 = 3 - it.f_log2;
    PairDesc* spd = reinterpret_cast<PairDesc*>(smem + 2 * buf_chunks);   // [W] descriptors of this ring
    for (int r = threadIdx.x; r < W; r += kThreads) spd[r] = p.pairs[(size_t)it.i0 * W + r];
    __syncthreads();

    uint64_t acc[kP];
#pragma unroll
    for (int q = 0; q < kP; q++) acc[q] = 0ull;

    WideStage cur; cur.r = 0; cur.e0 = 0;
    wide_seek(p, it, L, cur, spd);
    int buf = 0;
    // prologue: stage the first block directly
    if (cur.r < W) {
        uint4* zs = smem;
        const float* row_n = in + (size_t)cur.j * p.n_phi;
        const float* row_s = in + (size_t)(p.n_theta - 1 - cur.j) * p.n_phi;
        for (int q = threadIdx.x; q < cur.nq; q += kThreads)
            quad_store(zs, q, quad_load(row_n, row_s, wrap_phi(cur.phi4 + 4 * q, p.n_phi)));
        float* ws = reinterpret_cast<float*>(smem + cap_pairs / 2);
        for (int q = threadIdx.x; q < (cur.nt >> 2); q += kThreads) cp_async16(ws + 4 * q, p.weights + (size_t)cur.w_off + 4 * q);
        cp_async_wait_all();
    }
    __syncthreads();
    while (cur.r < W) {
        WideStage nxt; nxt.r = cur.r; nxt.e0 = cur.e0 + TB;
        wide_seek(p, it, L, nxt, spd);
        const bool more = nxt.r < W;
        uint4* zs = smem + buf * buf_chunks;
        const float* ws = reinterpret_cast<const float*>(zs + cap_pairs / 2);
        uint4* zs_n = smem + (buf ^ 1) * buf_chunks;
        float* ws_n = reinterpret_cast<float*>(zs_n + cap_pairs / 2);
        // ---- prefetch the next stage: global loads into registers, weights by cp.async --------------
        Quad pf[kPrefetchWide];
        if (more) {
            const float* row_n = in + (size_t)nxt.j * p.n_phi;
            const float* row_s = in + (size_t)(p.n_theta - 1 - nxt.j) * p.n_phi;
#pragma unroll
            for (int u = 0; u < kPrefetchWide; u++) {
                const int q = threadIdx.x + u * kThreads;
                if (q < nxt.nq) pf[u] = quad_load(row_n, row_s, wrap_phi(nxt.phi4 + 4 * q, p.n_phi));
            }
            for (int q = threadIdx.x; q < (nxt.nt >> 2); q += kThreads) cp_async16(ws_n + 4 * q, p.weights + (size_t)nxt.w_off + 4 * q);
        }
        // ---- compute this warp's share of the taps of the current stage --------------------------------
        {
            const int chunk_taps = (((cur.nt >> 2) + S - 1) >> s_log2) << 2;
            const int e_lo = s * chunk_taps;
            const int e_hi = min(cur.nt, e_lo + chunk_taps);
            conv_taps(acc, zs, ws, (uint32_t)cur.delta + lane_pair0, e_lo, e_hi);
        }
        // ---- commit the prefetched stage to the other buffer ---------------------------------------------
        if (more) {
#pragma unroll
            for (int u = 0; u < kPrefetchWide; u++) {
                const int q = threadIdx.x + u * kThreads;
                if (q < nxt.nq) quad_store(zs_n, q, pf[u]);
            }
            cp_async_wait_all();
        }
        __syncthreads();
        cur = nxt; buf ^= 1;
    }

    // ---- epilogue -----------------------------------------------------------------------------------------
    const int i = it.i0, i_s = p.n_theta - 1 - i;
    if (S == 1) {
        store_outputs(p, out, i, it.k0 + (int)lane_pair0, acc);
    } else {
        // fixed-order sum of the S tap splits through shared memory (all stage buffers are free now)
        __syncthreads();
        uint64_t* red = reinterpret_cast<uint64_t*>(smem);
#pragma unroll
        for (int q = 0; q < kP; q++) red[(warp * kP + q) * 32 + lane] = acc[q];
        __syncthreads();
        const int per = kP / S;
        for (int q = s * per; q < (s + 1) * per; q++) {
            float n = 0.f, so = 0.f;
            for (int s2 = 0; s2 < S; s2++) {
                const uint64_t v = red[((s2 * F + f) * kP + q) * 32 + lane];
                float a, b;
                asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
                n += a; so += b;
            }
            const int phi = it.k0 + (int)lane_pair0 + q;
            if (phi < p.n_phi) {
                out[(size_t)i * p.n_phi + phi] = n;
                if (i_s != i) out[(size_t)i_s * p.n_phi + phi] = so;
            }
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
