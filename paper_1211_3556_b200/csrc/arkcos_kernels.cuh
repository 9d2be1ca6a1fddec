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
//   once to FP32; zero outside the window (so the convolution kernels need no masks).  The table is
//   uniform in theta, or the paper's two-zone table with half the nodes in the innermost part of the
//   support (arkcos_plan_create_biased).
//   One warp per work unit; persistent CTAs so the table is loaded into shared memory once per SM.
// ================================================================================================
struct GenParams {
    const GenUnit* units;
    const double* s2;        // [n_phi/2+1] sin^2(d dphi / 2)
    const double* table;     // [n_table]
    float* weights;
    int n_units, n_phi, n_table;
    double t_scale;          // (n_table-1)/theta_cut; two-zone table: m_split/theta_split
    int table_in_smem;       // 1: the table was copied to dynamic shared memory
    int m_split;             // 0: uniform table.  > 0: two-zone table, node m_split at theta_split
    double theta_split;
    double t_scale2;         // (n_table-1-m_split)/(theta_cut-theta_split)
};

constexpr int kGenThreads = 512;
constexpr int kGenSmemMax = 200 * 1024;   // largest table (bytes) the generator keeps in shared memory

__device__ __forceinline__ float gen_weight(const GenParams& p, const GenUnit& g, const double* tab, const int d) {
    const int ad = d < 0 ? -d : d;
    const bool inside = (g.half == p.n_phi) ? (d >= -(p.n_phi / 2) && d < p.n_phi / 2) : (ad <= g.half);
    if (!inside) return 0.0f;
    double h = fma(g.b, p.s2[ad], g.a);
    h = fmin(h, 1.0);
    const double gam = 2.0 * asin(sqrt(h));
    double t = gam * p.t_scale;
    if (p.m_split > 0 && gam >= p.theta_split) t = (double)p.m_split + (gam - p.theta_split) * p.t_scale2;
    int m = (int)t;
    m = min(m, p.n_table - 2);
    const double f = t - (double)m;
    const double k = (1.0 - f) * tab[m] + f * tab[m + 1];
    return (float)(g.area * k);
}

__global__ void __launch_bounds__(kGenThreads) k_generate_weights(const GenParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ double s_table[];
#else
    double* s_table = reinterpret_cast<double*>(emu::g_smem);
#endif
    const double* tab = p.table;
    if (p.table_in_smem) {
        for (int m = threadIdx.x; m < p.n_table; m += blockDim.x) s_table[m] = p.table[m];
        __syncthreads();
        tab = s_table;
    }
    const int warps = kGenThreads / 32, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // the next unit's descriptor is fetched while the current unit is computed (a warp handles ~20 units
    // one after the other; each descriptor would otherwise cost a full global-memory round trip)
    const int stride = gridDim.x * warps;
    int u = blockIdx.x * warps + warp;
    if (u >= p.n_units) return;
    GenUnit g = p.units[u];
    for (; u < p.n_units; u += stride) {
        const GenUnit nxt = p.units[u + stride < p.n_units ? u + stride : u];
        for (int e = lane; e < g.count; e += 32) p.weights[(size_t)g.w_base + e] = gen_weight(p, g, tab, g.d0 + e);
        g = nxt;
    }
}

// ================================================================================================
// S3 / S3w - convolution (BASELINE.json north_star (c))
//
//   out[i,k] = sum_r sum_e w_{i,i+r}[e] * in[i+r, (k + start + e) mod n_phi]
//
// A lane owns kLaneP = 32 consecutive outputs of one ring in registers and slides a register window
// of the input row over the taps:  acc[m] += w[e] * z[m + e].  The weight is warp uniform, so the
// inner loop is plain FFMA acc, z, w.reuse, acc - the form that issues at 124 of 128 FMA/clk/SM on
// B200 (the packed FFMA2 form tops out at 94, register-read bound).  Everything else is
// kept off the issue slots: input rows are staged with cp.async as they are in memory, in a lane-tile
// layout (8 chunks + 1 pad chunk per lane) that makes the window loads conflict free.
//
//   WIDE items   (polar / high-latitude rings, windows of 64 .. n_phi taps): one ring; every warp
//                streams its share of the ring's taps through private double-buffered stages.
//   NARROW items (windows inside [-32, 32)): a band of rings of one hemisphere marches through a
//                shared-memory ring of 2R+2S input rows, S rings per pass, so every input row is
//                staged once per band; the window loads of a row use immediate offsets only; a lane
//                owns kNarrowP = 16 outputs so that two CTAs fit an SM (kernel k_convolve_narrow).
// Southern rings use the weights of their northern mirror (A_j and sin t are N/S symmetric).
// ================================================================================================
struct ConvParams {
    const float* in;
    float* out;
    const PairDesc* pairs;
    const Item* items;       // the items of THIS launch (the wide or the narrow part of the work list)
    const float* weights;
    const NarrowRun* runs;   // [n_north - first_narrow][2R+1]
    int n_theta, n_phi, R;
    int first_narrow;        // first northern ring of the narrow class
    uint32_t narrow_w_base;  // its weights start here; one block of wslot floats per narrow ring
    int wslot;               // floats per ring in the (global) narrow weight buffer
    int wcap;                // floats of the weight area in conv_narrow's shared memory
    long long map_stride;    // elements between consecutive maps of a batch
};

// ---- the PTX this file uses, in one place --------------------------------------------------------
// (ARKCOS_HOST_EMU: tests/emu/ compiles this very file for the host to check the index logic of the
//  kernels against the oracle without a GPU; the emulation replaces only these wrappers.)
#ifndef ARKCOS_HOST_EMU
__device__ __forceinline__ void cp_async16(const uint32_t smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_dst), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Shared-memory loads that the compiler may not sink, hoist or drop: they are software prefetches
// issued one step ahead of their first use.
__device__ __forceinline__ void lds128(float& a, float& b, float& c, float& d, const uint32_t addr) {
    asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "r"(addr));
}
template <int OFF>
__device__ __forceinline__ void lds128i(float& a, float& b, float& c, float& d, const uint32_t addr) {
    asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "r"(addr), "n"(OFF));
}
template <int OFF>
__device__ __forceinline__ void lds64i(float& a, float& b, const uint32_t addr) {
    asm volatile("ld.volatile.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(a), "=f"(b) : "r"(addr), "n"(OFF));
}
__device__ __forceinline__ void lds128u(int& a, int& b, int& c, int& d, const uint32_t addr) {
    asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(addr));
}
#else
__device__ __forceinline__ void cp_async16(const uint32_t smem_dst, const void* gmem_src) { emu::cp_async_enqueue(smem_dst, gmem_src); }
__device__ __forceinline__ void cp_async_commit() { emu::cp_async_commit_group(); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { emu::cp_async_wait(N); }
__device__ __forceinline__ void cp_async_wait_all() { emu::cp_async_wait(0); }
__device__ __forceinline__ void lds128(float& a, float& b, float& c, float& d, const uint32_t addr) {
    const float* q = reinterpret_cast<const float*>(emu::smem_read(addr, 16));
    a = q[0]; b = q[1]; c = q[2]; d = q[3];
}
template <int OFF>
__device__ __forceinline__ void lds128i(float& a, float& b, float& c, float& d, const uint32_t addr) { lds128(a, b, c, d, addr + (uint32_t)OFF); }
template <int OFF>
__device__ __forceinline__ void lds64i(float& a, float& b, const uint32_t addr) {
    const float* q = reinterpret_cast<const float*>(emu::smem_read(addr + (uint32_t)OFF, 8));
    a = q[0]; b = q[1];
}
__device__ __forceinline__ void lds128u(int& a, int& b, int& c, int& d, const uint32_t addr) {
    const int* q = reinterpret_cast<const int*>(emu::smem_read(addr, 16));
    a = q[0]; b = q[1]; c = q[2]; d = q[3];
}
#endif

__device__ __forceinline__ int wrap_phi(int phi, int n_phi) {   // phi may be any int; result in [0, n_phi)
    int r = phi % n_phi;
    return r < 0 ? r + n_phi : r;
}

// ------------------------------------------------------------------------------------------------
// WIDE item: one output ring (either hemisphere), F sub-tiles of kWarpSpan outputs x S tap splits.
//
// Every warp is autonomous: it streams ITS share of the ring's taps through two private stage buffers
// filled with cp.async (no CTA barrier until the final reduction of the S splits), so the warps of an
// SM drift apart and the FMA pipe never waits for a common stage hand-over.
//
// Stage layout: logical float m of the stage = x[(phi0 + m) mod n_phi] in the lane-tile layout
// (16-byte chunk c at physical chunk c + (c >> 3)); then the stage's weights, one float per tap.
// ------------------------------------------------------------------------------------------------
constexpr int kZRing = 10;                // register window: 10 chunks = 40 floats (36 live + 4 prefetched)

// One step (4 taps) at window phase PH.  Live chunks q .. q+8 sit in ring slots (PH + c) % 10;
// chunk q+9 is fetched into the slot chunk q-1 has just left, the weights of step q+1 into the other
// half of the weight double buffer.
// Even taps accumulate into a0, odd taps into a1: the register file has two banks (register number
// parity) and an FFMA whose two register operands (accumulator, window float; the weight comes from the
// operand re-use cache) share a bank issues at half rate.  z[m + t] alternates bank with t, so one
// accumulator per output would collide on every other tap; with two sets ptxas places a0[m] opposite
// z[m] and a1[m] opposite z[m + 1].
template <int PH>
__device__ __forceinline__ void wide_step(float (&a0)[kLaneP], float (&a1)[kLaneP], float (&z)[4 * kZRing], float (&w)[2][4],
                                          const uint32_t zlane, const uint32_t ws, const int q) {
    constexpr int B = PH & 1;
    constexpr int N = (4 * (PH + 9)) % (4 * kZRing);
    const int u = q + 9;
    lds128(z[N], z[N + 1], z[N + 2], z[N + 3], zlane + (uint32_t)((u + (u >> 3)) << 4));
    lds128(w[B ^ 1][0], w[B ^ 1][1], w[B ^ 1][2], w[B ^ 1][3], ws + (uint32_t)(16 * q + 16));
#pragma unroll
    for (int t = 0; t < 4; t += 2) {
#pragma unroll
        for (int m = 0; m < kLaneP; m++) a0[m] = fmaf(z[(4 * PH + m + t) % (4 * kZRing)], w[B][t], a0[m]);
#pragma unroll
        for (int m = 0; m < kLaneP; m++) a1[m] = fmaf(z[(4 * PH + m + t + 1) % (4 * kZRing)], w[B][t + 1], a1[m]);
    }
}

// a0[m] + a1[m] += sum_{e < 4 nq} ws[e] * Z[m + e];  zlane / ws: shared-memory addresses of the lane's tile and
// of the stage's weights.
__device__ __forceinline__ void wide_taps(float (&a0)[kLaneP], float (&a1)[kLaneP], const uint32_t zlane, const uint32_t ws, const int nq) {
    float z[4 * kZRing];
#pragma unroll
    for (int c = 0; c < 9; c++) lds128(z[4 * c], z[4 * c + 1], z[4 * c + 2], z[4 * c + 3], zlane + (uint32_t)((c + (c >> 3)) << 4));
    z[36] = z[37] = z[38] = z[39] = 0.f;
    float w[2][4];
    lds128(w[0][0], w[0][1], w[0][2], w[0][3], ws);
    int q = 0;
    for (;;) {
        wide_step<0>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<1>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<2>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<3>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<4>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<5>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<6>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<7>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<8>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
        wide_step<9>(a0, a1, z, w, zlane, ws, q); if (++q == nq) break;
    }
}

struct WideStage {
    const float* row;    // input ring
    int phi0;            // phi of logical float 0 of the stage, in [0, n_phi), multiple of 4
    int nq;              // steps (4 taps each), 1 .. kWideStage/4
    uint32_t w_off;      // first weight of the stage (floats)
};

__device__ void conv_wide(const ConvParams& p, const Item& it, char* smem, const float* in, float* out) {
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int W = 2 * p.R + 1;
    const int i = it.i0;
    const bool mirrored = 2 * i >= p.n_theta;                  // southern ring: weights of its mirror pair
    const int i_n = mirrored ? p.n_theta - 1 - i : i;
    const uint32_t wsm = (uint32_t)__cvta_generic_to_shared(smem) + (uint32_t)(warp * 2 * kWideStageBytes);
    PairDesc* spd = reinterpret_cast<PairDesc*>(smem + (size_t)kWarps * 2 * kWideStageBytes);
    for (int r = threadIdx.x; r < W; r += kThreads) spd[r] = p.pairs[(size_t)i_n * W + r];
    __syncthreads();

    const int K0 = it.k0 + f * kWarpSpan;                      // first output of this warp
    // this warp's share [g_lo, g_hi) of the ring's steps (rows concatenated)
    int G = 0;
    for (int r = 0; r < W; r++) G += spd[r].ntaps >> 2;
    int g_lo = (int)(((long long)G * s) / S), g_hi = (int)(((long long)G * (s + 1)) / S);
    if (K0 >= p.n_phi) g_hi = g_lo;                            // ragged tile: no outputs here
    int r = 0, q = 0, remaining = g_hi - g_lo;
    for (int a = 0; r < W; r++) {
        const int n = spd[r].ntaps >> 2;
        if (g_lo < a + n) { q = g_lo - a; break; }
        a += n;
    }
    auto next_stage = [&](WideStage& st) -> bool {
        if (remaining <= 0) return false;
        while (q >= (spd[r].ntaps >> 2)) { r++; q = 0; }
        const PairDesc pd = spd[r];
        st.nq = min(min(kWideStage / 4, (pd.ntaps >> 2) - q), remaining);
        const int j = mirrored ? i - (r - p.R) : i + (r - p.R);
        st.row = in + (size_t)j * p.n_phi;
        st.phi0 = wrap_phi(K0 + pd.start + 4 * q, p.n_phi);
        st.w_off = pd.w_off + 4u * (uint32_t)q;
        q += st.nq; remaining -= st.nq;
        return true;
    };
    // lane-constant parts of the stage fill: chunk c = lane + 32 n sits at physical chunk
    // (lane + (lane >> 3)) + 36 n, its input at phi0 + 4 lane + 128 n (mod n_phi)
    const int lane_phi = (4 * lane) % p.n_phi, phi_step = 128 % p.n_phi;
    const uint32_t lane_dst = (uint32_t)((lane + (lane >> 3)) << 4);
    auto issue = [&](const WideStage& st, const int b) {
        const uint32_t zb = wsm + (uint32_t)(b * kWideStageBytes);
        const int nchunks = kWarpSpan / 4 + st.nq + 1;
        int phi = st.phi0 + lane_phi;
        if (phi >= p.n_phi) phi -= p.n_phi;
        uint32_t dst = zb + lane_dst;
#pragma unroll 4
        for (int c = lane; c < nchunks; c += 32) {
            cp_async16(dst, st.row + phi);
            dst += 36 * 16;
            phi += phi_step;
            if (phi >= p.n_phi) phi -= p.n_phi;
        }
        const uint32_t wb = zb + kWideZBytes;
        const float* wsrc = p.weights + st.w_off;
        for (int c = lane; c < st.nq; c += 32) cp_async16(wb + 16 * c, wsrc + 4 * c);
        cp_async_commit();
    };

    float a0[kLaneP], a1[kLaneP];
#pragma unroll
    for (int m = 0; m < kLaneP; m++) { a0[m] = 0.f; a1[m] = 0.f; }
    // Blocked summation: after every >= kWideFlushSteps steps the register accumulators are added to a per-lane
    // partial sum in shared memory (outside the hot loop, 0.3 % of its instructions) and restart from zero, so an
    // FP32 chain is at most ~2500 products long whatever the ring band: the polar sums of 1e5 .. 1.5e6 products
    // and the R = 91 regime of the paper stay inside the 1e-6 tolerance (error budget).
    float* part = reinterpret_cast<float*>(smem + (size_t)kWarps * 2 * kWideStageBytes + (size_t)W * sizeof(PairDesc)) + warp * kLaneP * 32 + lane;
    int since = 0;
    bool flushed = false;

    WideStage cur, nxt;
    bool have = next_stage(cur);
    int b = 0;
    if (have) issue(cur, 0);
    while (have) {
        const bool more = next_stage(nxt);
        if (more) { issue(nxt, b ^ 1); cp_async_wait_group<1>(); } else { cp_async_wait_group<0>(); }
        __syncwarp();
        const uint32_t zb = wsm + (uint32_t)(b * kWideStageBytes);
        wide_taps(a0, a1, zb + (uint32_t)(lane * kTileBytes), zb + (uint32_t)kWideZBytes, cur.nq);
        __syncwarp();                                          // buffer b is free for the stage after next
        since += cur.nq;
        if (more && since >= kWideFlushSteps) {                // warp uniform; every lane touches its own words only
#pragma unroll
            for (int m = 0; m < kLaneP; m++) {
                float v = a0[m] + a1[m];
                if (flushed) v += part[m * 32];
                part[m * 32] = v;
                a0[m] = 0.f; a1[m] = 0.f;
            }
            flushed = true; since = 0;
        }
        cur = nxt; have = more; b ^= 1;
    }

    // ---- epilogue: sum the S splits in a fixed order, store float4 ------------------------------------
    float acc[kLaneP];
#pragma unroll
    for (int m = 0; m < kLaneP; m++) acc[m] = a0[m] + a1[m];
    if (flushed) {
#pragma unroll
        for (int m = 0; m < kLaneP; m++) acc[m] += part[m * 32];
    }
    float* orow = out + (size_t)i * p.n_phi;
    if (S == 1) {
        const int phi = K0 + lane * kLaneP;
#pragma unroll
        for (int g = 0; g < kLaneP / 4; g++)
            if (phi + 4 * g < p.n_phi)
                *reinterpret_cast<float4*>(orow + phi + 4 * g) = make_float4(acc[4 * g], acc[4 * g + 1], acc[4 * g + 2], acc[4 * g + 3]);
    } else {
        __syncthreads();                                       // every warp is done with its stage buffers
        float* red = reinterpret_cast<float*>(smem);           // [warp][p][lane]
#pragma unroll
        for (int pp = 0; pp < kLaneP; pp++) red[(warp * kLaneP + pp) * 32 + lane] = acc[pp];
        __syncthreads();
        const int per = (kLaneP / 4) / S;                      // float4 groups of this lane's 32 outputs per split
        for (int g = s * per; g < (s + 1) * per; g++) {
            float o[4];
#pragma unroll
            for (int x = 0; x < 4; x++) {
                float sum = 0.f;
                for (int s2 = 0; s2 < S; s2++) sum += red[((s2 * F + f) * kLaneP + 4 * g + x) * 32 + lane];
                o[x] = sum;
            }
            const int phi = K0 + lane * kLaneP + 4 * g;
            if (phi < p.n_phi) *reinterpret_cast<float4*>(orow + phi) = make_float4(o[0], o[1], o[2], o[3]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// NARROW item: band marching (kernel v5: 16 outputs per lane, two CTAs per SM).
//
// A (ring, input row) run of the narrow class is only 6 .. 32 taps long, so what limits it is not the FFMA
// rate of its inner loop but the latency of its start (descriptor, jump table, window loads); v4 ran it with 32
// outputs per lane in 8 warps per SM and reached 35 % of the FP32 peak (ncu: issue slots 59 % busy, stalls
// wait / short scoreboard / no instruction).  v5 halves the lane's outputs (kNarrowP = 16): 80 instead of 151
// registers and half the shared memory per CTA, so TWO CTAs (16 warps) are resident per SM and cover each
// other's run starts; the unrolled chain shrinks from 35 KB to 18 KB (fits the 32 KB instruction cache level).
//
// Window geometry.  The origin of the tap axis is d = -32 = the start of the tile TWO to the left of the
// lane's own tile (a tile = 16 floats = 4 chunks of 16 bytes, + 1 pad chunk in shared memory).  Step K handles
// taps d = -32 + 2K and d + 1 and needs floats [2K, 2K + 16] of the row = chunks (K >> 1) .. (K >> 1) + 4.
// The register window is a ring of 6 chunks (5 live + 1 prefetched by every EVEN step, two steps ahead of its
// first use, as one conflict-free LDS.128).  A run enters the fully unrolled chain of 32 steps at
// k0 = (32 + start) / 2 and leaves it after ntaps / 2 steps: every shared-memory offset is an immediate.
// ------------------------------------------------------------------------------------------------
constexpr int kNarrowRing = 6;            // chunks of the register window
constexpr int kNarrowSteps = kHaloNarrow; // steps of the chain (2 taps each)

// byte offset of chunk q of the tap axis relative to the lane's own tile
__host__ __device__ constexpr int narrow_chunk_off(int q) { return ((q >> 2) - 2) * kNarrowTileBytes + (q & 3) * 16; }

template <int Q>
__device__ __forceinline__ void narrow_load_chunk(float (&z)[4 * kNarrowRing], const uint32_t zt) {
    constexpr int sl = 4 * (Q % kNarrowRing);
    lds128i<narrow_chunk_off(Q)>(z[sl], z[sl + 1], z[sl + 2], z[sl + 3], zt);
}

template <int K>
__device__ __forceinline__ void narrow_init(float (&z)[4 * kNarrowRing], float (&w)[2][2], const uint32_t zt, const uint32_t wq) {
    constexpr int C = K >> 1;
    narrow_load_chunk<C>(z, zt); narrow_load_chunk<C + 1>(z, zt); narrow_load_chunk<C + 2>(z, zt);
    narrow_load_chunk<C + 3>(z, zt); narrow_load_chunk<C + 4>(z, zt);
    if constexpr ((K & 1) != 0) narrow_load_chunk<C + 5>(z, zt);   // an odd entry step is followed by an even one that needs it
    lds64i<8 * K>(w[K & 1][0], w[K & 1][1], wq);
}

template <int K>
__device__ __forceinline__ void narrow_step(float (&a0)[kNarrowP], float (&a1)[kNarrowP], float (&z)[4 * kNarrowRing], float (&w)[2][2],
                                            const uint32_t zt, const uint32_t wq) {
    if constexpr ((K & 1) == 0) narrow_load_chunk<(K >> 1) + 5>(z, zt);   // first used by step K + 2
    lds64i<8 * (K + 1)>(w[(K + 1) & 1][0], w[(K + 1) & 1][1], wq);
#pragma unroll
    for (int m = 0; m < kNarrowP; m++) a0[m] = fmaf(z[(2 * K + m) % (4 * kNarrowRing)], w[K & 1][0], a0[m]);
#pragma unroll
    for (int m = 0; m < kNarrowP; m++) a1[m] = fmaf(z[(2 * K + m + 1) % (4 * kNarrowRing)], w[K & 1][1], a1[m]);
}

// a0[m] + a1[m] += sum_{e < 2 n} wrow[e] * Z[m + 2 k0 + e],  Z = the row from the start of the tile two to the left.
// zt: shared address of the lane's own tile in the row slot; wq = address of wrow - 8 k0 bytes.
#pragma nv_diag_suppress 177   // the chain's labels past K = 16 are only fallen into
__device__ __forceinline__ void narrow_row(float (&a0)[kNarrowP], float (&a1)[kNarrowP], const uint32_t zt, const uint32_t wq, const int k0, const int n) {
    float z[4 * kNarrowRing];
    float w[2][2];
    const int kend = k0 + n;                                   // the exit test of a step is one compare with an immediate
#define ARKCOS_NR_CASE(K) case K: narrow_init<K>(z, w, zt, wq); goto nr_step_##K;
#define ARKCOS_NR_STEP(K) nr_step_##K: narrow_step<K>(a0, a1, z, w, zt, wq); if (kend == K + 1) goto nr_done;
    switch (k0) {
        ARKCOS_NR_CASE(0) ARKCOS_NR_CASE(1) ARKCOS_NR_CASE(2) ARKCOS_NR_CASE(3) ARKCOS_NR_CASE(4) ARKCOS_NR_CASE(5)
        ARKCOS_NR_CASE(6) ARKCOS_NR_CASE(7) ARKCOS_NR_CASE(8) ARKCOS_NR_CASE(9) ARKCOS_NR_CASE(10) ARKCOS_NR_CASE(11)
        ARKCOS_NR_CASE(12) ARKCOS_NR_CASE(13) ARKCOS_NR_CASE(14) ARKCOS_NR_CASE(15) ARKCOS_NR_CASE(16)
        default: return;
    }
    ARKCOS_NR_STEP(0) ARKCOS_NR_STEP(1) ARKCOS_NR_STEP(2) ARKCOS_NR_STEP(3) ARKCOS_NR_STEP(4) ARKCOS_NR_STEP(5)
    ARKCOS_NR_STEP(6) ARKCOS_NR_STEP(7) ARKCOS_NR_STEP(8) ARKCOS_NR_STEP(9) ARKCOS_NR_STEP(10) ARKCOS_NR_STEP(11)
    ARKCOS_NR_STEP(12) ARKCOS_NR_STEP(13) ARKCOS_NR_STEP(14) ARKCOS_NR_STEP(15) ARKCOS_NR_STEP(16) ARKCOS_NR_STEP(17)
    ARKCOS_NR_STEP(18) ARKCOS_NR_STEP(19) ARKCOS_NR_STEP(20) ARKCOS_NR_STEP(21) ARKCOS_NR_STEP(22) ARKCOS_NR_STEP(23)
    ARKCOS_NR_STEP(24) ARKCOS_NR_STEP(25) ARKCOS_NR_STEP(26) ARKCOS_NR_STEP(27) ARKCOS_NR_STEP(28) ARKCOS_NR_STEP(29)
    ARKCOS_NR_STEP(30) ARKCOS_NR_STEP(31)
nr_done:;
#undef ARKCOS_NR_CASE
#undef ARKCOS_NR_STEP
}
#pragma nv_diag_default 177

// A band of `nr` rings of one hemisphere x a phi tile of kNarrowSpan outputs, in "logical" (northern) ring
// indices lam: the physical ring of logical ring lam is lam (north) or n_theta-1-lam (south); descriptors and
// weights are those of lam.  The band marches through a shared-memory ring of 2R + 2S row slots, S = kWarps rings
// per pass (one warp per ring), so every input row is staged once per band; the S rows, the weight blocks and
// the run descriptors of the NEXT pass are copied by cp.async during the current pass (one barrier per pass).
__device__ void conv_narrow(const ConvParams& p, const Item& it, char* smem, const float* in, float* out) {
    constexpr int S = kWarps;
    const bool south = it.nrings < 0;
    const int nr = south ? -it.nrings : it.nrings;
    const int s = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int W = 2 * p.R + 1;
    const int NS = 2 * p.R + 2 * S;                           // row slots
    constexpr int slot_bytes = kNarrowSlotBytes;
    const uint32_t rows = (uint32_t)__cvta_generic_to_shared(smem);
    // shared memory: row slots | run descriptors [2][S][W] | weight area: [2][S][wstride] if that fits (the tables of
    // the next pass are then copied during the current one), else [S][wstride] (every warp reloads its own ring's
    // block at the start of a pass; only the polar-most bands of the class, whose blocks are the largest)
    const uint32_t pdbuf_addr = rows + (uint32_t)(NS * slot_bytes);
    const uint32_t wbuf_addr = pdbuf_addr + (uint32_t)(2 * S * W * sizeof(NarrowRun));
    const int wstride = it.wcopy + kNarrowWPad;
    const bool dbl = 2 * S * wstride <= p.wcap;
    const int lam0 = it.i0, lam_end = it.i0 + nr;
    const int npass = (nr + S - 1) / S;

    // ---- staging, one warp per row / per ring (all addresses warp uniform except the lane's chunk) ------------
    // chunk idx of a row slot = floats [4 idx, 4 idx + 4) from phi = k0 - 32, at physical chunk idx + (idx >> 2)
    constexpr int row_chunks = kNarrowSpan / 4 + 2 * (kHaloNarrow / 4);     // own tiles + a halo of 32 floats on either side
    const int lane_phi = wrap_phi(it.k0 - kHaloNarrow + 4 * lane, p.n_phi), phi_step = 128 % p.n_phi;
    const uint32_t lane_dst = (uint32_t)((lane + (lane >> 2)) << 4);
    auto stage_row = [&](const int lam_j) {
        if (lam_j < 0 || lam_j >= p.n_theta) return;          // beyond the pole: no ring pair uses it
        const float* row = in + (size_t)(south ? p.n_theta - 1 - lam_j : lam_j) * p.n_phi;
        int sl = lam_j % NS; if (sl < 0) sl += NS;
        uint32_t dst = rows + (uint32_t)(sl * slot_bytes) + lane_dst;
        int phi = lane_phi;
#pragma unroll
        for (int idx = lane; idx < row_chunks; idx += 32) {
            cp_async16(dst, row + phi);
            dst += 40 * 16;                                   // 32 chunks + their 8 pad chunks
            phi += phi_step;
            if (phi >= p.n_phi) phi -= p.n_phi;
        }
    };
    // weights and run descriptors of ring lam -> buffer slot tb (no dependent global loads: both live at
    // computable addresses)
    const int n4 = it.wcopy >> 2;
    auto stage_ring_tables = [&](const int lam, const int tb) {
        if (lam >= lam_end) return;
        const NarrowRun* psrc = p.runs + (size_t)(lam - p.first_narrow) * W;
        const uint32_t pdst = pdbuf_addr + (uint32_t)((tb * W) * sizeof(NarrowRun));
        for (int q = lane; q < W; q += 32) cp_async16(pdst + 16 * q, psrc + q);
        const float* src = p.weights + p.narrow_w_base + (size_t)(lam - p.first_narrow) * p.wslot;
        const uint32_t dst = wbuf_addr + (uint32_t)((tb * wstride) * 4);
        for (int q = lane; q < n4; q += 32) cp_async16(dst + 16 * q, src + 4 * q);
    };
    for (int q = s; q < 2 * p.R + S; q += S) stage_row(lam0 - p.R + q);
    if (dbl) stage_ring_tables(lam0 + s, s);

    const uint32_t lane_tile = (uint32_t)((kHaloNarrow / kNarrowP + lane) * kNarrowTileBytes);
    for (int pass = 0; pass < npass; pass++) {
        const int lbase = lam0 + pass * S;
        cp_async_wait_all();
        __syncthreads();                                      // this pass's rows and tables have landed; pass-1 is done
        const int lam = lbase + s;
        if (!dbl) {                                           // this warp's own tables: nobody else reads buffer s
            stage_ring_tables(lam, s);
            cp_async_wait_all();
            __syncwarp();
        }
        if (pass + 1 < npass) {                               // next pass: S new rows into the slots pass-1 freed
            stage_row(lbase + S + p.R + s);
            if (dbl) stage_ring_tables(lbase + S + s, ((pass + 1) & 1) * S + s);
        }
        if (lam < lam_end) {
            float a0[kNarrowP], a1[kNarrowP];
#pragma unroll
            for (int m = 0; m < kNarrowP; m++) { a0[m] = 0.f; a1[m] = 0.f; }
            const int tb = dbl ? (pass & 1) * S + s : s;
            const uint32_t wring = wbuf_addr + (uint32_t)(tb * wstride * 4);
            const uint32_t spd = pdbuf_addr + (uint32_t)(tb * W * sizeof(NarrowRun));
            int slot = (lam - p.R) % NS; if (slot < 0) slot += NS;
            uint32_t zt = rows + (uint32_t)(slot * slot_bytes) + lane_tile;
            const uint32_t zt_end = rows + (uint32_t)(NS * slot_bytes) + lane_tile;
            // Run descriptors are double buffered in registers: the descriptor of run r+1 is loaded into
            // the other set while run r executes, and only copied out of it one run later.
            int dA[4], dB[4];
            lds128u(dA[0], dA[1], dA[2], dA[3], spd);
#pragma unroll 1
            for (int r = 0; r < W; r++) {
                const uint32_t nxt = spd + (uint32_t)((r + 1 < W ? r + 1 : r) * sizeof(NarrowRun));
                int wq_rel, k0, n;
                if (r & 1) { wq_rel = dB[0]; k0 = dB[1]; n = dB[2]; lds128u(dA[0], dA[1], dA[2], dA[3], nxt); }
                else { wq_rel = dA[0]; k0 = dA[1]; n = dA[2]; lds128u(dB[0], dB[1], dB[2], dB[3], nxt); }
                if (n != 0) narrow_row(a0, a1, zt, wring + (uint32_t)wq_rel, k0, n);
                zt += (uint32_t)slot_bytes;
                if (zt == zt_end) zt -= (uint32_t)(NS * slot_bytes);
            }
            const int phi = it.k0 + lane * kNarrowP;
            float* orow = out + (size_t)(south ? p.n_theta - 1 - lam : lam) * p.n_phi + phi;
#pragma unroll
            for (int g = 0; g < kNarrowP / 4; g++)
                if (phi + 4 * g < p.n_phi)
                    *reinterpret_cast<float4*>(orow + 4 * g) = make_float4(a0[4 * g] + a1[4 * g], a0[4 * g + 1] + a1[4 * g + 1],
                                                                           a0[4 * g + 2] + a1[4 * g + 2], a0[4 * g + 3] + a1[4 * g + 3]);
        }
    }
}

// ---- the two convolution kernels of a launch: WIDE items (1 CTA of 8 warps per SM), NARROW items (2 per SM) ----
// The descriptors were validated on the host (validate_schedule) before they were uploaded; the guards only keep
// a work item that was corrupted in device memory from being turned into addresses.
__global__ void __launch_bounds__(kThreads, 1) k_convolve_wide(const ConvParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ uint4 smem4[];
    char* smem = reinterpret_cast<char*>(smem4);
#else
    char* smem = reinterpret_cast<char*>(emu::g_smem);
#endif
    const Item it = p.items[blockIdx.x];
    if ((unsigned)it.f_log2 > 3u || (unsigned)it.k0 >= (unsigned)p.n_phi || (unsigned)it.i0 >= (unsigned)p.n_theta || it.kind != kWide) return;
    conv_wide(p, it, smem, p.in + (long long)blockIdx.y * p.map_stride, p.out + (long long)blockIdx.y * p.map_stride);
}

__global__ void __launch_bounds__(kThreads, 2) k_convolve_narrow(const ConvParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ uint4 smem4[];
    char* smem = reinterpret_cast<char*>(smem4);
#else
    char* smem = reinterpret_cast<char*>(emu::g_smem);
#endif
    const Item it = p.items[blockIdx.x];
    if ((unsigned)it.k0 >= (unsigned)p.n_phi || (unsigned)it.i0 >= (unsigned)p.n_theta || it.kind != kNarrow || it.nrings == 0) return;
    conv_narrow(p, it, smem, p.in + (long long)blockIdx.y * p.map_stride, p.out + (long long)blockIdx.y * p.map_stride);
}

}  // namespace arkcos
