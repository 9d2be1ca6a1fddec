// arkcos_tensor.cuh - N1(a): the WIDE work items of step S3 on the tensor cores (
// BASELINE.json north_star: "Tensor cores are not used unless a ring-pair circulant is recast as a genuinely
// dense contraction and ncu shows that it wins").  An EXPERIMENT behind ARKCOS_PLAN_WIDE_TENSOR
// (include/arkcos_measure.h); the product's default WIDE kernel is k_convolve_wide (arkcos_kernels.cuh).
// Product code; shares nothing with oracle/.
//
// The contraction.  One stage of a WIDE item is  out[o] += sum_{e < ntaps} w[e] Z[o + e],  o = 0 .. 1023 (the
// outputs of a warp), Z = the staged window of one input ring.  Writing o = 128 nt + 16 a + m  (m = 0..15,
// a = 0..7, nt = 0..7) turns it into eight GEMMs of shape 16 x 8 x K:
//
//     C_nt[m][a] = sum_k T[m][k] X_nt[k][a],   T[m][k] = w[k - m]  (banded Toeplitz, 16 x (ntaps + 15)),
//                                              X_nt[k][a] = Z[128 nt + 16 a + k]  (overlapping-stride view)
//
// T is (ntaps)/(ntaps + 15) dense: with the M = 16 of the warp-level mma every WIDE row (>= 64 taps) is >= 81 %
// dense, where the M = 128 of a tcgen05 tile would need >= 512 taps for the same density.
// The instruction is mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 (the warp-level tensor path; SASS HMMA):
// no descriptors, no TMEM, operands from registers - the Toeplitz fragment of a thread is 8 weights read from
// shared memory once per 16 taps and re-used for all 8 n-tiles, the X fragment one conflict-free LDS.128.
//
// FP32 accuracy from TF32 products (3 x TF32): both operands are split  v = hi + lo  with hi = rna_tf32(v),
// lo = rna_tf32(v - hi), and the product is  hi hi + lo hi + hi lo  (the lo lo term is 2^-22 relative).  The
// tensor core adds with truncation, so a long accumulation inside it drifts; every group of 16 taps is
// therefore accumulated from ZERO inside the tensor core (6 mma: the four small terms first) and added to the
// FP32 accumulator with a plain FADD (round to nearest) - the scheme of Ootomo & Yokota (2022), restated.
// Error against FP64 on the sums of this path (numpy study with emulated TF32 rounding): rel-rms
// 1.2-1.6e-7, inside the north_star tolerance (1e-6); the host emulation of this file is checked against the
// oracle at that tolerance (tests/test_tensor_wide.py).
//
// K order.  The k index of an mma is a dummy, so k slots are assigned to taps such that a thread's operands are
// contiguous: over a group of 16 taps (two mma k blocks) thread t of a quad owns taps 4t .. 4t+3: k block 0
// takes (4t, 4t+1) as its slots (t, t+4), k block 1 takes (4t+2, 4t+3).
//
// Fragment layout of mma.m16n8k8 .tf32 (PTX ISA "Matrix Fragments for mma.m16n8k8"; g = lane >> 2, t = lane & 3):
//     A (16 x 8, row):  a0 = A[g][t]      a1 = A[g+8][t]    a2 = A[g][t+4]    a3 = A[g+8][t+4]
//     B ( 8 x 8, col):  b0 = B[t][g]      b1 = B[t+4][g]
//     C (16 x 8):       c0 = C[g][2t]     c1 = C[g][2t+1]   c2 = C[g+8][2t]   c3 = C[g+8][2t+1]
#pragma once
#include "arkcos_kernels.cuh"

namespace arkcos {

// Stage layout of the tensor path (same stage size as conv_wide, kWideStageBytes): the input window LINEAR
// (float x at byte 4x: the LDS.128 of a quarter warp reads 128 contiguous bytes), then the weights with
// kTcLead zero floats before (rows m > k of the Toeplitz) and kTcTail zero floats after them.
constexpr int kTcLead = 16;
constexpr int kTcTail = 32;
constexpr int kTcZBytes = kWideZChunks * 16;
constexpr int kTcWBytes = (kTcLead + kWideStage + kTcTail) * 4;
static_assert(kTcZBytes + kTcWBytes <= kWideStageBytes, "the tensor path's stage must fit the WIDE stage buffers");
static_assert(kWarpSpan / 4 + kWideStage / 4 + 8 <= kWideZChunks, "input window of a stage + the 32 floats the last k group over-reads");

#ifndef ARKCOS_HOST_EMU
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t a0, const uint32_t a1, const uint32_t a2, const uint32_t a3,
                                         const uint32_t b0, const uint32_t b1) {
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%0, %1, %2, %3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// plain shared-memory accesses through the generic pointer (ordered by the "memory" clobbers of the cp.async
// wrappers and by __syncwarp / __syncthreads; the compiler is free to schedule them inside a stage)
__device__ __forceinline__ float4 tc_lds128(const char* smem, const uint32_t off) { return *reinterpret_cast<const float4*>(smem + off); }
__device__ __forceinline__ float tc_lds32(const char* smem, const uint32_t off) { return *reinterpret_cast<const float*>(smem + off); }
__device__ __forceinline__ void tc_sts128_zero(char* smem, const uint32_t off) { *reinterpret_cast<float4*>(smem + off) = make_float4(0.f, 0.f, 0.f, 0.f); }
#else
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t a0, const uint32_t a1, const uint32_t a2, const uint32_t a3,
                                         const uint32_t b0, const uint32_t b1) { emu::mma_m16n8k8_tf32(c, a0, a1, a2, a3, b0, b1); }
__device__ __forceinline__ float4 tc_lds128(const char*, const uint32_t off) {
    const float* q = reinterpret_cast<const float*>(emu::smem_read(off, 16));
    return make_float4(q[0], q[1], q[2], q[3]);
}
__device__ __forceinline__ float tc_lds32(const char*, const uint32_t off) { return *reinterpret_cast<const float*>(emu::smem_read(off, 4)); }
__device__ __forceinline__ void tc_sts128_zero(char*, const uint32_t off) { std::memset(emu::smem_write(off, 16), 0, 16); }
#endif

// v = hi + lo, both exactly representable in TF32 (10 mantissa bits; the tensor core reads the upper 19 bits of a
// register): round to nearest, ties away from zero = what cvt.rna.tf32.f32 does, written as two full-rate integer
// instructions (add half an ulp of TF32 to the magnitude, clear the 13 low bits); v - hi is exact in FP32.
__device__ __forceinline__ uint32_t tc_round_tf32(const float v) { return (__float_as_uint(v) + 0x1000u) & 0xFFFFE000u; }
__device__ __forceinline__ void tc_split(const float v, uint32_t& hi, uint32_t& lo) {
    hi = tc_round_tf32(v);
    lo = tc_round_tf32(v - __uint_as_float(hi));
}

// acc[4 nt + c] += sum_{e < 4 nq} w[e] Z[o + e]  for the four outputs o = 128 nt + 16 (2t + (c & 1)) + g + 8 (c >> 1)
// this thread holds of n-tile nt.  zoff / woff: byte offsets, in the CTA's shared memory, of the stage's input
// window and of its weight area (kTcLead zeros, the 4 nq weights, kTcTail zeros).
__device__ __forceinline__ void tc_taps(float (&acc)[kLaneP], const char* smem, const uint32_t zoff, const uint32_t woff, const int nq, const int lane) {
    const int g = lane >> 2, t = lane & 3;
    const int ngroups = (4 * nq + 15 + 15) >> 4;               // groups of 16 k: k = 0 .. 4 nq + 14
    const uint32_t zt = zoff + (uint32_t)(4 * (16 * g + 4 * t));
    uint32_t wt = woff + (uint32_t)(4 * (kTcLead + 4 * t - g));   // w[16 kk + 4 t - g]; rows g + 8: 8 floats below
#pragma unroll 1
    for (int kk = 0; kk < ngroups; kk++) {
        uint32_t ah[8], al[8];                                 // [2 i + row half], i = tap 4t + i of the group
#pragma unroll
        for (int i = 0; i < 4; i++) {
            tc_split(tc_lds32(smem, wt + 4 * i), ah[2 * i], al[2 * i]);
            tc_split(tc_lds32(smem, wt + 4 * i - 32), ah[2 * i + 1], al[2 * i + 1]);
        }
        const uint32_t zk = zt + (uint32_t)(64 * kk);
#pragma unroll
        for (int nt = 0; nt < 8; nt++) {
            const float4 z = tc_lds128(smem, zk + (uint32_t)(512 * nt));
            uint32_t bh[4], bl[4];
            tc_split(z.x, bh[0], bl[0]); tc_split(z.y, bh[1], bl[1]); tc_split(z.z, bh[2], bl[2]); tc_split(z.w, bh[3], bl[3]);
            float c[4] = {0.f, 0.f, 0.f, 0.f};
            mma_tf32(c, al[0], al[1], al[2], al[3], bh[0], bh[1]);     // small terms first
            mma_tf32(c, al[4], al[5], al[6], al[7], bh[2], bh[3]);
            mma_tf32(c, ah[0], ah[1], ah[2], ah[3], bl[0], bl[1]);
            mma_tf32(c, ah[4], ah[5], ah[6], ah[7], bl[2], bl[3]);
            mma_tf32(c, ah[0], ah[1], ah[2], ah[3], bh[0], bh[1]);
            mma_tf32(c, ah[4], ah[5], ah[6], ah[7], bh[2], bh[3]);
#pragma unroll
            for (int x = 0; x < 4; x++) acc[4 * nt + x] += c[x];
        }
        wt += 64;
    }
}

// One WIDE item (as conv_wide: one output ring, F sub-tiles of kWarpSpan outputs x S tap splits, every warp
// streaming its share of the ring's taps through two private cp.async stages) with the taps of a stage applied
// by tc_taps.  Same work items, same pair descriptors, same FP32 weight buffer as conv_wide.
__device__ void conv_wide_tc(const ConvParams& p, const Item& it, char* smem, const float* in, float* out) {
    const int F = 1 << it.f_log2, S = kWarps >> it.f_log2;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int f = warp & (F - 1), s = warp >> it.f_log2;
    const int W = 2 * p.R + 1;
    const int i = it.i0;
    const bool mirrored = 2 * i >= p.n_theta;
    const int i_n = mirrored ? p.n_theta - 1 - i : i;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t woff0 = (uint32_t)(warp * 2 * kWideStageBytes);            // this warp's two stages, offset in the CTA's shared memory
    PairDesc* spd = reinterpret_cast<PairDesc*>(smem + (size_t)kWarps * 2 * kWideStageBytes);
    for (int r = threadIdx.x; r < W; r += kThreads) spd[r] = p.pairs[(size_t)i_n * W + r];
    // the kTcLead zero floats in front of either stage's weights are written once
    if (lane < 2 * (kTcLead / 4)) tc_sts128_zero(smem, woff0 + (uint32_t)((lane & 1) * kWideStageBytes + kTcZBytes + 16 * (lane >> 1)));
    __syncthreads();

    const int K0 = it.k0 + f * kWarpSpan;
    int G = 0;
    for (int r = 0; r < W; r++) G += spd[r].ntaps >> 2;
    int g_lo = (int)(((long long)G * s) / S), g_hi = (int)(((long long)G * (s + 1)) / S);
    if (K0 >= p.n_phi) g_hi = g_lo;
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
    const int lane_phi = (4 * lane) % p.n_phi, phi_step = 128 % p.n_phi;
    auto issue = [&](const WideStage& st, const int b) {
        const uint32_t zb = woff0 + (uint32_t)(b * kWideStageBytes);
        const int nchunks = kWarpSpan / 4 + st.nq + 8;         // the last k group reads up to 32 floats past the window
        int phi = st.phi0 + lane_phi;
        if (phi >= p.n_phi) phi -= p.n_phi;
        uint32_t dst = sbase + zb + (uint32_t)(16 * lane);
#pragma unroll 4
        for (int c = lane; c < nchunks; c += 32) {
            cp_async16(dst, st.row + phi);
            dst += 32 * 16;
            phi += phi_step;
            if (phi >= p.n_phi) phi -= p.n_phi;
        }
        const uint32_t wb = zb + (uint32_t)(kTcZBytes + 4 * kTcLead);
        const float* wsrc = p.weights + st.w_off;
        for (int c = lane; c < st.nq; c += 32) cp_async16(sbase + wb + 16 * c, wsrc + 4 * c);
        if (lane < kTcTail / 4) tc_sts128_zero(smem, wb + (uint32_t)(16 * (st.nq + lane)));
        cp_async_commit();
    };

    float acc[kLaneP];
#pragma unroll
    for (int m = 0; m < kLaneP; m++) acc[m] = 0.f;
    // blocked summation as in conv_wide: the FP32 accumulators (one FADD per 16 taps) are flushed to per-lane partial
    // sums in shared memory after every full stage, so a chain is ~32 additions long whatever the ring band
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
        const uint32_t zb = woff0 + (uint32_t)(b * kWideStageBytes);
        tc_taps(acc, smem, zb, zb + (uint32_t)kTcZBytes, cur.nq, lane);
        __syncwarp();
        since += cur.nq;
        if (more && since >= kWideFlushSteps) {                // warp uniform; every lane touches its own words only
#pragma unroll
            for (int m = 0; m < kLaneP; m++) {
                float v = acc[m];
                if (flushed) v += part[m * 32];
                part[m * 32] = v;
                acc[m] = 0.f;
            }
            flushed = true; since = 0;
        }
        cur = nxt; have = more; b ^= 1;
    }
    if (flushed) {
#pragma unroll
        for (int m = 0; m < kLaneP; m++) acc[m] += part[m * 32];
    }

    // ---- epilogue: acc[4 nt + c] is output K0 + 128 nt + 32 t + 16 (c & 1) + 8 (c >> 1) + g --------------------
    const int g = lane >> 2, t = lane & 3;
    float* orow = out + (size_t)i * p.n_phi;
    const int phi_t = K0 + 32 * t + g;
    if (S == 1) {
#pragma unroll
        for (int x = 0; x < kLaneP; x++) {
            const int phi = phi_t + 128 * (x >> 2) + 16 * (x & 1) + 8 * ((x >> 1) & 1);
            if (phi < p.n_phi) orow[phi] = acc[x];
        }
    } else {
        __syncthreads();
        float* red = reinterpret_cast<float*>(smem);           // [warp][register][lane]
#pragma unroll
        for (int x = 0; x < kLaneP; x++) red[(warp * kLaneP + x) * 32 + lane] = acc[x];
        __syncthreads();
        const int per = kLaneP / S;                            // registers summed and stored by this split
        for (int x = s * per; x < (s + 1) * per; x++) {
            float sum = 0.f;
            for (int s2 = 0; s2 < S; s2++) sum += red[((s2 * F + f) * kLaneP + x) * 32 + lane];
            const int phi = phi_t + 128 * (x >> 2) + 16 * (x & 1) + 8 * ((x >> 1) & 1);
            if (phi < p.n_phi) orow[phi] = sum;
        }
    }
}

__global__ void __launch_bounds__(kThreads, 1) k_convolve_wide_tc(const ConvParams p) {
#ifndef ARKCOS_HOST_EMU
    extern __shared__ uint4 smem4[];
    char* smem = reinterpret_cast<char*>(smem4);
#else
    char* smem = reinterpret_cast<char*>(emu::g_smem);
#endif
    const Item it = p.items[blockIdx.x];
    if ((unsigned)it.f_log2 > 3u || (unsigned)it.k0 >= (unsigned)p.n_phi || (unsigned)it.i0 >= (unsigned)p.n_theta || it.kind != kWide) return;
    conv_wide_tc(p, it, smem, p.in + (long long)blockIdx.y * p.map_stride, p.out + (long long)blockIdx.y * p.map_stride);
}

}  // namespace arkcos
