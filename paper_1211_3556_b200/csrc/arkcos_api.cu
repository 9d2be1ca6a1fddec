// arkcos_api.cu - the C ABI of include/arkcos.h: plan creation (S1 + uploads), the hot-path launches
// (S2 weight generator, S3 convolution) and the introspection / measurement hooks.
// Product code; shares nothing with oracle/.  No CPU fallback: compute entry points need a CUDA device.
#ifdef ARKCOS_HOST_EMU
#include "emu_runtime.h"   // tests/emu: the CUDA runtime emulated on the host (test builds only, never the product)
#define ARKCOS_LAUNCH(kernel, grid, block, smem, stream, params) emu::launch(kernel, dim3(grid), dim3(block), (size_t)(smem), params)
#else
#include <cuda_runtime.h>
#define ARKCOS_LAUNCH(kernel, grid, block, smem, stream, params) kernel<<<grid, block, smem, stream>>>(params)
#endif

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/arkcos.h"
#include "../../include/arkcos_measure.h"
#include "../../include/arkcos_spectral.h"
#include "arkcos_internal.h"
#include "arkcos_kernels.cuh"
#include "arkcos_spectral.cuh"
#include "arkcos_tensor.cuh"

using namespace arkcos;

namespace {
thread_local std::string g_last_cuda_error;

bool cuda_ok(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return true;
    g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
    (void)cudaGetLastError();
    return false;
}
#define CU(call) do { if (!cuda_ok((call), #call)) return ARKCOS_ECUDA; } while (0)
}  // namespace

struct arkcos_plan {
    Schedule sched;
    std::vector<double> table;
    int n_table = 0;
    int m_split = 0;                  // two-zone table (arkcos_plan_create_biased); 0 = uniform
    double theta_split = 0.0;
    unsigned flags = 0;
    int device = -1, sm_count = 0;
    bool weights_ready = false;       // cached plans: generator already ran
    // device memory
    PairDesc* d_pairs = nullptr;
    Item* d_items = nullptr;
    GenUnit* d_units = nullptr;
    double *d_s2 = nullptr, *d_table = nullptr;
    NarrowRun* d_runs = nullptr;
    float* d_weights = nullptr;
    float *d_io_in = nullptr, *d_io_out = nullptr;   // arkcos_convolve_host staging (arkcos_plan_reserve_host_io)
    // arkcos_convolve_host pipeline (arkcos_plan_reserve_host_io)
    Pipeline pipe;
    Item* d_pipe_items = nullptr;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    std::vector<cudaEvent_t> ev_h2d, ev_comp;
    cudaEvent_t ev_fork = nullptr;
    // N2, spectral path (ARKCOS_PLAN_SPECTRAL)
    float* d_wspec = nullptr;         // [n_north][2R+1][n_phi/2+1] What_ij[m] * 2/n
    float2 *d_tw_h = nullptr, *d_tw_n = nullptr;
    size_t device_bytes = 0;
    size_t gen_smem = 0;
    int gen_grid = 0, table_in_smem = 0;
};

namespace {

template <typename T>
arkcos_status upload(size_t* counter, T** dst, const std::vector<T>& src) {
    size_t bytes = src.size() * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    cudaError_t e = cudaMalloc((void**)dst, bytes);
    if (e == cudaErrorMemoryAllocation) { (void)cudaGetLastError(); return ARKCOS_ENOMEM; }
    CU(e);
    *counter += bytes;
    if (!src.empty()) CU(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return ARKCOS_OK;
}
template <typename T>
arkcos_status upload(arkcos_plan* pl, T** dst, const std::vector<T>& src) { return upload(&pl->device_bytes, dst, src); }

arkcos_status launch_generate(const arkcos_plan* pl, cudaStream_t st) {
    GenParams g;
    g.units = pl->d_units; g.s2 = pl->d_s2; g.table = pl->d_table; g.weights = pl->d_weights;
    g.n_units = (int)pl->sched.gen_units.size(); g.n_phi = pl->sched.n_phi; g.n_table = pl->n_table;
    g.t_scale = (double)(pl->n_table - 1) / pl->sched.theta_cut;
    g.m_split = pl->m_split; g.theta_split = pl->theta_split; g.t_scale2 = 0.0;
    if (pl->m_split > 0) {
        g.t_scale = (double)pl->m_split / pl->theta_split;
        g.t_scale2 = (double)(pl->n_table - 1 - pl->m_split) / (pl->sched.theta_cut - pl->theta_split);
    }
    g.table_in_smem = pl->table_in_smem;
    ARKCOS_LAUNCH(k_generate_weights, pl->gen_grid, kGenThreads, pl->gen_smem, st, g);
    CU(cudaGetLastError());
    return ARKCOS_OK;
}

ConvParams conv_params(const arkcos_plan* pl, const float* d_in, float* d_out) {
    const Schedule& s = pl->sched;
    ConvParams c;
    c.in = d_in; c.out = d_out; c.pairs = pl->d_pairs; c.items = pl->d_items; c.weights = pl->d_weights;
    c.runs = pl->d_runs; c.first_narrow = s.first_narrow; c.narrow_w_base = s.narrow_w_base;
    c.n_theta = s.n_theta; c.n_phi = s.n_phi; c.R = s.R; c.wslot = s.narrow_wslot; c.wcap = s.narrow_wcap;
    c.map_stride = (long long)s.n_theta * s.n_phi;
    return c;
}

// n_wide WIDE items at `wide`, n_narrow NARROW items at `narrow` (device pointers), back to back on `st`
arkcos_status launch_items(const arkcos_plan* pl, ConvParams c, const Item* wide, int n_wide, const Item* narrow, int n_narrow,
                           int n_maps, cudaStream_t st) {
    if (pl->flags & ARKCOS_PLAN_ONLY_NARROW) n_wide = 0;
    if (pl->flags & ARKCOS_PLAN_ONLY_WIDE) n_narrow = 0;
    if (n_wide > 0) {
        c.items = wide;
        if (pl->flags & ARKCOS_PLAN_WIDE_TENSOR)                  // N1(a): the same items on the tensor cores
            ARKCOS_LAUNCH(k_convolve_wide_tc, dim3((unsigned)n_wide, (unsigned)n_maps, 1), kThreads, pl->sched.smem_wide, st, c);
        else
            ARKCOS_LAUNCH(k_convolve_wide, dim3((unsigned)n_wide, (unsigned)n_maps, 1), kThreads, pl->sched.smem_wide, st, c);
        CU(cudaGetLastError());
    }
    if (n_narrow > 0) {
        c.items = narrow;
        ARKCOS_LAUNCH(k_convolve_narrow, dim3((unsigned)n_narrow, (unsigned)n_maps, 1), kThreads, pl->sched.smem_narrow, st, c);
        CU(cudaGetLastError());
    }
    return ARKCOS_OK;
}

// S3 / S3w: the WIDE items (k_convolve_wide, one CTA per SM) and the NARROW items (k_convolve_narrow, two CTAs per
// SM) of the plan, back to back on the caller's stream.  The two kernels write disjoint output rings.
arkcos_status launch_convolve(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps, cudaStream_t st) {
    const Schedule& s = pl->sched;
    return launch_items(pl, conv_params(pl, d_in, d_out), pl->d_items, s.n_wide_items, pl->d_items + s.n_wide_items,
                        (int)s.items.size() - s.n_wide_items, n_maps, st);
}

// N2: the weight spectra What_ij[m] of every northern ring pair, once per plan (FP64 on the device, rounded to FP32)
arkcos_status build_spectral(arkcos_plan* pl) {
    const Schedule& s = pl->sched;
    const int n = s.n_phi, h = n / 2, W = 2 * s.R + 1;
    const double kPi = 3.14159265358979323846264338327950288;
    std::vector<SpecPair> sp((size_t)s.n_north * W);
    for (int i = 0; i < s.n_north; i++)
        for (int r = 0; r < W; r++) {
            const int j = i + r - s.R;
            SpecPair& g = sp[(size_t)i * W + r];
            g.half = s.pairs[(size_t)i * W + r].half; g.pad_ = 0;
            const bool live = g.half >= 0 && j >= 0 && j < s.n_theta;
            g.a = s.a_r[std::abs(r - s.R)]; g.b = live ? s.sin_t[i] * s.sin_t[j] : 0.0; g.area = live ? s.area[j] : 0.0;
            if (!live) g.half = -1;
        }
    std::vector<double> costab(n);
    for (int k = 0; k < n; k++) costab[k] = std::cos(2.0 * kPi * k / n);
    std::vector<float2> tw_h(std::max(1, h / 2)), tw_n(h + 1);
    for (int k = 0; k < h / 2; k++) tw_h[k] = make_float2((float)std::cos(2.0 * kPi * k / h), (float)-std::sin(2.0 * kPi * k / h));
    for (int m = 0; m <= h; m++) tw_n[m] = make_float2((float)std::cos(2.0 * kPi * m / n), (float)-std::sin(2.0 * kPi * m / n));
    SpecPair* d_sp = nullptr; double* d_cos = nullptr;
    arkcos_status st = ARKCOS_OK;
    do {
        if ((st = upload(pl, &pl->d_tw_h, tw_h)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_tw_n, tw_n)) != ARKCOS_OK) break;
        size_t tmp_bytes = 0;                                     // temporaries of this function, not plan memory
        if ((st = upload(&tmp_bytes, &d_sp, sp)) != ARKCOS_OK) break;
        if ((st = upload(&tmp_bytes, &d_cos, costab)) != ARKCOS_OK) break;
        const size_t bytes = sp.size() * (size_t)(h + 1) * sizeof(float);
        cudaError_t e = cudaMalloc((void**)&pl->d_wspec, bytes);
        if (e == cudaErrorMemoryAllocation) { (void)cudaGetLastError(); st = ARKCOS_ENOMEM; break; }
        if (!cuda_ok(e, "cudaMalloc(wspec)")) { st = ARKCOS_ECUDA; break; }
        pl->device_bytes += bytes;
        SpecWeightParams w;
        w.pairs = d_sp; w.s2 = pl->d_s2; w.table = pl->d_table; w.costab = d_cos; w.wspec = pl->d_wspec;
        w.n_pairs = (int)sp.size(); w.n_phi = n; w.n_table = pl->n_table;
        w.t_scale = (double)(pl->n_table - 1) / s.theta_cut; w.m_split = pl->m_split; w.theta_split = pl->theta_split; w.t_scale2 = 0.0;
        if (pl->m_split > 0) {
            w.t_scale = (double)pl->m_split / pl->theta_split;
            w.t_scale2 = (double)(pl->n_table - 1 - pl->m_split) / (s.theta_cut - pl->theta_split);
        }
        const size_t smem = (size_t)(h + 1) * sizeof(double);
        if (!cuda_ok(cudaFuncSetAttribute(k_spectral_weights, cudaFuncAttributeMaxDynamicSharedMemorySize, (kSpecMaxPhi / 2 + 1) * 8),
                     "cudaFuncSetAttribute(k_spectral_weights)") ||
            !cuda_ok(cudaFuncSetAttribute(k_rfft_rings, cudaFuncAttributeMaxDynamicSharedMemorySize, kSpecMaxPhi * 10 + 16),
                     "cudaFuncSetAttribute(k_rfft_rings)") ||
            !cuda_ok(cudaFuncSetAttribute(k_spectral_apply, cudaFuncAttributeMaxDynamicSharedMemorySize, kSpecMaxPhi * 10 + 16),
                     "cudaFuncSetAttribute(k_spectral_apply)")) { st = ARKCOS_ECUDA; break; }
        const int grid = std::min<int>((int)sp.size(), 8 * std::max(1, pl->sm_count));
        ARKCOS_LAUNCH(k_spectral_weights, grid, kSpecThreads, smem, 0, w);
        if (!cuda_ok(cudaGetLastError(), "k_spectral_weights") || !cuda_ok(cudaDeviceSynchronize(), "k_spectral_weights sync")) { st = ARKCOS_ECUDA; break; }
    } while (0);
    cudaFree(d_sp); cudaFree(d_cos);
    return st;
}

arkcos_status check_io(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps) {
    if (!pl || !d_in || !d_out || n_maps < 1) return ARKCOS_EINVAL;
    if (pl->flags & ARKCOS_PLAN_HOST_ONLY) return ARKCOS_EUNSUPPORTED;
    int dev = -1;
    if (!cuda_ok(cudaGetDevice(&dev), "cudaGetDevice")) return ARKCOS_ECUDA;
    if (dev != pl->device) return ARKCOS_EINVAL;                // the plan's memory lives on another device
    if (((uintptr_t)d_in & 15u) || ((uintptr_t)d_out & 15u)) return ARKCOS_EINVAL;
    const size_t bytes = (size_t)n_maps * pl->sched.n_theta * pl->sched.n_phi * sizeof(float);
    const uintptr_t a = (uintptr_t)d_in, b = (uintptr_t)d_out;
    if (a < b + bytes && b < a + bytes) return ARKCOS_EINVAL;   // overlap
    return ARKCOS_OK;
}

arkcos_status run(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps, cudaStream_t st) {
    const bool cached = (pl->flags & ARKCOS_PLAN_CACHE_WEIGHTS) != 0;
    if (!cached) { arkcos_status s = launch_generate(pl, st); if (s != ARKCOS_OK) return s; }
    return launch_convolve(pl, d_in, d_out, n_maps, st);
}

}  // namespace

extern "C" {

const char* arkcos_status_string(arkcos_status s) {
    switch (s) {
        case ARKCOS_OK: return "ARKCOS_OK";
        case ARKCOS_EINVAL: return "ARKCOS_EINVAL: invalid argument";
        case ARKCOS_ENOMEM: return "ARKCOS_ENOMEM: out of memory";
        case ARKCOS_ECUDA: return "ARKCOS_ECUDA: CUDA runtime error";
        case ARKCOS_EUNSUPPORTED: return "ARKCOS_EUNSUPPORTED: not supported by this build";
        case ARKCOS_EINTERNAL: return "ARKCOS_EINTERNAL: the schedule failed its own validation";
    }
    return "ARKCOS_?: unknown status";
}

const char* arkcos_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

arkcos_status arkcos_plan_destroy(arkcos_plan* pl) {
    if (!pl) return ARKCOS_OK;
    if (!(pl->flags & ARKCOS_PLAN_HOST_ONLY)) {
        cudaFree(pl->d_pairs); cudaFree(pl->d_items); cudaFree(pl->d_units); cudaFree(pl->d_runs); cudaFree(pl->d_s2); cudaFree(pl->d_table);
        cudaFree(pl->d_weights); cudaFree(pl->d_io_in); cudaFree(pl->d_io_out);
        cudaFree(pl->d_wspec); cudaFree(pl->d_tw_h); cudaFree(pl->d_tw_n); cudaFree(pl->d_pipe_items);
        for (auto& e : pl->ev_h2d) if (e) cudaEventDestroy(e);
        for (auto& e : pl->ev_comp) if (e) cudaEventDestroy(e);
        if (pl->ev_fork) cudaEventDestroy(pl->ev_fork);
        if (pl->s_h2d) cudaStreamDestroy(pl->s_h2d);
        if (pl->s_d2h) cudaStreamDestroy(pl->s_d2h);
        (void)cudaGetLastError();
    }
    delete pl;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_create_ex(arkcos_plan** plan, int n_theta, int n_phi, const double* k_table, int n_table,
                                    double theta_cut, unsigned flags) {
    return arkcos_plan_create_biased(plan, n_theta, n_phi, k_table, n_table, theta_cut, 0, 0.0, flags);
}

arkcos_status arkcos_plan_create_biased(arkcos_plan** plan, int n_theta, int n_phi, const double* k_table, int n_table,
                                        double theta_cut, int m_split, double theta_split, unsigned flags) {
    if (!plan) return ARKCOS_EINVAL;
    *plan = nullptr;
    if (m_split < 0) return ARKCOS_EINVAL;
    if (m_split > 0 && (m_split > n_table - 2 || !(theta_split > 0.0) || !(theta_split < theta_cut))) return ARKCOS_EINVAL;
    if (!k_table || n_table < 2 || n_theta < 1 || n_phi < 1) return ARKCOS_EINVAL;
    if (!(theta_cut > 0.0) || !std::isfinite(theta_cut)) return ARKCOS_EINVAL;
    if (flags & ~(ARKCOS_PLAN_HOST_ONLY | ARKCOS_PLAN_CACHE_WEIGHTS | ARKCOS_PLAN_ONLY_WIDE | ARKCOS_PLAN_ONLY_NARROW | ARKCOS_PLAN_SPECTRAL |
                  ARKCOS_PLAN_WIDE_TENSOR | ARKCOS_PLAN_ALL_WIDE)) return ARKCOS_EINVAL;
    if ((flags & ARKCOS_PLAN_SPECTRAL) && (n_phi < 16 || n_phi > kSpecMaxPhi || (n_phi & (n_phi - 1)) != 0)) return ARKCOS_EUNSUPPORTED;
    if ((flags & ARKCOS_PLAN_ONLY_WIDE) && (flags & ARKCOS_PLAN_ONLY_NARROW)) return ARKCOS_EINVAL;
    for (int m = 0; m < n_table; m++) if (!std::isfinite(k_table[m])) return ARKCOS_EINVAL;
    arkcos_plan* pl = new (std::nothrow) arkcos_plan();
    if (!pl) return ARKCOS_ENOMEM;
    pl->flags = flags; pl->n_table = n_table;
    pl->m_split = m_split; pl->theta_split = m_split > 0 ? theta_split : 0.0;
    arkcos_status st = ARKCOS_OK;
    try {
        pl->table.assign(k_table, k_table + n_table);
        if (!(flags & ARKCOS_PLAN_HOST_ONLY)) {
            cudaDeviceProp prop;
            if (!cuda_ok(cudaGetDevice(&pl->device), "cudaGetDevice") ||
                !cuda_ok(cudaGetDeviceProperties(&prop, pl->device), "cudaGetDeviceProperties")) {
                delete pl; return ARKCOS_ECUDA;
            }
            pl->sm_count = prop.multiProcessorCount;
            if (prop.major < 10) { g_last_cuda_error = "arkcos needs an sm_100 class device"; delete pl; return ARKCOS_EUNSUPPORTED; }
        }
        int rc = build_schedule(n_theta, n_phi, theta_cut, pl->sm_count, pl->sched, (flags & ARKCOS_PLAN_ALL_WIDE) != 0);
        if (rc != 0) { delete pl; return (arkcos_status)rc; }
    } catch (const std::bad_alloc&) { delete pl; return ARKCOS_ENOMEM; }
    if (flags & ARKCOS_PLAN_HOST_ONLY) { *plan = pl; return ARKCOS_OK; }

    const Schedule& s = pl->sched;
    do {
        if ((st = upload(pl, &pl->d_pairs, s.pairs)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_items, s.items)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_units, s.gen_units)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_runs, s.runs)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_s2, s.s2)) != ARKCOS_OK) break;
        if ((st = upload(pl, &pl->d_table, pl->table)) != ARKCOS_OK) break;
        {
            size_t bytes = (size_t)s.weight_slots * sizeof(float) + 16;
            cudaError_t e = cudaMalloc((void**)&pl->d_weights, bytes);
            if (e == cudaErrorMemoryAllocation) { (void)cudaGetLastError(); st = ARKCOS_ENOMEM; break; }
            if (!cuda_ok(e, "cudaMalloc(weights)")) { st = ARKCOS_ECUDA; break; }
            pl->device_bytes += bytes;
            // gaps between ring blocks and window padding stay zero for the life of the plan.  The memset runs on
            // the legacy default stream, which non-blocking user streams do not wait for: finish it here.
            if (!cuda_ok(cudaMemset(pl->d_weights, 0, bytes), "cudaMemset(weights)") ||
                !cuda_ok(cudaDeviceSynchronize(), "cudaDeviceSynchronize(weights)")) { st = ARKCOS_ECUDA; break; }
        }
        // launch configuration.  The dynamic shared-memory limit is an attribute of the KERNEL, shared by every
        // plan of the process: always set it to the library's maximum, never to this plan's own size (a later,
        // smaller plan must not lower it under an earlier plan's launches).
        if (!cuda_ok(cudaFuncSetAttribute(k_convolve_wide, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBudget),
                     "cudaFuncSetAttribute(k_convolve_wide)") ||
            !cuda_ok(cudaFuncSetAttribute(k_convolve_wide_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBudget),
                     "cudaFuncSetAttribute(k_convolve_wide_tc)") ||
            !cuda_ok(cudaFuncSetAttribute(k_convolve_narrow, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBudget),
                     "cudaFuncSetAttribute(k_convolve_narrow)") ||
            // two NARROW CTAs of up to kSmemTwoPerSm share an SM only with the largest shared-memory carve-out
            !cuda_ok(cudaFuncSetAttribute(k_convolve_narrow, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared),
                     "cudaFuncSetAttribute(k_convolve_narrow, carveout)")) { st = ARKCOS_ECUDA; break; }
        size_t tab_bytes = (size_t)n_table * sizeof(double);
        pl->table_in_smem = tab_bytes <= (size_t)kGenSmemMax ? 1 : 0;
        pl->gen_smem = pl->table_in_smem ? tab_bytes : 0;
        if (!cuda_ok(cudaFuncSetAttribute(k_generate_weights, cudaFuncAttributeMaxDynamicSharedMemorySize, kGenSmemMax),
                     "cudaFuncSetAttribute(k_generate_weights)")) { st = ARKCOS_ECUDA; break; }
        const int units = (int)s.gen_units.size(), per_cta = kGenThreads / 32;
        const int want = (units + per_cta - 1) / per_cta;
        pl->gen_grid = want < pl->sm_count ? (want > 0 ? want : 1) : pl->sm_count;
        if ((flags & ARKCOS_PLAN_SPECTRAL) && (st = build_spectral(pl)) != ARKCOS_OK) break;
        if (flags & ARKCOS_PLAN_CACHE_WEIGHTS) {
            if ((st = launch_generate(pl, 0)) != ARKCOS_OK) break;
            if (!cuda_ok(cudaDeviceSynchronize(), "cudaDeviceSynchronize")) { st = ARKCOS_ECUDA; break; }
            pl->weights_ready = true;
        }
    } while (0);
    if (st != ARKCOS_OK) { arkcos_plan_destroy(pl); return st; }
    *plan = pl;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_create(arkcos_plan** plan, int n_theta, int n_phi, const double* k_table, int n_table,
                                 double theta_cut) {
    return arkcos_plan_create_ex(plan, n_theta, n_phi, k_table, n_table, theta_cut, ARKCOS_PLAN_DEFAULT);
}

arkcos_status arkcos_convolve_batch(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps, void* stream) {
    arkcos_status s = check_io(pl, d_in, d_out, n_maps);
    if (s != ARKCOS_OK) return s;
    if (n_maps > 65535) return ARKCOS_EINVAL;
    return run(pl, d_in, d_out, n_maps, (cudaStream_t)stream);
}

arkcos_status arkcos_convolve(const arkcos_plan* pl, const float* d_in, float* d_out, void* stream) {
    return arkcos_convolve_batch(pl, d_in, d_out, 1, stream);
}

arkcos_status arkcos_measure_convolve(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps, void* stream,
                                      float* ms_generate, float* ms_convolve) {
    arkcos_status s = check_io(pl, d_in, d_out, n_maps);
    if (s != ARKCOS_OK) return s;
    if (n_maps > 65535) return ARKCOS_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const bool cached = (pl->flags & ARKCOS_PLAN_CACHE_WEIGHTS) != 0;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};             // per call: the entry point is re-entrant
    for (auto& e : ev)
        if (!cuda_ok(cudaEventCreate(&e), "cudaEventCreate")) { for (auto& x : ev) if (x) cudaEventDestroy(x); return ARKCOS_ECUDA; }
    float a = 0.f, b = 0.f;
    s = ARKCOS_ECUDA;
    do {
        if (!cuda_ok(cudaEventRecord(ev[0], st), "cudaEventRecord")) break;
        if (!cached && (s = launch_generate(pl, st)) != ARKCOS_OK) break;
        s = ARKCOS_ECUDA;
        if (!cuda_ok(cudaEventRecord(ev[1], st), "cudaEventRecord")) break;
        if ((s = launch_convolve(pl, d_in, d_out, n_maps, st)) != ARKCOS_OK) break;
        s = ARKCOS_ECUDA;
        if (!cuda_ok(cudaEventRecord(ev[2], st), "cudaEventRecord")) break;
        if (!cuda_ok(cudaEventSynchronize(ev[2]), "cudaEventSynchronize")) break;
        if (!cuda_ok(cudaEventElapsedTime(&a, ev[0], ev[1]), "cudaEventElapsedTime")) break;
        if (!cuda_ok(cudaEventElapsedTime(&b, ev[1], ev[2]), "cudaEventElapsedTime")) break;
        s = ARKCOS_OK;
    } while (0);
    for (auto& e : ev) cudaEventDestroy(e);
    if (s != ARKCOS_OK) return s;
    if (ms_generate) *ms_generate = cached ? 0.f : a;
    if (ms_convolve) *ms_convolve = b;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_reserve_host_io(arkcos_plan* pl) { return arkcos_plan_reserve_host_io_chunks(pl, 0); }

arkcos_status arkcos_plan_reserve_host_io_chunks(arkcos_plan* pl, int n_chunks) {
    if (!pl || n_chunks < 0) return ARKCOS_EINVAL;
    if (pl->flags & ARKCOS_PLAN_HOST_ONLY) return ARKCOS_EUNSUPPORTED;
    if (pl->d_io_in) return ARKCOS_OK;
    const size_t bytes = (size_t)pl->sched.n_theta * pl->sched.n_phi * sizeof(float);
    // chunks of about 8 MB: long enough for the copy engines, short enough that compute and the copy back start early
    if (n_chunks == 0) n_chunks = (int)std::max<size_t>(1, std::min<size_t>(16, bytes / (8u << 20)));
    arkcos_status st = ARKCOS_OK;
    try { build_pipeline(pl->sched, n_chunks, pl->pipe); } catch (const std::bad_alloc&) { return ARKCOS_ENOMEM; }
    cudaError_t e = cudaMalloc((void**)&pl->d_io_in, bytes);
    if (e == cudaSuccess) e = cudaMalloc((void**)&pl->d_io_out, bytes);
    if (e != cudaSuccess) {
        cudaFree(pl->d_io_in); pl->d_io_in = nullptr; pl->d_io_out = nullptr;
        if (e == cudaErrorMemoryAllocation) { (void)cudaGetLastError(); return ARKCOS_ENOMEM; }
        CU(e);
    }
    pl->device_bytes += 2 * bytes;
    if ((st = upload(pl, &pl->d_pipe_items, pl->pipe.items)) != ARKCOS_OK) return st;
    CU(cudaStreamCreateWithFlags(&pl->s_h2d, cudaStreamNonBlocking));
    CU(cudaStreamCreateWithFlags(&pl->s_d2h, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming));
    pl->ev_h2d.assign(pl->pipe.n_chunks, nullptr); pl->ev_comp.assign(pl->pipe.n_chunks, nullptr);
    for (auto& ev : pl->ev_h2d) CU(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    for (auto& ev : pl->ev_comp) CU(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    CU(cudaDeviceSynchronize());                                  // the item upload has landed
    return ARKCOS_OK;
}

// HOST map in, HOST map out, as a pipeline over bands of rings (Pipeline, arkcos_internal.h): the copy of chunk
// c + 1 to the device, the convolution of the items whose last input ring lies in chunk c, and the copy back of the
// chunks those items completed run concurrently on three streams.  The work items, their kernels and therefore
// the result are those of arkcos_convolve.
arkcos_status arkcos_convolve_host(arkcos_plan* pl, const float* h_in, float* h_out, void* stream) {
    if (!pl || !h_in || !h_out) return ARKCOS_EINVAL;
    if (pl->flags & ARKCOS_PLAN_HOST_ONLY) return ARKCOS_EUNSUPPORTED;
    arkcos_status s = arkcos_plan_reserve_host_io(pl);           // no-op once reserved
    if (s != ARKCOS_OK) return s;
    if ((s = check_io(pl, pl->d_io_in, pl->d_io_out, 1)) != ARKCOS_OK) return s;
    const Pipeline& pp = pl->pipe;
    const size_t row = (size_t)pl->sched.n_phi;
    cudaStream_t st = (cudaStream_t)stream;
    // the copy streams start after whatever the caller has queued on `stream`
    CU(cudaEventRecord(pl->ev_fork, st));
    CU(cudaStreamWaitEvent(pl->s_h2d, pl->ev_fork, 0));
    CU(cudaStreamWaitEvent(pl->s_d2h, pl->ev_fork, 0));
    if (!(pl->flags & ARKCOS_PLAN_CACHE_WEIGHTS) && (s = launch_generate(pl, st)) != ARKCOS_OK) return s;
    const ConvParams c = conv_params(pl, pl->d_io_in, pl->d_io_out);
    for (int g = 0; g < pp.n_chunks; g++) {
        const size_t lo = (size_t)pp.chunk_lo[g] * row, n = (size_t)(pp.chunk_lo[g + 1] - pp.chunk_lo[g]) * row;
        CU(cudaMemcpyAsync(pl->d_io_in + lo, h_in + lo, n * sizeof(float), cudaMemcpyHostToDevice, pl->s_h2d));
        CU(cudaEventRecord(pl->ev_h2d[g], pl->s_h2d));
        CU(cudaStreamWaitEvent(st, pl->ev_h2d[g], 0));
        s = launch_items(pl, c, pl->d_pipe_items + pp.wide_begin[g], pp.narrow_begin[g] - pp.wide_begin[g],
                         pl->d_pipe_items + pp.narrow_begin[g], pp.wide_begin[g + 1] - pp.narrow_begin[g], 1, st);
        if (s != ARKCOS_OK) return s;
        CU(cudaEventRecord(pl->ev_comp[g], st));
        bool waited = false;
        for (int ch = 0; ch < pp.n_chunks; ch++) {
            if (pp.ready_group[ch] != g) continue;
            if (!waited) { CU(cudaStreamWaitEvent(pl->s_d2h, pl->ev_comp[g], 0)); waited = true; }
            const size_t clo = (size_t)pp.chunk_lo[ch] * row, cn = (size_t)(pp.chunk_lo[ch + 1] - pp.chunk_lo[ch]) * row;
            CU(cudaMemcpyAsync(h_out + clo, pl->d_io_out + clo, cn * sizeof(float), cudaMemcpyDeviceToHost, pl->s_d2h));
        }
    }
    CU(cudaStreamSynchronize(pl->s_d2h));
    CU(cudaStreamSynchronize(st));
    return ARKCOS_OK;
}

arkcos_status arkcos_spectral_workspace_bytes(const arkcos_plan* pl, int n_maps, unsigned long long* bytes) {
    if (!pl || !bytes || n_maps < 1) return ARKCOS_EINVAL;
    if (!(pl->flags & ARKCOS_PLAN_SPECTRAL)) return ARKCOS_EUNSUPPORTED;
    *bytes = (unsigned long long)n_maps * pl->sched.n_theta * (pl->sched.n_phi / 2 + 1) * sizeof(float2);
    return ARKCOS_OK;
}

arkcos_status arkcos_convolve_spectral(const arkcos_plan* pl, const float* d_in, float* d_out, int n_maps, void* d_work,
                                       unsigned long long work_bytes, void* stream) {
    arkcos_status st = check_io(pl, d_in, d_out, n_maps);
    if (st != ARKCOS_OK) return st;
    if (!(pl->flags & ARKCOS_PLAN_SPECTRAL)) return ARKCOS_EUNSUPPORTED;
    unsigned long long need = 0;
    (void)arkcos_spectral_workspace_bytes(pl, n_maps, &need);
    if (!d_work || ((uintptr_t)d_work & 15u) || work_bytes < need || n_maps > 65535) return ARKCOS_EINVAL;
    const Schedule& s = pl->sched;
    const int h = s.n_phi / 2;
    SpecParams p;
    p.in = d_in; p.out = d_out; p.xspec = reinterpret_cast<float2*>(d_work); p.wspec = pl->d_wspec; p.pairs = pl->d_pairs;
    p.tw_h = pl->d_tw_h; p.tw_n = pl->d_tw_n; p.n_theta = s.n_theta; p.n_phi = s.n_phi; p.R = s.R;
    const dim3 grid((unsigned)s.n_theta, (unsigned)n_maps, 1);
    cudaStream_t cs = (cudaStream_t)stream;
    ARKCOS_LAUNCH(k_rfft_rings, grid, kSpecThreads, (size_t)(2 * h + h / 2) * sizeof(float2), cs, p);
    CU(cudaGetLastError());
    ARKCOS_LAUNCH(k_spectral_apply, grid, kSpecThreads, (size_t)(2 * h + 1 + h / 2) * sizeof(float2), cs, p);
    CU(cudaGetLastError());
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_work(const arkcos_plan* pl, unsigned long long* pair_evals, unsigned long long* weights,
                               int* ring_halfband) {
    if (!pl) return ARKCOS_EINVAL;
    if (pair_evals) *pair_evals = pl->sched.pair_evals;
    if (weights) *weights = pl->sched.weights;
    if (ring_halfband) *ring_halfband = pl->sched.R;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_get_info(const arkcos_plan* pl, arkcos_plan_info* info) {
    if (!pl || !info) return ARKCOS_EINVAL;
    std::memset(info, 0, sizeof(*info));
    const Schedule& s = pl->sched;
    info->n_theta = s.n_theta; info->n_phi = s.n_phi; info->n_table = pl->n_table; info->theta_cut = s.theta_cut;
    info->ring_halfband = s.R; info->pair_evals = s.pair_evals; info->weights = s.weights;
    info->fma_slots = s.fma_slots; info->weight_slots = s.weight_slots;
    info->n_items = (int)s.items.size(); info->n_gen_units = (int)s.gen_units.size();
    {
        const int n_wide = (pl->flags & ARKCOS_PLAN_ONLY_NARROW) ? 0 : s.n_wide_items;
        const int n_narrow = (pl->flags & ARKCOS_PLAN_ONLY_WIDE) ? 0 : (int)s.items.size() - s.n_wide_items;
        info->kernels_per_convolve = ((pl->flags & ARKCOS_PLAN_CACHE_WEIGHTS) ? 0 : 1) + (n_wide > 0) + (n_narrow > 0);
    }
    info->sm_count = pl->sm_count; info->flags = pl->flags; info->device_bytes = pl->device_bytes;
    info->fma_slots_wide = s.fma_slots_wide; info->first_narrow_ring = s.first_narrow;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_item(const arkcos_plan* pl, int index, int* fields) {
    if (!pl || !fields || index < 0 || index >= (int)pl->sched.items.size()) return ARKCOS_EINVAL;
    const Item& it = pl->sched.items[index];
    fields[0] = it.kind; fields[1] = it.i0; fields[2] = it.nrings; fields[3] = it.k0;
    fields[4] = it.kind == kWide ? kWarpSpan << it.f_log2 : kNarrowSpan;
    fields[5] = it.kind == kWide ? kWarps >> it.f_log2 : kWarps;
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_validate(const arkcos_plan* pl, char* why, int cap) {
    if (!pl || cap < 0 || (cap > 0 && !why)) return ARKCOS_EINVAL;
    std::string msg;
    const int rc = validate_schedule(pl->sched, &msg);
    if (cap > 0) { std::strncpy(why, msg.c_str(), (size_t)cap - 1); why[cap - 1] = 0; }
    return rc == 0 ? ARKCOS_OK : ARKCOS_EINTERNAL;
}

arkcos_status arkcos_plan_window(const arkcos_plan* pl, int i, int j, int* half_width) {
    if (!pl || !half_width) return ARKCOS_EINVAL;
    if (i < 0 || i >= pl->sched.n_theta || j < 0 || j >= pl->sched.n_theta) return ARKCOS_EINVAL;
    *half_width = pl->sched.window(i, j);
    return ARKCOS_OK;
}

arkcos_status arkcos_plan_pair_weights(const arkcos_plan* pl, int i, int j, float* h_w, int cap, int* n) {
    if (!pl || !h_w || !n || cap < 0) return ARKCOS_EINVAL;
    if (pl->flags & ARKCOS_PLAN_HOST_ONLY) return ARKCOS_EUNSUPPORTED;
    const Schedule& s = pl->sched;
    if (i < 0 || i >= s.n_theta || j < 0 || j >= s.n_theta) return ARKCOS_EINVAL;
    *n = 0;
    // southern output rings use their northern mirror pair (identical weights)
    int in_ = i, jn = j;
    if (i >= s.n_north) { in_ = s.n_theta - 1 - i; jn = s.n_theta - 1 - j; }
    const PairDesc* pd = s.pair(in_, jn);
    if (!pd || pd->ntaps == 0) return ARKCOS_OK;
    if (!pl->weights_ready) {
        arkcos_status st = launch_generate(pl, 0);
        if (st != ARKCOS_OK) return st;
    }
    CU(cudaDeviceSynchronize());
    int dmax = pd->half == s.n_phi ? s.n_phi / 2 : pd->half;
    int cnt = dmax + 1 < cap ? dmax + 1 : cap;
    const size_t floats = (size_t)pd->ntaps;
    std::vector<float> all(floats);
    CU(cudaMemcpy(all.data(), pl->d_weights + pd->w_off, sizeof(float) * floats, cudaMemcpyDeviceToHost));
    for (int d = 0; d < cnt; d++) {
        // tap +d is stored at e = d - start, except d = n_phi/2 of a whole ring, stored as d = -n_phi/2
        int e = d - pd->start;
        if (pd->half == s.n_phi && d == s.n_phi / 2) e = -d - pd->start;
        h_w[d] = all[e];
    }
    *n = cnt;
    return ARKCOS_OK;
}

}  // extern "C"
