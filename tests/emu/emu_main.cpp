// emu_main.cpp - HOST EMULATION harness of the arkcos CUDA kernels.  Test infrastructure only.
//
// Compiles paper_1211_3556_b200/csrc/arkcos_kernels.cuh (the product's kernel source, unchanged) and
// arkcos_schedule.cpp for the host against tests/emu/stub/cuda_runtime.h and runs, for one plan:
//   k_generate_weights  ->  k_convolve  (every work item, one CTA at a time, one OS thread per CUDA
//   thread, real barriers for __syncthreads / __syncwarp, cp.async performed only at its wait).
// Shared memory is a heap block of exactly the launch's dynamic size (AddressSanitizer sees overruns),
// every ld.shared wrapper checks bounds and alignment, every cp.async source must lie in a registered
// global buffer.  Shared memory and the output start as NaN, so a value consumed before it was staged
// shows up in the result.  EMU_EAGER=1 performs cp.async copies at issue instead of at the wait, which exposes
// a copy that lands in a buffer still being read.
//
//   emu_arkcos n_theta n_phi theta_cut n_table table.f64 in.f32 out.f32 [only_wide|only_narrow]
//
// It does not replace the GPU parity tests: it checks the index logic (windows, staging, wrap-around,
// pass structure, weight layout), not the compiled SASS.
#include "emu_runtime.h"

#include "arkcos_internal.h"
#include "arkcos_kernels.cuh"
#include "arkcos_tensor.cuh"


template <typename T>
static std::vector<T> read_file(const char* path, size_t n) {
    std::vector<T> v(n);
    FILE* f = std::fopen(path, "rb");
    if (!f || std::fread(v.data(), sizeof(T), n, f) != n) { std::fprintf(stderr, "cannot read %s\n", path); std::exit(2); }
    std::fclose(f);
    return v;
}

// Self-test of the hazard checker: tiny two-warp "kernels" with and without the barrier that orders a cp.async
// write and an ld.shared read.  Modes 1 and 3 must die with EMU FAILURE (exit 3), modes 2 and 4 must pass.
// Modes 5 and 6: barriers that can never complete (a hang on the device) must be reported as a DEADLOCK - one lane
// waits at __syncwarp while the rest of its warp waits at __syncthreads; a lane skips a warp-collective mma.
static int hazard_selftest(int mode) {
    static float src[8] = {1, 2, 3, 4, 5, 6, 7, 8};
    emu::g_global = {{(const unsigned char*)src, (const unsigned char*)(src + 8)}};
    emu::g_kernel_name = "selftest";
    emu::run_cta(0, 0, 64, mode == 7 ? 8192 : 64, [&] {
        const unsigned t = threadIdx.x;
        float a, b, c, d;
        if (mode == 7) {                                   // bank-conflict accounting: known patterns (EMU_BANKS=<file>)
            float a, b, c, d;
            if (t < 32) {
                arkcos::lds64i<0>(a, b, t * 144);          // round 1's NARROW layout: lanes l and l + 8 collide -> 2 wavefronts per half warp
                arkcos::lds128(a, b, c, d, t * 80);        // v5's lane tiles: conflict free
                arkcos::lds128(a, b, c, d, (t & 7) * 16);  // four lanes per address: broadcast, conflict free
                arkcos::lds128(a, b, c, d, t * 128);       // every lane in the same four banks: 8 wavefronts per quarter warp
            }
            return;
        }
        if (mode == 5) { if (t == 3) __syncwarp(); __syncthreads(); return; }
        if (mode == 6) { float c[4] = {0, 0, 0, 0}; if (t != 7) emu::mma_m16n8k8_tf32(c, 0, 0, 0, 0, 0, 0); return; }
        if (mode == 1 || mode == 2) {                      // write by thread 0, read by thread 40 (another warp)
            if (t == 0) { arkcos::cp_async16(0, src); arkcos::cp_async_wait_all(); }
            if (mode == 2) __syncthreads();
            if (t == 40) arkcos::lds128(a, b, c, d, 0);
            if (mode == 1) __syncthreads();                // a barrier AFTER the read does not order it
        } else {                                           // read by thread 1, then cp.async by thread 2 (same warp)
            if (t == 1) arkcos::lds128(a, b, c, d, 16);
            if (mode == 4) __syncwarp();
            if (t == 2) { arkcos::cp_async16(16, src + 4); arkcos::cp_async_wait_all(); }
            if (mode == 3) __syncwarp();
        }
    });
    emu::bank_report();
    std::printf("selftest %d passed the checker\n", mode);
    return 0;
}

int main(int argc, char** argv) {
    using namespace arkcos;
    if (argc == 3 && std::string(argv[1]) == "selftest") return hazard_selftest(std::atoi(argv[2]));
    if (argc < 8) { std::fprintf(stderr, "usage: emu_arkcos n_theta n_phi theta_cut n_table table.f64 in.f32 out.f32 [only_wide|only_narrow]\n"); return 2; }
    const int n_theta = std::atoi(argv[1]), n_phi = std::atoi(argv[2]);
    const double theta_cut = std::atof(argv[3]);
    const int n_table = std::atoi(argv[4]);
    const std::string only = argc > 8 ? argv[8] : "";
    std::vector<double> table = read_file<double>(argv[5], (size_t)n_table);
    const size_t n_pix = (size_t)n_theta * n_phi;
    std::vector<float> in = read_file<float>(argv[6], n_pix);
    std::vector<float> out(n_pix, std::nanf(""));

    Schedule s;
    const int rc = build_schedule(n_theta, n_phi, theta_cut, 148, s);
    if (rc != 0) { std::fprintf(stderr, "build_schedule failed: %d\n", rc); return 2; }
    std::vector<float> weights((size_t)s.weight_slots + 4, 0.0f);
    emu::g_global = {{(const unsigned char*)in.data(), (const unsigned char*)(in.data() + in.size())},
                     {(const unsigned char*)weights.data(), (const unsigned char*)(weights.data() + weights.size())},
                     {(const unsigned char*)s.pairs.data(), (const unsigned char*)(s.pairs.data() + s.pairs.size())}};

    // ---- S2: weight generator ----------------------------------------------------------------------
    GenParams g;
    g.units = s.gen_units.data(); g.s2 = s.s2.data(); g.table = table.data(); g.weights = weights.data();
    g.n_units = (int)s.gen_units.size(); g.n_phi = n_phi; g.n_table = n_table;
    g.t_scale = (double)(n_table - 1) / theta_cut; g.table_in_smem = 1;
    g.m_split = 0; g.theta_split = 0.0; g.t_scale2 = 0.0;
    if (const char* e = std::getenv("EMU_M_SPLIT")) {            // two-zone table: EMU_M_SPLIT, EMU_THETA_SPLIT
        g.m_split = std::atoi(e); g.theta_split = std::atof(std::getenv("EMU_THETA_SPLIT"));
        g.t_scale = (double)g.m_split / g.theta_split;
        g.t_scale2 = (double)(n_table - 1 - g.m_split) / (theta_cut - g.theta_split);
    }
    const int gen_grid = 4;
    emu::g_gridDim = dim3(gen_grid);
    emu::g_kernel_name = "k_generate_weights";
    for (int b = 0; b < gen_grid; b++)
        emu::run_cta((unsigned)b, 0, kGenThreads, (size_t)n_table * sizeof(double), [&] { k_generate_weights(g); });

    // ---- S3: convolution, one CTA per work item ------------------------------------------------------
    ConvParams c;
    c.in = in.data(); c.out = out.data(); c.pairs = s.pairs.data(); c.items = s.items.data(); c.weights = weights.data();
    c.runs = s.runs.data(); c.first_narrow = s.first_narrow; c.narrow_w_base = s.narrow_w_base;
    c.n_theta = n_theta; c.n_phi = n_phi; c.R = s.R; c.wslot = s.narrow_wslot; c.wcap = s.narrow_wcap;
    c.map_stride = (long long)n_pix;
    emu::g_global.push_back({(const unsigned char*)s.runs.data(), (const unsigned char*)(s.runs.data() + s.runs.size())});
    emu::g_gridDim = dim3((unsigned)s.items.size());
    int n_wide = 0, n_narrow = 0;
    // EMU_ITEM_STRIDE=n: run every n-th work item only (big grids; outputs of the skipped items stay NaN);
    // EMU_ITEM_OFFSET=o: ... the items o, o + n, o + 2n, ... (n processes with o = 0 .. n-1 cover the launch)
    const size_t item_stride = std::getenv("EMU_ITEM_STRIDE") ? (size_t)std::atoi(std::getenv("EMU_ITEM_STRIDE")) : 1;
    const size_t item_offset = std::getenv("EMU_ITEM_OFFSET") ? (size_t)std::atoi(std::getenv("EMU_ITEM_OFFSET")) : 0;   // items b = offset mod stride
    const bool wide_tensor = std::getenv("EMU_WIDE_TENSOR") != nullptr;   // WIDE items through k_convolve_wide_tc
    for (size_t b = 0; b < s.items.size(); b++) {
        const bool wide = s.items[b].kind == kWide;
        if (item_stride > 1 && b % item_stride != item_offset % item_stride) continue;
        if ((only == "only_wide" && !wide) || (only == "only_narrow" && wide)) continue;
        (wide ? n_wide : n_narrow)++;
        ConvParams cc = c;                                     // each kernel is launched on its own part of the work list
        emu::g_kernel_name = wide ? (wide_tensor ? "k_convolve_wide_tc" : "k_convolve_wide") : "k_convolve_narrow";
        if (wide && wide_tensor) emu::run_cta((unsigned)b, 0, kThreads, s.smem_wide, [&] { k_convolve_wide_tc(cc); });   // N1(a)
        else if (wide) emu::run_cta((unsigned)b, 0, kThreads, s.smem_wide, [&] { k_convolve_wide(cc); });
        else {
            cc.items = c.items + s.n_wide_items;
            emu::run_cta((unsigned)(b - s.n_wide_items), 0, kThreads, s.smem_narrow, [&] { k_convolve_narrow(cc); });
        }
    }
    emu::bank_report();
    FILE* f = std::fopen(argv[7], "wb");
    if (!f || std::fwrite(out.data(), sizeof(float), n_pix, f) != n_pix) { std::fprintf(stderr, "cannot write %s\n", argv[7]); return 2; }
    std::fclose(f);
    int n_single = 0;
    for (size_t b = (size_t)s.n_wide_items; b < s.items.size(); b++) n_single += 2 * kWarps * (s.items[b].wcopy + kNarrowWPad) > s.narrow_wcap;
    std::printf("single-buffered narrow items %d; ", n_single);
    std::printf("emu ok: R %d first_narrow %d n_north %d items wide %d narrow %d smem wide %zu narrow %zu weight_slots %llu\n", s.R,
                s.first_narrow, s.n_north, n_wide, n_narrow, s.smem_wide, s.smem_narrow, (unsigned long long)s.weight_slots);
    return 0;
}
