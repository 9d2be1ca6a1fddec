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
#include <barrier>
#include <memory>
#include <mutex>
#include <thread>

#include "cuda_runtime.h"

#include "arkcos_internal.h"
#include "arkcos_kernels.cuh"

namespace emu {
thread_local uint3 t_threadIdx, t_blockIdx;
dim3 g_blockDim, g_gridDim;
unsigned char* g_smem = nullptr;
size_t g_smem_bytes = 0;

static std::unique_ptr<std::barrier<>> g_cta_barrier;
static std::vector<std::unique_ptr<std::barrier<>>> g_warp_barriers;
struct Range { const unsigned char* lo; const unsigned char* hi; };
static std::vector<Range> g_global;

[[noreturn]] void fail(const char* what, long a, long b) {
    std::fprintf(stderr, "EMU FAILURE: %s (%ld, %ld) block %u thread %u\n", what, a, b, t_blockIdx.x, t_threadIdx.x);
    std::_Exit(3);
}
static thread_local uint32_t t_cta_epoch = 0, t_warp_epoch = 0;   // barriers this thread has passed (hazard checker below)
void sync_threads() { g_cta_barrier->arrive_and_wait(); ++t_cta_epoch; }
void sync_warp() { g_warp_barriers[t_threadIdx.x >> 5]->arrive_and_wait(); ++t_warp_epoch; }
void check_global(const void* p, size_t bytes) {
    const unsigned char* q = (const unsigned char*)p;
    if ((uintptr_t)q % 16) fail("misaligned global access of cp.async", (long)((uintptr_t)q % 16), (long)bytes);
    for (const Range& r : g_global)
        if (q >= r.lo && q + bytes <= r.hi) return;
    fail("cp.async source outside every global buffer", 0, (long)bytes);
}

// ---- shared-memory hazard checker -------------------------------------------------------------------
// What `compute-sanitizer --tool racecheck` reports on the device, for the accesses the emulation sees (the
// ld.shared wrappers and the cp.async copies): two accesses of one shared-memory word by different threads, at
// least one a write, with no barrier both threads took part in between them.  Every thread counts the CTA
// barriers and the warp barriers it has passed; an access by thread b is ordered after an earlier access by
// thread a iff b has passed a CTA barrier a had not yet passed at its access, or the two are in one warp and b
// has passed a warp barrier a had not.  A cp.async WRITE may land any time between its issue and its wait: it is
// checked against earlier readers / writers at issue and becomes the word's writer at the wait.
struct Stamp { uint16_t tid; uint16_t valid; uint32_t cta_epoch, warp_epoch; };
static std::vector<Stamp> g_writer, g_reader;                     // per 4-byte word: last writer, most recent reader
static std::mutex g_shadow_mutex;
static const bool g_racecheck = std::getenv("EMU_NO_RACECHECK") == nullptr;
static bool ordered_after(const Stamp& a) {                        // is the calling thread's access ordered after stamp a?
    if (!a.valid || a.tid == t_threadIdx.x) return true;
    if (t_cta_epoch > a.cta_epoch) return true;
    return (a.tid >> 5) == (t_threadIdx.x >> 5) && t_warp_epoch > a.warp_epoch;
}
static Stamp now() { return Stamp{(uint16_t)t_threadIdx.x, 1, t_cta_epoch, t_warp_epoch}; }
void note_read(uint32_t addr, uint32_t bytes) {
    if (!g_racecheck) return;
    std::lock_guard<std::mutex> lock(g_shadow_mutex);
    for (uint32_t w = addr / 4; w < (addr + bytes + 3) / 4; w++) {
        if (!ordered_after(g_writer[w])) fail("shared-memory hazard: read of a word another thread wrote without a barrier in between (word, writer)", w, g_writer[w].tid);
        const Stamp& r = g_reader[w];
        if (!r.valid || t_cta_epoch >= r.cta_epoch) g_reader[w] = now();
    }
}
static void note_write_issue(uint32_t addr, uint32_t bytes) {
    if (!g_racecheck) return;
    std::lock_guard<std::mutex> lock(g_shadow_mutex);
    for (uint32_t w = addr / 4; w < (addr + bytes + 3) / 4; w++) {
        if (!ordered_after(g_reader[w])) fail("shared-memory hazard: cp.async issued into a word another thread may still be reading (word, reader)", w, g_reader[w].tid);
        if (!ordered_after(g_writer[w])) fail("shared-memory hazard: two unordered writes of one word (word, writer)", w, g_writer[w].tid);
    }
}
static void note_write_done(uint32_t addr, uint32_t bytes) {
    if (!g_racecheck) return;
    std::lock_guard<std::mutex> lock(g_shadow_mutex);
    for (uint32_t w = addr / 4; w < (addr + bytes + 3) / 4; w++) g_writer[w] = now();
}

struct Pending { uint32_t dst; const void* src; };
static thread_local std::vector<std::vector<Pending>> t_groups;   // committed groups, oldest first
static thread_local std::vector<Pending> t_open;                  // not yet committed
// Two modes bracket what the hardware may do with a cp.async: DEFERRED (default) performs the copy only at
// the wait - a read before the wait sees stale data (RAW hazard); EAGER (EMU_EAGER=1) performs it at once - a
// copy into a buffer that other threads still read clobbers it (WAR hazard).
static const bool g_eager = std::getenv("EMU_EAGER") != nullptr;
void cp_async_enqueue(uint32_t dst, const void* src) {
    (void)smem_at(dst, 16);
    check_global(src, 16);
    note_write_issue(dst, 16);
    if (g_eager) { std::memcpy(smem_at(dst, 16), src, 16); note_write_done(dst, 16); return; }
    t_open.push_back(Pending{dst, src});
}
void cp_async_commit_group() { t_groups.push_back(std::move(t_open)); t_open.clear(); }
static void perform(const std::vector<Pending>& g) {
    for (const Pending& c : g) { std::memcpy(smem_at(c.dst, 16), c.src, 16); note_write_done(c.dst, 16); }
}
void cp_async_wait(int keep_groups) {
    if (keep_groups == 0) {            // wait_all / wait_group 0: everything, committed or not
        for (auto& g : t_groups) perform(g);
        t_groups.clear();
        perform(t_open); t_open.clear();
        return;
    }
    while ((int)t_groups.size() > keep_groups) { perform(t_groups.front()); t_groups.erase(t_groups.begin()); }
}
static void thread_exit_check() {
    if (!t_open.empty() || !t_groups.empty()) fail("thread exits with cp.async copies it never waited for", (long)t_groups.size(), 0);
}

// run one CTA of `threads` threads
template <typename F>
static void run_cta(unsigned bx, unsigned by, unsigned threads, size_t smem_bytes, F&& body) {
    g_smem_bytes = smem_bytes;
    g_smem = (unsigned char*)std::malloc(smem_bytes ? smem_bytes : 16);
    std::memset(g_smem, 0xFF, smem_bytes);                        // NaN pattern
    g_writer.assign(smem_bytes / 4 + 4, Stamp{0, 0, 0, 0}); g_reader.assign(smem_bytes / 4 + 4, Stamp{0, 0, 0, 0});
    g_blockDim = dim3(threads);
    g_cta_barrier = std::make_unique<std::barrier<>>((std::ptrdiff_t)threads);
    g_warp_barriers.clear();
    for (unsigned w = 0; w < threads / 32; w++) g_warp_barriers.push_back(std::make_unique<std::barrier<>>(32));
    std::vector<std::thread> pool;
    for (unsigned t = 0; t < threads; t++)
        pool.emplace_back([&, t] {
            t_threadIdx = uint3{t, 0, 0}; t_blockIdx = uint3{bx, by, 0};
            t_cta_epoch = 0; t_warp_epoch = 0;
            body();
            thread_exit_check();
        });
    for (auto& th : pool) th.join();
    std::free(g_smem);
    g_smem = nullptr;
}
}  // namespace emu

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
static int hazard_selftest(int mode) {
    static float src[8] = {1, 2, 3, 4, 5, 6, 7, 8};
    emu::g_global = {{(const unsigned char*)src, (const unsigned char*)(src + 8)}};
    emu::run_cta(0, 0, 64, 64, [&] {
        const unsigned t = threadIdx.x;
        float a, b, c, d;
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
    // EMU_ITEM_STRIDE=n: run every n-th work item only (big grids; outputs of the skipped items stay NaN)
    const size_t item_stride = std::getenv("EMU_ITEM_STRIDE") ? (size_t)std::atoi(std::getenv("EMU_ITEM_STRIDE")) : 1;
    for (size_t b = 0; b < s.items.size(); b++) {
        const bool wide = s.items[b].kind == kWide;
        if (item_stride > 1 && b % item_stride != 0) continue;
        if ((only == "only_wide" && !wide) || (only == "only_narrow" && wide)) continue;
        (wide ? n_wide : n_narrow)++;
        ConvParams cc = c;                                     // each kernel is launched on its own part of the work list
        if (wide) emu::run_cta((unsigned)b, 0, kThreads, s.smem_wide, [&] { k_convolve_wide(cc); });
        else {
            cc.items = c.items + s.n_wide_items;
            emu::run_cta((unsigned)(b - s.n_wide_items), 0, kThreads, s.smem_narrow, [&] { k_convolve_narrow(cc); });
        }
    }
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
