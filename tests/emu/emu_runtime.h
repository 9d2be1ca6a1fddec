// emu_runtime.h - the HOST EMULATION runtime of the arkcos CUDA kernels.  Test infrastructure only; included
// once per emulation binary (emu_main.cpp: the kernel-level command-line harness; emu_api.cpp: the whole C-ABI
// library compiled for the host).
//
// One OS thread per CUDA thread, one CTA at a time, real barriers for __syncthreads / __syncwarp, cp.async
// performed only at its wait (EMU_EAGER=1: at issue), shared memory a heap block of exactly the launch's dynamic
// size with bounds- and alignment-checked ld.shared wrappers, checked cp.async sources, NaN-initialised shared
// memory, and a shared-memory hazard checker (the CPU counterpart of compute-sanitizer racecheck).
#pragma once
#include <barrier>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <thread>

#include "cuda_runtime.h"

namespace emu {
thread_local uint3 t_threadIdx, t_blockIdx;
dim3 g_blockDim, g_gridDim;
unsigned char* g_smem = nullptr;
size_t g_smem_bytes = 0;

static std::unique_ptr<std::barrier<>> g_cta_barrier;
static std::vector<std::unique_ptr<std::barrier<>>> g_warp_barriers;
struct Range { const unsigned char* lo; const unsigned char* hi; };
static std::vector<Range> g_global;      // buffers a cp.async may read: registered by the harness, or by the emulated cudaMalloc

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
// The copy may have landed at any time since its issue: a reader that is not ordered BEFORE the issue (it read while
// the copy was in flight, with or without a barrier after the issue) is a hazard too.  `ic`, `iw` = the writer's
// barrier counts at issue.
static void note_write_done(uint32_t addr, uint32_t bytes, uint32_t ic, uint32_t iw) {
    if (!g_racecheck) return;
    std::lock_guard<std::mutex> lock(g_shadow_mutex);
    for (uint32_t w = addr / 4; w < (addr + bytes + 3) / 4; w++) {
        const Stamp& r = g_reader[w];
        const bool before_issue = !r.valid || r.tid == t_threadIdx.x || ic > r.cta_epoch ||
                                  ((r.tid >> 5) == (t_threadIdx.x >> 5) && iw > r.warp_epoch);
        if (!before_issue) fail("shared-memory hazard: a word was read by another thread while a cp.async into it was in flight (word, reader)", w, r.tid);
        g_writer[w] = now();
    }
}

void note_store(uint32_t addr, uint32_t bytes) {                  // plain st.shared: issue and completion coincide
    note_write_issue(addr, bytes);
    note_write_done(addr, bytes, t_cta_epoch, t_warp_epoch);
}

// ---- mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 -------------------------------------------------
// The 32 threads of a warp publish their fragment registers, meet, and each computes its four elements of
// D = A B + C from the fragment layout of the PTX ISA ("Matrix Fragments for mma.m16n8k8", .tf32; g = lane >> 2,
// t = lane & 3):  A[g + 8 (r & 1)][t + 4 (r >> 1)] = a_r,  B[t + 4 r][g] = b_r,  C[g + 8 (r >> 1)][2 t + (r & 1)] = c_r.
// The tensor core reads the upper 19 bits of an operand register (the 13 low mantissa bits are ignored), forms
// the products exactly and adds them to C with TRUNCATION; here: exact sum in FP64, then rounded toward zero to FP32.
// The meeting uses the warp's barrier WITHOUT counting it for the hazard checker: mma.sync converges the warp but
// orders no shared-memory access.
static uint32_t g_mma_a[64][32][4], g_mma_b[64][32][2];
void mma_m16n8k8_tf32(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    const unsigned warp = t_threadIdx.x >> 5, lane = t_threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    uint32_t (&A)[32][4] = g_mma_a[warp]; uint32_t (&B)[32][2] = g_mma_b[warp];
    A[lane][0] = a0; A[lane][1] = a1; A[lane][2] = a2; A[lane][3] = a3; B[lane][0] = b0; B[lane][1] = b1;
    g_warp_barriers[warp]->arrive_and_wait();
    auto tf32 = [](uint32_t u) { u &= 0xFFFFE000u; float f; std::memcpy(&f, &u, 4); return (double)f; };
    for (int r = 0; r < 4; r++) {
        const unsigned m = g + 8 * (r >> 1), n = 2 * t + (r & 1);
        double sum = (double)c[r];
        for (unsigned k = 0; k < 8; k++)
            sum += tf32(A[(m & 7) * 4 + (k & 3)][(m >> 3) + 2 * (k >> 2)]) * tf32(B[n * 4 + (k & 3)][k >> 2]);
        float f = (float)sum;                                     // round to nearest, then step back if that rounded away from zero
        if (std::fabs((double)f) > std::fabs(sum)) f = std::nextafterf(f, 0.0f);
        c[r] = f;
    }
    g_warp_barriers[warp]->arrive_and_wait();
}

struct Pending { uint32_t dst; const void* src; uint32_t ic, iw; };
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
    if (g_eager) { std::memcpy(smem_at(dst, 16), src, 16); note_write_done(dst, 16, t_cta_epoch, t_warp_epoch); return; }
    t_open.push_back(Pending{dst, src, t_cta_epoch, t_warp_epoch});
}
void cp_async_commit_group() { t_groups.push_back(std::move(t_open)); t_open.clear(); }
static void perform(const std::vector<Pending>& g) {
    for (const Pending& c : g) { std::memcpy(smem_at(c.dst, 16), c.src, 16); note_write_done(c.dst, 16, c.ic, c.iw); }
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

// ================================================================================================
// Emulated CUDA runtime for the API layer (csrc/arkcos_api.cu compiled with ARKCOS_HOST_EMU): "device" memory is
// host memory with red zones, streams and events are in-order no-ops (every launch runs to completion before it
// returns), cudaFuncSetAttribute is recorded and a launch that asks for more dynamic shared memory than its
// kernel was granted fails as on the device (cudaErrorInvalidValue).
// ================================================================================================
namespace emu {
constexpr size_t kRedZone = 4096;
struct Block { unsigned char* base; size_t bytes; };
static std::map<const void*, Block> g_blocks;                 // user pointer -> allocation
static std::map<const void*, int> g_max_dyn_smem;             // kernel -> MaxDynamicSharedMemorySize
static cudaError_t g_last_error = cudaSuccess;
static unsigned long long g_launches = 0, g_ctas = 0;

static void refresh_ranges() {
    g_global.clear();
    for (auto& kv : g_blocks) g_global.push_back(Range{(const unsigned char*)kv.first, (const unsigned char*)kv.first + kv.second.bytes});
}
static void* device_alloc(size_t bytes) {
    unsigned char* base = (unsigned char*)std::aligned_alloc(256, ((bytes + 255) / 256) * 256 + 2 * kRedZone);
    if (!base) return nullptr;
    std::memset(base, 0xA5, kRedZone);
    std::memset(base + kRedZone, 0xFF, ((bytes + 255) / 256) * 256);          // fresh device memory reads as NaN
    std::memset(base + kRedZone + ((bytes + 255) / 256) * 256, 0xA5, kRedZone);
    g_blocks[base + kRedZone] = Block{base, bytes};
    refresh_ranges();
    return base + kRedZone;
}
// 0 if every red zone is intact, else 1 + index of the first damaged block
static int check_red_zones() {
    int k = 0;
    for (auto& kv : g_blocks) {
        const unsigned char* lo = kv.second.base; const unsigned char* hi = (const unsigned char*)kv.first + ((kv.second.bytes + 255) / 256) * 256;
        for (size_t i = 0; i < kRedZone; i++) if (lo[i] != 0xA5 || hi[i] != 0xA5) return 1 + k;
        k++;
    }
    return 0;
}
template <typename P>
static void launch(void (*kernel)(P), dim3 grid, dim3 block, size_t smem, const P& params) {
    g_last_error = cudaSuccess;
    auto it = g_max_dyn_smem.find((const void*)kernel);
    const size_t granted = it == g_max_dyn_smem.end() ? 48 * 1024 : (size_t)it->second;
    if (smem > granted || block.x == 0 || block.x > 1024 || block.x % 32 || grid.x == 0 || grid.y == 0 || grid.y > 65535) { g_last_error = cudaErrorInvalidValue; return; }
    g_gridDim = grid;
    g_launches++;
    for (unsigned by = 0; by < grid.y; by++)
        for (unsigned bx = 0; bx < grid.x; bx++) { g_ctas++; run_cta(bx, by, block.x, smem, [&] { kernel(params); }); }
    if (check_red_zones()) fail("a kernel wrote outside a device allocation (block index)", check_red_zones() - 1, 0);
}
}  // namespace emu

inline cudaError_t cudaMalloc(void** p, size_t bytes) { *p = emu::device_alloc(bytes); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
inline cudaError_t cudaFree(void* p) {
    if (!p) return cudaSuccess;
    auto it = emu::g_blocks.find(p);
    if (it == emu::g_blocks.end()) emu::fail("cudaFree of an unknown pointer", 0, 0);
    std::free(it->second.base); emu::g_blocks.erase(it); emu::refresh_ranges();
    return cudaSuccess;
}
inline cudaError_t cudaMemcpy(void* d, const void* s, size_t n, int) { std::memcpy(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, int, cudaStream_t) { std::memcpy(d, s, n); return cudaSuccess; }
inline cudaError_t cudaMemset(void* d, int v, size_t n) { std::memset(d, v, n); return cudaSuccess; }
inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
inline cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int) { p->major = 10; p->minor = 0; p->multiProcessorCount = 148; return cudaSuccess; }
inline cudaError_t cudaGetLastError() { cudaError_t e = emu::g_last_error; emu::g_last_error = cudaSuccess; return e; }
inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : e == cudaErrorMemoryAllocation ? "out of memory" : "invalid value (emulated)"; }
template <typename K>
inline cudaError_t cudaFuncSetAttribute(K* kernel, int attr, int value) {
    if (attr == cudaFuncAttributeMaxDynamicSharedMemorySize) {
        if (value > 227 * 1024) return cudaErrorInvalidValue;     // sm_100: 227 KB per CTA
        emu::g_max_dyn_smem[(const void*)kernel] = value;
    }
    return cudaSuccess;
}
inline cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = new emu::Event{0.0}; return cudaSuccess; }
inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned) { return cudaEventCreate(e); }
inline cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
inline cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->t = emu::wall_ms(); return cudaSuccess; }
inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
inline cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) { *ms = (float)(b->t - a->t) + 1e-6f; return cudaSuccess; }
inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = new emu::Stream{}; return cudaSuccess; }
inline cudaError_t cudaStreamDestroy(cudaStream_t s) { delete s; return cudaSuccess; }
inline cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
