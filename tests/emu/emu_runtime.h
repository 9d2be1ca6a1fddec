// emu_runtime.h - the HOST EMULATION runtime of the arkcos CUDA kernels.  Test infrastructure only; included
// once per emulation binary (emu_main.cpp: the kernel-level command-line harness; emu_api.cpp: the whole C-ABI
// library compiled for the host).
//
// One FIBER per CUDA thread, one CTA at a time, scheduled round-robin by a single OS thread: a fiber runs
// until it reaches __syncthreads / __syncwarp / a warp-collective instruction, where it waits until every live
// thread of the CTA / warp has arrived (a barrier that can never complete - divergent barriers, a thread that exited
// while its warp waits - is reported as a DEADLOCK instead of hanging).  cp.async is
// performed only at its wait (EMU_EAGER=1: at issue), shared memory a heap block of exactly the launch's dynamic
// size with bounds- and alignment-checked ld.shared wrappers, checked cp.async sources, NaN-initialised shared
// memory, and a shared-memory hazard checker (the CPU counterpart of compute-sanitizer racecheck).
#pragma once
#if !defined(__x86_64__)
#include <ucontext.h>
#endif

#include <map>
#include <memory>
#include <string>
#include <unordered_map>
#if defined(__SANITIZE_ADDRESS__)
#include <sanitizer/common_interface_defs.h>
#endif

#include "cuda_runtime.h"

namespace emu {
thread_local uint3 t_threadIdx, t_blockIdx;
dim3 g_blockDim, g_gridDim;
unsigned char* g_smem = nullptr;
size_t g_smem_bytes = 0;

enum WaitKind { kRunnable = 0, kWaitCta = 1, kWaitWarp = 2, kWaitCollective = 3, kDone = 4 };
static void fiber_wait(int kind);        // yield to the scheduler until the barrier of that kind completes
struct Range { const unsigned char* lo; const unsigned char* hi; };
static std::vector<Range> g_global;      // buffers a cp.async may read: registered by the harness, or by the emulated cudaMalloc

[[noreturn]] void fail(const char* what, long a, long b) {
    std::fprintf(stderr, "EMU FAILURE: %s (%ld, %ld) block %u thread %u\n", what, a, b, t_blockIdx.x, t_threadIdx.x);
    std::_Exit(3);
}
static thread_local uint32_t t_cta_epoch = 0, t_warp_epoch = 0;   // barriers this thread has passed (hazard checker below)
void sync_threads() { fiber_wait(kWaitCta); ++t_cta_epoch; }
void sync_warp() { fiber_wait(kWaitWarp); ++t_warp_epoch; }
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
static const bool g_racecheck = std::getenv("EMU_NO_RACECHECK") == nullptr;
static bool ordered_after(const Stamp& a) {                        // is the calling thread's access ordered after stamp a?
    if (!a.valid || a.tid == t_threadIdx.x) return true;
    if (t_cta_epoch > a.cta_epoch) return true;
    return (a.tid >> 5) == (t_threadIdx.x >> 5) && t_warp_epoch > a.warp_epoch;
}
static Stamp now() { return Stamp{(uint16_t)t_threadIdx.x, 1, t_cta_epoch, t_warp_epoch}; }
void note_read(uint32_t addr, uint32_t bytes) {
    if (!g_racecheck) return;
    for (uint32_t w = addr / 4; w < (addr + bytes + 3) / 4; w++) {
        if (!ordered_after(g_writer[w])) fail("shared-memory hazard: read of a word another thread wrote without a barrier in between (word, writer)", w, g_writer[w].tid);
        const Stamp& r = g_reader[w];
        if (!r.valid || t_cta_epoch >= r.cta_epoch) g_reader[w] = now();
    }
}
static void note_write_issue(uint32_t addr, uint32_t bytes) {
    if (!g_racecheck) return;
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
// The meeting is a warp rendezvous that is NOT counted for the hazard checker: mma.sync converges the warp but
// orders no shared-memory access.
static uint32_t g_mma_a[2][32][32][4], g_mma_b[2][32][32][2];   // [parity of the warp's mma count][warp][lane][register]
static unsigned g_mma_count[32][32];                             // per warp and lane: mma instructions executed in this CTA
void mma_m16n8k8_tf32(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1) {
    const unsigned warp = t_threadIdx.x >> 5, lane = t_threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    // two exchange buffers used alternately: one rendezvous per instruction is enough, because a lane can only
    // overwrite buffer p two instructions later, after every lane has passed the rendezvous in between
    const unsigned par = g_mma_count[warp][lane]++ & 1u;
    uint32_t (&A)[32][4] = g_mma_a[par][warp]; uint32_t (&B)[32][2] = g_mma_b[par][warp];
    A[lane][0] = a0; A[lane][1] = a1; A[lane][2] = a2; A[lane][3] = a3; B[lane][0] = b0; B[lane][1] = b1;
    fiber_wait(kWaitCollective);
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
}

// ---- shared-memory bank-conflict accounting (EMU_BANKS=<report file>) --------------------------------------
// What ncu reports as l1tex__data_bank_conflicts_pipe_lsu_mem_shared, from the addresses the emulation sees: the
// accesses of the 32 lanes of a warp that belong to one executed instruction are matched by (warp, barrier counts,
// call site = the instruction's address in the emulation binary, occurrence of that site since the last barrier);
// shared memory has 32 banks of 4 bytes, a 16-byte access is served a quarter warp at a time, an 8-byte access a
// half warp, and a phase takes as many wavefronts as the largest number of DIFFERENT words it touches in one bank
// (equal words are a broadcast).  Report per (kernel, site): instructions, wavefronts, conflict-free wavefronts.
bool g_banks = std::getenv("EMU_BANKS") != nullptr;
const char* g_kernel_name = "?";
struct BankKey {
    uint32_t warp, ce, we, occ; uintptr_t site;
    bool operator==(const BankKey& o) const { return warp == o.warp && ce == o.ce && we == o.we && occ == o.occ && site == o.site; }
};
struct BankKeyHash { size_t operator()(const BankKey& k) const { return std::hash<uint64_t>()(((uint64_t)k.warp << 48) ^ ((uint64_t)k.ce << 40) ^ ((uint64_t)k.we << 20) ^ k.occ ^ (k.site * 0x9E3779B97F4A7C15ull)); } };
struct BankEntry { uint32_t addr[32]; uint32_t mask = 0; uint8_t bytes = 0, kind = 0; };
struct SiteStat { unsigned long long instrs = 0, waves = 0, ideal = 0; unsigned worst = 0; unsigned bytes = 0, kind = 0; };
static std::unordered_map<BankKey, BankEntry, BankKeyHash> g_bank_entries;                 // of the running CTA
static std::map<std::pair<std::string, uintptr_t>, SiteStat> g_site_stats;                // of the whole run
struct Occurrences { uint32_t ce = ~0u, we = ~0u; std::unordered_map<uintptr_t, uint32_t> count; };
static std::vector<Occurrences> g_occ;                                                     // per thread of the CTA
__attribute__((noinline)) void bank_note(uint32_t addr, uint32_t bytes, int kind) {
    const uintptr_t site = (uintptr_t)__builtin_return_address(0);
    const unsigned tid = t_threadIdx.x;
    if (g_occ.size() <= tid) g_occ.resize(tid + 1);
    Occurrences& oc = g_occ[tid];
    if (oc.ce != t_cta_epoch || oc.we != t_warp_epoch) { oc.ce = t_cta_epoch; oc.we = t_warp_epoch; oc.count.clear(); }
    const uint32_t occ = oc.count[site]++;
    BankEntry& e = g_bank_entries[BankKey{tid >> 5, t_cta_epoch, t_warp_epoch, occ, site}];
    e.addr[tid & 31] = addr; e.mask |= 1u << (tid & 31); e.bytes = (uint8_t)bytes; e.kind = (uint8_t)kind;
}
static void bank_finish_cta() {
    for (auto& kv : g_bank_entries) {
        const BankEntry& e = kv.second;
        const unsigned lanes_per_phase = e.bytes >= 16 ? 8 : e.bytes == 8 ? 16 : 32, words = e.bytes / 4 ? e.bytes / 4 : 1;
        unsigned waves = 0, ideal = 0;
        for (unsigned l0 = 0; l0 < 32; l0 += lanes_per_phase) {
            std::vector<uint32_t> per_bank[32];
            bool any = false;
            for (unsigned l = l0; l < l0 + lanes_per_phase; l++) {
                if (!(e.mask >> l & 1u)) continue;
                any = true;
                for (unsigned j = 0; j < words; j++) {
                    const uint32_t word = e.addr[l] / 4 + j;
                    auto& v = per_bank[word & 31];
                    if (std::find(v.begin(), v.end(), word) == v.end()) v.push_back(word);
                }
            }
            if (!any) continue;
            unsigned worst = 1;
            for (auto& v : per_bank) worst = std::max<unsigned>(worst, (unsigned)v.size());
            waves += worst; ideal += 1;
        }
        SiteStat& st = g_site_stats[{g_kernel_name, kv.first.site}];
        st.instrs++; st.waves += waves; st.ideal += ideal; st.worst = std::max(st.worst, ideal ? (waves + ideal - 1) / ideal : 0u);
        st.bytes = e.bytes; st.kind = e.kind;
    }
    g_bank_entries.clear();
    g_occ.clear();
}
// one line per (kernel, instruction site): kernel kind bytes instructions wavefronts conflict-free-wavefronts worst-factor
static void bank_report() {
    const char* path = std::getenv("EMU_BANKS");
    if (!path) return;
    FILE* f = std::fopen(path, "w");
    if (!f) return;
    for (auto& kv : g_site_stats)
        std::fprintf(f, "%s %s %u %llu %llu %llu %u\n", kv.first.first.c_str(), kv.second.kind == 0 ? "ld.shared" : kv.second.kind == 1 ? "st.shared" : "cp.async",
                     kv.second.bytes, kv.second.instrs, kv.second.waves, kv.second.ideal, kv.second.worst);
    std::fclose(f);
}

struct Pending { uint32_t dst; const void* src; uint32_t ic, iw; };
static thread_local std::vector<std::vector<Pending>> t_groups;   // committed groups, oldest first
static thread_local std::vector<Pending> t_open;                  // not yet committed
// Two modes bracket what the hardware may do with a cp.async: DEFERRED (default) performs the copy only at
// the wait - a read before the wait sees stale data (RAW hazard); EAGER (EMU_EAGER=1) performs it at once - a
// copy into a buffer that other threads still read clobbers it (WAR hazard).
static const bool g_eager = std::getenv("EMU_EAGER") != nullptr;
void cp_async_enqueue(uint32_t dst, const void* src) {
    if (g_banks) {                                       // the destination side of the LDGSTS; site = the caller's instruction
        const uintptr_t site = (uintptr_t)__builtin_return_address(0);
        const unsigned tid = t_threadIdx.x;
        if (g_occ.size() <= tid) g_occ.resize(tid + 1);
        Occurrences& oc = g_occ[tid];
        if (oc.ce != t_cta_epoch || oc.we != t_warp_epoch) { oc.ce = t_cta_epoch; oc.we = t_warp_epoch; oc.count.clear(); }
        const uint32_t occ = oc.count[site]++;
        BankEntry& e = g_bank_entries[BankKey{tid >> 5, t_cta_epoch, t_warp_epoch, occ, site}];
        e.addr[tid & 31] = dst; e.mask |= 1u << (tid & 31); e.bytes = 16; e.kind = 2;
    }
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

// ---- fibers ------------------------------------------------------------------------------------------------
// Context switch.  glibc's swapcontext makes two system calls per switch (it saves and restores the signal mask),
// which dominated the run time of the emulation; on x86-64 the switch is therefore a dozen instructions of our own
// (callee-saved registers + stack pointer, System V ABI), ucontext elsewhere.
#if defined(__x86_64__)
extern "C" void arkcos_emu_switch(void** save_sp, void* load_sp);
asm(".text\n.globl arkcos_emu_switch\n.type arkcos_emu_switch,@function\narkcos_emu_switch:\n"
    "  pushq %rbp\n  pushq %rbx\n  pushq %r12\n  pushq %r13\n  pushq %r14\n  pushq %r15\n"
    "  movq %rsp, (%rdi)\n  movq %rsi, %rsp\n"
    "  popq %r15\n  popq %r14\n  popq %r13\n  popq %r12\n  popq %rbx\n  popq %rbp\n  ret\n"
    ".size arkcos_emu_switch, .-arkcos_emu_switch\n");
struct Context { void* sp = nullptr; };
static void context_switch(Context& from, Context& to) { arkcos_emu_switch(&from.sp, to.sp); }
static void context_make(Context& c, unsigned char* stack, size_t bytes, void (*entry)()) {
    uintptr_t top = ((uintptr_t)stack + bytes) & ~(uintptr_t)15;
    void** sp = (void**)top;
    *--sp = nullptr;                       // the "return address" of entry (it never returns)
    *--sp = (void*)entry;                  // popped by the ret of the first switch: entry starts with rsp = 8 mod 16
    for (int r = 0; r < 6; r++) *--sp = nullptr;
    c.sp = sp;
}
#else
struct Context { ucontext_t uc; };
static void context_switch(Context& from, Context& to) { swapcontext(&from.uc, &to.uc); }
static void context_make(Context& c, unsigned char* stack, size_t bytes, void (*entry)()) {
    getcontext(&c.uc);
    c.uc.uc_stack.ss_sp = stack; c.uc.uc_stack.ss_size = bytes; c.uc.uc_link = nullptr;
    makecontext(&c.uc, entry, 0);
}
#endif

struct Fiber {
    Context ctx;
    std::unique_ptr<unsigned char[]> stack;
    uint3 tid{0, 0, 0};
    uint32_t cta_epoch = 0, warp_epoch = 0;
    std::vector<std::vector<Pending>> groups;
    std::vector<Pending> open;
    int state = kDone;
    void* fake_stack = nullptr;           // AddressSanitizer's bookkeeping across a switch
};
constexpr size_t kFiberStack = 512 * 1024;
static std::vector<Fiber> g_fibers;
static Fiber* g_cur = nullptr;
static Context g_sched_ctx;
static void* g_sched_fake_stack = nullptr;
static const void* g_sched_stack_bottom = nullptr;
static size_t g_sched_stack_size = 0;
static void (*g_body)(void*) = nullptr;
static void* g_body_arg = nullptr;

static void switch_to_scheduler(bool dying) {
    Fiber* f = g_cur;
#if defined(__SANITIZE_ADDRESS__)
    __sanitizer_start_switch_fiber(dying ? nullptr : &f->fake_stack, g_sched_stack_bottom, g_sched_stack_size);
#endif
    context_switch(f->ctx, g_sched_ctx);
#if defined(__SANITIZE_ADDRESS__)
    __sanitizer_finish_switch_fiber(f->fake_stack, &g_sched_stack_bottom, &g_sched_stack_size);
#endif
}
static void fiber_wait(int kind) {
    Fiber* f = g_cur;
    f->state = kind;
    f->cta_epoch = t_cta_epoch; f->warp_epoch = t_warp_epoch;
    std::swap(f->groups, t_groups); std::swap(f->open, t_open);
    switch_to_scheduler(false);
}
static void fiber_entry() {
#if defined(__SANITIZE_ADDRESS__)
    __sanitizer_finish_switch_fiber(nullptr, &g_sched_stack_bottom, &g_sched_stack_size);
#endif
    g_body(g_body_arg);
    thread_exit_check();
    g_cur->state = kDone;
    switch_to_scheduler(true);
}
static void resume(Fiber& f) {
    g_cur = &f;
    t_threadIdx = f.tid; t_cta_epoch = f.cta_epoch; t_warp_epoch = f.warp_epoch;
    std::swap(f.groups, t_groups); std::swap(f.open, t_open);
    f.state = kRunnable;
#if defined(__SANITIZE_ADDRESS__)
    __sanitizer_start_switch_fiber(&g_sched_fake_stack, f.stack.get(), kFiberStack);
#endif
    context_switch(g_sched_ctx, f.ctx);
#if defined(__SANITIZE_ADDRESS__)
    __sanitizer_finish_switch_fiber(g_sched_fake_stack, nullptr, nullptr);
#endif
    g_cur = nullptr;
}

// run one CTA of `threads` threads
template <typename F>
static void run_cta(unsigned bx, unsigned by, unsigned threads, size_t smem_bytes, F&& body) {
    g_smem_bytes = smem_bytes;
    g_smem = (unsigned char*)std::malloc(smem_bytes ? smem_bytes : 16);
    std::memset(g_smem, 0xFF, smem_bytes);                        // NaN pattern
    g_writer.assign(smem_bytes / 4 + 4, Stamp{0, 0, 0, 0}); g_reader.assign(smem_bytes / 4 + 4, Stamp{0, 0, 0, 0});
    g_blockDim = dim3(threads);
    t_blockIdx = uint3{bx, by, 0};
    std::memset(g_mma_count, 0, sizeof(g_mma_count));
    if (g_fibers.size() < threads) g_fibers.resize(threads);
    auto thunk = [](void* p) { (*static_cast<std::remove_reference_t<F>*>(p))(); };
    g_body = thunk; g_body_arg = &body;
    for (unsigned t = 0; t < threads; t++) {
        Fiber& f = g_fibers[t];
        if (!f.stack) f.stack.reset(new unsigned char[kFiberStack]);
        f.tid = uint3{t, 0, 0}; f.cta_epoch = f.warp_epoch = 0; f.groups.clear(); f.open.clear(); f.state = kRunnable; f.fake_stack = nullptr;
        context_make(f.ctx, f.stack.get(), kFiberStack, fiber_entry);
    }
    const unsigned warps = threads / 32;
    for (;;) {
        bool ran = false, all_done = true;
        for (unsigned t = 0; t < threads; t++)
            if (g_fibers[t].state == kRunnable) { resume(g_fibers[t]); ran = true; }
        // barriers complete when every LIVE thread of the CTA / warp waits at the same kind of barrier
        unsigned live = 0, at_cta = 0;
        for (unsigned t = 0; t < threads; t++) { const int st = g_fibers[t].state; live += st != kDone; at_cta += st == kWaitCta; all_done &= st == kDone; }
        if (all_done) break;
        bool released = false;
        if (live > 0 && at_cta == live) { for (unsigned t = 0; t < threads; t++) if (g_fibers[t].state == kWaitCta) g_fibers[t].state = kRunnable; released = true; }
        for (unsigned w = 0; w < warps; w++)
            for (const int kind : {kWaitWarp, kWaitCollective}) {
                unsigned wl = 0, at = 0;
                for (unsigned l = 0; l < 32; l++) { const int st = g_fibers[32 * w + l].state; wl += st != kDone; at += st == kind; }
                if (wl > 0 && at == wl) { for (unsigned l = 0; l < 32; l++) if (g_fibers[32 * w + l].state == kind) g_fibers[32 * w + l].state = kRunnable; released = true; }
                // a warp-collective instruction needs all 32 lanes
                if (kind == kWaitCollective && at > 0 && at == wl && wl != 32) fail("warp-collective instruction executed by a partial warp (warp, lanes)", w, wl);
            }
        if (!ran && !released) {
            for (unsigned t = 0; t < threads; t++)
                if (g_fibers[t].state != kDone) { t_threadIdx = g_fibers[t].tid; fail("DEADLOCK: a barrier can never complete (waiting thread's barrier kind 1 = CTA, 2 = warp, 3 = collective; live threads)", g_fibers[t].state, live); }
        }
    }
    if (g_banks) bank_finish_cta();
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
