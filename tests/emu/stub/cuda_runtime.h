// Stub <cuda_runtime.h> for the HOST EMULATION of the arkcos CUDA kernels (tests/emu/).  Test
// infrastructure only: it lets `-m "not gpu"` tests execute the very kernel source of
// paper_1211_3556_b200/csrc/arkcos_kernels.cuh on CPU threads (one OS thread per CUDA thread, one CTA
// at a time) with bounds- and alignment-checked shared memory, so that index logic can be checked
// against the oracle on machines without a GPU.  Nothing in the product links or includes this.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __launch_bounds__(...)
#define __shared__
#define __restrict__

struct dim3 { unsigned x = 1, y = 1, z = 1; dim3(unsigned a = 1, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {} };
struct uint3 { unsigned x, y, z; };
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) uint4 { unsigned x, y, z, w; };
struct alignas(8) float2 { float x, y; };
static inline float4 make_float4(float a, float b, float c, float d) { return float4{a, b, c, d}; }
static inline float2 make_float2(float a, float b) { return float2{a, b}; }

using std::max;
using std::min;

// ---- the part of the CUDA runtime API the library's API layer uses (implemented in emu_runtime.h) ----
#include <chrono>
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2 };
enum { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2 };
enum { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributePreferredSharedMemoryCarveout = 9, cudaSharedmemCarveoutMaxShared = 100 };
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };
namespace emu {
struct Event { double t; };
struct Stream {};
static inline double wall_ms() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count(); }
}
typedef emu::Event* cudaEvent_t;
typedef emu::Stream* cudaStream_t;
struct cudaDeviceProp { int major, minor, multiProcessorCount; };

namespace emu {
extern thread_local uint3 t_threadIdx, t_blockIdx;
extern dim3 g_blockDim, g_gridDim;
extern unsigned char* g_smem;         // base of the CTA's dynamic shared memory
extern size_t g_smem_bytes;           // its size for the current launch
void sync_threads();                  // CTA barrier
void sync_warp();                     // warp barrier
[[noreturn]] void fail(const char* what, long a, long b);
// checked shared-memory window [addr, addr + bytes), aligned to `bytes`
static inline unsigned char* smem_at(uint32_t addr, uint32_t bytes) {
    if ((size_t)addr + bytes > g_smem_bytes) fail("shared-memory access out of bounds", addr, bytes);
    if (addr % bytes) fail("misaligned shared-memory access", addr, bytes);
    return g_smem + addr;
}
// shared-memory hazard checker (emu_main.cpp): the CPU counterpart of `compute-sanitizer --tool racecheck` for the
// accesses that go through the kernels' PTX wrappers (ld.shared reads, cp.async writes)
void note_read(uint32_t addr, uint32_t bytes);
// bank-conflict accounting (EMU_BANKS=<report file>; emu_runtime.h): the call site identifies the instruction
extern bool g_banks;
void bank_note(uint32_t addr, uint32_t bytes, int kind);   // kind: 0 = ld.shared, 1 = st.shared, 2 = cp.async destination
static inline __attribute__((always_inline)) unsigned char* smem_read(uint32_t addr, uint32_t bytes) {
    unsigned char* p = smem_at(addr, bytes); note_read(addr, bytes);
    if (g_banks) bank_note(addr, bytes, 0);
    return p;
}
void note_store(uint32_t addr, uint32_t bytes);   // a plain st.shared: checked against earlier readers / writers, visible at once
static inline __attribute__((always_inline)) unsigned char* smem_write(uint32_t addr, uint32_t bytes) {
    unsigned char* p = smem_at(addr, bytes); note_store(addr, bytes);
    if (g_banks) bank_note(addr, bytes, 1);
    return p;
}
// warp-level tensor-core instruction mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 (arkcos_tensor.cuh)
void mma_m16n8k8_tf32(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0, uint32_t b1);
void check_global(const void* p, size_t bytes);   // must lie inside a registered global buffer, 16-byte aligned
// cp.async emulation: copies are queued per thread and only performed by the wait calls
void cp_async_enqueue(uint32_t dst, const void* src) __attribute__((noinline));
void cp_async_commit_group();
void cp_async_wait(int keep_groups);
}  // namespace emu

#define threadIdx (emu::t_threadIdx)
#define blockIdx (emu::t_blockIdx)
#define blockDim (emu::g_blockDim)
#define gridDim (emu::g_gridDim)
static inline void __syncthreads() { emu::sync_threads(); }
static inline void __syncwarp() { emu::sync_warp(); }
static inline double __ldg(const double* p) { return *p; }
static inline float __uint_as_float(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }
static inline uint32_t __float_as_uint(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
static inline size_t __cvta_generic_to_shared(const void* p) { return (size_t)((const unsigned char*)p - emu::g_smem); }
