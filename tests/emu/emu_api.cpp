// emu_api.cpp - the WHOLE C-ABI library (csrc/arkcos_api.cu: plan creation, uploads, launch configuration, the host
// pipeline, the spectral path) compiled for the host against the emulated CUDA runtime of emu_runtime.h.
// Test infrastructure only: tests/test_emu_api.py loads the resulting tests/emu/libarkcos_emu.so through the same
// ctypes binding as the product's libarkcos.so and runs the API-level scenarios of the GPU suite on small grids,
// with "device" buffers that are host memory with red zones.  The product never loads this library.
#include "../../paper_1211_3556_b200/csrc/arkcos_api.cu"

extern "C" {
void* arkcos_emu_device_alloc(unsigned long long bytes) { return emu::device_alloc((size_t)bytes); }
void arkcos_emu_device_free(void* p) { (void)cudaFree(p); }
int arkcos_emu_check_red_zones(void) { return emu::check_red_zones(); }
unsigned long long arkcos_emu_launches(void) { return emu::g_launches; }
unsigned long long arkcos_emu_ctas(void) { return emu::g_ctas; }
}
