// emu_spectral.cpp - HOST EMULATION harness of the spectral-path kernels (csrc/arkcos_spectral.cuh, N2).  Test
// infrastructure only; same runtime as emu_main.cpp (tests/emu/emu_runtime.h: one fiber per CUDA thread, barriers with
// deadlock detection, shared memory a heap block of exactly the launch's size under AddressSanitizer).
//
//   emu_spectral n_theta n_phi theta_cut n_table table.f64 in.f32 out.f32
#include "emu_runtime.h"

#include "arkcos_internal.h"
#include "arkcos_spectral.cuh"

template <typename T>
static std::vector<T> read_file(const char* path, size_t n) {
    std::vector<T> v(n);
    FILE* f = std::fopen(path, "rb");
    if (!f || std::fread(v.data(), sizeof(T), n, f) != n) { std::fprintf(stderr, "cannot read %s\n", path); std::exit(2); }
    std::fclose(f);
    return v;
}

int main(int argc, char** argv) {
    using namespace arkcos;
    if (argc < 8) { std::fprintf(stderr, "usage: emu_spectral n_theta n_phi theta_cut n_table table.f64 in.f32 out.f32\n"); return 2; }
    const int n_theta = std::atoi(argv[1]), n = std::atoi(argv[2]);
    const double theta_cut = std::atof(argv[3]);
    const int n_table = std::atoi(argv[4]);
    std::vector<double> table = read_file<double>(argv[5], (size_t)n_table);
    const size_t n_pix = (size_t)n_theta * n;
    std::vector<float> in = read_file<float>(argv[6], n_pix);
    std::vector<float> out(n_pix, std::nanf(""));
    if (n < 16 || n > kSpecMaxPhi || (n & (n - 1))) { std::fprintf(stderr, "n_phi must be a power of two\n"); return 2; }

    Schedule s;
    if (build_schedule(n_theta, n, theta_cut, 148, s) != 0) { std::fprintf(stderr, "build_schedule failed\n"); return 2; }
    const int h = n / 2, W = 2 * s.R + 1;
    const double kPi = 3.14159265358979323846264338327950288;
    // what build_spectral (csrc/arkcos_api.cu) uploads
    std::vector<SpecPair> sp((size_t)s.n_north * W);
    for (int i = 0; i < s.n_north; i++)
        for (int r = 0; r < W; r++) {
            const int j = i + r - s.R;
            SpecPair& g = sp[(size_t)i * W + r];
            g.half = s.pairs[(size_t)i * W + r].half; g.pad_ = 0;
            const bool live = g.half >= 0 && j >= 0 && j < n_theta;
            g.a = s.a_r[std::abs(r - s.R)]; g.b = live ? s.sin_t[i] * s.sin_t[j] : 0.0; g.area = live ? s.area[j] : 0.0;
            if (!live) g.half = -1;
        }
    std::vector<double> costab(n);
    for (int k = 0; k < n; k++) costab[k] = std::cos(2.0 * kPi * k / n);
    std::vector<float2> tw_h(std::max(1, h / 2)), tw_n(h + 1);
    for (int k = 0; k < h / 2; k++) tw_h[k] = make_float2((float)std::cos(2.0 * kPi * k / h), (float)-std::sin(2.0 * kPi * k / h));
    for (int m = 0; m <= h; m++) tw_n[m] = make_float2((float)std::cos(2.0 * kPi * m / n), (float)-std::sin(2.0 * kPi * m / n));
    std::vector<float> wspec(sp.size() * (size_t)(h + 1), std::nanf(""));
    std::vector<float2> xspec((size_t)n_theta * (h + 1), make_float2(std::nanf(""), std::nanf("")));

    SpecWeightParams w;
    w.pairs = sp.data(); w.s2 = s.s2.data(); w.table = table.data(); w.costab = costab.data(); w.wspec = wspec.data();
    w.n_pairs = (int)sp.size(); w.n_phi = n; w.n_table = n_table;
    w.t_scale = (double)(n_table - 1) / theta_cut; w.m_split = 0; w.theta_split = 0.0; w.t_scale2 = 0.0;
    const int wgrid = 3;
    emu::g_gridDim = dim3(wgrid);
    for (int b = 0; b < wgrid; b++) emu::run_cta((unsigned)b, 0, kSpecThreads, (size_t)(h + 1) * sizeof(double), [&] { k_spectral_weights(w); });

    SpecParams p;
    p.in = in.data(); p.out = out.data(); p.xspec = xspec.data(); p.wspec = wspec.data(); p.pairs = s.pairs.data();
    p.tw_h = tw_h.data(); p.tw_n = tw_n.data(); p.n_theta = n_theta; p.n_phi = n; p.R = s.R;
    emu::g_gridDim = dim3((unsigned)n_theta);
    for (int i = 0; i < n_theta; i++) emu::run_cta((unsigned)i, 0, kSpecThreads, (size_t)(2 * h + h / 2) * sizeof(float2), [&] { k_rfft_rings(p); });
    for (int i = 0; i < n_theta; i++) emu::run_cta((unsigned)i, 0, kSpecThreads, (size_t)(2 * h + 1 + h / 2) * sizeof(float2), [&] { k_spectral_apply(p); });

    FILE* f = std::fopen(argv[7], "wb");
    if (!f || std::fwrite(out.data(), sizeof(float), n_pix, f) != n_pix) { std::fprintf(stderr, "cannot write %s\n", argv[7]); return 2; }
    std::fclose(f);
    std::printf("emu spectral ok: R %d n_north %d pairs %zu\n", s.R, s.n_north, sp.size());
    return 0;
}
