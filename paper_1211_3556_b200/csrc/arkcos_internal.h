// arkcos_internal.h - data structures shared by the host scheduler (S1) and the CUDA kernels (S2, S3).
// Product code; shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

#ifdef __CUDACC__
#define ARKCOS_HD __host__ __device__
#else
#define ARKCOS_HD
#endif

namespace arkcos {

// ---- tiling constants of the convolution kernel ---------------------
constexpr int kP = 16;                 // outputs per thread in phi (register-blocked sliding window)
constexpr int kWarpSpan = 32 * kP;     // 512 contiguous phi outputs per warp
constexpr int kWarps = 8;              // warps per CTA
constexpr int kThreads = 32 * kWarps;
constexpr int kMaxF = 8;               // a CTA covers F phi sub-tiles x S = kWarps/F tap splits
constexpr int kGenUnitTaps = 1024;     // taps per weight-generator work unit

// Tap block (taps staged per shared-memory fill) as a function of log2(F).
ARKCOS_HD constexpr int tap_block(int f_log2) { return f_log2 == 3 ? 512 : (f_log2 == 2 ? 1024 : 2048); }

// One (north output ring i, input ring j = i + r) pair.  The southern mirror pair
// (n_theta-1-i, n_theta-1-j) has identical weights and is computed by the same CTA (FFMA2 lanes).
struct PairDesc {
    uint32_t w_off;   // offset, in floats, of the stored weights; multiple of 4
    int32_t start;    // dphi index d of stored tap 0 (even, <= 0)
    int32_t ntaps;    // stored taps, multiple of 4; 0 = nothing to do
    int32_t half;     // D (taps -D..D inside theta_cut); n_phi = whole ring; -1 = empty
};

// One CTA of the convolution launch.
struct Item {
    int32_t i_north;  // output ring in the northern half; the CTA also produces ring n_theta-1-i
    int32_t k0;       // first output phi of the tile
    int32_t f_log2;   // F = 1 << f_log2 sub-tiles of 512 outputs; S = kWarps / F tap splits
    int32_t row_lo;   // first input-row slot r (0..2R) this CTA sums (cluster splitting; 0 in v1)
};

struct GenUnit {
    uint32_t pair;    // index into the PairDesc array
    uint32_t e0;      // first stored tap of the unit
};

// Host-side result of step S1 (the ring-pair scheduler).  FP64 throughout.
struct Schedule {
    int n_theta = 0, n_phi = 0;
    double theta_cut = 0.0;
    int R = 0;                              // ring half band
    int n_north = 0;                        // ceil(n_theta / 2)
    double h_cut = 0.0;                     // sin^2(theta_cut / 2)
    std::vector<double> sin_t;              // [n_theta] sin(theta_i)
    std::vector<double> area;               // [n_theta] exact ring pixel area A_j
    std::vector<double> a_r;                // [R+1] sin^2(r dtheta / 2)
    std::vector<double> s2;                 // [n_phi/2+1] sin^2(d dphi / 2)
    std::vector<PairDesc> pairs;            // [n_north][2R+1]
    std::vector<Item> items;                // cost-sorted, heaviest first
    std::vector<GenUnit> gen_units;
    unsigned long long pair_evals = 0;      // useful FMAs per map
    unsigned long long weights = 0;         // in-support weights, no symmetry reduction
    unsigned long long fma_slots = 0;       // FMA lanes issued per map (padding included)
    unsigned long long weight_slots = 0;    // floats in the weight buffer

    // window of ring pair (i, j) for ANY i (southern rings through the mirror): -1 / D / n_phi
    int window(int i, int j) const;
    const PairDesc* pair(int i_north, int j) const {
        int r = j - i_north + R;
        if (i_north < 0 || i_north >= n_north || r < 0 || r > 2 * R) return nullptr;
        return &pairs[(size_t)i_north * (2 * R + 1) + r];
    }
};

// Builds the schedule.  Returns 0 on success, 1 = invalid argument, 4 = unsupported (matches arkcos_status).
int build_schedule(int n_theta, int n_phi, double theta_cut, int sm_count, Schedule& out);

}  // namespace arkcos
