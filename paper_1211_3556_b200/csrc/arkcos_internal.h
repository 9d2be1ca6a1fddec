// arkcos_internal.h - data structures shared by the host scheduler (S1) and the CUDA kernels (S2, S3).
// Product code; shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#ifdef __CUDACC__
#define ARKCOS_HD __host__ __device__
#else
#define ARKCOS_HD
#endif

namespace arkcos {

// ---- tiling constants of the convolution kernel ---------------------
// A lane owns kLaneP consecutive phi outputs of one ring in registers; a warp owns kWarpSpan.  The hot
// loops are plain FP32 FFMA with the (warp-uniform) weight as the re-used operand: measured on B200,
// that form issues at 124 of the 128 FMA/clk/SM, against 94 for the packed FFMA2 form.
constexpr int kLaneP = 32;             // outputs per lane in phi
constexpr int kWarpSpan = 32 * kLaneP; // 1024 contiguous phi outputs per warp
constexpr int kWarps = 8;              // warps per CTA
constexpr int kThreads = 32 * kWarps;
constexpr int kHaloNarrow = 32;        // narrow rings: every stored tap window lies inside [-32, 32)
constexpr int kGenUnitTaps = 1024;     // taps per weight-generator work unit (one warp)
constexpr int kSmemBudget = 220 * 1024;
constexpr int kSmemTwoPerSm = 113 * 1024; // dynamic shared memory of a CTA when two are to share an SM (228 KB - 2 x 1 KB reserved)

// Shared-memory rows are stored in lane tiles: 8 chunks of 16 bytes (the kLaneP floats one lane owns)
// followed by one pad chunk, so that the 16-byte / 8-byte loads of the 32 lanes of a warp (lane stride
// 144 bytes) are bank-conflict free.  Logical 16-byte chunk c sits at physical chunk c + (c >> 3).
constexpr int kTileBytes = 144;

// ---- NARROW items: band marching, kNarrowP outputs per lane ----------------------------------------
// A warp owns kNarrowSpan contiguous outputs of one ring; a lane's tile is kNarrowP floats = 4 chunks of 16
// bytes + 1 pad chunk (lane stride 80 bytes: the 16-byte window loads of a warp are bank-conflict free).
// Row slot = 2 left halo tiles + 32 own tiles + 2 right halo tiles + one spare tile (the software prefetch of
// the sliding window reads at most one tile past the right halo).
constexpr int kNarrowP = 16;
constexpr int kNarrowSpan = 32 * kNarrowP;           // 512 contiguous phi outputs per warp = per NARROW item
constexpr int kNarrowTileBytes = 80;
constexpr int kNarrowSlotBytes = (32 + 2 * (kHaloNarrow / kNarrowP) + 1) * kNarrowTileBytes;
// A ring's weight block of wcopy floats takes wcopy + kNarrowWPad floats of the shared weight area: the chain
// prefetches the 8 bytes after a run's last weight, and that read must not land in the neighbouring block, which in
// the double-buffered case is being filled for the next pass (harmless - the value is never used - but a
// shared-memory hazard for a race checker all the same).
constexpr int kNarrowWPad = 4;

// ---- WIDE items (windows of 64 .. n_phi taps): warp-autonomous path ------------------------------
// A warp owns kWarpSpan contiguous outputs of ONE ring and streams its share of the ring's taps through
// a private, double-buffered shared-memory stage of up to kWideStage taps.
constexpr int kWideStage = 512;                     // taps per stage; multiple of 4
constexpr int kWideZChunks = (kWarpSpan + kWideStage) / 4 + 8;          // logical chunks of a stage's input window (+ prefetch slack)
constexpr int kWideZBytes = (kWideZChunks + kWideZChunks / 8 + 1) * 16; // ... in the padded tile layout
constexpr int kWideWBytes = (kWideStage + 8) * 4;   // weights of a stage (+ prefetch slack)
constexpr int kWideStageBytes = kWideZBytes + kWideWBytes;
constexpr int kWideFlushSteps = 128;                // blocked summation: flush the register accumulators every >= 512 taps (one full stage)
constexpr int kWidePartBytes = kWarps * kLaneP * 32 * 4;   // per-lane partial sums of the blocked summation, [warp][output][lane]

// One (north output ring i, input ring j = i + r) pair.  The southern mirror pair
// (n_theta-1-i, n_theta-1-j) has identical weights.  `ntaps` FP32 weights w[e], tap e <-> dphi index
// d = start + e; zero outside the window.
//   NARROW rings: start and ntaps even (8-byte steps), window inside [-32, 32).
//   WIDE rings:   start and ntaps multiples of 4 (16-byte steps).
struct PairDesc {
    uint32_t w_off;   // offset, in floats, of the stored weights; even (narrow) / multiple of 4 (wide)
    int32_t start;    // dphi index d of stored tap 0 (<= 0)
    int32_t ntaps;    // stored taps; 0 = nothing to do
    int32_t half;     // D (taps -D..D inside theta_cut); n_phi = whole ring; -1 = empty
};

// Kernel-ready form of a NARROW ring pair (what conv_narrow stages instead of PairDesc): the run enters
// the unrolled step chain at step k0 = (32 + start) / 2 and executes n = ntaps / 2 steps.
struct NarrowRun {
    int32_t wq_rel;   // byte offset of the run's weights in the ring's weight block, minus 8 * k0
    int32_t k0;       // entry step
    int32_t n;        // steps; 0 = nothing to do
    int32_t pad_;
};

enum ItemKind : int16_t { kWide = 0, kNarrow = 1 };

// One CTA of the convolution launch.
struct Item {
    int32_t i0;       // kWide: the output ring (either hemisphere).  kNarrow: first NORTHERN output ring
                      //   (the CTA also produces the mirror rings)
    int32_t k0;       // first output phi of the tile
    int16_t f_log2;   // kWide: F = 1 << f_log2 phi sub-tiles of kWarpSpan outputs; S = kWarps / F.  kNarrow: 0
                      //   (the tile is kNarrowSpan outputs; kWarps rings per pass)
    int16_t kind;     // kWide: one ring, S tap splits.  kNarrow: `nrings` rings
    int32_t nrings;   // kNarrow: rings of the band; negative = the band is the southern mirror of
                      //   northern rings [i0, i0 - nrings)
    int32_t wcopy;    // kNarrow: floats of a ring's weight block to stage (max over the band; multiple of 4)
};

// Work unit of the weight generator (one warp) for one ring pair: `count` taps d0, d0+1, ...
struct GenUnit {
    uint32_t w_base;  // destination offset in the weight buffer
    int32_t d0;       // first dphi index
    int32_t count;    // taps / steps to write (<= kGenUnitTaps)
    int32_t half;     // D, or n_phi for a whole ring
    double a;         // sin^2((t_i - t_j)/2)
    double b;         // sin t_i sin t_j
    double area;      // A_j
    int32_t pad_[2];
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
    std::vector<NarrowRun> runs;            // [n_north - first_narrow][2R+1]
    uint32_t narrow_w_base = 0;             // weights of narrow ring i start at narrow_w_base + (i - first_narrow) * narrow_wslot
    std::vector<uint32_t> ring_w_off;       // [n_north] offset of the ring's (contiguous) weights
    std::vector<uint32_t> ring_slots;       // [n_north] stored taps of the ring (sum over rows, padded to 4)
    std::vector<Item> items;                // the WIDE items, then the NARROW items; each part cost-sorted, heaviest first
    int n_wide_items = 0;                   // items[0 .. n_wide_items) are WIDE (kernel k_convolve_wide), the rest NARROW
    std::vector<GenUnit> gen_units;
    int first_narrow = 0;                   // rings [first_narrow, n_north) use the narrow kernel path
    int narrow_wslot = 0;                   // floats per ring in the GLOBAL narrow weight buffer (uniform stride)
    int narrow_wcap = 0;                    // floats of the weight area in shared memory (conv_narrow)
    size_t smem_wide = 0, smem_narrow = 0;  // dynamic shared memory of the two convolution kernels
    unsigned long long pair_evals = 0;      // useful FMAs per map
    unsigned long long weights = 0;         // in-support weights, no symmetry reduction
    unsigned long long fma_slots = 0;       // FMA lanes issued per map (padding included)
    unsigned long long fma_slots_wide = 0;  // ... of which by the WIDE items
    unsigned long long weight_slots = 0;    // floats in the weight buffer

    // window of ring pair (i, j) for ANY i (southern rings through the mirror): -1 / D / n_phi
    int window(int i, int j) const;
    const PairDesc* pair(int i_north, int j) const {
        int r = j - i_north + R;
        if (i_north < 0 || i_north >= n_north || r < 0 || r > 2 * R) return nullptr;
        return &pairs[(size_t)i_north * (2 * R + 1) + r];
    }
};

// Host <-> device pipeline of arkcos_convolve_host: the map is cut into `n_chunks` bands of rings; chunk c is copied to
// the device, then the work items whose LAST input ring lies in chunk c (their "group") are launched, and a chunk's
// output rings are copied back as soon as every item that writes into it has been launched.  Same items, same
// arithmetic as one arkcos_convolve: only the launches are grouped, so the result is bit-identical.
struct Pipeline {
    int n_chunks = 0;
    std::vector<int> chunk_lo;              // [n_chunks + 1] first ring of each chunk; chunk_lo[n_chunks] = n_theta
    std::vector<Item> items;                // the schedule's items ordered by (group, class, cost)
    std::vector<int> wide_begin;            // [n_chunks + 1] items[wide_begin[g] .. narrow_begin[g]) = WIDE items of group g
    std::vector<int> narrow_begin;          // [n_chunks + 1] items[narrow_begin[g] .. wide_begin[g + 1]) = NARROW items of group g
    std::vector<int> ready_group;           // [n_chunks] chunk c's output is complete once groups <= ready_group[c] have run
};
// physical output rings [lo, hi] of a work item
void item_output_rings(const Schedule& s, const Item& it, int& lo, int& hi);
void build_pipeline(const Schedule& s, int n_chunks, Pipeline& out);

// shared memory of a WIDE item (two private stage buffers per warp), and of the NARROW path
size_t wide_smem_bytes(int R);
size_t narrow_smem_bytes(int R, int wcap);

// Builds the schedule.  Returns 0 on success, 1 = invalid argument, 4 = unsupported (matches arkcos_status).
// all_wide: every ring goes to the WIDE class (measurement hook ARKCOS_PLAN_ALL_WIDE: the NARROW kernel against the
// WIDE kernel on the same rings).
int build_schedule(int n_theta, int n_phi, double theta_cut, int sm_count, Schedule& out, bool all_wide = false);

// Re-derives, as plain integer arithmetic, every global-memory range and every shared-memory offset the
// kernels will form from the schedule's descriptors (work items, pair descriptors, narrow runs, generator
// units) and checks that each lies inside its buffer, is aligned as the instruction that uses it needs, and
// that every input ring a non-empty pair names exists.  Called by build_schedule before it returns (a
// schedule that fails is never uploaded: arkcos_plan_create returns ARKCOS_EINTERNAL) and by the CPU tests on
// every BASELINE.json workload.  Returns 0, or a positive code; `why` (may be null) receives a description.
int validate_schedule(const Schedule& s, std::string* why);

}  // namespace arkcos
