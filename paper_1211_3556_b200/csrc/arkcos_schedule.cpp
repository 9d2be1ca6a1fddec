// arkcos_schedule.cpp - step S1, the ring-pair scheduler (host, FP64).  BASELINE.json north_star (a):
// "a ring-pair scheduler that exploits the ECP grid's azimuthal symmetry, so each (output ring i,
// input ring j) pair inside the theta_cut band is a banded circular 1-D convolution in dphi".
// SURVEY.md §8(a)-S1, §8(c) G3 (support decided in FP64), G12 (poles / whole-ring windows).
//
// Geometry uses the cancellation-free haversine form, algebraically identical to
// cos(gamma) = cos t_i cos t_j + sin t_i sin t_j cos(dphi):
//     sin^2(gamma/2) = sin^2((t_i - t_j)/2) + sin t_i sin t_j sin^2(dphi/2)
// and the support test  gamma <= theta_cut  <=>  sin^2(gamma/2) <= sin^2(theta_cut/2).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <string>

#include "arkcos_internal.h"

namespace arkcos {

namespace {
constexpr double kPi = 3.14159265358979323846264338327950288;

// The single FP64 expression that decides whether tap d of ring pair (a_r, b) is inside the support.
inline bool inside(const Schedule& s, double a_r, double b, int d) { return a_r + b * s.s2[d] <= s.h_cut; }

// -1 empty, n_phi whole ring, else largest D with tap D inside (monotone in d on [0, n_phi/2]).
int window_of(const Schedule& s, int i, int j) {
    int r = std::abs(i - j);
    if (r > s.R) return -1;
    double a_r = s.a_r[r];
    double b = s.sin_t[i] * s.sin_t[j];
    if (!inside(s, a_r, b, 0)) return -1;
    int half = s.n_phi / 2;
    if (inside(s, a_r, b, half)) return s.n_phi;
    int lo = 0, hi = half;  // inside(lo) true, inside(hi) false
    while (hi - lo > 1) {
        int mid = (lo + hi) / 2;
        if (inside(s, a_r, b, mid)) lo = mid; else hi = mid;
    }
    return lo;
}
}  // namespace

int Schedule::window(int i, int j) const {
    if (i < 0 || i >= n_theta || j < 0 || j >= n_theta) return -1;
    return window_of(*this, i, j);
}

int build_schedule(int n_theta, int n_phi, double theta_cut, int sm_count, Schedule& s, bool all_wide) {
    if (n_theta < 1 || n_phi < 4 || !(theta_cut > 0.0) || !(theta_cut <= kPi * (1.0 + 1e-15))) return 1;
    if (n_phi % 4 != 0) return 4;
    if (sm_count < 1) sm_count = 148;
    s = Schedule();
    s.n_theta = n_theta; s.n_phi = n_phi; s.theta_cut = theta_cut;
    s.n_north = (n_theta + 1) / 2;
    const double dtheta = kPi / n_theta, dphi = 2.0 * kPi / n_phi;
    {
        double sh = std::sin(0.5 * std::min(theta_cut, kPi));
        s.h_cut = sh * sh;
    }
    s.sin_t.resize(n_theta); s.area.resize(n_theta);
    for (int i = 0; i < n_theta; i++) {
        s.sin_t[i] = std::sin((i + 0.5) * dtheta);
        // exact ring pixel area dphi (cos(j dt) - cos((j+1) dt)) in its product form (no cancellation)
        s.area[i] = 2.0 * dphi * s.sin_t[i] * std::sin(0.5 * dtheta);
    }
    s.s2.resize(n_phi / 2 + 1);
    for (int d = 0; d <= n_phi / 2; d++) { double v = std::sin(0.5 * d * dphi); s.s2[d] = v * v; }
    // ring half band R: largest r whose d = 0 tap is inside (gamma >= |t_i - t_j|, equality at d = 0)
    s.a_r.clear();
    for (int r = 0; r < n_theta; r++) {
        double v = std::sin(0.5 * r * dtheta); v *= v;
        if (v > s.h_cut) break;
        s.a_r.push_back(v);
    }
    s.R = (int)s.a_r.size() - 1;
    const int W = 2 * s.R + 1;

    // ---- windows of the northern ring pairs; work counters over ALL rings --------------------------
    s.pairs.assign((size_t)s.n_north * W, PairDesc{0u, 0, 0, -1});
    for (int i = 0; i < n_theta; i++) {
        for (int r = -s.R; r <= s.R; r++) {
            int j = i + r;
            if (j < 0 || j >= n_theta) continue;            // no wrap over the pole (G12)
            int D = window_of(s, i, j);
            if (D < 0) continue;
            unsigned long long taps = (D == n_phi) ? (unsigned long long)n_phi : (unsigned long long)(2 * D + 1);
            s.weights += taps;
            s.pair_evals += taps * (unsigned long long)n_phi;
            if (i < s.n_north) s.pairs[(size_t)i * W + (r + s.R)].half = D;
        }
    }
    // stored tap range of a pair in the NARROW layout: start and ntaps even (8-byte steps)
    auto narrow_range = [&](int D, int& start, int& ntaps) {
        if (D == n_phi) { start = -(n_phi / 2); ntaps = n_phi; }
        else { start = -(D + (D & 1)); ntaps = ((D - start + 1) + 1) & ~1; }
    };
    // ... and in the WIDE layout: start and ntaps multiples of 4 (16-byte steps)
    auto wide_range = [&](int D, int& start, int& ntaps) {
        const int dmin = (D == n_phi) ? -(n_phi / 2) : -D;
        const int dmax = (D == n_phi) ? n_phi / 2 - 1 : D;
        start = -(((-dmin) + 3) & ~3);
        ntaps = ((dmax - start + 1) + 3) & ~3;
    };

    // ---- ring classes -----------------------------------------------------------------------------
    // NARROW rings: every stored window lies inside [-kHaloNarrow, kHaloNarrow).  Windows widen
    // towards the pole, so the narrow rings are the band [first_narrow, n_north) next to the equator.
    auto ring_is_narrow = [&](int i) {
        for (int r = 0; r < W; r++) {
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            if (p.half < 0) continue;
            if (p.half == n_phi) return false;
            int start, ntaps;
            narrow_range(p.half, start, ntaps);
            if (start < -kHaloNarrow || start + ntaps > kHaloNarrow) return false;
        }
        return true;
    };
    s.first_narrow = s.n_north;
    while (!all_wide && s.first_narrow > 0 && ring_is_narrow(s.first_narrow - 1)) s.first_narrow--;
    // stored windows of the narrow rings
    std::vector<int> nw_start((size_t)s.n_north * W, 0), nw_ntaps((size_t)s.n_north * W, 0);
    for (int i = s.first_narrow; i < s.n_north; i++)
        for (int r = 0; r < W; r++) {
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            if (p.half >= 0) narrow_range(p.half, nw_start[(size_t)i * W + r], nw_ntaps[(size_t)i * W + r]);
        }
    // Band marching keeps 2R + 2 kWarps row slots, the run descriptors and the ring weight blocks of kWarps rings in
    // shared memory.  Whatever the row slots leave of the launch's shared memory is the weight area, `narrow_wcap`
    // floats: an item whose rings' blocks fit twice (2 kWarps wcopy <= wcap) double-buffers them across passes,
    // one whose blocks fit once reloads them at the start of every pass (conv_narrow), a ring whose block does
    // not fit at all is WIDE.  Two launch sizes are tried: half an SM's shared memory, so that two CTAs (16
    // warps) share an SM - taken when at least 70 % of the narrow FMA slots can then be double-buffered - or else
    // one CTA per SM with the full budget.  The weight block of a ring grows towards the pole, so the narrow
    // class shrinks from its polar end; for a large ring band (R > ~25) nothing fits and every ring is WIDE.
    {
        std::vector<unsigned long long> slots(s.n_north, 0);
        for (int i = s.first_narrow; i < s.n_north; i++) {
            for (int r = 0; r < W; r++) slots[i] += (unsigned long long)nw_ntaps[(size_t)i * W + r];
            slots[i] = (slots[i] + 3) & ~3ull;
        }
        const long long fixed = (long long)narrow_smem_bytes(s.R, 0);
        auto wcap_of = [&](long long budget) { return budget > fixed ? (budget - fixed) / 4 / 4 * 4 : 0ll; };
        auto first_fit = [&](long long wcap, int mult) {           // first ring of the class whose block fits `mult` x kWarps times
            int fn = s.first_narrow;
            while (fn < s.n_north && (long long)mult * kWarps * (long long)(slots[fn] + kNarrowWPad) > wcap) fn++;
            return fn;
        };
        const long long wcap2 = wcap_of(kSmemTwoPerSm), wcap1 = wcap_of(kSmemBudget);
        unsigned long long all = 0, dbl2 = 0;
        for (int i = s.first_narrow; i < s.n_north; i++) all += slots[i];
        for (int i = first_fit(wcap2, 2); i < s.n_north; i++) dbl2 += slots[i];
        long long wcap = 0;
        if (all > 0 && (double)dbl2 >= 0.7 * (double)all) { wcap = wcap2; s.smem_narrow = (size_t)kSmemTwoPerSm; }
        else { wcap = wcap1; s.smem_narrow = (size_t)kSmemBudget; }
        s.first_narrow = first_fit(wcap, 1);
        if (s.first_narrow >= s.n_north) { s.first_narrow = s.n_north; s.narrow_wslot = 0; s.narrow_wcap = 0; s.smem_narrow = 0; }
        else {
            unsigned long long wslot = 0;
            for (int i = s.first_narrow; i < s.n_north; i++) wslot = std::max(wslot, slots[i]);
            s.narrow_wslot = (int)wslot;
            // no more shared memory than the largest item needs (double-buffered if it can be)
            const long long need = std::min<long long>(wcap, 2ll * kWarps * (long long)(wslot + kNarrowWPad));
            s.narrow_wcap = (int)need;
            s.smem_narrow = (size_t)(fixed + 4 * need);
        }
    }

    // ---- weight layout ------------------------------------------------------------------------------
    // WIDE rings: one contiguous block per ring.  NARROW rings: blocks at a uniform stride of narrow_wslot
    // floats, so that conv_narrow can stage a ring's block without reading an offset table first.
    unsigned long long w_off = 0;
    std::vector<unsigned long long> ring_slots(s.n_north, 0);  // stored taps per output phi
    s.ring_w_off.assign(s.n_north, 0u); s.ring_slots.assign(s.n_north, 0u);
    for (int i = 0; i < s.n_north; i++) {
        const bool wide = i < s.first_narrow;
        if (i == s.first_narrow) s.narrow_w_base = (uint32_t)w_off;
        const unsigned long long ring_base = w_off;
        s.ring_w_off[i] = (uint32_t)w_off;
        for (int r = 0; r < W; r++) {
            PairDesc& p = s.pairs[(size_t)i * W + r];
            if (p.half < 0) continue;
            if (wide) wide_range(p.half, p.start, p.ntaps);
            else { p.start = nw_start[(size_t)i * W + r]; p.ntaps = nw_ntaps[(size_t)i * W + r]; }
            const unsigned long long floats = (unsigned long long)p.ntaps;
            if (w_off + floats > 0xFFFFFFF0ull) return 4;
            p.w_off = (uint32_t)w_off;
            w_off += floats;
            ring_slots[i] += (unsigned long long)p.ntaps;
        }
        s.ring_slots[i] = (uint32_t)((ring_slots[i] + 3) & ~3ull);
        if (wide) w_off = (w_off + 3) & ~3ull;                         // every ring's block is 16-byte aligned
        else w_off = ring_base + (unsigned long long)s.narrow_wslot;
        if (w_off > 0xFFFFFFF0ull) return 4;
    }
    s.weight_slots = w_off;
    s.runs.assign((size_t)(s.n_north - s.first_narrow) * W, NarrowRun{0, 0, 0, 0});
    for (int i = s.first_narrow; i < s.n_north; i++)
        for (int r = 0; r < W; r++) {
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            if (p.ntaps == 0) continue;
            NarrowRun& u = s.runs[(size_t)(i - s.first_narrow) * W + r];
            u.k0 = (kHaloNarrow + p.start) / 2;
            u.n = p.ntaps / 2;
            u.wq_rel = 4 * (int32_t)(p.w_off - s.ring_w_off[i]) - 8 * u.k0;
        }

    // ---- generator work units: one warp writes up to kGenUnitTaps taps (steps) of one ring pair -----
    for (int i = 0; i < s.n_north; i++) {
        for (int r = 0; r < W; r++) {
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            const int j = i + r - s.R;
            const int n = p.ntaps;
            for (int e0 = 0; e0 < n; e0 += kGenUnitTaps) {
                GenUnit g;
                g.w_base = p.w_off + (uint32_t)e0; g.d0 = p.start + e0;
                g.count = std::min(kGenUnitTaps, n - e0); g.half = p.half;
                g.a = s.a_r[std::abs(r - s.R)]; g.b = s.sin_t[i] * s.sin_t[j]; g.area = s.area[j];
                g.pad_[0] = g.pad_[1] = 0;
                s.gen_units.push_back(g);
            }
        }
    }

    // ---- work items, heaviest first (H1: polar imbalance) -------------------------------------------
    unsigned long long total = 0;
    for (int i = 0; i < s.n_north; i++) total += ring_slots[i] * (unsigned long long)n_phi * (2 * i + 1 == n_theta ? 1ull : 2ull);
    const double c_max = (double)total / (double)sm_count / 8.0;   // no item above 1/8 of an SM's share, if possible
    struct Tmp { Item it; double cost; };
    std::vector<Tmp> tmp_wide, tmp_narrow;
    // WIDE: (ring of either hemisphere, phi tile of F sub-tiles of kWarpSpan outputs); S = 8/F tap splits
    if (s.first_narrow > 0) {
        s.smem_wide = wide_smem_bytes(s.R);
        int wf_cap = 0;
        while (wf_cap < 3 && (kWarpSpan << wf_cap) < n_phi) wf_cap++;
        for (int i = 0; i < s.first_narrow; i++) {
            int fl = wf_cap;
            while (fl > 0 && (double)ring_slots[i] * (double)std::min(n_phi, kWarpSpan << fl) > c_max) fl--;
            const int L = kWarpSpan << fl;
            const int i_s = n_theta - 1 - i;
            for (int k0 = 0; k0 < n_phi; k0 += L) {
                const int valid = std::min(L, n_phi - k0);
                const double cost = (double)ring_slots[i] * (double)valid + 4000.0;
                for (int hemi = 0; hemi < (i_s != i ? 2 : 1); hemi++) {
                    tmp_wide.push_back(Tmp{Item{hemi ? i_s : i, k0, (int16_t)fl, (int16_t)kWide, 1, 0}, cost});
                    s.fma_slots += ring_slots[i] * (unsigned long long)L;
                    s.fma_slots_wide += ring_slots[i] * (unsigned long long)L;
                }
            }
        }
    }
    // NARROW: (band of B rings of one hemisphere, phi tile of kNarrowSpan outputs); kWarps rings advance together.
    // Two CTAs share an SM, so a band is cut at half the WIDE items' cost cap.
    if (s.first_narrow < s.n_north) {
        constexpr int S = kWarps, L = kNarrowSpan;
        auto doubles = [&](int i) { return 2ll * S * (long long)(s.ring_slots[i] + kNarrowWPad) <= (long long)s.narrow_wcap; };
        const int b_min = ((2 * (2 * s.R + S)) + S - 1) / S * S;       // keep the band prologue below ~50 % extra staging
        int i = s.first_narrow;
        while (i < s.n_north) {
            // a band does not straddle the ring from which the weight blocks fit twice (its wcopy is that of its
            // polar-most ring, and the kernel double-buffers an item iff 2 kWarps wcopy <= wcap)
            int limit = s.n_north;
            if (!doubles(i)) { limit = i + 1; while (limit < s.n_north && !doubles(limit)) limit++; }
            double c = 0.0; int b = 0;
            while (i + b < limit && (b < b_min || c < 0.5 * c_max) && b < 512) { c += (double)ring_slots[i + b] * (double)L; b++; }
            b = std::min((b + S - 1) / S * S, limit - i);
            if (limit - (i + b) < b_min / 2) b = limit - i;             // do not leave a tiny tail band
            // the southern mirror band leaves out a ring that is its own mirror (odd n_theta: the equator)
            const int b_south = (2 * (i + b - 1) + 1 == n_theta) ? b - 1 : b;
            for (int hemi = 0; hemi < 2; hemi++) {
                const int nb = hemi ? b_south : b;
                if (nb <= 0) continue;
                c = 0.0;
                uint32_t wcopy = 4;
                for (int q = 0; q < nb; q++) { c += (double)ring_slots[i + q] * (double)L; wcopy = std::max(wcopy, s.ring_slots[i + q]); }
                for (int k0 = 0; k0 < n_phi; k0 += L) {
                    tmp_narrow.push_back(Tmp{Item{i, k0, (int16_t)0, (int16_t)kNarrow, hemi ? -nb : nb, (int32_t)wcopy}, c + 4000.0});
                    for (int q = 0; q < nb; q++) s.fma_slots += ring_slots[i + q] * (unsigned long long)L;
                }
            }
            i += b;
        }
    }
    auto by_cost = [](const Tmp& a, const Tmp& b) { return a.cost > b.cost; };
    std::stable_sort(tmp_wide.begin(), tmp_wide.end(), by_cost);
    std::stable_sort(tmp_narrow.begin(), tmp_narrow.end(), by_cost);
    s.items.reserve(tmp_wide.size() + tmp_narrow.size());
    for (auto& t : tmp_wide) s.items.push_back(t.it);
    s.n_wide_items = (int)s.items.size();
    for (auto& t : tmp_narrow) s.items.push_back(t.it);
    return validate_schedule(s, nullptr) == 0 ? 0 : 5;
}

// ---- validate_schedule ---------------------------------------------------------------------------
// Every check below restates, in integers, an address the kernels of arkcos_kernels.cuh form from the
// descriptor it names (the function and line of thought are given with each group).  The kernels trust the
// descriptors: there is no bounds check in the hot loops, so nothing that fails here may reach the device.
int validate_schedule(const Schedule& s, std::string* why) {
    int code = 0;
    auto fail = [&](int c, const char* what, long long a, long long b) {
        if (code == 0) {
            code = c;
            if (why) *why = std::string(what) + " (" + std::to_string(a) + ", " + std::to_string(b) + ")";
        }
        return c;
    };
    const int W = 2 * s.R + 1, n_theta = s.n_theta, n_phi = s.n_phi;
    if (n_theta < 1 || n_phi < 4 || n_phi % 4 != 0 || s.R < 0 || s.R >= n_theta) return fail(1, "grid / R", n_phi, s.R);
    if (s.n_north != (n_theta + 1) / 2 || s.first_narrow < 0 || s.first_narrow > s.n_north) return fail(2, "ring classes", s.first_narrow, s.n_north);
    if (s.pairs.size() != (size_t)s.n_north * W) return fail(3, "pairs size", (long long)s.pairs.size(), W);
    if (s.runs.size() != (size_t)(s.n_north - s.first_narrow) * W) return fail(4, "runs size", (long long)s.runs.size(), W);
    if (s.s2.size() != (size_t)n_phi / 2 + 1) return fail(5, "s2 size", (long long)s.s2.size(), n_phi);
    if (s.ring_w_off.size() != (size_t)s.n_north || s.ring_slots.size() != (size_t)s.n_north) return fail(6, "ring tables", 0, 0);
    if (s.weight_slots > 0xFFFFFFF0ull) return fail(7, "weight buffer over 2^32 floats", (long long)s.weight_slots, 0);
    if (s.smem_wide > (size_t)kSmemBudget || s.smem_narrow > (size_t)kSmemBudget) return fail(8, "shared memory over budget", (long long)s.smem_wide, (long long)s.smem_narrow);
    if (s.n_wide_items < 0 || s.n_wide_items > (int)s.items.size()) return fail(8, "n_wide_items", s.n_wide_items, (long long)s.items.size());
    const long long wtot = (long long)s.weight_slots;
    const bool have_narrow = s.first_narrow < s.n_north;
    if (have_narrow) {
        if (s.narrow_wslot < 4 || s.narrow_wslot % 4 != 0 || s.narrow_w_base % 4 != 0) return fail(10, "narrow weight stride", s.narrow_wslot, s.narrow_w_base);
        if (s.narrow_wcap < 0 || s.narrow_wcap % 4 || narrow_smem_bytes(s.R, s.narrow_wcap) > s.smem_narrow) return fail(11, "narrow shared memory", (long long)s.smem_narrow, s.narrow_wcap);
    }
    if (s.first_narrow > 0 && wide_smem_bytes(s.R) > s.smem_wide) return fail(12, "wide shared memory", (long long)s.smem_wide, 0);

    // ---- pair descriptors (conv_wide: stage source rows and weight ranges; plan_pair_weights) ----------
    unsigned long long stored = 0;
    for (int i = 0; i < s.n_north; i++) {
        const bool wide = i < s.first_narrow;
        unsigned long long ring = 0;
        for (int r = 0; r < W; r++) {
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            const int j = i + r - s.R;
            if (p.ntaps == 0) { if (p.half >= 0) return fail(20, "in-support pair without stored taps", i, r); continue; }
            if (p.half < 0 || j < 0 || j >= n_theta) return fail(21, "stored taps for a ring pair that does not exist", i, j);
            const int q = wide ? 4 : 2;                          // conv_wide: 16-byte steps; conv_narrow: 8-byte steps
            if (p.ntaps < 0 || p.ntaps % q || p.start > 0 || (-p.start) % q || p.w_off % q) return fail(22, "tap range granularity", i, r);
            if (p.half != n_phi && (p.half >= n_phi / 2 || p.start > -p.half || p.start + p.ntaps <= p.half)) return fail(23, "stored range does not cover the window", i, r);
            if (p.half == n_phi && (p.start > -(n_phi / 2) || p.start + p.ntaps < n_phi / 2)) return fail(24, "stored range does not cover the whole ring", i, r);
            if (-p.start > n_phi / 2 + 3 || p.start + p.ntaps > n_phi / 2 + 4) return fail(25, "stored range beyond one turn", i, r);
            if ((long long)p.w_off + p.ntaps > wtot) return fail(26, "weights beyond the buffer", i, r);
            if ((long long)p.w_off < s.ring_w_off[i] || (long long)p.w_off + p.ntaps > (long long)s.ring_w_off[i] + s.ring_slots[i]) return fail(27, "weights outside the ring's block", i, r);
            if (!wide && (p.start < -kHaloNarrow || p.start + p.ntaps > kHaloNarrow)) return fail(28, "narrow window outside the halo", i, r);
            ring += (unsigned long long)p.ntaps;
        }
        if (((ring + 3) & ~3ull) != s.ring_slots[i]) return fail(29, "ring_slots", i, (long long)ring);
        if (!wide && (s.ring_w_off[i] != s.narrow_w_base + (unsigned long long)(i - s.first_narrow) * s.narrow_wslot ||
                      s.ring_slots[i] > (unsigned)s.narrow_wslot)) return fail(30, "narrow ring block", i, s.ring_slots[i]);
        stored += ring;
    }
    // ---- narrow run descriptors (conv_narrow / narrow_row: jump-table entry, step count, weight address) ---
    for (int i = s.first_narrow; i < s.n_north; i++)
        for (int r = 0; r < W; r++) {
            const NarrowRun& u = s.runs[(size_t)(i - s.first_narrow) * W + r];
            const PairDesc& p = s.pairs[(size_t)i * W + r];
            if (u.n == 0) { if (p.ntaps != 0) return fail(40, "pair without a run", i, r); continue; }
            if (u.k0 < 0 || u.k0 > 16 || u.n < 1 || u.k0 + u.n > kHaloNarrow) return fail(41, "run outside the step chain", u.k0, u.n);
            if (2 * u.k0 - kHaloNarrow != p.start || 2 * u.n != p.ntaps) return fail(42, "run does not match its pair", i, r);
            const long long woff = (long long)u.wq_rel + 8ll * u.k0;       // byte offset of the run's weights in the ring block
            if (woff < 0 || woff % 8 || woff != 4ll * (p.w_off - s.ring_w_off[i])) return fail(43, "run weight offset", i, r);
            if (woff / 4 + p.ntaps > (long long)s.ring_slots[i]) return fail(44, "run weights beyond the staged block", i, r);
        }
    // ---- generator units (k_generate_weights: destination range, s2 index) ---------------------------------
    unsigned long long gen = 0;
    for (const GenUnit& g : s.gen_units) {
        if (g.count < 1 || g.count > kGenUnitTaps || (long long)g.w_base + g.count > wtot) return fail(50, "generator unit range", g.w_base, g.count);
        if (!(g.half == n_phi || (g.half >= 0 && g.half < n_phi / 2))) return fail(51, "generator unit window", g.half, 0);
        const long long lo = g.d0, hi = (long long)g.d0 + g.count - 1;   // taps written; inside-the-window taps index s2[|d|]
        if (lo < -(long long)(n_phi / 2) - 3 || hi > n_phi / 2 + 3) return fail(52, "generator unit taps beyond one turn", lo, hi);
        gen += (unsigned long long)g.count;
    }
    if (gen != stored) return fail(53, "generator units do not tile the stored taps", (long long)gen, (long long)stored);
    // ---- work items (k_convolve_wide / k_convolve_narrow) and coverage: every output ring x 512-pixel tile once ----
    const int tiles = (n_phi + kNarrowSpan - 1) / kNarrowSpan;
    std::vector<unsigned char> cover((size_t)n_theta * tiles, 0);
    for (size_t k = 0; k < s.items.size(); k++) {
        const Item& it = s.items[k];
        if ((it.kind == kWide) != ((int)k < s.n_wide_items)) return fail(59, "item in the wrong part of the work list", (long long)k, it.kind);
        if (it.kind == kWide) {
            if (it.f_log2 < 0 || it.f_log2 > 3) return fail(60, "item f_log2", it.f_log2, 0);
            const int L = kWarpSpan << it.f_log2;
            if (it.k0 < 0 || it.k0 >= n_phi || it.k0 % L) return fail(61, "item k0", it.k0, L);
            if (it.i0 < 0 || it.i0 >= n_theta) return fail(62, "wide item ring", it.i0, 0);
            const int i_n = 2 * it.i0 >= n_theta ? n_theta - 1 - it.i0 : it.i0;
            if (i_n >= s.first_narrow) return fail(63, "wide item on a narrow ring", it.i0, s.first_narrow);
            const int t0 = it.k0 / kNarrowSpan, t1 = std::min(tiles, t0 + L / kNarrowSpan);
            for (int t = t0; t < t1; t++) cover[(size_t)it.i0 * tiles + t]++;
        } else if (it.kind == kNarrow) {
            const int nr = it.nrings < 0 ? -it.nrings : it.nrings;
            if (!have_narrow || it.f_log2 != 0) return fail(64, "narrow item tile", it.f_log2, 0);
            if (it.k0 < 0 || it.k0 >= n_phi || it.k0 % kNarrowSpan) return fail(61, "item k0", it.k0, kNarrowSpan);
            if (nr < 1 || it.i0 < s.first_narrow || it.i0 + nr > s.n_north) return fail(65, "narrow item band", it.i0, nr);
            if (it.wcopy < 4 || it.wcopy % 4 || it.wcopy > s.narrow_wslot) return fail(66, "narrow item wcopy", it.wcopy, s.narrow_wslot);
            // conv_narrow keeps kWarps (single-buffered) or 2 kWarps (double-buffered) blocks of wcopy floats in the weight area
            if ((long long)kWarps * (it.wcopy + kNarrowWPad) > (long long)s.narrow_wcap) return fail(66, "narrow item weight blocks beyond the shared weight area", it.wcopy, s.narrow_wcap);
            // stage_ring_tables reads wcopy floats of each ring's block
            if ((long long)s.narrow_w_base + (long long)(it.i0 + nr - 1 - s.first_narrow) * s.narrow_wslot + it.wcopy > wtot) return fail(67, "narrow weight block beyond the buffer", it.i0, nr);
            for (int q = 0; q < nr; q++) {
                if (s.ring_slots[it.i0 + q] > (unsigned)it.wcopy) return fail(68, "ring block larger than wcopy", it.i0 + q, it.wcopy);
                const int i_phys = it.nrings < 0 ? n_theta - 1 - (it.i0 + q) : it.i0 + q;
                if (it.nrings < 0 && 2 * (it.i0 + q) + 1 == n_theta) return fail(69, "self-mirrored ring in a southern band", it.i0 + q, 0);
                cover[(size_t)i_phys * tiles + it.k0 / kNarrowSpan]++;
            }
        } else return fail(70, "item kind", it.kind, 0);
    }
    for (size_t c = 0; c < cover.size(); c++)
        if (cover[c] != 1) return fail(71, "output tile not written exactly once (ring, count)", (long long)(c / tiles), cover[c]);
    return 0;
}

void item_output_rings(const Schedule& s, const Item& it, int& lo, int& hi) {
    if (it.kind == kWide) { lo = hi = it.i0; return; }
    const int nr = it.nrings < 0 ? -it.nrings : it.nrings;
    if (it.nrings < 0) { lo = s.n_theta - it.i0 - nr; hi = s.n_theta - 1 - it.i0; }
    else { lo = it.i0; hi = it.i0 + nr - 1; }
}

void build_pipeline(const Schedule& s, int n_chunks, Pipeline& p) {
    p = Pipeline();
    n_chunks = std::max(1, std::min(n_chunks, s.n_theta));
    p.n_chunks = n_chunks;
    p.chunk_lo.resize(n_chunks + 1);
    for (int c = 0; c <= n_chunks; c++) p.chunk_lo[c] = (int)((long long)s.n_theta * c / n_chunks);
    auto chunk_of = [&](int ring) { return (int)(std::upper_bound(p.chunk_lo.begin(), p.chunk_lo.end(), ring) - p.chunk_lo.begin()) - 1; };
    struct Tmp { int group, kind; size_t order; };
    std::vector<Tmp> key(s.items.size());
    p.ready_group.assign(n_chunks, 0);
    for (size_t k = 0; k < s.items.size(); k++) {
        int lo, hi;
        item_output_rings(s, s.items[k], lo, hi);
        const int g = chunk_of(std::min(s.n_theta - 1, hi + s.R));   // the last input ring the item reads
        key[k] = Tmp{g, s.items[k].kind, k};
        for (int c = chunk_of(lo); c <= chunk_of(hi); c++) p.ready_group[c] = std::max(p.ready_group[c], g);
    }
    std::stable_sort(key.begin(), key.end(), [](const Tmp& a, const Tmp& b) { return a.group != b.group ? a.group < b.group : a.kind < b.kind; });
    p.items.reserve(key.size());
    p.wide_begin.assign(n_chunks + 1, 0); p.narrow_begin.assign(n_chunks + 1, 0);
    size_t k = 0;
    for (int g = 0; g < n_chunks; g++) {
        p.wide_begin[g] = (int)p.items.size();
        while (k < key.size() && key[k].group == g && key[k].kind == kWide) p.items.push_back(s.items[key[k++].order]);
        p.narrow_begin[g] = (int)p.items.size();
        while (k < key.size() && key[k].group == g) p.items.push_back(s.items[key[k++].order]);
    }
    p.wide_begin[n_chunks] = p.narrow_begin[n_chunks] = (int)p.items.size();
}

size_t wide_smem_bytes(int R) {
    const size_t stage = (size_t)kWarps * 2 * kWideStageBytes + (size_t)(2 * R + 1) * sizeof(PairDesc) + (size_t)kWidePartBytes;
    const size_t red = (size_t)kWarps * kWarpSpan * 4;
    return stage > red ? stage : red;
}

// (2R + 2S) row slots (the S rows of the next pass land in the slots the previous pass freed), two
// buffers of S x (2R+1) run descriptors, and a weight area of `wcap` floats
size_t narrow_smem_bytes(int R, int wcap) {
    constexpr int S = kWarps;
    // (every weight block carries kNarrowWPad floats of its own for the chain's weight prefetch: conv_narrow)
    return (size_t)(2 * R + 2 * S) * (size_t)kNarrowSlotBytes + 2ull * S * (2 * R + 1) * sizeof(NarrowRun) + 4ull * (size_t)wcap;
}

}  // namespace arkcos
