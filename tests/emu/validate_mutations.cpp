// validate_mutations.cpp - test of the host-side schedule validator (csrc/arkcos_schedule.cpp: validate_schedule).
// Test infrastructure only.  Builds the schedule of one grid, checks that it validates, then corrupts ONE
// descriptor field at a time - each corruption is an address the kernels would form out of range, or an
// output tile written twice / never - and requires the validator to reject every one of them.
//
//   validate_mutations n_theta n_phi theta_cut        -> prints "ok: N mutations rejected", exit 0
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <string>
#include <vector>

#include "arkcos_internal.h"

using namespace arkcos;

int main(int argc, char** argv) {
    if (argc < 4) { std::fprintf(stderr, "usage: validate_mutations n_theta n_phi theta_cut\n"); return 2; }
    const int n_theta = std::atoi(argv[1]), n_phi = std::atoi(argv[2]);
    const double theta_cut = std::atof(argv[3]);
    Schedule base;
    const int rc = build_schedule(n_theta, n_phi, theta_cut, 148, base);
    if (rc != 0) { std::fprintf(stderr, "build_schedule failed: %d\n", rc); return 1; }
    std::string why;
    if (validate_schedule(base, &why) != 0) { std::fprintf(stderr, "fresh schedule rejected: %s\n", why.c_str()); return 1; }
    const int W = 2 * base.R + 1;
    int first_wide = -1, first_narrow_item = -1;
    for (size_t k = 0; k < base.items.size(); k++) {
        if (base.items[k].kind == kWide && first_wide < 0) first_wide = (int)k;
        if (base.items[k].kind == kNarrow && first_narrow_item < 0) first_narrow_item = (int)k;
    }
    size_t live_pair = 0;                              // some pair with stored taps
    for (size_t q = 0; q < base.pairs.size(); q++) if (base.pairs[q].ntaps > 0) { live_pair = q; break; }
    size_t live_run = 0; bool have_run = false;
    for (size_t q = 0; q < base.runs.size(); q++) if (base.runs[q].n > 0) { live_run = q; have_run = true; break; }

    struct Mut { const char* name; std::function<bool(Schedule&)> apply; };   // apply returns false if not applicable
    std::vector<Mut> muts = {
        {"wide item ring beyond the map", [&](Schedule& s) { if (first_wide < 0) return false; s.items[first_wide].i0 = n_theta; return true; }},
        {"wide item on a narrow ring", [&](Schedule& s) { if (first_wide < 0 || s.first_narrow >= s.n_north) return false; s.items[first_wide].i0 = s.first_narrow; return true; }},
        {"item k0 off its tile grid", [&](Schedule& s) { s.items[0].k0 += 4; return true; }},
        {"item k0 beyond the ring", [&](Schedule& s) { s.items[0].k0 = (n_phi + kWarpSpan * 8) / (kWarpSpan * 8) * (kWarpSpan * 8); return true; }},
        {"item f_log2", [&](Schedule& s) { s.items[0].f_log2 = 4; return true; }},
        {"item kind", [&](Schedule& s) { s.items[0].kind = 7; return true; }},
        {"item dropped", [&](Schedule& s) { s.items.pop_back(); return true; }},
        {"item duplicated", [&](Schedule& s) { s.items.push_back(s.items[0]); return true; }},
        {"narrow band beyond the equator", [&](Schedule& s) { if (first_narrow_item < 0) return false; Item& it = s.items[first_narrow_item]; it.nrings = (it.nrings < 0 ? -1 : 1) * (s.n_north - it.i0 + 1); return true; }},
        {"narrow band starts in the wide class", [&](Schedule& s) { if (first_narrow_item < 0 || s.first_narrow == 0) return false; s.items[first_narrow_item].i0 = s.first_narrow - 1; return true; }},
        {"narrow wcopy beyond the ring stride", [&](Schedule& s) { if (first_narrow_item < 0) return false; s.items[first_narrow_item].wcopy = s.narrow_wslot + 4; return true; }},
        {"narrow wcopy smaller than a ring block", [&](Schedule& s) { if (first_narrow_item < 0) return false; Item& it = s.items[first_narrow_item]; if (s.ring_slots[it.i0] <= 4) return false; it.wcopy = (int)s.ring_slots[it.i0] - 4; return true; }},
        {"narrow wcopy misaligned", [&](Schedule& s) { if (first_narrow_item < 0) return false; s.items[first_narrow_item].wcopy += 2; return true; }},
        {"narrow item with the wrong tile width", [&](Schedule& s) { if (first_narrow_item < 0) return false; s.items[first_narrow_item].f_log2 = 1; return true; }},
        {"pair weights beyond the buffer", [&](Schedule& s) { s.pairs[live_pair].w_off = (uint32_t)s.weight_slots; return true; }},
        {"pair weights misaligned", [&](Schedule& s) { s.pairs[live_pair].w_off += 1; return true; }},
        {"pair taps overrun the ring block", [&](Schedule& s) { s.pairs[live_pair].ntaps += 4096; return true; }},
        {"pair window not covered", [&](Schedule& s) { if (s.pairs[live_pair].half < 2 || s.pairs[live_pair].half == n_phi) return false; s.pairs[live_pair].start += 4; return true; }},
        {"pair for a ring beyond the pole", [&](Schedule& s) { if (s.R == 0) return false; PairDesc& p = s.pairs[0]; p.ntaps = 4; p.half = 1; p.start = -4; return true; }},
        {"run entry step", [&](Schedule& s) { if (!have_run) return false; s.runs[live_run].k0 = 17; return true; }},
        {"run length", [&](Schedule& s) { if (!have_run) return false; s.runs[live_run].n = 40; return true; }},
        {"run weight offset", [&](Schedule& s) { if (!have_run) return false; s.runs[live_run].wq_rel += 8; return true; }},
        {"run weight offset negative", [&](Schedule& s) { if (!have_run) return false; s.runs[live_run].wq_rel = -4096; return true; }},
        {"run without its pair", [&](Schedule& s) { if (!have_run) return false; s.runs[live_run].n = 0; return true; }},
        {"generator unit beyond the buffer", [&](Schedule& s) { s.gen_units.back().w_base = (uint32_t)s.weight_slots - 1; s.gen_units.back().count = 8; return true; }},
        {"generator unit too long", [&](Schedule& s) { s.gen_units[0].count = kGenUnitTaps + 1; return true; }},
        {"generator unit window", [&](Schedule& s) { s.gen_units[0].half = n_phi / 2; return true; }},
        {"generator unit taps beyond one turn", [&](Schedule& s) { s.gen_units[0].d0 = -n_phi; return true; }},
        {"generator unit dropped", [&](Schedule& s) { s.gen_units.pop_back(); return true; }},
        {"wide shared memory too small", [&](Schedule& s) { if (s.first_narrow == 0) return false; s.smem_wide = 1024; return true; }},
        {"narrow shared memory too small", [&](Schedule& s) { if (s.first_narrow >= s.n_north) return false; s.smem_narrow = 1024; return true; }},
        {"shared memory over budget", [&](Schedule& s) { s.smem_wide = kSmemBudget + 16; return true; }},
        {"wide / narrow split of the work list", [&](Schedule& s) { if (first_wide < 0 || first_narrow_item < 0) return false; s.n_wide_items -= 1; return true; }},
        {"narrow weight stride misaligned", [&](Schedule& s) { if (s.first_narrow >= s.n_north) return false; s.narrow_wslot += 2; return true; }},
        {"runs table truncated", [&](Schedule& s) { if (s.runs.empty()) return false; s.runs.pop_back(); return true; }},
        {"pairs table truncated", [&](Schedule& s) { s.pairs.pop_back(); return true; }},
    };
    int rejected = 0, skipped = 0;
    for (const Mut& m : muts) {
        Schedule s = base;
        if (!m.apply(s)) { skipped++; continue; }
        std::string w;
        if (validate_schedule(s, &w) == 0) { std::fprintf(stderr, "NOT rejected: %s\n", m.name); return 1; }
        rejected++;
    }
    (void)W;
    std::printf("ok: %d mutations rejected, %d not applicable; items %zu, R %d, first_narrow %d of %d\n", rejected, skipped,
                base.items.size(), base.R, base.first_narrow, base.n_north);
    return 0;
}
