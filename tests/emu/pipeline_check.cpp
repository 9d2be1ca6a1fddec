// pipeline_check.cpp - test of the host<->device pipeline schedule of arkcos_convolve_host (build_pipeline in
// csrc/arkcos_schedule.cpp).  Test infrastructure only.  For one grid and several chunk counts it checks that
//   1. the pipeline's items are exactly the schedule's items, each once, grouped as (group, WIDE | NARROW);
//   2. every item of group g reads input rings below the end of chunk g only (they are on the device when it runs);
//   3. every item that writes into chunk c belongs to a group <= ready_group[c] (the chunk is complete when it is
//      copied back), and ready_group[c] >= c.
//   pipeline_check n_theta n_phi theta_cut
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "arkcos_internal.h"

using namespace arkcos;

static bool same(const Item& a, const Item& b) { return std::memcmp(&a, &b, sizeof(Item)) == 0; }

int main(int argc, char** argv) {
    if (argc < 4) return 2;
    const int n_theta = std::atoi(argv[1]), n_phi = std::atoi(argv[2]);
    Schedule s;
    if (build_schedule(n_theta, n_phi, std::atof(argv[3]), 148, s) != 0) { std::fprintf(stderr, "build_schedule failed\n"); return 1; }
    int checked = 0;
    for (int n_chunks : {1, 2, 3, 5, 8, 16, 1000}) {
        Pipeline p;
        build_pipeline(s, n_chunks, p);
        const int nc = p.n_chunks;
        if (nc < 1 || nc > n_theta || (int)p.chunk_lo.size() != nc + 1 || p.chunk_lo[0] != 0 || p.chunk_lo[nc] != n_theta) { std::fprintf(stderr, "chunks\n"); return 1; }
        for (int c = 0; c < nc; c++) if (p.chunk_lo[c + 1] <= p.chunk_lo[c]) { std::fprintf(stderr, "empty chunk\n"); return 1; }
        if (p.items.size() != s.items.size()) { std::fprintf(stderr, "item count\n"); return 1; }
        std::vector<char> used(s.items.size(), 0);
        for (int g = 0; g < nc; g++) {
            if (p.wide_begin[g] > p.narrow_begin[g] || p.narrow_begin[g] > p.wide_begin[g + 1]) { std::fprintf(stderr, "ranges\n"); return 1; }
            for (int k = p.wide_begin[g]; k < p.wide_begin[g + 1]; k++) {
                const Item& it = p.items[k];
                if ((it.kind == kWide) != (k < p.narrow_begin[g])) { std::fprintf(stderr, "class order in group %d\n", g); return 1; }
                size_t q = 0;
                while (q < s.items.size() && (used[q] || !same(s.items[q], it))) q++;
                if (q == s.items.size()) { std::fprintf(stderr, "item not in the schedule (or twice)\n"); return 1; }
                used[q] = 1;
                int lo, hi;
                item_output_rings(s, it, lo, hi);
                if (lo < 0 || hi >= n_theta || lo > hi) { std::fprintf(stderr, "output rings\n"); return 1; }
                if (std::min(n_theta - 1, hi + s.R) >= p.chunk_lo[g + 1]) { std::fprintf(stderr, "item of group %d reads ring %d beyond its chunk\n", g, hi + s.R); return 1; }
                for (int c = 0; c < nc; c++) {
                    const bool writes = lo < p.chunk_lo[c + 1] && hi >= p.chunk_lo[c];
                    if (writes && p.ready_group[c] < g) { std::fprintf(stderr, "chunk %d copied back before group %d wrote it\n", c, g); return 1; }
                }
            }
        }
        for (int c = 0; c < nc; c++) if (p.ready_group[c] < c || p.ready_group[c] >= nc) { std::fprintf(stderr, "ready_group\n"); return 1; }
        checked++;
    }
    std::printf("ok: %d chunkings, %zu items\n", checked, s.items.size());
    return 0;
}
