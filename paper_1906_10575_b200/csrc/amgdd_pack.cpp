// Host packer of the SELL-32 group streams (layout: amgdd_stream.hpp).  Index work only; no
// arithmetic of the method.  One routine cuts the rows into slices and deals them to the ways;
// the planner and the writer both run it, so they cannot disagree.
#include "amgdd_stream.hpp"

#include <algorithm>
#include <cstring>
#include <vector>

namespace amgdd {

namespace {

inline int64_t align128(int64_t x) { return (x + 127) & ~(int64_t)127; }

struct Slice {
    int nrows;                    // rows in the slice (<= 32)
    int group;                    // 0: rows < n_real, 1: the rest
    int rows[SLICE_ROWS];         // row of lane j (sorted by descending length, stable); -1: none
    int len[SLICE_ROWS];
    int K;                        // groups of the slice = max(1, ceil(longest row / 4))
};

void build_slices(int nrows, const int32_t* rp, int n_real, int window, std::vector<Slice>& out) {
    out.clear();
    std::vector<int> order;
    const int gb[3] = {0, std::min(n_real, nrows), nrows};
    for (int g = 0; g < 2; ++g)
        for (int w0 = gb[g]; w0 < gb[g + 1]; w0 += window) {
            const int w1 = std::min(w0 + window, gb[g + 1]);
            order.resize(w1 - w0);
            for (int i = 0; i < w1 - w0; ++i) order[i] = w0 + i;
            std::stable_sort(order.begin(), order.end(),
                             [&](int a, int b) { return rp[a + 1] - rp[a] > rp[b + 1] - rp[b]; });
            for (int s0 = 0; s0 < w1 - w0; s0 += SLICE_ROWS) {
                Slice sl;
                sl.group = g;
                sl.nrows = std::min(SLICE_ROWS, w1 - w0 - s0);
                for (int j = 0; j < SLICE_ROWS; ++j) {
                    sl.rows[j] = j < sl.nrows ? order[s0 + j] : -1;
                    sl.len[j] = j < sl.nrows ? rp[sl.rows[j] + 1] - rp[sl.rows[j]] : 0;
                }
                sl.K = std::max(1, (sl.len[0] + GROUP_STEPS - 1) / GROUP_STEPS);
                out.push_back(sl);
            }
        }
}

// slices -> ways: in slice order, each to the way with the fewest bytes so far (ties: lowest way)
void deal(const std::vector<Slice>& slices, int gbytes, int hbytes, std::vector<int> (&of_way)[NUM_WAYS]) {
    int64_t load[NUM_WAYS];
    for (int w = 0; w < NUM_WAYS; ++w) { load[w] = 0; of_way[w].clear(); }
    for (size_t i = 0; i < slices.size(); ++i) {
        int best = 0;
        for (int w = 1; w < NUM_WAYS; ++w) if (load[w] < load[best]) best = w;
        load[best] += (int64_t)slices[i].K * gbytes + hbytes;
        of_way[best].push_back((int)i);
    }
}

PackPlan make_plan(const std::vector<Slice>& slices, const std::vector<int> (&of_way)[NUM_WAYS], int gbytes, int hbytes) {
    PackPlan p;
    std::memset(&p, 0, sizeof(p));
    for (int w = 0; w < NUM_WAYS; ++w) {
        WayDesc& d = p.way[w];
        for (int si : of_way[w]) {
            const Slice& sl = slices[si];
            d.ngroups += (uint32_t)sl.K;
            d.nslices += 1;
            if (sl.group == 0) { d.ngroups_real += (uint32_t)sl.K; d.nslices_real += 1; }
        }
        p.ngroups += d.ngroups; p.ngroups_real += d.ngroups_real;
        p.nslices += d.nslices; p.nslices_real += d.nslices_real;
    }
    int64_t off = 0;
    for (int w = 0; w < NUM_WAYS; ++w) { p.way[w].grp_off128 = (uint32_t)(off / 128); off += (int64_t)p.way[w].ngroups * gbytes; }
    for (int w = 0; w < NUM_WAYS; ++w) { p.way[w].hdr_off128 = (uint32_t)(off / 128); off = align128(off + (int64_t)p.way[w].nslices * hbytes); }
    p.bytes = off;
    p.bytes_real = p.ngroups_real * gbytes + p.nslices_real * hbytes;
    p.padded_nnz = p.ngroups * GROUP_STEPS * SLICE_ROWS;
    return p;
}

}  // namespace

PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, int n_real, int window) {
    std::vector<Slice> slices;
    build_slices(nrows, rp, n_real, window, slices);
    std::vector<int> of_way[NUM_WAYS];
    deal(slices, group_bytes(wide), header_bytes(wide), of_way);
    return make_plan(slices, of_way, group_bytes(wide), header_bytes(wide));
}

void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, bool wide,
                  int n_real, int window, char* dst, const uint8_t* row_flags) {
    const int gbytes = group_bytes(wide), hbytes = header_bytes(wide);
    std::vector<Slice> slices;
    build_slices(nrows, rp, n_real, window, slices);
    std::vector<int> of_way[NUM_WAYS];
    deal(slices, gbytes, hbytes, of_way);
    const PackPlan p = make_plan(slices, of_way, gbytes, hbytes);
    std::memset(dst, 0, (size_t)p.bytes);
    for (int w = 0; w < NUM_WAYS; ++w) {
        char* g = dst + 128 * (int64_t)p.way[w].grp_off128;
        char* h = dst + 128 * (int64_t)p.way[w].hdr_off128;
        for (int si : of_way[w]) {
            const Slice& sl = slices[si];
            for (int j = 0; j < SLICE_ROWS; ++j) {
                const uint32_t flag = (row_flags && sl.rows[j] >= 0 && row_flags[sl.rows[j]]) ? 0x80000000u : 0u;
                if (wide) {                                                  // { row, K | flag << 31 }
                    const uint32_t row = sl.rows[j] >= 0 ? (uint32_t)sl.rows[j] : NO_ROW;
                    const uint32_t k = (uint32_t)sl.K | flag;
                    std::memcpy(h + 8 * j, &row, 4); std::memcpy(h + 8 * j + 4, &k, 4);
                } else {                                                     // row | K << 16 | flag << 31
                    const uint32_t w = (sl.rows[j] >= 0 ? (uint32_t)sl.rows[j] : (uint32_t)NO_ROW16) | ((uint32_t)sl.K << 16) | flag;
                    std::memcpy(h + 4 * j, &w, 4);
                }
            }
            h += hbytes;
            for (int kg = 0; kg < sl.K; ++kg, g += gbytes)
                for (int j = 0; j < sl.nrows; ++j)
                    for (int s = 0; s < GROUP_STEPS; ++s) {
                        const int k = kg * GROUP_STEPS + s;
                        if (k >= sl.len[j]) break;                          // padding stays 0.0 / column 0
                        const int src = rp[sl.rows[j]] + k;
                        std::memcpy(g + (s >> 1) * 512 + 16 * j + 8 * (s & 1), &v[src], 8);
                        if (wide) { const uint32_t c = (uint32_t)ci[src]; std::memcpy(g + 1024 + 16 * j + 4 * s, &c, 4); }
                        else { const uint16_t c = (uint16_t)ci[src]; std::memcpy(g + 1024 + 8 * j + 2 * s, &c, 2); }
                    }
        }
    }
}

}  // namespace amgdd
