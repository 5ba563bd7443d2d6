// Host packer of the slice-JDS way/block streams (layout: amgdd_stream.hpp).  Index work only; no
// arithmetic of the method.  One walker lays the pieces down; the planner and the writer are two
// sets of callbacks on it, so they cannot disagree.
#include "amgdd_stream.hpp"

#include <algorithm>
#include <cstring>
#include <vector>

namespace amgdd {

namespace {

inline int64_t align16(int64_t x) { return (x + 15) & ~(int64_t)15; }

struct Slice {
    int row_base;                 // first row of the window
    int nrows;                    // rows in the slice (<= 32)
    int group;                    // 0: rows < n_real, 1: the rest
    int rows[SLICE_ROWS];         // row of lane j (sorted by descending length, stable)
    int len[SLICE_ROWS];
    int K;                        // longest row
    int64_t nnz;
};

struct Piece {
    const Slice* sl;
    int k0, nk, nnz;
    int64_t data_bytes;           // padded to 16
};

inline int prefix_bytes(bool has_aux) { return SLICE_ROWS * 2 * 2 + (has_aux ? SLICE_ROWS * 8 : 0); }

// entries of step k of a slice = rows longer than k (a prefix of the lanes)
inline int step_count(const Slice& s, int k) {
    int c = 0;
    while (c < s.nrows && s.len[c] > k) ++c;
    return c;
}

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
                sl.row_base = w0;
                sl.group = g;
                sl.nrows = std::min(SLICE_ROWS, w1 - w0 - s0);
                sl.nnz = 0;
                for (int j = 0; j < SLICE_ROWS; ++j) {
                    sl.rows[j] = j < sl.nrows ? order[s0 + j] : -1;
                    sl.len[j] = j < sl.nrows ? rp[sl.rows[j] + 1] - rp[sl.rows[j]] : 0;
                    sl.nnz += sl.len[j];
                }
                sl.K = sl.len[0];
                out.push_back(sl);
            }
        }
}

// slices -> ways: in slice order, each to the way with the fewest bytes so far (ties: lowest way)
void deal(const std::vector<Slice>& slices, bool wide, bool has_aux, std::vector<int> (&of_way)[NUM_WAYS]) {
    int64_t load[NUM_WAYS];
    for (int w = 0; w < NUM_WAYS; ++w) { load[w] = 0; of_way[w].clear(); }
    for (size_t i = 0; i < slices.size(); ++i) {
        int best = 0;
        for (int w = 1; w < NUM_WAYS; ++w) if (load[w] < load[best]) best = w;
        load[best] += PIECE_DESC_BYTES + prefix_bytes(has_aux) + slices[i].nnz * (wide ? 12 : 10);
        of_way[best].push_back((int)i);
    }
}

inline int64_t block_used_bytes(const std::vector<Piece>& pcs) {
    int64_t b = BLOCK_HEADER_BYTES;
    for (const Piece& p : pcs) b += PIECE_DESC_BYTES + p.data_bytes;
    return b;
}

// Lays the slices of one way down; calls on_block(block_index, pieces) for every block, in order.
// Returns {nblocks, nblocks_real, nslices_real, bytes of the last block}.
struct WayResult { int nblocks, nblocks_real, nslices_real; int64_t last_bytes; };

template <class OnBlock>
WayResult walk_way(const std::vector<Slice>& slices, const std::vector<int>& mine, bool wide, bool has_aux, int block_bytes,
                   OnBlock on_block) {
    const int cw = wide ? 4 : 2;
    std::vector<Piece> pending;
    int64_t used = BLOCK_HEADER_BYTES;
    int block = 0;
    WayResult res = {0, 0, 0, 0};
    auto close = [&]() {
        if (pending.empty()) return;
        res.last_bytes = block_used_bytes(pending);
        on_block(block, pending);
        pending.clear();
        used = BLOCK_HEADER_BYTES;
        ++block;
    };
    for (int si : mine) {
        const Slice& sl = slices[si];
        int k = 0;
        for (;;) {                                                 // at least one piece, also for K = 0
            const int64_t fixed = PIECE_DESC_BYTES + (k == 0 ? prefix_bytes(has_aux) : 0);
            const int64_t room = block_bytes - used - fixed;
            int nk = 0, nnz = 0;
            if (room >= 0) {
                while (k + nk < sl.K) {
                    const int c = step_count(sl, k + nk);
                    if (nnz + c > 65535 || align16((int64_t)(nnz + c) * (8 + cw)) > room) break;
                    nnz += c;
                    ++nk;
                }
            }
            if (room < 0 || (nk == 0 && sl.K > 0)) { close(); continue; }   // nothing fits: next block
            Piece pc;
            pc.sl = &sl; pc.k0 = k; pc.nk = nk; pc.nnz = nnz;
            pc.data_bytes = (k == 0 ? prefix_bytes(has_aux) : 0) + align16((int64_t)nnz * (8 + cw));
            used += PIECE_DESC_BYTES + pc.data_bytes;
            pending.push_back(pc);
            k += nk;
            if (k >= sl.K) break;
        }
        if (sl.group == 0) { ++res.nslices_real; res.nblocks_real = block + 1; }
    }
    close();
    res.nblocks = block;
    return res;
}

void write_block(const std::vector<Piece>& pcs, const int32_t* rp, const int32_t* ci, const double* v, const double* aux,
                 bool wide, char* out) {
    const bool has_aux = aux != nullptr;
    std::memset(out, 0, (size_t)block_used_bytes(pcs));
    uint32_t hdr[4] = {(uint32_t)pcs.size(), 0, 0, 0};
    std::memcpy(out, hdr, 16);
    int64_t off = BLOCK_HEADER_BYTES + (int64_t)PIECE_DESC_BYTES * (int64_t)pcs.size();
    for (size_t i = 0; i < pcs.size(); ++i) {
        const Piece& pc = pcs[i];
        const Slice& sl = *pc.sl;
        PieceDesc d;
        d.off = (uint32_t)off; d.row_base = (uint32_t)sl.row_base;
        d.k0 = (uint16_t)pc.k0; d.nk = (uint16_t)pc.nk; d.K = (uint16_t)sl.K; d.nnz = (uint16_t)pc.nnz;
        std::memcpy(out + BLOCK_HEADER_BYTES + i * PIECE_DESC_BYTES, &d, sizeof(d));
        char* q = out + off;
        if (pc.k0 == 0) {
            uint16_t* rowid = (uint16_t*)q;
            uint16_t* len = rowid + SLICE_ROWS;
            for (int j = 0; j < SLICE_ROWS; ++j) {
                rowid[j] = sl.rows[j] >= 0 ? (uint16_t)(sl.rows[j] - sl.row_base) : NO_ROW;
                len[j] = (uint16_t)sl.len[j];
            }
            q += SLICE_ROWS * 4;
            if (has_aux) {
                double* a = (double*)q;
                for (int j = 0; j < SLICE_ROWS; ++j) a[j] = sl.rows[j] >= 0 ? aux[sl.rows[j]] : 0.0;
                q += SLICE_ROWS * 8;
            }
        }
        double* vv = (double*)q;
        char* cc = q + (int64_t)pc.nnz * 8;
        int e = 0;
        for (int k = pc.k0; k < pc.k0 + pc.nk; ++k)
            for (int j = 0; j < sl.nrows && sl.len[j] > k; ++j, ++e) {
                const int src = rp[sl.rows[j]] + k;
                vv[e] = v[src];
                if (wide) ((uint32_t*)cc)[e] = (uint32_t)ci[src];
                else ((uint16_t*)cc)[e] = (uint16_t)ci[src];
            }
        off += pc.data_bytes;
    }
}

}  // namespace

PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, bool has_aux, int block_bytes, int n_real, int window) {
    PackPlan p;
    std::memset(&p, 0, sizeof(p));
    std::vector<Slice> slices;
    build_slices(nrows, rp, n_real, window, slices);
    std::vector<int> of_way[NUM_WAYS];
    deal(slices, wide, has_aux, of_way);
    p.nslices = (int)slices.size();
    int64_t off = 0;
    for (int w = 0; w < NUM_WAYS; ++w) {
        const WayResult r = walk_way(slices, of_way[w], wide, has_aux, block_bytes, [](int, const std::vector<Piece>&) {});
        WayDesc& d = p.way[w];
        d.off16 = (uint32_t)(off / 16);
        d.nblocks = (uint32_t)r.nblocks; d.nblocks_real = (uint32_t)r.nblocks_real;
        d.last16 = (uint16_t)(r.last_bytes / 16); d.nslices_real = (uint16_t)r.nslices_real;
        if (r.nblocks > 0) off += (int64_t)(r.nblocks - 1) * block_bytes + r.last_bytes;
        p.nblocks += r.nblocks; p.nblocks_real += r.nblocks_real; p.nslices_real += r.nslices_real;
    }
    p.bytes = off;
    return p;
}

void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, const double* aux, bool wide,
                  int block_bytes, int n_real, int window, char* dst) {
    const bool has_aux = aux != nullptr;
    std::vector<Slice> slices;
    build_slices(nrows, rp, n_real, window, slices);
    std::vector<int> of_way[NUM_WAYS];
    deal(slices, wide, has_aux, of_way);
    int64_t off = 0;
    for (int w = 0; w < NUM_WAYS; ++w) {
        char* base = dst + off;
        const WayResult r = walk_way(slices, of_way[w], wide, has_aux, block_bytes, [&](int b, const std::vector<Piece>& pcs) {
            write_block(pcs, rp, ci, v, aux, wide, base + (int64_t)b * block_bytes);
        });
        if (r.nblocks > 0) off += (int64_t)(r.nblocks - 1) * block_bytes + r.last_bytes;
    }
}

}  // namespace amgdd
