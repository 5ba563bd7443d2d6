// Host packer of the slice-JDS chunk stream (layout: amgdd_stream.hpp).  Index work only; no
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
    int rows[SLICE_ROWS];         // row of lane j (sorted by descending length, stable)
    int len[SLICE_ROWS];
    int K;                        // longest row
};

struct Piece {
    Slice sl;
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

// Calls on_chunk(chunk_index, pieces) for every chunk, in order.  Returns {nslices, nslices_real,
// chunk index holding the end of the last slice of the first group (-1 if that group is empty)}.
struct WalkResult { int nslices, nslices_real, last_real_chunk; };

template <class OnChunk>
WalkResult walk(int nrows, const int32_t* rp, bool wide, bool has_aux, int chunk_bytes, int n_real, int window,
                OnChunk on_chunk) {
    const int cw = wide ? 4 : 2;
    std::vector<Piece> pending;
    int64_t used = CHUNK_HEADER_BYTES;
    int chunk = 0;
    WalkResult res = {0, 0, -1};
    auto close = [&]() {
        if (pending.empty()) return;
        on_chunk(chunk, pending);
        pending.clear();
        used = CHUNK_HEADER_BYTES;
        ++chunk;
    };
    std::vector<int> order;
    const int gb[3] = {0, std::min(n_real, nrows), nrows};
    for (int g = 0; g < 2; ++g) {
        for (int w0 = gb[g]; w0 < gb[g + 1]; w0 += window) {
            const int w1 = std::min(w0 + window, gb[g + 1]);
            order.resize(w1 - w0);
            for (int i = 0; i < w1 - w0; ++i) order[i] = w0 + i;
            std::stable_sort(order.begin(), order.end(),
                             [&](int a, int b) { return rp[a + 1] - rp[a] > rp[b + 1] - rp[b]; });
            for (int s0 = 0; s0 < w1 - w0; s0 += SLICE_ROWS) {
                Slice sl;
                sl.row_base = w0;
                sl.nrows = std::min(SLICE_ROWS, w1 - w0 - s0);
                for (int j = 0; j < SLICE_ROWS; ++j) {
                    sl.rows[j] = j < sl.nrows ? order[s0 + j] : -1;
                    sl.len[j] = j < sl.nrows ? rp[sl.rows[j] + 1] - rp[sl.rows[j]] : 0;
                }
                sl.K = sl.len[0];
                ++res.nslices;
                if (g == 0) ++res.nslices_real;
                int k = 0;
                for (;;) {                                         // at least one piece, also for K = 0
                    const int64_t fixed = PIECE_DESC_BYTES + (k == 0 ? prefix_bytes(has_aux) : 0);
                    const int64_t room = chunk_bytes - used - fixed;
                    int nk = 0, nnz = 0;
                    if (room >= 0) {
                        while (k + nk < sl.K && nk < 65535) {
                            const int c = step_count(sl, k + nk);
                            if (nnz + c > 65535 || align16((int64_t)(nnz + c) * (8 + cw)) > room) break;
                            nnz += c;
                            ++nk;
                        }
                    }
                    if (room < 0 || (nk == 0 && sl.K > 0)) { close(); continue; }   // nothing fits: next chunk
                    Piece pc;
                    pc.sl = sl; pc.k0 = k; pc.nk = nk; pc.nnz = nnz;
                    pc.data_bytes = (k == 0 ? prefix_bytes(has_aux) : 0) + align16((int64_t)nnz * (8 + cw));
                    used += PIECE_DESC_BYTES + pc.data_bytes;
                    pending.push_back(pc);
                    k += nk;
                    if (k >= sl.K) break;
                }
                if (g == 0) res.last_real_chunk = chunk;
            }
        }
    }
    close();
    return res;
}

inline int64_t chunk_used_bytes(const std::vector<Piece>& pcs) {
    int64_t b = CHUNK_HEADER_BYTES;
    for (const Piece& p : pcs) b += PIECE_DESC_BYTES + p.data_bytes;
    return b;
}

}  // namespace

PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, bool has_aux, int chunk_bytes, int n_real, int window) {
    PackPlan p;
    p.bytes = 0; p.nchunks = 0; p.nchunks_real = 0; p.last_bytes = 0; p.nslices = 0; p.nslices_real = 0;
    const WalkResult r = walk(nrows, rp, wide, has_aux, chunk_bytes, n_real, window, [&](int, const std::vector<Piece>& pcs) {
        ++p.nchunks;
        p.last_bytes = (int)chunk_used_bytes(pcs);
    });
    p.nslices = r.nslices; p.nslices_real = r.nslices_real;
    p.nchunks_real = r.last_real_chunk + 1;
    if (p.nchunks > 0) p.bytes = (int64_t)(p.nchunks - 1) * chunk_bytes + p.last_bytes;
    return p;
}

void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, const double* aux, bool wide,
                  int chunk_bytes, int n_real, int window, char* dst) {
    const bool has_aux = aux != nullptr;
    int slice_counter = 0;                                         // slices started so far
    walk(nrows, rp, wide, has_aux, chunk_bytes, n_real, window, [&](int c, const std::vector<Piece>& pcs) {
        char* out = dst + (int64_t)c * chunk_bytes;
        const int64_t used = chunk_used_bytes(pcs);
        std::memset(out, 0, (size_t)used);
        // piece 0 continues the slice started last iff its k0 > 0
        const uint32_t slice0 = (uint32_t)(pcs[0].k0 > 0 ? slice_counter - 1 : slice_counter);
        uint32_t hdr[4] = {(uint32_t)pcs.size(), slice0, 0, 0};
        std::memcpy(out, hdr, 16);
        int64_t off = CHUNK_HEADER_BYTES + (int64_t)PIECE_DESC_BYTES * (int64_t)pcs.size();
        for (size_t i = 0; i < pcs.size(); ++i) {
            const Piece& pc = pcs[i];
            if (pc.k0 == 0) ++slice_counter;
            PieceDesc d;
            d.off = (uint32_t)off; d.row_base = (uint32_t)pc.sl.row_base;
            d.k0 = (uint16_t)pc.k0; d.nk = (uint16_t)pc.nk; d.K = (uint16_t)pc.sl.K; d.nnz = (uint16_t)pc.nnz;
            std::memcpy(out + CHUNK_HEADER_BYTES + i * PIECE_DESC_BYTES, &d, sizeof(d));
            char* q = out + off;
            if (pc.k0 == 0) {
                uint16_t* rowid = (uint16_t*)q;
                uint16_t* len = rowid + SLICE_ROWS;
                for (int j = 0; j < SLICE_ROWS; ++j) {
                    rowid[j] = pc.sl.rows[j] >= 0 ? (uint16_t)(pc.sl.rows[j] - pc.sl.row_base) : NO_ROW;
                    len[j] = (uint16_t)pc.sl.len[j];
                }
                q += SLICE_ROWS * 4;
                if (has_aux) {
                    double* a = (double*)q;
                    for (int j = 0; j < SLICE_ROWS; ++j) a[j] = pc.sl.rows[j] >= 0 ? aux[pc.sl.rows[j]] : 0.0;
                    q += SLICE_ROWS * 8;
                }
            }
            double* vv = (double*)q;
            char* cc = q + (int64_t)pc.nnz * 8;
            int e = 0;
            for (int k = pc.k0; k < pc.k0 + pc.nk; ++k)
                for (int j = 0; j < pc.sl.nrows && pc.sl.len[j] > k; ++j, ++e) {
                    const int src = rp[pc.sl.rows[j]] + k;
                    vv[e] = v[src];
                    if (wide) ((uint32_t*)cc)[e] = (uint32_t)ci[src];
                    else ((uint16_t*)cc)[e] = (uint16_t)ci[src];
                }
            off += pc.data_bytes;
        }
    });
}

}  // namespace amgdd
