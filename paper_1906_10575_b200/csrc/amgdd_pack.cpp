// Host packer of the chunked CSR stream format (layout: amgdd_stream.hpp).  Rows are packed
// greedily: a chunk takes consecutive whole rows while header + values + column indices + row
// ends fit `chunk_bytes`.  Index work only; no arithmetic of the method.
#include "amgdd_stream.hpp"

#include <cstring>

namespace amgdd {

namespace {

inline int64_t align16(int64_t x) { return (x + 15) & ~(int64_t)15; }

// calls emit(row_begin, row_end) for every chunk; returns a row that fits no chunk, or -1
template <class Emit>
int64_t for_each_chunk(int nrows, const int32_t* rp, bool wide, int chunk_bytes, Emit emit) {
    int r = 0;
    while (r < nrows) {
        int e = r;
        int64_t nnz = 0;
        while (e < nrows) {
            const int64_t len = rp[e + 1] - rp[e];
            if (nnz + len > 65535) break;                                   // rowend is 16-bit
            if (chunk_payload_bytes(e + 1 - r, nnz + len, wide) > chunk_bytes) break;
            nnz += len;
            ++e;
        }
        if (e == r) return r;                                               // row r alone is too long
        emit(r, e);
        r = e;
    }
    return -1;
}

}  // namespace

PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, int chunk_bytes, int n_real) {
    PackPlan p;
    p.bytes = 0; p.nchunks = 0; p.nchunks_real = 0; p.last_bytes = 0;
    p.too_long_row = for_each_chunk(nrows, rp, wide, chunk_bytes, [&](int r, int e) {
        ++p.nchunks;
        if (r < n_real) p.nchunks_real = p.nchunks;
        p.last_bytes = (int)align16(chunk_payload_bytes(e - r, rp[e] - rp[r], wide));
    });
    if (p.nchunks > 0) p.bytes = (int64_t)(p.nchunks - 1) * chunk_bytes + p.last_bytes;
    return p;
}

void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, bool wide, int chunk_bytes,
                  char* dst) {
    int c = 0;
    for_each_chunk(nrows, rp, wide, chunk_bytes, [&](int r, int e) {
        char* out = dst + (int64_t)c * chunk_bytes;
        const int nnz = rp[e] - rp[r], nr = e - r;
        const int64_t used = chunk_payload_bytes(nr, nnz, wide);
        const int64_t padded = align16(used);
        int32_t hdr[4] = {r, nr, nnz, 0};
        std::memcpy(out, hdr, 16);
        std::memcpy(out + 16, v + rp[r], (size_t)nnz * 8);
        char* pci = out + 16 + (int64_t)nnz * 8;
        if (wide) {
            std::memcpy(pci, ci + rp[r], (size_t)nnz * 4);
            pci += (int64_t)nnz * 4;
        } else {
            uint16_t* c16 = (uint16_t*)pci;
            for (int k = 0; k < nnz; ++k) c16[k] = (uint16_t)ci[rp[r] + k];
            pci += (int64_t)nnz * 2;
        }
        uint16_t* re = (uint16_t*)pci;
        for (int i = 0; i < nr; ++i) re[i] = (uint16_t)(rp[r + i + 1] - rp[r]);
        std::memset(out + used, 0, (size_t)(padded - used));
        ++c;
    });
}

}  // namespace amgdd
