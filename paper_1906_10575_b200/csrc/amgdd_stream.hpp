// HBM layout of the AMG-DD solve phase: packed CSR streams and the per-(subdomain, level)
// descriptor tables.  Plain structs shared by the host packer (amgdd_pack.cpp, amgdd_composite.cpp,
// amgdd_api.cu) and the device kernel (amgdd_fac.cu); no CUDA types, no arithmetic of the method.
//
// PACKED CSR STREAM.  Every local matrix of a composite level (A_l, P_l, R_l = P_l^T; paper P:49,
// P:248) is stored as a sequence of fixed-stride CHUNKS of `chunk_bytes` bytes.  A chunk holds a
// run of whole consecutive rows and is moved HBM -> shared memory by ONE bulk async copy
// (cp.async.bulk, the 1-D TMA path), so the matrix crosses HBM exactly once per mat-vec in large
// contiguous requests that do not depend on any warp's progress:
//
//     byte  0  int32 row_begin      first row of the chunk
//           4  int32 nrows          rows in the chunk
//           8  int32 nnz            nonzeros in the chunk (<= 65535)
//          12  int32 reserved (0)
//          16  double  v[nnz]       values, row after row
//   16+8 nnz   colT    ci[nnz]      column indices: uint16 (narrow) or uint32 (wide stream)
//        ...   uint16  rowend[nrows]  exclusive end offset of each row inside v / ci
//     (padded with zeros to a multiple of 16 bytes; the last chunk of a stream is cut there)
//
// 10 bytes per nonzero + 2 per row in the narrow form (local column indices of a composite level
// fit 16 bits whenever |D-bar_l^p| <= 65536), against 12 + 4 of textbook CSR.
#pragma once
#include <cstdint>

namespace amgdd {

constexpr int CHUNK_HEADER_BYTES = 16;
constexpr int MIN_CHUNK_BYTES = 1024;
constexpr int MAX_CHUNK_BYTES = 65536;       // rowend offsets are 16-bit
constexpr int NARROW_MAX_COLS = 65536;       // uint16 column indices

// bytes a chunk with these counts occupies (before padding to 16)
inline int64_t chunk_payload_bytes(int64_t nrows, int64_t nnz, bool wide) {
    return CHUNK_HEADER_BYTES + nnz * (8 + (wide ? 4 : 2)) + nrows * 2;
}

struct StreamDesc {
    const char* base;      // DEVICE, 16-byte aligned; chunk c starts at base + c * chunk_bytes
    int nchunks;           // chunks holding all rows
    int nchunks_real;      // chunks holding at least one of the first n_real rows (A streams)
    int last_bytes;        // size of the last chunk (multiple of 16, <= chunk_bytes)
    int lanes;             // threads that share one row (power of two, <= 32)
    int wide;              // 1: uint32 column indices
    int pad_;
};

// one (subdomain, level) block; pointers are device addresses (private blob or the shared global copy)
struct DevLevel {
    int n_real;            // |D_l^p|
    int n_bar;             // |D-bar_l^p| = real + ghost
    const int* gid;        // n_bar global indices (real ascending, then ghost ascending; S7)
    const double* dinv;    // n_real
    StreamDesc A;          // n_bar rows: real rows complete, ghost rows restricted to real columns (A12)
    StreamDesc P;          // n_bar rows, columns local to level l+1 (unused on L)
    StreamDesc R;          // n_bar(l+1) rows, columns local to level l (unused on L)
    long long voff;        // offset (doubles) of this level's vectors u|t|s|f inside a workspace slot
};

struct DevSub {
    const int* owned;      // local indices (level 0) of the owned dofs Omega_0^p
    int n_owned;
    int pad_;
};

struct FacParams {
    const DevLevel* lev;       // [P][L+1]
    const DevSub* sub;         // [P]
    const int* order;          // processing order of the subdomains (largest first)
    int num_sub;
    int L;                     // coarsest level index
    const double* r_all;       // concatenated restricted residuals r_0 | r_1 | ... | r_L
    const long long* r_off;    // L+1 offsets into r_all
    double* x;                 // fine iterate, updated on owned dofs
    double* workspace;         // gridDim.x * slot_stride doubles
    long long slot_stride;
    long long scratch_off;     // offset of the scratch vector w inside a slot
    int* work_counter;
    int nfac;
    int nu;
    const double* lu;          // dense LU of A_L, column-major, unit lower
    const int* rowperm;
    int nL;
    // shared-memory plan of one CTA
    int chunk_bytes;           // ring slot size = stream chunk stride
    int stages;                // ring depth
    int x_cap;                 // doubles in the shared-memory gather buffer
};

struct FacLaunch {
    int grid;
    int block;                 // 32 * (1 producer warp + consumer warps)
    int smem_bytes;
};

// host-side packing (amgdd_pack.cpp) ---------------------------------------------------------
struct PackPlan {
    int64_t bytes;             // total stream bytes (16-aligned)
    int nchunks;
    int nchunks_real;          // chunks that contain a row < n_real
    int last_bytes;
    int64_t too_long_row;      // -1, or a row that does not fit one chunk
};
// rp: nrows+1 int32 offsets (rp[0] = 0)
PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, int chunk_bytes, int n_real);
// writes plan.bytes bytes (the gap between a chunk's padded end and the next chunk is left untouched)
void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, bool wide, int chunk_bytes,
                  char* dst);

int fac_smem_bytes(int chunk_bytes, int stages, int x_cap);
int fac_max_stages();
void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream);
int fac_configure(int device, int max_smem_optin);   // sets the kernel's dynamic-smem attribute; 0 on success

}  // namespace amgdd
