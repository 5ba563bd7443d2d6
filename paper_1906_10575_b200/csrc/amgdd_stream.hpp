// HBM layout of the AMG-DD solve phase: packed "slice-JDS" matrix streams and the per-(subdomain,
// level) descriptor tables.  Plain structs shared by the host packer (amgdd_pack.cpp,
// amgdd_composite.cpp, amgdd_api.cu) and the device kernel (amgdd_fac.cu); no CUDA types, no
// arithmetic of the method.
//
// PACKED STREAM.  Every local matrix of a composite level (A_l, P_l, R_l = P_l^T; paper P:49,
// P:248) is stored as a sequence of fixed-stride CHUNKS of `chunk_bytes` bytes, each moved
// HBM -> shared memory by ONE bulk async copy (cp.async.bulk, the 1-D TMA path), so the matrix
// crosses HBM exactly once per mat-vec in large contiguous requests.
//
// Rows are grouped for a 32-wide warp with ONE LANE PER ROW:
//   * the rows [0, n_real) and [n_real, nrows) are two GROUPS (real / ghost rows of A_l; other
//     matrices have one group); a group is cut into WINDOWS of `window` consecutive rows; inside a
//     window the rows are sorted by descending length (stable) and cut into SLICES of 32 rows
//     (the last slice of a group may hold fewer).  Lane j of a slice owns its j-th longest row.
//   * a slice with longest row K is stored as K STEPS (jagged diagonals): step k holds entry k of
//     every row of the slice that has more than k entries -- lanes [0, cnt_k) because of the
//     sort -- so nothing is padded: 8 + 2 (or 4) bytes per nonzero.
//   * a slice is laid down as one or more PIECES (consecutive step ranges); a piece never crosses
//     a chunk, a slice may.  The pieces of all slices follow each other in slice order.
//
//   chunk:  byte 0  uint32 npieces
//                4  uint32 slice0        stream-wide index of the slice of piece 0 (piece i belongs
//                                        to slice slice0 + i: only piece 0 can continue a slice)
//                8  uint32 reserved[2]
//               16  PieceDesc[npieces]   16 bytes each
//              ...  piece data, each piece 16-byte aligned
//           (the last chunk of a stream is cut at its 16-byte padded end)
//   piece:  [only if k0 == 0]  uint16 rowid[32]   row of lane j minus desc.row_base; 0xFFFF = no row
//                              uint16 len[32]     entries of that row (0 for "no row")
//                              double aux[32]     only in streams packed with an aux vector (A_l:
//                                                 the l1 diagonal inverse of the row, S8)
//           double v[nnz]      step after step
//           colT   ci[nnz]     uint16 (narrow) or uint32 (wide), same order
//           (zero padding to a multiple of 16 bytes)
#pragma once
#include <cstdint>

namespace amgdd {

constexpr int CHUNK_HEADER_BYTES = 16;
constexpr int PIECE_DESC_BYTES = 16;
constexpr int SLICE_ROWS = 32;
constexpr int MIN_CHUNK_BYTES = 1024;
constexpr int MAX_CHUNK_BYTES = 65536;
constexpr int NARROW_MAX_COLS = 65536;       // uint16 column indices
constexpr int MAX_WINDOW = 32768;            // rowid is 16-bit relative to the window, 0xFFFF reserved
constexpr int DEFAULT_WINDOW = 256;
constexpr uint16_t NO_ROW = 0xFFFF;

struct PieceDesc {
    uint32_t off;          // byte offset of the piece data from the start of the chunk (16-aligned)
    uint32_t row_base;     // first row of the slice's window
    uint16_t k0;           // first step of the slice held by this piece
    uint16_t nk;           // steps in this piece
    uint16_t K;            // steps of the whole slice (= its longest row); the piece is the last iff k0 + nk == K
    uint16_t nnz;          // entries in this piece
};
static_assert(sizeof(PieceDesc) == PIECE_DESC_BYTES, "PieceDesc layout");

struct StreamDesc {
    const char* base;      // DEVICE, 16-byte aligned; chunk c starts at base + c * chunk_bytes
    int nchunks;           // chunks holding all slices
    int nchunks_real;      // chunks holding the slices of the first group (rows < n_real)
    int last_bytes;        // size of the last chunk (multiple of 16, <= chunk_bytes)
    int nslices_real;      // slices of the first group
    int wide;              // 1: uint32 column indices
    int has_aux;           // 1: first pieces carry aux[32]
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
    long long* prof;           // optional: gridDim.x * FAC_PROF_SLOTS cycle counters (debugging), or nullptr
};
constexpr int FAC_PROF_SLOTS = 16;

struct FacLaunch {
    int grid;
    int block;                 // 32 * (1 producer warp + consumer warps)
    int smem_bytes;
};

// host-side packing (amgdd_pack.cpp) ---------------------------------------------------------
struct PackPlan {
    int64_t bytes;             // total stream bytes (16-aligned)
    int nchunks;
    int nchunks_real;          // chunks that hold the slices of the first group (rows < n_real)
    int last_bytes;
    int nslices;
    int nslices_real;
};
// rp: nrows+1 int32 offsets (rp[0] = 0); window: rows per sort window (multiple of 32, <= MAX_WINDOW)
PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, bool has_aux, int chunk_bytes, int n_real, int window);
// writes plan.bytes bytes (the gap between a chunk's padded end and the next chunk is left untouched);
// aux: nrows doubles or nullptr (must match has_aux of the plan)
void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, const double* aux, bool wide,
                  int chunk_bytes, int n_real, int window, char* dst);

int fac_smem_bytes(int chunk_bytes, int stages, int x_cap);
int fac_max_stages();
void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream);
int fac_configure(int device, int max_smem_optin);   // sets the kernel's dynamic-smem attribute; 0 on success

}  // namespace amgdd
