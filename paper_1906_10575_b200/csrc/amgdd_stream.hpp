// HBM layout of the AMG-DD solve phase: packed "slice-JDS" matrix streams and the per-(subdomain,
// level) descriptor tables.  Plain structs shared by the host packer (amgdd_pack.cpp,
// amgdd_composite.cpp, amgdd_api.cu) and the device kernel (amgdd_fac.cu); no CUDA types, no
// arithmetic of the method.
//
// PACKED STREAM.  Every local matrix of a composite level (A_l, P_l, R_l = P_l^T; paper P:49,
// P:248) is stored as NUM_WAYS independent sub-streams ("ways"), one per consumer warp of the
// AlgFAC kernel.  A way is a sequence of fixed-stride BLOCKS of `block_bytes` bytes; warp w moves
// the blocks of way w HBM -> its own shared-memory ring with one bulk async copy each
// (cp.async.bulk, the 1-D TMA path) and consumes them in order, so a mat-vec needs no
// communication between warps and the matrix crosses HBM exactly once, in contiguous requests.
//
// Rows are grouped for a 32-wide warp with ONE LANE PER ROW:
//   * the rows [0, n_real) and [n_real, nrows) are two GROUPS (real / ghost rows of A_l; other
//     matrices have one group); a group is cut into WINDOWS of `window` consecutive rows; inside a
//     window the rows are sorted by descending length (stable) and cut into SLICES of 32 rows
//     (the last slice of a group may hold fewer).  Lane j of a slice owns its j-th longest row.
//   * a slice with longest row K is stored as K STEPS (jagged diagonals): step k holds entry k of
//     every row of the slice that has more than k entries -- lanes [0, cnt_k) because of the
//     sort -- so nothing is padded: 8 + 2 (or 4) bytes per nonzero.
//   * slices are dealt to the ways in slice order, each to the way with the fewest bytes so far
//     (ties: lowest way), first all slices of the first group, then those of the second; inside a
//     way they keep that order.  A slice is laid down as one or more PIECES (consecutive step
//     ranges); a piece never crosses a block, a slice may.
//
//   way w:  blocks at  base + 16 * way[w].off16 + j * block_bytes,  j < way[w].nblocks; the last
//           block of a way is cut at its 16-byte padded end (16 * way[w].last16 bytes)
//   block:  byte 0  uint32 npieces
//                4  uint32 reserved[3]
//               16  PieceDesc[npieces]   16 bytes each
//              ...  piece data, each piece 16-byte aligned
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

constexpr int NUM_WAYS = 16;                 // consumer warps of the AlgFAC kernel = sub-streams per matrix
constexpr int BLOCK_HEADER_BYTES = 16;
constexpr int PIECE_DESC_BYTES = 16;
constexpr int SLICE_ROWS = 32;
constexpr int MIN_BLOCK_BYTES = 1024;
constexpr int MAX_BLOCK_BYTES = 32768;
constexpr int DEFAULT_BLOCK_BYTES = 2048;
constexpr int NARROW_MAX_COLS = 65536;       // uint16 column indices
constexpr int MAX_WINDOW = 32768;            // rowid is 16-bit relative to the window, 0xFFFF reserved
constexpr int DEFAULT_WINDOW = 256;
constexpr uint16_t NO_ROW = 0xFFFF;

struct PieceDesc {
    uint32_t off;          // byte offset of the piece data from the start of the block (16-aligned)
    uint32_t row_base;     // first row of the slice's window
    uint16_t k0;           // first step of the slice held by this piece
    uint16_t nk;           // steps in this piece
    uint16_t K;            // steps of the whole slice (= its longest row); the piece is the last iff k0 + nk == K
    uint16_t nnz;          // entries in this piece
};
static_assert(sizeof(PieceDesc) == PIECE_DESC_BYTES, "PieceDesc layout");

struct WayDesc {           // one sub-stream (same layout as amgdd_way_t of include/amgdd.h)
    uint32_t off16;        // start of the way, in units of 16 bytes from the stream base
    uint32_t nblocks;      // blocks of the way
    uint32_t nblocks_real; // blocks that hold the way's slices of the first group
    uint16_t last16;       // size of the last block in units of 16 bytes (<= block_bytes / 16)
    uint16_t nslices_real; // the way's slices of the first group
};
static_assert(sizeof(WayDesc) == 16, "WayDesc layout");

struct StreamDesc {
    const char* base;      // DEVICE, 16-byte aligned
    WayDesc way[NUM_WAYS];
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
    int nops;                  // steps in the program of one subdomain = fac_num_ops(L, nfac, nu)
    const double* lu;          // dense LU of A_L, column-major, unit lower
    const int* rowperm;
    int nL;
    // shared-memory plan of one CTA
    int block_bytes;           // ring slot size = stream block stride
    int stages;                // ring depth of every warp
    int x_cap;                 // doubles in the shared-memory gather buffer
    int table_bytes;           // bytes of one descriptor table slot = (L+1) * sizeof(DevLevel), 16-aligned
    long long* prof;           // optional: gridDim.x * FAC_PROF_SLOTS cycle counters (debugging), or nullptr
};
constexpr int FAC_PROF_SLOTS = 16;

struct FacLaunch {
    int grid;
    int block;                 // 32 * NUM_WAYS
    int smem_bytes;
};

// host-side packing (amgdd_pack.cpp) ---------------------------------------------------------
struct PackPlan {
    int64_t bytes;             // total stream bytes (16-aligned)
    WayDesc way[NUM_WAYS];
    int64_t nblocks;           // blocks over all ways
    int64_t nblocks_real;
    int nslices, nslices_real;
};
// rp: nrows+1 int32 offsets (rp[0] = 0); window: rows per sort window (multiple of 32, <= MAX_WINDOW);
// rows must have at most 65535 entries
PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, bool has_aux, int block_bytes, int n_real, int window);
// writes plan.bytes bytes; aux: nrows doubles or nullptr (must match has_aux of the plan)
void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, const double* aux, bool wide,
                  int block_bytes, int n_real, int window, char* dst);

int fac_smem_bytes(int block_bytes, int stages, int x_cap, int table_bytes);
int fac_max_stages();
int fac_num_ops(int L, int nfac, int nu);   // steps in the program of one subdomain
int fac_max_ops();                          // the longest program the kernel has room for
void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream);
int fac_configure(int device, int max_smem_optin);   // sets the kernel's dynamic-smem attribute; 0 on success

}  // namespace amgdd
