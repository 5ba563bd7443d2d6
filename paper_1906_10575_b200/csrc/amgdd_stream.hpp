// HBM layout of the AMG-DD solve phase: packed "SELL-32 group" matrix streams, the per-(subdomain,
// level) descriptor tables and the static program of one subdomain.  Plain structs shared by the
// host packer (amgdd_pack.cpp, amgdd_composite.cpp, amgdd_api.cu) and the device kernel
// (amgdd_fac.cu); no CUDA types, no arithmetic of the method.
//
// PACKED STREAM.  Every local matrix of a composite level (A_l, P_l, R_l = P_l^T; paper P:49,
// P:248) is stored as NUM_WAYS independent sub-streams ("ways"), one per warp of the AlgFAC
// kernel.  Warp w reads way w with coalesced 128-bit loads straight into a ring of registers and
// runs several groups ahead of its arithmetic, so a mat-vec needs no communication between warps
// and the matrix crosses HBM exactly once, in 512-byte requests.
//
// Rows are grouped for a 32-wide warp with ONE LANE PER ROW (sliced ELLPACK, slice height 32):
//   * the rows [0, n_real) and [n_real, nrows) are two ROW GROUPS (real / ghost rows of A_l; other
//     matrices have one); a row group is cut into WINDOWS of `window` consecutive rows; inside a
//     window the rows are sorted by descending length (stable) and cut into SLICES of 32 rows (the
//     last slice of a row group may hold fewer).  Lane j of a slice owns its j-th longest row.
//   * a slice whose longest row has len entries is stored as K = max(1, ceil(len / 4)) GROUPS of
//     4 STEPS; step k of lane j is entry k of the lane's row, in stored (= CSR) order; steps past
//     the end of a row are padding (value 0.0, column 0).
//   * slices are dealt to the ways in slice order, each to the way with the fewest bytes so far
//     (ties: lowest way), first all slices of the first row group, then those of the second;
//     inside a way they keep that order, so the slices of the first row group are a prefix of
//     every way (what a real-rows-only mat-vec reads).
//
//   stream:  [groups of way 0] ... [groups of way 15] [headers of way 0] ... [headers of way 15]
//   way w:   groups at   base + 128 * way[w].grp_off128 + g * group_bytes,   g < way[w].ngroups
//            headers at  base + 128 * way[w].hdr_off128 + s * header_bytes,  s < way[w].nslices
//   group (narrow, 1280 bytes):  32 x { double v[step 0], v[step 1] }     lane j at byte 16 j
//                                32 x { double v[step 2], v[step 3] }     lane j at 512 + 16 j
//                                32 x { uint16 col[step 0..3] }           lane j at 1024 + 8 j
//   group (wide, 1536 bytes):    the same two value planes, then 32 x { uint32 col[step 0..3] },
//                                lane j at 1024 + 16 j
//   header (narrow, 128 bytes):  32 x uint32  row | K << 16 | flag << 31      lane j at 4 j
//   header (wide, 256 bytes):    32 x { uint32 row, uint32 K | flag << 31 }    lane j at 8 j
//            row = the lane's row (0xFFFF / NO_ROW: the slice has fewer than 32 rows), K = groups of the
//            slice (the same in every lane), flag = the row is a C-point of its level (the CF smoother relaxes
//            the two classes in turn).  The l1 diagonal inverse a relaxing epilogue needs is NOT in the
//            stream: the kernel fetches it from the level's dinv array together with the other row-local
//            operands (round 1 kept it in a 16-byte header per row; the headers were 4-30 % of a stream).
//            A narrow stream has at most 65536 columns AND at most 65535 rows.
#pragma once
#include <cstdint>

namespace amgdd {

#ifndef AMGDD_RING_DEPTH
#define AMGDD_RING_DEPTH 3
#endif
#ifndef AMGDD_WAYS
#define AMGDD_WAYS 16
#endif
#ifndef AMGDD_CTAS_PER_SM
#define AMGDD_CTAS_PER_SM 1
#endif
constexpr int NUM_WAYS = AMGDD_WAYS;          // warps of an AlgFAC CTA = sub-streams per matrix
constexpr int CTAS_PER_SM = AMGDD_CTAS_PER_SM;   // resident AlgFAC CTAs per SM (each works on its own subdomain)
constexpr int SLICE_ROWS = 32;
constexpr int GROUP_STEPS = 4;
constexpr int GROUP_BYTES_NARROW = 1280;
constexpr int GROUP_BYTES_WIDE = 1536;
constexpr int HEADER_BYTES_NARROW = 128;     // 32 x uint32 { row | K << 16 | flag << 31 }
constexpr int HEADER_BYTES_WIDE = 256;       // 32 x { uint32 row, uint32 K | flag << 31 }
inline int header_bytes(bool wide) { return wide ? HEADER_BYTES_WIDE : HEADER_BYTES_NARROW; }
constexpr uint16_t NO_ROW16 = 0xFFFFu;
constexpr int NARROW_MAX_COLS = 65536;       // uint16 column indices
constexpr int NARROW_MAX_ROWS = 65535;       // uint16 row in the header word (0xFFFF: no row)
constexpr int DEFAULT_WINDOW = 256;
#ifndef AMGDD_THIN_WINDOW
#define AMGDD_THIN_WINDOW 256
#endif
constexpr int THIN_WINDOW = AMGDD_THIN_WINDOW;    // sort window of the P_l / R_l streams
constexpr int MAX_WINDOW = 1 << 20;
constexpr uint32_t NO_ROW = 0xFFFFFFFFu;
constexpr uint32_t HDR_GROUPS_MASK = 0x7FFFFFFFu;   // header info: groups of the slice; bit 31: the row's flag
constexpr int RING_DEPTH = AMGDD_RING_DEPTH;  // groups per register block = groups per burst of loads; a warp holds two blocks

inline int group_bytes(bool wide) { return wide ? GROUP_BYTES_WIDE : GROUP_BYTES_NARROW; }

struct WayDesc {           // one sub-stream (same layout as amgdd_way_t of include/amgdd.h)
    uint32_t grp_off128;   // start of the way's groups, in units of 128 bytes from the stream base
    uint32_t hdr_off128;   // start of the way's slice headers, same unit
    uint32_t ngroups;      // groups of the way
    uint32_t ngroups_real; // groups of the way's slices of the first row group (a prefix)
    uint32_t nslices;      // slices of the way
    uint32_t nslices_real; // slices of the first row group (a prefix)
    uint32_t pad_[2];
};
static_assert(sizeof(WayDesc) == 32, "WayDesc layout");

constexpr uint32_t STREAM_WIDE = 1u;         // StreamDesc::flags
constexpr uint32_t STREAM_SHARED = 4u;       // the single copy of a fully covered level: every CTA reads it, keep it in L2

struct StreamDesc {
    const char* base;      // DEVICE, 128-byte aligned
    uint32_t flags;        // STREAM_WIDE | STREAM_SHARED
    uint32_t pad_;
    WayDesc way[NUM_WAYS];
};
static_assert(sizeof(StreamDesc) == 16 + 32 * NUM_WAYS, "StreamDesc layout");

// one (subdomain, level) block; pointers are device addresses (private blob or the shared global copy)
struct DevLevel {
    int n_real;            // |D_l^p|
    int n_bar;             // |D-bar_l^p| = real + ghost
    const int* gid;        // n_bar global indices (real ascending, then ghost ascending; S7)
    const double* dinv;    // n_real
    long long voff;        // offset (doubles) of this level's vectors u|t|s|f inside a workspace slot
    StreamDesc A;          // n_bar rows: real rows complete, ghost rows restricted to real columns (A12); aux = dinv
    StreamDesc P;          // n_bar rows, columns local to level l+1 (unused on L); no aux
    StreamDesc R;          // n_bar(l+1) rows, columns local to level l (unused on L); aux = dinv of level l+1
};
static_assert(sizeof(DevLevel) % 16 == 0, "DevLevel is read with 128-bit loads");

struct DevSub {
    const int* owned;      // local indices (level 0) of the owned dofs Omega_0^p
    int n_owned;
    int pad_;
};

// ---- the static program of one subdomain (built on the host by fac_build_program) ------------
enum OpKind : uint8_t {
    OPK_BEGIN = 0,         // Alg. 2 P:475 + Alg. 4
    OPK_FIRST0 = 1,        // level 0, first AlgFAC iteration: u_0 = 0, so the first sweep is delta = D^-1 f (no matrix)
    OPK_RELAX = 2,         // one l1-Jacobi sweep on the real points (P:507-508 / P:517-518), stream A_l real rows
    OPK_AT = 3,            // w = s_l + A_l t_l on D-bar_l, stream A_l
    OPK_RESTRICT = 4,      // s_{l+1} = R_l w [+ P:511 and the first sweep of level l+1 in the first iteration]
    OPK_RECALC = 5,        // f_{l+1} -= A_{l+1} u_{l+1} + s_{l+1} [+ the first sweep of level l+1]
    OPK_INTERP = 6,        // u_l += P_l u_{l+1} on D-bar_l
    OPK_COARSE = 7,        // u_L = A_L^-1 f_L
    OPK_END = 8            // Alg. 2
};
constexpr uint8_t OPF_FIRST = 1;      // first AlgFAC iteration of the cycle
constexpr uint8_t OPF_TSMEM = 2;      // the shared-memory output is t (the gather vector of the A t step), else u
constexpr uint8_t OPF_COARSEST = 4;   // RESTRICT / RECALC whose target level is L: no relaxation follows
constexpr uint8_t OPF_HALF_C = 8;     // CF smoother: this relaxation step updates the C-points only
constexpr uint8_t OPF_HALF_F = 16;    // ... the F-points only
constexpr uint8_t OPF_CF = 32;        // CF smoother: a fused first sweep (u = 0) is its C half only, the F half follows as a step

struct FacOp {
    uint8_t kind;          // OpKind
    uint8_t level;         // l of the step as written in Alg. 4 (RESTRICT: R_l; RECALC: A_{l+1} has level = l+1; INTERP: P_l)
    uint8_t gbuf;          // shared-memory vector buffer (0/1) the mat-vec gathers from; it writes the other
    uint8_t flags;         // OPF_*
    int16_t next_mat;      // index of the next mat-vec op of the program (-1: none): its first groups and header are prefetched
    int16_t pad_;
};
static_assert(sizeof(FacOp) == 8, "FacOp layout");
constexpr int MAX_OPS = 1024;

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
    long long xg_off;          // offset of the two global vector buffers (x_cap_global doubles each) inside a slot, or -1
    int* work_counter;
    const FacOp* ops;          // DEVICE, nops entries
    int nops;
    const double* lu;          // dense LU of A_L, column-major, unit lower
    const int* rowperm;
    int nL;
    const int8_t* cf0;         // C/F flags of level 0 (global numbering), for the matrix-free first sweep of the CF smoother
    int x_cap;                 // doubles in each of the two shared-memory vector buffers (0: vectors in global memory)
    long long* prof;           // optional: gridDim.x * FAC_PROF_SLOTS cycle counters (debugging), or nullptr
    int prof_smem_off;         // byte offset of the profiling counters in dynamic shared memory (PROF_SMEM_BYTES), with prof != nullptr
    long long* prof_ops;       // optional: gridDim.x * PROF_OPS_STRIDE: per step of the program: cycles | barrier wait after it | waits for ring blocks | waits for staged slice operands
};
constexpr int FAC_PROF_SLOTS = 16;
constexpr int PROF_OPS_STRIDE = 4 * MAX_OPS;
constexpr int PROF_OPS_SMEM = 256;           // steps of the program that the per-step counters cover (they live in shared memory)
constexpr int PROF_SMEM_BYTES = (FAC_PROF_SLOTS + 4 * PROF_OPS_SMEM) * 8;

struct FacLaunch {
    int grid;
    int block;                 // 32 * NUM_WAYS
    int smem_bytes;
};

// host-side packing (amgdd_pack.cpp) ---------------------------------------------------------
struct PackPlan {
    int64_t bytes;             // total stream bytes (multiple of 128)
    int64_t bytes_real;        // groups + headers of the first row group
    WayDesc way[NUM_WAYS];
    int64_t ngroups, ngroups_real;
    int64_t nslices, nslices_real;
    int64_t padded_nnz;        // 4 * 32 * ngroups: entries stored, padding included
};
// rp: nrows+1 int32 offsets (rp[0] = 0); window: rows per sort window (multiple of 32)
// wide must be true when the matrix has more than NARROW_MAX_COLS columns or more than NARROW_MAX_ROWS rows
PackPlan plan_stream(int nrows, const int32_t* rp, bool wide, int n_real, int window);
// writes plan.bytes bytes; row_flags: nrows bytes (0/1) or nullptr
void write_stream(int nrows, const int32_t* rp, const int32_t* ci, const double* v, bool wide,
                  int n_real, int window, char* dst, const uint8_t* row_flags = nullptr);
inline bool needs_wide(long long nrows, long long ncols) { return ncols > NARROW_MAX_COLS || nrows > NARROW_MAX_ROWS; }

// the program of one subdomain: num_fac_cycles AlgFAC V(nu,nu)-cycles (Alg. 4); returns the op count
// (ops may be nullptr to count only)
int fac_build_program(int L, int nfac, int nu, int smoother, FacOp* ops);   // smoother: 0 l1-Jacobi, 1 CF l1-Jacobi
int fac_smem_bytes(int x_cap, int L, int nops);
void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream);
int fac_configure(int device, int max_smem_optin);   // sets the kernel's dynamic-smem attribute; 0 on success

}  // namespace amgdd
