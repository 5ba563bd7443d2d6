// Device-side assembly of the composite-grid matrices (paper P:335: "a clear
// dominant cost: setting up local indices ... (primarily mapping global to local column indices for the
// matrices A_l on each level)").  The host only grows the index sets D_l^p / D-bar_l^p (breadth-first
// search, amgdd_composite.cpp); the rows of the global A_l, P_l, R_l are then cut out, renumbered and
// packed into the SELL-32 group streams (amgdd_stream.hpp) by two kernels, straight into the subdomain's
// device blob.  The streams are byte-identical to the ones the host packer writes (amgdd_pack.cpp);
// tests/test_gpu_assembly.py compares them.  Index work only: values are copied, never computed.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "amgdd_stream.hpp"

namespace amgdd {

struct DevCsr64 {               // a whole level matrix on the device, row pointers as the host keeps them
    const long long* rp;
    const int* ci;
    const double* v;
};

struct DevHierLevel {
    DevCsr64 A, P, R;           // P, R: null pointers on the coarsest level
    const double* dinv;         // l1 diagonal inverse (S8)
    const int8_t* cf;           // +1 C / -1 F; null when the level has no splitting (coarsest)
    const int* coarse_of;       // fine index -> coarse index of a C-point (null on the coarsest level)
    long long n;
};

enum AsmKind : int { ASM_A = 0, ASM_P = 1, ASM_R = 2 };

// One stream of one private (subdomain, level) block.
struct AsmJob {
    int kind;                   // AsmKind
    int level;                  // l: A_l, P_l, R_l
    int nrows;                  // rows of the stream (A, P: n_bar(l); R: n_bar(l+1))
    int nrows_first;            // rows of the first row group (A: n_real(l); P, R: nrows)
    int nr, ng;                 // |D_l^p|, ghosts of level l
    int nrc, ngc;               // the same of level l+1 (ngc = 0 and gidc = null when l+1 is fully covered)
    const int* gid;             // DEVICE: global indices of level l, real ascending then ghost ascending
    const int* gidc;            // DEVICE: the same of level l+1, or null: local index = global index
    int window;                 // sort window of the stream (<= ASM_MAX_WINDOW)
    int wide;                   // 32-bit column indices
    long long scratch_row;      // offset (ints) of this job's row scratch: len[nrows], order[nrows]
    long long scratch_slice;    // offset (AsmSlice) of its slice scratch
    char* dst;                  // DEVICE: where the stream goes (set between the two passes)
};

struct AsmSlice { uint32_t K, way, g_off, h_idx; };   // groups; way; groups / slices of the way before it

struct AsmPlan {                // what the plan pass reports per job
    WayDesc way[NUM_WAYS];
    long long bytes, bytes_real, padded_nnz, nnz;
    int dropped;                // P entries that point outside D-bar_{l+1} (A7)
    int too_long_row;           // a row with more than 65535 entries (-1: none)
    int bad_col;                // write pass: entries of a real row of A_l outside D-bar_l (eq. 1 violated; must stay 0)
    int pad_;
};

struct AsmCopy {                // gid / owned-index copies and the gather of the l1 diagonal of the real points
    const int* src;             // DEVICE ints
    int* dst;                   // DEVICE
    int n;
    int gather;                 // 1: dst is double*, dst[i] = dinv[src[i]] for i < n_gather, 0.0 behind (ghost points)
    const double* dinv;
    int n_gather;
    int pad_;
};

// ---- composite index sets on the device (S6, S7; eq. 1): breadth-first growth with bitmaps -----------------
// One CTA per subdomain.  Pass 1 (asm_sets_grow) walks the levels top down: D_l^p = points within eta of B_l^p in the graph
// of A_l, the ghost layers around it, B_{l+1}^p = coarse images of the C-points of D_l^p; membership lives in two bitmaps
// per (subdomain, level), the frontiers in a scratch of min(SET_FRONTIER_CAP, n_0) indices (a larger frontier raises `overflow` and
// the host path takes the batch).  Pass 2 (asm_sets_extract) turns the bitmaps into the ascending index lists (S7) at the
// offsets the host laid out from the sizes, sums the row lengths the layout needs, and clears the bitmaps again.
struct SetLevelOut {            // per (subdomain, level), written by pass 1 (sizes, range) and pass 2 (sums)
    int n_real, n_ghost;
    int lo_word, hi_word;       // bitmap words that hold the sets (inclusive range; hi < lo: empty)
    long long nnzA_real;        // sum of the global row lengths of A_l over D_l^p
    long long nnzA_ghost_bound; // the same over the ghost points (bound of the local ghost rows)
    long long nnzP_bound;       // sum of the global row lengths of P_l over D-bar_l^p
};
struct SetJob {
    const int* owned;           // DEVICE: Omega_0^p, global indices ascending
    int n_owned;
    int overflow;               // out: a frontier exceeded the scratch
    unsigned* bm_real;          // DEVICE scratch: bitmaps of all levels, level l at word offset bm_off[l]
    unsigned* bm_ghost;
    int* frontier;              // DEVICE scratch: 3 * frontier_cap ints
    int frontier_cap;           // capacity of each of the three index buffers: min(SET_FRONTIER_CAP, largest level size)
    SetLevelOut* out;           // DEVICE: L + 1 records
    int* const* list_dst;       // pass 2: DEVICE array of L + 1 pointers: where real | ghost of level l go (null: shared level)
    int* owned_local_dst;       // pass 2: n_owned local indices (level 0) of the owned dofs
};
constexpr int SET_FRONTIER_CAP = 1 << 18;
cudaError_t launch_sets_grow(SetJob* jobs, int njobs, const DevHierLevel* hier, const long long* bm_off, int L, int eta, int num_ghost,
                             cudaStream_t st);
cudaError_t launch_sets_extract(SetJob* jobs, int njobs, const DevHierLevel* hier, const long long* bm_off, int L, cudaStream_t st);

constexpr int ASM_MAX_WINDOW = 1024;

cudaError_t launch_asm_plan(const AsmJob* jobs, int njobs, const DevHierLevel* hier, int* row_scratch, AsmSlice* slice_scratch,
                            AsmPlan* plans, cudaStream_t st);
cudaError_t launch_asm_write(const AsmJob* jobs, int njobs, const DevHierLevel* hier, const int* row_scratch,
                             const AsmSlice* slice_scratch, AsmPlan* plans, cudaStream_t st);
cudaError_t launch_asm_copy(const AsmCopy* jobs, int njobs, cudaStream_t st);

}  // namespace amgdd
