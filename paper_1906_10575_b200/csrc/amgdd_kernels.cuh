// Device-side data layout and kernels of the AMG-DD solve phase (sm_100a).
//
// One persistent CTA per resident slot; each CTA takes whole subdomains from a work counter and
// runs ALL num_fac_cycles AlgFAC V(nu,nu)-cycles of that subdomain (Alg. 4) start to
// finish: gather of the restricted residuals (Alg. 2), every level's relax / A t /
// restrict / recalculate / interpolate step, the dense coarse solve, and the owned-dof update
// (P:479).  Subdomains never communicate, so the only synchronisation is __syncthreads.
// The level vectors u, f, t, s live in a per-slot workspace that is reused by every subdomain
// the slot processes, so they stay in L1/L2 and never stream from HBM; what streams from HBM is
// the matrix data (values, column indices, row pointers), read exactly once per mat-vec.
#pragma once
#include <cstdint>

namespace amgdd {

// one (subdomain, level) block; pointers are device addresses (private blob or the shared global copy)
struct DevLevel {
    int n_real;            // |D_l^p|
    int n_bar;             // |D-bar_l^p| = real + ghost
    int lanes_a;           // threads cooperating on one row of A / P / R (power of two, <= 32)
    int lanes_p;
    int lanes_r;
    int pad_;
    const int* gid;        // n_bar global indices (real ascending, then ghost ascending; S7)
    const double* dinv;    // n_real
    const int* a_rp;       // n_bar + 1
    const int* a_ci;
    const double* a_v;
    const int* p_rp;       // n_bar + 1, columns local to level l+1 (unused on L)
    const int* p_ci;
    const double* p_v;
    const int* r_rp;       // n_bar(l+1) + 1, columns local to level l (unused on L)
    const int* r_ci;
    const double* r_v;
    long long voff;        // offset (doubles) of this level's vectors inside a workspace slot
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
    double* workspace;         // num_slots * slot_stride doubles
    long long slot_stride;
    long long scratch_off;     // offset of the two scratch vectors (w, delta) inside a slot
    long long scratch_len;     // length of one scratch vector
    int* work_counter;
    int nfac;
    int nu;
    const double* lu;          // dense LU of A_L, column-major, unit lower
    const int* rowperm;
    int nL;
};

void launch_fac(const FacParams& prm, int grid, int block, void* stream);

// r = b - A x and per-block partial sums of r^2; A global CSR with int32 row pointers
void launch_residual(const int* rp, const int* ci, const double* v, long long n, int lanes, const double* b,
                     const double* x, double* r, double* partial, int* nblocks_out, void* stream);
int residual_num_blocks(long long n, int lanes);
// out[0] = sqrt(sum partial[0..nb))
void launch_norm_finalize(const double* partial, int nb, double* out, void* stream);
// y = M x, M global CSR (used with M = R_l = P_l^T for Alg. 2)
void launch_spmv(const int* rp, const int* ci, const double* v, long long nrows, int lanes, const double* x,
                 double* y, void* stream);

int pick_lanes(double avg_row_nnz);

}  // namespace amgdd
