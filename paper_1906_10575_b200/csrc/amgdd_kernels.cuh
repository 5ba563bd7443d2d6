// Global (whole-grid) kernels of the AMG-DD cycle (Alg. 2 P:471-473 and the residual norm).
// The AlgFAC kernel and the device data layout are in amgdd_fac.cu / amgdd_stream.hpp.
#pragma once
#include <cstdint>

namespace amgdd {

// r = b - A x and per-block partial sums of r^2 (nblk of them); A global CSR with int32 row pointers.  blk: DEVICE, nblk + 1
// row offsets of the kernel's blocks: consecutive rows, at most stream_block_rows() rows and stream_block_nnz() entries
// each (a longer row is a block of its own), built on the host once per matrix
void launch_residual(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* b,
                     const double* x, double* r, double* partial, void* stream);
int stream_block_rows();
int stream_block_nnz();
int residual_num_blocks(long long n, int lanes);
// out[0] = sqrt(sum partial[0..nb))
void launch_norm_finalize(const double* partial, int nb, double* out, void* stream);
// y = M x, M global CSR (used with M = R_l = P_l^T for Alg. 2)
void launch_spmv(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* x,
                 double* y, void* stream);

// AMG V-cycle pieces (Alg. 1): one l1-Jacobi sweep (u_in = nullptr: from u = 0); y = f - A x, y = A x or
// y += A x; dense coarse solve with the LU factors of setup (n <= 4096, one CTA)
void launch_relax(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* dinv, const double* f,
                  const double* u_in, double* u_out, const signed char* cf, int cls, void* stream);   // cf: one class of points only (CF smoother)
void launch_spmv_axpy(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* x, const double* f,
                      double* y, int accumulate, void* stream);
void launch_coarse_solve(const double* lu, const int* rowperm, int n, const double* f, double* u, void* stream);

int pick_lanes(double avg_row_nnz);

// ---- sharded cycle (NEXT 4): the same row arithmetic restricted to a list of rows, and the pack / unpack of a stage ----
// r[rows[k]] = b[rows[k]] - (A x)[rows[k]], partial sums of r^2 over the listed rows (nblocks_out blocks)
void launch_residual_rows(const int* rp, const int* ci, const double* v, const int* rows, long long nrows, const double* b,
                          const double* x, double* r, double* partial, int* nblocks_out, void* stream);
// y[rows[k]] = (M x)[rows[k]]
void launch_spmv_rows(const int* rp, const int* ci, const double* v, const int* rows, long long nrows, const double* x,
                      double* y, void* stream);
void launch_gather(const double* src, const long long* pos, long long n, double* dst, void* stream);    // dst[k] = src[pos[k]]
void launch_scatter(const double* src, const long long* pos, long long n, double* dst, void* stream);   // dst[pos[k]] = src[k]
void launch_gather32(const double* src, const int* pos, long long n, double* dst, void* stream);
void launch_scatter32(const double* src, const int* pos, long long n, double* dst, void* stream);
// out[0] = sum partial[0..nb) (no square root)
void launch_sum_finalize(const double* partial, int nb, double* out, void* stream);

}  // namespace amgdd
