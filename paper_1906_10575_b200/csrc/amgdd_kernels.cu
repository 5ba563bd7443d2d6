// Global kernels of the AMG-DD cycle (sm_100a): fine residual + norm, restriction chain.
#include "amgdd_kernels.cuh"

#include <cuda_runtime.h>

namespace amgdd {

namespace {

// ---------------------------------------------------------------------------------------------
// global kernels (Alg. 2 P:471-473 and the residual norm)
// ---------------------------------------------------------------------------------------------
constexpr int GLOBAL_BLOCK = 256;

// Row sums of the global kernels (a1, a2): the entries of a row are multiplied and added ONE BY ONE in stored order
// (__dmul_rn, __dadd_rn: no contraction), whichever kernel computes the row -- the whole-matrix "CSR stream" kernel below
// or the row-list kernel of the sharded cycle -- so a row's result does not depend on who owns it.
constexpr int STREAM_ROWS = 256;             // rows of a block of the stream kernel (one thread per row in the second phase)
constexpr int STREAM_NNZ = 2304;             // entries of a block (their products wait in shared memory)

// y = M x (MODE 0), r = b - M x with per-block sums of r^2 (MODE 1), one l1-Jacobi sweep y = x + D^-1 (b - M x) on the rows
// of one C/F class or on all rows (MODE 2; x = nullptr: from zero), y = b - M x (MODE 3) or y += M x (MODE 4) over consecutive rows.  Block k owns the rows
// [blk[k], blk[k+1]) (host-built: at most STREAM_ROWS rows and STREAM_NNZ entries; a longer row is a block of its own).
// Phase 1: all threads walk the block's contiguous entries (coalesced loads of values and columns, x gathered through
// L2) and leave the products in shared memory; phase 2: thread t adds the products of row t in order.
template <int MODE>
__global__ void __launch_bounds__(GLOBAL_BLOCK) csr_stream_kernel(const int* __restrict__ rp, const int* __restrict__ ci,
                                                                  const double* __restrict__ v, const int* __restrict__ blk,
                                                                  const double* __restrict__ x, const double* __restrict__ b,
                                                                  double* __restrict__ y, double* __restrict__ partial,
                                                                  const double* __restrict__ dinv, const signed char* __restrict__ cf, int cls) {
    __shared__ double prod[STREAM_NNZ];
    __shared__ int srp[STREAM_ROWS + 1];
    __shared__ double red[GLOBAL_BLOCK / 32];
    const int r0 = __ldg(blk + blockIdx.x), r1 = __ldg(blk + blockIdx.x + 1), n = r1 - r0;
    for (int t = threadIdx.x; t <= n; t += GLOBAL_BLOCK) srp[t] = __ldg(rp + r0 + t);
    __syncthreads();
    const int e0 = srp[0], e1 = srp[n];
    double sq = 0.0;
    auto finish = [&](int row, double sum) {
        if (MODE == 1) {
            const double ri = b[row] - sum;
            if (y) y[row] = ri;
            sq = ri * ri;
        } else if (MODE == 2) {                // CF smoother: cf != nullptr restricts the update to one class (cls > 0: C-points)
            const bool active = !cf || ((cf[row] > 0) == (cls > 0));
            y[row] = (x ? x[row] : 0.0) + (active ? dinv[row] * (b[row] - sum) : 0.0);
        } else if (MODE == 3) y[row] = b[row] - sum;
        else if (MODE == 4) y[row] = y[row] + sum;
        else y[row] = sum;
    };
    const bool have_x = MODE != 2 || x != nullptr;                      // a sweep from u = 0 needs no products
    if (e1 - e0 <= STREAM_NNZ) {
        if (have_x)
            for (int e = e0 + threadIdx.x; e < e1; e += GLOBAL_BLOCK) prod[e - e0] = __dmul_rn(__ldg(v + e), __ldg(x + __ldg(ci + e)));
        __syncthreads();
        if (threadIdx.x < n) {
            double sum = 0.0;
            if (have_x)
                for (int k = srp[threadIdx.x] - e0; k < srp[threadIdx.x + 1] - e0; ++k) sum = __dadd_rn(sum, prod[k]);
            finish(r0 + threadIdx.x, sum);
        }
    } else if (threadIdx.x == 0) {             // one row longer than a block holds: the same order, one thread
        double sum = 0.0;
        if (have_x)
            for (int e = e0; e < e1; ++e) sum = __dadd_rn(sum, __dmul_rn(__ldg(v + e), __ldg(x + __ldg(ci + e))));
        finish(r0, sum);
    }
    if (MODE == 1) {
        for (int o = 16; o > 0; o >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int k = 0; k < GLOBAL_BLOCK / 32; ++k) tot += red[k];
            partial[blockIdx.x] = tot;
        }
    }
}

// the same rows for a LIST of rows (sharded cycle: the rows a rank owns), one thread per row
template <int MODE>
__global__ void __launch_bounds__(GLOBAL_BLOCK) csr_rows_kernel(const int* __restrict__ rp, const int* __restrict__ ci,
                                                                const double* __restrict__ v, const int* __restrict__ rows, long long n,
                                                                const double* __restrict__ x, const double* __restrict__ b,
                                                                double* __restrict__ y, double* __restrict__ partial) {
    __shared__ double red[GLOBAL_BLOCK / 32];
    const long long idx = (long long)blockIdx.x * GLOBAL_BLOCK + threadIdx.x;
    double sq = 0.0;
    if (idx < n) {
        const int row = __ldg(rows + idx);
        double sum = 0.0;
        for (int k = __ldg(rp + row); k < __ldg(rp + row + 1); ++k) sum = __dadd_rn(sum, __dmul_rn(__ldg(v + k), __ldg(x + __ldg(ci + k))));
        if (MODE == 1) {
            const double ri = b[row] - sum;
            if (y) y[row] = ri;
            sq = ri * ri;
        } else y[row] = sum;
    }
    if (MODE == 1) {
        for (int o = 16; o > 0; o >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int k = 0; k < GLOBAL_BLOCK / 32; ++k) tot += red[k];
            partial[blockIdx.x] = tot;
        }
    }
}

__global__ void __launch_bounds__(1024) norm_finalize_kernel(const double* __restrict__ partial, int nb, double* out) {
    __shared__ double red[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += 1024) s += partial[i];       // fixed order: deterministic
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = red[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) out[0] = sqrt(s);
    }
}

// pack / unpack of one exchange stage of the sharded cycle (positions: 64-bit into x or the residual vector; 32-bit dof lists)
template <class I>
__global__ void __launch_bounds__(GLOBAL_BLOCK) gather_kernel(const double* __restrict__ src, const I* __restrict__ pos, long long n,
                                                              double* __restrict__ dst) {
    const long long k = (long long)blockIdx.x * GLOBAL_BLOCK + threadIdx.x;
    if (k < n) dst[k] = src[pos[k]];
}
template <class I>
__global__ void __launch_bounds__(GLOBAL_BLOCK) scatter_kernel(const double* __restrict__ src, const I* __restrict__ pos, long long n,
                                                               double* __restrict__ dst) {
    const long long k = (long long)blockIdx.x * GLOBAL_BLOCK + threadIdx.x;
    if (k < n) dst[pos[k]] = src[k];
}

__global__ void __launch_bounds__(1024) sum_finalize_kernel(const double* __restrict__ partial, int nb, double* out) {
    __shared__ double red[32];
    double s = 0.0;
    for (int i = threadIdx.x; i < nb; i += 1024) s += partial[i];       // fixed order: deterministic
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        s = red[threadIdx.x];
        for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) out[0] = s;
    }
}

// ---------------------------------------------------------------------------------------------
// AMG V-cycle on the global hierarchy (Alg. 1): the paper's comparison method
// ---------------------------------------------------------------------------------------------
// u = A_L^-1 f with the LU factors of setup (column-major, unit lower; rowperm[i] = source row of row i); one CTA
__global__ void __launch_bounds__(256) coarse_solve_kernel(const double* __restrict__ lu, const int* __restrict__ rowperm, int n,
                                                           const double* __restrict__ f, double* __restrict__ u) {
    extern __shared__ double y[];
    for (int i = threadIdx.x; i < n; i += blockDim.x) y[i] = f[rowperm[i]];
    __syncthreads();
    for (int c = 0; c < n; ++c) {                              // forward: L y = P f
        const double yc = y[c];
        for (int i = c + 1 + threadIdx.x; i < n; i += blockDim.x) y[i] -= lu[(size_t)c * n + i] * yc;
        __syncthreads();
    }
    for (int c = n - 1; c >= 0; --c) {                         // backward: U u = y
        if (threadIdx.x == 0) y[c] = y[c] / lu[(size_t)c * n + c];
        __syncthreads();
        const double yc = y[c];
        for (int i = threadIdx.x; i < c; i += blockDim.x) y[i] -= lu[(size_t)c * n + i] * yc;
        __syncthreads();
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) u[i] = y[i];
}

}  // namespace

void launch_relax(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* dinv, const double* f,
                  const double* u_in, double* u_out, const signed char* cf, int cls, void* stream) {
    if (nblk > 0) csr_stream_kernel<2><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, u_in, f, u_out, nullptr, dinv, cf, cls);
}

void launch_spmv_axpy(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* x, const double* f,
                      double* y, int accumulate, void* stream) {
    if (nblk <= 0) return;
    if (accumulate) csr_stream_kernel<4><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, x, nullptr, y, nullptr, nullptr, nullptr, 0);
    else if (f) csr_stream_kernel<3><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, x, f, y, nullptr, nullptr, nullptr, 0);
    else csr_stream_kernel<0><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, x, nullptr, y, nullptr, nullptr, nullptr, 0);
}

void launch_coarse_solve(const double* lu, const int* rowperm, int n, const double* f, double* u, void* stream) {
    coarse_solve_kernel<<<1, 256, (size_t)n * sizeof(double), (cudaStream_t)stream>>>(lu, rowperm, n, f, u);
}

int pick_lanes(double avg) {
    int g = 2;
    while (g < 32 && g * 2 <= avg) g *= 2;      // lanes <= avg row length < 2*lanes (at least 2)
    return g;
}

int residual_num_blocks(long long n, int lanes) {
    const int rows_per_block = GLOBAL_BLOCK / lanes;
    return (int)((n + rows_per_block - 1) / rows_per_block);
}

int stream_block_rows() { return STREAM_ROWS; }
int stream_block_nnz() { return STREAM_NNZ; }

void launch_residual(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* b,
                     const double* x, double* r, double* partial, void* stream) {
    if (nblk > 0) csr_stream_kernel<1><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, x, b, r, partial, nullptr, nullptr, 0);
}

void launch_residual_rows(const int* rp, const int* ci, const double* v, const int* rows, long long nrows, const double* b,
                          const double* x, double* r, double* partial, int* nblocks_out, void* stream) {
    const int nb = (int)((nrows + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK);
    if (nb > 0) csr_rows_kernel<1><<<nb, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, rows, nrows, x, b, r, partial);
    if (nblocks_out) *nblocks_out = nb;
}

void launch_spmv_rows(const int* rp, const int* ci, const double* v, const int* rows, long long nrows, const double* x,
                      double* y, void* stream) {
    if (nrows <= 0) return;
    const int nb = (int)((nrows + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK);
    csr_rows_kernel<0><<<nb, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, rows, nrows, x, nullptr, y, nullptr);
}

void launch_gather(const double* src, const long long* pos, long long n, double* dst, void* stream) {
    if (n > 0) gather_kernel<long long><<<(unsigned)((n + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK), GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(src, pos, n, dst);
}
void launch_scatter(const double* src, const long long* pos, long long n, double* dst, void* stream) {
    if (n > 0) scatter_kernel<long long><<<(unsigned)((n + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK), GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(src, pos, n, dst);
}
void launch_gather32(const double* src, const int* pos, long long n, double* dst, void* stream) {
    if (n > 0) gather_kernel<int><<<(unsigned)((n + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK), GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(src, pos, n, dst);
}
void launch_scatter32(const double* src, const int* pos, long long n, double* dst, void* stream) {
    if (n > 0) scatter_kernel<int><<<(unsigned)((n + GLOBAL_BLOCK - 1) / GLOBAL_BLOCK), GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(src, pos, n, dst);
}
void launch_sum_finalize(const double* partial, int nb, double* out, void* stream) {
    sum_finalize_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(partial, nb, out);
}

void launch_norm_finalize(const double* partial, int nb, double* out, void* stream) {
    norm_finalize_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(partial, nb, out);
}

void launch_spmv(const int* rp, const int* ci, const double* v, const int* blk, int nblk, const double* x,
                 double* y, void* stream) {
    if (nblk > 0) csr_stream_kernel<0><<<nblk, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, blk, x, nullptr, y, nullptr, nullptr, nullptr, 0);
}

}  // namespace amgdd
