// Global kernels of the AMG-DD cycle (sm_100a): fine residual + norm, restriction chain.
#include "amgdd_kernels.cuh"

#include <cuda_runtime.h>

namespace amgdd {

namespace {

// ---------------------------------------------------------------------------------------------
// global kernels (Alg. 2 P:471-473 and the residual norm)
// ---------------------------------------------------------------------------------------------
constexpr int GLOBAL_BLOCK = 256;

__global__ void __launch_bounds__(GLOBAL_BLOCK) residual_kernel(const int* __restrict__ rp, const int* __restrict__ ci,
                                                                const double* __restrict__ v, long long n, int lanes,
                                                                const double* __restrict__ b, const double* __restrict__ x,
                                                                double* __restrict__ r, double* __restrict__ partial) {
    __shared__ double red[GLOBAL_BLOCK / 32];
    const int lane = threadIdx.x & (lanes - 1);
    const long long row = (long long)blockIdx.x * (GLOBAL_BLOCK / lanes) + threadIdx.x / lanes;
    double sum = 0.0;
    if (row < n) {
        const int bgn = __ldg(rp + row), end = __ldg(rp + row + 1);
        for (int k = bgn + lane; k < end; k += lanes) sum += __ldg(v + k) * __ldg(x + __ldg(ci + k));
    }
    for (int o = lanes >> 1; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o, lanes);
    double sq = 0.0;
    if (row < n && lane == 0) {
        const double ri = b[row] - sum;
        if (r) r[row] = ri;
        sq = ri * ri;
    }
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < GLOBAL_BLOCK / 32; ++k) tot += red[k];
        partial[blockIdx.x] = tot;
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

__global__ void __launch_bounds__(GLOBAL_BLOCK) spmv_kernel(const int* __restrict__ rp, const int* __restrict__ ci,
                                                            const double* __restrict__ v, long long n, int lanes,
                                                            const double* __restrict__ x, double* __restrict__ y) {
    const int lane = threadIdx.x & (lanes - 1);
    const long long row = (long long)blockIdx.x * (GLOBAL_BLOCK / lanes) + threadIdx.x / lanes;
    double sum = 0.0;
    if (row < n) {
        const int bgn = __ldg(rp + row), end = __ldg(rp + row + 1);
        for (int k = bgn + lane; k < end; k += lanes) sum += __ldg(v + k) * __ldg(x + __ldg(ci + k));
    }
    for (int o = lanes >> 1; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o, lanes);
    if (row < n && lane == 0) y[row] = sum;
}

}  // namespace

int pick_lanes(double avg) {
    int g = 2;
    while (g < 32 && g * 2 <= avg) g *= 2;      // lanes <= avg row length < 2*lanes (at least 2)
    return g;
}

int residual_num_blocks(long long n, int lanes) {
    const int rows_per_block = GLOBAL_BLOCK / lanes;
    return (int)((n + rows_per_block - 1) / rows_per_block);
}

void launch_residual(const int* rp, const int* ci, const double* v, long long n, int lanes, const double* b,
                     const double* x, double* r, double* partial, int* nblocks_out, void* stream) {
    const int nb = residual_num_blocks(n, lanes);
    residual_kernel<<<nb, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, n, lanes, b, x, r, partial);
    if (nblocks_out) *nblocks_out = nb;
}

void launch_norm_finalize(const double* partial, int nb, double* out, void* stream) {
    norm_finalize_kernel<<<1, 1024, 0, (cudaStream_t)stream>>>(partial, nb, out);
}

void launch_spmv(const int* rp, const int* ci, const double* v, long long nrows, int lanes, const double* x,
                 double* y, void* stream) {
    if (nrows <= 0) return;
    const int nb = residual_num_blocks(nrows, lanes);
    spmv_kernel<<<nb, GLOBAL_BLOCK, 0, (cudaStream_t)stream>>>(rp, ci, v, nrows, lanes, x, y);
}

}  // namespace amgdd
