// Hand-written sm_100a kernels of the AMG-DD solve phase.  See amgdd_kernels.cuh for the layout.
#include "amgdd_kernels.cuh"

#include <cuda_runtime.h>

namespace amgdd {

namespace {

// streaming loads of matrix data: read once per mat-vec, never written by the kernel
__device__ __forceinline__ int ld_stream(const int* p) { return __ldg(p); }
__device__ __forceinline__ double ld_stream(const double* p) { return __ldg(p); }

// Row-parallel CSR traversal by one CTA: `lanes` consecutive threads share a row, a warp covers
// 32/lanes consecutive rows, so the index and value streams are read contiguously.  epi(row, sum)
// runs on the first lane of the row's group.  All threads of the CTA must call this.
template <class Epi>
__device__ __forceinline__ void cta_spmv(int nrows, const int* __restrict__ rp, const int* __restrict__ ci,
                                         const double* __restrict__ v, const double* x, int lanes, Epi epi) {
    const int lane = threadIdx.x & (lanes - 1);
    const int group = threadIdx.x / lanes;
    const int ngroups = blockDim.x / lanes;
    for (int base = 0; base < nrows; base += ngroups) {
        const int row = base + group;
        double sum = 0.0;
        if (row < nrows) {
            const int b = ld_stream(rp + row), e = ld_stream(rp + row + 1);
            for (int k = b + lane; k < e; k += lanes) sum += ld_stream(v + k) * x[ld_stream(ci + k)];
        }
        for (int o = lanes >> 1; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o, lanes);
        if (row < nrows && lane == 0) epi(row, sum);
    }
}

// One l1-Jacobi sweep on the real points (paper §4.1): delta from the OLD u for
// every real row, then u += delta, t += delta (Alg. 4 P:507-508 / P:517-518).
__device__ __forceinline__ void relax_sweep(const DevLevel& d, double* u, const double* f, double* t,
                                            double* delta) {
    const double* dinv = d.dinv;
    cta_spmv(d.n_real, d.a_rp, d.a_ci, d.a_v, u, d.lanes_a,
             [&](int i, double au) { delta[i] = __ldg(dinv + i) * (f[i] - au); });
    __syncthreads();
    for (int i = threadIdx.x; i < d.n_real; i += blockDim.x) {
        const double dl = delta[i];
        u[i] += dl;
        t[i] += dl;
    }
    __syncthreads();
}

// u_L = A_L^{-1} f_L with the LU factors computed at setup (Alg. 4).  One warp, columns of
// the unit-lower / upper factors are contiguous (column-major), y lives in shared or global memory.
__device__ __forceinline__ void coarse_solve(const FacParams& prm, const double* f, double* y) {
    const int n = prm.nL;
    const double* __restrict__ lu = prm.lu;
    for (int i = threadIdx.x; i < n; i += blockDim.x) y[i] = f[__ldg(prm.rowperm + i)];
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        for (int c = 0; c < n; ++c) {                      // forward: L y = P f
            const double yc = y[c];
            for (int i = c + 1 + lane; i < n; i += 32) y[i] -= __ldg(lu + (size_t)c * n + i) * yc;
            __syncwarp();
        }
        for (int c = n - 1; c >= 0; --c) {                 // backward: U u = y
            if (lane == 0) y[c] = y[c] / __ldg(lu + (size_t)c * n + c);
            __syncwarp();
            const double yc = y[c];
            for (int i = lane; i < c; i += 32) y[i] -= __ldg(lu + (size_t)c * n + i) * yc;
            __syncwarp();
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(512) fac_kernel(const FacParams prm) {
    __shared__ int s_p;
    const int L = prm.L;
    double* ws = prm.workspace + (size_t)blockIdx.x * prm.slot_stride;
    double* w = ws + prm.scratch_off;                      // scratch: s_l + A_l t_l
    double* delta = w + prm.scratch_len;                   // scratch: relaxation update
    const int tid = threadIdx.x, nt = blockDim.x;

    for (;;) {
        if (tid == 0) s_p = atomicAdd(prm.work_counter, 1);
        __syncthreads();
        const int q = s_p;
        __syncthreads();
        if (q >= prm.num_sub) break;
        const int p = prm.order[q];
        const DevLevel* lev = prm.lev + (size_t)p * (L + 1);

        // vectors of level l inside the slot: u | t | s | f, each n_bar long
        auto U = [&](int l) { return ws + lev[l].voff; };
        auto T = [&](int l) { return ws + lev[l].voff + lev[l].n_bar; };
        auto S = [&](int l) { return ws + lev[l].voff + 2 * (size_t)lev[l].n_bar; };
        auto F = [&](int l) { return ws + lev[l].voff + 3 * (size_t)lev[l].n_bar; };

        // ---- Alg. 2 P:475 + Alg. 4: f_l = r_l on D_l ; u = t = s = 0 ----
        for (int l = 0; l <= L; ++l) {
            const DevLevel d = lev[l];
            const double* r = prm.r_all + prm.r_off[l];
            double* u = U(l);
            for (int i = tid; i < 3 * d.n_bar; i += nt) u[i] = 0.0;
            double* f = F(l);
            for (int i = tid; i < d.n_real; i += nt) f[i] = r[__ldg(d.gid + i)];
        }
        __syncthreads();

        for (int it = 0; it < prm.nfac; ++it) {
            // ------------------------------ downsweep ------------------------------
            for (int l = 0; l < L; ++l) {
                const DevLevel d = lev[l];
                const DevLevel c = lev[l + 1];
                double *u = U(l), *t = T(l), *s = S(l), *f = F(l);
                int sweeps = prm.nu;
                if (l != 0) {
                    // P:506 u_l <- 0, then the first sweep needs no matrix: delta = D^{-1} f
                    for (int i = tid; i < d.n_bar; i += nt) {
                        double dl = 0.0;
                        if (i < d.n_real) { dl = __ldg(d.dinv + i) * f[i]; t[i] += dl; }
                        u[i] = dl;
                    }
                    __syncthreads();
                    --sweeps;
                }
                for (int k = 0; k < sweeps; ++k) relax_sweep(d, u, f, t, delta);
                // P:509  w = s_l + A_l t_l on all of D-bar_l (ghost rows: real columns only)
                cta_spmv(d.n_bar, d.a_rp, d.a_ci, d.a_v, t, d.lanes_a, [&](int i, double at) { w[i] = s[i] + at; });
                __syncthreads();
                // P:509  s_{l+1} = R_l w ; P:512 reset t_l, s_l
                double *sc = S(l + 1), *fc = F(l + 1), *uc = U(l + 1);
                cta_spmv(c.n_bar, d.r_rp, d.r_ci, d.r_v, w, d.lanes_r, [&](int I, double rw) { sc[I] = rw; });
                for (int i = tid; i < 2 * d.n_bar; i += nt) t[i] = 0.0;      // t and s are adjacent
                __syncthreads();
                // P:510-511  f_{l+1} <- f_{l+1} - A_{l+1} u_{l+1} - s_{l+1}  (u_{l+1} of the previous
                // iteration; identically zero in the first one)
                if (it > 0) {
                    cta_spmv(c.n_real, c.a_rp, c.a_ci, c.a_v, uc, c.lanes_a,
                             [&](int I, double au) { fc[I] = (fc[I] - au) - sc[I]; });
                } else {
                    for (int I = tid; I < c.n_real; I += nt) fc[I] -= sc[I];
                }
                __syncthreads();
            }
            // ------------------------------ coarse solve -------------------------------
            coarse_solve(prm, F(L), U(L));
            // ------------------------------ upsweep --------------------------------
            for (int l = L - 1; l >= 0; --l) {
                const DevLevel d = lev[l];
                double *u = U(l), *t = T(l), *f = F(l);
                const double* uc = U(l + 1);
                cta_spmv(d.n_bar, d.p_rp, d.p_ci, d.p_v, uc, d.lanes_p, [&](int i, double pu) { u[i] += pu; });
                __syncthreads();
                for (int k = 0; k < prm.nu; ++k) relax_sweep(d, u, f, t, delta);
            }
        }
        // ---- Alg. 2: x <- x + u_0^p on Omega_0^p (disjoint targets across subdomains) ----
        {
            const DevSub sb = prm.sub[p];
            const double* u0 = U(0);
            const int* gid0 = lev[0].gid;
            for (int k = tid; k < sb.n_owned; k += nt) {
                const int li = __ldg(sb.owned + k);
                prm.x[__ldg(gid0 + li)] += u0[li];
            }
        }
        __syncthreads();
    }
}

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

void launch_fac(const FacParams& prm, int grid, int block, void* stream) {
    fac_kernel<<<grid, block, 0, (cudaStream_t)stream>>>(prm);
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
