// amgdd_residual_norm_static (include/amgdd.h): || b - A x ||_2 of a CSR matrix that already sits on the device,
// computed WITHOUT any device allocation.  Who this is for: code that must not call cudaMalloc / cudaFree where the
// norm is needed -- a solver loop inside an application whose memory pool already holds all of the GPU's memory
// (config 3 of this repository leaves under 70 GB of 180 free, a framework's caching allocator may leave nothing), or
// a latency-critical loop that cannot afford the device-wide synchronisation cudaFree implies.  The handle-based
// amgdd_residual_norm needs amgdd_setup first, which allocates the whole hierarchy; this entry needs no handle.
//
// The per-CTA sums of squares (the scratch memory of the residual kernel: one double per CTA, summed in a fixed order by
// the CTA that finishes last) and the arrival counter live in g_rn_scratch below, a file-scope __device__ array of
// fixed size.  Every GPU on which this library is loaded keeps those 512.25 KiB until the process exits.
//
// Row arithmetic is the one of csr_stream_kernel<1> (amgdd_kernels.cu): products with __dmul_rn, added one by one in
// stored order with __dadd_rn, so r is bit-identical to the handle-based path; the norm can differ from it in the last
// bits (another grouping of the partial sums).
#include "../../include/amgdd.h"

#include <cuda_runtime.h>

#include <mutex>
#include <string>

namespace amgdd {
void set_error_detail(const std::string& s);    // amgdd_api.cu: the thread-local string behind amgdd_last_error_detail
}

namespace {

constexpr int RN_BLOCK = 256;                                // threads of a CTA = rows of a CTA
constexpr int RN_CHUNK = 2304;                               // products that wait in shared memory per pass
constexpr int RN_MAX_BLOCKS = AMGDD_STATIC_MAX_ROWS / RN_BLOCK;
static_assert(AMGDD_STATIC_MAX_ROWS % RN_BLOCK == 0, "the row limit is a whole number of CTAs");
constexpr int RN_COUNTER_SLOT = RN_MAX_BLOCKS;               // the arrival counter sits behind the partial sums

// [0, RN_MAX_BLOCKS): sum of r_i^2 of CTA k;  [RN_COUNTER_SLOT]: CTAs that have stored their sum (as unsigned int).
// In HOST code this name is only a stand-in for the symbol: its device address comes from cudaGetSymbolAddress
// (scratch_of_current_device below); handing &g_rn_scratch to a kernel from host code would pass a host address.
static __device__ __align__(256) double g_rn_scratch[RN_MAX_BLOCKS + 32];

__global__ void __launch_bounds__(RN_BLOCK) residual_norm_static_kernel(const long long* __restrict__ rp, const int* __restrict__ ci,
                                                                        const double* __restrict__ v, long long n,
                                                                        const double* __restrict__ b, const double* __restrict__ x,
                                                                        double* __restrict__ r, double* scratch, double* out) {
    __shared__ double prod[RN_CHUNK];
    __shared__ long long srp[RN_BLOCK + 1];
    __shared__ double red[RN_BLOCK / 32];
    __shared__ bool last;
    const long long r0 = (long long)blockIdx.x * RN_BLOCK;
    const int nr = (int)(n - r0 < RN_BLOCK ? n - r0 : RN_BLOCK);
    for (int t = threadIdx.x; t <= nr; t += RN_BLOCK) srp[t] = rp[r0 + t];
    __syncthreads();
    const long long e0 = srp[0], e1 = srp[nr];
    const bool have_row = (int)threadIdx.x < nr;
    const long long rs = have_row ? srp[threadIdx.x] : 0, re = have_row ? srp[threadIdx.x + 1] : 0;
    double sum = 0.0;
    // the CTA's entries in passes of RN_CHUNK: coalesced loads, products to shared memory, then every thread adds the
    // products of ITS row that fall into the pass -- passes ascend, so a row is summed in stored order whatever its length
    for (long long c0 = e0; c0 < e1; c0 += RN_CHUNK) {
        const long long c1 = c0 + RN_CHUNK < e1 ? c0 + RN_CHUNK : e1;
        for (long long e = c0 + threadIdx.x; e < c1; e += RN_BLOCK) prod[e - c0] = __dmul_rn(__ldg(v + e), __ldg(x + __ldg(ci + e)));
        __syncthreads();
        const long long k0 = rs > c0 ? rs : c0, k1 = re < c1 ? re : c1;
        for (long long k = k0; k < k1; ++k) sum = __dadd_rn(sum, prod[k - c0]);
        __syncthreads();
    }
    double sq = 0.0;
    if (have_row) {
        const double ri = b[r0 + threadIdx.x] - sum;
        if (r) r[r0 + threadIdx.x] = ri;
        sq = ri * ri;
    }
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_down_sync(0xffffffffu, sq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    unsigned int* arrived = reinterpret_cast<unsigned int*>(scratch + RN_COUNTER_SLOT);
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < RN_BLOCK / 32; ++k) tot += red[k];
        scratch[blockIdx.x] = tot;
        __threadfence();                                       // the sum is visible before the arrival is
        last = atomicAdd(arrived, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    // the CTA that arrives last adds the gridDim.x sums in a fixed order (deterministic whichever CTA it is); only
    // entries written by THIS launch are read, so what an earlier call left behind them does not matter
    __threadfence();
    double s = 0.0;
    for (unsigned int i = threadIdx.x; i < gridDim.x; i += RN_BLOCK) s += __ldcg(scratch + i);
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        for (int k = 0; k < RN_BLOCK / 32; ++k) tot += red[k];
        out[0] = sqrt(tot);
        *arrived = 0u;                                         // left at zero for the next call (the host clears it as well)
    }
}

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch_dev[MAX_DEVICES] = {};    // device address of g_rn_scratch on device d, once looked up

// Device address of the scratch array on the calling thread's current device; the first call on a device asks the
// runtime for it (cudaGetSymbolAddress may load the module there: not something to do while a stream is capturing).
int scratch_of_current_device(double** p) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { amgdd::set_error_detail(std::string("cudaGetDevice: ") + cudaGetErrorString(e)); return AMGDD_ERR_CUDA; }
    if (dev < 0 || dev >= MAX_DEVICES) { amgdd::set_error_detail("device ordinal " + std::to_string(dev) + " is beyond the 64 this entry point keeps track of"); return AMGDD_ERR_BAD_ARG; }
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_dev[dev]) {
        void* sym = nullptr;
        e = cudaGetSymbolAddress(&sym, g_rn_scratch);
        if (e != cudaSuccess || !sym) {
            amgdd::set_error_detail(std::string("cudaGetSymbolAddress(g_rn_scratch) on device ") + std::to_string(dev) + ": " + cudaGetErrorString(e));
            return AMGDD_ERR_CUDA;
        }
        g_scratch_dev[dev] = static_cast<double*>(sym);
    }
    *p = g_scratch_dev[dev];
    return AMGDD_SUCCESS;
}

}  // namespace

extern "C" int amgdd_residual_norm_static(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* b,
                                          const double* x, double* r, double* out_norm, void* cuda_stream) {
    if (n <= 0) { amgdd::set_error_detail("n must be positive"); return AMGDD_ERR_BAD_ARG; }
    if (!rowptr || !colind || !vals || !b || !x || !out_norm) { amgdd::set_error_detail("null pointer argument"); return AMGDD_ERR_BAD_ARG; }
    if (n > (int64_t)AMGDD_STATIC_MAX_ROWS) {
        amgdd::set_error_detail("amgdd_residual_norm_static: n = " + std::to_string(n) + " rows exceed AMGDD_STATIC_MAX_ROWS = " +
                                std::to_string((long long)AMGDD_STATIC_MAX_ROWS) + " (the fixed scratch array holds one partial sum per 256 rows); use amgdd_residual_norm");
        return AMGDD_ERR_BAD_ARG;
    }
    double* scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != AMGDD_SUCCESS) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the arrival counter must start at zero even if an earlier launch died half way (a memset node, no allocation)
    cudaError_t e = cudaMemsetAsync(scratch + RN_COUNTER_SLOT, 0, sizeof(unsigned int), st);
    if (e != cudaSuccess) { amgdd::set_error_detail(std::string("cudaMemsetAsync: ") + cudaGetErrorString(e)); return AMGDD_ERR_CUDA; }
    const unsigned int nb = (unsigned int)((n + RN_BLOCK - 1) / RN_BLOCK);
    static_assert(sizeof(long long) == sizeof(int64_t), "rowptr is passed to the kernel as long long");
    residual_norm_static_kernel<<<nb, RN_BLOCK, 0, st>>>(reinterpret_cast<const long long*>(rowptr), colind, vals, (long long)n, b, x, r, scratch, out_norm);
    e = cudaGetLastError();
    if (e != cudaSuccess) { amgdd::set_error_detail(std::string("residual_norm_static_kernel launch: ") + cudaGetErrorString(e)); return AMGDD_ERR_CUDA; }
    return AMGDD_SUCCESS;
}
