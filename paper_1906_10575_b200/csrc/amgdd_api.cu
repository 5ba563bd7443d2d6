// C ABI of the AMG-DD library (include/amgdd.h): setup orchestration (host hierarchy, threaded
// composite-grid construction streamed to the device), the solve driver, introspection.
#include "../../include/amgdd.h"
#include "amgdd_assemble.cuh"
#include "amgdd_host.hpp"
#include "amgdd_kernels.cuh"
#include "amgdd_stream.hpp"

#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <mutex>
#include <new>
#include <numeric>
#include <string>

using namespace amgdd;

namespace {

thread_local std::string g_detail;

struct GlobalLevelDev {          // the single device copy of a whole level
    // plain CSR (int32 row pointers) for the global kernels: A_0 (Alg. 2) and every R_l
    int* a_rp = nullptr; int* a_ci = nullptr; double* a_v = nullptr;
    int* r_rp = nullptr; int* r_ci = nullptr; double* r_v = nullptr;
    int lanes_a = 2, lanes_r = 2;
    // row blocks of the CSR stream kernel (amgdd_kernels.cuh) for A_0 and R_l
    int* a_blk = nullptr; int a_nblk = 0;
    int* r_blk = nullptr; int r_nblk = 0;
    // packed streams for the AlgFAC kernel, present when some subdomain covers the whole level
    char* sA = nullptr; char* sP = nullptr; char* sR = nullptr;
    StreamLayout layA, layP, layR;
    double* dinv = nullptr; int* ident = nullptr;
    // AMG V-cycle (amgdd_vcycle; uploaded on first use): A_l and P_l as plain CSR, the l1 diagonal, level vectors
    int* p_rp = nullptr; int* p_ci = nullptr; double* p_v = nullptr;
    int lanes_p = 2;
    int* p_blk = nullptr; int p_nblk = 0;
    double* vdinv = nullptr; double *vu0 = nullptr, *vu1 = nullptr, *vf = nullptr, *vr = nullptr;
    int8_t* vcf = nullptr;
};

struct SubMeta {                 // host-side record of one subdomain's blob
    SubdomainBlob plan;
    char* dev_base = nullptr;
};

}  // namespace

namespace amgdd {
// for entry points in other translation units (amgdd_static.cu): the string amgdd_last_error_detail returns
void set_error_detail(const std::string& s) { g_detail = s; }
}  // namespace amgdd

struct amgdd_shard_plan_s {                     // a plan on its own (host only: amgdd_shard_plan_create) or the one of a handle
    std::unique_ptr<Hierarchy> H;
    std::unique_ptr<ShardPlan> own;
    ShardPlan* S = nullptr;
};

struct amgdd_handle_s {
    Hierarchy H;
    int P = 0, eta = 0, nghost = 1;
    i64 n = 0;
    int device = 0;
    cudaStream_t stream = nullptr;
    std::vector<SubMeta> subs;
    std::vector<GlobalLevelDev> glev;
    std::vector<void*> allocs;                  // every cudaMalloc the handle owns
    i64 device_bytes = 0;
    // tables
    DevLevel* d_lev = nullptr;
    DevSub* d_sub = nullptr;
    int* d_order = nullptr;
    double* d_r_all = nullptr;
    long long* d_r_off = nullptr;
    std::vector<long long> r_off;
    double* d_workspace = nullptr;
    long long slot_stride = 0, xg_off = -1, x_need = 0;
    int window = DEFAULT_WINDOW, x_cap = 0, smem_cta = 0;
    FacLaunch fac_cfg = {1, 32 * NUM_WAYS, 0};
    FacOp* d_ops = nullptr;                     // the program of one subdomain (fac_build_program)
    int prof_smem_off = 0;
    int prog_nfac = -1, prog_nu = -1, prog_smoother = -1, prog_nops = 0;
    int* d_counter = nullptr;
    long long* d_prof_ops = nullptr;
    long long* d_prof = nullptr;                // AMGDD_FAC_PROFILE=1: per-CTA cycle counters of the AlgFAC kernel
    double* d_lu = nullptr; int* d_rowperm = nullptr;
    int8_t* d_cf0 = nullptr;                    // C/F flags of level 0
    int smoother = 0;                           // 0: l1-Jacobi, 1: CF l1-Jacobi (amgdd_set_smoother)
    double* d_partial = nullptr; int partial_cap = 0;
    double* d_norms = nullptr; int norms_cap = 0;
    double* d_b_stage = nullptr; double* d_x_stage = nullptr;   // for amgdd_solve_host
    std::vector<cudaEvent_t> events;                            // phase timers of amgdd_solve, created once and reused
    amgdd_stats_t stats;
    double prof_ms[4] = {0, 0, 0, 0};
    long long prof_launches[3] = {0, 0, 0};
    std::string detail;
    bool vcycle_ready = false;
    // sharding over ranks (NEXT 4): this handle holds the subdomains [sub_lo, sub_lo + P) of P_global
    int P_global = 0, sub_lo = 0;
    std::unique_ptr<ShardPlan> shard;
    std::unique_ptr<struct amgdd_shard_plan_s> shard_view;       // what amgdd_get_shard_plan hands out (borrows `shard`)
    struct StageDev {                            // one exchange stage on the device (amgdd_shard_commit)
        long long* send_pos = nullptr; long long* recv_pos = nullptr;
        long long nsend = 0, nrecv = 0;
        std::vector<long long> send_counts, recv_counts;
    };
    std::vector<StageDev> stage_dev;
    std::vector<int*> d_owned_rows;              // per level: the rows this rank owns
    int* d_owned0_all = nullptr;                 // level 0: the dofs of every rank, rank after rank
    std::vector<long long> owned0_off;           // nranks + 1 offsets into d_owned0_all
    double* d_sq = nullptr;                      // sum of r_0^2 over the owned rows (amgdd_shard_sqnorm)
    // one AMG-DD cycle captured as a CUDA graph (asynchronous amgdd_solve calls: 4 + L launches become one)
    cudaGraphExec_t cycle_graph = nullptr;
    cudaStream_t capture_stream = nullptr;
    const double* graph_b = nullptr; double* graph_x = nullptr;
    int graph_nfac = -1, graph_nu = -1, graph_smoother = -1, graph_nops = -1;
    bool graph_off = false;
    bool shard_committed = false;
};


namespace {

#define CUDA_TRY(expr)                                                                    \
    do {                                                                                  \
        cudaError_t e__ = (expr);                                                         \
        if (e__ != cudaSuccess) {                                                         \
            g_detail = std::string(#expr) + ": " + cudaGetErrorString(e__);               \
            return e__ == cudaErrorMemoryAllocation ? AMGDD_ERR_OUT_OF_MEMORY : AMGDD_ERR_CUDA; \
        }                                                                                 \
    } while (0)

int dev_alloc(amgdd_handle_s* h, void** p, size_t bytes) {
    if (bytes == 0) bytes = 16;
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) {
        g_detail = "cudaMalloc of " + std::to_string(bytes) + " bytes failed (" + std::to_string(h->device_bytes) +
                   " bytes already held): " + cudaGetErrorString(e);
        cudaGetLastError();
        return AMGDD_ERR_OUT_OF_MEMORY;
    }
    h->allocs.push_back(*p);
    h->device_bytes += (i64)bytes;
    return AMGDD_SUCCESS;
}

template <class T>
int upload(amgdd_handle_s* h, T** dptr, const T* src, size_t count) {
    int rc = dev_alloc(h, (void**)dptr, count * sizeof(T));
    if (rc) return rc;
    if (count) CUDA_TRY(cudaMemcpy(*dptr, src, count * sizeof(T), cudaMemcpyHostToDevice));
    return AMGDD_SUCCESS;
}

int upload_csr32(amgdd_handle_s* h, const HostCsr& M, int** rp, int** ci, double** v) {
    if (M.nnz() > (i64)INT32_MAX) { g_detail = "a level matrix has more than 2^31-1 nonzeros"; return AMGDD_ERR_INDEX_RANGE; }
    std::vector<int> rp32(M.rp.begin(), M.rp.end());
    int rc = upload(h, rp, rp32.data(), rp32.size());
    if (rc) return rc;
    if ((rc = upload(h, ci, M.ci.data(), M.ci.size()))) return rc;
    return upload(h, v, M.v.data(), M.v.size());
}

double avg_row(const HostCsr& M) { return M.nrows ? (double)M.nnz() / (double)M.nrows : 1.0; }

// blocks of consecutive rows for the CSR stream kernel: at most stream_block_rows() rows and stream_block_nnz() entries
// (a row longer than that is a block of its own); returns the nblk + 1 row offsets
std::vector<int> stream_row_blocks(const HostCsr& M) {
    const i64 max_rows = stream_block_rows(), max_nnz = stream_block_nnz();
    std::vector<int> blk(1, 0);
    i64 r = 0;
    while (r < M.nrows) {
        i64 e = r;
        while (e < M.nrows && e - r < max_rows && M.rp[e + 1] - M.rp[r] <= max_nnz) ++e;
        if (e == r) e = r + 1;
        blk.push_back((int)e);
        r = e;
    }
    return blk;
}

void free_handle(amgdd_handle_s* h) {
    if (!h) return;
    for (void* p : h->allocs) cudaFree(p);
    for (cudaEvent_t e : h->events) cudaEventDestroy(e);
    if (h->cycle_graph) cudaGraphExecDestroy(h->cycle_graph);
    if (h->capture_stream) cudaStreamDestroy(h->capture_stream);
    delete h;
}

// ------------------------------------------------------------------------------------------
// composite grids: worker threads plan + fill blobs into pinned staging and copy them into a
// chunked device arena (SURVEY.md §7 hard part 2: stream, never hold everything on the host)
// ------------------------------------------------------------------------------------------
struct Arena {
    std::mutex mu;
    char* cur = nullptr;
    size_t left = 0;
    size_t chunk = (size_t)1 << 30;
};

int env_int(const char* name, int dflt) {
    const char* v = std::getenv(name);
    if (!v || !*v) return dflt;
    return std::atoi(v);
}

// reserves `bytes` of the chunked device arena (thread-safe); chunks are owned by the handle
int arena_take(amgdd_handle_s* h, Arena& arena, size_t bytes, char** out, std::string& why) {
    std::lock_guard<std::mutex> g(arena.mu);
    if (arena.left < bytes) {
        const size_t want = std::max(arena.chunk, bytes);
        void* ptr = nullptr;
        cudaError_t e = cudaMalloc(&ptr, want);
        if (e != cudaSuccess) {
            cudaGetLastError();
            why = "device arena: cudaMalloc of " + std::to_string(want) + " bytes failed with " + std::to_string(h->device_bytes) +
                  " bytes already held";
            return AMGDD_ERR_OUT_OF_MEMORY;
        }
        h->allocs.push_back(ptr);
        h->device_bytes += (i64)want;
        arena.cur = (char*)ptr;
        arena.left = want;
    }
    *out = arena.cur;
    const size_t adv = (bytes + 255) & ~(size_t)255;
    arena.cur += std::min(adv, arena.left);
    arena.left -= std::min(adv, arena.left);
    return AMGDD_SUCCESS;
}

int build_composites(amgdd_handle_s* h, const std::vector<i32>& owner, int nthreads) {
    const int P = h->P, L = h->H.L;
    std::vector<std::vector<i32>> owned(P);
    for (i64 i = 0; i < h->n; ++i) if (owner[i] >= 0) owned[owner[i]].push_back((i32)i);      // (-1: a subdomain of another rank)
    h->subs.assign(P, SubMeta());
    Arena arena;
    std::atomic<int> status(AMGDD_SUCCESS);
    std::string fail_detail;
    std::mutex fail_mu;
    auto fail = [&](int code, const std::string& d) {
        std::lock_guard<std::mutex> g(fail_mu);
        if (status.load() == AMGDD_SUCCESS) { status.store(code); fail_detail = d; }
    };
    const int dev = h->device;
    const int nw = std::max(1, std::min(nthreads, P));
    std::atomic<int> next(0);
    run_threads(nw, [&](int) {
        try {
            if (cudaSetDevice(dev) != cudaSuccess) { fail(AMGDD_ERR_CUDA, "cudaSetDevice failed in a setup worker"); return; }
            cudaStream_t st;
            if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) { fail(AMGDD_ERR_CUDA, "stream create failed"); return; }
            char* stage = nullptr;
            size_t stage_cap = 0;
            CompositeBuilder cb(h->H, owner, owned, h->eta, h->nghost, h->window);
            for (;;) {
                const int p = next.fetch_add(1);
                if (p >= P || status.load() != AMGDD_SUCCESS) break;
                SubMeta& sm = h->subs[p];
                cb.plan(p, sm.plan);
                if (sm.plan.dropped > 0) {
                    fail(AMGDD_ERR_NOT_CONNECTED_UPWARD, "subdomain " + std::to_string(p) + ": " + std::to_string(sm.plan.dropped) +
                                                             " interpolation entries of composite rows fall outside D-bar_{l+1}");
                    break;
                }
                bool too_big = false;
                for (int l = 0; l <= L; ++l)
                    if (sm.plan.lev[l].nnzA > INT32_MAX || sm.plan.lev[l].nnzP > INT32_MAX) too_big = true;
                if (too_big) { fail(AMGDD_ERR_INDEX_RANGE, "a composite level exceeds 2^31-1 local nonzeros"); break; }
                if (sm.plan.too_long_row >= 0) {
                    fail(AMGDD_ERR_INDEX_RANGE, "subdomain " + std::to_string(p) + ", level " + std::to_string(sm.plan.too_long_level) +
                                                    ": a local matrix row has more than 65535 entries");
                    break;
                }
                const size_t bytes = (size_t)std::max<i64>(sm.plan.bytes, 16);
                {
                    std::string why;
                    const int arc = arena_take(h, arena, bytes, &sm.dev_base, why);
                    if (arc) { fail(arc, why); break; }
                }
                cudaStreamSynchronize(st);                         // previous copy out of `stage` finished
                if (stage_cap < bytes) {
                    if (stage) cudaFreeHost(stage);
                    stage_cap = bytes + bytes / 4;
                    if (cudaHostAlloc((void**)&stage, stage_cap, cudaHostAllocDefault) != cudaSuccess) {
                        cudaGetLastError();
                        stage = nullptr;
                        fail(AMGDD_ERR_OUT_OF_MEMORY, "pinned staging buffer of " + std::to_string(stage_cap) + " bytes failed");
                        break;
                    }
                }
                cb.fill(sm.plan, stage);
                if (cudaMemcpyAsync(sm.dev_base, stage, (size_t)sm.plan.bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) {
                    fail(AMGDD_ERR_CUDA, "blob upload failed");
                    break;
                }
            }
            cudaStreamSynchronize(st);
            if (stage) cudaFreeHost(stage);
            cudaStreamDestroy(st);
        } catch (const std::bad_alloc&) { fail(AMGDD_ERR_OUT_OF_MEMORY, "host allocation failed in a setup worker"); }
        catch (const std::exception& e) { fail(AMGDD_ERR_OUT_OF_MEMORY, std::string("setup worker failed: ") + e.what()); }
    });
    if (status.load() != AMGDD_SUCCESS) { g_detail = fail_detail; return status.load(); }
    return AMGDD_SUCCESS;
}

// ------------------------------------------------------------------------------------------
// Device-side assembly (NEXT 3, paper P:335): the host grows the index sets only; the local
// matrices are cut out of the global level matrices, renumbered and packed on the device
// (amgdd_assemble.cu), batch by batch, straight into the arena.  Same blobs, byte for byte, as
// build_composites writes.
// ------------------------------------------------------------------------------------------
struct TempDev {                                    // device / pinned scratch that lives only during setup
    std::vector<void*> dev, pinned;
    ~TempDev() { for (void* p : dev) cudaFree(p); for (void* p : pinned) cudaFreeHost(p); }
    template <class T> cudaError_t alloc(T** p, size_t count) {
        cudaError_t e = cudaMalloc((void**)p, std::max<size_t>(count, 1) * sizeof(T));
        if (e == cudaSuccess) dev.push_back(*p);
        return e;
    }
    template <class T> cudaError_t put(T** p, const T* src, size_t count) {
        cudaError_t e = alloc(p, count);
        if (e == cudaSuccess && count) e = cudaMemcpy(*p, src, count * sizeof(T), cudaMemcpyHostToDevice);
        return e;
    }
};

template <class T>
struct GrowBuf {                                    // a device array that is re-allocated when a batch needs more
    T* p = nullptr; size_t cap = 0;
    cudaError_t need(size_t n) {
        if (n <= cap) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        const size_t want = n + n / 4 + 1024;
        cudaError_t e = cudaMalloc((void**)&p, want * sizeof(T));
        if (e == cudaSuccess) cap = want;
        return e;
    }
    ~GrowBuf() { if (p) cudaFree(p); }
};

int build_composites_device(amgdd_handle_s* h, const std::vector<i32>& owner, int nthreads) {
    const int P = h->P, L = h->H.L;
    std::vector<std::vector<i32>> owned(P);
    for (i64 i = 0; i < h->n; ++i) if (owner[i] >= 0) owned[owner[i]].push_back((i32)i);      // (-1: a subdomain of another rank)
    h->subs.assign(P, SubMeta());
    auto tA = std::chrono::steady_clock::now();
    // the hierarchy on the device, for the duration of the assembly
    TempDev tmp;
    std::vector<DevHierLevel> hier(L + 1);
    auto put_csr = [&](const HostCsr& M, DevCsr64& d) -> cudaError_t {
        static_assert(sizeof(long long) == sizeof(i64), "row pointers are uploaded as they are");
        long long* rp = nullptr; int* ci = nullptr; double* v = nullptr;
        cudaError_t e = tmp.put(&rp, (const long long*)M.rp.data(), M.rp.size());
        if (e == cudaSuccess) e = tmp.put(&ci, M.ci.data(), M.ci.size());
        if (e == cudaSuccess) e = tmp.put(&v, M.v.data(), M.v.size());
        d.rp = rp; d.ci = ci; d.v = v;
        return e;
    };
    for (int l = 0; l <= L; ++l) {
        const HostLevel& lv = h->H.lv[l];
        DevHierLevel& d = hier[l];
        std::memset(&d, 0, sizeof(d));
        d.n = lv.A.nrows;
        CUDA_TRY(put_csr(lv.A, d.A));
        if (l < L) { CUDA_TRY(put_csr(lv.P, d.P)); CUDA_TRY(put_csr(lv.R, d.R)); }
        double* dinv = nullptr;
        CUDA_TRY(tmp.put(&dinv, lv.dinv.data(), lv.dinv.size()));
        d.dinv = dinv;
        if (!lv.cf.empty()) { int8_t* cf = nullptr; CUDA_TRY(tmp.put(&cf, lv.cf.data(), lv.cf.size())); d.cf = cf; }
        if (!lv.coarse_of.empty()) { int* co = nullptr; CUDA_TRY(tmp.put(&co, lv.coarse_of.data(), lv.coarse_of.size())); d.coarse_of = co; }
    }
    DevHierLevel* d_hier = nullptr;
    CUDA_TRY(tmp.put(&d_hier, hier.data(), hier.size()));

    const int nw = std::max(1, std::min(nthreads, P));
    std::vector<std::unique_ptr<CompositeBuilder>> builders(nw);
    const int batch = std::min(P, std::max(1, env_int("AMGDD_SETUP_BATCH", 256)));   // scratch is sized per subdomain of a batch
    const int thin = std::min(h->window, THIN_WINDOW);
    Arena arena;
    cudaStream_t st = h->stream;
    GrowBuf<int> d_idx, d_rows;
    GrowBuf<AsmSlice> d_slices;
    GrowBuf<AsmJob> d_jobs;
    GrowBuf<AsmPlan> d_plans;
    GrowBuf<AsmCopy> d_copies;
    std::vector<std::vector<i32>> lists;              // per subdomain of the batch: owned local indices, then gid of every private level
    std::vector<AsmJob> jobs;
    std::vector<AsmPlan> plans;
    std::vector<AsmCopy> copies;
    std::vector<i32> flat;
    struct JobRef { int p, l, kind; };
    std::vector<JobRef> refs;
    double t_sets = 0, t_dev = 0;
    // AMGDD_INDEX_SETS=host keeps the breadth-first growth of the index sets on the host (the reference the device
    // path is tested against); the device path: amgdd_assemble.cuh, "composite index sets on the device"
    const char* sets_env = std::getenv("AMGDD_INDEX_SETS");
    bool dev_sets = !(sets_env && std::strcmp(sets_env, "host") == 0);
    std::vector<long long> bm_off(L + 2, 0);
    for (int l = 0; l <= L; ++l) bm_off[l + 1] = bm_off[l] + (h->H.lv[l].A.nrows + 31) / 32;
    long long* d_bm_off = nullptr;
    unsigned* d_bm = nullptr;
    int* d_frontier = nullptr;
    // a frontier (or a seed list) holds distinct points of one level, so it never exceeds the largest level: the scratch of a
    // small problem is small (it used to be 3 MiB per subdomain of the batch whatever the size)
    long long max_nl = 1;
    for (int l = 0; l <= L; ++l) max_nl = std::max<long long>(max_nl, h->H.lv[l].A.nrows);
    const int frontier_cap = (int)std::min<long long>(SET_FRONTIER_CAP, max_nl);
    int* d_owned_all = nullptr;
    SetLevelOut* d_set_out = nullptr;
    int** d_list_dst = nullptr;
    SetJob* d_set_jobs = nullptr;
    std::vector<long long> owned_off(P + 1, 0);
    std::vector<SetJob> set_jobs;
    std::vector<SetLevelOut> set_out;
    std::vector<int*> list_dst;
    if (dev_sets) {
        CUDA_TRY(tmp.put(&d_bm_off, bm_off.data(), bm_off.size()));
        CUDA_TRY(tmp.alloc(&d_bm, (size_t)batch * 2 * (size_t)bm_off[L + 1]));
        CUDA_TRY(cudaMemsetAsync(d_bm, 0, (size_t)batch * 2 * (size_t)bm_off[L + 1] * sizeof(unsigned), st));
        CUDA_TRY(tmp.alloc(&d_frontier, (size_t)batch * 3 * (size_t)frontier_cap));
        std::vector<int> flat_owned;
        flat_owned.reserve((size_t)h->n);
        for (int p = 0; p < P; ++p) { flat_owned.insert(flat_owned.end(), owned[p].begin(), owned[p].end()); owned_off[p + 1] = (long long)flat_owned.size(); }
        CUDA_TRY(tmp.put(&d_owned_all, flat_owned.data(), flat_owned.size()));
        CUDA_TRY(tmp.alloc(&d_set_out, (size_t)batch * (L + 1)));
        CUDA_TRY(tmp.alloc(&d_list_dst, (size_t)batch * (L + 1)));
        CUDA_TRY(tmp.alloc(&d_set_jobs, (size_t)batch));
    }
    for (int p0 = 0; p0 < P; p0 += batch) {
        const int p1 = std::min(P, p0 + batch), nb_ = p1 - p0;
        auto t0 = std::chrono::steady_clock::now();
        size_t total = 0;
        std::vector<size_t> base(nb_);
        bool sets_done = false;
        auto t1 = t0;
        if (dev_sets) {
            // a'. index sets on the device: grow (sizes), lay out, extract (ascending lists, row-length sums)
            set_jobs.assign(nb_, SetJob());
            for (int k = 0; k < nb_; ++k) {
                SetJob& j = set_jobs[k];
                std::memset(&j, 0, sizeof(j));
                j.owned = d_owned_all + owned_off[p0 + k]; j.n_owned = (int)(owned_off[p0 + k + 1] - owned_off[p0 + k]);
                j.bm_real = d_bm + (size_t)k * 2 * (size_t)bm_off[L + 1];
                j.bm_ghost = j.bm_real + bm_off[L + 1];
                j.frontier = d_frontier + (size_t)k * 3 * (size_t)frontier_cap; j.frontier_cap = frontier_cap;
                j.out = d_set_out + (size_t)k * (L + 1);
                j.list_dst = d_list_dst + (size_t)k * (L + 1);
            }
            CUDA_TRY(cudaMemcpyAsync(d_set_jobs, set_jobs.data(), set_jobs.size() * sizeof(SetJob), cudaMemcpyHostToDevice, st));
            CUDA_TRY(launch_sets_grow(d_set_jobs, nb_, d_hier, d_bm_off, L, h->eta, h->nghost, st));
            set_out.resize((size_t)nb_ * (L + 1));
            CUDA_TRY(cudaMemcpyAsync(set_out.data(), d_set_out, set_out.size() * sizeof(SetLevelOut), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaMemcpyAsync(set_jobs.data(), d_set_jobs, set_jobs.size() * sizeof(SetJob), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            bool overflow = false;
            for (int k = 0; k < nb_; ++k) overflow = overflow || set_jobs[k].overflow != 0;
            if (overflow) {
                // a frontier larger than the scratch: the host grows the sets of this and all later batches (bitmaps are left dirty)
                dev_sets = false;
            } else {
                for (int k = 0; k < nb_; ++k) {
                    SubdomainBlob& sb = h->subs[p0 + k].plan;
                    sb.lev.assign(L + 1, BlockLayout());
                    sb.dropped = 0; sb.too_long_row = -1; sb.too_long_level = -1;
                    sb.n_owned = set_jobs[k].n_owned;
                    base[k] = total;
                    size_t cnt = (size_t)sb.n_owned;
                    for (int l = 0; l <= L; ++l) {
                        const SetLevelOut& o = set_out[(size_t)k * (L + 1) + l];
                        BlockLayout& b = sb.lev[l];
                        b.n_real = o.n_real; b.n_ghost = o.n_ghost;
                        b.shared = (i64)o.n_real == h->H.lv[l].A.nrows;
                        if (!b.shared) cnt += (size_t)o.n_real + o.n_ghost;
                    }
                    total += (cnt + 3) & ~(size_t)3;
                }
                CUDA_TRY(d_idx.need(total));
                list_dst.assign((size_t)nb_ * (L + 1), nullptr);
                for (int k = 0; k < nb_; ++k) {
                    const SubdomainBlob& sb = h->subs[p0 + k].plan;
                    size_t o = base[k] + (size_t)sb.n_owned;
                    set_jobs[k].owned_local_dst = d_idx.p + base[k];
                    for (int l = 0; l <= L; ++l) {
                        if (sb.lev[l].shared) continue;
                        list_dst[(size_t)k * (L + 1) + l] = d_idx.p + o;
                        o += (size_t)sb.lev[l].n_real + sb.lev[l].n_ghost;
                    }
                }
                CUDA_TRY(cudaMemcpyAsync(d_list_dst, list_dst.data(), list_dst.size() * sizeof(int*), cudaMemcpyHostToDevice, st));
                CUDA_TRY(cudaMemcpyAsync(d_set_jobs, set_jobs.data(), set_jobs.size() * sizeof(SetJob), cudaMemcpyHostToDevice, st));
                CUDA_TRY(launch_sets_extract(d_set_jobs, nb_, d_hier, d_bm_off, L, st));
                CUDA_TRY(cudaMemcpyAsync(set_out.data(), d_set_out, set_out.size() * sizeof(SetLevelOut), cudaMemcpyDeviceToHost, st));
                CUDA_TRY(cudaStreamSynchronize(st));
                for (int k = 0; k < nb_; ++k) {
                    SubdomainBlob& sb = h->subs[p0 + k].plan;
                    for (int l = 0; l <= L; ++l) {
                        const SetLevelOut& o = set_out[(size_t)k * (L + 1) + l];
                        BlockLayout& b = sb.lev[l];
                        b.nnzA_real = o.nnzA_real;
                        if (b.shared) { b.nnzA = b.nnzA_real; b.nnzP = (l < L) ? h->H.lv[l].P.nnz() : 0; }
                        else if (o.nnzA_real + o.nnzA_ghost_bound > (i64)INT32_MAX || o.nnzP_bound > (i64)INT32_MAX) {
                            g_detail = "a composite level exceeds 2^31-1 local nonzeros";
                            return AMGDD_ERR_INDEX_RANGE;
                        }
                    }
                }
                sets_done = true;
                t1 = std::chrono::steady_clock::now();
                t_sets += std::chrono::duration<double>(t1 - t0).count();
            }
        }
        if (!sets_done) {
        // a. index sets on the host (breadth-first growth, S6/S7), one subdomain per task
        lists.assign(nb_, std::vector<i32>());
        std::atomic<int> next(p0);
        std::atomic<int> status(AMGDD_SUCCESS);
        std::string fail_detail;
        std::mutex fail_mu;
        auto work = [&](int t) {
          try {
            if (!builders[t]) builders[t].reset(new CompositeBuilder(h->H, owner, owned, h->eta, h->nghost, h->window));
            CompositeBuilder& cb = *builders[t];
            std::vector<i32> own;
            for (;;) {
                const int p = next.fetch_add(1);
                if (p >= p1 || status.load() != AMGDD_SUCCESS) break;
                SubMeta& sm = h->subs[p];
                if (!cb.plan_sets(p, sm.plan)) {
                    std::lock_guard<std::mutex> g(fail_mu);
                    status.store(AMGDD_ERR_INDEX_RANGE);
                    fail_detail = "a composite level exceeds 2^31-1 local nonzeros";
                    break;
                }
                std::vector<i32>& out = lists[p - p0];
                cb.owned_local(own);
                out.insert(out.end(), own.begin(), own.end());
                for (int l = 0; l <= L; ++l) {
                    if (sm.plan.lev[l].shared) continue;
                    out.insert(out.end(), cb.real(l).begin(), cb.real(l).end());
                    out.insert(out.end(), cb.ghost(l).begin(), cb.ghost(l).end());
                }
            }
          } catch (const std::exception& e) {                              // bad_alloc of the per-thread maps / lists: report, do not terminate
              std::lock_guard<std::mutex> g(fail_mu);
              if (status.load() == AMGDD_SUCCESS) { status.store(AMGDD_ERR_OUT_OF_MEMORY); fail_detail = std::string("host allocation failed while growing the index sets: ") + e.what(); }
          }
        };
        run_threads(nw, work);
        if (status.load() != AMGDD_SUCCESS) { g_detail = fail_detail; return status.load(); }
        t1 = std::chrono::steady_clock::now();
        t_sets += std::chrono::duration<double>(t1 - t0).count();
        // b. index lists to the device; jobs of the batch
        total = 0;
        for (int k = 0; k < nb_; ++k) { base[k] = total; total += (lists[k].size() + 3) & ~(size_t)3; }
        flat.assign(total, 0);
        for (int k = 0; k < nb_; ++k) std::copy(lists[k].begin(), lists[k].end(), flat.begin() + base[k]);
        CUDA_TRY(d_idx.need(total));
        CUDA_TRY(cudaMemcpyAsync(d_idx.p, flat.data(), total * sizeof(i32), cudaMemcpyHostToDevice, st));
        }
        jobs.clear(); refs.clear();
        long long row_off = 0, slice_off = 0;
        std::vector<std::vector<const int*>> gidp(nb_, std::vector<const int*>(L + 1, nullptr));
        for (int k = 0; k < nb_; ++k) {
            const SubdomainBlob& sb = h->subs[p0 + k].plan;
            size_t o = base[k] + (size_t)sb.n_owned;
            for (int l = 0; l <= L; ++l) {
                if (sb.lev[l].shared) continue;
                gidp[k][l] = d_idx.p + o;
                o += (size_t)sb.lev[l].n_real + sb.lev[l].n_ghost;
            }
            for (int l = 0; l < L; ++l) {
                const BlockLayout& b = sb.lev[l];
                if (b.shared) continue;
                const BlockLayout& c = sb.lev[l + 1];
                const int nb = b.n_real + b.n_ghost, nbc = c.n_real + c.n_ghost;
                for (int kind = 0; kind < 3; ++kind) {
                    AsmJob j;
                    std::memset(&j, 0, sizeof(j));
                    j.kind = kind; j.level = l;
                    j.nrows = kind == ASM_R ? nbc : nb;
                    j.nrows_first = kind == ASM_A ? b.n_real : j.nrows;
                    j.nr = b.n_real; j.ng = b.n_ghost; j.nrc = c.n_real; j.ngc = c.n_ghost;
                    j.gid = gidp[k][l]; j.gidc = gidp[k][l + 1];
                    j.window = kind == ASM_A ? h->window : thin;
                    j.wide = needs_wide(j.nrows, kind == ASM_P ? nbc : nb);
                    j.scratch_row = row_off; j.scratch_slice = slice_off;
                    row_off += 2LL * j.nrows;
                    slice_off += (j.nrows_first + SLICE_ROWS - 1) / SLICE_ROWS + (j.nrows - j.nrows_first + SLICE_ROWS - 1) / SLICE_ROWS;
                    jobs.push_back(j);
                    refs.push_back({p0 + k, l, kind});
                }
            }
        }
        const int njobs = (int)jobs.size();
        CUDA_TRY(d_rows.need((size_t)row_off));
        CUDA_TRY(d_slices.need((size_t)slice_off));
        CUDA_TRY(d_jobs.need(jobs.size()));
        CUDA_TRY(d_plans.need(jobs.size()));
        // c. plan pass: row lengths, sort, slices, dealing -> sizes and way tables
        if (njobs) {
            CUDA_TRY(cudaMemcpyAsync(d_jobs.p, jobs.data(), jobs.size() * sizeof(AsmJob), cudaMemcpyHostToDevice, st));
            CUDA_TRY(launch_asm_plan(d_jobs.p, njobs, d_hier, d_rows.p, d_slices.p, d_plans.p, st));
            plans.resize(jobs.size());
            CUDA_TRY(cudaMemcpyAsync(plans.data(), d_plans.p, jobs.size() * sizeof(AsmPlan), cudaMemcpyDeviceToHost, st));
        }
        CUDA_TRY(cudaStreamSynchronize(st));
        // d. layouts, arena space, destinations
        for (int q = 0; q < njobs; ++q) {
            const JobRef& r = refs[q];
            const AsmPlan& pl = plans[q];
            SubdomainBlob& sb = h->subs[r.p].plan;
            BlockLayout& b = sb.lev[r.l];
            if (pl.dropped > 0) {
                g_detail = "subdomain " + std::to_string(r.p) + ": " + std::to_string(pl.dropped) +
                           " interpolation entries of composite rows fall outside D-bar_{l+1}";
                return AMGDD_ERR_NOT_CONNECTED_UPWARD;
            }
            if (pl.too_long_row >= 0) {
                g_detail = "subdomain " + std::to_string(r.p) + ", level " + std::to_string(r.l) + ": a local matrix row has more than 65535 entries";
                return AMGDD_ERR_INDEX_RANGE;
            }
            StreamLayout& sl = r.kind == ASM_A ? b.A : (r.kind == ASM_P ? b.P : b.R);
            sl.nrows = jobs[q].nrows; sl.nnz = pl.nnz; sl.wide = jobs[q].wide != 0;
            sl.bytes = pl.bytes; sl.bytes_real = pl.bytes_real; sl.padded_nnz = pl.padded_nnz;
            for (int w = 0; w < NUM_WAYS; ++w) sl.way[w] = pl.way[w];
            if (r.kind == ASM_A) { b.nnzA = pl.nnz; b.nnzA_ghost = b.nnzA - b.nnzA_real; }
            if (r.kind == ASM_P) b.nnzP = pl.nnz;
        }
        copies.clear();
        {   // one arena chunk per batch instead of many 1 GB chunks (cudaMalloc is not cheap)
            size_t total = 0;
            for (int k = 0; k < nb_; ++k) {
                layout_blob(h->subs[p0 + k].plan);
                total += ((size_t)std::max<i64>(h->subs[p0 + k].plan.bytes, 16) + 255) & ~(size_t)255;
            }
            arena.chunk = std::max<size_t>((size_t)1 << 30, total);
        }
        for (int k = 0; k < nb_; ++k) {
            SubMeta& sm = h->subs[p0 + k];
            std::string why;
            const int arc = arena_take(h, arena, (size_t)std::max<i64>(sm.plan.bytes, 16), &sm.dev_base, why);
            if (arc) { g_detail = why; return arc; }
            AsmCopy c;
            std::memset(&c, 0, sizeof(c));
            c.src = d_idx.p + base[k]; c.dst = (int*)(sm.dev_base + sm.plan.off_owned); c.n = sm.plan.n_owned;
            copies.push_back(c);
            for (int l = 0; l <= L; ++l) {
                const BlockLayout& b = sm.plan.lev[l];
                if (b.shared) continue;
                c.src = gidp[k][l]; c.dst = (int*)(sm.dev_base + b.off_gid); c.n = b.n_real + b.n_ghost; c.gather = 0; c.dinv = nullptr;
                copies.push_back(c);
                c.dst = (int*)(sm.dev_base + b.off_dinv); c.n = b.n_real + b.n_ghost; c.n_gather = b.n_real; c.gather = 1; c.dinv = hier[l].dinv;
                copies.push_back(c);
            }
        }
        for (int q = 0; q < njobs; ++q) {
            const JobRef& r = refs[q];
            const SubMeta& sm = h->subs[r.p];
            const BlockLayout& b = sm.plan.lev[r.l];
            jobs[q].dst = sm.dev_base + (r.kind == ASM_A ? b.A.off : (r.kind == ASM_P ? b.P.off : b.R.off));
        }
        // e. write pass
        CUDA_TRY(d_copies.need(copies.size()));
        CUDA_TRY(cudaMemcpyAsync(d_copies.p, copies.data(), copies.size() * sizeof(AsmCopy), cudaMemcpyHostToDevice, st));
        CUDA_TRY(launch_asm_copy(d_copies.p, (int)copies.size(), st));
        if (njobs) {
            CUDA_TRY(cudaMemcpyAsync(d_jobs.p, jobs.data(), jobs.size() * sizeof(AsmJob), cudaMemcpyHostToDevice, st));
            CUDA_TRY(launch_asm_write(d_jobs.p, njobs, d_hier, d_rows.p, d_slices.p, d_plans.p, st));
            CUDA_TRY(cudaMemcpyAsync(plans.data(), d_plans.p, jobs.size() * sizeof(AsmPlan), cudaMemcpyDeviceToHost, st));
        }
        CUDA_TRY(cudaStreamSynchronize(st));
        for (int q = 0; q < njobs; ++q)
            if (plans[q].bad_col) {
                g_detail = "subdomain " + std::to_string(refs[q].p) + ", level " + std::to_string(refs[q].l) +
                           ": a real row of A_l leaves D-bar_l (eq. 1 violated)";
                return AMGDD_ERR_INDEX_RANGE;
            }
        t_dev += std::chrono::duration<double>(std::chrono::steady_clock::now() - t1).count();
    }
    h->stats.setup_seconds_index_sets = t_sets;
    h->stats.setup_seconds_assembly = t_dev;
    h->stats.setup_seconds_upload = std::chrono::duration<double>(std::chrono::steady_clock::now() - tA).count() - t_sets - t_dev;
    h->stats.assembled_on_device = 1;
    h->stats.index_sets_on_device = dev_sets ? 1 : 0;
    return AMGDD_SUCCESS;
}

// the SURVEY.md §8(d) traffic model (nu = 1) and the bytes this build's kernel actually streams
void traffic_model(amgdd_handle_s* h) {
    amgdd_stats_t& s = h->stats;
    const int L = h->H.L;
    double model[2] = {0, 0}, stream[2] = {0, 0}, useful[2] = {0, 0};
    for (const SubMeta& sm : h->subs) {
        auto layA = [&](int l) -> const StreamLayout& { return sm.plan.lev[l].shared ? h->glev[l].layA : sm.plan.lev[l].A; };
        auto layP = [&](int l) -> const StreamLayout& { return sm.plan.lev[l].shared ? h->glev[l].layP : sm.plan.lev[l].P; };
        auto layR = [&](int l) -> const StreamLayout& { return sm.plan.lev[l].shared ? h->glev[l].layR : sm.plan.lev[l].R; };
        for (int l = 0; l < L; ++l) {
            const BlockLayout& b = sm.plan.lev[l];
            const BlockLayout& c = sm.plan.lev[l + 1];
            const double nr = b.n_real, ng = b.n_ghost, nb = nr + ng;
            const double nrc = c.n_real, nbc = (double)c.n_real + c.n_ghost;
            const double Ar = 12.0 * b.nnzA_real + 4.0 * nr, Ag = 12.0 * b.nnzA_ghost + 4.0 * ng;
            const double Pm = 12.0 * b.nnzP + 4.0 * nb, Pt = 12.0 * b.nnzP + 4.0 * nbc;
            const double Arc = 12.0 * c.nnzA_real + 4.0 * nrc;
            const double pre = (l == 0) ? (Ar + 8 * nb + 40 * nr) : 32 * nr;
            const double at = Ar + Ag + 8 * nr + 16 * nb;
            const double rs = Pt + 8 * nb + 8 * nbc;
            const double rc = Arc + 16 * nbc + 16 * nrc;
            const double ip = Pm + 8 * nbc + 16 * nb;
            const double post = Ar + 8 * nb + 40 * nr;
            model[0] += 32 * nr + at + rs + ip + post;             // first iteration: u_l = 0 on every level, the first sweep needs no matrix (a4)
            model[1] += pre + at + rs + rc + ip + post;
            const StreamLayout& A = layA(l);
            const double a_real = (double)A.bytes_real;
            const double a_all = (double)A.bytes;
            const StreamLayout& Ac = layA(l + 1);
            const double ac_real = (double)Ac.bytes_real;
            // pre-relaxation: matrix-free on every level in the first iteration (u = 0: OPK_FIRST0 on level 0, fused into the
            // restriction on l >= 1); in later iterations level 0 runs a real sweep over A_0's real rows
            const double common = a_all + (double)layR(l).bytes + (double)layP(l).bytes + a_real;
            stream[0] += common;
            stream[1] += common + (l == 0 ? a_real : 0.0) + ac_real;
            // the entries themselves: A_l (A t: all rows; post-relaxation: real rows), R_l, P_l; later iterations add the
            // pre-relaxation of level 0 and the recalculation on level l+1
            const double eA = A.wide ? 12.0 : 10.0, eAc = Ac.wide ? 12.0 : 10.0;
            const double eP = layP(l).wide ? 12.0 : 10.0, eR = layR(l).wide ? 12.0 : 10.0;
            const double ucommon = eA * (2.0 * b.nnzA_real + b.nnzA_ghost) + (eP + eR) * b.nnzP;
            useful[0] += ucommon;
            useful[1] += ucommon + (l == 0 ? eA * b.nnzA_real : 0.0) + eAc * c.nnzA_real;
        }
    }
    s.model_bytes_fac_iter[0] = model[0]; s.model_bytes_fac_iter[1] = model[1];
    s.stream_bytes_fac_iter[0] = stream[0]; s.stream_bytes_fac_iter[1] = stream[1];
    s.useful_bytes_fac_iter[0] = useful[0]; s.useful_bytes_fac_iter[1] = useful[1];
    double g = 12.0 * h->H.lv[0].A.nnz() + 4.0 * h->n + 24.0 * h->n;            // a1: A_0, x, b, r
    for (int l = 0; l < L; ++l) g += 12.0 * h->H.lv[l].P.nnz() + 4.0 * h->H.lv[l + 1].A.nrows + 8.0 * (h->H.lv[l].A.nrows + h->H.lv[l + 1].A.nrows);
    g += 12.0 * (double)s.sum_real + 24.0 * h->n;                                // a3 gather, a10 update
    s.model_bytes_global = g;
}

StreamDesc make_desc(const char* base, const StreamLayout& lay, bool shared = false) {
    StreamDesc d;
    std::memset(&d, 0, sizeof(d));
    d.base = base;
    for (int w = 0; w < NUM_WAYS; ++w) d.way[w] = lay.way[w];
    d.flags = (lay.wide ? STREAM_WIDE : 0u) | (shared ? STREAM_SHARED : 0u);
    return d;
}

int upload_packed(amgdd_handle_s* h, const HostCsr& M, const std::vector<int8_t>* cf, char** dptr, StreamLayout& lay, const char* what, int l) {
    std::vector<uint8_t> flags;                                      // C-points of the rows' level (CF smoother)
    if (cf && !cf->empty()) { flags.resize(cf->size()); for (size_t i = 0; i < cf->size(); ++i) flags[i] = (*cf)[i] > 0 ? 1 : 0; }
    const int window = what[0] == 'A' ? h->window : std::min(h->window, THIN_WINDOW);
    PackedLevelStream ps;
    i64 bad = -1;
    if (!pack_global_stream(M, flags.empty() ? nullptr : flags.data(), window, ps, bad)) { g_detail = "a level matrix has more than 2^31-1 nonzeros"; return AMGDD_ERR_INDEX_RANGE; }
    if (bad >= 0) {
        g_detail = std::string("row ") + std::to_string(bad) + " of " + what + "_" + std::to_string(l) + " has more than 65535 entries";
        return AMGDD_ERR_INDEX_RANGE;
    }
    lay = ps.lay;
    return upload(h, dptr, ps.data.data(), ps.data.size());
}

int finish_tables(amgdd_handle_s* h) {
    const int P = h->P, L = h->H.L;
    // which levels are used through the shared global copy
    std::vector<char> need(L + 1, 0);
    i64 shared_inst = 0;
    for (const SubMeta& sm : h->subs)
        for (int l = 0; l <= L; ++l)
            if (sm.plan.lev[l].shared) { need[l] = 1; ++shared_inst; }
    h->glev.assign(L + 1, GlobalLevelDev());
    int rc;
    for (int l = 0; l <= L; ++l) {
        const HostLevel& lv = h->H.lv[l];
        GlobalLevelDev& g = h->glev[l];
        g.lanes_a = pick_lanes(avg_row(lv.A));
        if (l < L) g.lanes_r = pick_lanes(avg_row(lv.R));
        if (l == 0) {
            if ((rc = upload_csr32(h, lv.A, &g.a_rp, &g.a_ci, &g.a_v))) return rc;   // Alg. 2
            const std::vector<int> blk = stream_row_blocks(lv.A);
            g.a_nblk = (int)blk.size() - 1;
            if ((rc = upload(h, &g.a_blk, blk.data(), blk.size()))) return rc;
        }
        if (l < L) {
            if ((rc = upload_csr32(h, lv.R, &g.r_rp, &g.r_ci, &g.r_v))) return rc;   // Alg. 2 P:473 needs every R_l
            const std::vector<int> blk = stream_row_blocks(lv.R);
            g.r_nblk = (int)blk.size() - 1;
            if ((rc = upload(h, &g.r_blk, blk.data(), blk.size()))) return rc;
        }
        if (need[l]) {
            if ((rc = upload_packed(h, lv.A, &lv.cf, &g.sA, g.layA, "A", l))) return rc;
            if (l < L) {
                if ((rc = upload_packed(h, lv.P, nullptr, &g.sP, g.layP, "P", l))) return rc;
                if ((rc = upload_packed(h, lv.R, &h->H.lv[l + 1].cf, &g.sR, g.layR, "R", l))) return rc;
            }
            if ((rc = upload(h, &g.dinv, lv.dinv.data(), lv.dinv.size()))) return rc;
            std::vector<int> id((size_t)lv.A.nrows);
            std::iota(id.begin(), id.end(), 0);
            if ((rc = upload(h, &g.ident, id.data(), id.size()))) return rc;
        }
    }
    // workspace geometry: per level u | t | s | f (n_bar each), then one scratch vector
    long long max_sum = 0, max_nb = 0;
    std::vector<DevLevel> lev((size_t)P * (L + 1));
    std::vector<DevSub> sub(P);
    amgdd_stats_t& st = h->stats;
    for (int p = 0; p < P; ++p) {
        const SubMeta& sm = h->subs[p];
        long long off = 0;
        for (int l = 0; l <= L; ++l) {
            const BlockLayout& b = sm.plan.lev[l];
            DevLevel& d = lev[(size_t)p * (L + 1) + l];
            std::memset(&d, 0, sizeof(d));
            d.n_real = b.n_real;
            d.n_bar = b.n_real + b.n_ghost;
            max_nb = std::max<long long>(max_nb, d.n_bar);
            st.sum_real += b.n_real; st.sum_ghost += b.n_ghost; st.nnz_composite_real += b.nnzA_real;
            if (b.shared) {
                const GlobalLevelDev& g = h->glev[l];
                d.gid = g.ident; d.dinv = g.dinv;
                d.A = make_desc(g.sA, g.layA, true);
                if (l < L) { d.P = make_desc(g.sP, g.layP, true); d.R = make_desc(g.sR, g.layR, true); }
            } else {
                char* base = sm.dev_base;
                d.gid = (const int*)(base + b.off_gid); d.dinv = (const double*)(base + b.off_dinv);
                d.A = make_desc(base + b.A.off, b.A);
                d.P = make_desc(base + b.P.off, b.P);
                d.R = make_desc(base + b.R.off, b.R);
            }
        }
        // vectors of a level: u | t | s | f, n_bar doubles each, consecutive; levels 16-byte aligned
        off = 0;
        for (int l = 0; l <= L; ++l) {
            DevLevel& d = lev[(size_t)p * (L + 1) + l];
            d.voff = off;
            off += 4LL * d.n_bar;
            off = (off + 1) & ~1LL;
        }
        max_sum = std::max(max_sum, off);
        sub[p].owned = (const int*)(sm.dev_base + sm.plan.off_owned);
        sub[p].n_owned = sm.plan.n_owned;
    }
    st.shared_level_instances = shared_inst;

    // launch plan of the persistent AlgFAC kernel: one CTA of NUM_WAYS warps per SM.  The two vector
    // buffers (the gather vector of a step and the one the step writes for the next) live in shared
    // memory when the largest composite level fits twice next to the tables of the longest program;
    // otherwise they live in the workspace slot (slow path, same arithmetic).
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, h->device));
    h->smem_cta = CTAS_PER_SM == 1 ? (int)prop.sharedMemPerBlockOptin
                                   : std::min((int)prop.sharedMemPerBlockOptin, (int)prop.sharedMemPerMultiprocessor / CTAS_PER_SM - 1024);
    h->x_need = (max_nb + 15) & ~15LL;
    h->xg_off = (max_sum + 15) & ~15LL;                          // the slot always has room for the slow path's buffers
    h->slot_stride = h->xg_off + 2 * h->x_need;
    h->x_cap = (int)h->x_need;                                   // refined per solve: the program length decides whether it fits
    h->fac_cfg.block = 32 * NUM_WAYS;
    h->fac_cfg.smem_bytes = fac_smem_bytes(h->x_cap, L, MAX_OPS);       // refined per solve (program length)
    h->fac_cfg.grid = std::max(1, std::min(P, prop.multiProcessorCount * CTAS_PER_SM));
    if (fac_configure(h->device, (int)prop.sharedMemPerBlockOptin) != 0) { g_detail = "cudaFuncSetAttribute(max dynamic shared memory) failed"; cudaGetLastError(); return AMGDD_ERR_CUDA; }
    if ((rc = dev_alloc(h, (void**)&h->d_ops, (size_t)MAX_OPS * sizeof(FacOp)))) return rc;

    if ((rc = dev_alloc(h, (void**)&h->d_workspace, (size_t)h->fac_cfg.grid * h->slot_stride * sizeof(double)))) return rc;
    if ((rc = upload(h, &h->d_lev, lev.data(), lev.size()))) return rc;
    if ((rc = upload(h, &h->d_sub, sub.data(), sub.size()))) return rc;
    // largest subdomains first (longest-processing-time order for the dynamic scheduler)
    std::vector<int> order(P);
    std::iota(order.begin(), order.end(), 0);
    std::vector<i64> cost(P, 0);
    for (int p = 0; p < P; ++p) for (int l = 0; l <= L; ++l) cost[p] += h->subs[p].plan.lev[l].nnzA + h->subs[p].plan.lev[l].nnzP;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return cost[a] > cost[b]; });
    if ((rc = upload(h, &h->d_order, order.data(), order.size()))) return rc;
    // residual vectors of all levels, concatenated
    h->r_off.assign(L + 2, 0);
    for (int l = 0; l <= L; ++l) h->r_off[l + 1] = h->r_off[l] + (((long long)h->H.lv[l].A.nrows + 1) & ~1LL);
    if ((rc = dev_alloc(h, (void**)&h->d_r_all, (size_t)h->r_off[L + 1] * sizeof(double)))) return rc;
    if ((rc = upload(h, &h->d_r_off, h->r_off.data(), (size_t)L + 1))) return rc;
    if ((rc = dev_alloc(h, (void**)&h->d_counter, sizeof(int)))) return rc;
    if (env_int("AMGDD_FAC_PROFILE", 0) > 0) {
        const size_t bytes = (size_t)h->fac_cfg.grid * FAC_PROF_SLOTS * sizeof(long long);
        if ((rc = dev_alloc(h, (void**)&h->d_prof, bytes))) return rc;
        CUDA_TRY(cudaMemset(h->d_prof, 0, bytes));
        const size_t b2 = (size_t)h->fac_cfg.grid * PROF_OPS_STRIDE * sizeof(long long);
        if ((rc = dev_alloc(h, (void**)&h->d_prof_ops, b2))) return rc;
        CUDA_TRY(cudaMemset(h->d_prof_ops, 0, b2));
    }
    if ((rc = upload(h, &h->d_lu, h->H.lu.data(), h->H.lu.size()))) return rc;
    if ((rc = upload(h, &h->d_rowperm, h->H.rowperm.data(), h->H.rowperm.size()))) return rc;
    if (L > 0) { if ((rc = upload(h, &h->d_cf0, h->H.lv[0].cf.data(), h->H.lv[0].cf.size()))) return rc; }
    h->partial_cap = std::max(h->glev[0].a_nblk, residual_num_blocks(h->n, 1));          // stream blocks, or 256 listed rows per block
    if ((rc = dev_alloc(h, (void**)&h->d_partial, (size_t)h->partial_cap * sizeof(double)))) return rc;
    h->norms_cap = 1024;
    if ((rc = dev_alloc(h, (void**)&h->d_norms, (size_t)h->norms_cap * sizeof(double)))) return rc;
    // statistics
    st.num_levels = L + 1; st.num_subdomains = P; st.n_fine = h->n;
    st.nnz_hierarchy = 0;
    for (int l = 0; l <= L; ++l) st.nnz_hierarchy += h->H.lv[l].A.nnz();
    st.overhead = (double)st.nnz_composite_real / (double)st.nnz_hierarchy;
    st.operator_complexity = (double)st.nnz_hierarchy / (double)h->H.lv[0].A.nnz();
    st.dropped_interp_entries = 0;
    traffic_model(h);
    st.device_bytes = h->device_bytes;
    st.block_bytes = GROUP_BYTES_NARROW; st.num_ways = NUM_WAYS; st.window = h->window; st.ring_stages = RING_DEPTH; st.x_cap = h->x_cap;
    st.fac_grid = h->fac_cfg.grid; st.fac_block = h->fac_cfg.block; st.fac_smem_bytes = h->fac_cfg.smem_bytes;
    st.max_n_bar = max_nb;
    return AMGDD_SUCCESS;
}

bool bad_handle(amgdd_handle_t h) {
    if (!h) { g_detail = "null handle"; return true; }
    return false;
}

// every compute entry runs on the device the handle was set up on, whatever the caller's current device is
// (the handle's pointers and the kernels' attributes belong to that device); the caller's device is restored
struct DeviceScope {
    int prev = -1;
    bool ok = true;
    explicit DeviceScope(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceScope() { int cur = -1; if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev); }
};
#define DEVICE_SCOPE(h)                                                                       \
    DeviceScope dev_scope__((h)->device);                                                     \
    if (!dev_scope__.ok) { g_detail = "cannot select the handle's device"; cudaGetLastError(); return AMGDD_ERR_CUDA; }

}  // namespace

extern "C" {

const char* amgdd_strerror(int code) {
    switch (code) {
        case AMGDD_SUCCESS: return "success";
        case AMGDD_ERR_BAD_ARG: return "bad argument";
        case AMGDD_ERR_BAD_CSR: return "malformed CSR matrix";
        case AMGDD_ERR_BAD_OWNER: return "bad owner array";
        case AMGDD_ERR_COARSE_TOO_LARGE: return "coarsest level too large for the dense solve";
        case AMGDD_ERR_SINGULAR_COARSE: return "coarsest-level matrix is singular";
        case AMGDD_ERR_NOT_CONNECTED_UPWARD: return "interpolation stencil of a composite row leaves the composite grid";
        case AMGDD_ERR_OUT_OF_MEMORY: return "out of memory";
        case AMGDD_ERR_CUDA: return "CUDA runtime error";
        case AMGDD_ERR_INDEX_RANGE: return "32-bit local index range exceeded";
        default: return "unknown status";
    }
}

const char* amgdd_last_error_detail(void) { return g_detail.c_str(); }

static int setup_impl(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                      int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                      int32_t max_levels, double theta, int32_t coarse_max, int32_t rank, int32_t nranks, bool sharded,
                      amgdd_handle_t* out);

int amgdd_setup(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                int32_t max_levels, double theta, int32_t coarse_max, amgdd_handle_t* out) {
    return setup_impl(n, rowptr, colind, vals, num_subdomains, owner, eta, num_ghost, max_levels, theta, coarse_max, 0, 1, false, out);
}

int amgdd_setup_shard(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                      int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                      int32_t max_levels, double theta, int32_t coarse_max, int32_t rank, int32_t nranks, amgdd_handle_t* out) {
    if (nranks < 1 || rank < 0 || rank >= nranks || nranks > num_subdomains) {
        if (out) *out = nullptr;
        g_detail = "need 0 <= rank < nranks <= num_subdomains";
        return AMGDD_ERR_BAD_ARG;
    }
    return setup_impl(n, rowptr, colind, vals, num_subdomains, owner, eta, num_ghost, max_levels, theta, coarse_max, rank, nranks, true, out);
}

static int setup_impl(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                      int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                      int32_t max_levels, double theta, int32_t coarse_max, int32_t rank, int32_t nranks, bool sharded,
                      amgdd_handle_t* out) {
    if (out) *out = nullptr;
    g_detail.clear();
    if (!out || !rowptr || !colind || !vals || !owner) { g_detail = "null pointer argument"; return AMGDD_ERR_BAD_ARG; }
    if (n <= 0 || n > (i64)INT32_MAX) { g_detail = "n must be in [1, 2^31-1]"; return AMGDD_ERR_BAD_ARG; }
    if (num_subdomains <= 0 || eta < 0 || num_ghost < 1 || max_levels < 1 || coarse_max < 1 || !(theta > 0.0 && theta <= 1.0)) {
        g_detail = "need P > 0, eta >= 0, num_ghost >= 1, max_levels >= 1, coarse_max >= 1, 0 < theta <= 1";
        return AMGDD_ERR_BAD_ARG;
    }
    int rc = validate_csr(n, rowptr, colind, vals, g_detail);
    if (rc) return rc;
    {
        std::vector<char> seen((size_t)num_subdomains, 0);
        for (i64 i = 0; i < n; ++i) {
            if (owner[i] < 0 || owner[i] >= num_subdomains) { g_detail = "owner[" + std::to_string(i) + "] out of range"; return AMGDD_ERR_BAD_OWNER; }
            seen[owner[i]] = 1;
        }
        for (int p = 0; p < num_subdomains; ++p)
            if (!seen[p]) { g_detail = "subdomain " + std::to_string(p) + " owns no dof"; return AMGDD_ERR_BAD_OWNER; }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g_detail = "no CUDA device: this library has no CPU fallback";
        return AMGDD_ERR_CUDA;
    }
    amgdd_handle_s* h = new (std::nothrow) amgdd_handle_s();
    if (!h) return AMGDD_ERR_OUT_OF_MEMORY;
    std::memset(&h->stats, 0, sizeof(h->stats));
    if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; g_detail = "cudaGetDevice failed"; return AMGDD_ERR_CUDA; }
    h->n = n; h->P = num_subdomains; h->eta = eta; h->nghost = num_ghost;
    h->P_global = num_subdomains;
    if (sharded) {                               // the rank's block of subdomains: [ceil(rank P / R), ceil((rank + 1) P / R))
        h->sub_lo = (int)(((i64)rank * num_subdomains + nranks - 1) / nranks);
        h->P = (int)(((i64)(rank + 1) * num_subdomains + nranks - 1) / nranks) - h->sub_lo;
    }
    h->window = env_int("AMGDD_WINDOW", DEFAULT_WINDOW);
    if (h->window < SLICE_ROWS || h->window > MAX_WINDOW || (h->window % SLICE_ROWS)) {
        delete h;
        g_detail = "AMGDD_WINDOW must be a multiple of 32 in [32, 1048576]";
        return AMGDD_ERR_BAD_ARG;
    }
    const int nthreads = default_threads();
    try {
        auto t0 = std::chrono::steady_clock::now();
        HostCsr A0;
        A0.nrows = A0.ncols = n;
        A0.rp.assign(rowptr, rowptr + n + 1);
        A0.ci.assign(colind, colind + rowptr[n]);
        A0.v.assign(vals, vals + rowptr[n]);
        rc = build_hierarchy(std::move(A0), theta, max_levels, coarse_max, nthreads, h->H, g_detail);
        if (rc) { free_handle(h); return rc; }
        auto t1 = std::chrono::steady_clock::now();
        std::vector<i32> own(owner, owner + n);
        if (sharded) {
            h->shard.reset(new ShardPlan());
            shard_build(h->H, owner, num_subdomains, eta, rank, nranks, *h->shard);
            for (i64 i = 0; i < n; ++i) own[i] = (own[i] >= h->sub_lo && own[i] < h->sub_lo + h->P) ? own[i] - h->sub_lo : -1;
        }
        // AMGDD_ASSEMBLE=host keeps the local matrices and the packing on the host (the reference the device
        // assembly is tested against); windows beyond the device sort's tile also take that path
        const char* asm_env = std::getenv("AMGDD_ASSEMBLE");
        const bool on_host = (asm_env && std::strcmp(asm_env, "host") == 0) || h->window > ASM_MAX_WINDOW;
        rc = on_host ? build_composites(h, own, std::min(nthreads, 32)) : build_composites_device(h, own, std::min(nthreads, 32));
        if (rc) { free_handle(h); return rc; }
        rc = finish_tables(h);
        if (rc) { free_handle(h); return rc; }
        auto t2 = std::chrono::steady_clock::now();
        h->stats.setup_seconds_hierarchy = std::chrono::duration<double>(t1 - t0).count();
        h->stats.setup_seconds_composite = std::chrono::duration<double>(t2 - t1).count();
    } catch (const std::bad_alloc&) {
        free_handle(h);
        g_detail = "host allocation failed during setup";
        return AMGDD_ERR_OUT_OF_MEMORY;
    } catch (const std::exception& e) {                                  // length_error, system_error (thread creation), ...
        free_handle(h);
        g_detail = std::string("setup failed: ") + e.what();
        return AMGDD_ERR_OUT_OF_MEMORY;
    } catch (...) {
        free_handle(h);
        g_detail = "setup failed with an unknown exception";
        return AMGDD_ERR_OUT_OF_MEMORY;
    }
    *out = h;
    return AMGDD_SUCCESS;
}

int amgdd_destroy(amgdd_handle_t h) {
    free_handle(h);
    return AMGDD_SUCCESS;
}

int amgdd_set_smoother(amgdd_handle_t h, int32_t type) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (type != AMGDD_SMOOTHER_L1_JACOBI && type != AMGDD_SMOOTHER_CF_L1_JACOBI) { g_detail = "unknown smoother"; return AMGDD_ERR_BAD_ARG; }
    h->smoother = type;
    return AMGDD_SUCCESS;
}

int amgdd_set_stream(amgdd_handle_t h, void* s) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    h->stream = (cudaStream_t)s;
    return AMGDD_SUCCESS;
}

}  // extern "C"

namespace {

// (re)builds the static program of one subdomain and the launch plan that depends on its length
int ensure_program(amgdd_handle_s* h, int num_fac_cycles, int relax_sweeps) {
    const int L = h->H.L;
    if (h->prog_nfac != num_fac_cycles || h->prog_nu != relax_sweeps || h->prog_smoother != h->smoother) {       // (re)build the program of one subdomain
        const int nops = fac_build_program(L, num_fac_cycles, relax_sweeps, h->smoother, nullptr);
        if (nops > MAX_OPS || L > 84) {
            g_detail = "num_fac_cycles x relax_sweeps x levels gives a program of " + std::to_string(nops) + " steps; the kernel holds " +
                       std::to_string(MAX_OPS);
            return AMGDD_ERR_BAD_ARG;
        }
        std::vector<FacOp> ops((size_t)nops);
        fac_build_program(L, num_fac_cycles, relax_sweeps, h->smoother, ops.data());
        CUDA_TRY(cudaMemcpyAsync(h->d_ops, ops.data(), ops.size() * sizeof(FacOp), cudaMemcpyHostToDevice, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        h->prog_nfac = num_fac_cycles; h->prog_nu = relax_sweeps; h->prog_smoother = h->smoother; h->prog_nops = nops;
        // shared-memory vector buffers: as large as the largest level needs, but leave the L1 (which
        // shares the SM's 228 KB with shared memory) room for the loads in flight: with less than
        // ~48 KB of L1 the streaming rate of this kernel drops by 15% (profiles/).  Levels that do
        // not fit are gathered through L1 from the workspace slot instead.
        const int budget = std::min(h->smem_cta, env_int("AMGDD_SMEM_BUDGET", 180 * 1024));
        const int prof_bytes = h->d_prof ? PROF_SMEM_BYTES : 0;
        long long cap = ((long long)budget - fac_smem_bytes(0, L, nops) - prof_bytes) / 16;
        cap = std::max(0LL, std::min(cap, h->x_need)) & ~15LL;
        if (env_int("AMGDD_FORCE_GLOBAL_X", 0) > 0) cap = 0;
        h->x_cap = (int)cap;
        h->stats.x_cap = h->x_cap;
        h->prof_smem_off = fac_smem_bytes(h->x_cap, L, nops);
        h->fac_cfg.smem_bytes = std::min(h->smem_cta, h->prof_smem_off + prof_bytes);
        h->stats.fac_smem_bytes = h->fac_cfg.smem_bytes;
    }
    return AMGDD_SUCCESS;
}

FacParams fac_params(amgdd_handle_s* h, double* x) {
    const int L = h->H.L;
    FacParams prm;
    prm.lev = h->d_lev; prm.sub = h->d_sub; prm.order = h->d_order;
    prm.num_sub = h->P; prm.L = L;
    prm.r_all = h->d_r_all; prm.r_off = h->d_r_off;
    prm.x = x; prm.workspace = h->d_workspace;
    prm.slot_stride = h->slot_stride; prm.xg_off = h->xg_off;
    prm.work_counter = h->d_counter;
    prm.ops = h->d_ops; prm.nops = h->prog_nops;
    prm.lu = h->d_lu; prm.rowperm = h->d_rowperm; prm.nL = (int)h->H.nL;
    prm.cf0 = h->d_cf0;
    prm.x_cap = h->x_cap;
    prm.prof = h->d_prof;
    prm.prof_smem_off = h->prof_smem_off;
    prm.prof_ops = h->d_prof_ops;
    return prm;
}

// r_0 = b - A_0 x with ||r_0||_2 into d_norms[slot]
int enqueue_residual(amgdd_handle_s* h, const double* b, const double* x, double* r, int norm_slot) {
    const GlobalLevelDev& g = h->glev[0];
    int nb = 0;
    nb = g.a_nblk;
    launch_residual(g.a_rp, g.a_ci, g.a_v, g.a_blk, g.a_nblk, b, x, r, h->d_partial, h->stream);
    launch_norm_finalize(h->d_partial, nb, h->d_norms + norm_slot, h->stream);
    return AMGDD_SUCCESS;
}

}  // namespace

extern "C" {

int amgdd_solve(amgdd_handle_t h, const double* b, double* x, int32_t num_cycles, int32_t num_fac_cycles,
                int32_t relax_sweeps, double* resnorm_host) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (!b || !x || num_cycles < 0 || num_fac_cycles < 1 || relax_sweeps < 1 || num_cycles + 1 > h->norms_cap) {
        g_detail = "need b, x non-null, 0 <= num_cycles < 1024, num_fac_cycles >= 1, relax_sweeps >= 1";
        return AMGDD_ERR_BAD_ARG;
    }
    DEVICE_SCOPE(h);
    const int L = h->H.L;
    const bool timed = resnorm_host != nullptr;
    std::vector<cudaEvent_t>& ev = h->events;                   // owned by the handle: nothing to release on an early return
    size_t nev = 0;
    if (timed) {
        const size_t want = 3 * (size_t)num_cycles + 2;
        while (ev.size() < want) {
            cudaEvent_t e;
            CUDA_TRY(cudaEventCreate(&e));
            ev.push_back(e);
        }
    }
    auto mark = [&]() {
        if (timed) cudaEventRecord(ev[nev++], h->stream);
    };
    {
        const int prc = ensure_program(h, num_fac_cycles, relax_sweeps);
        if (prc) return prc;
    }
    const FacParams prm = fac_params(h, x);
    long long launches[3] = {0, 0, 0};
    // Asynchronous calls (no norms wanted, no phase timers): the cycle is a fixed sequence of 4 + L launches on fixed
    // pointers, so it is captured once as a CUDA graph (on a stream of the handle's own: the caller's may be the legacy
    // default stream, which cannot capture) and replayed on the caller's stream.  AMGDD_GRAPH=0 launches kernel by kernel.
    if (!timed && num_cycles > 0 && !h->graph_off) {
        const bool hit = h->cycle_graph && h->graph_b == b && h->graph_x == x && h->graph_nfac == num_fac_cycles &&
                         h->graph_nu == relax_sweeps && h->graph_smoother == h->smoother && h->graph_nops == h->prog_nops;
        if (!hit) {
            if (env_int("AMGDD_GRAPH", 1) <= 0) h->graph_off = true;
            if (h->cycle_graph) { cudaGraphExecDestroy(h->cycle_graph); h->cycle_graph = nullptr; }
            if (!h->graph_off && !h->capture_stream && cudaStreamCreateWithFlags(&h->capture_stream, cudaStreamNonBlocking) != cudaSuccess) h->graph_off = true;
            if (!h->graph_off) {
                cudaStream_t user = h->stream;
                cudaGraph_t graph = nullptr;
                const char* why = "cudaStreamBeginCapture";
                cudaError_t ce = cudaStreamBeginCapture(h->capture_stream, cudaStreamCaptureModeThreadLocal);
                bool ok = ce == cudaSuccess;
                if (ok) {
                    h->stream = h->capture_stream;
                    enqueue_residual(h, b, x, h->d_r_all, 0);
                    for (int l = 0; l < L; ++l) {
                        const GlobalLevelDev& g = h->glev[l];
                        launch_spmv(g.r_rp, g.r_ci, g.r_v, g.r_blk, g.r_nblk, h->d_r_all + h->r_off[l],
                                    h->d_r_all + h->r_off[l + 1], h->stream);
                    }
                    ce = cudaGetLastError();                                 // a launch-configuration error of the global kernels
                    if (ce != cudaSuccess) { ok = false; why = "a residual / restriction launch during capture"; }
                    if (ok && (ce = cudaMemsetAsync(h->d_counter, 0, sizeof(int), h->stream)) != cudaSuccess) { ok = false; why = "cudaMemsetAsync during capture"; }
                    launch_fac(prm, h->fac_cfg, h->stream);
                    if (ok && (ce = cudaGetLastError()) != cudaSuccess) { ok = false; why = "the fac_kernel launch during capture"; }
                    h->stream = user;
                    const cudaError_t ee = cudaStreamEndCapture(h->capture_stream, &graph);
                    if (ok && (ee != cudaSuccess || !graph)) { ok = false; ce = ee; why = "cudaStreamEndCapture"; }
                }
                if (ok && (ce = cudaGraphInstantiate(&h->cycle_graph, graph, 0)) != cudaSuccess) { ok = false; why = "cudaGraphInstantiate"; }
                if (graph) cudaGraphDestroy(graph);
                if (!ok) {
                    // fall back to kernel-by-kernel launches for the rest of the handle's life, and say why: the call itself
                    // still succeeds if those launches do (a real launch error is reported by them below)
                    cudaGetLastError();
                    h->cycle_graph = nullptr; h->graph_off = true;
                    g_detail = std::string("CUDA graph of the cycle not used (") + why + ": " + cudaGetErrorString(ce) + "); launching kernel by kernel";
                }
                else {
                    h->graph_b = b; h->graph_x = x; h->graph_nfac = num_fac_cycles; h->graph_nu = relax_sweeps;
                    h->graph_smoother = h->smoother; h->graph_nops = h->prog_nops;
                }
            }
        }
        if (h->cycle_graph) {
            for (int k = 0; k < num_cycles; ++k) CUDA_TRY(cudaGraphLaunch(h->cycle_graph, h->stream));
            CUDA_TRY(cudaGetLastError());
            launches[0] = 2LL * num_cycles; launches[1] = (long long)L * num_cycles; launches[2] = num_cycles;
            for (int i = 0; i < 3; ++i) h->prof_launches[i] = launches[i];
            return AMGDD_SUCCESS;
        }
    }
    mark();
    for (int k = 0; k < num_cycles; ++k) {
        enqueue_residual(h, b, x, h->d_r_all, k);                                   // Alg. 2 P:471 (+ a11)
        launches[0] += 2;
        mark();
        for (int l = 0; l < L; ++l) {                                               // Alg. 2
            const GlobalLevelDev& g = h->glev[l];
            launch_spmv(g.r_rp, g.r_ci, g.r_v, g.r_blk, g.r_nblk, h->d_r_all + h->r_off[l],
                        h->d_r_all + h->r_off[l + 1], h->stream);
            launches[1] += 1;
        }
        mark();
        CUDA_TRY(cudaMemsetAsync(h->d_counter, 0, sizeof(int), h->stream));
        launch_fac(prm, h->fac_cfg, h->stream);                                     // Alg. 2
        launches[2] += 1;
        mark();
    }
    if (timed) {                                                                    // ||b - A x|| of the final iterate; nobody can read it
        enqueue_residual(h, b, x, nullptr, num_cycles);                             // in an asynchronous call (resnorm_host = NULL)
        launches[0] += 2;
    }
    mark();
    CUDA_TRY(cudaGetLastError());
    if (timed) {
        CUDA_TRY(cudaMemcpyAsync(resnorm_host, h->d_norms, (size_t)(num_cycles + 1) * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(cudaStreamSynchronize(h->stream));
        double ms[4] = {0, 0, 0, 0};
        for (int k = 0; k < num_cycles; ++k) {
            float a = 0, bb = 0, c = 0;
            cudaEventElapsedTime(&a, ev[3 * k], ev[3 * k + 1]);
            cudaEventElapsedTime(&bb, ev[3 * k + 1], ev[3 * k + 2]);
            cudaEventElapsedTime(&c, ev[3 * k + 2], ev[3 * k + 3]);
            ms[0] += a; ms[1] += bb; ms[2] += c;
        }
        float last = 0, tot = 0;
        cudaEventElapsedTime(&last, ev[3 * num_cycles], ev[3 * num_cycles + 1]);
        cudaEventElapsedTime(&tot, ev[0], ev[nev - 1]);
        ms[0] += last; ms[3] = tot;
        for (int i = 0; i < 4; ++i) h->prof_ms[i] = ms[i];
    }
    for (int i = 0; i < 3; ++i) h->prof_launches[i] = launches[i];
    return AMGDD_SUCCESS;
}

int amgdd_solve_host(amgdd_handle_t h, const double* b_host, double* x_host, int32_t num_cycles,
                     int32_t num_fac_cycles, int32_t relax_sweeps, double* resnorm_host) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (!b_host || !x_host) { g_detail = "null host vector"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    int rc;
    if (!h->d_b_stage || !h->d_x_stage) {                        // both or neither: a failed second allocation leaves the handle usable
        double *sb = nullptr, *sx = nullptr;
        if ((rc = dev_alloc(h, (void**)&sb, (size_t)h->n * sizeof(double)))) return rc;
        if ((rc = dev_alloc(h, (void**)&sx, (size_t)h->n * sizeof(double)))) return rc;    // (sb stays owned by the handle's allocation list)
        h->d_b_stage = sb; h->d_x_stage = sx;
    }
    CUDA_TRY(cudaMemcpyAsync(h->d_b_stage, b_host, (size_t)h->n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(cudaMemcpyAsync(h->d_x_stage, x_host, (size_t)h->n * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    rc = amgdd_solve(h, h->d_b_stage, h->d_x_stage, num_cycles, num_fac_cycles, relax_sweeps, resnorm_host);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(x_host, h->d_x_stage, (size_t)h->n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return AMGDD_SUCCESS;
}

int amgdd_residual_norm(amgdd_handle_t h, const double* b, const double* x, double* out_host) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (!b || !x || !out_host) { g_detail = "null pointer argument"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    enqueue_residual(h, b, x, nullptr, 0);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(out_host, h->d_norms, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return AMGDD_SUCCESS;
}

// AMG V(nu1,nu2)-cycles on the global hierarchy (Alg. 1): the paper's comparison method (Fig. 14)
static int ensure_vcycle(amgdd_handle_s* h) {
    if (h->vcycle_ready) return AMGDD_SUCCESS;
    const int L = h->H.L;
    int rc;
    for (int l = 0; l <= L; ++l) {
        const HostLevel& lv = h->H.lv[l];
        GlobalLevelDev& g = h->glev[l];
        const size_t nl = (size_t)lv.A.nrows;
        if (!g.a_rp) { if ((rc = upload_csr32(h, lv.A, &g.a_rp, &g.a_ci, &g.a_v))) return rc; }
        if (!g.a_blk) {
            const std::vector<int> blk = stream_row_blocks(lv.A);
            g.a_nblk = (int)blk.size() - 1;
            if ((rc = upload(h, &g.a_blk, blk.data(), blk.size()))) return rc;
        }
        if (l < L) {
            if ((rc = upload_csr32(h, lv.P, &g.p_rp, &g.p_ci, &g.p_v))) return rc;
            const std::vector<int> blk = stream_row_blocks(lv.P);
            g.p_nblk = (int)blk.size() - 1;
            if ((rc = upload(h, &g.p_blk, blk.data(), blk.size()))) return rc;
        }
        if ((rc = upload(h, &g.vdinv, lv.dinv.data(), lv.dinv.size()))) return rc;
        if (l < L) { if ((rc = upload(h, &g.vcf, lv.cf.data(), lv.cf.size()))) return rc; }
        if ((rc = dev_alloc(h, (void**)&g.vu0, nl * sizeof(double)))) return rc;
        if ((rc = dev_alloc(h, (void**)&g.vu1, nl * sizeof(double)))) return rc;
        if ((rc = dev_alloc(h, (void**)&g.vf, nl * sizeof(double)))) return rc;
        if ((rc = dev_alloc(h, (void**)&g.vr, nl * sizeof(double)))) return rc;
    }
    h->vcycle_ready = true;
    return AMGDD_SUCCESS;
}

int amgdd_vcycle(amgdd_handle_t h, const double* b, double* x, int32_t num_cycles, int32_t nu1, int32_t nu2, double* resnorm_host) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (!b || !x || num_cycles < 0 || nu1 < 0 || nu2 < 0 || nu1 + nu2 < 1 || num_cycles + 1 > h->norms_cap) {
        g_detail = "need b, x non-null, 0 <= num_cycles < 1024, nu1, nu2 >= 0, nu1 + nu2 >= 1";
        return AMGDD_ERR_BAD_ARG;
    }
    DEVICE_SCOPE(h);
    int rc = ensure_vcycle(h);
    if (rc) return rc;
    const int L = h->H.L;
    const bool cfm = h->smoother == AMGDD_SMOOTHER_CF_L1_JACOBI;
    cudaStream_t st = h->stream;
    auto nrows = [&](int l) { return (long long)h->H.lv[l].A.nrows; };
    for (int k = 0; k < num_cycles; ++k) {
        enqueue_residual(h, b, x, nullptr, k);                                  // ||b - A x_k|| (metric only)
        for (int l = 0; l < L; ++l) {                                           // downsweep P:449-455
            GlobalLevelDev& g = h->glev[l];
            const double* f = l == 0 ? b : g.vf;
            bool have_u = l == 0;                                               // coarse levels start from u = 0
            if (l == 0) CUDA_TRY(cudaMemcpyAsync(g.vu0, x, (size_t)nrows(0) * sizeof(double), cudaMemcpyDeviceToDevice, st));
            for (int s = 0; s < nu1; ++s)                                       // the level's iterate lives in vu0
                for (int half = 0; half < (cfm ? 2 : 1); ++half) {              // CF smoother: C-points, then F-points
                    launch_relax(g.a_rp, g.a_ci, g.a_v, g.a_blk, g.a_nblk, g.vdinv, f, have_u ? g.vu0 : nullptr, g.vu1,
                                 cfm ? (const signed char*)g.vcf : nullptr, half == 0 ? +1 : -1, st);
                    std::swap(g.vu0, g.vu1);
                    have_u = true;
                }
            if (!have_u) CUDA_TRY(cudaMemsetAsync(g.vu0, 0, (size_t)nrows(l) * sizeof(double), st));
            launch_spmv_axpy(g.a_rp, g.a_ci, g.a_v, g.a_blk, g.a_nblk, g.vu0, f, g.vr, 0, st);          // r = f - A u
            launch_spmv(g.r_rp, g.r_ci, g.r_v, g.r_blk, g.r_nblk, g.vr, h->glev[l + 1].vf, st);         // f_{l+1} = P^T r
        }
        launch_coarse_solve(h->d_lu, h->d_rowperm, (int)h->H.nL, L == 0 ? b : h->glev[L].vf, L == 0 ? x : h->glev[L].vu0, st);
        for (int l = L - 1; l >= 0; --l) {                                      // upsweep P:459-464
            GlobalLevelDev& g = h->glev[l];
            const double* f = l == 0 ? b : g.vf;
            launch_spmv_axpy(g.p_rp, g.p_ci, g.p_v, g.p_blk, g.p_nblk, h->glev[l + 1].vu0, nullptr, g.vu0, 1, st);   // u += P u_{l+1}
            for (int s = 0; s < nu2; ++s)
                for (int half = 0; half < (cfm ? 2 : 1); ++half) {              // CF smoother: F-points, then C-points
                    launch_relax(g.a_rp, g.a_ci, g.a_v, g.a_blk, g.a_nblk, g.vdinv, f, g.vu0, g.vu1,
                                 cfm ? (const signed char*)g.vcf : nullptr, half == 0 ? -1 : +1, st);
                    std::swap(g.vu0, g.vu1);
                }
            if (l == 0) CUDA_TRY(cudaMemcpyAsync(x, g.vu0, (size_t)nrows(0) * sizeof(double), cudaMemcpyDeviceToDevice, st));
        }
    }
    enqueue_residual(h, b, x, nullptr, num_cycles);
    CUDA_TRY(cudaGetLastError());
    if (resnorm_host) {
        CUDA_TRY(cudaMemcpyAsync(resnorm_host, h->d_norms, (size_t)(num_cycles + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
    }
    return AMGDD_SUCCESS;
}

// ---------------------------------------------------------------------------------------------
// Sharding over ranks (paper section 5 and Alg. 5): index protocol and stages
// ---------------------------------------------------------------------------------------------
int amgdd_shard_plan_create(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, int32_t num_subdomains,
                            const int32_t* owner, int32_t eta, int32_t max_levels, double theta, int32_t coarse_max, int32_t rank,
                            int32_t nranks, amgdd_shard_plan_t* out) {
    if (out) *out = nullptr;
    g_detail.clear();
    if (!out || !rowptr || !colind || !vals || !owner || n <= 0 || n > (i64)INT32_MAX || num_subdomains <= 0 || eta < 0 || max_levels < 1 ||
        coarse_max < 1 || !(theta > 0.0 && theta <= 1.0) || nranks < 1 || rank < 0 || rank >= nranks || nranks > num_subdomains) {
        g_detail = "bad argument to amgdd_shard_plan_create";
        return AMGDD_ERR_BAD_ARG;
    }
    int rc = validate_csr(n, rowptr, colind, vals, g_detail);
    if (rc) return rc;
    for (i64 i = 0; i < n; ++i)
        if (owner[i] < 0 || owner[i] >= num_subdomains) { g_detail = "owner[" + std::to_string(i) + "] out of range"; return AMGDD_ERR_BAD_OWNER; }
    try {
        std::unique_ptr<amgdd_shard_plan_s> p(new amgdd_shard_plan_s());
        p->H.reset(new Hierarchy());
        HostCsr A0;
        A0.nrows = A0.ncols = n;
        A0.rp.assign(rowptr, rowptr + n + 1);
        A0.ci.assign(colind, colind + rowptr[n]);
        A0.v.assign(vals, vals + rowptr[n]);
        rc = build_hierarchy(std::move(A0), theta, max_levels, coarse_max, default_threads(), *p->H, g_detail);
        if (rc) return rc;
        p->own.reset(new ShardPlan());
        shard_build(*p->H, owner, num_subdomains, eta, rank, nranks, *p->own);
        p->S = p->own.get();
        *out = p.release();
    } catch (const std::exception& e) {
        g_detail = std::string("amgdd_shard_plan_create failed: ") + e.what();
        return AMGDD_ERR_OUT_OF_MEMORY;
    }
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_destroy(amgdd_shard_plan_t p) {
    delete p;
    return AMGDD_SUCCESS;
}

int amgdd_get_shard_plan(amgdd_handle_t h, amgdd_shard_plan_t* out) {
    if (bad_handle(h) || !out) return AMGDD_ERR_BAD_ARG;
    if (!h->shard) { g_detail = "the handle was not set up with amgdd_setup_shard"; return AMGDD_ERR_BAD_ARG; }
    if (!h->shard_view) { h->shard_view.reset(new amgdd_shard_plan_s()); h->shard_view->S = h->shard.get(); }
    *out = h->shard_view.get();
    return AMGDD_SUCCESS;
}

#define PLAN_OK(p) if (!(p) || !(p)->S) { g_detail = "null shard plan"; return AMGDD_ERR_BAD_ARG; }
#define STAGE_PEER_OK(S, stage, peer)                                                                  \
    if ((stage) < 0 || (stage) >= (int)(S).stages.size() || (peer) < 0 || (peer) >= (S).nranks) {      \
        g_detail = "stage or rank out of range"; return AMGDD_ERR_BAD_ARG; }

int amgdd_shard_plan_info(amgdd_shard_plan_t p, int32_t info[6]) {
    PLAN_OK(p);
    if (!info) return AMGDD_ERR_BAD_ARG;
    const ShardPlan& S = *p->S;
    info[0] = S.rank; info[1] = S.nranks; info[2] = S.L + 1; info[3] = (int32_t)S.stages.size(); info[4] = S.sub_lo; info[5] = S.sub_hi;
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_level(amgdd_shard_plan_t p, int32_t l, int64_t* n_l, int64_t* r_offset, int64_t* n_owned) {
    PLAN_OK(p);
    const ShardPlan& S = *p->S;
    if (l < 0 || l > S.L) { g_detail = "level out of range"; return AMGDD_ERR_BAD_ARG; }
    if (n_l) *n_l = (int64_t)S.owner_rank[l].size();
    if (r_offset) *r_offset = S.r_off[l];
    if (n_owned) *n_owned = (int64_t)S.owned[l].size();
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_owner_rank(amgdd_shard_plan_t p, int32_t l, int32_t* owner_rank) {
    PLAN_OK(p);
    const ShardPlan& S = *p->S;
    if (l < 0 || l > S.L || !owner_rank) { g_detail = "level out of range"; return AMGDD_ERR_BAD_ARG; }
    std::copy(S.owner_rank[l].begin(), S.owner_rank[l].end(), owner_rank);
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_list(amgdd_shard_plan_t p, int32_t which, int32_t stage, int32_t peer, int64_t* pos, int64_t* count) {
    PLAN_OK(p);
    const ShardPlan& S = *p->S;
    STAGE_PEER_OK(S, stage, peer);
    if (!count || (which != 0 && which != 1)) return AMGDD_ERR_BAD_ARG;
    const std::vector<i64>& v = which == 0 ? S.stages[stage].send[peer] : S.stages[stage].recv[peer];
    *count = (int64_t)v.size();
    if (pos) std::copy(v.begin(), v.end(), pos);
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_stage_vector(amgdd_shard_plan_t p, int32_t stage, int32_t* vec) {
    PLAN_OK(p);
    if (stage < 0 || stage >= (int)p->S->stages.size() || !vec) return AMGDD_ERR_BAD_ARG;
    *vec = p->S->stages[stage].vec;
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_recv_filter(amgdd_shard_plan_t p, int32_t stage, int32_t src, const int64_t* announced, int64_t count,
                                 int64_t* redundant, int64_t* nredundant) {
    PLAN_OK(p);
    ShardPlan& S = *p->S;
    STAGE_PEER_OK(S, stage, src);
    if (count < 0 || (count > 0 && (!announced || !redundant)) || !nredundant) return AMGDD_ERR_BAD_ARG;
    const i64 limit = S.stages[stage].vec == 0 ? (i64)S.have_x.size() : (i64)S.have.size();
    for (int64_t k = 0; k < count; ++k)
        if (announced[k] < 0 || announced[k] >= limit) { g_detail = "announced position out of range"; return AMGDD_ERR_BAD_ARG; }
    std::vector<uint8_t>& done = S.stages[stage].filtered;
    done.resize((size_t)S.nranks, 0);
    if (done[src]) {
        g_detail = "the index protocol already ran for stage " + std::to_string(stage) + ", source " + std::to_string(src) +
                   " (it is not repeatable on a plan: set the handle or plan up again)";
        return AMGDD_ERR_BAD_ARG;
    }
    done[src] = 1;
    std::vector<i64> red;
    shard_recv_filter(S, stage, src, announced, count, red);
    *nredundant = (int64_t)red.size();
    std::copy(red.begin(), red.end(), redundant);
    return AMGDD_SUCCESS;
}

int amgdd_shard_plan_apply_drop(amgdd_shard_plan_t p, int32_t stage, int32_t dest, const int64_t* redundant, int64_t count) {
    PLAN_OK(p);
    ShardPlan& S = *p->S;
    STAGE_PEER_OK(S, stage, dest);
    if (count < 0 || (count > 0 && !redundant)) return AMGDD_ERR_BAD_ARG;
    std::vector<uint8_t>& done = S.stages[stage].dropped;
    done.resize((size_t)S.nranks, 0);
    if (done[dest]) {
        g_detail = "redundant positions were already removed for stage " + std::to_string(stage) + ", destination " + std::to_string(dest);
        return AMGDD_ERR_BAD_ARG;
    }
    done[dest] = 1;
    shard_apply_drop(S, stage, dest, redundant, count);
    return AMGDD_SUCCESS;
}

#define SHARD_OK(h) if (bad_handle(h)) return AMGDD_ERR_BAD_ARG; \
    if (!(h)->shard) { g_detail = "the handle was not set up with amgdd_setup_shard"; return AMGDD_ERR_BAD_ARG; }
#define SHARD_READY(h) SHARD_OK(h) \
    if (!(h)->shard_committed) { g_detail = "run the index protocol and amgdd_shard_commit first"; return AMGDD_ERR_BAD_ARG; }

int amgdd_shard_commit(amgdd_handle_t h) {
    SHARD_OK(h);
    if (h->shard_committed) { g_detail = "amgdd_shard_commit already ran on this handle (its device lists are in use)"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    const ShardPlan& S = *h->shard;
    const int R = S.nranks;
    int rc;
    h->stage_dev.assign(S.stages.size(), amgdd_handle_s::StageDev());
    for (size_t s = 0; s < S.stages.size(); ++s) {
        amgdd_handle_s::StageDev& d = h->stage_dev[s];
        d.send_counts.assign(R, 0); d.recv_counts.assign(R, 0);
        std::vector<long long> sp, rv;
        for (int q = 0; q < R; ++q) {
            d.send_counts[q] = (long long)S.stages[s].send[q].size();
            d.recv_counts[q] = (long long)S.stages[s].recv[q].size();
            sp.insert(sp.end(), S.stages[s].send[q].begin(), S.stages[s].send[q].end());
            rv.insert(rv.end(), S.stages[s].recv[q].begin(), S.stages[s].recv[q].end());
        }
        d.nsend = (long long)sp.size(); d.nrecv = (long long)rv.size();
        if ((rc = upload(h, &d.send_pos, sp.data(), sp.size()))) return rc;
        if ((rc = upload(h, &d.recv_pos, rv.data(), rv.size()))) return rc;
    }
    h->d_owned_rows.assign(S.L + 1, nullptr);
    for (int l = 0; l <= S.L; ++l)
        if ((rc = upload(h, &h->d_owned_rows[l], S.owned[l].data(), S.owned[l].size()))) return rc;
    std::vector<int> all;
    h->owned0_off.assign(R + 1, 0);
    for (int q = 0; q < R; ++q) { all.insert(all.end(), S.owned0_all[q].begin(), S.owned0_all[q].end()); h->owned0_off[q + 1] = (long long)all.size(); }
    if ((rc = upload(h, &h->d_owned0_all, all.data(), all.size()))) return rc;
    if ((rc = dev_alloc(h, (void**)&h->d_sq, sizeof(double)))) return rc;
    h->shard_committed = true;
    return AMGDD_SUCCESS;
}

int amgdd_shard_stage_counts(amgdd_handle_t h, int32_t stage, int64_t* send_counts, int64_t* recv_counts) {
    SHARD_READY(h);
    if (stage < 0 || stage >= (int)h->stage_dev.size() || !send_counts || !recv_counts) { g_detail = "stage out of range"; return AMGDD_ERR_BAD_ARG; }
    for (int q = 0; q < h->shard->nranks; ++q) { send_counts[q] = h->stage_dev[stage].send_counts[q]; recv_counts[q] = h->stage_dev[stage].recv_counts[q]; }
    return AMGDD_SUCCESS;
}

int amgdd_shard_stage_pack(amgdd_handle_t h, int32_t stage, const double* b, const double* x, double* sendbuf) {
    SHARD_READY(h);
    const ShardPlan& S = *h->shard;
    const int L = S.L;
    if (stage < 0 || stage >= (int)h->stage_dev.size() || !b || !x) { g_detail = "stage out of range or null vector"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    // the part of Alg. 2 that must precede the stage: r_l on the rows this rank owns, l = stage - 1
    if (stage >= 1 && stage <= L + 1) {
        const int l = stage - 1;
        const long long nrows = (long long)S.owned[l].size();
        if (l == 0) {
            const GlobalLevelDev& g = h->glev[0];
            int nb = 0;
            launch_residual_rows(g.a_rp, g.a_ci, g.a_v, h->d_owned_rows[0], nrows, b, x, h->d_r_all, h->d_partial, &nb, h->stream);
            launch_sum_finalize(h->d_partial, nb, h->d_sq, h->stream);
        } else {
            const GlobalLevelDev& g = h->glev[l - 1];
            launch_spmv_rows(g.r_rp, g.r_ci, g.r_v, h->d_owned_rows[l], nrows, h->d_r_all + h->r_off[l - 1], h->d_r_all + h->r_off[l], h->stream);
        }
    }
    const amgdd_handle_s::StageDev& d = h->stage_dev[stage];
    if (d.nsend > 0) {
        if (!sendbuf) { g_detail = "null send buffer"; return AMGDD_ERR_BAD_ARG; }
        launch_gather(S.stages[stage].vec == 0 ? x : h->d_r_all, d.send_pos, d.nsend, sendbuf, h->stream);
    }
    CUDA_TRY(cudaGetLastError());
    return AMGDD_SUCCESS;
}

int amgdd_shard_stage_unpack(amgdd_handle_t h, int32_t stage, double* x, const double* recvbuf) {
    SHARD_READY(h);
    if (stage < 0 || stage >= (int)h->stage_dev.size() || !x) { g_detail = "stage out of range or null vector"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    const amgdd_handle_s::StageDev& d = h->stage_dev[stage];
    if (d.nrecv > 0) {
        if (!recvbuf) { g_detail = "null receive buffer"; return AMGDD_ERR_BAD_ARG; }
        launch_scatter(recvbuf, d.recv_pos, d.nrecv, h->shard->stages[stage].vec == 0 ? x : h->d_r_all, h->stream);
    }
    CUDA_TRY(cudaGetLastError());
    return AMGDD_SUCCESS;
}

int amgdd_shard_local_solve(amgdd_handle_t h, double* x, int32_t num_fac_cycles, int32_t relax_sweeps) {
    SHARD_OK(h);
    if (!x || num_fac_cycles < 1 || relax_sweeps < 1) { g_detail = "need x non-null, num_fac_cycles >= 1, relax_sweeps >= 1"; return AMGDD_ERR_BAD_ARG; }
    DEVICE_SCOPE(h);
    const int prc = ensure_program(h, num_fac_cycles, relax_sweeps);
    if (prc) return prc;
    const FacParams prm = fac_params(h, x);
    CUDA_TRY(cudaMemsetAsync(h->d_counter, 0, sizeof(int), h->stream));
    launch_fac(prm, h->fac_cfg, h->stream);                                         // Alg. 2 P:475-479 on this rank's subdomains
    CUDA_TRY(cudaGetLastError());
    return AMGDD_SUCCESS;
}

int amgdd_shard_sqnorm(amgdd_handle_t h, double* out_host) {
    SHARD_READY(h);
    if (!out_host) return AMGDD_ERR_BAD_ARG;
    DEVICE_SCOPE(h);
    CUDA_TRY(cudaMemcpyAsync(out_host, h->d_sq, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return AMGDD_SUCCESS;
}

int amgdd_shard_owned_count(amgdd_handle_t h, int32_t rank, int64_t* count) {
    SHARD_READY(h);
    if (rank < 0 || rank >= h->shard->nranks || !count) { g_detail = "rank out of range"; return AMGDD_ERR_BAD_ARG; }
    *count = h->owned0_off[rank + 1] - h->owned0_off[rank];
    return AMGDD_SUCCESS;
}

int amgdd_shard_pack_owned(amgdd_handle_t h, const double* x, double* buf) {
    SHARD_READY(h);
    if (!x || !buf) return AMGDD_ERR_BAD_ARG;
    DEVICE_SCOPE(h);
    const int r = h->shard->rank;
    launch_gather32(x, h->d_owned0_all + h->owned0_off[r], h->owned0_off[r + 1] - h->owned0_off[r], buf, h->stream);
    CUDA_TRY(cudaGetLastError());
    return AMGDD_SUCCESS;
}

int amgdd_shard_unpack_owned(amgdd_handle_t h, int32_t src_rank, const double* buf, double* x) {
    SHARD_READY(h);
    if (!x || !buf || src_rank < 0 || src_rank >= h->shard->nranks) return AMGDD_ERR_BAD_ARG;
    DEVICE_SCOPE(h);
    launch_scatter32(buf, h->d_owned0_all + h->owned0_off[src_rank], h->owned0_off[src_rank + 1] - h->owned0_off[src_rank], x, h->stream);
    CUDA_TRY(cudaGetLastError());
    return AMGDD_SUCCESS;
}

int amgdd_pack_stream(int32_t nrows, int32_t n_real, const int32_t* rowptr32, const int32_t* colind, const double* vals,
                      const uint8_t* row_flags, int32_t wide, int32_t window, void* out, int64_t out_capacity,
                      int64_t* out_bytes, amgdd_way_t* out_ways) {
    g_detail.clear();
    if (nrows < 0 || n_real < 0 || n_real > nrows || !rowptr32 || (!colind && rowptr32[nrows] > 0) ||
        (!vals && rowptr32[nrows] > 0) || rowptr32[0] != 0 || window < SLICE_ROWS || window > MAX_WINDOW || (window % SLICE_ROWS)) {
        g_detail = "bad argument to amgdd_pack_stream";
        return AMGDD_ERR_BAD_ARG;
    }
    for (int32_t i = 0; i < nrows; ++i) {
        if (rowptr32[i + 1] < rowptr32[i]) { g_detail = "row pointers not monotone"; return AMGDD_ERR_BAD_ARG; }
        if (rowptr32[i + 1] - rowptr32[i] > 65535) { g_detail = "row " + std::to_string(i) + " has more than 65535 entries"; return AMGDD_ERR_INDEX_RANGE; }
    }
    if (!wide) {
        if (nrows > NARROW_MAX_ROWS) { g_detail = "more than 65535 rows need the wide form"; return AMGDD_ERR_BAD_ARG; }
        for (int32_t k = 0; k < rowptr32[nrows]; ++k)
            if (colind[k] < 0 || colind[k] >= NARROW_MAX_COLS) { g_detail = "column index needs the wide form"; return AMGDD_ERR_BAD_ARG; }
    }
    const PackPlan pp = plan_stream(nrows, rowptr32, wide != 0, n_real, window);
    if (out_bytes) *out_bytes = pp.bytes;
    static_assert(sizeof(amgdd_way_t) == sizeof(WayDesc), "amgdd_way_t mirrors WayDesc");
    if (out_ways) std::memcpy(out_ways, pp.way, sizeof(pp.way));
    if (out) {
        if (out_capacity < pp.bytes) { g_detail = "output buffer too small"; return AMGDD_ERR_BAD_ARG; }
        write_stream(nrows, rowptr32, colind, vals, wide != 0, n_real, window, (char*)out, row_flags);
    }
    return AMGDD_SUCCESS;
}

int amgdd_last_solve_profile(amgdd_handle_t h, double ms[4], int64_t launches[3]) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (ms) for (int i = 0; i < 4; ++i) ms[i] = h->prof_ms[i];
    if (launches) for (int i = 0; i < 3; ++i) launches[i] = h->prof_launches[i];
    return AMGDD_SUCCESS;
}

int amgdd_debug_fac_cycles(amgdd_handle_t h, int64_t out[16], int32_t reset) {
    if (bad_handle(h) || !out) return AMGDD_ERR_BAD_ARG;
    for (int i = 0; i < 16; ++i) out[i] = 0;
    if (!h->d_prof) { g_detail = "set AMGDD_FAC_PROFILE=1 before amgdd_setup"; return AMGDD_ERR_BAD_ARG; }
    const size_t cnt = (size_t)h->fac_cfg.grid * FAC_PROF_SLOTS;
    std::vector<long long> host(cnt);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    CUDA_TRY(cudaMemcpy(host.data(), h->d_prof, cnt * sizeof(long long), cudaMemcpyDeviceToHost));
    for (size_t i = 0; i < cnt; ++i) out[i % FAC_PROF_SLOTS] += host[i];
    if (reset) CUDA_TRY(cudaMemset(h->d_prof, 0, cnt * sizeof(long long)));
    return AMGDD_SUCCESS;
}

int amgdd_debug_fac_op_cycles(amgdd_handle_t h, int64_t* out, int32_t n, int32_t* kinds_levels) {
    if (bad_handle(h) || !out) return AMGDD_ERR_BAD_ARG;
    if (!h->d_prof_ops) { g_detail = "set AMGDD_FAC_PROFILE=1 before amgdd_setup"; return AMGDD_ERR_BAD_ARG; }
    const size_t cnt = (size_t)h->fac_cfg.grid * PROF_OPS_STRIDE;
    std::vector<long long> host(cnt);
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    CUDA_TRY(cudaMemcpy(host.data(), h->d_prof_ops, cnt * sizeof(long long), cudaMemcpyDeviceToHost));
    for (int i = 0; i < 4 * n; ++i) out[i] = 0;
    for (int b = 0; b < h->fac_cfg.grid; ++b)
        for (int j = 0; j < n && j < MAX_OPS; ++j)
            for (int q = 0; q < 4; ++q) out[q * n + j] += host[(size_t)b * PROF_OPS_STRIDE + q * MAX_OPS + j];
    if (kinds_levels) {
        std::vector<FacOp> ops((size_t)std::max(1, h->prog_nops));
        fac_build_program(h->H.L, h->prog_nfac, h->prog_nu, h->prog_smoother, ops.data());
        for (int j = 0; j < n && j < h->prog_nops; ++j) kinds_levels[j] = ops[j].kind * 256 + ops[j].level;
    }
    CUDA_TRY(cudaMemset(h->d_prof_ops, 0, cnt * sizeof(long long)));
    return AMGDD_SUCCESS;
}

int amgdd_debug_read_block(amgdd_handle_t h, int32_t p, int32_t level, int32_t which, void* out, int64_t out_capacity, int64_t* out_bytes) {
    if (bad_handle(h) || !out_bytes) return AMGDD_ERR_BAD_ARG;
    if (p < 0 || p >= h->P || level < 0 || level > h->H.L || which < 0 || which > 5) { g_detail = "index out of range"; return AMGDD_ERR_BAD_ARG; }
    const SubMeta& sm = h->subs[p];
    const BlockLayout& b = sm.plan.lev[level];
    i64 off = -1, bytes = 0;
    if (which == 5) { off = sm.plan.off_owned; bytes = 4LL * sm.plan.n_owned; }
    else if (!b.shared) {
        switch (which) {
            case 0: off = b.off_gid; bytes = 4LL * (b.n_real + b.n_ghost); break;
            case 1: off = b.off_dinv; bytes = 8LL * (b.n_real + b.n_ghost); break;
            case 2: off = b.A.off; bytes = b.A.bytes; break;
            case 3: off = b.P.off; bytes = b.P.bytes; break;
            default: off = b.R.off; bytes = b.R.bytes; break;
        }
    }
    *out_bytes = bytes;
    if (!out || bytes == 0) return AMGDD_SUCCESS;
    if (out_capacity < bytes) { g_detail = "out_capacity too small"; return AMGDD_ERR_BAD_ARG; }
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    CUDA_TRY(cudaMemcpy(out, sm.dev_base + off, (size_t)bytes, cudaMemcpyDeviceToHost));
    return AMGDD_SUCCESS;
}

// ---- introspection ------------------------------------------------------------------------
int amgdd_num_levels(amgdd_handle_t h, int32_t* out) {
    if (bad_handle(h) || !out) return AMGDD_ERR_BAD_ARG;
    *out = h->H.L + 1;
    return AMGDD_SUCCESS;
}

int amgdd_level_size(amgdd_handle_t h, int32_t l, int64_t* n_l, int64_t* nnzA, int64_t* nnzP) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (l < 0 || l > h->H.L) { g_detail = "level out of range"; return AMGDD_ERR_BAD_ARG; }
    if (n_l) *n_l = h->H.lv[l].A.nrows;
    if (nnzA) *nnzA = h->H.lv[l].A.nnz();
    if (nnzP) *nnzP = h->H.lv[l].P.nnz();
    return AMGDD_SUCCESS;
}

int amgdd_get_cf(amgdd_handle_t h, int32_t l, int8_t* cf) {
    if (bad_handle(h) || !cf) return AMGDD_ERR_BAD_ARG;
    if (l < 0 || l >= h->H.L) { g_detail = "level out of range (cf exists for l < L)"; return AMGDD_ERR_BAD_ARG; }
    std::copy(h->H.lv[l].cf.begin(), h->H.lv[l].cf.end(), cf);
    return AMGDD_SUCCESS;
}

int amgdd_get_level_matrix(amgdd_handle_t h, int32_t l, int32_t which, int64_t* rp, int32_t* ci, double* v) {
    if (bad_handle(h) || !rp || !ci || !v) return AMGDD_ERR_BAD_ARG;
    if (l < 0 || l > h->H.L || (which != 0 && which != 1) || (which == 1 && l == h->H.L)) {
        g_detail = "level / matrix selector out of range";
        return AMGDD_ERR_BAD_ARG;
    }
    const HostCsr& M = which == 0 ? h->H.lv[l].A : h->H.lv[l].P;
    std::copy(M.rp.begin(), M.rp.end(), rp);
    std::copy(M.ci.begin(), M.ci.end(), ci);
    std::copy(M.v.begin(), M.v.end(), v);
    return AMGDD_SUCCESS;
}

int amgdd_composite_size(amgdd_handle_t h, int32_t p, int32_t l, int64_t* n_real, int64_t* n_ghost) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (p < 0 || p >= h->P || l < 0 || l > h->H.L) { g_detail = "subdomain / level out of range"; return AMGDD_ERR_BAD_ARG; }
    const BlockLayout& b = h->subs[p].plan.lev[l];
    if (n_real) *n_real = b.n_real;
    if (n_ghost) *n_ghost = b.n_ghost;
    return AMGDD_SUCCESS;
}

int amgdd_get_composite(amgdd_handle_t h, int32_t p, int32_t l, int32_t* real_gid, int32_t* ghost_gid) {
    if (bad_handle(h)) return AMGDD_ERR_BAD_ARG;
    if (p < 0 || p >= h->P || l < 0 || l > h->H.L) { g_detail = "subdomain / level out of range"; return AMGDD_ERR_BAD_ARG; }
    const BlockLayout& b = h->subs[p].plan.lev[l];
    if (b.shared) {
        if (real_gid) for (int i = 0; i < b.n_real; ++i) real_gid[i] = i;
        return AMGDD_SUCCESS;
    }
    const char* base = h->subs[p].dev_base + b.off_gid;          // read the device copy back: what the kernels use
    if (real_gid && b.n_real) CUDA_TRY(cudaMemcpy(real_gid, base, (size_t)b.n_real * 4, cudaMemcpyDeviceToHost));
    if (ghost_gid && b.n_ghost) CUDA_TRY(cudaMemcpy(ghost_gid, base + (size_t)b.n_real * 4, (size_t)b.n_ghost * 4, cudaMemcpyDeviceToHost));
    return AMGDD_SUCCESS;
}

int amgdd_get_stats(amgdd_handle_t h, amgdd_stats_t* s) {
    if (bad_handle(h) || !s) return AMGDD_ERR_BAD_ARG;
    h->stats.device_bytes = h->device_bytes;
    *s = h->stats;
    return AMGDD_SUCCESS;
}

}  // extern "C"
