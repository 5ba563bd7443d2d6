// Host-side data structures of the AMG-DD library (setup phase, runs once).
// Independent of oracle/: nothing here is shared with, included by, or derived from it.
#pragma once
#include <atomic>
#include <cstdint>
#include <exception>
#include <functional>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "amgdd_stream.hpp"

namespace amgdd {

typedef int64_t i64;
typedef int32_t i32;

struct HostCsr {
    i64 nrows = 0, ncols = 0;
    std::vector<i64> rp;
    std::vector<i32> ci;
    std::vector<double> v;
    i64 nnz() const { return rp.empty() ? 0 : rp.back(); }
};

struct HostLevel {
    HostCsr A;                   // A_l
    HostCsr P;                   // P_l (n_l x n_{l+1}); empty on the coarsest level
    HostCsr R;                   // R_l = P_l^T, stored explicitly (deterministic restriction, no atomics)
    std::vector<int8_t> cf;      // +1 C / -1 F
    std::vector<i32> coarse_of;  // fine index -> coarse index (C-points), -1 otherwise
    std::vector<double> dinv;    // 1 / sum_j |a_ij|   (S8)
};

struct Hierarchy {
    std::vector<HostLevel> lv;
    int L = 0;                   // coarsest level index
    // dense LU of A_L: P A = L U, stored column-major (lu[i + j*nL]); rowperm[i] = source row of row i
    std::vector<double> lu;
    std::vector<i32> rowperm;
    i64 nL = 0;
};

// status codes mirror include/amgdd.h (kept numeric here so this header stays free of the C ABI)
int validate_csr(i64 n, const i64* rowptr, const i32* colind, const double* vals, std::string& detail);
int build_hierarchy(HostCsr&& A0, double theta, int max_levels, int coarse_max, int nthreads, Hierarchy& H,
                    std::string& detail);

// ---- tiny fork-join helper: fn(thread_id, item) over items [0,n) with dynamic scheduling ----
inline int default_threads() {
    unsigned h = std::thread::hardware_concurrency();
    if (h == 0) h = 4;
    return (int)(h > 64 ? 64 : h);
}

// Runs body(t) on nthreads threads (t = 0 on the calling thread) and joins them.  An exception thrown by any
// body (std::bad_alloc from the scratch vectors, std::system_error from thread creation) is caught on its thread;
// the first one is re-thrown on the CALLING thread after all threads have joined, so that nothing can reach
// std::terminate and amgdd_setup can turn it into an error code (no exception crosses the C ABI).
template <class F>
void run_threads(int nthreads, F&& body) {
    std::exception_ptr first;
    std::mutex mu;
    auto guarded = [&](int t) {
        try { body(t); }
        catch (...) { std::lock_guard<std::mutex> g(mu); if (!first) first = std::current_exception(); }
    };
    std::vector<std::thread> th;
    try {
        th.reserve(nthreads > 1 ? nthreads - 1 : 0);
        for (int t = 1; t < nthreads; ++t) th.emplace_back(guarded, t);
    } catch (...) { std::lock_guard<std::mutex> g(mu); if (!first) first = std::current_exception(); }
    guarded(0);
    for (auto& x : th) x.join();
    if (first) std::rethrow_exception(first);
}

template <class F>
void parallel_for(i64 n, int nthreads, i64 chunk, F&& fn) {
    if (nthreads <= 1 || n <= chunk) {
        for (i64 i = 0; i < n; ++i) fn(0, i);
        return;
    }
    std::atomic<i64> next(0);
    std::atomic<bool> stop(false);
    run_threads(nthreads, [&](int t) {
        try {
            for (;;) {
                const i64 b = next.fetch_add(chunk);
                if (b >= n || stop.load(std::memory_order_relaxed)) break;
                const i64 e = b + chunk < n ? b + chunk : n;
                for (i64 i = b; i < e; ++i) fn(t, i);
            }
        } catch (...) { stop.store(true); throw; }
    });
}

// ---- composite grids (S6, S7) --------------------------------------------------------------
// Where one packed stream (amgdd_stream.hpp) sits inside a blob, and its ways.
struct StreamLayout {
    i64 off = -1;                // byte offset inside the blob (16-byte aligned)
    i64 bytes = 0;               // all ways: groups and slice headers
    i64 bytes_real = 0;          // groups and headers of the first row group (what a real-rows-only mat-vec reads)
    i64 padded_nnz = 0;          // entries stored, padding included
    WayDesc way[NUM_WAYS] = {};
    i32 nrows = 0;
    i64 nnz = 0;
    bool wide = false;           // uint32 column indices
};

// Sizes of one (subdomain, level) block and where its arrays sit inside the subdomain's blob.
struct BlockLayout {
    i32 n_real = 0, n_ghost = 0;
    bool shared = false;         // D_l^p = Omega_l: the single global copy of the level is used
    i64 nnzA = 0, nnzP = 0;      // local nonzeros (ghost rows of A: real columns only)
    i64 nnzA_real = 0;           // over real rows only (overhead statistic)
    i64 nnzA_ghost = 0;          // ghost rows x real columns
    i64 off_gid = -1, off_dinv = -1;     // byte offsets inside the blob; -1 where absent
    StreamLayout A, P, R;
};

struct SubdomainBlob {
    std::vector<BlockLayout> lev;     // L+1 entries
    i64 off_owned = -1;               // int32 local indices (into level-0 real) of the owned dofs
    i32 n_owned = 0;
    i64 bytes = 0;                    // blob size
    i64 dropped = 0;                  // A7 count
    i64 too_long_row = -1;            // a local row with more than 65535 entries (-1: none)
    i32 too_long_level = -1;
};

// local CSR with 32-bit offsets (what the packer takes)
struct LocalCsr {
    std::vector<i32> rp, ci;
    std::vector<double> v;
};

// Per-thread scratch for building composite grids; one instance per worker thread.
class CompositeBuilder {
public:
    CompositeBuilder(const Hierarchy& H, const std::vector<i32>& owner, const std::vector<std::vector<i32>>& owned,
                     int eta, int num_ghost, int window);
    // Phase 1: index sets, local matrices and the blob layout of subdomain p (= plan_sets, plan_matrices, layout_blob).
    void plan(int p, SubdomainBlob& out);
    // Phase 1 in parts (the device-side assembly runs only the first on the host)
    bool plan_sets(int p, SubdomainBlob& out);
    void plan_matrices(SubdomainBlob& out);
    // local indices (level 0) of the owned dofs of the subdomain planned last
    void owned_local(std::vector<i32>& out) const;
    int thin_window_of() const { return thin_window(); }
    // Phase 2: write the arrays of the subdomain planned last into dst (out.bytes bytes).
    void fill(const SubdomainBlob& plan, char* dst);
    // index sets of the subdomain planned last
    const std::vector<i32>& real(int l) const { return real_[l]; }
    const std::vector<i32>& ghost(int l) const { return ghost_[l]; }

private:
    void grow(int l, const std::vector<i32>& seed, int dist, std::vector<i32>& out);
    const Hierarchy& H_;
    const std::vector<i32>& owner_;
    const std::vector<std::vector<i32>>& owned_;
    int eta_, nghost_, window_, p_ = -1;
    // P_l and R_l have a few entries per row: their slices end after one or two groups, and every slice end
    // touches its 32 rows' vector entries; rows of one slice are kept within a few cache lines
    int thin_window() const { return window_ < THIN_WINDOW ? window_ : THIN_WINDOW; }
    std::vector<std::vector<i32>> real_, ghost_;
    std::vector<LocalCsr> A_, P_, R_;                 // local matrices of the subdomain planned last
    // epoch-stamped global->local maps, one per level
    std::vector<std::vector<i32>> loc_, stamp_;
    std::vector<i32> epoch_;
    std::vector<i32> frontier_, next_, cursor_;
    std::vector<uint8_t> flg_;
    i32 local_of(int l, i32 g) const { return stamp_[l][g] == epoch_[l] ? loc_[l][g] : -1; }
};

// offsets of the arrays inside a subdomain's blob, from the sizes in out.lev (out.n_owned set)
void layout_blob(SubdomainBlob& out);

// ---- sharding over ranks (amgdd_shard.cpp) ---------------------------------
struct ShardStage {
    int vec = 1;                               // 0: positions index x, 1: the concatenated residual vector r_0 | r_1 | ...
    std::vector<std::vector<i64>> send, recv;  // per peer rank: positions, in the order both sides agree on
    // the index protocol runs ONCE: recv_filter marks positions as held for good, so a second pass over a (stage, peer)
    // pair would report every position redundant and empty the send lists; these flags make the C ABI refuse it
    std::vector<uint8_t> filtered, dropped;    // per peer rank, sized on first use
};
struct ShardPlan {
    int rank = 0, nranks = 1, L = 0, sub_lo = 0, sub_hi = 0;
    std::vector<i64> r_off;                    // L + 2 offsets of the levels in the residual vector
    std::vector<std::vector<i32>> owner_rank;  // per level: the rank that owns each point (Omega_l^r)
    std::vector<std::vector<i32>> owned;       // per level: the points of this rank, ascending
    std::vector<std::vector<i32>> owned0_all;  // level 0: the points of every rank (all-gather of x)
    std::vector<ShardStage> stages;            // 2 L + 2
    std::vector<uint8_t> have, have_x;         // receiver side of the redundancy removal: owned or already promised
};
int shard_rank_of_sub(int p, int P, int nranks);
void shard_build(const Hierarchy& H, const i32* owner, int P, int eta, int rank, int nranks, ShardPlan& S);
void shard_recv_filter(ShardPlan& S, int stage, int src, const i64* announced, i64 count, std::vector<i64>& redundant);
void shard_apply_drop(ShardPlan& S, int stage, int dest, const i64* redundant, i64 count);

// packs a whole level matrix (the shared global copy) into a host buffer
struct PackedLevelStream {
    std::vector<char> data;
    StreamLayout lay;
};
// row_flags: M.nrows bytes (1: C-point of the rows' level) or nullptr
bool pack_global_stream(const HostCsr& M, const uint8_t* row_flags, int window, PackedLevelStream& out, i64& too_long_row);

}  // namespace amgdd
