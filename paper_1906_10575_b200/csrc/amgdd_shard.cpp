// Sharding of the AMG-DD cycle over R ranks: the index sets of the residual
// communication algorithm (paper section 5; Alg. 5) and of the mat-vec halos of Alg. 2
// (P:471), built on the host.  No arithmetic of the method; independent of oracle/.
//
// A "processor" of the paper is a RANK here: rank r holds the contiguous block of subdomains
// [ceil(r P / R), ceil((r + 1) P / R)) and owns Omega_l^r, the union of their owned points on level l (level 0: the
// owner array; level l + 1: the coarse images of the C-points of Omega_l^r).  Its composite grid is the union of
// the composite grids of its subdomains (padding and coarsening commute with unions).
//
// One sharded cycle exchanges values in 2 L + 2 STAGES:
//   stage 0            x at the columns that the rank's rows of A_0 read outside Omega_0^r
//   stage 1 + l, l < L r_l at the columns that its rows of R_l read outside Omega_l^r
//   stage L + 1 + k    Alg. 5 for level l = L - k: to every rank q with a point of Omega_l^r within eta_l of Omega_l^q
//                      the residuals at Psi = { i in Omega_l^r : dist(i, Omega_l^q) <= eta_l } and at Psi_c, the
//                      composite grid built from Psi on the coarser levels (C-points of Psi, padded, and so on;
//                      the whole coarsest level, reading A5; eta_L = infinity: every rank gets all of level L)
// A position is an index into x (stage 0) or into the concatenated residual vector r_0 | r_1 | ... (all others).
//
// Redundancy: (1) a rank never announces to q a position it announced to q in an earlier Alg. 5 stage;
// (2) the RECEIVER filters what is announced to it, stage by stage and source by source in ascending rank: a
// position it owns or was already promised is reported back as redundant and the sender drops it.  The protocol
// runs once at setup (amgdd_shard_plan_send_list -> recv_filter -> apply_drop); afterwards every needed value arrives
// exactly once.
#include "amgdd_host.hpp"

#include <algorithm>
#include <cstring>

namespace amgdd {

int shard_rank_of_sub(int p, int P, int nranks) { return (int)(((i64)p * nranks) / P); }

namespace {

// points of level l within graph distance `dist` of the seeds (seeds included), appended to `out` unsorted;
// stamp[i] == ep marks membership
void pad_set(const HostCsr& A, const std::vector<i32>& seeds, int dist, std::vector<i32>& stamp, i32 ep, std::vector<i32>& out) {
    std::vector<i32> frontier, next;
    for (i32 i : seeds)
        if (stamp[i] != ep) { stamp[i] = ep; out.push_back(i); frontier.push_back(i); }
    for (int d = 0; d < dist && !frontier.empty(); ++d) {
        next.clear();
        for (i32 i : frontier)
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
                const i32 j = A.ci[k];
                if (stamp[j] != ep) { stamp[j] = ep; out.push_back(j); next.push_back(j); }
            }
        frontier.swap(next);
    }
}

}  // namespace

void shard_build(const Hierarchy& H, const i32* owner, int P, int eta, int rank, int nranks, ShardPlan& S) {
    const int L = H.L;
    S.rank = rank; S.nranks = nranks; S.L = L;
    S.sub_lo = (int)(((i64)rank * P + nranks - 1) / nranks);
    S.sub_hi = (int)(((i64)(rank + 1) * P + nranks - 1) / nranks);
    S.r_off.assign(L + 2, 0);
    for (int l = 0; l <= L; ++l) S.r_off[l + 1] = S.r_off[l] + ((H.lv[l].A.nrows + 1) & ~(i64)1);
    // ---- ownership on every level ----
    S.owner_rank.assign(L + 1, std::vector<i32>());
    S.owner_rank[0].resize((size_t)H.lv[0].A.nrows);
    for (i64 i = 0; i < H.lv[0].A.nrows; ++i) S.owner_rank[0][i] = shard_rank_of_sub(owner[i], P, nranks);
    for (int l = 0; l < L; ++l) {
        const HostLevel& lv = H.lv[l];
        S.owner_rank[l + 1].assign((size_t)H.lv[l + 1].A.nrows, -1);
        for (i64 i = 0; i < lv.A.nrows; ++i)
            if (lv.cf[i] > 0) S.owner_rank[l + 1][lv.coarse_of[i]] = S.owner_rank[l][i];
    }
    S.owned.assign(L + 1, std::vector<i32>());
    for (int l = 0; l <= L; ++l)
        for (i64 i = 0; i < H.lv[l].A.nrows; ++i)
            if (S.owner_rank[l][i] == rank) S.owned[l].push_back((i32)i);
    S.owned0_all.assign(nranks, std::vector<i32>());
    for (i64 i = 0; i < H.lv[0].A.nrows; ++i) S.owned0_all[S.owner_rank[0][i]].push_back((i32)i);
    // receiver-side record: positions this rank owns or has been promised (r space; x halo kept apart)
    S.have.assign((size_t)S.r_off[L + 1], 0);
    for (int l = 0; l <= L; ++l)
        for (i32 i : S.owned[l]) S.have[(size_t)(S.r_off[l] + i)] = 1;
    S.have_x.assign((size_t)H.lv[0].A.nrows, 0);
    for (i32 i : S.owned[0]) S.have_x[i] = 1;

    const int nstages = 2 * L + 2;
    S.stages.assign(nstages, ShardStage());
    for (ShardStage& st : S.stages) { st.send.assign(nranks, std::vector<i64>()); st.recv.assign(nranks, std::vector<i64>()); }
    // ---- mat-vec halos: stage 0 (A_0, columns of x), stage 1 + l (R_l, columns of r_l) ----
    auto halo = [&](const HostCsr& M, const std::vector<i32>& row_owner, const std::vector<i32>& col_owner, i64 base, ShardStage& st) {
        for (i64 i = 0; i < M.nrows; ++i) {
            const i32 ri = row_owner[i];
            for (i64 k = M.rp[i]; k < M.rp[i + 1]; ++k) {
                const i32 j = M.ci[k], rj = col_owner[j];
                if (ri == rj) continue;
                if (rj == rank) st.send[ri].push_back(base + j);          // rank ri reads my point j
            }
        }
        for (int q = 0; q < nranks; ++q) {
            std::vector<i64>& v = st.send[q];
            std::sort(v.begin(), v.end());
            v.erase(std::unique(v.begin(), v.end()), v.end());
        }
    };
    S.stages[0].vec = 0;
    halo(H.lv[0].A, S.owner_rank[0], S.owner_rank[0], 0, S.stages[0]);
    for (int l = 0; l < L; ++l) {
        S.stages[1 + l].vec = 1;
        halo(H.lv[l].R, S.owner_rank[l + 1], S.owner_rank[l], S.r_off[l], S.stages[1 + l]);
    }
    // ---- Alg. 5: stage L + 1 + (L - l) for l = L .. 0 ----
    std::vector<std::vector<i32>> stamp(L + 1);
    for (int l = 0; l <= L; ++l) stamp[l].assign((size_t)H.lv[l].A.nrows, 0);
    i32 epoch = 0;
    std::vector<std::vector<uint8_t>> sent(nranks);                          // redundancy (1): what I announced to q before
    for (int q = 0; q < nranks; ++q)
        if (q != rank) sent[q].assign((size_t)S.r_off[L + 1], 0);
    std::vector<i32> cur, nxt, seeds;
    for (int l = L; l >= 0; --l) {
        ShardStage& st = S.stages[L + 1 + (L - l)];
        st.vec = 1;
        for (int q = 0; q < nranks; ++q) {
            if (q == rank) continue;
            // Psi: my points within eta_l of Omega_l^q (the whole of Omega_l^r on the coarsest level)
            cur.clear();
            if (l == L) cur = S.owned[l];
            else {
                seeds.clear();
                for (i64 i = 0; i < H.lv[l].A.nrows; ++i)
                    if (S.owner_rank[l][i] == q) seeds.push_back((i32)i);
                nxt.clear();
                ++epoch;
                pad_set(H.lv[l].A, seeds, eta, stamp[l], epoch, nxt);
                for (i32 i : nxt)
                    if (S.owner_rank[l][i] == rank) cur.push_back(i);
            }
            if (cur.empty()) continue;                                        // q is not a distance-eta_l neighbour on this level
            std::sort(cur.begin(), cur.end());
            std::vector<i64>& out = st.send[q];
            auto announce = [&](int m, const std::vector<i32>& pts) {          // ascending within a level; skips what q already got from me
                for (i32 i : pts) {
                    const size_t pos = (size_t)(S.r_off[m] + i);
                    if (!sent[q][pos]) { sent[q][pos] = 1; out.push_back((i64)pos); }
                }
            };
            announce(l, cur);
            // Psi_c: the composite grid built from Psi on the coarser levels
            for (int m = l + 1; m <= L; ++m) {
                nxt.clear();
                if (m == L) {                                                  // reading A5: the whole coarsest level
                    nxt.resize((size_t)H.lv[L].A.nrows);
                    for (i64 i = 0; i < H.lv[L].A.nrows; ++i) nxt[i] = (i32)i;
                } else {
                    seeds.clear();
                    const HostLevel& lf = H.lv[m - 1];
                    for (i32 i : cur)
                        if (lf.cf[i] > 0) seeds.push_back(lf.coarse_of[i]);
                    ++epoch;
                    pad_set(H.lv[m].A, seeds, eta, stamp[m], epoch, nxt);
                    std::sort(nxt.begin(), nxt.end());
                }
                announce(m, nxt);
                cur.swap(nxt);
            }
        }
    }
}

// receiver side of redundancy (2): `announced` is what `src` will send in `stage`; positions this rank owns or was
// promised before go to `redundant`, the others become the receive list of (stage, src), in announced order
void shard_recv_filter(ShardPlan& S, int stage, int src, const i64* announced, i64 count, std::vector<i64>& redundant) {
    redundant.clear();
    std::vector<i64>& rl = S.stages[stage].recv[src];
    rl.clear();
    std::vector<uint8_t>& have = S.stages[stage].vec == 0 ? S.have_x : S.have;
    for (i64 k = 0; k < count; ++k) {
        const i64 pos = announced[k];
        if (have[(size_t)pos]) redundant.push_back(pos);
        else { have[(size_t)pos] = 1; rl.push_back(pos); }
    }
}

// sender side: remove the positions the receiver reported as redundant (both lists are in announced order)
void shard_apply_drop(ShardPlan& S, int stage, int dest, const i64* redundant, i64 count) {
    if (count == 0) return;
    std::vector<i64>& sl = S.stages[stage].send[dest];
    std::vector<i64> keep;
    keep.reserve(sl.size());
    i64 k = 0;
    for (i64 pos : sl) {
        if (k < count && redundant[k] == pos) ++k;
        else keep.push_back(pos);
    }
    sl.swap(keep);
}

}  // namespace amgdd
