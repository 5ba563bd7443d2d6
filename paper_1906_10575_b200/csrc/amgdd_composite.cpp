// Composite grids of one subdomain (paper P:57, eq. 1; readings S6, S7, A5-A8, A12) and
// their local CSR blocks, built on the host by worker threads and shipped to the device as one
// contiguous "blob" per subdomain.  Independent of oracle/ (epoch-stamped maps, local matrices).
//
// Local numbering of level l (S7): real points D_l^p in ascending global index get 0..n_real-1,
// ghost points D-bar_l^p \ D_l^p in ascending global index get n_real..n_real+n_ghost-1.
// Blocks stored per private (subdomain, level):
//   gid   int32[n_bar]            global index of every local point
//   dinv  double[n_real]          l1 diagonal of the full global row (S8)
//   A     CSR, n_bar rows: real rows hold the whole global row (all columns lie in D-bar_l by
//         eq. 1); ghost rows hold only their real columns (t_l vanishes off D_l, A12)
//   P     CSR, n_bar rows, columns local to level l+1 (rows over all of D-bar_l)
//   R     CSR, n_bar(l+1) rows, columns local to level l: the explicit transpose of the local P,
//         so restriction is a gather with a fixed summation order (no atomics)
// A level on which D_l^p = Omega_l (always true on L, reading A5) is "shared": nothing is stored
// for it, the single global copy of the level is used ("each processor stores the entire
// coarsest grid ... may be true for a few of the coarsest grids").
#include "amgdd_host.hpp"

#include <algorithm>
#include <cstring>

namespace amgdd {

namespace {
inline i64 align16(i64 x) { return (x + 15) & ~(i64)15; }
}

CompositeBuilder::CompositeBuilder(const Hierarchy& H, const std::vector<i32>& owner,
                                   const std::vector<std::vector<i32>>& owned, int eta, int num_ghost)
    : H_(H), owner_(owner), owned_(owned), eta_(eta), nghost_(num_ghost) {
    const int nl = H.L + 1;
    real_.resize(nl); ghost_.resize(nl); loc_.resize(nl); stamp_.resize(nl);
    epoch_.assign(nl, 0);
    for (int l = 0; l < nl; ++l) {
        loc_[l].assign((size_t)H.lv[l].A.nrows, -1);
        stamp_[l].assign((size_t)H.lv[l].A.nrows, 0);
    }
}

// Breadth-first growth by `dist` edges from `seed` (already stamped); newly reached points are
// appended to `out` (unsorted) and stamped with a placeholder local index.
void CompositeBuilder::grow(int l, const std::vector<i32>& seed, int dist, std::vector<i32>& out) {
    const HostCsr& A = H_.lv[l].A;
    const i32 ep = epoch_[l];
    frontier_ = seed;
    for (int d = 0; d < dist && !frontier_.empty(); ++d) {
        next_.clear();
        for (i32 i : frontier_)
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
                const i32 j = A.ci[k];
                if (stamp_[l][j] != ep) { stamp_[l][j] = ep; loc_[l][j] = -2; next_.push_back(j); out.push_back(j); }
            }
        frontier_.swap(next_);
    }
}

void CompositeBuilder::plan(int p, SubdomainBlob& out) {
    const int L = H_.L;
    p_ = p;
    out.lev.assign(L + 1, BlockLayout());
    out.dropped = 0;
    std::vector<i32> seed = owned_[p];                                   // B_0^p = Omega_0^p
    for (int l = 0; l <= L; ++l) {
        const i64 nl = H_.lv[l].A.nrows;
        BlockLayout& b = out.lev[l];
        if (++epoch_[l] == INT32_MAX) { std::fill(stamp_[l].begin(), stamp_[l].end(), 0); epoch_[l] = 1; }
        const i32 ep = epoch_[l];
        std::vector<i32>& re = real_[l];
        std::vector<i32>& gh = ghost_[l];
        re.clear(); gh.clear();
        if (l == L) {                                                    // A5: D_L = Omega_L, no ghosts
            re.resize((size_t)nl);
            for (i64 i = 0; i < nl; ++i) { re[i] = (i32)i; stamp_[l][i] = ep; loc_[l][i] = (i32)i; }
        } else {
            for (i32 i : seed) { stamp_[l][i] = ep; loc_[l][i] = -2; }
            re = seed;
            grow(l, seed, eta_, re);                                     // D_l^p
            std::sort(re.begin(), re.end());
            for (size_t k = 0; k < re.size(); ++k) loc_[l][re[k]] = (i32)k;
            grow(l, re, nghost_, gh);                                    // D-bar_l^p \ D_l^p
            std::sort(gh.begin(), gh.end());
            for (size_t k = 0; k < gh.size(); ++k) loc_[l][gh[k]] = (i32)(re.size() + k);
            seed.clear();                                                // B_{l+1}^p
            const HostLevel& lv = H_.lv[l];
            for (i32 i : re) if (lv.cf[i] > 0) seed.push_back(lv.coarse_of[i]);
        }
        b.n_real = (i32)re.size();
        b.n_ghost = (i32)gh.size();
        b.shared = ((i64)re.size() == nl);
    }
    // sizes
    for (int l = 0; l <= L; ++l) {
        BlockLayout& b = out.lev[l];
        const HostLevel& lv = H_.lv[l];
        const i32 nr = b.n_real;
        for (i32 g : real_[l]) b.nnzA_real += lv.A.rp[g + 1] - lv.A.rp[g];
        for (i32 g : ghost_[l])
            for (i64 k = lv.A.rp[g]; k < lv.A.rp[g + 1]; ++k) {
                const i32 c = local_of(l, lv.A.ci[k]);
                b.nnzA_ghost += (c >= 0 && c < nr);
            }
        b.nnzA = b.nnzA_real + b.nnzA_ghost;
        if (l < L) {
            auto count_rows = [&](const std::vector<i32>& rows) {
                for (i32 g : rows)
                    for (i64 k = lv.P.rp[g]; k < lv.P.rp[g + 1]; ++k) {
                        if (local_of(l + 1, lv.P.ci[k]) >= 0) ++b.nnzP;
                        else ++out.dropped;                              // A7
                    }
            };
            count_rows(real_[l]);
            count_rows(ghost_[l]);
        }
    }
    // layout
    i64 off = 0;
    auto take = [&](i64 bytes) { const i64 o = off; off = align16(off + bytes); return o; };
    out.n_owned = (i32)owned_[p].size();
    out.off_owned = take((i64)out.n_owned * 4);
    for (int l = 0; l <= L; ++l) {
        BlockLayout& b = out.lev[l];
        if (b.shared) continue;
        const i64 nb = (i64)b.n_real + b.n_ghost;
        const i64 nbc = (i64)out.lev[l + 1].n_real + out.lev[l + 1].n_ghost;    // l < L here
        b.off_gid = take(nb * 4);
        b.off_dinv = take((i64)b.n_real * 8);
        b.off_a_rp = take((nb + 1) * 4);
        b.off_a_ci = take(b.nnzA * 4);
        b.off_a_v = take(b.nnzA * 8);
        b.off_p_rp = take((nb + 1) * 4);
        b.off_p_ci = take(b.nnzP * 4);
        b.off_p_v = take(b.nnzP * 8);
        b.off_r_rp = take((nbc + 1) * 4);
        b.off_r_ci = take(b.nnzP * 4);
        b.off_r_v = take(b.nnzP * 8);
    }
    out.bytes = off;
}

void CompositeBuilder::fill(const SubdomainBlob& plan, char* dst) {
    const int L = H_.L;
    {
        i32* own = (i32*)(dst + plan.off_owned);
        const std::vector<i32>& o = owned_[p_];
        for (size_t k = 0; k < o.size(); ++k) own[k] = loc_[0][o[k]];
    }
    std::vector<i32> cursor;
    for (int l = 0; l <= L; ++l) {
        const BlockLayout& b = plan.lev[l];
        if (b.shared) continue;
        const HostLevel& lv = H_.lv[l];
        const i32 nr = b.n_real, ng = b.n_ghost, nb = nr + ng;
        i32* gid = (i32*)(dst + b.off_gid);
        std::memcpy(gid, real_[l].data(), (size_t)nr * 4);
        std::memcpy(gid + nr, ghost_[l].data(), (size_t)ng * 4);
        double* dinv = (double*)(dst + b.off_dinv);
        for (i32 i = 0; i < nr; ++i) dinv[i] = lv.dinv[gid[i]];
        // A
        i32* arp = (i32*)(dst + b.off_a_rp);
        i32* aci = (i32*)(dst + b.off_a_ci);
        double* av = (double*)(dst + b.off_a_v);
        i32 q = 0;
        for (i32 i = 0; i < nb; ++i) {
            arp[i] = q;
            const i32 g = gid[i];
            for (i64 k = lv.A.rp[g]; k < lv.A.rp[g + 1]; ++k) {
                const i32 c = loc_[l][lv.A.ci[k]];                       // real rows: always stamped (eq. 1)
                if (i < nr) { aci[q] = c; av[q] = lv.A.v[k]; ++q; }
                else {
                    const i32 cc = local_of(l, lv.A.ci[k]);
                    if (cc >= 0 && cc < nr) { aci[q] = cc; av[q] = lv.A.v[k]; ++q; }
                }
            }
        }
        arp[nb] = q;
        // P (columns local to level l+1)
        const i32 nbc = plan.lev[l + 1].n_real + plan.lev[l + 1].n_ghost;
        i32* prp = (i32*)(dst + b.off_p_rp);
        i32* pci = (i32*)(dst + b.off_p_ci);
        double* pv = (double*)(dst + b.off_p_v);
        i32* rrp = (i32*)(dst + b.off_r_rp);
        i32* rci = (i32*)(dst + b.off_r_ci);
        double* rv = (double*)(dst + b.off_r_v);
        std::memset(rrp, 0, (size_t)(nbc + 1) * 4);
        q = 0;
        for (i32 i = 0; i < nb; ++i) {
            prp[i] = q;
            const i32 g = gid[i];
            for (i64 k = lv.P.rp[g]; k < lv.P.rp[g + 1]; ++k) {
                const i32 c = local_of(l + 1, lv.P.ci[k]);
                if (c >= 0) { pci[q] = c; pv[q] = lv.P.v[k]; ++q; rrp[c + 1]++; }
            }
        }
        prp[nb] = q;
        // R = local P transposed (counting sort: columns come out ascending)
        for (i32 c = 0; c < nbc; ++c) rrp[c + 1] += rrp[c];
        cursor.assign(rrp, rrp + nbc);
        for (i32 i = 0; i < nb; ++i)
            for (i32 k = prp[i]; k < prp[i + 1]; ++k) {
                const i32 pos = cursor[pci[k]]++;
                rci[pos] = i; rv[pos] = pv[k];
            }
    }
}

}  // namespace amgdd
