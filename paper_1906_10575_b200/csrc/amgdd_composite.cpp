// Composite grids of one subdomain (paper P:57, eq. 1; readings S6, S7, A5-A8, A12) and
// their local matrices, built on the host by worker threads and shipped to the device as one
// contiguous "blob" per subdomain.  Independent of oracle/ (epoch-stamped maps, local matrices,
// packed streams).
//
// Local numbering of level l (S7): real points D_l^p in ascending global index get 0..n_real-1,
// ghost points D-bar_l^p \ D_l^p in ascending global index get n_real..n_real+n_ghost-1.
// Stored per private (subdomain, level):
//   gid   int32[n_bar]            global index of every local point
//   dinv  double[n_bar]           l1 diagonal inverse of the full global row (S8); 0.0 on the ghost points
//   A     packed stream, n_bar rows: real rows hold the whole global row (all columns lie in
//         D-bar_l by eq. 1); ghost rows hold only their real columns (t_l vanishes off D_l,
//         P:230, A12)
//   P     packed stream, n_bar rows, columns local to level l+1 (rows over all of D-bar_l)
//   R     packed stream, n_bar(l+1) rows, columns local to level l: the explicit transpose of the
//         local P, so restriction is a gather with a fixed summation order (no atomics)
// (stream format: amgdd_stream.hpp).  A level on which D_l^p = Omega_l (always true on L, reading
// A5) is "shared": nothing is stored for it, the single global copy of the level is used (P:57
// "each processor stores the entire coarsest grid ... may be true for a few of the coarsest grids").
#include "amgdd_host.hpp"
#include "amgdd_stream.hpp"

#include <algorithm>
#include <cstring>

namespace amgdd {

namespace {

void layout_stream(const LocalCsr& M, int nrows, int ncols, int window, int n_real, StreamLayout& s,
                   i64& too_long_row) {
    s.nrows = nrows;
    s.nnz = M.rp[nrows];
    s.wide = needs_wide(nrows, ncols);
    for (int i = 0; i < nrows && too_long_row < 0; ++i)
        if (M.rp[i + 1] - M.rp[i] > 65535) too_long_row = i;             // group counts of a slice stay small
    if (too_long_row >= 0) return;
    const PackPlan pp = plan_stream(nrows, M.rp.data(), s.wide, n_real, window);
    s.bytes = pp.bytes;
    s.bytes_real = pp.bytes_real;
    s.padded_nnz = pp.padded_nnz;
    for (int w = 0; w < NUM_WAYS; ++w) s.way[w] = pp.way[w];
}
}  // namespace

CompositeBuilder::CompositeBuilder(const Hierarchy& H, const std::vector<i32>& owner,
                                   const std::vector<std::vector<i32>>& owned, int eta, int num_ghost, int window)
    : H_(H), owner_(owner), owned_(owned), eta_(eta), nghost_(num_ghost), window_(window) {
    const int nl = H.L + 1;
    real_.resize(nl); ghost_.resize(nl); loc_.resize(nl); stamp_.resize(nl);
    A_.resize(nl); P_.resize(nl); R_.resize(nl);
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
    if (!plan_sets(p, out)) return;
    plan_matrices(out);
    layout_blob(out);
}

// Index sets D_l^p, D-bar_l^p of every level (S6, S7, eq. 1) and the sizes that follow from them alone.
// Returns false (out.bytes = 0, the offending counts in out.lev[l]) when a level would overflow 32-bit local offsets.
bool CompositeBuilder::plan_sets(int p, SubdomainBlob& out) {
    const int L = H_.L;
    p_ = p;
    out.lev.assign(L + 1, BlockLayout());
    out.dropped = 0;
    out.too_long_row = -1; out.too_long_level = -1;
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
    out.n_owned = (i32)owned_[p].size();
    for (int l = 0; l <= L; ++l) {
        BlockLayout& b = out.lev[l];
        const HostLevel& lv = H_.lv[l];
        const i32 nr = b.n_real, nb = b.n_real + b.n_ghost;
        for (i32 g : real_[l]) b.nnzA_real += lv.A.rp[g + 1] - lv.A.rp[g];
        if (b.shared) {                                                  // no ghosts, whole level
            b.nnzA = b.nnzA_real;
            b.nnzP = (l < L) ? lv.P.nnz() : 0;
            continue;
        }
        auto gid_of = [&](i32 i) { return i < nr ? real_[l][i] : ghost_[l][i - nr]; };
        // 32-bit local offsets: refuse (AMGDD_ERR_INDEX_RANGE in the caller) before anything overflows
        i64 bound = b.nnzA_real, boundP = 0;
        for (i32 g : ghost_[l]) bound += lv.A.rp[g + 1] - lv.A.rp[g];
        for (i32 i = 0; i < nb; ++i) boundP += lv.P.rp[gid_of(i) + 1] - lv.P.rp[gid_of(i)];
        if (bound > (i64)INT32_MAX || boundP > (i64)INT32_MAX) { b.nnzA = bound; b.nnzP = boundP; out.bytes = 0; return false; }
    }
    return true;
}

void CompositeBuilder::owned_local(std::vector<i32>& out) const {
    const std::vector<i32>& o = owned_[p_];
    out.resize(o.size());
    for (size_t k = 0; k < o.size(); ++k) out[k] = loc_[0][o[k]];
}

// Local matrices of the private levels (host assembly) and the plans of their streams.
void CompositeBuilder::plan_matrices(SubdomainBlob& out) {
    const int L = H_.L;
    for (int l = 0; l <= L; ++l) {
        BlockLayout& b = out.lev[l];
        const HostLevel& lv = H_.lv[l];
        const i32 nr = b.n_real, nb = b.n_real + b.n_ghost;
        if (b.shared) continue;
        auto gid_of = [&](i32 i) { return i < nr ? real_[l][i] : ghost_[l][i - nr]; };
        LocalCsr& A = A_[l];
        A.rp.assign((size_t)nb + 1, 0); A.ci.clear(); A.v.clear();
        for (i32 i = 0; i < nb; ++i) {
            const i32 g = gid_of(i);
            for (i64 k = lv.A.rp[g]; k < lv.A.rp[g + 1]; ++k) {
                const i32 c = local_of(l, lv.A.ci[k]);
                if (i < nr) { A.ci.push_back(c); A.v.push_back(lv.A.v[k]); }       // real rows: always inside (eq. 1)
                else if (c >= 0 && c < nr) { A.ci.push_back(c); A.v.push_back(lv.A.v[k]); }
            }
            A.rp[i + 1] = (i32)A.ci.size();
        }
        b.nnzA = A.rp[nb];
        b.nnzA_ghost = b.nnzA - b.nnzA_real;
        // P (columns local to level l+1) and R = local P transposed; l < L here
        const i32 nbc = out.lev[l + 1].n_real + out.lev[l + 1].n_ghost;
        LocalCsr& P = P_[l];
        LocalCsr& R = R_[l];
        P.rp.assign((size_t)nb + 1, 0); P.ci.clear(); P.v.clear();
        R.rp.assign((size_t)nbc + 1, 0);
        for (i32 i = 0; i < nb; ++i) {
            const i32 g = gid_of(i);
            for (i64 k = lv.P.rp[g]; k < lv.P.rp[g + 1]; ++k) {
                const i32 c = local_of(l + 1, lv.P.ci[k]);
                if (c >= 0) { P.ci.push_back(c); P.v.push_back(lv.P.v[k]); R.rp[c + 1]++; }
                else ++out.dropped;                                      // A7
            }
            P.rp[i + 1] = (i32)P.ci.size();
        }
        b.nnzP = P.rp[nb];
        for (i32 c = 0; c < nbc; ++c) R.rp[c + 1] += R.rp[c];            // counting sort: columns ascending
        R.ci.resize((size_t)b.nnzP); R.v.resize((size_t)b.nnzP);
        cursor_.assign(R.rp.begin(), R.rp.end() - 1);
        for (i32 i = 0; i < nb; ++i)
            for (i32 k = P.rp[i]; k < P.rp[i + 1]; ++k) {
                const i32 pos = cursor_[P.ci[k]]++;
                R.ci[pos] = i; R.v[pos] = P.v[k];
            }
        i64 bad = -1;
        layout_stream(A, nb, nb, window_, nr, b.A, bad);
        layout_stream(P, nb, nbc, thin_window(), nb, b.P, bad);
        layout_stream(R, nbc, nb, thin_window(), nbc, b.R, bad);
        if (bad >= 0 && out.too_long_row < 0) { out.too_long_row = bad; out.too_long_level = l; }
    }
}

// Where the arrays of a subdomain sit inside its blob (sizes of all streams known).
void layout_blob(SubdomainBlob& out) {
    const int L = (int)out.lev.size() - 1;
    i64 off = 0;
    auto take = [&](i64 bytes) { const i64 o = off; off = (off + bytes + 127) & ~(i64)127; return o; };   // streams need 128-byte alignment
    out.off_owned = take((i64)out.n_owned * 4);
    for (int l = 0; l <= L; ++l) {
        BlockLayout& b = out.lev[l];
        if (b.shared) continue;
        const i64 nb = (i64)b.n_real + b.n_ghost;
        b.off_gid = take(nb * 4);
        b.off_dinv = take(nb * 8);                       // n_bar entries: 0.0 on the ghost points (they never relax, A4)
        b.A.off = take(b.A.bytes);
        b.P.off = take(b.P.bytes);
        b.R.off = take(b.R.bytes);
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
        for (i32 i = nr; i < nb; ++i) dinv[i] = 0.0;                     // ghost rows never relax (A4)
        const i32 nbc = plan.lev[l + 1].n_real + plan.lev[l + 1].n_ghost;
        flg_.assign((size_t)nb, 0);                                      // C-points among the real rows (CF smoother)
        for (i32 i = 0; i < nr; ++i) flg_[i] = lv.cf[gid[i]] > 0 ? 1 : 0;
        write_stream(nb, A_[l].rp.data(), A_[l].ci.data(), A_[l].v.data(), b.A.wide, nr, window_, dst + b.A.off, flg_.data());
        write_stream(nb, P_[l].rp.data(), P_[l].ci.data(), P_[l].v.data(), b.P.wide, nb, thin_window(), dst + b.P.off);
        {   // R_l rows are the points of level l+1: flag = their C/F class
            const BlockLayout& c = plan.lev[l + 1];
            const HostLevel& lc = H_.lv[l + 1];
            flg_.assign((size_t)nbc, 0);
            for (i32 i = 0; i < c.n_real; ++i)
                if (!lc.cf.empty()) flg_[i] = lc.cf[real_[l + 1][i]] > 0 ? 1 : 0;
            write_stream(nbc, R_[l].rp.data(), R_[l].ci.data(), R_[l].v.data(), b.R.wide, nbc, thin_window(), dst + b.R.off, flg_.data());
        }
    }
}

bool pack_global_stream(const HostCsr& M, const uint8_t* row_flags, int window, PackedLevelStream& out, i64& too_long_row) {
    if (M.nnz() > (i64)INT32_MAX || M.nrows > (i64)INT32_MAX) return false;
    LocalCsr T;
    T.rp.assign(M.rp.begin(), M.rp.end());
    i64 bad = -1;
    layout_stream(T, (int)M.nrows, (int)M.ncols, window, (int)M.nrows, out.lay, bad);
    too_long_row = bad;
    if (bad >= 0) return true;
    out.data.assign((size_t)out.lay.bytes, 0);
    write_stream((int)M.nrows, T.rp.data(), M.ci.data(), M.v.data(), out.lay.wide, (int)M.nrows, window, out.data.data(), row_flags);
    return true;
}

}  // namespace amgdd
