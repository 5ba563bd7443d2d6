// AMG hierarchy on the host (setup phase): classical Ruge-Stueben strength + first-pass C/F
// colouring, direct interpolation, explicit R = P^T, Galerkin A_{l+1} = R_l A_l P_l (paper P:49),
// l1 diagonals and the dense LU of the coarsest operator.  Follows readings S1-S5, S8 of
// DESIGN.md.  Written independently of oracle/ (different data structures and algorithms:
// per-entry strength flags, bucketed bitmap colouring, threaded symbolic/numeric triple product).
#include "amgdd_host.hpp"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <memory>

namespace amgdd {

namespace {
enum { ST_OK = 0, ST_BAD_CSR = -2, ST_COARSE_TOO_LARGE = -4, ST_SINGULAR = -5 };
}

int validate_csr(i64 n, const i64* rp, const i32* ci, const double* v, std::string& detail) {
    if (rp[0] != 0) { detail = "rowptr[0] != 0"; return ST_BAD_CSR; }
    for (i64 i = 0; i < n; ++i) {
        if (rp[i + 1] < rp[i]) { detail = "rowptr not monotone at row " + std::to_string(i); return ST_BAD_CSR; }
        bool diag = false;
        for (i64 k = rp[i]; k < rp[i + 1]; ++k) {
            if (ci[k] < 0 || ci[k] >= n) { detail = "column out of range in row " + std::to_string(i); return ST_BAD_CSR; }
            if (k > rp[i] && ci[k] <= ci[k - 1]) { detail = "columns not strictly ascending in row " + std::to_string(i); return ST_BAD_CSR; }
            // the AlgFAC kernel streams the values unchecked (and orders its load bursts by an Inf/NaN test of data
            // it has already received): non-finite input is refused here
            if (!std::isfinite(v[k])) { detail = "non-finite value in row " + std::to_string(i); return ST_BAD_CSR; }
            if (ci[k] == i) {
                diag = true;
                if (!(v[k] > 0.0)) { detail = "non-positive diagonal in row " + std::to_string(i); return ST_BAD_CSR; }
            }
        }
        if (!diag) { detail = "missing diagonal in row " + std::to_string(i); return ST_BAD_CSR; }
    }
    // structural symmetry: count entries per column, then check (i,j) <-> (j,i) by binary search
    for (i64 i = 0; i < n; ++i)
        for (i64 k = rp[i]; k < rp[i + 1]; ++k) {
            const i32 j = ci[k];
            if (j == i) continue;
            const i32* b = ci + rp[j];
            const i32* e = ci + rp[j + 1];
            if (!std::binary_search(b, e, (i32)i)) {
                detail = "pattern not symmetric: (" + std::to_string(i) + "," + std::to_string(j) + ") has no mirror";
                return ST_BAD_CSR;
            }
        }
    return ST_OK;
}

namespace {

// S1: flag[k] = 1 iff entry k of A is a strong off-diagonal connection of its row.
void strength_flags(const HostCsr& A, double theta, int nthreads, std::vector<uint8_t>& flag) {
    flag.assign((size_t)A.nnz(), 0);
    parallel_for(A.nrows, nthreads, 4096, [&](int, i64 i) {
        const i64 b = A.rp[i], e = A.rp[i + 1];
        double biggest = 0.0;                          // max over off-diagonals of -a_ik, if positive
        for (i64 k = b; k < e; ++k)
            if (A.ci[k] != i && -A.v[k] > biggest) biggest = -A.v[k];
        if (biggest <= 0.0) return;
        const double cut = theta * biggest * (1.0 - 1e-10);
        for (i64 k = b; k < e; ++k)
            if (A.ci[k] != i && A.v[k] < 0.0 && -A.v[k] >= cut) flag[k] = 1;
    });
}

// A set of indices in [0, n) with "lowest member" in a few word operations: a bitmap with two summary levels.
struct IndexSet {
    std::vector<uint64_t> l0, l1, l2;
    i64 count = 0;
    explicit IndexSet(i64 n) : l0((size_t)((n + 63) >> 6), 0), l1((l0.size() + 63) >> 6, 0), l2((l1.size() + 63) >> 6, 0) {}
    void insert(i64 i) {
        const i64 w0 = i >> 6, w1 = w0 >> 6;
        l0[w0] |= 1ull << (i & 63); l1[w1] |= 1ull << (w0 & 63); l2[w1 >> 6] |= 1ull << (w1 & 63);
        ++count;
    }
    void erase(i64 i) {
        const i64 w0 = i >> 6, w1 = w0 >> 6;
        l0[w0] &= ~(1ull << (i & 63));
        if (!l0[w0]) { l1[w1] &= ~(1ull << (w0 & 63)); if (!l1[w1]) l2[w1 >> 6] &= ~(1ull << (w1 & 63)); }
        --count;
    }
    i64 lowest() const {
        for (size_t k = 0; k < l2.size(); ++k)
            if (l2[k]) {
                const i64 w1 = (i64)k * 64 + __builtin_ctzll(l2[k]);
                const i64 w0 = w1 * 64 + __builtin_ctzll(l1[w1]);
                return w0 * 64 + __builtin_ctzll(l0[w0]);
            }
        return -1;
    }
};

// S2: first pass of the RS colouring.  The undecided points sit in one IndexSet per weight lambda; the next
// C-point is the lowest index of the highest non-empty weight (lambda desc, index asc), a weight change moves
// a point to the next set.
void colour(const HostCsr& A, const std::vector<uint8_t>& strong, std::vector<int8_t>& cf) {
    const i64 n = A.nrows;
    // transpose lists of the strength graph: who strongly depends on i
    std::vector<i64> tp(n + 1, 0);
    for (i64 k = 0; k < A.nnz(); ++k) if (strong[k]) tp[A.ci[k] + 1]++;
    for (i64 i = 0; i < n; ++i) tp[i + 1] += tp[i];
    std::vector<i32> tl((size_t)tp[n]);
    {
        std::vector<i64> cur(tp.begin(), tp.end() - 1);
        for (i64 i = 0; i < n; ++i)
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k)
                if (strong[k]) tl[cur[A.ci[k]]++] = (i32)i;
    }
    std::vector<i32> weight(n);
    cf.assign(n, 0);
    std::vector<std::unique_ptr<IndexSet>> bucket;
    auto set_of = [&](i32 w) -> IndexSet& {
        if ((size_t)w >= bucket.size()) bucket.resize((size_t)w + 1);
        if (!bucket[w]) bucket[w].reset(new IndexSet(n));
        return *bucket[w];
    };
    i32 maxw = 0;
    for (i64 i = 0; i < n; ++i) {
        weight[i] = (i32)(tp[i + 1] - tp[i]);
        bool has_strong = false;
        for (i64 k = A.rp[i]; k < A.rp[i + 1] && !has_strong; ++k) has_strong = strong[k];
        if (!has_strong && weight[i] == 0) cf[i] = -1;
        else { set_of(weight[i]).insert(i); maxw = std::max(maxw, weight[i]); }
    }
    for (;;) {
        while (maxw >= 0 && ((size_t)maxw >= bucket.size() || !bucket[maxw] || bucket[maxw]->count == 0)) --maxw;
        if (maxw < 0) break;
        const i32 i = (i32)bucket[maxw]->lowest();
        bucket[maxw]->erase(i);
        cf[i] = 1;
        for (i64 a = tp[i]; a < tp[i + 1]; ++a) {
            const i32 j = tl[a];
            if (cf[j] != 0) continue;
            cf[j] = -1;
            bucket[weight[j]]->erase(j);
            for (i64 k = A.rp[j]; k < A.rp[j + 1]; ++k) {
                if (!strong[k]) continue;
                const i32 m = A.ci[k];
                if (cf[m] == 0) {
                    bucket[weight[m]]->erase(m);
                    set_of(++weight[m]).insert(m);
                    maxw = std::max(maxw, weight[m]);
                }
            }
        }
    }
}

// S3: direct interpolation.
void interpolation(const HostCsr& A, const std::vector<uint8_t>& strong, const std::vector<int8_t>& cf,
                   int nthreads, std::vector<i32>& coarse_of, HostCsr& P) {
    const i64 n = A.nrows;
    coarse_of.assign(n, -1);
    i32 nc = 0;
    for (i64 i = 0; i < n; ++i) if (cf[i] > 0) coarse_of[i] = nc++;
    P.nrows = n; P.ncols = nc;
    P.rp.assign(n + 1, 0);
    for (i64 i = 0; i < n; ++i) {
        i64 cnt = 0;
        if (cf[i] > 0) cnt = 1;
        else for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) cnt += (strong[k] && cf[A.ci[k]] > 0);
        P.rp[i + 1] = P.rp[i] + cnt;
    }
    P.ci.resize((size_t)P.rp[n]);
    P.v.resize((size_t)P.rp[n]);
    parallel_for(n, nthreads, 4096, [&](int, i64 i) {
        i64 q = P.rp[i];
        if (cf[i] > 0) { P.ci[q] = coarse_of[i]; P.v[q] = 1.0; return; }
        if (P.rp[i + 1] == q) return;                  // F-point without a strong C neighbour: empty row
        double diag = 0.0, plus = 0.0, minus = 0.0, strongC = 0.0;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
            const double a = A.v[k];
            if (A.ci[k] == i) diag = a;
            else if (a > 0.0) plus += a;
            else if (a < 0.0) minus += a;
            if (strong[k] && cf[A.ci[k]] > 0) strongC += a;
        }
        const double alpha = minus / strongC, denom = diag + plus;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k)
            if (strong[k] && cf[A.ci[k]] > 0) { P.ci[q] = coarse_of[A.ci[k]]; P.v[q] = -alpha * A.v[k] / denom; ++q; }
    });
}

void transpose_csr(const HostCsr& M, HostCsr& T) {
    T.nrows = M.ncols; T.ncols = M.nrows;
    T.rp.assign(M.ncols + 1, 0);
    const i64 nz = M.nnz();
    for (i64 k = 0; k < nz; ++k) T.rp[M.ci[k] + 1]++;
    for (i64 c = 0; c < M.ncols; ++c) T.rp[c + 1] += T.rp[c];
    T.ci.resize((size_t)nz); T.v.resize((size_t)nz);
    std::vector<i64> cur(T.rp.begin(), T.rp.end() - 1);
    for (i64 i = 0; i < M.nrows; ++i)
        for (i64 k = M.rp[i]; k < M.rp[i + 1]; ++k) {
            const i64 q = cur[M.ci[k]]++;
            T.ci[q] = (i32)i; T.v[q] = M.v[k];
        }
}

// C = X * Y with every structural entry kept, columns ascending; threaded symbolic + numeric phases.  Entry (i,c)
// accumulates x_ij * y_jc with j ascending: one fixed order, independent of the thread count.
void spgemm(const HostCsr& X, const HostCsr& Y, int nthreads, HostCsr& C) {
    const i64 n = X.nrows, m = Y.ncols;
    C.nrows = n; C.ncols = m;
    C.rp.assign(n + 1, 0);
    std::vector<std::vector<i32>> mark(nthreads);
    std::vector<std::vector<double>> acc(nthreads);
    std::vector<std::vector<i32>> cols(nthreads);
    for (int t = 0; t < nthreads; ++t) mark[t].assign(m, -1);
    parallel_for(n, nthreads, 2048, [&](int t, i64 i) {
        std::vector<i32>& mk = mark[t];
        i64 cnt = 0;
        for (i64 a = X.rp[i]; a < X.rp[i + 1]; ++a) {
            const i32 j = X.ci[a];
            for (i64 b = Y.rp[j]; b < Y.rp[j + 1]; ++b)
                if (mk[Y.ci[b]] != (i32)i) { mk[Y.ci[b]] = (i32)i; ++cnt; }
        }
        C.rp[i + 1] = cnt;
    });
    for (i64 i = 0; i < n; ++i) C.rp[i + 1] += C.rp[i];
    C.ci.resize((size_t)C.rp[n]);
    C.v.resize((size_t)C.rp[n]);
    for (int t = 0; t < nthreads; ++t) { mark[t].assign(m, -1); acc[t].assign(m, 0.0); }
    parallel_for(n, nthreads, 2048, [&](int t, i64 i) {
        std::vector<i32>& mk = mark[t];
        std::vector<double>& ac = acc[t];
        std::vector<i32>& cl = cols[t];
        cl.clear();
        for (i64 a = X.rp[i]; a < X.rp[i + 1]; ++a) {
            const i32 j = X.ci[a];
            const double xv = X.v[a];
            for (i64 b = Y.rp[j]; b < Y.rp[j + 1]; ++b) {
                const i32 c = Y.ci[b];
                if (mk[c] != (i32)i) { mk[c] = (i32)i; cl.push_back(c); ac[c] = xv * Y.v[b]; }
                else ac[c] += xv * Y.v[b];
            }
        }
        std::sort(cl.begin(), cl.end());
        i64 q = C.rp[i];
        for (i32 c : cl) { C.ci[q] = c; C.v[q] = ac[c]; ++q; }
    });
}

// Galerkin operator A_{l+1} = R_l A_l P_l (reading S4: every structural entry kept, the terms of an entry
// summed "in any order").  DEFAULT: two sparse products, R (A P): entry (I,J) = sum_i r_Ii (sum_j a_ij p_jJ), an
// association and a rounding of its own (it is NOT the order of the oracle's triple loop, so parity is shown with
// coarse operators that differ from the oracle's in the last bits).  AMGDD_GALERKIN=fused selects the one-pass
// triple product below, whose terms (r_Ii a_ij) p_jJ are added with i, then j, then J ascending.
// Fused variant: Galerkin triple product C = R A P in one pass per coarse row, every structural entry kept,
// columns ascending; threaded symbolic + numeric phases.  Entry (I,J) accumulates the terms
// (r_Ii * a_ij) * p_jJ with i, then j, then J ascending, a fixed order, so the coarse operators
// do not depend on the thread count.
void galerkin_rap(const HostCsr& R, const HostCsr& A, const HostCsr& P, int nthreads, HostCsr& C) {
    const i64 nc = R.nrows;
    C.nrows = nc; C.ncols = nc;
    C.rp.assign(nc + 1, 0);
    std::vector<std::vector<i32>> mark(nthreads);
    std::vector<std::vector<double>> acc(nthreads);
    std::vector<std::vector<i32>> cols(nthreads);
    for (int t = 0; t < nthreads; ++t) mark[t].assign(nc, -1);
    parallel_for(nc, nthreads, 512, [&](int t, i64 I) {
        std::vector<i32>& mk = mark[t];
        i64 cnt = 0;
        for (i64 a = R.rp[I]; a < R.rp[I + 1]; ++a) {
            const i32 i = R.ci[a];
            for (i64 b = A.rp[i]; b < A.rp[i + 1]; ++b) {
                const i32 j = A.ci[b];
                for (i64 c = P.rp[j]; c < P.rp[j + 1]; ++c)
                    if (mk[P.ci[c]] != (i32)I) { mk[P.ci[c]] = (i32)I; ++cnt; }
            }
        }
        C.rp[I + 1] = cnt;
    });
    for (i64 I = 0; I < nc; ++I) C.rp[I + 1] += C.rp[I];
    C.ci.resize((size_t)C.rp[nc]);
    C.v.resize((size_t)C.rp[nc]);
    for (int t = 0; t < nthreads; ++t) { mark[t].assign(nc, -1); acc[t].assign(nc, 0.0); }
    parallel_for(nc, nthreads, 512, [&](int t, i64 I) {
        std::vector<i32>& mk = mark[t];
        std::vector<double>& ac = acc[t];
        std::vector<i32>& cl = cols[t];
        cl.clear();
        for (i64 a = R.rp[I]; a < R.rp[I + 1]; ++a) {
            const i32 i = R.ci[a];
            const double rv = R.v[a];
            for (i64 b = A.rp[i]; b < A.rp[i + 1]; ++b) {
                const i32 j = A.ci[b];
                const double ra = rv * A.v[b];
                for (i64 c = P.rp[j]; c < P.rp[j + 1]; ++c) {
                    const i32 J = P.ci[c];
                    if (mk[J] != (i32)I) { mk[J] = (i32)I; cl.push_back(J); ac[J] = 0.0; }
                    ac[J] += ra * P.v[c];
                }
            }
        }
        std::sort(cl.begin(), cl.end());
        i64 q = C.rp[I];
        for (i32 J : cl) { C.ci[q] = J; C.v[q] = ac[J]; ++q; }
    });
}

void l1_diagonal(const HostCsr& A, int nthreads, std::vector<double>& dinv) {
    dinv.resize((size_t)A.nrows);
    parallel_for(A.nrows, nthreads, 8192, [&](int, i64 i) {
        double s = 0.0;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) s += std::fabs(A.v[k]);
        dinv[i] = 1.0 / s;
    });
}

// column-major right-looking LU with partial pivoting; rowperm[i] = original row now in position i
bool factor_dense(const HostCsr& A, std::vector<double>& lu, std::vector<i32>& rowperm) {
    const i64 n = A.nrows;
    lu.assign((size_t)(n * n), 0.0);
    for (i64 i = 0; i < n; ++i)
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) lu[(size_t)(i + A.ci[k] * n)] = A.v[k];
    rowperm.resize(n);
    for (i64 i = 0; i < n; ++i) rowperm[i] = (i32)i;
    for (i64 c = 0; c < n; ++c) {
        i64 piv = c;
        double big = std::fabs(lu[(size_t)(c + c * n)]);
        for (i64 i = c + 1; i < n; ++i) {
            const double a = std::fabs(lu[(size_t)(i + c * n)]);
            if (a > big) { big = a; piv = i; }
        }
        if (big == 0.0) return false;
        if (piv != c) {
            for (i64 j = 0; j < n; ++j) std::swap(lu[(size_t)(c + j * n)], lu[(size_t)(piv + j * n)]);
            std::swap(rowperm[c], rowperm[piv]);
        }
        const double d = lu[(size_t)(c + c * n)];
        for (i64 i = c + 1; i < n; ++i) lu[(size_t)(i + c * n)] /= d;
        for (i64 j = c + 1; j < n; ++j) {
            const double ucj = lu[(size_t)(c + j * n)];
            if (ucj == 0.0) continue;
            for (i64 i = c + 1; i < n; ++i) lu[(size_t)(i + j * n)] -= lu[(size_t)(i + c * n)] * ucj;
        }
    }
    return true;
}

}  // namespace

int build_hierarchy(HostCsr&& A0, double theta, int max_levels, int coarse_max, int nthreads, Hierarchy& H,
                    std::string& detail) {
    typedef std::chrono::steady_clock Clock;
    const char* tenv = std::getenv("AMGDD_SETUP_TIMING");                        // 1: stage times per level on stderr
    const bool timing = tenv && tenv[0] == '1';
    const char* genv = std::getenv("AMGDD_GALERKIN");                            // "fused": one-pass triple product (see galerkin_rap)
    const bool fused_rap = genv && std::string(genv) == "fused";
    H.lv.clear();
    H.lv.emplace_back();
    H.lv[0].A = std::move(A0);
    int l = 0;
    for (;;) {
        HostLevel& cur = H.lv[l];
        l1_diagonal(cur.A, nthreads, cur.dinv);
        const i64 n = cur.A.nrows;
        if (n <= coarse_max || l + 1 >= max_levels) break;                       // S5
        const auto t0 = Clock::now();
        std::vector<uint8_t> strong;
        strength_flags(cur.A, theta, nthreads, strong);
        const auto t1 = Clock::now();
        std::vector<int8_t> cf;
        colour(cur.A, strong, cf);
        const auto t2 = Clock::now();
        i64 nc = 0;
        for (i64 i = 0; i < n; ++i) nc += cf[i] > 0;
        if (nc == 0 || nc == n) break;                                           // S5
        cur.cf = std::move(cf);
        interpolation(cur.A, strong, cur.cf, nthreads, cur.coarse_of, cur.P);
        const auto t3 = Clock::now();
        transpose_csr(cur.P, cur.R);
        const auto t4 = Clock::now();
        HostCsr Ac;
        if (fused_rap) galerkin_rap(cur.R, cur.A, cur.P, nthreads, Ac);
        else {
            HostCsr AP;
            spgemm(cur.A, cur.P, nthreads, AP);
            spgemm(cur.R, AP, nthreads, Ac);
        }
        if (timing) {
            const auto t5 = Clock::now();
            auto sec = [](Clock::time_point a, Clock::time_point b) { return std::chrono::duration<double>(b - a).count(); };
            std::fprintf(stderr, "amgdd setup: level %d n %lld nnz %lld: strength %.3f colour %.3f interpolation %.3f transpose %.3f rap %.3f s\n",
                         l, (long long)n, (long long)cur.A.nnz(), sec(t0, t1), sec(t1, t2), sec(t2, t3), sec(t3, t4), sec(t4, t5));
        }
        for (double a : Ac.v)
            if (!std::isfinite(a)) { detail = "the Galerkin operator of level " + std::to_string(l + 1) + " has a non-finite entry"; return ST_BAD_CSR; }
        H.lv.emplace_back();
        H.lv[l + 1].A = std::move(Ac);
        ++l;
    }
    H.L = l;
    H.nL = H.lv[l].A.nrows;
    if (H.nL > 4096) {
        detail = "coarsest level has " + std::to_string(H.nL) + " dofs (> 4096)";
        return ST_COARSE_TOO_LARGE;
    }
    if (!factor_dense(H.lv[l].A, H.lu, H.rowperm)) { detail = "zero pivot in the coarsest-level LU"; return ST_SINGULAR; }
    return ST_OK;
}

}  // namespace amgdd
