// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU implementation of the AMG-DD hot
// path (Mitchell, Strzodka, Falgout, arXiv 1906.10575), written from the paper.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may call this.  It
// shares no code with paper_1906_10575_b200/ (the CUDA path) and neither includes the other.
//
// Citations "P:NNN" are line numbers of /root/reference/PAPER.md; "S1..S8", "A1..A20" are the
// readings listed in SURVEY.md §8(c) and restated in DESIGN.md.
//
// Structure: everything works on the GLOBAL level matrices A_l, P_l.  A subdomain's composite
// grid is two sorted index lists per level (real D_l, ghost D-bar_l \ D_l) and a scratch
// global->local array; no local matrices are ever formed.  There is no blocking, fusion or
// reordering beyond what Alg. 2 and Alg. 4 state.
//
// Parity pins (tests/test_oracle_pins.py): 1D Poisson closed form for S1-S4; brute-force graph
// distances for S6; masked global V-cycle for Alg. 4; P=1 => V(nu,nu)-cycle; Jacobi
// eigenvalues for the relaxation; dense LU for the whole solve; mat-vec counts of P:53/P:232;
// the overhead definition of P:293-299.  No function here is "parity unpinned".
#include <algorithm>
#include <cassert>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <memory>
#include <set>
#include <utility>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef int64_t i64;
typedef int32_t i32;

namespace {

struct Csr {
    i64 nrows = 0, ncols = 0;
    std::vector<i64> rp;
    std::vector<i32> ci;
    std::vector<double> v;
    i64 nnz() const { return rp.empty() ? 0 : rp.back(); }
};

struct Level {
    Csr A;                      // A_l
    Csr P;                      // P_l : n_l x n_{l+1}; empty on the coarsest level
    std::vector<int8_t> cf;     // +1 C, -1 F (empty on the coarsest level)
    std::vector<i32> cidx;      // coarse index of a C-point, -1 otherwise
    std::vector<double> dinv;   // S8: 1 / sum_j |a_ij|
};

struct Comp {                   // one subdomain's composite grid (eq. 1)
    std::vector<std::vector<i32>> real, ghost;   // per level, ascending global index (S7)
};

struct Counters { i64 A = 0, P = 0, R = 0; };

struct Oracle {
    std::vector<Level> lev;
    int L = 0;                  // index of the coarsest level
    std::vector<double> lu;     // dense LU of A_L, row-major, partial pivoting
    std::vector<i32> piv;
    // decomposition
    int nsub = 0, eta = 0, nghost = 1;
    std::vector<i32> owner;
    std::vector<std::vector<i32>> owned;          // B_0^p = Omega_0^p
    std::vector<std::unique_ptr<Comp>> comp;      // built lazily, one per subdomain
    i64 dropped = 0;            // A7: P entries of composite rows that fall outside D-bar_{l+1}
    Counters cnt;               // mat-vec counters
    int smoother = 0;           // 0: l1-Jacobi (BASELINE), 1: CF l1-Jacobi (C then F before, F then C after the coarse correction)
};

// ------------------------------------------------------------------------------------------
// S1  strength of connection (classical RS, threshold theta; "strong influence")
// ------------------------------------------------------------------------------------------
void strength(const Csr& A, double theta, std::vector<i64>& srp, std::vector<i32>& sci) {
    const i64 n = A.nrows;
    srp.assign(n + 1, 0);
    sci.clear();
    for (i64 i = 0; i < n; ++i) {
        double m = -INFINITY;
        bool any = false;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k)
            if (A.ci[k] != i) { m = std::max(m, -A.v[k]); any = true; }
        if (any && m > 0.0) {
            const double thr = theta * m * (1.0 - 1e-10);     // A9: relative slack for ties
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k)
                if (A.ci[k] != i && -A.v[k] > 0.0 && -A.v[k] >= thr) sci.push_back(A.ci[k]);
        }
        srp[i + 1] = (i64)sci.size();
    }
}

void transpose_pattern(i64 nrows, i64 ncols, const std::vector<i64>& rp, const std::vector<i32>& ci,
                       std::vector<i64>& trp, std::vector<i32>& tci) {
    trp.assign(ncols + 1, 0);
    for (i32 c : ci) trp[c + 1]++;
    for (i64 c = 0; c < ncols; ++c) trp[c + 1] += trp[c];
    tci.resize(ci.size());
    std::vector<i64> pos(trp.begin(), trp.end() - 1);
    for (i64 i = 0; i < nrows; ++i)
        for (i64 k = rp[i]; k < rp[i + 1]; ++k) tci[pos[ci[k]]++] = (i32)i;   // rows ascending
}

// ------------------------------------------------------------------------------------------
// S2  C/F splitting: first pass of the Ruge-Stueben colouring, ties to the smallest index
// ------------------------------------------------------------------------------------------
void cf_split(i64 n, const std::vector<i64>& srp, const std::vector<i32>& sci,
              const std::vector<i64>& trp, const std::vector<i32>& tci, std::vector<int8_t>& cf) {
    cf.assign(n, 0);                                      // 0 = undecided
    std::vector<i64> lam(n);
    std::set<std::pair<i64, i32>> q;                      // (-lambda, index): begin() = max lambda, min index
    for (i64 i = 0; i < n; ++i) {
        lam[i] = trp[i + 1] - trp[i];
        if (srp[i + 1] == srp[i] && lam[i] == 0) cf[i] = -1;
        else q.insert({-lam[i], (i32)i});
    }
    while (!q.empty()) {
        const i32 i = q.begin()->second;
        q.erase(q.begin());
        cf[i] = 1;
        for (i64 a = trp[i]; a < trp[i + 1]; ++a) {       // j in S_i^T, ascending
            const i32 j = tci[a];
            if (cf[j] != 0) continue;
            cf[j] = -1;
            q.erase({-lam[j], j});
            for (i64 b = srp[j]; b < srp[j + 1]; ++b) {   // k in S_j
                const i32 k = sci[b];
                if (cf[k] != 0) continue;
                q.erase({-lam[k], k});
                lam[k] += 1;
                q.insert({-lam[k], k});
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// S3  direct interpolation (injection at C-points, weights at F-points from distance-1 C)
// ------------------------------------------------------------------------------------------
void direct_interp(const Csr& A, const std::vector<i64>& srp, const std::vector<i32>& sci,
                   const std::vector<int8_t>& cf, std::vector<i32>& cidx, Csr& P) {
    const i64 n = A.nrows;
    cidx.assign(n, -1);
    i32 nc = 0;
    for (i64 i = 0; i < n; ++i) if (cf[i] == 1) cidx[i] = nc++;
    P = Csr();
    P.nrows = n; P.ncols = nc;
    P.rp.assign(n + 1, 0);
    for (i64 i = 0; i < n; ++i) {
        if (cf[i] == 1) {
            P.ci.push_back(cidx[i]); P.v.push_back(1.0);
        } else {
            double aii = 0.0, pos = 0.0, neg = 0.0, sumC = 0.0;
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
                if (A.ci[k] == i) aii = A.v[k];
                else if (A.v[k] > 0.0) pos += A.v[k];
                else if (A.v[k] < 0.0) neg += A.v[k];
            }
            // C_i = S_i intersect C ; both lists ascending -> merge
            std::vector<i64> ks;
            i64 b = srp[i];
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
                while (b < srp[i + 1] && sci[b] < A.ci[k]) ++b;
                if (b < srp[i + 1] && sci[b] == A.ci[k] && cf[A.ci[k]] == 1) { ks.push_back(k); sumC += A.v[k]; }
            }
            if (!ks.empty()) {
                const double d = aii + pos;               // A11: positive off-diagonals lumped
                const double alpha = neg / sumC;
                for (i64 k : ks) { P.ci.push_back(cidx[A.ci[k]]); P.v.push_back(-alpha * A.v[k] / d); }
            }
        }
        P.rp[i + 1] = (i64)P.ci.size();
    }
}

Csr transpose(const Csr& M) {
    Csr T;
    T.nrows = M.ncols; T.ncols = M.nrows;
    T.rp.assign(M.ncols + 1, 0);
    for (i32 c : M.ci) T.rp[c + 1]++;
    for (i64 c = 0; c < M.ncols; ++c) T.rp[c + 1] += T.rp[c];
    T.ci.resize(M.ci.size()); T.v.resize(M.v.size());
    std::vector<i64> pos(T.rp.begin(), T.rp.end() - 1);
    for (i64 i = 0; i < M.nrows; ++i)
        for (i64 k = M.rp[i]; k < M.rp[i + 1]; ++k) {
            const i64 q = pos[M.ci[k]]++;
            T.ci[q] = (i32)i; T.v[q] = M.v[k];
        }
    return T;
}

// ------------------------------------------------------------------------------------------
// S4  Galerkin product A_{l+1} = P^T A P, every structural entry kept
// ------------------------------------------------------------------------------------------
Csr galerkin(const Csr& A, const Csr& P) {
    const Csr R = transpose(P);                           // R_l = P_l^T
    const i64 nc = P.ncols;
    Csr C;
    C.nrows = nc; C.ncols = nc;
    C.rp.assign(nc + 1, 0);
    std::vector<double> acc(nc, 0.0);
    std::vector<char> mark(nc, 0);
    std::vector<i32> cols;
    for (i64 I = 0; I < nc; ++I) {
        cols.clear();
        for (i64 a = R.rp[I]; a < R.rp[I + 1]; ++a) {
            const i32 i = R.ci[a];
            const double r = R.v[a];
            for (i64 b = A.rp[i]; b < A.rp[i + 1]; ++b) {
                const i32 j = A.ci[b];
                const double ra = r * A.v[b];
                for (i64 c = P.rp[j]; c < P.rp[j + 1]; ++c) {
                    const i32 J = P.ci[c];
                    if (!mark[J]) { mark[J] = 1; cols.push_back(J); }
                    acc[J] += ra * P.v[c];
                }
            }
        }
        std::sort(cols.begin(), cols.end());
        for (i32 J : cols) { C.ci.push_back(J); C.v.push_back(acc[J]); acc[J] = 0.0; mark[J] = 0; }
        C.rp[I + 1] = (i64)C.ci.size();
    }
    return C;
}

// S8  l1 diagonal: D_ii = sum_j |a_ij| over the full row (ref. 23; reading A2)
void l1_dinv(const Csr& A, std::vector<double>& dinv) {
    dinv.resize(A.nrows);
    for (i64 i = 0; i < A.nrows; ++i) {
        double s = 0.0;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) s += std::fabs(A.v[k]);
        dinv[i] = 1.0 / s;
    }
}

// dense LU with partial pivoting (Gaussian elimination, "a direct method such as ...")
bool dense_lu(int n, std::vector<double>& a, std::vector<i32>& piv) {
    piv.resize(n);
    for (int k = 0; k < n; ++k) {
        int p = k;
        double best = std::fabs(a[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i)
            if (std::fabs(a[(size_t)i * n + k]) > best) { best = std::fabs(a[(size_t)i * n + k]); p = i; }
        piv[k] = p;
        if (best == 0.0) return false;
        if (p != k) for (int j = 0; j < n; ++j) std::swap(a[(size_t)k * n + j], a[(size_t)p * n + j]);
        for (int i = k + 1; i < n; ++i) {
            const double m = a[(size_t)i * n + k] / a[(size_t)k * n + k];
            a[(size_t)i * n + k] = m;
            for (int j = k + 1; j < n; ++j) a[(size_t)i * n + j] -= m * a[(size_t)k * n + j];
        }
    }
    return true;
}

void dense_lu_solve(int n, const std::vector<double>& a, const std::vector<i32>& piv, double* x) {
    for (int k = 0; k < n; ++k) if (piv[k] != k) std::swap(x[k], x[piv[k]]);
    for (int i = 1; i < n; ++i) {
        double s = x[i];
        for (int j = 0; j < i; ++j) s -= a[(size_t)i * n + j] * x[j];
        x[i] = s;
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = x[i];
        for (int j = i + 1; j < n; ++j) s -= a[(size_t)i * n + j] * x[j];
        x[i] = s / a[(size_t)i * n + i];
    }
}

// ------------------------------------------------------------------------------------------
// setup S1-S5, S8
// ------------------------------------------------------------------------------------------
int build_hierarchy(Oracle& o, Csr A0, double theta, int max_levels, int coarse_max) {
    o.lev.clear();
    o.lev.emplace_back();
    o.lev[0].A = std::move(A0);
    int l = 0;
    for (;;) {
        Level& cur = o.lev[l];
        l1_dinv(cur.A, cur.dinv);
        const i64 n = cur.A.nrows;
        if (n <= coarse_max || l + 1 >= max_levels) break;            // S5
        std::vector<i64> srp, trp;
        std::vector<i32> sci, tci;
        strength(cur.A, theta, srp, sci);
        transpose_pattern(n, n, srp, sci, trp, tci);
        std::vector<int8_t> cf;
        cf_split(n, srp, sci, trp, tci, cf);
        i64 nc = 0;
        for (i64 i = 0; i < n; ++i) nc += (cf[i] == 1);
        if (nc == 0 || nc == n) break;                                // S5: coarsening stagnated
        cur.cf = std::move(cf);
        direct_interp(cur.A, srp, sci, cur.cf, cur.cidx, cur.P);
        Csr Ac = galerkin(cur.A, cur.P);
        o.lev.emplace_back();
        o.lev[l + 1].A = std::move(Ac);
        ++l;
    }
    o.L = l;
    const i64 nL = o.lev[l].A.nrows;
    if (nL > 4096) return -4;                                         // COARSE_TOO_LARGE
    o.lu.assign((size_t)nL * nL, 0.0);
    const Csr& AL = o.lev[l].A;
    for (i64 i = 0; i < nL; ++i)
        for (i64 k = AL.rp[i]; k < AL.rp[i + 1]; ++k) o.lu[(size_t)i * nL + AL.ci[k]] = AL.v[k];
    if (!dense_lu((int)nL, o.lu, o.piv)) return -5;
    return 0;
}

// ------------------------------------------------------------------------------------------
// S6/S7  composite sets: points within graph distance `dist` of `seed` (edges = stored
// off-diagonal entries of the rows, eq. 1; reading A8).  Returns them ascending.
// ------------------------------------------------------------------------------------------
std::vector<i32> grow(const Csr& A, const std::vector<i32>& seed, int dist, std::vector<i32>& stamp) {
    // stamp: scratch of size n, all -1 on entry and on exit
    std::vector<i32> all(seed), frontier(seed), next;
    for (i32 i : seed) stamp[i] = 0;
    for (int d = 1; d <= dist; ++d) {
        next.clear();
        for (i32 i : frontier)
            for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) {
                const i32 j = A.ci[k];
                if (stamp[j] < 0) { stamp[j] = d; next.push_back(j); all.push_back(j); }
            }
        frontier.swap(next);
    }
    for (i32 i : all) stamp[i] = -1;
    std::sort(all.begin(), all.end());
    return all;
}

void build_comp(const Oracle& o, int p, Comp& c, std::vector<std::vector<i32>>& stamp) {
    const int L = o.L;
    c.real.assign(L + 1, {});
    c.ghost.assign(L + 1, {});
    std::vector<i32> B = o.owned[p];                                   // B_0^p
    for (int l = 0; l <= L; ++l) {
        const Csr& A = o.lev[l].A;
        if (l == L) {                                                  // A5: D_L = Omega_L, no ghosts
            c.real[l].resize(A.nrows);
            for (i64 i = 0; i < A.nrows; ++i) c.real[l][i] = (i32)i;
            break;
        }
        c.real[l] = grow(A, B, o.eta, stamp[l]);                       // D_l^p
        std::vector<i32> bar = grow(A, c.real[l], o.nghost, stamp[l]); // D-bar_l^p (eq. 1)
        std::set_difference(bar.begin(), bar.end(), c.real[l].begin(), c.real[l].end(),
                            std::back_inserter(c.ghost[l]));
        B.clear();                                                     // B_{l+1}^p: C-points of D_l^p
        for (i32 i : c.real[l]) if (o.lev[l].cf[i] == 1) B.push_back(o.lev[l].cidx[i]);
    }
}

// per-thread scratch: one global->local array per level, all -1 between uses
struct Scratch {
    std::vector<std::vector<i32>> g2l;
    explicit Scratch(const Oracle& o) {
        g2l.resize(o.L + 1);
        for (int l = 0; l <= o.L; ++l) g2l[l].assign(o.lev[l].A.nrows, -1);
    }
};

const Comp& get_comp(Oracle& o, int p, Scratch& sc) {
    if (!o.comp[p]) {
        std::unique_ptr<Comp> c(new Comp());
        build_comp(o, p, *c, sc.g2l);
        o.comp[p] = std::move(c);
    }
    return *o.comp[p];
}

// ------------------------------------------------------------------------------------------
// relaxation on the real points of one composite level (§4.1; readings A2-A4):
// one l1-Jacobi sweep, delta = D^{-1}(f - A u) from the OLD u, then u += delta, t += delta.
// ------------------------------------------------------------------------------------------
void relax_level(const Csr& A, const double* dinv_global, const std::vector<i32>& real,
                 const std::vector<i32>& g2l, std::vector<double>& u, const std::vector<double>& f,
                 std::vector<double>* t, std::vector<double>& delta, Counters& cnt,
                 const int8_t* cf = nullptr, int first_class = 0) {
    // cf == nullptr: plain l1-Jacobi (one pass over all real points).  Otherwise "CF l1-scaled Jacobi" (P:275,
    // reading A2b): two half-sweeps, each an l1-Jacobi update of one class of points (C: cf > 0, F: cf < 0)
    // from the current u; first_class = +1: C-points then F-points, -1: F-points then C-points.
    const size_t nr = real.size();
    delta.resize(nr);
    const int npass = cf ? 2 : 1;
    for (int pass = 0; pass < npass; ++pass) {
        const int cls = cf ? (pass == 0 ? first_class : -first_class) : 0;
        for (size_t i = 0; i < nr; ++i) {
            const i32 g = real[i];
            delta[i] = 0.0;
            if (cf && ((cf[g] > 0) != (cls > 0))) continue;
            double au = 0.0;
            for (i64 k = A.rp[g]; k < A.rp[g + 1]; ++k) {
                const i32 lj = g2l[A.ci[k]];
                assert(lj >= 0);                                       // eq. 1: the row stencil is in D-bar_l
                au += A.v[k] * u[lj];
            }
            delta[i] = dinv_global[g] * (f[i] - au);
        }
        for (size_t i = 0; i < nr; ++i) { u[i] += delta[i]; if (t) (*t)[i] += delta[i]; }
    }
    cnt.A += 1;
}

// ------------------------------------------------------------------------------------------
// AlgFAC V(nu,nu)-cycles on the composite grid of subdomain p (Alg. 4).
// r[l] = globally restricted residual on level l (Alg. 2; reading A14).
// On return u0 holds u_0 on D-bar_0^p (real points first, then ghosts).
// ------------------------------------------------------------------------------------------
void fac_subdomain(Oracle& o, int p, const std::vector<std::vector<double>>& r, int nfac, int nu,
                   Scratch& sc, std::vector<double>& u0, Counters& cnt, i64& dropped) {
    const int L = o.L;
    const Comp& c = get_comp(o, p, sc);
    std::vector<std::vector<double>> u(L + 1), f(L + 1), t(L + 1), s(L + 1);
    std::vector<double> w, delta;
    for (int l = 0; l <= L; ++l) {
        const size_t nr = c.real[l].size(), ng = c.ghost[l].size();
        for (size_t i = 0; i < nr; ++i) sc.g2l[l][c.real[l][i]] = (i32)i;
        for (size_t i = 0; i < ng; ++i) sc.g2l[l][c.ghost[l][i]] = (i32)(nr + i);
        u[l].assign(nr + ng, 0.0);
        t[l].assign(nr, 0.0);
        s[l].assign(nr + ng, 0.0);
        f[l].resize(nr);
        for (size_t i = 0; i < nr; ++i) f[l][i] = r[l][c.real[l][i]];
    }
    auto gid = [&](int l, size_t li) -> i32 {
        const size_t nr = c.real[l].size();
        return li < nr ? c.real[l][li] : c.ghost[l][li - nr];
    };
    for (int it = 0; it < nfac; ++it) {
        for (int l = 0; l < L; ++l) {                                  // downsweep P:505
            const Level& lv = o.lev[l];
            const size_t nr = c.real[l].size(), nb = u[l].size();
            if (l != 0) std::fill(u[l].begin(), u[l].end(), 0.0);
            for (int k = 0; k < nu; ++k)
                relax_level(lv.A, lv.dinv.data(), c.real[l], sc.g2l[l], u[l], f[l], &t[l], delta, cnt,
                            o.smoother ? lv.cf.data() : nullptr, +1);
            // P:509  w = s_l + A_l t_l on D-bar_l ; t_l is zero off D_l (reading A12)
            w = s[l];
            for (size_t li = 0; li < nb; ++li) {
                const i32 g = gid(l, li);
                double at = 0.0;
                for (i64 k = lv.A.rp[g]; k < lv.A.rp[g + 1]; ++k) {
                    const i32 lj = sc.g2l[l][lv.A.ci[k]];
                    if (lj >= 0 && (size_t)lj < nr) at += lv.A.v[k] * t[l][lj];
                }
                w[li] += at;
            }
            cnt.A += 1;
            // P:509  s_{l+1} = R_l w = P_l^T w restricted to D-bar_{l+1}
            std::fill(s[l + 1].begin(), s[l + 1].end(), 0.0);
            for (size_t li = 0; li < nb; ++li) {
                const i32 g = gid(l, li);
                for (i64 k = lv.P.rp[g]; k < lv.P.rp[g + 1]; ++k) {
                    const i32 lI = sc.g2l[l + 1][lv.P.ci[k]];
                    if (lI < 0) { if (it == 0) ++dropped; continue; }  // A7
                    s[l + 1][lI] += lv.P.v[k] * w[li];
                }
            }
            cnt.R += 1;
            // P:510  f_{l+1} <- f_{l+1} - A_{l+1} u_{l+1}   (u_{l+1} of the previous iteration, A1)
            const Level& lc = o.lev[l + 1];
            const size_t nrc = c.real[l + 1].size();
            if (it > 0) {                                              // zero on the first downsweep
                for (size_t i = 0; i < nrc; ++i) {
                    const i32 g = c.real[l + 1][i];
                    double au = 0.0;
                    for (i64 k = lc.A.rp[g]; k < lc.A.rp[g + 1]; ++k) {
                        const i32 lj = sc.g2l[l + 1][lc.A.ci[k]];
                        assert(lj >= 0);
                        au += lc.A.v[k] * u[l + 1][lj];
                    }
                    f[l + 1][i] -= au;
                }
                cnt.A += 1;
            }
            for (size_t i = 0; i < nrc; ++i) f[l + 1][i] -= s[l + 1][i];
            std::fill(t[l].begin(), t[l].end(), 0.0);
            std::fill(s[l].begin(), s[l].end(), 0.0);
        }
        // P:514  coarse solve u_L = A_L^{-1} f_L (D_L = Omega_L, reading A5)
        u[L] = f[L];
        dense_lu_solve((int)u[L].size(), o.lu, o.piv, u[L].data());
        for (int l = L - 1; l >= 0; --l) {                             // upsweep P:515
            const Level& lv = o.lev[l];
            const size_t nb = u[l].size();
            for (size_t li = 0; li < nb; ++li) {                       // P:516 on all of D-bar_l (§4.2)
                const i32 g = gid(l, li);
                double pu = 0.0;
                for (i64 k = lv.P.rp[g]; k < lv.P.rp[g + 1]; ++k) {
                    const i32 lI = sc.g2l[l + 1][lv.P.ci[k]];
                    if (lI >= 0) pu += lv.P.v[k] * u[l + 1][lI];
                }
                u[l][li] += pu;
            }
            cnt.P += 1;
            for (int k = 0; k < nu; ++k)
                relax_level(lv.A, lv.dinv.data(), c.real[l], sc.g2l[l], u[l], f[l], &t[l], delta, cnt,
                            o.smoother ? lv.cf.data() : nullptr, -1);
        }
    }
    u0 = u[0];
    for (int l = 0; l <= L; ++l) {
        for (i32 g : c.real[l]) sc.g2l[l][g] = -1;
        for (i32 g : c.ghost[l]) sc.g2l[l][g] = -1;
    }
}

void spmv(const Csr& A, const double* x, double* y) {
    for (i64 i = 0; i < A.nrows; ++i) {
        double s = 0.0;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) s += A.v[k] * x[A.ci[k]];
        y[i] = s;
    }
}

void spmv_t(const Csr& P, const double* x, double* y) {            // y = P^T x
    std::fill(y, y + P.ncols, 0.0);
    for (i64 i = 0; i < P.nrows; ++i)
        for (i64 k = P.rp[i]; k < P.rp[i + 1]; ++k) y[P.ci[k]] += P.v[k] * x[i];
}

// Alg. 2 lines P:471-473: r_0 = b - A_0 x ; r_{l+1} = P_l^T r_l (no relaxation)
void global_residuals(const Oracle& o, const double* b, const double* x, std::vector<std::vector<double>>& r) {
    r.resize(o.L + 1);
    const i64 n = o.lev[0].A.nrows;
    r[0].resize(n);
    spmv(o.lev[0].A, x, r[0].data());
    for (i64 i = 0; i < n; ++i) r[0][i] = b[i] - r[0][i];
    for (int l = 0; l < o.L; ++l) {
        r[l + 1].resize(o.lev[l + 1].A.nrows);
        spmv_t(o.lev[l].P, r[l].data(), r[l + 1].data());
    }
}

// one AMG-DD cycle (Alg. 2) on the listed subdomains (all if list == nullptr)
void amgdd_cycle(Oracle& o, const double* b, double* x, int nfac, int nu, const i32* list, int nlist,
                 int nthreads) {
    std::vector<std::vector<double>> r;
    global_residuals(o, b, x, r);
    const int cnt = list ? nlist : o.nsub;
    i64 dropped = 0;
    Counters total;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
#endif
    {
        Scratch sc(o);
        std::vector<double> u0;
        Counters c;
        i64 dr = 0;
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
        for (int q = 0; q < cnt; ++q) {
            const int p = list ? list[q] : q;
            Counters cp;
            fac_subdomain(o, p, r, nfac, nu, sc, u0, cp, dr);
            if (q == 0) c = cp;                                        // counters of one subdomain
            const Comp& cm = *o.comp[p];
            // P:479  u_0 <- u_0 + delta u_0^p on Omega_0^p (disjoint targets)
            for (size_t i = 0; i < cm.real[0].size(); ++i) {
                const i32 g = cm.real[0][i];
                if (o.owner[g] == p) x[g] += u0[i];
            }
        }
#ifdef _OPENMP
#pragma omp critical
#endif
        { dropped += dr; total.A += c.A; total.P += c.P; total.R += c.R; }
    }
    o.dropped = dropped;
    o.cnt = total;
}

double residual_norm(const Oracle& o, const double* b, const double* x) {
    const Csr& A = o.lev[0].A;
    double ss = 0.0;
    for (i64 i = 0; i < A.nrows; ++i) {
        double s = 0.0;
        for (i64 k = A.rp[i]; k < A.rp[i + 1]; ++k) s += A.v[k] * x[A.ci[k]];
        const double ri = b[i] - s;
        ss += ri * ri;
    }
    return std::sqrt(ss);
}

}  // namespace

// ==========================================================================================
// C entry points (ctypes binding in oracle/__init__.py)
// ==========================================================================================
extern "C" {

void* orc_create(i64 n, const i64* rowptr, const i32* colind, const double* vals, double theta,
                 int max_levels, int coarse_max, int* err) {
    Oracle* o = new Oracle();
    Csr A;
    A.nrows = A.ncols = n;
    A.rp.assign(rowptr, rowptr + n + 1);
    A.ci.assign(colind, colind + rowptr[n]);
    A.v.assign(vals, vals + rowptr[n]);
    const int rc = build_hierarchy(*o, std::move(A), theta, max_levels, coarse_max);
    if (err) *err = rc;
    if (rc != 0) { delete o; return nullptr; }
    return o;
}

void orc_destroy(void* h) { delete (Oracle*)h; }

// 0: l1-Jacobi, 1: CF l1-Jacobi (relaxation of orc_cycle, orc_solve, orc_fac_local, orc_vcycle)
void orc_set_smoother(void* h, int type) { ((Oracle*)h)->smoother = type; }

int orc_num_levels(void* h) { return ((Oracle*)h)->L + 1; }

void orc_level_size(void* h, int l, i64* n, i64* nnzA, i64* nnzP) {
    const Level& lv = ((Oracle*)h)->lev[l];
    *n = lv.A.nrows; *nnzA = lv.A.nnz(); *nnzP = lv.P.nnz();
}

void orc_get_cf(void* h, int l, int8_t* cf) {
    const Level& lv = ((Oracle*)h)->lev[l];
    std::copy(lv.cf.begin(), lv.cf.end(), cf);
}

void orc_get_matrix(void* h, int l, int which, i64* rp, i32* ci, double* v) {
    const Level& lv = ((Oracle*)h)->lev[l];
    const Csr& M = which == 0 ? lv.A : lv.P;
    std::copy(M.rp.begin(), M.rp.end(), rp);
    std::copy(M.ci.begin(), M.ci.end(), ci);
    std::copy(M.v.begin(), M.v.end(), v);
}

void orc_get_dinv(void* h, int l, double* d) {
    const Level& lv = ((Oracle*)h)->lev[l];
    std::copy(lv.dinv.begin(), lv.dinv.end(), d);
}

// TEST SUPPORT, no arithmetic of the method: overwrite the stored VALUES of A_l (same pattern, l >= 1) with the caller's
// and refresh what is derived from them with the routines above -- the l1 diagonal (S8) and, on the coarsest level, the
// dense LU.  P_l, the C/F splitting and the composite index sets (patterns only) stay.  Reading S4 leaves the summation
// order of a Galerkin entry open; with this entry a test can build a SECOND valid oracle whose coarse operators were
// summed in another order (scipy's P^T (A P) of this oracle's own A_l, P_l) and measure how far two valid oracles are
// apart: the yardstick of DESIGN.md section 12.  Returns 0, -1 for a bad level, -5 for a singular A_L.
int orc_set_level_values(void* h, int l, const double* vals) {
    Oracle& o = *(Oracle*)h;
    if (l < 1 || l > o.L) return -1;
    Level& lv = o.lev[l];
    std::copy(vals, vals + lv.A.nnz(), lv.A.v.begin());
    l1_dinv(lv.A, lv.dinv);
    if (l == o.L) {
        const i64 nL = lv.A.nrows;
        o.lu.assign((size_t)nL * nL, 0.0);
        for (i64 i = 0; i < nL; ++i)
            for (i64 k = lv.A.rp[i]; k < lv.A.rp[i + 1]; ++k) o.lu[(size_t)i * nL + lv.A.ci[k]] = lv.A.v[k];
        if (!dense_lu((int)nL, o.lu, o.piv)) return -5;
    }
    return 0;
}

// S6: owner partition, padding eta (one value for every level l < L, reading A6), ghost layers
int orc_set_partition(void* h, int nsub, const i32* owner, int eta, int num_ghost) {
    Oracle& o = *(Oracle*)h;
    const i64 n = o.lev[0].A.nrows;
    if (nsub < 1 || eta < 0 || num_ghost < 1) return -1;
    o.nsub = nsub; o.eta = eta; o.nghost = num_ghost;
    o.owner.assign(owner, owner + n);
    o.owned.assign(nsub, {});
    for (i64 i = 0; i < n; ++i) {
        if (owner[i] < 0 || owner[i] >= nsub) return -3;
        o.owned[owner[i]].push_back((i32)i);
    }
    for (int p = 0; p < nsub; ++p) if (o.owned[p].empty()) return -3;
    o.comp.clear();
    o.comp.resize(nsub);
    return 0;
}

void orc_composite_size(void* h, int p, int l, i64* nr, i64* ng) {
    Oracle& o = *(Oracle*)h;
    if (!o.comp[p]) { Scratch sc(o); get_comp(o, p, sc); }             // (the scratch arrays are of global size: only when the grid is not built yet)
    const Comp& c = *o.comp[p];
    *nr = (i64)c.real[l].size(); *ng = (i64)c.ghost[l].size();
}

void orc_get_composite(void* h, int p, int l, i32* real, i32* ghost) {
    Oracle& o = *(Oracle*)h;
    if (!o.comp[p]) { Scratch sc(o); get_comp(o, p, sc); }
    const Comp& c = *o.comp[p];
    std::copy(c.real[l].begin(), c.real[l].end(), real);
    std::copy(c.ghost[l].begin(), c.ghost[l].end(), ghost);
}

// one AMG-DD cycle, x updated in place on the owned dofs of the listed subdomains
void orc_cycle(void* h, const double* b, double* x, int nfac, int nu, const i32* list, int nlist, int nthreads) {
    amgdd_cycle(*(Oracle*)h, b, x, nfac, nu, list, nlist, nthreads);
}

double orc_residual_norm(void* h, const double* b, const double* x) {
    return residual_norm(*(Oracle*)h, b, x);
}

// num_cycles AMG-DD cycles; resnorm[k] = ||b - A x_k||_2, k = 0..num_cycles (reading A16)
void orc_solve(void* h, const double* b, double* x, int num_cycles, int nfac, int nu, double* resnorm,
               int nthreads) {
    Oracle& o = *(Oracle*)h;
    if (resnorm) resnorm[0] = residual_norm(o, b, x);
    for (int k = 0; k < num_cycles; ++k) {
        amgdd_cycle(o, b, x, nfac, nu, nullptr, 0, nthreads);
        if (resnorm) resnorm[k + 1] = residual_norm(o, b, x);
    }
}

// AlgFAC on one subdomain from a given global fine residual r0: returns u_0 on D-bar_0^p
void orc_fac_local(void* h, int p, const double* r0, int nfac, int nu, double* u0_out) {
    Oracle& o = *(Oracle*)h;
    std::vector<std::vector<double>> r(o.L + 1);
    r[0].assign(r0, r0 + o.lev[0].A.nrows);
    for (int l = 0; l < o.L; ++l) {
        r[l + 1].resize(o.lev[l + 1].A.nrows);
        spmv_t(o.lev[l].P, r[l].data(), r[l + 1].data());
    }
    Scratch sc(o);
    std::vector<double> u0;
    Counters c;
    i64 dr = 0;
    fac_subdomain(o, p, r, nfac, nu, sc, u0, c, dr);
    o.cnt = c; o.dropped = dr;
    std::copy(u0.begin(), u0.end(), u0_out);
}

// The relaxation routine of Alg. 4 applied to a whole level: real points = mask != 0 (all points
// if mask == NULL); `dinv` overrides the l1 diagonal if not NULL.  nsweeps Jacobi sweeps on u.
void orc_relax(void* h, int l, double* u, const double* f, const int8_t* mask, const double* dinv, int nsweeps) {
    Oracle& o = *(Oracle*)h;
    const Level& lv = o.lev[l];
    const i64 n = lv.A.nrows;
    std::vector<i32> real, g2l(n);
    for (i64 i = 0; i < n; ++i) { g2l[i] = (i32)i; if (!mask || mask[i]) real.push_back((i32)i); }
    // local numbering = global numbering here; u and f are addressed through `real`
    std::vector<double> uu(u, u + n), delta, ff(real.size());
    // relax_level addresses u by local index of D-bar (= global here) but f, delta by real index
    // and updates u[i] for i < nr, so permute: real points first.
    std::vector<i32> perm(n, -1);
    i32 q = 0;
    for (i32 g : real) perm[g] = q++;
    for (i64 i = 0; i < n; ++i) if (perm[i] < 0) perm[i] = q++;
    std::vector<double> up(n);
    for (i64 i = 0; i < n; ++i) up[perm[i]] = u[i];
    for (size_t i = 0; i < real.size(); ++i) ff[i] = f[real[i]];
    Counters c;
    for (int k = 0; k < nsweeps; ++k)
        relax_level(lv.A, dinv ? dinv : lv.dinv.data(), real, perm, up, ff, nullptr, delta, c, o.smoother ? lv.cf.data() : nullptr, +1);
    for (i64 i = 0; i < n; ++i) u[i] = up[perm[i]];
}

// AMG V(nu1,nu2)-cycle on the global hierarchy (Alg. 1) with the same relaxation
void orc_vcycle(void* h, const double* b, double* x, int nu1, int nu2) {
    Oracle& o = *(Oracle*)h;
    const int L = o.L;
    std::vector<std::vector<double>> u(L + 1), f(L + 1);
    std::vector<double> delta, tmp;
    Counters c;
    u[0].assign(x, x + o.lev[0].A.nrows);
    f[0].assign(b, b + o.lev[0].A.nrows);
    std::vector<std::vector<i32>> id(L + 1);
    for (int l = 0; l <= L; ++l) { id[l].resize(o.lev[l].A.nrows); for (size_t i = 0; i < id[l].size(); ++i) id[l][i] = (i32)i; }
    for (int l = 0; l < L; ++l) {
        const Level& lv = o.lev[l];
        for (int k = 0; k < nu1; ++k) relax_level(lv.A, lv.dinv.data(), id[l], id[l], u[l], f[l], nullptr, delta, c, o.smoother ? lv.cf.data() : nullptr, +1);
        tmp.resize(lv.A.nrows);
        spmv(lv.A, u[l].data(), tmp.data());
        for (size_t i = 0; i < tmp.size(); ++i) tmp[i] = f[l][i] - tmp[i];
        f[l + 1].resize(o.lev[l + 1].A.nrows);
        spmv_t(lv.P, tmp.data(), f[l + 1].data());
        u[l + 1].assign(o.lev[l + 1].A.nrows, 0.0);
    }
    u[L] = f[L];
    dense_lu_solve((int)u[L].size(), o.lu, o.piv, u[L].data());
    for (int l = L - 1; l >= 0; --l) {
        const Level& lv = o.lev[l];
        for (i64 i = 0; i < lv.A.nrows; ++i) {
            double pu = 0.0;
            for (i64 k = lv.P.rp[i]; k < lv.P.rp[i + 1]; ++k) pu += lv.P.v[k] * u[l + 1][lv.P.ci[k]];
            u[l][i] += pu;
        }
        for (int k = 0; k < nu2; ++k) relax_level(lv.A, lv.dinv.data(), id[l], id[l], u[l], f[l], nullptr, delta, c, o.smoother ? lv.cf.data() : nullptr, -1);
    }
    std::copy(u[0].begin(), u[0].end(), x);
}

// dense solve with the stored LU of A_L (pin: against a library solve)
void orc_coarse_solve(void* h, double* x) {
    Oracle& o = *(Oracle*)h;
    dense_lu_solve((int)o.lev[o.L].A.nrows, o.lu, o.piv, x);
}

// counters of the last orc_fac_local / first subdomain of the last orc_cycle: A, P, R mat-vecs
void orc_counters(void* h, i64* out) {
    Oracle& o = *(Oracle*)h;
    out[0] = o.cnt.A; out[1] = o.cnt.P; out[2] = o.cnt.R;
}

i64 orc_dropped(void* h) { return ((Oracle*)h)->dropped; }

// Composite-grid overhead: sum over subdomains and levels of nnz(A_l) on real rows,
// divided by sum over levels of nnz(A_l).  Builds every composite grid.
double orc_overhead(void* h, int nthreads) {
    Oracle& o = *(Oracle*)h;
    double num = 0.0, den = 0.0;
    for (int l = 0; l <= o.L; ++l) den += (double)o.lev[l].A.nnz();
#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads < 1 ? 1 : nthreads)
#endif
    {
        Scratch sc(o);
        double part = 0.0;
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
        for (int p = 0; p < o.nsub; ++p) {
            const Comp& c = get_comp(o, p, sc);
            for (int l = 0; l <= o.L; ++l)
                for (i32 g : c.real[l]) part += (double)(o.lev[l].A.rp[g + 1] - o.lev[l].A.rp[g]);
        }
#ifdef _OPENMP
#pragma omp critical
#endif
        num += part;
    }
    return num / den;
}

int orc_max_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
