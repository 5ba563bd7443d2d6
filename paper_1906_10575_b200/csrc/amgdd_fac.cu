// The persistent AlgFAC kernel (sm_100a): Alg. 2 lines P:475-479 with Alg. 4 inside.
//
// One CTA per SM takes whole subdomains from a work counter and runs ALL num_fac_cycles AlgFAC
// V(nu,nu)-cycles of a subdomain start to finish; subdomains never communicate.
//
// Every warp is a consumer AND its own producer.  A matrix is stored as NUM_WAYS independent
// sub-streams (amgdd_stream.hpp); warp w owns way w of every matrix: it streams the blocks of its
// way HBM -> its PRIVATE shared-memory ring with cp.async.bulk (TMA, SASS UBLKCP; completion on one
// mbarrier per ring slot) and consumes them in order.  Matrix data does not depend on computed
// values, so the warp's issue cursor walks the same static "program" of mat-vecs as its consume
// cursor, `stages` blocks ahead -- across mat-vec, level and subdomain boundaries -- and the only
// synchronisation between warps is the CTA barrier between two steps of Alg. 4.
//
// Inside a block, lane j owns row j of a 32-row slice (slice-JDS layout): it adds the entries of
// its row in stored (= column) order, so there is no cross-lane reduction and every row sum has
// one fixed summation order (run-to-run identical results); a row-local epilogue applies the
// AlgFAC update.  The gather vector of a mat-vec is staged in shared memory.
// The level vectors u, t, s, f live in a per-CTA workspace slot in global memory that every
// subdomain of the CTA reuses; what streams from HBM is matrix data, once per mat-vec.
#include "amgdd_stream.hpp"

#include <cuda_runtime.h>

#include <climits>

namespace amgdd {

namespace {

constexpr int MAX_STAGES = 8;
constexpr int NTHREADS = 32 * NUM_WAYS;

enum OpKind { OP_RELAX = 0, OP_AT = 1, OP_RESTRICT = 2, OP_RECALC = 3, OP_INTERP = 4, OP_RELAX_DELTA = 5,
              OP_FIRST = 6, OP_COARSE = 7, OP_BEGIN = 8, OP_END = 9 };
// slots of the optional per-CTA cycle counters (FAC_PROF_SLOTS each; amgdd_debug_fac_cycles)
enum ProfSlot { PROF_SYNC = 0, PROF_WAIT_FULL = 1, PROF_CONSUME = 2, PROF_STAGE = 3, PROF_ISSUE = 4, PROF_BEGIN = 5,
                PROF_END = 6, PROF_FIRST = 7, PROF_COARSE = 8, PROF_TOTAL = 9, PROF_OP0 = 10 };

// an op of the program: kind | level << 4 | (first AlgFAC iteration) << 12
__host__ __device__ constexpr unsigned short make_op(int kind, int level, int first) {
    return (unsigned short)(kind | (level << 4) | (first << 12));
}
__device__ __forceinline__ int op_kind(unsigned short op) { return op & 15; }
__device__ __forceinline__ int op_level(unsigned short op) { return (op >> 4) & 255; }
__device__ __forceinline__ int op_first(unsigned short op) { return (op >> 12) & 1; }

// The static program of one subdomain: the steps of num_fac_cycles AlgFAC V(nu,nu)-cycles (Alg. 4)
// in order.  emit(op) is called for each; fac_num_ops() counts with the same routine.
struct OpSink {                       // counts the ops and, if out != nullptr, stores them
    unsigned short* out;
    int n;
    __host__ __device__ void operator()(unsigned short op) {
        if (out) out[n] = op;
        ++n;
    }
};

__host__ __device__ inline void fac_program(int L, int nfac, int nu, OpSink& emit) {
    emit(make_op(OP_BEGIN, 0, 0));                                         // Alg. 2, Alg. 4
    for (int it = 0; it < nfac; ++it) {
        const int first = it == 0;
        for (int l = 0; l < L; ++l) {                                      // downsweep P:505-513
            int sweeps = nu;
            if (l != 0) { emit(make_op(OP_FIRST, l, first)); --sweeps; }   // u_l = 0, so delta = D^-1 f
            for (int k = 0; k < sweeps; ++k) emit(make_op(OP_RELAX, l, first));
            emit(make_op(OP_AT, l, first));                                // P:509  w = s_l + A_l t_l
            emit(make_op(OP_RESTRICT, l, first));                          // P:509  s_{l+1} = R_l w 
            if (!first) emit(make_op(OP_RECALC, l, first));                // P:510  (identically zero at it = 0)
        }
        emit(make_op(OP_COARSE, L, first));
        for (int l = L - 1; l >= 0; --l) {                                 // upsweep P:515-519
            emit(make_op(OP_INTERP, l, first));
            for (int k = 0; k < nu; ++k) emit(make_op(OP_RELAX, l, first));
        }
    }
    emit(make_op(OP_END, 0, 0));                                           // Alg. 2
}

struct Ctrl {
    unsigned long long full[NUM_WAYS][MAX_STAGES];   // ring slot s of warp w holds a complete block
    unsigned long long tbl_full[2];                  // descriptor table slot q is loaded
    int sub_id[2];                                   // subdomain whose table sits in slot q (-1: no more work)
};
constexpr int CTRL_BYTES = 1152;
static_assert(sizeof(Ctrl) <= CTRL_BYTES, "control block too large");

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 1-D bulk async copy global -> shared (TMA), completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s_plain(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}
// orders this thread's earlier generic-proxy accesses to shared memory before later async-proxy ones
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// shared-memory loads by 32-bit shared address (no generic-address arithmetic in the inner loop)
__device__ __forceinline__ double lds_f64(uint32_t a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t a) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint4 lds_v4(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
// the gather vector: staged in shared memory, or read from the workspace (global memory)
struct SmemVec {
    uint32_t base;
    __device__ __forceinline__ double at(uint32_t c) const { return lds_f64(base + (c << 3)); }
};
struct GlobalVec {
    const double* base;
    __device__ __forceinline__ double at(uint32_t c) const { return base[c]; }
};

// What a row does with its finished sum (the Alg. 4 step of the mat-vec); the pointers index the
// level vectors in this CTA's workspace slot.
struct Epilogue {
    int kind;              // OpKind
    int limit;             // OP_RESTRICT: rows below this are real rows of level l+1
    int first;             // OP_RESTRICT: first AlgFAC iteration
    double* a;             // RELAX u | AT w | RESTRICT s_{l+1} | RECALC f_{l+1} | INTERP u | RELAX_DELTA delta
    double* b;             // RELAX t | RESTRICT f_{l+1}
    const double* c;       // RELAX f | AT s | RECALC s_{l+1} | RELAX_DELTA f
};

__device__ __forceinline__ void apply(const Epilogue& ep, int i, double sum, double aux) {
    switch (ep.kind) {
        case OP_RELAX: {                   // one l1-Jacobi update (§4.1); aux = 1 / sum_j |a_ij| (S8)
            const double dl = aux * (ep.c[i] - sum);
            ep.a[i] += dl;
            ep.b[i] += dl;
            break;
        }
        case OP_RELAX_DELTA: ep.a[i] = aux * (ep.c[i] - sum); break;
        case OP_AT: ep.a[i] = ep.c[i] + sum; break;                        // P:509 w = s_l + A_l t_l
        case OP_RESTRICT:                                                  // P:509 s_{l+1} = R_l w ; P:511 (first iteration)
            ep.a[i] = sum;
            if (ep.first && i < ep.limit) ep.b[i] -= sum;
            break;
        case OP_RECALC: ep.a[i] = (ep.a[i] - sum) - ep.c[i]; break;
        default: ep.a[i] += sum; break;                                    // OP_INTERP
    }
}

// What a warp carries from piece to piece of the slice it is working on (a slice may span blocks).
struct SliceState {
    double acc, aux;
    int row;               // row of this lane, -1: none
    int len;               // entries of that row
    int slices_left;       // slices still to finish in this mat-vec (real-rows-only mat-vecs stop early)
};

// One block in shared memory (layout: amgdd_stream.hpp), `blk` = its shared address.  Lane j owns
// row j of the slice and adds its entries in stored (= column) order.  Lanes whose row has ended
// re-read entry 0 of the piece and discard it: every load is unconditional, so the four steps of
// an unrolled block overlap.
template <bool WIDE, class X>
__device__ __forceinline__ void consume_block(uint32_t blk, X xs, int has_aux, SliceState& st, const Epilogue& ep) {
    constexpr int CS = WIDE ? 2 : 1;                               // log2 bytes per column index
    const int np = (int)lds_u32(blk);
    const int lane = threadIdx.x & 31;
    for (int i = 0; i < np && st.slices_left > 0; ++i) {
        const uint4 raw = lds_v4(blk + BLOCK_HEADER_BYTES + i * PIECE_DESC_BYTES);
        const int k0 = (int)(raw.z & 0xFFFFu), nk = (int)(raw.z >> 16), K = (int)(raw.w & 0xFFFFu), nnz = (int)(raw.w >> 16);
        uint32_t q = blk + raw.x;
        if (k0 == 0) {
            const int rid = (int)lds_u16(q + 2 * lane);
            st.len = (int)lds_u16(q + 2 * (SLICE_ROWS + lane));
            st.row = rid == (int)NO_ROW ? -1 : (int)raw.y + rid;
            st.acc = 0.0;
            q += SLICE_ROWS * 4;
            if (has_aux) { st.aux = lds_f64(q + 8 * lane); q += SLICE_ROWS * 8; }
        }
        const uint32_t vb = q, cb = q + (uint32_t)nnz * 8;
        uint32_t e = (uint32_t)lane;
        double acc = st.acc;
        const int len = st.len;
        int k = k0;
        const int kend = k0 + nk;
        auto col = [&](uint32_t ee) { return WIDE ? lds_u32(cb + (ee << CS)) : lds_u16(cb + (ee << CS)); };
        for (; k + 4 <= kend; k += 4) {
            const bool a0 = k < len, a1 = k + 1 < len, a2 = k + 2 < len, a3 = k + 3 < len;
            const uint32_t e0 = e;
            const uint32_t e1 = e0 + __popc(__ballot_sync(0xffffffffu, a0));
            const uint32_t e2 = e1 + __popc(__ballot_sync(0xffffffffu, a1));
            const uint32_t e3 = e2 + __popc(__ballot_sync(0xffffffffu, a2));
            e = e3 + __popc(__ballot_sync(0xffffffffu, a3));
            const uint32_t f0 = a0 ? e0 : 0u, f1 = a1 ? e1 : 0u, f2 = a2 ? e2 : 0u, f3 = a3 ? e3 : 0u;
            const uint32_t c0 = col(f0), c1 = col(f1), c2 = col(f2), c3 = col(f3);
            const double v0 = lds_f64(vb + (f0 << 3)), v1 = lds_f64(vb + (f1 << 3));
            const double v2 = lds_f64(vb + (f2 << 3)), v3 = lds_f64(vb + (f3 << 3));
            const double x0 = xs.at(c0), x1 = xs.at(c1), x2 = xs.at(c2), x3 = xs.at(c3);
            if (a0) acc = fma(v0, x0, acc);
            if (a1) acc = fma(v1, x1, acc);
            if (a2) acc = fma(v2, x2, acc);
            if (a3) acc = fma(v3, x3, acc);
        }
        for (; k < kend; ++k) {
            const bool a0 = k < len;
            const uint32_t cnt = __popc(__ballot_sync(0xffffffffu, a0));
            const uint32_t f0 = a0 ? e : 0u;
            const double v0 = lds_f64(vb + (f0 << 3));
            const double x0 = xs.at(col(f0));
            if (a0) acc = fma(v0, x0, acc);
            e += cnt;
        }
        st.acc = acc;
        if (kend != K) break;                                   // the slice continues in the next block
        if (st.row >= 0) apply(ep, st.row, acc, st.aux);
        --st.slices_left;
    }
}

// which packed stream a mat-vec reads, and whether it stops after the real rows
__device__ __forceinline__ const StreamDesc* stream_of(const DevLevel* T, int kind, int l, bool& real_only) {
    real_only = (kind == OP_RELAX || kind == OP_RECALC);
    if (kind == OP_RELAX || kind == OP_AT) return &T[l].A;
    if (kind == OP_RESTRICT) return &T[l].R;
    if (kind == OP_RECALC) return &T[l + 1].A;
    return &T[l].P;
}

template <bool PROF>
struct Worker {
    // ---- constants of the launch ----
    const FacParams* prm;
    Ctrl* ctrl;
    const unsigned short* ops;     // the program (shared memory)
    unsigned char* tbl_base;       // two descriptor-table slots (shared memory)
    double* xbuf;                  // shared-memory gather buffer, x_cap doubles
    uint32_t x_addr, ring_addr, bar_addr, tbl_bar_addr;   // shared addresses: xbuf, this warp's ring, its barriers, tbl_full[0]
    double* ws;                    // this CTA's workspace slot
    double* w;                     // scratch vector inside the slot
    long long* prof;               // this CTA's cycle counters (PROF only)
    uint64_t policy;
    int nops, stages, block_bytes, x_cap;
    int tid, lane, wid;
    // ---- consume cursor ----
    const DevLevel* lev;           // table of the current subdomain
    int ksub;                      // sequence number of the current subdomain of this CTA
    int cslot;
    uint32_t cphase;
    int inflight;                  // blocks issued and not yet consumed (<= stages)
    // ---- issue cursor: runs ahead of the consume cursor through the same program ----
    int iksub, iop, islot;
    uint32_t iblk, inb, itail, ilast;
    const char* isrc;
    bool idone;

    __device__ __forceinline__ long long tick() const { return PROF ? clock64() : 0; }
    __device__ __forceinline__ void tock(int idx, long long t0) const { if (PROF && tid == 0) prof[idx] += clock64() - t0; }
    __device__ __forceinline__ void sync() {
        const long long t0 = tick();
        __syncthreads();
        tock(PROF_SYNC, t0);
    }
    __device__ __forceinline__ const DevLevel* table(int q) const { return reinterpret_cast<const DevLevel*>(tbl_base + (size_t)q * prm->table_bytes); }
    __device__ __forceinline__ double* U(int l) const { return ws + lev[l].voff; }
    __device__ __forceinline__ double* T(int l) const { return ws + lev[l].voff + lev[l].n_bar; }
    __device__ __forceinline__ double* S(int l) const { return ws + lev[l].voff + 2 * (size_t)lev[l].n_bar; }
    __device__ __forceinline__ double* F(int l) const { return ws + lev[l].voff + 3 * (size_t)lev[l].n_bar; }

    // Issue the next block of this warp's way (if the ring has room the caller checked).  Returns
    // false when there is nothing to issue: no more work, or the cursor would run two subdomains ahead.
    __device__ __forceinline__ bool issue_one() {
        while (iblk >= inb) {
            if (idone) return false;
            if (iop + 1 >= nops) {                                       // the program of subdomain iksub is issued
                if (iksub > ksub) return false;
                const int nk = iksub + 1, nq = nk & 1;
                mbar_wait(tbl_bar_addr + 8 * nq, (uint32_t)(nk >> 1) & 1u);
                if (ctrl->sub_id[nq] < 0) { idone = true; return false; }
                iksub = nk;
                iop = -1;
            }
            ++iop;
            const unsigned short op = ops[iop];
            const int kind = op_kind(op);
            iblk = inb = 0;
            if (kind <= OP_INTERP) {
                bool real_only;
                const StreamDesc* sd = stream_of(table(iksub & 1), kind, op_level(op), real_only);
                const WayDesc wd = sd->way[wid];
                inb = real_only ? wd.nblocks_real : wd.nblocks;
                isrc = sd->base + 16ull * wd.off16;
                itail = wd.nblocks - 1u;
                ilast = 16u * wd.last16;
            }
        }
        if (lane == 0) {
            const uint32_t bytes = (iblk == itail) ? ilast : (uint32_t)block_bytes;
            const uint32_t bar = bar_addr + 8 * islot;
            fence_proxy_async();
            mbar_arrive_expect_tx(bar, bytes);
            bulk_copy_g2s(ring_addr + (uint32_t)islot * (uint32_t)block_bytes, isrc, bytes, bar, policy);
        }
        isrc += block_bytes;
        ++iblk;
        ++inflight;
        if (++islot == stages) islot = 0;
        return true;
    }
    __device__ __forceinline__ void top_up() {
        const long long t0 = tick();
        while (inflight < stages && issue_one()) {}
        tock(PROF_ISSUE, t0);
    }

    // ---- Alg. 2 P:475 + Alg. 4: f_l = r_l on D_l ; u = t = s = 0 ----
    __device__ __forceinline__ void begin_subdomain() {
        const long long tp0 = tick();
        const int L = prm->L;
        for (int l = 0; l <= L; ++l) {
            const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
            const int* gid = lev[l].gid;
            const double* r = prm->r_all + prm->r_off[l];
            double* u = U(l);
            for (int i = tid; i < 3 * n_bar; i += NTHREADS) u[i] = 0.0;   // u | t | s are adjacent
            double* f = F(l);
            for (int i = tid; i < n_real; i += NTHREADS) f[i] = r[__ldg(gid + i)];
        }
        tock(PROF_BEGIN, tp0);
    }
    // ---- Alg. 2: x <- x + u_0^p on Omega_0^p (disjoint targets across subdomains) ----
    __device__ __forceinline__ void end_subdomain(int p) {
        const long long tp0 = tick();
        const DevSub sb = prm->sub[p];
        const double* u0 = U(0);
        const int* gid0 = lev[0].gid;
        for (int k = tid; k < sb.n_owned; k += NTHREADS) {
            const int li = __ldg(sb.owned + k);
            prm->x[__ldg(gid0 + li)] += u0[li];
        }
        tock(PROF_END, tp0);
    }
    // P:506 u_l <- 0, then the first sweep needs no matrix: delta = D^{-1} f
    __device__ __forceinline__ void first_sweep(int l) {
        const long long tp0 = tick();
        const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
        const double* dinv = lev[l].dinv;
        double *u = U(l), *t = T(l);
        const double* f = F(l);
        for (int i = tid; i < n_bar; i += NTHREADS) {
            double dl = 0.0;
            if (i < n_real) { dl = __ldg(dinv + i) * f[i]; t[i] += dl; }
            u[i] = dl;
        }
        tock(PROF_FIRST, tp0);
    }
    // u_L = A_L^{-1} f_L with the LU factors computed at setup (Alg. 4).  One warp; columns
    // of the unit-lower / upper factors are contiguous (column-major).
    __device__ __forceinline__ void coarse() {
        const long long tp0 = tick();
        const int L = prm->L, n = prm->nL;
        const double* __restrict__ lu = prm->lu;
        const double* f = F(L);
        double* y = (n <= x_cap) ? xbuf : w;
        for (int i = tid; i < n; i += NTHREADS) y[i] = f[__ldg(prm->rowperm + i)];
        sync();
        if (wid == 0) {
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
        sync();
        double* uL = U(L);
        for (int i = tid; i < n; i += NTHREADS) uL[i] = y[i];
        tock(PROF_COARSE, tp0);
    }

    // one mat-vec: the blocks of this warp's way, in order; `staged`: the gather vector is in xbuf
    __device__ __forceinline__ void run_blocks(const StreamDesc* sd, bool real_only, bool staged, const double* xg, const Epilogue& ep) {
        const WayDesc wd = sd->way[wid];
        const uint32_t nb = real_only ? wd.nblocks_real : wd.nblocks;
        const int has_aux = sd->has_aux, wide = sd->wide;
        SliceState st;
        st.acc = 0.0; st.aux = 0.0; st.row = -1; st.len = 0;
        st.slices_left = real_only ? (int)wd.nslices_real : INT_MAX;
        for (uint32_t b = 0; b < nb; ++b) {
            top_up();                                                    // the block waited for below is issued now
            const long long t0 = tick();
            mbar_wait(bar_addr + 8 * cslot, cphase);
            tock(PROF_WAIT_FULL, t0);
            const long long t1 = tick();
            const uint32_t blk = ring_addr + (uint32_t)cslot * (uint32_t)block_bytes;
            if (staged) {
                SmemVec xs;
                xs.base = x_addr;
                consume_block<false>(blk, xs, has_aux, st, ep);
            } else {
                GlobalVec xs;
                xs.base = xg;
                if (wide) consume_block<true>(blk, xs, has_aux, st, ep);
                else consume_block<false>(blk, xs, has_aux, st, ep);
            }
            __syncwarp();
            tock(PROF_CONSUME, t1);
            --inflight;
            if (++cslot == stages) { cslot = 0; cphase ^= 1u; }
        }
        top_up();
    }

    // stage the gather vector of the next mat-vec in shared memory (if it fits; wide streams never do)
    __device__ __forceinline__ bool stage_x(const double* x, int n) {
        if (n > x_cap) return false;
        const long long t0 = tick();
        for (int i = tid; i < n; i += NTHREADS) xbuf[i] = x[i];
        tock(PROF_STAGE, t0);
        return true;
    }

    __device__ __forceinline__ void matvec(int K, int l, int first) {
        const long long top0 = tick();
        Epilogue ep;
        ep.kind = K; ep.limit = 0; ep.first = 0; ep.a = nullptr; ep.b = nullptr; ep.c = nullptr;
        bool real_only;
        const StreamDesc* sd = stream_of(lev, K, l, real_only);
        if (K == OP_RELAX) {
            // one l1-Jacobi sweep on the real points (§4.1): delta from the OLD u
            // (the staged copy), then u += delta, t += delta (P:507-508 / P:517-518)
            const int n_real = lev[l].n_real;
            double *u = U(l), *t = T(l);
            const bool staged = stage_x(u, lev[l].n_bar);
            sync();
            ep.c = F(l);
            if (staged) {
                ep.a = u; ep.b = t;
                run_blocks(sd, true, true, u, ep);
            } else {                                                     // gather from global: two passes
                double* delta = w;
                ep.kind = OP_RELAX_DELTA; ep.a = delta;
                run_blocks(sd, true, false, u, ep);
                sync();
                for (int i = tid; i < n_real; i += NTHREADS) {
                    const double dl = delta[i];
                    u[i] += dl;
                    t[i] += dl;
                }
            }
        } else if (K == OP_AT) {
            // P:509  w = s_l + A_l t_l on all of D-bar_l (ghost rows: real columns only)
            const double* t = T(l);
            const bool staged = stage_x(t, lev[l].n_bar);
            sync();
            ep.a = w; ep.c = S(l);
            run_blocks(sd, false, staged, t, ep);
        } else if (K == OP_RESTRICT) {
            // P:509  s_{l+1} = R_l w ; P:512 reset t_l, s_l ; first iteration: P:511 f_{l+1} -= s_{l+1}
            const int n_bar = lev[l].n_bar;
            const bool staged = stage_x(w, n_bar);
            double* t = T(l);
            for (int i = tid; i < 2 * n_bar; i += NTHREADS) t[i] = 0.0;  // t and s are adjacent
            sync();
            ep.a = S(l + 1); ep.b = F(l + 1); ep.limit = lev[l + 1].n_real; ep.first = first;
            run_blocks(sd, false, staged, w, ep);
        } else if (K == OP_RECALC) {
            // P:510-511  f_{l+1} <- f_{l+1} - A_{l+1} u_{l+1} - s_{l+1}  (u_{l+1} of the previous iteration)
            const double* uc = U(l + 1);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            ep.a = F(l + 1); ep.c = S(l + 1);
            run_blocks(sd, true, staged, uc, ep);
        } else {
            // P:516  u_l += P_l u_{l+1} on all of D-bar_l (§4.2)
            const double* uc = U(l + 1);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            ep.a = U(l);
            run_blocks(sd, false, staged, uc, ep);
        }
        tock(PROF_OP0 + K, top0);
    }
};

constexpr int OPS_RESERVE_BYTES = 2048;        // room for the program (2 bytes per op)

template <bool PROF>
__global__ void __launch_bounds__(NTHREADS, 1) fac_kernel(const FacParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem);
    unsigned short* ops = reinterpret_cast<unsigned short*>(smem + CTRL_BYTES);
    unsigned char* tbl = smem + CTRL_BYTES + OPS_RESERVE_BYTES;
    double* xbuf = reinterpret_cast<double*>(tbl + 2 * (size_t)prm.table_bytes);
    unsigned char* rings = reinterpret_cast<unsigned char*>(xbuf + prm.x_cap);
    const int L = prm.L;
    const uint32_t tbl_exact = (uint32_t)((L + 1) * sizeof(DevLevel));

    // thread 0: draw the next subdomain for sequence number k and start loading its descriptor table
    auto load_table = [&](int k) {
        const int q = k & 1;
        const int id = atomicAdd(prm.work_counter, 1);
        const int p = id < prm.num_sub ? prm.order[id] : -1;
        ctrl->sub_id[q] = p;
        const uint32_t bar = smem_addr(&ctrl->tbl_full[q]);
        if (p >= 0) {
            fence_proxy_async();
            mbar_arrive_expect_tx(bar, tbl_exact);
            bulk_copy_g2s_plain(smem_addr(tbl + (size_t)q * prm.table_bytes), prm.lev + (size_t)p * (L + 1), tbl_exact, bar);
        } else {
            mbar_arrive(bar);
        }
    };

    if (threadIdx.x == 0) {
        for (int w = 0; w < NUM_WAYS; ++w)
            for (int s = 0; s < prm.stages; ++s) mbar_init(&ctrl->full[w][s], 1);
        mbar_init(&ctrl->tbl_full[0], 1);
        mbar_init(&ctrl->tbl_full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        OpSink sink = {ops, 0};
        fac_program(L, prm.nfac, prm.nu, sink);
        load_table(0);
        load_table(1);
    }
    __syncthreads();

    Worker<PROF> W;
    W.prm = &prm; W.ctrl = ctrl; W.ops = ops; W.tbl_base = tbl; W.xbuf = xbuf;
    W.tid = threadIdx.x; W.lane = threadIdx.x & 31; W.wid = threadIdx.x >> 5;
    W.nops = prm.nops; W.stages = prm.stages; W.block_bytes = prm.block_bytes; W.x_cap = prm.x_cap;
    W.x_addr = smem_addr(xbuf);
    W.ring_addr = smem_addr(rings) + (uint32_t)W.wid * (uint32_t)(prm.stages * prm.block_bytes);
    W.bar_addr = smem_addr(&ctrl->full[W.wid][0]);
    W.tbl_bar_addr = smem_addr(&ctrl->tbl_full[0]);
    W.ws = prm.workspace + (size_t)blockIdx.x * prm.slot_stride;
    W.w = W.ws + prm.scratch_off;
    W.prof = PROF ? prm.prof + (size_t)blockIdx.x * FAC_PROF_SLOTS : nullptr;
    W.policy = policy_evict_first();
    W.ksub = 0; W.cslot = 0; W.cphase = 0; W.inflight = 0;
    W.iksub = 0; W.iop = -1; W.islot = 0; W.iblk = 0; W.inb = 0; W.itail = 0; W.ilast = 0; W.isrc = nullptr; W.idone = false;

    const long long tk0 = W.tick();
    for (;;) {
        const int q = W.ksub & 1;
        mbar_wait(W.tbl_bar_addr + 8 * q, (uint32_t)(W.ksub >> 1) & 1u);
        const int p = ctrl->sub_id[q];
        if (p < 0) break;
        W.lev = W.table(q);
        for (int j = 0; j < W.nops; ++j) {
            const unsigned short op = ops[j];
            const int kind = op_kind(op), l = op_level(op);
            W.sync();                                                    // the previous step is complete
            if (kind == OP_BEGIN) W.begin_subdomain();
            else if (kind == OP_FIRST) W.first_sweep(l);
            else if (kind == OP_COARSE) W.coarse();
            else if (kind == OP_END) W.end_subdomain(p);
            else W.matvec(kind, l, op_first(op));
        }
        W.sync();                                   // every warp is done with table slot q and with the workspace
        if (threadIdx.x == 0) load_table(W.ksub + 2);
        ++W.ksub;
    }
    W.tock(PROF_TOTAL, tk0);
}

}  // namespace

int fac_smem_bytes(int block_bytes, int stages, int x_cap, int table_bytes) {
    return CTRL_BYTES + OPS_RESERVE_BYTES + 2 * table_bytes + x_cap * 8 + NUM_WAYS * stages * block_bytes;
}

int fac_max_stages() { return MAX_STAGES; }

int fac_num_ops(int L, int nfac, int nu) {
    OpSink sink = {nullptr, 0};
    fac_program(L, nfac, nu, sink);
    return sink.n;
}

int fac_max_ops() { return OPS_RESERVE_BYTES / 2; }

int fac_configure(int /*device*/, int max_smem_optin) {
    cudaError_t e = cudaFuncSetAttribute(fac_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fac_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
    return e == cudaSuccess ? 0 : (int)e;
}

void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream) {
    if (prm.prof) fac_kernel<true><<<cfg.grid, cfg.block, cfg.smem_bytes, (cudaStream_t)stream>>>(prm);
    else fac_kernel<false><<<cfg.grid, cfg.block, cfg.smem_bytes, (cudaStream_t)stream>>>(prm);
}

}  // namespace amgdd
