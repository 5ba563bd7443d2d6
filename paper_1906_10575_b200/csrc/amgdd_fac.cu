// The persistent AlgFAC kernel (sm_100a): Alg. 2 lines P:475-479 with Alg. 4 inside.
//
// One CTA per SM takes whole subdomains from a work counter and runs ALL num_fac_cycles AlgFAC
// V(nu,nu)-cycles of a subdomain start to finish; subdomains never communicate.
//
// MATRIX DATA.  A matrix is stored as NUM_WAYS independent sub-streams of SELL-32 groups
// (amgdd_stream.hpp); warp w owns way w of every matrix.  It reads its groups with coalesced
// 128-bit loads (ld.global.nc, L1 no-allocate, L2 evict-first) straight into a RING OF REGISTERS
// of two blocks of RING_DEPTH groups -- the register file is the staging buffer.  While one block
// is consumed the other is in flight (one burst of loads per block), and the ring runs ahead of
// the arithmetic across mat-vec boundaries: the burst after the last block of a mat-vec fetches
// the first groups of the NEXT mat-vec of the program, so the HBM pipe does not drain at the CTA
// barrier between two steps of Alg. 4.  All loads of the ring are unconditional (clamped
// addresses): a predicated asm load forces the compiler to wait for it at once.
//
// ARITHMETIC.  Lane j owns row j of a 32-row slice: it adds the entries of its row in stored
// (= column) order, so there is no cross-lane reduction and every row sum has one fixed summation
// order (run-to-run identical results); a row-local epilogue applies the Alg. 4 update.
//
// VECTORS.  The gather vector of a mat-vec lives in one of two vector buffers; the epilogue writes
// the gather vector of the NEXT step into the other (u after interpolation for the relaxation, t
// for the A t step, w for the restriction, ...), so no step needs a staging pass and there is
// exactly one CTA barrier per step.  A buffer is in shared memory for the levels that fit the
// shared-memory budget (the L1 must keep ~44 KB for the loads in flight) and in the workspace
// slot, gathered through L1, for larger ones.  u, t, s, f of all levels are kept in a per-CTA
// workspace slot in global memory (L2 resident); a slice's header and the operands of its epilogue
// are staged in shared memory by cp.async one slice ahead (own scoreboard: waiting for them does
// not wait for the ring).
#include "amgdd_stream.hpp"

#include <cuda_runtime.h>

namespace amgdd {

namespace {

constexpr int NTHREADS = 32 * NUM_WAYS;
constexpr int D = RING_DEPTH;
#ifndef AMGDD_SINGLE_BUFFER
#define AMGDD_SINGLE_BUFFER 0
#endif
#ifndef AMGDD_EARLY_COMMIT
#define AMGDD_EARLY_COMMIT 1     // commit every batch of asynchronous copies where it is issued (0: cp.async.wait_all at the wait)
#endif
constexpr int STAGE_BYTES = 512 + 3 * 256;     // per warp: one slice header + three operand vectors of 32 doubles

// slots of the optional per-CTA cycle counters (FAC_PROF_SLOTS each; amgdd_debug_fac_cycles)
enum ProfSlot { PROF_SYNC = 0, PROF_SETUP = 1, PROF_PRE = 2, PROF_PRIME = 3, PROF_TOTAL = 4, PROF_OP0 = 5 };   // PROF_OP0 + OpKind

struct LevInfo {           // shared-memory copy of the scalar part of DevLevel
    int n_real, n_bar;
    long long voff;
    const int* gid;
    const double* dinv;
};
struct WayEnt {            // shared memory: what warp w needs to read stream s (offsets from the stream base, sbase[s])
    uint32_t grp_off128, hdr_off128;
    uint32_t n_all, n_real, nsl_all, nsl_real;
};
static_assert(sizeof(WayEnt) == 24 && sizeof(LevInfo) == 32, "shared-memory table layout");

struct Grp { uint4 a, b, c; };     // values of steps 0,1 | values of steps 2,3 | column indices (narrow: c.x, c.y)

// ---- loads ------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint4 ldg_stream128(const void* p, uint64_t pol) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ uint2 ldg_stream64(const void* p, uint64_t pol) {
    uint2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.u32 {%0,%1}, [%2], %3;" : "=r"(v.x), "=r"(v.y) : "l"(p), "l"(pol));
    return v;
}
template <bool WIDE>
__device__ __forceinline__ Grp load_grp(const char* p, int lane, uint64_t pol) {
    Grp g;
    g.a = ldg_stream128(p + 16 * lane, pol);
    g.b = ldg_stream128(p + 512 + 16 * lane, pol);
    if (WIDE) g.c = ldg_stream128(p + 1024 + 16 * lane, pol);
    else { const uint2 t = ldg_stream64(p + 1024 + 8 * lane, pol); g.c.x = t.x; g.c.y = t.y; g.c.z = 0; g.c.w = 0; }
    return g;
}
// asynchronous copies global -> shared (LDGSTS): they complete on their own scoreboard
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
#if AMGDD_EARLY_COMMIT
// every batch of copies is committed where it is issued (cp_async_issued), so the wait does not plant a new
// completion marker behind the ring's loads that were issued in between
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_issued() { cp_async_commit(); }
#else
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_issued() {}
#endif
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_u64(uint32_t a) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_f64(uint32_t a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ double mkdouble(uint32_t lo, uint32_t hi) { return __hiloint2double((int)hi, (int)lo); }

// One of the two vector buffers.  A vector of level l lives in shared memory when |D-bar_l| <= x_cap
// (gathers cost a few shared-memory wavefronts), otherwise in the workspace slot (gathers go through
// L1).  x_cap is chosen so that the L1 keeps enough room for the loads in flight (fac_pick_x_cap).
struct XB {
    uint32_t a;            // shared address
    double* p;             // the same buffer's twin in the workspace slot
    bool s;                // which one is in use for this vector
    template <bool GS> __device__ __forceinline__ double ldt(uint32_t i) const {
        if (GS) {
            double v;
            asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a + (i << 3)));
            return v;
        }
        return p[i];
    }
    __device__ __forceinline__ double ld(uint32_t i) const { return s ? ldt<true>(i) : ldt<false>(i); }
    __device__ __forceinline__ void st(uint32_t i, double v) const {
        if (s) asm volatile("st.shared.f64 [%0], %1;" ::"r"(a + (i << 3)), "d"(v) : "memory");
        else p[i] = v;
    }
};

__device__ __forceinline__ int stream_of(const FacOp& op) {           // 3 * level + {0: A, 1: P, 2: R}
    const int which = op.kind == OPK_INTERP ? 1 : op.kind == OPK_RESTRICT ? 2 : 0;
    return 3 * op.level + which;
}
__device__ __forceinline__ bool real_rows_only(const FacOp& op) { return op.kind == OPK_RELAX || op.kind == OPK_RECALC; }
__device__ __forceinline__ bool is_matvec(int kind) { return kind >= OPK_RELAX && kind <= OPK_INTERP; }
// level of the vector a step gathers from / of the vector it leaves in the other buffer
__device__ __forceinline__ int gather_level(const FacOp& op) { return op.kind == OPK_INTERP ? op.level + 1 : op.level; }
__device__ __forceinline__ int out_level(const FacOp& op) { return op.kind == OPK_RESTRICT ? op.level + 1 : op.level; }

template <bool PROF>
struct Worker {
    const FacParams* prm;
    const FacOp* ops;              // shared memory
    const LevInfo* lev;            // shared memory, L+1
    const WayEnt* wt;              // shared memory, [stream][way]
    const uint32_t* sflags;        // shared memory, per stream
    const char* const* sbase;      // shared memory, per stream: base address of the packed stream
    uint32_t xs0, xs1;             // the two vector buffers in shared memory (x_cap doubles each)
    double *xg0, *xg1;             // and in the workspace slot
    int x_cap;
    __device__ __forceinline__ XB xbuf_of(int b, int level) const {
        XB x;
        x.a = b ? xs1 : xs0; x.p = b ? xg1 : xg0; x.s = lev[level].n_bar <= x_cap;
        return x;
    }
    double* ws;                    // this CTA's workspace slot
    long long* prof;
    long long* prof_s;             // shared-memory copy of the counters (PROF)
    uint64_t pol_stream, pol_keep; // L2 policies: private streams are read once per mat-vec (evict first), shared levels by every CTA (keep)
    int tid, lane, wid, L;
    // ring state carried from mat-vec to mat-vec
    Grp ra[D], rb[D];              // two blocks of D groups; `phase` tells which one holds the coming block
    int phase;
    bool ring_valid;               // the ring holds the first groups of the coming mat-vec
    bool hdr_ready;                // the staging area holds (or is receiving) the header of its slice 0
    uint32_t stage;                // shared address of this warp's staging area (STAGE_BYTES)
    int opj;                       // index of the current step in the program (profiling)

    __device__ __forceinline__ long long tick() const { return PROF ? clock64() : 0; }
    // profiling counters live in shared memory while the kernel runs (a global read-modify-write per event would
    // cost thread 0 a round trip to L2 each time and distort what is measured); flushed once at the end
    __device__ __forceinline__ void tock(int idx, long long t0) const { if (PROF && tid == 0) prof_s[idx] += clock64() - t0; }
    __device__ __forceinline__ void tock_op(int which, long long t0) const {
        if (PROF && tid == 0 && opj < PROF_OPS_SMEM) prof_s[FAC_PROF_SLOTS + which * PROF_OPS_SMEM + opj] += clock64() - t0;
    }
    __device__ __forceinline__ void sync() {
        const long long t0 = tick();
        __syncthreads();
        tock(PROF_SYNC, t0);
    }
    __device__ __forceinline__ double* U(int l) const { return ws + lev[l].voff; }
    __device__ __forceinline__ double* T(int l) const { return ws + lev[l].voff + lev[l].n_bar; }
    __device__ __forceinline__ double* S(int l) const { return ws + lev[l].voff + 2 * (size_t)lev[l].n_bar; }
    __device__ __forceinline__ double* F(int l) const { return ws + lev[l].voff + 3 * (size_t)lev[l].n_bar; }

    // ---- Alg. 2 P:475 + Alg. 4: f_l = r_l on D_l ; u = t = s = 0 ----
    __device__ __forceinline__ void begin_subdomain() {
        for (int l = 0; l <= L; ++l) {
            const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
            const int* gid = lev[l].gid;
            const double* r = prm->r_all + prm->r_off[l];
            double* u = U(l);
            for (int i = tid; i < 3 * n_bar; i += NTHREADS) u[i] = 0.0;   // u | t | s are adjacent
            double* f = F(l);
            for (int i = tid; i < n_real; i += NTHREADS) f[i] = __ldg(r + __ldg(gid + i));
        }
    }
    // ---- Alg. 2: x <- x + u_0^p on Omega_0^p (disjoint targets across subdomains) ----
    __device__ __forceinline__ void end_subdomain(int p) {
        const DevSub sb = prm->sub[p];
        const double* u0 = U(0);
        const int* gid0 = lev[0].gid;
        for (int k = tid; k < sb.n_owned; k += NTHREADS) {
            const int li = __ldg(sb.owned + k);
            prm->x[__ldg(gid0 + li)] += u0[li];
        }
    }
    // level 0, first iteration: u_0 = 0, so the first sweep is delta = D^{-1} f (P:507 with A u = 0)
    __device__ __forceinline__ void first0(const FacOp op) {
        const XB xo = xbuf_of(op.gbuf ^ 1, 0);
        const int n_real = lev[0].n_real, n_bar = lev[0].n_bar;
        const double* dinv = lev[0].dinv;
        double *u = U(0), *t = T(0);
        const double* f = F(0);
        const bool cfmode = op.flags & OPF_CF;                               // CF smoother: the C half of the sweep; the F half follows
        const int* gid = lev[0].gid;
        for (int i = tid; i < n_bar; i += NTHREADS) {
            double dl = 0.0;
            if (i < n_real && !(cfmode && prm->cf0[__ldg(gid + i)] <= 0)) { dl = __ldg(dinv + i) * f[i]; u[i] = dl; t[i] += dl; }
            xo.st(i, dl);
        }
    }
    // u_L = A_L^{-1} f_L with the LU factors computed at setup (Alg. 4).  One warp; columns
    // of the unit-lower / upper factors are contiguous (column-major).  The solve runs in place in
    // the output vector buffer.
    __device__ __forceinline__ void coarse(const FacOp op) {
        const XB y = xbuf_of(op.gbuf ^ 1, L);
        const int n = prm->nL;
        const double* __restrict__ lu = prm->lu;
        const double* f = F(L);
        for (int i = tid; i < n; i += NTHREADS) y.st(i, f[__ldg(prm->rowperm + i)]);
        sync();
        if (wid == 0) {
            for (int c = 0; c < n; ++c) {                      // forward: L y = P f
                const double yc = y.ld(c);
                for (int i = c + 1 + lane; i < n; i += 32) y.st(i, y.ld(i) - __ldg(lu + (size_t)c * n + i) * yc);
                __syncwarp();
            }
            for (int c = n - 1; c >= 0; --c) {                 // backward: U u = y
                if (lane == 0) y.st(c, y.ld(c) / __ldg(lu + (size_t)c * n + c));
                __syncwarp();
                const double yc = y.ld(c);
                for (int i = lane; i < c; i += 32) y.st(i, y.ld(i) - __ldg(lu + (size_t)c * n + i) * yc);
                __syncwarp();
            }
        }
        sync();
        double* uL = U(L);
        for (int i = tid; i < n; i += NTHREADS) uL[i] = y.ld(i);
    }

    // work of a step that is not row-local to the mat-vec's rows (all threads; touches only data
    // that neither the gathers nor the epilogues of THIS step use, so no barrier follows it)
    __device__ __forceinline__ void pre_actions(const FacOp op) {
        const XB xg = xbuf_of(op.gbuf, gather_level(op)), xo = xbuf_of(op.gbuf ^ 1, out_level(op));
        const int l = op.level;
        if (op.kind == OPK_RELAX) {                 // ghost values are fixed (A4): carry them (u) or clear them (t)
            const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
            if (op.flags & OPF_TSMEM) { for (int i = n_real + tid; i < n_bar; i += NTHREADS) xo.st(i, 0.0); }
            else { for (int i = n_real + tid; i < n_bar; i += NTHREADS) xo.st(i, xg.ld(i)); }
        } else if (op.kind == OPK_AT) {             // P:512 t_l <- 0 (its values are in the gather buffer)
            double* t = T(l);
            const int n_real = lev[l].n_real;
            for (int i = tid; i < n_real; i += NTHREADS) t[i] = 0.0;
        } else if (op.kind == OPK_RESTRICT) {       // later iterations: stage u_{l+1} for the recalculation that follows
            if (!(op.flags & OPF_FIRST)) {
                const double* uc = U(l + 1);
                const int nbc = lev[l + 1].n_bar;
                for (int i = tid; i < nbc; i += NTHREADS) xo.st(i, uc[i]);
            }
        } else if (op.kind == OPK_RECALC) {         // P:506 u_{l+1} <- 0 on the ghost points too
            if (!(op.flags & OPF_COARSEST)) {
                const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
                double* u = U(l);
                for (int i = n_real + tid; i < n_bar; i += NTHREADS) { xo.st(i, 0.0); u[i] = 0.0; }
            }
        }
    }

    // one mat-vec of the program: the groups of this warp's way, in order
    template <bool WIDE, bool GS>
    __device__ __forceinline__ void matvec(const FacOp op) {
        constexpr int GB = WIDE ? GROUP_BYTES_WIDE : GROUP_BYTES_NARROW;
        const long long tp0 = tick();
        const int kind = op.kind, l = op.level;
        const bool first = op.flags & OPF_FIRST, tsmem = op.flags & OPF_TSMEM, coarsest = op.flags & OPF_COARSEST;
        const bool half_c = op.flags & OPF_HALF_C, half_f = op.flags & OPF_HALF_F, cfmode = op.flags & OPF_CF;
        const XB xg = xbuf_of(op.gbuf, gather_level(op)), xo = xbuf_of(op.gbuf ^ 1, out_level(op));
        // ---- this warp's way of the stream, and of the next mat-vec's stream ----
        const WayEnt we = wt[stream_of(op) * NUM_WAYS + wid];
        const char* const sb = sbase[stream_of(op)];
        const uint64_t pol = (sflags[stream_of(op)] & STREAM_SHARED) ? pol_keep : pol_stream;
        uint64_t pol_nxt = pol_stream;
        const char* const we_hdr = sb + 128ull * we.hdr_off128;
        const bool ronly = real_rows_only(op);
        const int n = (int)(ronly ? we.n_real : we.n_all);
        const int nsl = (int)(ronly ? we.nsl_real : we.nsl_all);
        const char* const cur = sb + 128ull * we.grp_off128;
        const char* const dummy = reinterpret_cast<const char*>(prm->lev);     // always readable (>= 1536 bytes)
        const char* nxt = dummy;
        const char* nxt_hdr = dummy;
        int n_next = 0;
        if (op.next_mat >= 0 && (bool)(sflags[stream_of(ops[op.next_mat])] & STREAM_WIDE) == WIDE) {   // (the ring holds one group shape)
            const FacOp nop = ops[op.next_mat];
            const WayEnt w2 = wt[stream_of(nop) * NUM_WAYS + wid];
            n_next = (int)(real_rows_only(nop) ? w2.n_real : w2.n_all);
            if (sflags[stream_of(nop)] & STREAM_SHARED) pol_nxt = pol_keep;
            if (n_next > 0) { const char* b2 = sbase[stream_of(nop)]; nxt = b2 + 128ull * w2.grp_off128; nxt_hdr = b2 + 128ull * w2.hdr_off128; }
        }
        const int next_last = n_next > 0 ? n_next - 1 : 0;
        // ---- groups of this mat-vec that are not in the ring yet (first mat-vec of a subdomain, or after a short one) ----
        if (!ring_valid && n > 0) {
            if (phase == 0) {
#pragma unroll
                for (int d = 0; d < D; ++d) ra[d] = load_grp<WIDE>(cur + (long long)(d < n - 1 ? d : n - 1) * GB, lane, pol);
            } else {
#pragma unroll
                for (int d = 0; d < D; ++d) rb[d] = load_grp<WIDE>(cur + (long long)(d < n - 1 ? d : n - 1) * GB, lane, pol);
            }
        }
        // ---- the row-local operands of the epilogue (level vectors in the workspace slot) ----
        double* pu = nullptr; double* pt = nullptr; double* ps = nullptr; double* pf = nullptr;
        const double *cA = nullptr, *cB = nullptr, *cC = nullptr;
        int nr = 0;                                                          // real rows of the epilogue's level
        if (kind == OPK_RELAX) { pu = U(l); pt = T(l); cA = F(l); cB = pt; }
        else if (kind == OPK_AT) { cA = S(l); }
        else if (kind == OPK_RESTRICT) {
            ps = S(l + 1); nr = lev[l + 1].n_real;
            if (first) { pf = F(l + 1); pu = U(l + 1); pt = T(l + 1); cA = pf; cB = pt; }
        } else if (kind == OPK_RECALC) { pf = F(l); pu = U(l); pt = T(l); cA = pf; cB = S(l); cC = pt; }
        else { pu = U(l); cA = pu; nr = lev[l].n_real; }
        // ---- slice bookkeeping ----
        // The header of a slice and the row-local operands of its epilogue reach the warp through a
        // small lane-private staging area in shared memory, filled by cp.async one slice ahead:
        // asynchronous copies complete on their own scoreboard, so waiting for them does not wait
        // for the ring's loads in flight (all ordinary global loads of a warp share one).
        //   stage:  H  32 x 4 (wide: 8) bytes  header of the next slice (after the last slice: slice 0 of the next mat-vec)
        //           D  32 x 8 bytes at 256    the l1 diagonal inverse of the current slice's rows (where the step relaxes)
        //           C  3 x 32 x 8 bytes at 512  operands e0 | e1 | e2 of the current slice's epilogue
        if (n == 0) {
            // Nothing to do for this warp in this step (a stream with fewer slices than ways): use the time
            // to fetch the first block and the first header of the next mat-vec, so that the steps on the
            // small coarse levels do not each start with a full round trip to memory.
            ring_valid = hdr_ready = n_next > 0;
            if (n_next > 0) {
                if (phase == 0) {
#pragma unroll
                    for (int d = 0; d < D; ++d) ra[d] = load_grp<WIDE>(nxt + (long long)(d < next_last ? d : next_last) * GB, lane, pol_nxt);
                } else {
#pragma unroll
                    for (int d = 0; d < D; ++d) rb[d] = load_grp<WIDE>(nxt + (long long)(d < next_last ? d : next_last) * GB, lane, pol_nxt);
                }
                cp_async_wait_all();
                if (WIDE) cp_async8(stage + 8 * lane, nxt_hdr + 8 * lane);
                else cp_async4(stage + 4 * lane, nxt_hdr + 4 * lane);
                cp_async_issued();
            }
            tock(PROF_OP0 + kind, tp0);
            return;
        }
        constexpr int HL = WIDE ? 8 : 4, HB = WIDE ? HEADER_BYTES_WIDE : HEADER_BYTES_NARROW;   // header bytes per lane / per slice
        const char* const hdr = we_hdr + HL * lane;
        const uint32_t stH = stage + HL * lane, stD = stage + 256 + 8 * lane, stC = stage + 512 + 8 * lane;
        const char* const hdr_after = nxt_hdr + HL * lane;
        auto fetch_ctx = [&](uint32_t r) {
            if (r != NO_ROW) {
                if (cA) cp_async8(stC, cA + r);
                if (cB) cp_async8(stC + 256, cB + r);
                if (cC) cp_async8(stC + 512, cC + r);
                // the l1 diagonal inverse of the rows that relax (S8; the level's dinv array has n_bar entries, 0.0 on ghosts);
                // the pointer is read from the level table where it is needed: it is not worth two registers of the ring loop
                if (kind == OPK_RELAX || ((kind == OPK_RECALC || (kind == OPK_RESTRICT && first)) && !coarsest))
                    cp_async8(stD, lev[kind == OPK_RESTRICT ? l + 1 : l].dinv + r);
            }
        };
        auto fetch_hdr = [&](const char* src) { if (WIDE) cp_async8(stH, src); else cp_async4(stH, src); };
        uint32_t row;
        int left;
        bool is_c;                                                          // the row is a C-point of its level
        auto read_hdr = [&]() {                                             // narrow: row | K << 16 | flag << 31; wide: row, K | flag << 31
            if (WIDE) { const uint2 w = lds_u64(stH); row = w.x; left = (int)(w.y & HDR_GROUPS_MASK); is_c = (w.y >> 31) != 0; }
            else {
                const uint32_t w = lds_u32(stH);
                row = (w & 0xFFFFu) == 0xFFFFu ? NO_ROW : (w & 0xFFFFu);
                left = (int)((w >> 16) & 0x7FFFu); is_c = (w >> 31) != 0;
            }
        };
        if (!hdr_ready) { cp_async_wait_all(); fetch_hdr(hdr); cp_async_issued(); }       // (never two copies in flight to one slot)
        cp_async_wait_all();
        read_hdr();
        double aux = 0.0;
        fetch_ctx(row);
        fetch_hdr(nsl > 1 ? hdr + HB : hdr_after);
        cp_async_issued();
        hdr_ready = n_next > 0;
        int sidx = 0;
        double acc = 0.0;
        auto consume = [&](const Grp& g) {
            uint32_t c0, c1, c2, c3;
            if (WIDE) { c0 = g.c.x; c1 = g.c.y; c2 = g.c.z; c3 = g.c.w; }
            else { c0 = g.c.x & 0xffffu; c1 = g.c.x >> 16; c2 = g.c.y & 0xffffu; c3 = g.c.y >> 16; }
            const double x0 = xg.template ldt<GS>(c0), x1 = xg.template ldt<GS>(c1), x2 = xg.template ldt<GS>(c2), x3 = xg.template ldt<GS>(c3);
            acc = fma(mkdouble(g.a.x, g.a.y), x0, acc);
            acc = fma(mkdouble(g.a.z, g.a.w), x1, acc);
            acc = fma(mkdouble(g.b.x, g.b.y), x2, acc);
            acc = fma(mkdouble(g.b.z, g.b.w), x3, acc);
        };
        auto slice_end = [&]() {
            const long long tw0 = tick();
            cp_async_wait_all();
            const uint32_t stE = stC;
            tock(14, tw0);
            tock_op(3, tw0);
            if (row != NO_ROW) {
                const double e0 = lds_f64(stE), e1 = lds_f64(stE + 256), e2 = lds_f64(stE + 512);   // unused ones are stale, never read
                aux = lds_f64(stD);
                if (kind == OPK_RELAX) {           // one l1-Jacobi update (§4.1); aux = 1 / sum_j |a_ij| (S8)
                    const double uo = xg.ld(row);
                    if ((half_c && !is_c) || (half_f && is_c)) {   // CF smoother: not this half-sweep's class
                        xo.st(row, tsmem ? e1 : uo);
                    } else {
                        const double dl = aux * (e0 - acc);
                        const double un = uo + dl, tn = e1 + dl;
                        pu[row] = un; pt[row] = tn;
                        xo.st(row, tsmem ? tn : un);
                    }
                } else if (kind == OPK_AT) {       // P:509 w = s_l + A_l t_l
                    xo.st(row, e0 + acc);
                } else if (kind == OPK_RESTRICT) { // P:509 s_{l+1} = R_l w
                    ps[row] = acc;
                    if (first) {                   // P:511 with A u = 0, then P:506-508 of level l+1: delta = D^-1 f
                        if ((int)row < nr) {
                            const double f = e0 - acc;
                            pf[row] = f;
                            if (!coarsest) {
                                const double u = (cfmode && !is_c) ? 0.0 : aux * f, tn = e1 + u;   // CF smoother: the C half of the sweep
                                pu[row] = u; pt[row] = tn;
                                xo.st(row, tsmem ? tn : u);
                            }
                        } else if (!coarsest) xo.st(row, 0.0);
                    }
                } else if (kind == OPK_RECALC) {   // P:510-511, then P:506-508 of the same level
                    const double f = (e0 - acc) - e1;
                    pf[row] = f;
                    if (!coarsest) {
                        const double u = (cfmode && !is_c) ? 0.0 : aux * f, tn = e2 + u;           // CF smoother: the C half of the sweep
                        pu[row] = u; pt[row] = tn;
                        xo.st(row, tsmem ? tn : u);
                    }
                } else {                           // OPK_INTERP
                    const double un = e0 + acc;
                    xo.st(row, un);
                    if ((int)row >= nr) pu[row] = un;              // ghost values are not relaxed: keep them
                }
            }
            ++sidx;
            acc = 0.0;
            if (sidx < nsl) {
                read_hdr();
                fetch_ctx(row);
                fetch_hdr(sidx + 1 < nsl ? hdr + (long long)(sidx + 1) * HB : hdr_after);
                cp_async_issued();
            }
        };
        tock(PROF_PRIME, tp0);
        // Blocks of D groups, double buffered in registers: WAIT for block j (buffer X), then issue
        // the burst of block j+1 into the other buffer (the next D groups of this mat-vec or, after
        // its last block, the first D groups of the next mat-vec), then consume block j while
        // that burst is in flight.  All ordinary global loads of a warp share one hardware
        // scoreboard, so a wait on any of them waits for all: the burst must not be issued before
        // the data of block j has arrived.  That order is forced by a data dependence: the
        // burst's base address is selected by a bit pattern of block j's first value that no
        // finite matrix entry has (Inf/NaN exponent), so the address cannot be formed earlier.
        auto step = [&](Grp (&X)[D], Grp (&Y)[D], int p0) {
            const bool more = p0 + D < n;
            const long long tr0 = tick();
            const bool never = (X[0].a.y & 0x7FF00000u) == 0x7FF00000u;
            if (PROF && never) prof_s[15] += 1;          // (keeps the read of X[0] before the second clock read)
            tock(15, tr0);
            tock_op(2, tr0);
            const char* rbase = never ? dummy : (more ? cur : nxt);
            const int r0 = more ? p0 + D : 0, rlast = never ? 0 : (more ? n - 1 : next_last);
            const uint64_t pol_b = more ? pol : pol_nxt;
#if !AMGDD_SINGLE_BUFFER
#pragma unroll
            for (int d = 0; d < D; ++d) Y[d] = load_grp<WIDE>(rbase + (long long)(r0 + d < rlast ? r0 + d : rlast) * GB, lane, pol_b);
#endif
            const int nv = n - p0 < D ? n - p0 : D;     // groups of this block (the last block of a mat-vec may be short)
            if (left > nv && nv == D) {                 // no slice ends inside this block: straight-line code
#pragma unroll
                for (int d = 0; d < D; ++d) consume(X[d]);
                left -= D;
            } else {
                // general case: consume up to the next slice end, run the epilogue (ONE copy of its code per
                // buffer: the kernel's instruction footprint matters), resume behind it
                int d = 0;
                bool ended;
                do {
                    ended = false;
#pragma unroll
                    for (int dd = 0; dd < D; ++dd)
                        if (!ended && dd >= d && dd < nv) {
                            consume(X[dd]);
                            d = dd + 1;
                            if (--left == 0) ended = true;
                        }
                    if (ended) slice_end();
                } while (ended && d < nv);
            }
#if AMGDD_SINGLE_BUFFER
#pragma unroll
            for (int d = 0; d < D; ++d) X[d] = load_grp<WIDE>(rbase + (long long)(r0 + d < rlast ? r0 + d : rlast) * GB, lane, pol_b);
#endif
        };
        int ph = phase;
        for (int p0 = 0; p0 < n; p0 += D) {
#if AMGDD_SINGLE_BUFFER
            step(ra, ra, p0);
#else
            if (ph == 0) step(ra, rb, p0);
            else step(rb, ra, p0);
            ph ^= 1;
#endif
        }
        phase = ph;
        ring_valid = n_next > 0;
        tock(PROF_OP0 + kind, tp0);
    }
};

template <bool PROF>
__global__ void __launch_bounds__(NTHREADS, CTAS_PER_SM) fac_kernel(const FacParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const int L = prm.L, nstreams = 3 * (L + 1);
    // shared-memory plan (fac_smem_bytes): control | ops | LevInfo | stream flags | stream bases | way table | staging areas | two vector buffers
    int* ctrl = reinterpret_cast<int*>(smem);
    FacOp* ops = reinterpret_cast<FacOp*>(smem + 128);
    LevInfo* lev = reinterpret_cast<LevInfo*>(smem + 128 + (((size_t)prm.nops * sizeof(FacOp) + 127) & ~(size_t)127));
    uint32_t* sflags = reinterpret_cast<uint32_t*>(lev + (L + 1));
    const char** sbase = reinterpret_cast<const char**>(reinterpret_cast<unsigned char*>(sflags) + (((size_t)nstreams * 4 + 127) & ~(size_t)127));
    WayEnt* wt = reinterpret_cast<WayEnt*>(reinterpret_cast<unsigned char*>(sbase) + (((size_t)nstreams * 8 + 127) & ~(size_t)127));
    unsigned char* stage = reinterpret_cast<unsigned char*>(wt) + (((size_t)nstreams * NUM_WAYS * sizeof(WayEnt) + 127) & ~(size_t)127);
    double* xbuf = reinterpret_cast<double*>(stage + NUM_WAYS * STAGE_BYTES);

    Worker<PROF> W;
    W.prm = &prm; W.ops = ops; W.lev = lev; W.wt = wt; W.sflags = sflags; W.sbase = sbase;
    W.tid = threadIdx.x; W.lane = threadIdx.x & 31; W.wid = threadIdx.x >> 5; W.L = L;
    W.ws = prm.workspace + (size_t)blockIdx.x * prm.slot_stride;
    W.xs0 = (uint32_t)__cvta_generic_to_shared(xbuf);
    W.xs1 = W.xs0 + (uint32_t)prm.x_cap * 8u;
    W.xg0 = W.ws + prm.xg_off;
    W.xg1 = W.xg0 + (prm.slot_stride - prm.xg_off) / 2;
    W.x_cap = prm.x_cap;
    W.prof = PROF ? prm.prof + (size_t)blockIdx.x * FAC_PROF_SLOTS : nullptr;
    W.prof_s = reinterpret_cast<long long*>(smem + prm.prof_smem_off);
    if (PROF) { for (int i = threadIdx.x; i < FAC_PROF_SLOTS + 4 * PROF_OPS_SMEM; i += NTHREADS) W.prof_s[i] = 0; }
    W.pol_stream = policy_evict_first(); W.pol_keep = policy_evict_last();
    W.ring_valid = false; W.hdr_ready = false;
    W.stage = (uint32_t)__cvta_generic_to_shared(stage) + (uint32_t)W.wid * STAGE_BYTES;
#pragma unroll
    for (int d = 0; d < D; ++d) W.ra[d].a = W.ra[d].b = W.ra[d].c = W.rb[d].a = W.rb[d].b = W.rb[d].c = make_uint4(0, 0, 0, 0);
    W.phase = 0;

    for (int j = threadIdx.x; j < prm.nops; j += NTHREADS) ops[j] = prm.ops[j];
    const long long tk0 = W.tick();
    for (;;) {
        const long long ts0 = W.tick();
        if (threadIdx.x == 0) {
            const int id = atomicAdd(prm.work_counter, 1);
            ctrl[0] = id < prm.num_sub ? prm.order[id] : -1;
        }
        __syncthreads();
        const int p = ctrl[0];
        if (p < 0) break;
        const DevLevel* tbl = prm.lev + (size_t)p * (L + 1);
        for (int l = threadIdx.x; l <= L; l += NTHREADS) {
            LevInfo li;
            li.n_real = tbl[l].n_real; li.n_bar = tbl[l].n_bar; li.voff = tbl[l].voff; li.gid = tbl[l].gid; li.dinv = tbl[l].dinv;
            lev[l] = li;
        }
        for (int idx = threadIdx.x; idx < nstreams * NUM_WAYS; idx += NTHREADS) {
            const int s = idx / NUM_WAYS, w = idx % NUM_WAYS;
            const StreamDesc* sd = &tbl[s / 3].A + (s % 3);                  // A, P, R are consecutive members
            const char* base = sd->base;
            const WayDesc wd = sd->way[w];
            WayEnt e;
            e.grp_off128 = wd.grp_off128; e.hdr_off128 = wd.hdr_off128;
            e.n_all = wd.ngroups; e.n_real = wd.ngroups_real; e.nsl_all = wd.nslices; e.nsl_real = wd.nslices_real;
            wt[idx] = e;
            if (w == 0) { sflags[s] = sd->flags; sbase[s] = base; }
        }
        __syncthreads();
        W.tock(PROF_SETUP, ts0);
        W.ring_valid = false; W.hdr_ready = false;
        for (int j = 0; j < prm.nops; ++j) {
            const FacOp op = ops[j];
            W.opj = j;
            const long long tp0 = W.tick();
            if (op.kind == OPK_BEGIN) W.begin_subdomain();
            else if (op.kind == OPK_FIRST0) W.first0(op);
            else if (op.kind == OPK_COARSE) W.coarse(op);
            else if (op.kind == OPK_END) W.end_subdomain(p);
            else {
                W.pre_actions(op);
                W.tock(PROF_PRE, tp0);
                if (sflags[stream_of(op)] & STREAM_WIDE) W.template matvec<true, false>(op);
                else if (lev[gather_level(op)].n_bar <= prm.x_cap) W.template matvec<false, true>(op);
                else W.template matvec<false, false>(op);
            }
            if (!is_matvec(op.kind)) W.tock(PROF_OP0 + op.kind, tp0);
            long long tq0 = 0;
            if (PROF) { W.tock_op(0, tp0); tq0 = clock64(); }
            W.sync();                                                    // the step is complete
            if (PROF) W.tock_op(1, tq0);
        }
    }
    W.tock(PROF_TOTAL, tk0);
    if (PROF && threadIdx.x == 0) {                                          // flush the counters of this CTA
        for (int i = 0; i < FAC_PROF_SLOTS; ++i) W.prof[i] += W.prof_s[i];
        if (prm.prof_ops)
            for (int q = 0; q < 4; ++q)
                for (int j = 0; j < PROF_OPS_SMEM && j < prm.nops; ++j)
                    prm.prof_ops[(size_t)blockIdx.x * PROF_OPS_STRIDE + q * MAX_OPS + j] += W.prof_s[FAC_PROF_SLOTS + q * PROF_OPS_SMEM + j];
    }
}

}  // namespace

// The static program of one subdomain: the steps of num_fac_cycles AlgFAC V(nu,nu)-cycles (Alg. 4)
// in order, with the shared-memory buffer each mat-vec gathers from (it writes the other one).
int fac_build_program(int L, int nfac, int nu, int smoother, FacOp* ops) {
    int n = 0;
    auto emit = [&](int kind, int level, int gbuf, int flags) {
        if (ops && n < MAX_OPS) {
            FacOp o;
            o.kind = (uint8_t)kind; o.level = (uint8_t)level; o.gbuf = (uint8_t)gbuf; o.flags = (uint8_t)flags;
            o.next_mat = -1; o.pad_ = 0;
            ops[n] = o;
        }
        ++n;
    };
    const bool cf = smoother == 1;                                           // CF l1-Jacobi: two half-sweeps per sweep
    int cur = 0;                                                             // buffer that holds the live gather vector
    // one relaxation sweep on level l (P:507-508 / P:517-518); `last_pre`: the A t step follows, leave t behind;
    // `skip_first_half`: the sweep's first half was the matrix-free sweep from u = 0 fused into the step before
    auto sweep = [&](int l, int first, bool pre, bool last_pre, bool skip_first_half) {
        if (!cf) { emit(OPK_RELAX, l, cur, first | (last_pre ? OPF_TSMEM : 0)); cur ^= 1; return; }
        const int h1 = pre ? OPF_HALF_C : OPF_HALF_F, h2 = pre ? OPF_HALF_F : OPF_HALF_C;   // C then F before, F then C after the coarse correction
        if (!skip_first_half) { emit(OPK_RELAX, l, cur, first | h1); cur ^= 1; }
        emit(OPK_RELAX, l, cur, first | h2 | (last_pre ? OPF_TSMEM : 0)); cur ^= 1;
    };
    const int cff = cf ? OPF_CF : 0;
    emit(OPK_BEGIN, 0, 0, 0);                                                // Alg. 2, Alg. 4
    for (int it = 0; it < nfac; ++it) {
        const int first = it == 0 ? OPF_FIRST : 0;
        // does the sweep from u = 0, fused into the step before, leave t (not u) in the buffer?  only if nothing follows it
        const int fused_t = (nu == 1 && !cf) ? OPF_TSMEM : 0;
        for (int l = 0; l < L; ++l) {                                        // downsweep P:505-513
            const int coarsest = (l + 1 == L) ? OPF_COARSEST : 0;
            int k = 0;
            bool fused = false;
            if (l == 0 && first) { emit(OPK_FIRST0, 0, cur, first | fused_t | cff); cur ^= 1; fused = true; }
            if (l != 0) fused = true;                                        // fused into the restriction / recalculation before
            if (fused) { if (cf) sweep(l, first, true, nu == 1, true); k = 1; }
            for (; k < nu; ++k) sweep(l, first, true, k == nu - 1, false);
            emit(OPK_AT, l, cur, first); cur ^= 1;                           // P:509  w = s_l + A_l t_l
            const int fl = first | coarsest | fused_t | cff;
            emit(OPK_RESTRICT, l, cur, fl); cur ^= 1;                        // P:509  s_{l+1} = R_l w 
            if (!first) { emit(OPK_RECALC, l + 1, cur, fl); cur ^= 1; }      // P:510  (identically zero at it = 0)
        }
        emit(OPK_COARSE, L, cur, first); cur ^= 1;
        for (int l = L - 1; l >= 0; --l) {                                   // upsweep P:515-519
            emit(OPK_INTERP, l, cur, first); cur ^= 1;
            for (int k = 0; k < nu; ++k) sweep(l, first, false, false, false);
        }
    }
    emit(OPK_END, 0, 0, 0);                                                  // Alg. 2
    if (ops && n <= MAX_OPS) {
        int nm = -1;
        for (int j = n - 1; j >= 0; --j) {
            ops[j].next_mat = (int16_t)nm;
            if (ops[j].kind >= OPK_RELAX && ops[j].kind <= OPK_INTERP) nm = j;
        }
    }
    return n;
}

int fac_smem_bytes(int x_cap, int L, int nops) {
    const int nstreams = 3 * (L + 1);
    size_t b = 128;
    b += ((size_t)nops * sizeof(FacOp) + 127) & ~(size_t)127;
    b += (size_t)(L + 1) * sizeof(LevInfo);
    b += ((size_t)nstreams * 4 + 127) & ~(size_t)127;
    b += ((size_t)nstreams * 8 + 127) & ~(size_t)127;
    b += ((size_t)nstreams * NUM_WAYS * sizeof(WayEnt) + 127) & ~(size_t)127;
    b += (size_t)NUM_WAYS * STAGE_BYTES;
    b += 2 * (size_t)x_cap * 8;
    return (int)b;
}

int fac_configure(int /*device*/, int max_smem_optin) {
    cudaError_t e = cudaFuncSetAttribute(fac_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fac_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
    return e == cudaSuccess ? 0 : (int)e;
}

void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    if (prm.prof) fac_kernel<true><<<cfg.grid, cfg.block, cfg.smem_bytes, st>>>(prm);
    else fac_kernel<false><<<cfg.grid, cfg.block, cfg.smem_bytes, st>>>(prm);
}

}  // namespace amgdd
