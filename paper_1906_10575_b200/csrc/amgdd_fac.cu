// The persistent AlgFAC kernel (sm_100a): Alg. 2 lines P:475-479 with Alg. 4 inside.
//
// One CTA per SM slot takes whole subdomains from a work counter and runs ALL num_fac_cycles
// AlgFAC V(nu,nu)-cycles of a subdomain start to finish; subdomains never communicate.
// The CTA is warp-specialised:
//   warp 0 (one elected lane) = PRODUCER.  It walks the same static "program" of mat-vecs as the
//     consumers and streams every matrix chunk (amgdd_stream.hpp) HBM -> shared-memory ring with
//     cp.async.bulk (TMA, SASS UBLKCP), completion on an mbarrier per ring slot.  Matrix data does
//     not depend on computed values, so the producer runs ahead across mat-vec, level and even
//     subdomain boundaries, as far as the ring allows: HBM requests are large, contiguous and
//     independent of any warp's progress.  It also draws the next subdomain from the counter and
//     announces it through a zero-byte "control" slot of the ring.
//   warps 1.. = CONSUMERS.  Per mat-vec they stage the gather vector in shared memory, then take
//     ring slots in order; inside a chunk, `lanes` threads share a row, rows go round-robin to
//     warps by global row index (balanced across chunk boundaries), the row sum is reduced by
//     shuffles and a row-local epilogue applies the AlgFAC update.  Consumers sync among
//     themselves with a named barrier; a warp releases a ring slot with one mbarrier arrive.
// The level vectors u, t, s, f live in a per-CTA workspace slot in global memory that every
// subdomain of the CTA reuses (L2-resident); what streams from HBM is matrix data, once per
// mat-vec.  Every row sum has a fixed summation order, so results are run-to-run identical.
#include "amgdd_stream.hpp"

#include <cuda_runtime.h>

#include <climits>
#include <type_traits>

namespace amgdd {

namespace {

constexpr int MAX_STAGES = 24;
constexpr int CTRL_BYTES = 1024;

struct Ctrl {
    unsigned long long full[MAX_STAGES];    // producer arrive (+ TMA bytes) -> consumers wait
    unsigned long long empty[MAX_STAGES];   // one arrive per consumer warp -> producer waits
    int slot_sub[MAX_STAGES];               // control slots: subdomain id, or -1 = no more work
};
static_assert(sizeof(Ctrl) <= CTRL_BYTES, "control block too large");

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(void* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void* bar) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(void* bar, uint32_t bytes) {
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(smem_addr(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(void* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(void* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 1-D bulk async copy global -> shared (TMA), completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_copy_g2s(void* dst, const void* src, uint32_t bytes, void* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(smem_addr(dst)),
        "l"(src), "r"(bytes), "r"(smem_addr(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void bar_consumers(int nthreads) {
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}

enum OpKind { OP_RELAX = 0, OP_AT = 1, OP_RESTRICT = 2, OP_RECALC = 3, OP_INTERP = 4 };
// slots of the optional per-CTA cycle counters (FAC_PROF_SLOTS each; amgdd_debug_fac_cycles)
enum ProfSlot { PROF_SYNC = 0, PROF_WAIT_FULL = 1, PROF_CONSUME = 2, PROF_STAGE = 3, PROF_WAIT_EMPTY = 4, PROF_BEGIN = 5,
                PROF_END = 6, PROF_FIRST = 7, PROF_COARSE = 8, PROF_TOTAL = 9, PROF_OP0 = 10 };

// The static program of one subdomain: the order of the mat-vecs of num_fac_cycles AlgFAC
// V(nu,nu)-cycles (Alg. 4).  Producer and consumers both run it, so they agree on the sequence
// of ring slots by construction.
template <class Role>
__device__ __forceinline__ void fac_program(Role& r, int L, int nfac, int nu) {
    r.begin_subdomain();
    for (int it = 0; it < nfac; ++it) {
        for (int l = 0; l < L; ++l) {                                      // downsweep P:505-513
            int sweeps = nu;
            if (l != 0) { r.first_sweep(l); --sweeps; }                    // u_l = 0, so delta = D^-1 f
            for (int k = 0; k < sweeps; ++k) r.template stream<OP_RELAX>(l, it);
            r.template stream<OP_AT>(l, it);                               // P:509  w = s_l + A_l t_l
            r.template stream<OP_RESTRICT>(l, it);                         // P:509  s_{l+1} = R_l w 
            if (it > 0) r.template stream<OP_RECALC>(l, it);               // P:510  (identically zero at it = 0)
        }
        r.coarse();
        for (int l = L - 1; l >= 0; --l) {                                 // upsweep P:515-519
            r.template stream<OP_INTERP>(l, it);
            for (int k = 0; k < nu; ++k) r.template stream<OP_RELAX>(l, it);
        }
    }
    r.end_subdomain();
}

// ---- producer -------------------------------------------------------------------------------
struct Producer {
    Ctrl* ctrl;
    char* ring;
    const DevLevel* lev;
    int stages, chunk_bytes;
    int slot;
    uint32_t phase;
    uint64_t policy;

    long long* prof;
    __device__ __forceinline__ void acquire() {
        const long long t0 = prof ? clock64() : 0;
        mbar_wait(&ctrl->empty[slot], phase ^ 1u);
        if (prof) prof[PROF_WAIT_EMPTY] += clock64() - t0;
    }
    __device__ __forceinline__ void advance() {
        if (++slot == stages) { slot = 0; phase ^= 1u; }
    }
    __device__ __forceinline__ void control(int p) {
        acquire();
        ctrl->slot_sub[slot] = p;
        mbar_arrive(&ctrl->full[slot]);
        advance();
    }
    __device__ __forceinline__ void push(const StreamDesc& d, int nchunks) {
        const char* src = d.base;
        for (int c = 0; c < nchunks; ++c) {
            acquire();
            const uint32_t bytes = (c == d.nchunks - 1) ? (uint32_t)d.last_bytes : (uint32_t)chunk_bytes;
            mbar_arrive_expect_tx(&ctrl->full[slot], bytes);
            bulk_copy_g2s(ring + (size_t)slot * chunk_bytes, src + (size_t)c * chunk_bytes, bytes, &ctrl->full[slot], policy);
            advance();
        }
    }
    __device__ __forceinline__ void begin_subdomain() {}
    __device__ __forceinline__ void end_subdomain() {}
    __device__ __forceinline__ void first_sweep(int) {}
    __device__ __forceinline__ void coarse() {}
    template <int K>
    __device__ __forceinline__ void stream(int l, int) {
        if (K == OP_RELAX) { const StreamDesc d = lev[l].A; push(d, d.nchunks_real); }
        else if (K == OP_AT) { const StreamDesc d = lev[l].A; push(d, d.nchunks); }
        else if (K == OP_RESTRICT) { const StreamDesc d = lev[l].R; push(d, d.nchunks); }
        else if (K == OP_RECALC) { const StreamDesc d = lev[l + 1].A; push(d, d.nchunks_real); }
        else { const StreamDesc d = lev[l].P; push(d, d.nchunks); }
    }
};

// ---- consumers ------------------------------------------------------------------------------
// What a row does with its finished sum (Alg. 4 step of the mat-vec); all pointers index the
// current level's vectors in this CTA's workspace slot.
struct Epilogue {
    int kind;              // OpKind, or OP_RELAX_DELTA
    int limit;             // OP_RESTRICT: rows below this are real rows of level l+1
    int first;             // OP_RESTRICT: first AlgFAC iteration
    double* a;             // RELAX u | AT w | RESTRICT s_{l+1} | RECALC f_{l+1} | INTERP u | RELAX_DELTA delta
    double* b;             // RELAX t | RESTRICT f_{l+1}
    const double* c;       // RELAX f | AT s | RECALC s_{l+1} | RELAX_DELTA f
};
constexpr int OP_RELAX_DELTA = 5;

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

// What a warp carries from piece to piece of the slice it is working on (a slice may span chunks).
struct SliceState {
    double acc, aux;
    int row;               // row of this lane, -1: none
    int len;               // entries of that row
    int snext;             // next slice of this warp (slices go round-robin to the consumer warps)
};

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

// One chunk in shared memory (layout: amgdd_stream.hpp), `slot` = its shared address.  The warp
// takes the pieces of its own slices; lane j owns row j of the slice and adds its entries in stored
// (= column) order, so there is no cross-lane reduction and every row sum has one fixed summation
// order.  Lanes whose row has ended re-read entry 0 of the piece and discard it: every load is
// unconditional, so the four steps of an unrolled block overlap.
template <bool WIDE, class X>
__device__ __forceinline__ void consume_chunk(uint32_t slot, X xs, int ncw, int slice_limit, int has_aux, SliceState& st,
                                              const Epilogue& ep) {
    constexpr int CS = WIDE ? 2 : 1;                               // log2 bytes per column index
    const int np = (int)lds_u32(slot), slice0 = (int)lds_u32(slot + 4);
    const int lane = threadIdx.x & 31;
    for (;;) {
        const int i = st.snext - slice0;
        if (i >= np || st.snext >= slice_limit) break;
        const uint4 raw = lds_v4(slot + CHUNK_HEADER_BYTES + i * PIECE_DESC_BYTES);
        const int k0 = (int)(raw.z & 0xFFFFu), nk = (int)(raw.z >> 16), K = (int)(raw.w & 0xFFFFu), nnz = (int)(raw.w >> 16);
        uint32_t q = slot + raw.x;
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
        if (kend != K) break;                                   // the slice continues in the next chunk
        if (st.row >= 0) apply(ep, st.row, acc, st.aux);
        st.snext += ncw;
    }
}

struct Consumer {
    Ctrl* ctrl;
    const char* ring;
    double* xbuf;              // shared-memory gather buffer, x_cap doubles
    const FacParams* prm;
    const DevLevel* lev;
    double* ws;                // this CTA's workspace slot
    double* w;                 // scratch vector inside the slot
    int p;                     // current subdomain
    int stages, chunk_bytes, x_cap;
    int slot;
    uint32_t phase;
    int ctid, nct, cw, ncw;    // consumer thread id / count, consumer warp id / count
    long long* prof;           // this CTA's cycle counters, or nullptr

    __device__ __forceinline__ double* U(int l) const { return ws + lev[l].voff; }
    __device__ __forceinline__ double* T(int l) const { return ws + lev[l].voff + lev[l].n_bar; }
    __device__ __forceinline__ double* S(int l) const { return ws + lev[l].voff + 2 * (size_t)lev[l].n_bar; }
    __device__ __forceinline__ double* F(int l) const { return ws + lev[l].voff + 3 * (size_t)lev[l].n_bar; }
    // optional cycle counters of this CTA (FacParams::prof), written by consumer thread 0 only
    __device__ __forceinline__ long long tick() const { return prof ? clock64() : 0; }
    __device__ __forceinline__ void tock(int idx, long long t0) const { if (prof && ctid == 0) prof[idx] += clock64() - t0; }
    __device__ __forceinline__ void sync() {
        const long long t0 = tick();
        bar_consumers(nct);
        tock(PROF_SYNC, t0);
    }
    __device__ __forceinline__ void advance() {
        if (++slot == stages) { slot = 0; phase ^= 1u; }
    }
    __device__ __forceinline__ void release() {
        __syncwarp();
        if ((threadIdx.x & 31) == 0) mbar_arrive(&ctrl->empty[slot]);
        advance();
    }
    // next control slot: the subdomain announced by the producer (-1: none left)
    __device__ __forceinline__ int next_subdomain() {
        mbar_wait(&ctrl->full[slot], phase);
        const int q = ctrl->slot_sub[slot];
        release();
        return q;
    }

    // ---- Alg. 2 P:475 + Alg. 4: f_l = r_l on D_l ; u = t = s = 0 ----
    __device__ __forceinline__ void begin_subdomain() {
        sync();
        const long long tp0 = tick();
        const int L = prm->L;
        for (int l = 0; l <= L; ++l) {
            const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
            const int* gid = lev[l].gid;
            const double* r = prm->r_all + prm->r_off[l];
            double* u = U(l);
            for (int i = ctid; i < 3 * n_bar; i += nct) u[i] = 0.0;      // u | t | s are adjacent
            double* f = F(l);
            for (int i = ctid; i < n_real; i += nct) f[i] = r[__ldg(gid + i)];
        }
        tock(PROF_BEGIN, tp0);
    }
    // ---- Alg. 2: x <- x + u_0^p on Omega_0^p (disjoint targets across subdomains) ----
    __device__ __forceinline__ void end_subdomain() {
        sync();
        const long long tp0 = tick();
        const DevSub sb = prm->sub[p];
        const double* u0 = U(0);
        const int* gid0 = lev[0].gid;
        for (int k = ctid; k < sb.n_owned; k += nct) {
            const int li = __ldg(sb.owned + k);
            prm->x[__ldg(gid0 + li)] += u0[li];
        }
        tock(PROF_END, tp0);
    }
    // P:506 u_l <- 0, then the first sweep needs no matrix: delta = D^{-1} f
    __device__ __forceinline__ void first_sweep(int l) {
        sync();
        const long long tp0 = tick();
        const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
        const double* dinv = lev[l].dinv;
        double *u = U(l), *t = T(l);
        const double* f = F(l);
        for (int i = ctid; i < n_bar; i += nct) {
            double dl = 0.0;
            if (i < n_real) { dl = __ldg(dinv + i) * f[i]; t[i] += dl; }
            u[i] = dl;
        }
        tock(PROF_FIRST, tp0);
    }
    // u_L = A_L^{-1} f_L with the LU factors computed at setup (Alg. 4).  One warp; columns
    // of the unit-lower / upper factors are contiguous (column-major).
    __device__ __forceinline__ void coarse() {
        sync();
        const long long tp0 = tick();
        const int L = prm->L, n = prm->nL;
        const double* __restrict__ lu = prm->lu;
        const double* f = F(L);
        double* y = (n <= x_cap) ? xbuf : w;
        for (int i = ctid; i < n; i += nct) y[i] = f[__ldg(prm->rowperm + i)];
        sync();
        if (cw == 0) {
            const int lane = threadIdx.x & 31;
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
        for (int i = ctid; i < n; i += nct) uL[i] = y[i];
        tock(PROF_COARSE, tp0);
    }

    // one mat-vec: every chunk of the stream prefix, in ring order; `staged`: the gather vector is in xbuf
    __device__ __forceinline__ void run_chunks(const StreamDesc& d, int nchunks, int slice_limit, bool staged, const double* xg,
                                               const Epilogue& ep) {
        extern __shared__ __align__(128) unsigned char smem_dyn[];      // same base as in fac_kernel: keeps LDS addressing
        SliceState st;
        st.acc = 0.0; st.aux = 0.0; st.row = -1; st.len = 0; st.snext = cw;
        for (int c = 0; c < nchunks; ++c) {
            const long long t0 = tick();
            mbar_wait(&ctrl->full[slot], phase);
            tock(PROF_WAIT_FULL, t0);
            const long long t1 = tick();
            const uint32_t sl = smem_addr(smem_dyn) + CTRL_BYTES + (uint32_t)x_cap * 8u + (uint32_t)slot * (uint32_t)chunk_bytes;
            if (staged) {
                SmemVec xs;
                xs.base = smem_addr(smem_dyn) + CTRL_BYTES;
                consume_chunk<false>(sl, xs, ncw, slice_limit, d.has_aux, st, ep);
            } else {
                GlobalVec xs;
                xs.base = xg;
                if (d.wide) consume_chunk<true>(sl, xs, ncw, slice_limit, d.has_aux, st, ep);
                else consume_chunk<false>(sl, xs, ncw, slice_limit, d.has_aux, st, ep);
            }
            tock(PROF_CONSUME, t1);
            release();
        }
    }

    // stage the gather vector of the next mat-vec in shared memory (if it fits; wide streams never do)
    __device__ __forceinline__ bool stage_x(const double* x, int n) {
        if (n > x_cap) return false;
        const long long t0 = tick();
        for (int i = ctid; i < n; i += nct) xbuf[i] = x[i];
        tock(PROF_STAGE, t0);
        return true;
    }

    template <int K>
    __device__ __forceinline__ void stream(int l, int it) {
        sync();                                                          // the previous step is complete
        const long long top0 = tick();
        Epilogue ep;
        ep.kind = K; ep.limit = 0; ep.first = 0; ep.a = nullptr; ep.b = nullptr; ep.c = nullptr;
        if (K == OP_RELAX) {
            // one l1-Jacobi sweep on the real points (§4.1): delta from the OLD u
            // (the staged copy), then u += delta, t += delta (P:507-508 / P:517-518)
            const StreamDesc d = lev[l].A;
            const int n_real = lev[l].n_real;
            double *u = U(l), *t = T(l);
            const bool staged = stage_x(u, lev[l].n_bar);
            sync();
            ep.c = F(l);
            if (staged) {
                ep.a = u; ep.b = t;
                run_chunks(d, d.nchunks_real, d.nslices_real, true, u, ep);
            } else {                                                     // gather from global: two passes
                double* delta = w;
                ep.kind = OP_RELAX_DELTA; ep.a = delta;
                run_chunks(d, d.nchunks_real, d.nslices_real, false, u, ep);
                sync();
                for (int i = ctid; i < n_real; i += nct) {
                    const double dl = delta[i];
                    u[i] += dl;
                    t[i] += dl;
                }
            }
        } else if (K == OP_AT) {
            // P:509  w = s_l + A_l t_l on all of D-bar_l (ghost rows: real columns only)
            const StreamDesc d = lev[l].A;
            const double* t = T(l);
            const bool staged = stage_x(t, lev[l].n_bar);
            sync();
            ep.a = w; ep.c = S(l);
            run_chunks(d, d.nchunks, INT_MAX, staged, t, ep);
        } else if (K == OP_RESTRICT) {
            // P:509  s_{l+1} = R_l w ; P:512 reset t_l, s_l ; first iteration: P:511 f_{l+1} -= s_{l+1}
            const StreamDesc d = lev[l].R;
            const int n_bar = lev[l].n_bar;
            const bool staged = stage_x(w, n_bar);
            double* t = T(l);
            for (int i = ctid; i < 2 * n_bar; i += nct) t[i] = 0.0;      // t and s are adjacent
            sync();
            ep.a = S(l + 1); ep.b = F(l + 1); ep.limit = lev[l + 1].n_real; ep.first = (it == 0);
            run_chunks(d, d.nchunks, INT_MAX, staged, w, ep);
        } else if (K == OP_RECALC) {
            // P:510-511  f_{l+1} <- f_{l+1} - A_{l+1} u_{l+1} - s_{l+1}  (u_{l+1} of the previous iteration)
            const StreamDesc d = lev[l + 1].A;
            const double* uc = U(l + 1);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            ep.a = F(l + 1); ep.c = S(l + 1);
            run_chunks(d, d.nchunks_real, d.nslices_real, staged, uc, ep);
        } else {
            // P:516  u_l += P_l u_{l+1} on all of D-bar_l (§4.2)
            const StreamDesc d = lev[l].P;
            const double* uc = U(l + 1);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            ep.a = U(l);
            run_chunks(d, d.nchunks, INT_MAX, staged, uc, ep);
        }
        tock(PROF_OP0 + K, top0);
    }
};

__global__ void __launch_bounds__(1024, 1) fac_kernel(const FacParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    Ctrl* ctrl = reinterpret_cast<Ctrl*>(smem);
    double* xbuf = reinterpret_cast<double*>(smem + CTRL_BYTES);
    char* ring = reinterpret_cast<char*>(smem + CTRL_BYTES + (size_t)prm.x_cap * 8);
    const int nwarps = blockDim.x >> 5;
    const int ncw = nwarps - 1;
    const int warp = threadIdx.x >> 5;

    if (threadIdx.x == 0) {
        for (int s = 0; s < prm.stages; ++s) {
            mbar_init(&ctrl->full[s], 1);
            mbar_init(&ctrl->empty[s], (uint32_t)ncw);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int L = prm.L;
    if (warp == 0) {
        if (threadIdx.x == 0) {
            Producer pr;
            pr.ctrl = ctrl; pr.ring = ring; pr.stages = prm.stages; pr.chunk_bytes = prm.chunk_bytes;
            pr.slot = 0; pr.phase = 0; pr.policy = policy_evict_first();
            pr.prof = prm.prof ? prm.prof + (size_t)blockIdx.x * FAC_PROF_SLOTS : nullptr;
            for (;;) {
                const int q = atomicAdd(prm.work_counter, 1);
                const int p = q < prm.num_sub ? prm.order[q] : -1;
                pr.control(p);
                if (p < 0) break;
                pr.lev = prm.lev + (size_t)p * (L + 1);
                fac_program(pr, L, prm.nfac, prm.nu);
            }
        }
        return;
    }

    Consumer cs;
    cs.ctrl = ctrl; cs.ring = ring; cs.xbuf = xbuf; cs.prm = &prm;
    cs.ws = prm.workspace + (size_t)blockIdx.x * prm.slot_stride;
    cs.w = cs.ws + prm.scratch_off;
    cs.stages = prm.stages; cs.chunk_bytes = prm.chunk_bytes; cs.x_cap = prm.x_cap;
    cs.slot = 0; cs.phase = 0;
    cs.ctid = threadIdx.x - 32; cs.nct = blockDim.x - 32; cs.cw = warp - 1; cs.ncw = ncw;
    cs.prof = prm.prof ? prm.prof + (size_t)blockIdx.x * FAC_PROF_SLOTS : nullptr;
    const long long tk0 = cs.tick();
    for (;;) {
        const int p = cs.next_subdomain();
        if (p < 0) break;
        cs.p = p;
        cs.lev = prm.lev + (size_t)p * (L + 1);
        fac_program(cs, L, prm.nfac, prm.nu);
    }
    cs.tock(PROF_TOTAL, tk0);
}

}  // namespace

int fac_smem_bytes(int chunk_bytes, int stages, int x_cap) { return CTRL_BYTES + x_cap * 8 + stages * chunk_bytes; }

int fac_max_stages() { return MAX_STAGES; }

int fac_configure(int /*device*/, int max_smem_optin) {
    cudaError_t e = cudaFuncSetAttribute(fac_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin);
    return e == cudaSuccess ? 0 : (int)e;
}

void launch_fac(const FacParams& prm, const FacLaunch& cfg, void* stream) {
    fac_kernel<<<cfg.grid, cfg.block, cfg.smem_bytes, (cudaStream_t)stream>>>(prm);
}

}  // namespace amgdd
