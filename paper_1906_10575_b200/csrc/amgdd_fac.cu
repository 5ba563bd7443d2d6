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

    __device__ __forceinline__ void acquire() { mbar_wait(&ctrl->empty[slot], phase ^ 1u); }
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
// One chunk in shared memory.  Rows are dealt to the consumer warps in batches of G = 32/lanes
// consecutive rows, round-robin by GLOBAL batch index (so the deal stays balanced across chunk
// boundaries); `bnext` is the warp's next batch and is carried from chunk to chunk, which keeps
// the per-chunk bookkeeping free of integer division.  `lanes` threads stride over a row, the row
// sum is reduced by shuffles and epi(row, sum) runs on the first lane of the row.
template <bool WIDE, class X, class Epi>
__device__ __forceinline__ void consume_chunk(const char* slot, X xs, int ll /*log2 lanes*/, int ncw, int& bnext, int row_limit,
                                              Epi epi) {
    const int4 hdr = *reinterpret_cast<const int4*>(slot);
    const int rb = hdr.x, nr = hdr.y, nnz = hdr.z;
    const double* v = reinterpret_cast<const double*>(slot + CHUNK_HEADER_BYTES);
    const char* cbase = slot + CHUNK_HEADER_BYTES + (size_t)nnz * 8;
    const unsigned short* rowend = reinterpret_cast<const unsigned short*>(cbase + (size_t)nnz * (WIDE ? 4 : 2));
    const int lane = threadIdx.x & 31;
    const int lanes = 1 << ll, gl = 5 - ll;
    const int li = lane & (lanes - 1);
    const int sub = lane >> ll;
    const int b_last = (rb + nr - 1) >> gl;
    int b = bnext;
    for (; b <= b_last; b += ncw) {
        const int row = (b << gl) + sub;
        const int lr = row - rb;
        const bool valid = (lr >= 0) && (lr < nr) && (row < row_limit);
        double sum = 0.0;
        if (valid) {
            const int kb = lr > 0 ? (int)rowend[lr - 1] : 0, ke = (int)rowend[lr];
            if (WIDE) {
                const unsigned int* ci = reinterpret_cast<const unsigned int*>(cbase);
                for (int k = kb + li; k < ke; k += lanes) sum += v[k] * xs[ci[k]];
            } else {
                const unsigned short* ci = reinterpret_cast<const unsigned short*>(cbase);
                for (int k = kb + li; k < ke; k += lanes) sum += v[k] * xs[ci[k]];
            }
        }
        for (int o = lanes >> 1; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o, lanes);
        if (valid && li == 0) epi(row, sum);
    }
    // a batch cut by the end of the chunk continues in the next chunk
    if (b - ncw == b_last && ((rb + nr) & ((1 << gl) - 1)) != 0) b -= ncw;
    bnext = b;
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

    __device__ __forceinline__ double* U(int l) const { return ws + lev[l].voff; }
    __device__ __forceinline__ double* T(int l) const { return ws + lev[l].voff + lev[l].n_bar; }
    __device__ __forceinline__ double* S(int l) const { return ws + lev[l].voff + 2 * (size_t)lev[l].n_bar; }
    __device__ __forceinline__ double* F(int l) const { return ws + lev[l].voff + 3 * (size_t)lev[l].n_bar; }
    __device__ __forceinline__ void sync() { bar_consumers(nct); }
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
        sync();                                                          // previous subdomain fully done
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
    }
    // ---- Alg. 2: x <- x + u_0^p on Omega_0^p (disjoint targets across subdomains) ----
    __device__ __forceinline__ void end_subdomain() {
        sync();
        const DevSub sb = prm->sub[p];
        const double* u0 = U(0);
        const int* gid0 = lev[0].gid;
        for (int k = ctid; k < sb.n_owned; k += nct) {
            const int li = __ldg(sb.owned + k);
            prm->x[__ldg(gid0 + li)] += u0[li];
        }
    }
    // P:506 u_l <- 0, then the first sweep needs no matrix: delta = D^{-1} f
    __device__ __forceinline__ void first_sweep(int l) {
        sync();
        const int n_real = lev[l].n_real, n_bar = lev[l].n_bar;
        const double* dinv = lev[l].dinv;
        double *u = U(l), *t = T(l);
        const double* f = F(l);
        for (int i = ctid; i < n_bar; i += nct) {
            double dl = 0.0;
            if (i < n_real) { dl = __ldg(dinv + i) * f[i]; t[i] += dl; }
            u[i] = dl;
        }
    }
    // u_L = A_L^{-1} f_L with the LU factors computed at setup (Alg. 4).  One warp; columns
    // of the unit-lower / upper factors are contiguous (column-major).
    __device__ __forceinline__ void coarse() {
        sync();
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
    }

    template <class Epi>
    __device__ __forceinline__ void run_chunks(const StreamDesc& d, int nchunks, bool staged, const double* xg, int row_limit, Epi epi) {
        extern __shared__ __align__(128) unsigned char smem_dyn[];      // same base as in fac_kernel: keeps LDS addressing
        const int ll = __ffs(d.lanes) - 1;
        int bnext = cw;                                                  // batches cw, cw + ncw, ... are this warp's
        for (int c = 0; c < nchunks; ++c) {
            mbar_wait(&ctrl->full[slot], phase);
            const char* sl = reinterpret_cast<const char*>(smem_dyn + CTRL_BYTES + (size_t)x_cap * 8 + (size_t)slot * chunk_bytes);
            if (staged) {
                const double* xs = reinterpret_cast<const double*>(smem_dyn + CTRL_BYTES);
                if (d.wide) consume_chunk<true>(sl, xs, ll, ncw, bnext, row_limit, epi);
                else consume_chunk<false>(sl, xs, ll, ncw, bnext, row_limit, epi);
            } else {
                if (d.wide) consume_chunk<true>(sl, xg, ll, ncw, bnext, row_limit, epi);
                else consume_chunk<false>(sl, xg, ll, ncw, bnext, row_limit, epi);
            }
            release();
        }
    }

    // stage the gather vector of the next mat-vec in shared memory (if it fits)
    __device__ __forceinline__ bool stage_x(const double* x, int n) {
        if (n > x_cap) return false;
        for (int i = ctid; i < n; i += nct) xbuf[i] = x[i];
        return true;
    }

    template <int K>
    __device__ __forceinline__ void stream(int l, int it) {
        sync();                                                          // the previous step is complete
        if (K == OP_RELAX) {
            // one l1-Jacobi sweep on the real points (§4.1): delta from the OLD u
            // (the staged copy), then u += delta, t += delta (P:507-508 / P:517-518)
            const StreamDesc d = lev[l].A;
            const int n_real = lev[l].n_real;
            const double* dinv = lev[l].dinv;
            double *u = U(l), *t = T(l);
            const double* f = F(l);
            const bool staged = stage_x(u, lev[l].n_bar);
            sync();
            if (staged) {
                run_chunks(d, d.nchunks_real, true, u, n_real, [=](int i, double au) {
                    const double dl = __ldg(dinv + i) * (f[i] - au);
                    u[i] += dl;
                    t[i] += dl;
                });
            } else {                                                     // gather from global: two passes
                double* delta = w;
                run_chunks(d, d.nchunks_real, false, u, n_real, [=](int i, double au) { delta[i] = __ldg(dinv + i) * (f[i] - au); });
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
            const int n_bar = lev[l].n_bar;
            const double *t = T(l), *s = S(l);
            double* wv = w;
            const bool staged = stage_x(t, n_bar);
            sync();
            run_chunks(d, d.nchunks, staged, t, n_bar, [=](int i, double at) { wv[i] = s[i] + at; });
        } else if (K == OP_RESTRICT) {
            // P:509  s_{l+1} = R_l w ; P:512 reset t_l, s_l ; first iteration: P:511 f_{l+1} -= s_{l+1}
            const StreamDesc d = lev[l].R;
            const int n_bar = lev[l].n_bar, nc_bar = lev[l + 1].n_bar, nc_real = lev[l + 1].n_real;
            double *sc = S(l + 1), *fc = F(l + 1);
            const bool first = (it == 0);
            const bool staged = stage_x(w, n_bar);
            double* t = T(l);
            for (int i = ctid; i < 2 * n_bar; i += nct) t[i] = 0.0;      // t and s are adjacent
            sync();
            run_chunks(d, d.nchunks, staged, w, nc_bar, [=](int I, double rw) {
                sc[I] = rw;
                if (first && I < nc_real) fc[I] -= rw;
            });
        } else if (K == OP_RECALC) {
            // P:510-511  f_{l+1} <- f_{l+1} - A_{l+1} u_{l+1} - s_{l+1}  (u_{l+1} of the previous iteration)
            const StreamDesc d = lev[l + 1].A;
            const int nc_real = lev[l + 1].n_real;
            const double *uc = U(l + 1), *sc = S(l + 1);
            double* fc = F(l + 1);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            run_chunks(d, d.nchunks_real, staged, uc, nc_real, [=](int I, double au) { fc[I] = (fc[I] - au) - sc[I]; });
        } else {
            // P:516  u_l += P_l u_{l+1} on all of D-bar_l (§4.2)
            const StreamDesc d = lev[l].P;
            const int n_bar = lev[l].n_bar;
            const double* uc = U(l + 1);
            double* u = U(l);
            const bool staged = stage_x(uc, lev[l + 1].n_bar);
            sync();
            run_chunks(d, d.nchunks, staged, uc, n_bar, [=](int i, double pu) { u[i] += pu; });
        }
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
    for (;;) {
        const int p = cs.next_subdomain();
        if (p < 0) break;
        cs.p = p;
        cs.lev = prm.lev + (size_t)p * (L + 1);
        fac_program(cs, L, prm.nfac, prm.nu);
    }
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
