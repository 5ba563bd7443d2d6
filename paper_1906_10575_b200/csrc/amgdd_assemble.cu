// Kernels of the device-side composite-grid assembly (amgdd_assemble.cuh).  One CTA per stream of a
// (subdomain, level) block.  Pass 1 (plan): local row lengths, the stable sort by length inside the
// windows, the slices and their greedy dealing to the ways -- the same rules as the host packer, so
// both produce the same bytes.  Pass 2 (write): one warp per slice walks the global rows of its 32
// lanes, renumbers the columns by binary search in the sorted index lists of the block and stores
// headers and groups with coalesced 16-byte stores.
#include "amgdd_assemble.cuh"

#include <climits>

namespace amgdd {

namespace {

constexpr int ASM_THREADS = 256;

__device__ __forceinline__ int find_sorted(const int* __restrict__ a, int n, int g) {
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(a + mid) < g) lo = mid + 1; else hi = mid;
    }
    return (lo < n && __ldg(a + lo) == g) ? lo : -1;
}

// local index of global point g in a level given by its lists (real ascending, then ghost ascending; S7)
__device__ __forceinline__ int local_of(const int* __restrict__ gid, int nr, int ng, int g) {
    if (gid == nullptr) return g;                                    // fully covered level: identity
    const int r = find_sorted(gid, nr, g);
    if (r >= 0) return r;
    const int q = find_sorted(gid + nr, ng, g);
    return q >= 0 ? nr + q : -1;
}

// Enumerates the kept entries of local row i of a job in stored order:
//   A, real row:  the whole global row (eq. 1: all of it lies in D-bar_l)
//   A, ghost row: the entries whose column is a real point (A12)
//   P:            the entries whose column lies in D-bar_{l+1} (the others are counted: A7)
//   R:            the entries whose column (a point of level l) lies in D-bar_l, real columns first, then ghost
//                 columns (= ascending local index: the order of the host's counting-sort transpose)
struct RowCursor {
    const int* ci; const double* v;
    long long beg, cur, end;
    int pass;
};

__device__ __forceinline__ void row_open(const AsmJob& J, const DevHierLevel& H, int i, RowCursor& c) {
    const DevCsr64& M = J.kind == ASM_A ? H.A : (J.kind == ASM_P ? H.P : H.R);
    const int g = J.kind == ASM_R ? (J.gidc ? __ldg(J.gidc + i) : i) : __ldg(J.gid + i);
    c.ci = M.ci; c.v = M.v;
    c.beg = c.cur = M.rp[g];
    c.end = M.rp[g + 1];
    c.pass = 0;
}

// next kept entry: returns false when the row is exhausted; *bad is raised for an impossible column
__device__ __forceinline__ bool row_next(const AsmJob& J, int i, RowCursor& c, int& col, double& val, int& bad) {
    for (;;) {
        if (c.cur >= c.end) {
            if (J.kind == ASM_R && c.pass == 0) { c.pass = 1; c.cur = c.beg; continue; }
            return false;
        }
        const long long k = c.cur++;
        const int g = __ldg(c.ci + k);
        int loc;
        if (J.kind == ASM_A) {
            if (i < J.nr) { loc = local_of(J.gid, J.nr, J.ng, g); if (loc < 0) bad = 1; }
            else { loc = find_sorted(J.gid, J.nr, g); if (loc < 0) continue; }
        } else if (J.kind == ASM_P) {
            loc = local_of(J.gidc, J.nrc, J.ngc, g);
            if (loc < 0) continue;
        } else {
            if (c.pass == 0) { loc = find_sorted(J.gid, J.nr, g); if (loc < 0) continue; }
            else { loc = find_sorted(J.gid + J.nr, J.ng, g); if (loc < 0) continue; loc += J.nr; }
        }
        col = loc; val = c.v[k];
        return true;
    }
}

__device__ __forceinline__ int row_length(const AsmJob& J, const DevHierLevel& H, int i, int& dropped) {
    const DevCsr64& M = J.kind == ASM_A ? H.A : (J.kind == ASM_P ? H.P : H.R);
    const int g = J.kind == ASM_R ? (J.gidc ? __ldg(J.gidc + i) : i) : __ldg(J.gid + i);
    const long long b = M.rp[g], e = M.rp[g + 1];
    if (J.kind == ASM_A && i < J.nr) return (int)(e - b);
    int n = 0;
    for (long long k = b; k < e; ++k) {
        const int c = __ldg(M.ci + k);
        if (J.kind == ASM_A) n += find_sorted(J.gid, J.nr, c) >= 0;
        else if (J.kind == ASM_P) { const bool in = local_of(J.gidc, J.nrc, J.ngc, c) >= 0; n += in; dropped += !in; }
        else n += local_of(J.gid, J.nr, J.ng, c) >= 0;
    }
    return n;
}

// first sorted position of slice s and the rows it holds
__device__ __forceinline__ void slice_span(const AsmJob& J, int s, int& pos, int& cnt) {
    const int n0 = J.nrows_first, s0 = (n0 + SLICE_ROWS - 1) / SLICE_ROWS;
    if (s < s0) { pos = s * SLICE_ROWS; cnt = min(SLICE_ROWS, n0 - pos); }
    else { pos = n0 + (s - s0) * SLICE_ROWS; cnt = min(SLICE_ROWS, J.nrows - pos); }
}

__global__ void __launch_bounds__(ASM_THREADS) asm_plan_kernel(const AsmJob* __restrict__ jobs, const DevHierLevel* __restrict__ hier,
                                                                 int* __restrict__ row_scratch, AsmSlice* __restrict__ slice_scratch,
                                                                 AsmPlan* __restrict__ plans) {
    const AsmJob J = jobs[blockIdx.x];
    const DevHierLevel H = hier[J.level];
    int* len = row_scratch + J.scratch_row;
    int* order = len + J.nrows;
    AsmSlice* sl = slice_scratch + J.scratch_slice;
    __shared__ unsigned long long s_nnz;
    __shared__ int s_dropped, s_toolong;
    __shared__ int tile[ASM_MAX_WINDOW];
    const int tid = threadIdx.x;
    if (tid == 0) { s_nnz = 0; s_dropped = 0; s_toolong = INT_MAX; }
    __syncthreads();
    // 1. local row lengths
    {
        unsigned long long nnz = 0;
        int dropped = 0, toolong = INT_MAX;
        for (int i = tid; i < J.nrows; i += ASM_THREADS) {
            const int n = row_length(J, H, i, dropped);
            len[i] = n;
            nnz += (unsigned long long)n;
            if (n > 65535 && i < toolong) toolong = i;
        }
        if (nnz) atomicAdd(&s_nnz, nnz);
        if (dropped) atomicAdd(&s_dropped, dropped);
        if (toolong != INT_MAX) atomicMin(&s_toolong, toolong);
    }
    __syncthreads();
    // 2. inside every window of a row group: stable sort by descending length (rank by counting)
    const int gb[3] = {0, J.nrows_first, J.nrows};
    for (int g = 0; g < 2; ++g)
        for (int w0 = gb[g]; w0 < gb[g + 1]; w0 += J.window) {
            const int m = min(J.window, gb[g + 1] - w0);
            for (int k = tid; k < m; k += ASM_THREADS) tile[k] = len[w0 + k];
            __syncthreads();
            for (int k = tid; k < m; k += ASM_THREADS) {
                const int mine = tile[k];
                int rank = 0;
                for (int j = 0; j < m; ++j) { const int o = tile[j]; rank += (o > mine) || (o == mine && j < k); }
                order[w0 + rank] = w0 + k;
            }
            __syncthreads();
        }
    // 3. groups of every slice: its first lane holds the longest row
    const int n0 = J.nrows_first, n1 = J.nrows - n0;
    const int S0 = (n0 + SLICE_ROWS - 1) / SLICE_ROWS, S = S0 + (n1 + SLICE_ROWS - 1) / SLICE_ROWS;
    for (int s = tid; s < S; s += ASM_THREADS) {
        int pos, cnt;
        slice_span(J, s, pos, cnt);
        const int longest = len[order[pos]];
        sl[s].K = (uint32_t)max(1, (longest + GROUP_STEPS - 1) / GROUP_STEPS);
    }
    __syncthreads();
    // 4. deal the slices to the ways in slice order, each to the way with the fewest bytes so far (ties: lowest way)
    if (tid < 32) {
        const int lane = tid;
        const long long gbytes = J.wide ? GROUP_BYTES_WIDE : GROUP_BYTES_NARROW;
        const long long hbytes = J.wide ? HEADER_BYTES_WIDE : HEADER_BYTES_NARROW;
        long long load = 0;
        uint32_t ngr = 0, nsl = 0, ngr_first = 0, nsl_first = 0;
        for (int s = 0; s < S; ++s) {
            const uint32_t K = sl[s].K;
            long long key = lane < NUM_WAYS ? load : LLONG_MAX;
            int best = lane;
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) {
                const long long ok = __shfl_xor_sync(0xffffffffu, key, off);
                const int ob = __shfl_xor_sync(0xffffffffu, best, off);
                if (ok < key || (ok == key && ob < best)) { key = ok; best = ob; }
            }
            if (lane == best) {
                sl[s].way = (uint32_t)lane; sl[s].g_off = ngr; sl[s].h_idx = nsl;
                load += (long long)K * gbytes + hbytes;
                ngr += K; nsl += 1;
                if (s < S0) { ngr_first += K; nsl_first += 1; }
            }
        }
        // offsets: all groups way by way, then all headers way by way (128-byte units; both sizes are multiples of 128)
        const unsigned long long gb128 = (unsigned long long)ngr * (unsigned long long)(gbytes / 128);
        const unsigned long long hb128 = ((unsigned long long)nsl * (unsigned long long)hbytes + 127ull) / 128ull;      // a way's headers end 128-byte aligned
        unsigned long long gpre = gb128, hpre = hb128;                // inclusive scans over the lanes
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const unsigned long long a = __shfl_up_sync(0xffffffffu, gpre, off);
            const unsigned long long b = __shfl_up_sync(0xffffffffu, hpre, off);
            if (lane >= off) { gpre += a; hpre += b; }
        }
        const unsigned long long gtot = __shfl_sync(0xffffffffu, gpre, 31);
        const unsigned long long htot = __shfl_sync(0xffffffffu, hpre, 31);
        unsigned long long tg = ngr, ts = nsl, tgf = ngr_first, tsf = nsl_first;
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            tg += __shfl_xor_sync(0xffffffffu, tg, off); ts += __shfl_xor_sync(0xffffffffu, ts, off);
            tgf += __shfl_xor_sync(0xffffffffu, tgf, off); tsf += __shfl_xor_sync(0xffffffffu, tsf, off);
        }
        AsmPlan& pl = plans[blockIdx.x];
        if (lane < NUM_WAYS) {
            WayDesc d;
            d.grp_off128 = (uint32_t)(gpre - gb128);
            d.hdr_off128 = (uint32_t)(gtot + hpre - hb128);
            d.ngroups = ngr; d.ngroups_real = ngr_first; d.nslices = nsl; d.nslices_real = nsl_first;
            d.pad_[0] = d.pad_[1] = 0;
            pl.way[lane] = d;
        }
        if (lane == 0) {
            pl.bytes = (long long)((gtot + htot) * 128ull);
            pl.bytes_real = (long long)tgf * gbytes + (long long)tsf * hbytes;
            pl.padded_nnz = (long long)tg * GROUP_STEPS * SLICE_ROWS;
            pl.nnz = (long long)s_nnz;
            pl.dropped = s_dropped;
            pl.too_long_row = s_toolong == INT_MAX ? -1 : s_toolong;
            pl.bad_col = 0; pl.pad_ = 0;
        }
    }
}

__global__ void __launch_bounds__(ASM_THREADS) asm_write_kernel(const AsmJob* __restrict__ jobs, const DevHierLevel* __restrict__ hier,
                                                                  const int* __restrict__ row_scratch, const AsmSlice* __restrict__ slice_scratch,
                                                                  AsmPlan* __restrict__ plans) {
    const AsmJob J = jobs[blockIdx.x];
    const DevHierLevel H = hier[J.level];
    const int* len = row_scratch + J.scratch_row;
    const int* order = len + J.nrows;
    const AsmSlice* sl = slice_scratch + J.scratch_slice;
    const AsmPlan& pl = plans[blockIdx.x];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = ASM_THREADS / 32;
    const int n0 = J.nrows_first, n1 = J.nrows - n0;
    const int S = (n0 + SLICE_ROWS - 1) / SLICE_ROWS + (n1 + SLICE_ROWS - 1) / SLICE_ROWS;
    const int gbytes = J.wide ? GROUP_BYTES_WIDE : GROUP_BYTES_NARROW;
    // aux / flag of a row: A_l rows are points of level l, R_l rows points of level l+1; ghosts never relax (A4)
    const DevHierLevel Hr = J.kind == ASM_R ? hier[J.level + 1] : H;
    const int* rgid = J.kind == ASM_R ? J.gidc : J.gid;
    const int rreal = J.kind == ASM_R ? J.nrc : J.nr;
    int bad = 0;
    for (int s = warp; s < S; s += nwarps) {
        const AsmSlice rec = sl[s];
        int pos, cnt;
        slice_span(J, s, pos, cnt);
        const int row = lane < cnt ? order[pos + lane] : -1;
        char* h = J.dst + 128ll * pl.way[rec.way].hdr_off128 + (long long)rec.h_idx * (J.wide ? HEADER_BYTES_WIDE : HEADER_BYTES_NARROW);
        char* g = J.dst + 128ll * pl.way[rec.way].grp_off128 + (long long)rec.g_off * gbytes;
        {   // header: narrow row | K << 16 | flag << 31; wide { row, K | flag << 31 }
            uint32_t flag = 0;
            if (J.kind != ASM_P && row >= 0 && row < rreal) {
                const int gp = rgid ? __ldg(rgid + row) : row;
                if (Hr.cf != nullptr && Hr.cf[gp] > 0) flag = 0x80000000u;
            }
            if (J.wide) *reinterpret_cast<uint2*>(h + 8 * lane) = make_uint2(row >= 0 ? (uint32_t)row : NO_ROW, rec.K | flag);
            else *reinterpret_cast<uint32_t*>(h + 4 * lane) = (row >= 0 ? (uint32_t)row : (uint32_t)NO_ROW16) | (rec.K << 16) | flag;
        }
        RowCursor c;
        int mylen = 0;
        if (row >= 0) { mylen = len[row]; row_open(J, H, row, c); }
        int done = 0;
        for (uint32_t kg = 0; kg < rec.K; ++kg, g += gbytes) {
            double v[GROUP_STEPS];
            uint32_t col[GROUP_STEPS];
#pragma unroll
            for (int q = 0; q < GROUP_STEPS; ++q) {
                v[q] = 0.0; col[q] = 0;
                if (done < mylen) {
                    int cc = 0; double vv = 0.0;
                    if (row_next(J, row, c, cc, vv, bad)) { v[q] = vv; col[q] = (uint32_t)cc; }
                    ++done;
                }
            }
            *reinterpret_cast<double2*>(g + 16 * lane) = make_double2(v[0], v[1]);
            *reinterpret_cast<double2*>(g + 512 + 16 * lane) = make_double2(v[2], v[3]);
            if (J.wide) *reinterpret_cast<uint4*>(g + 1024 + 16 * lane) = make_uint4(col[0], col[1], col[2], col[3]);
            else *reinterpret_cast<uint2*>(g + 1024 + 8 * lane) = make_uint2((col[0] & 0xFFFFu) | (col[1] << 16), (col[2] & 0xFFFFu) | (col[3] << 16));
        }
    }
    if (bad) atomicOr(&plans[blockIdx.x].bad_col, 1);
}

__global__ void __launch_bounds__(ASM_THREADS) asm_copy_kernel(const AsmCopy* __restrict__ jobs) {
    const AsmCopy c = jobs[blockIdx.x];
    if (c.gather) {
        double* d = reinterpret_cast<double*>(c.dst);
        for (int i = threadIdx.x; i < c.n; i += ASM_THREADS) d[i] = i < c.n_gather ? c.dinv[c.src[i]] : 0.0;
    } else {
        for (int i = threadIdx.x; i < c.n; i += ASM_THREADS) c.dst[i] = c.src[i];
    }
}


// ---- composite index sets (amgdd_assemble.cuh) ----------------------------------------------------------------------------
constexpr int SET_THREADS = 256;

// one layer of breadth-first growth: every point of `cur` marks its unmarked neighbours in `mark` (those not in `skip`)
// and appends them to `next`; returns false when `next` overflowed
__device__ bool grow_layer(const DevCsr64& A, const int* cur, int ncur, unsigned* mark, const unsigned* skip, int* next, int cap, int* s_count,
                           int* s_lo, int* s_hi, int* s_over) {
    for (int q = threadIdx.x; q < ncur; q += SET_THREADS) {
        const int i = cur[q];
        for (long long k = A.rp[i]; k < A.rp[i + 1]; ++k) {
            const int j = __ldg(A.ci + k);
            const unsigned bit = 1u << (j & 31);
            if (skip && (skip[j >> 5] & bit)) continue;
            const unsigned old = atomicOr(mark + (j >> 5), bit);
            if (!(old & bit)) {
                const int pos = atomicAdd(s_count, 1);
                if (pos < cap) next[pos] = j; else *s_over = 1;
                atomicMin(s_lo, j >> 5);
                atomicMax(s_hi, j >> 5);
            }
        }
    }
    __syncthreads();
    return *s_over == 0;
}

__global__ void __launch_bounds__(SET_THREADS) asm_sets_grow_kernel(SetJob* __restrict__ jobs, const DevHierLevel* __restrict__ hier,
                                                                      const long long* __restrict__ bm_off, int L, int eta, int num_ghost) {
    SetJob& J = jobs[blockIdx.x];
    __shared__ int s_count, s_lo, s_hi, s_over, s_nseed;
    int* bufA = J.frontier;
    const int cap = J.frontier_cap;                  // min(SET_FRONTIER_CAP, n_0): no frontier holds more points than the largest level has
    int* bufB = J.frontier + cap;
    int* seeds = J.frontier + 2 * cap;
    if (threadIdx.x == 0) { s_over = 0; s_nseed = J.n_owned <= cap ? J.n_owned : 0; if (J.n_owned > cap) s_over = 1; }
    __syncthreads();
    for (int q = threadIdx.x; q < s_nseed; q += SET_THREADS) seeds[q] = J.owned[q];       // B_0^p = Omega_0^p
    __syncthreads();
    for (int l = 0; l <= L && s_over == 0; ++l) {
        const DevHierLevel H = hier[l];
        SetLevelOut& o = J.out[l];
        if (l == L) {                                                    // reading A5: D_L^p = Omega_L, no ghosts
            if (threadIdx.x == 0) { o.n_real = (int)H.n; o.n_ghost = 0; o.lo_word = 0; o.hi_word = -1; }
            break;
        }
        unsigned* real = J.bm_real + bm_off[l];
        unsigned* ghost = J.bm_ghost + bm_off[l];
        const int nseed = s_nseed;
        if (threadIdx.x == 0) { s_count = 0; s_lo = INT_MAX; s_hi = -1; }
        __syncthreads();
        for (int q = threadIdx.x; q < nseed; q += SET_THREADS) {         // the seeds are distinct
            const int i = seeds[q];
            atomicOr(real + (i >> 5), 1u << (i & 31));
            bufA[q] = i;
            atomicMin(&s_lo, i >> 5);
            atomicMax(&s_hi, i >> 5);
        }
        __syncthreads();
        int n_real = nseed, ncur = nseed;
        int* cur = bufA;
        int* nxt = bufB;
        for (int d = 0; d < eta && ncur > 0; ++d) {                       // D_l^p: within eta of B_l^p
            if (!grow_layer(H.A, cur, ncur, real, nullptr, nxt, cap, &s_count, &s_lo, &s_hi, &s_over)) break;
            ncur = s_count;
            n_real += ncur;
            __syncthreads();
            if (threadIdx.x == 0) s_count = 0;
            __syncthreads();
            int* t = cur; cur = nxt; nxt = t;
        }
        if (s_over) break;
        // ghost layers: only the points of the last real layer can have neighbours outside D_l^p
        int n_ghost = 0;
        for (int d = 0; d < num_ghost && ncur > 0; ++d) {
            if (!grow_layer(H.A, cur, ncur, ghost, real, nxt, cap, &s_count, &s_lo, &s_hi, &s_over)) break;
            ncur = s_count;
            n_ghost += ncur;
            __syncthreads();
            if (threadIdx.x == 0) s_count = 0;
            __syncthreads();
            int* t = cur; cur = nxt; nxt = t;
        }
        if (s_over) break;
        if (threadIdx.x == 0) { o.n_real = n_real; o.n_ghost = n_ghost; o.lo_word = s_lo == INT_MAX ? 0 : s_lo; o.hi_word = s_hi; s_nseed = 0; }
        __syncthreads();
        // B_{l+1}^p: coarse images of the C-points of D_l^p (order does not matter)
        const int lo = s_lo == INT_MAX ? 0 : s_lo, hi = s_hi;
        for (int w = lo + threadIdx.x; w <= hi; w += SET_THREADS) {
            unsigned bits = real[w];
            while (bits) {
                const int b = __ffs(bits) - 1;
                bits &= bits - 1;
                const int i = 32 * w + b;
                if (H.cf[i] > 0) {
                    const int pos = atomicAdd(&s_nseed, 1);
                    if (pos < cap) seeds[pos] = H.coarse_of[i]; else s_over = 1;
                }
            }
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) J.overflow = s_over;
}

// ascending extraction of a bitmap range into dst (returns the count); clears the words; all threads of the CTA
__device__ int extract_sorted(unsigned* bm, int lo, int hi, int* dst, int* s_scan, const DevHierLevel& H, bool is_real,
                              unsigned long long* s_sumA, unsigned long long* s_sumP) {
    int base = 0;
    unsigned long long sumA = 0, sumP = 0;
    for (int w0 = lo; w0 <= hi; w0 += SET_THREADS) {
        const int w = w0 + threadIdx.x;
        unsigned bits = w <= hi ? bm[w] : 0u;
        if (w <= hi && bits) bm[w] = 0u;
        const int cnt = __popc(bits);
        // block exclusive scan of cnt
        s_scan[threadIdx.x] = cnt;
        __syncthreads();
        for (int off = 1; off < SET_THREADS; off <<= 1) {
            const int v = threadIdx.x >= off ? s_scan[threadIdx.x - off] : 0;
            __syncthreads();
            s_scan[threadIdx.x] += v;
            __syncthreads();
        }
        int pos = base + s_scan[threadIdx.x] - cnt;
        const int total = s_scan[SET_THREADS - 1];
        while (bits) {
            const int b = __ffs(bits) - 1;
            bits &= bits - 1;
            const int i = 32 * w + b;
            if (dst) dst[pos] = i;
            ++pos;
            sumA += (unsigned long long)(H.A.rp[i + 1] - H.A.rp[i]);
            if (H.P.rp) sumP += (unsigned long long)(H.P.rp[i + 1] - H.P.rp[i]);
        }
        base += total;
        __syncthreads();
    }
    if (sumA) atomicAdd(s_sumA, sumA);
    if (sumP) atomicAdd(s_sumP, sumP);
    (void)is_real;
    return base;
}

__global__ void __launch_bounds__(SET_THREADS) asm_sets_extract_kernel(SetJob* __restrict__ jobs, const DevHierLevel* __restrict__ hier,
                                                                         const long long* __restrict__ bm_off, int L) {
    SetJob& J = jobs[blockIdx.x];
    __shared__ int s_scan[SET_THREADS];
    __shared__ unsigned long long s_sumA, s_sumP, s_sumAg;
    for (int l = 0; l <= L; ++l) {
        const DevHierLevel H = hier[l];
        SetLevelOut& o = J.out[l];
        if (threadIdx.x == 0) { s_sumA = 0; s_sumP = 0; s_sumAg = 0; }
        __syncthreads();
        if (l == L || o.n_real == (int)H.n) {
            // the whole level (shared copy): nothing to extract; the sums over the whole level; bitmaps still to be cleared
            if (l < L) {
                unsigned* real = J.bm_real + bm_off[l];
                unsigned* ghost = J.bm_ghost + bm_off[l];
                for (int w = o.lo_word + threadIdx.x; w <= o.hi_word; w += SET_THREADS) { real[w] = 0u; ghost[w] = 0u; }
            }
            if (threadIdx.x == 0) {
                o.nnzA_real = H.A.rp[H.n]; o.nnzA_ghost_bound = 0; o.nnzP_bound = H.P.rp ? H.P.rp[H.n] : 0;
            }
            __syncthreads();
            continue;
        }
        int* dst = J.list_dst[l];
        unsigned* real = J.bm_real + bm_off[l];
        unsigned* ghost = J.bm_ghost + bm_off[l];
        const int nr = extract_sorted(real, o.lo_word, o.hi_word, dst, s_scan, H, true, &s_sumA, &s_sumP);
        __syncthreads();
        extract_sorted(ghost, o.lo_word, o.hi_word, dst ? dst + nr : nullptr, s_scan, H, false, &s_sumAg, &s_sumP);
        __syncthreads();
        if (threadIdx.x == 0) { o.nnzA_real = (long long)s_sumA; o.nnzA_ghost_bound = (long long)s_sumAg; o.nnzP_bound = (long long)s_sumP; }
        __syncthreads();
    }
    // local indices (level 0) of the owned dofs: position in the ascending real list (identity on a fully covered level)
    const SetLevelOut& o0 = J.out[0];
    const bool shared0 = (L == 0) || o0.n_real == (int)hier[0].n;
    const int* real0 = shared0 ? nullptr : J.list_dst[0];
    for (int k = threadIdx.x; k < J.n_owned; k += SET_THREADS) {
        const int g = J.owned[k];
        int loc = g;
        if (!shared0) {                                                // (plain loads: the list was written by this kernel)
            int lo = 0, hi = o0.n_real;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (real0[mid] < g) lo = mid + 1; else hi = mid; }
            loc = lo;
        }
        J.owned_local_dst[k] = loc;
    }
}

}  // namespace

cudaError_t launch_asm_plan(const AsmJob* jobs, int njobs, const DevHierLevel* hier, int* row_scratch, AsmSlice* slice_scratch,
                            AsmPlan* plans, cudaStream_t st) {
    if (njobs > 0) asm_plan_kernel<<<njobs, ASM_THREADS, 0, st>>>(jobs, hier, row_scratch, slice_scratch, plans);
    return cudaGetLastError();
}

cudaError_t launch_asm_write(const AsmJob* jobs, int njobs, const DevHierLevel* hier, const int* row_scratch,
                             const AsmSlice* slice_scratch, AsmPlan* plans, cudaStream_t st) {
    if (njobs > 0) asm_write_kernel<<<njobs, ASM_THREADS, 0, st>>>(jobs, hier, row_scratch, slice_scratch, plans);
    return cudaGetLastError();
}

cudaError_t launch_sets_grow(SetJob* jobs, int njobs, const DevHierLevel* hier, const long long* bm_off, int L, int eta, int num_ghost,
                             cudaStream_t st) {
    if (njobs > 0) asm_sets_grow_kernel<<<njobs, SET_THREADS, 0, st>>>(jobs, hier, bm_off, L, eta, num_ghost);
    return cudaGetLastError();
}

cudaError_t launch_sets_extract(SetJob* jobs, int njobs, const DevHierLevel* hier, const long long* bm_off, int L, cudaStream_t st) {
    if (njobs > 0) asm_sets_extract_kernel<<<njobs, SET_THREADS, 0, st>>>(jobs, hier, bm_off, L);
    return cudaGetLastError();
}

cudaError_t launch_asm_copy(const AsmCopy* jobs, int njobs, cudaStream_t st) {
    if (njobs > 0) asm_copy_kernel<<<njobs, ASM_THREADS, 0, st>>>(jobs);
    return cudaGetLastError();
}

}  // namespace amgdd
