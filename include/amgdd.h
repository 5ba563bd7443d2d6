/* amgdd.h -- C ABI of the B200-native AMG-DD local-solve hot path.
 *
 * Method: Mitchell, Strzodka, Falgout, "Parallel Performance of Algebraic Multigrid Domain
 * Decomposition (AMG-DD)", arXiv 1906.10575.  "P:NNN" = line NNN of the paper text;
 * "S1..S8" / "A1..A20" = the readings fixed in DESIGN.md.
 *
 * What the library computes: the paper's P "processors" become P virtual subdomains on ONE GPU.
 *   setup  : AMG hierarchy A_l, P_l, R_l = P_l^T, A_{l+1} = R_l A_l P_l by classical
 *            Ruge-Stueben coarsening with threshold theta, direct interpolation and Galerkin
 *            products (S1-S5); per-subdomain composite grids D_l^p, D-bar_l^p grown by eta through
 *            the graph of A_l with one (or more) ghost layers (eq. 1; S6-S7); local CSR
 *            blocks uploaded to the device.  Runs once on the host.
 *   solve  : num_cycles AMG-DD cycles (Alg. 2): global residual r_0 = b - A_0 x,
 *            restriction r_{l+1} = P_l^T r_l to all levels, gather onto the composite grids, then
 *            num_fac_cycles AlgFAC V(nu,nu)-cycles per subdomain (Alg. 4) with
 *            l1-Jacobi relaxation and a dense direct solve on the coarsest level,
 *            and the update x <- x + u_0^p on the owned dofs.  All on the device.
 *
 * Conventions
 *   - All floating point is IEEE binary64; all indices are 0-based.
 *   - "HOST" / "DEVICE" says where a pointer must point.  The library never takes ownership of a
 *     caller's buffer: setup copies what it needs; b and x stay the caller's.
 *   - Every call returns AMGDD_SUCCESS (0) or a negative amgdd_status; nothing is printed and no
 *     exception crosses the boundary.  amgdd_last_error_detail() gives a one-line explanation of
 *     the last failure on the calling thread's handle-less calls (setup) or of the handle.
 *   - One solve at a time per handle.  Device work is enqueued on the handle's stream
 *     (amgdd_set_stream; default: the legacy default stream).
 *   - There is no CPU fallback: without a CUDA device every compute call returns AMGDD_ERR_CUDA.
 */
#ifndef AMGDD_H
#define AMGDD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct amgdd_handle_s* amgdd_handle_t; /* opaque; owned by the library */

typedef enum amgdd_status {
    AMGDD_SUCCESS = 0,
    AMGDD_ERR_BAD_ARG = -1,              /* null pointer, n <= 0, P <= 0, eta < 0, num_ghost < 1, theta not in (0,1],
                                            max_levels < 1, coarse_max < 1, num_fac_cycles < 1, relax_sweeps < 1,
                                            num_cycles < 0, level / subdomain index out of range */
    AMGDD_ERR_BAD_CSR = -2,              /* rowptr[0] != 0 or not monotone, column out of range, columns not strictly
                                            ascending in a row, missing or non-positive diagonal, a non-finite value,
                                            structurally unsymmetric pattern */
    AMGDD_ERR_BAD_OWNER = -3,            /* owner value outside [0,P) or a subdomain that owns no dof */
    AMGDD_ERR_COARSE_TOO_LARGE = -4,     /* coarsening stopped (max_levels or stagnation) with n_L > 4096 */
    AMGDD_ERR_SINGULAR_COARSE = -5,      /* zero pivot in the dense LU of A_L */
    AMGDD_ERR_NOT_CONNECTED_UPWARD = -6, /* a P_l entry of a composite row points outside D-bar_{l+1} (P:111,
                                            P:230: "not necessarily guaranteed"; reading A7): reported, never
                                            silently dropped */
    AMGDD_ERR_OUT_OF_MEMORY = -7,        /* host or device allocation failed; detail string has the byte count */
    AMGDD_ERR_CUDA = -8,                 /* any CUDA runtime error, including "no device" */
    AMGDD_ERR_INDEX_RANGE = -9           /* a composite level has more than 2^31-1 local nonzeros, or a matrix
                                            row has more than 65535 entries */
} amgdd_status;

/* Sizes and the traffic model of DESIGN.md §"Algorithmic bytes". */
typedef struct amgdd_stats {
    int32_t num_levels;              /* L + 1 */
    int32_t num_subdomains;          /* P */
    int64_t n_fine;                  /* N */
    int64_t nnz_hierarchy;           /* sum_l nnz(A_l): what plain AMG stores */
    int64_t nnz_composite_real;      /* sum_{p,l} nnz of A_l over real rows of D_l^p */
    double overhead;                 /* nnz_composite_real / nnz_hierarchy */
    double operator_complexity;      /* nnz_hierarchy / nnz(A_0) */
    int64_t sum_real;                /* sum_{p,l} |D_l^p| */
    int64_t sum_ghost;               /* sum_{p,l} |D-bar_l^p \ D_l^p| */
    int64_t dropped_interp_entries;  /* A7 count; setup fails if nonzero */
    int64_t device_bytes;            /* bytes held on the device by this handle */
    int64_t shared_level_instances;  /* number of (p,l) pairs that reuse the single global copy of a level */
    /* algorithmic bytes of one AlgFAC V(nu,nu) iteration over all subdomains with the PRIVATE
       12 B/nnz CSR model of SURVEY.md §8(d), for nu = 1: [0] first iteration (no residual
       recalculation), [1] every later iteration */
    double model_bytes_fac_iter[2];
    /* bytes of the packed matrix streams the kernel of THIS build actually requests from HBM per
       iteration (groups and slice headers; vectors stay in shared memory / L2), same two cases */
    double stream_bytes_fac_iter[2];
    double model_bytes_global;       /* a1+a2+a3+a10 per AMG-DD cycle: A_0 stream, R_l streams, gathers */
    double setup_seconds_hierarchy;  /* host: S1-S5 */
    double setup_seconds_composite;  /* host: S6-S7 + local matrices + packing + upload */
    /* launch plan of the persistent AlgFAC kernel */
    int32_t block_bytes;             /* bytes of one (narrow) group of a packed stream = one slot of a warp's register ring */
    int32_t num_ways;                /* sub-streams per matrix = warps per CTA */
    int32_t window;                  /* rows per sort window of the SELL-32 streams */
    int32_t ring_stages;             /* groups a warp keeps in flight */
    int32_t x_cap;                   /* doubles in each of the two shared-memory vector buffers (0: they live in global memory) */
    int32_t fac_grid, fac_block, fac_smem_bytes;
    int64_t max_n_bar;               /* largest |D-bar_l^p| over all subdomains and levels */
    /* composite-grid assembly (NEXT 3): 1 when the local matrices were cut out, renumbered and packed
       on the device (the default), 0 for the host path (AMGDD_ASSEMBLE=host); the three parts of
       setup_seconds_composite on the device path: host index sets, device kernels + small copies, hierarchy upload */
    int32_t assembled_on_device;
    int32_t index_sets_on_device;    /* 1: the composite index sets (S6, S7) were grown on the device too (default with the device
                                        assembly; AMGDD_INDEX_SETS=host, or a breadth-first frontier of more than 262144 points, keeps
                                        the host search) */
    double setup_seconds_index_sets;
    double setup_seconds_assembly;
    double setup_seconds_upload;
    /* the matrix entries one AlgFAC iteration reads at this build's widths (8-byte value + 2-byte column index,
       4-byte where a level has more than 65535 columns), no padding, no headers, no vectors: what a perfect
       packing of the same streams would move; same two cases as model_bytes_fac_iter */
    double useful_bytes_fac_iter[2];
} amgdd_stats_t;

/* ---------------------------------------------------------------------------------------------
 * amgdd_setup -- problem statement A u = f with owned partition Omega_0^p and padding eta
 * (Alg. 2).  HOST arrays, copied.
 *   n            N, number of fine dofs (> 0)
 *   rowptr       n+1 entries, rowptr[0] = 0, non-decreasing
 *   colind       rowptr[n] entries, strictly ascending inside each row; the diagonal must be stored
 *   vals         rowptr[n] entries; an explicitly stored zero IS an edge of the graph (reading A8)
 *   num_subdomains  P (> 0)
 *   owner        n entries in [0,P): owner[i] = p  <=>  i in Omega_0^p
 *   eta          padding eta_l, the same on every level l < L (>= 0; reading A6)
 *   num_ghost    ghost layers (>= 1; the paper needs exactly 1; reading A13)
 *   max_levels   stop coarsening at this many levels (>= 1)
 *   theta        strength threshold in (0,1]  (S1)
 *   coarse_max   stop coarsening when n_l <= coarse_max (>= 1); ADDED to the north_star signature,
 *                BASELINE configs 1 and 2 state it ("coarsen to <= 16 / <= 64 dofs")
 *   out          receives the handle; left NULL on failure
 * Needs a CUDA device (the composite grids are uploaded).
 * ------------------------------------------------------------------------------------------- */
int amgdd_setup(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                int32_t max_levels, double theta, int32_t coarse_max, amgdd_handle_t* out);

/* amgdd_solve -- num_cycles AMG-DD cycles (Alg. 2 with Alg. 4 inside).
 *   b, x          DEVICE, n doubles.  x is in/out: initial guess on entry, iterate on return.
 *   num_cycles    0 .. 1023 (0 only evaluates resnorm[0]; the norms of one call live in a fixed device buffer of
 *                 1024 doubles: AMGDD_ERR_BAD_ARG beyond that -- call again to continue, x carries the state)
 *   num_fac_cycles  AlgFAC iterations per cycle (>= 1; Fig. 10)
 *   relax_sweeps  nu: l1-Jacobi sweeps before and after each coarse correction (>= 1; V(nu,nu))
 *   resnorm_host  HOST, num_cycles+1 doubles or NULL.  resnorm[k] = || b - A_0 x_k ||_2, k = 0 is
 *                 the initial guess.  With NULL the call only enqueues work on the handle's
 *                 stream and returns (and the norm of the final iterate is not evaluated): the 4 + L
 *                 launches of a cycle are captured once as a CUDA graph (per b, x, num_fac_cycles,
 *                 relax_sweeps) and replayed, one graph launch per cycle; AMGDD_GRAPH=0 in the
 *                 environment launches kernel by kernel.  Otherwise the call synchronises the stream
 *                 before returning.
 * Limits: the steps of one subdomain's cycle form a static program of at most 1024 steps, about
 * num_fac_cycles * (L * (4 + 2 * relax_sweeps) + 1) (twice the relaxation steps with the CF smoother), and the
 * kernel's tables hold at most 85 levels (L <= 84): AMGDD_ERR_BAD_ARG with the step count in the detail string
 * otherwise.  The call runs on the device the handle was set up on, whatever the caller's current device is. */
int amgdd_solve(amgdd_handle_t h, const double* b, double* x, int32_t num_cycles,
                int32_t num_fac_cycles, int32_t relax_sweeps, double* resnorm_host);

/* Same computation with HOST b and x: copies b and x to the device, runs amgdd_solve, copies x
 * back.  This is the end-to-end entry (host buffers in, host buffers out). */
int amgdd_solve_host(amgdd_handle_t h, const double* b_host, double* x_host, int32_t num_cycles,
                     int32_t num_fac_cycles, int32_t relax_sweeps, double* resnorm_host);

/* amgdd_vcycle -- num_cycles AMG V(nu1,nu2)-cycles on the same hierarchy (Alg. 1): the method the
 * paper compares AMG-DD with (one V(1,1)-cycle against one AMG-DD iteration, Fig. 14).  Whole-level
 * kernels, no subdomains: l1-Jacobi relaxation (the same as in amgdd_solve), r = f - A u, restriction with
 * P^T, dense solve on the coarsest level, interpolation.  b, x DEVICE (x in/out); resnorm_host HOST,
 * num_cycles+1 entries or NULL (asynchronous).  nu1, nu2 >= 0, nu1 + nu2 >= 1.  The first call uploads A_l
 * and P_l of all levels as CSR (memory: about 12 bytes per nonzero of the hierarchy). */
int amgdd_vcycle(amgdd_handle_t h, const double* b, double* x, int32_t num_cycles, int32_t nu1, int32_t nu2,
                 double* resnorm_host);

/* || b - A_0 x ||_2 (metric of Fig. 6; reading A16).  b, x DEVICE; out HOST. Synchronises. */
int amgdd_residual_norm(amgdd_handle_t h, const double* b, const double* x, double* out_host);

/* amgdd_residual_norm_static -- the same norm, || b - A x ||_2 (Fig. 6; r = b - A x as in P:471), for callers
 * that cannot allocate device memory at the point where they need it: this call performs no cudaMalloc, no cudaFree and
 * calls no library routine that allocates.  Typical callers: an application whose own pool (or a framework's caching
 * allocator) already holds the GPU's memory, so that a cudaMalloc here would fail or force that pool to give memory
 * back; a time-critical loop that must not hit the device-wide synchronisation of cudaFree; code that has no
 * amgdd_handle_t, since amgdd_setup allocates the whole hierarchy.  Nothing is taken from a handle: the caller passes the
 * matrix, the vectors and the result, all DEVICE pointers on the calling thread's CURRENT device:
 *   n                 rows of A (> 0, at most AMGDD_STATIC_MAX_ROWS)
 *   rowptr            n+1 entries (int64, rowptr[0] = 0), colind / vals: rowptr[n] entries, as amgdd_setup takes them
 *   b, x              n doubles (read only)
 *   r                 n doubles that receive b - A x, or NULL
 *   out_norm          1 double that receives the norm
 *   cuda_stream       a cudaStream_t passed as void* (NULL = legacy default stream)
 * The call only ENQUEUES a 4-byte memset and one kernel on that stream and returns; read *out_norm after synchronising
 * the stream.  The kernel's scratch memory -- one partial sum per 256 rows and an arrival counter -- is a fixed
 * file-scope device array of 512.25 KiB, which every GPU that loads this library keeps until the process exits; that
 * array is why n is limited: AMGDD_ERR_BAD_ARG with the limit in the detail string beyond AMGDD_STATIC_MAX_ROWS (use
 * amgdd_residual_norm, whose scratch is sized by amgdd_setup, for larger systems).
 * First call on a device: it looks the array's device address up once (cudaGetSymbolAddress, with that device
 * current, which may make the runtime load this library's kernels there).  Make that first call at start-up, before any
 * stream capture begins on the device.
 * Sharing: all calls on a device use the one array.  A call clears the counter it needs and never reads partial sums of
 * an earlier call, so calls that follow each other on one stream are independent; two calls that can be in flight at
 * the same time (different streams, different host threads without ordering) race on it and return garbage norms.
 * Rows are summed as in amgdd_residual_norm (stored order, no contraction): r is bit-identical to that path, the norm
 * agrees to rounding.  Entries are not validated (a column index outside [0, n) reads out of bounds). */
#define AMGDD_STATIC_MAX_ROWS 16777216
int amgdd_residual_norm_static(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals, const double* b,
                               const double* x, double* r, double* out_norm, void* cuda_stream);

/* Relaxation used by amgdd_solve, amgdd_solve_host and amgdd_vcycle from the next call on.
 *   AMGDD_SMOOTHER_L1_JACOBI     (default) one l1-Jacobi sweep over the real points (reading A2, BASELINE)
 *   AMGDD_SMOOTHER_CF_L1_JACOBI  the paper's "CF l1-scaled Jacobi" (reading A2b): every sweep is two
 *                                half-sweeps, C-points then F-points before the coarse correction, F-points
 *                                then C-points after it; each half-sweep is one pass over the real rows of A_l */
#define AMGDD_SMOOTHER_L1_JACOBI 0
#define AMGDD_SMOOTHER_CF_L1_JACOBI 1
int amgdd_set_smoother(amgdd_handle_t h, int32_t type);

/* Use this CUDA stream (a cudaStream_t passed as void*; NULL = legacy default stream). */
int amgdd_set_stream(amgdd_handle_t h, void* cuda_stream);

/* Free everything the handle owns (device and host). NULL is accepted. */
int amgdd_destroy(amgdd_handle_t h);

/* Static string for a status code. */
const char* amgdd_strerror(int code);

/* One-line detail of the most recent failure (setup failures included). Thread-local storage. */
const char* amgdd_last_error_detail(void);

/* ---- introspection: the index-exact contract (S7) and the roofline model ------------------ */
int amgdd_num_levels(amgdd_handle_t h, int32_t* L_plus_1);
int amgdd_level_size(amgdd_handle_t h, int32_t l, int64_t* n_l, int64_t* nnzA, int64_t* nnzP);
/* cf_host: n_l entries, +1 C-point, -1 F-point; l < L. */
int amgdd_get_cf(amgdd_handle_t h, int32_t l, int8_t* cf_host);
/* which = 0: A_l (n_l x n_l), 1: P_l (n_l x n_{l+1}, l < L).  HOST outputs sized by amgdd_level_size. */
int amgdd_get_level_matrix(amgdd_handle_t h, int32_t l, int32_t which, int64_t* rowptr, int32_t* colind,
                           double* vals);
int amgdd_composite_size(amgdd_handle_t h, int32_t p, int32_t l, int64_t* n_real, int64_t* n_ghost);
/* real_gid: |D_l^p| global indices, ascending; ghost_gid: |D-bar_l^p \ D_l^p|, ascending (S7).  On a level that the
 * subdomain covers completely (D_l^p = Omega_l, always true on L; reading A5) real_gid is 0 .. n_l - 1, there are
 * no ghost points (amgdd_composite_size reports n_ghost = 0) and ghost_gid is not written. */
int amgdd_get_composite(amgdd_handle_t h, int32_t p, int32_t l, int32_t* real_gid, int32_t* ghost_gid);
int amgdd_get_stats(amgdd_handle_t h, amgdd_stats_t* s);

/* ---- sharding over ranks (paper section 5, and Alg. 5) -----------
 * One process per GPU; rank r of R holds the contiguous block of subdomains [ceil(r P / R), ceil((r + 1) P / R)) and owns
 * Omega_l^r, the union of their owned points on every level.  The library has no communication layer: one sharded
 * AMG-DD cycle is 2 L + 2 STAGES, each "compute + pack on the device -> the CALLER exchanges the packed doubles between
 * the ranks (torch.distributed all_to_all_single, send counts per rank from amgdd_shard_stage_counts) -> unpack":
 *   stage 0            x at the columns this rank's rows of A_0 read on other ranks ("mat-vec communication with A_0")
 *   stage 1 + l, l < L r_l likewise for its rows of R_l; before packing, r_l is computed on the owned rows
 *   stage L + 1 + k    Alg. 5 for level l = L - k: residuals at Psi = { i in Omega_l^r : dist(i, Omega_l^q) <= eta } and at
 *                      the composite grid Psi_c built from Psi on the coarser levels, to every such rank q (all of level
 *                      L to every rank, reading A5); values a rank received earlier are forwarded
 * then amgdd_shard_local_solve runs AlgFAC on the rank's subdomains and updates x on its dofs.  x, b and the residual
 * vector keep their global numbering on every rank; only the entries a rank owns or received are valid.
 *
 * Index protocol, once after setup (the redundancy removal of P:250).  For every stage in ascending order and every source
 * in ascending rank: the source's amgdd_shard_plan_list(which = 0) is ANNOUNCED to the destination; the destination runs
 * amgdd_shard_plan_recv_filter on it (positions it owns or was already promised come back as redundant; the rest
 * becomes its receive list) and returns the redundant positions; the source removes them with
 * amgdd_shard_plan_apply_drop.  Then amgdd_shard_commit uploads the final lists.  A position indexes x (stage 0) or the
 * concatenated residual vector r_0 | r_1 | ... (offsets: amgdd_shard_plan_level).  The protocol runs ONCE per plan: a second
 * amgdd_shard_plan_recv_filter or amgdd_shard_plan_apply_drop for the same (stage, peer) pair and a second amgdd_shard_commit
 * return AMGDD_ERR_BAD_ARG and change nothing (the filter marks positions as held for good; repeating it would empty the
 * send lists).  amgdd_shard_plan_create builds a plan
 * WITHOUT a CUDA device (the hierarchy is rebuilt on the host): tests of the protocol use it. */
typedef struct amgdd_shard_plan_s* amgdd_shard_plan_t;
int amgdd_setup_shard(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                      int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t num_ghost,
                      int32_t max_levels, double theta, int32_t coarse_max, int32_t rank, int32_t nranks,
                      amgdd_handle_t* out);      /* as amgdd_setup; builds the rank's subdomains only (local index p - sub_lo) */
int amgdd_shard_plan_create(int64_t n, const int64_t* rowptr, const int32_t* colind, const double* vals,
                            int32_t num_subdomains, const int32_t* owner, int32_t eta, int32_t max_levels, double theta,
                            int32_t coarse_max, int32_t rank, int32_t nranks, amgdd_shard_plan_t* out);
int amgdd_shard_plan_destroy(amgdd_shard_plan_t p);
int amgdd_get_shard_plan(amgdd_handle_t h, amgdd_shard_plan_t* out);   /* borrowed: valid until amgdd_destroy(h) */
/* info: rank, nranks, L + 1, stages, first and one-past-last subdomain of the rank */
int amgdd_shard_plan_info(amgdd_shard_plan_t p, int32_t info[6]);
int amgdd_shard_plan_level(amgdd_shard_plan_t p, int32_t l, int64_t* n_l, int64_t* r_offset, int64_t* n_owned);
int amgdd_shard_plan_owner_rank(amgdd_shard_plan_t p, int32_t l, int32_t* owner_rank);   /* HOST, n_l entries */
/* which = 0: positions this rank sends to `peer` in `stage`; 1: positions it receives from `peer` (after recv_filter).
 * pos = NULL returns the count only. */
int amgdd_shard_plan_list(amgdd_shard_plan_t p, int32_t which, int32_t stage, int32_t peer, int64_t* pos, int64_t* count);
int amgdd_shard_plan_stage_vector(amgdd_shard_plan_t p, int32_t stage, int32_t* vec);    /* 0: positions index x, 1: the residual vector */
int amgdd_shard_plan_recv_filter(amgdd_shard_plan_t p, int32_t stage, int32_t src, const int64_t* announced, int64_t count,
                                 int64_t* redundant, int64_t* nredundant);               /* redundant: room for count entries */
int amgdd_shard_plan_apply_drop(amgdd_shard_plan_t p, int32_t stage, int32_t dest, const int64_t* redundant, int64_t count);
int amgdd_shard_commit(amgdd_handle_t h);
/* send_counts, recv_counts: HOST, nranks entries: doubles to / from every rank in this stage (buffers: rank after rank) */
int amgdd_shard_stage_counts(amgdd_handle_t h, int32_t stage, int64_t* send_counts, int64_t* recv_counts);
int amgdd_shard_stage_pack(amgdd_handle_t h, int32_t stage, const double* b, const double* x, double* sendbuf);   /* DEVICE pointers */
int amgdd_shard_stage_unpack(amgdd_handle_t h, int32_t stage, double* x, const double* recvbuf);
int amgdd_shard_local_solve(amgdd_handle_t h, double* x, int32_t num_fac_cycles, int32_t relax_sweeps);            /* a3-a10 */
int amgdd_shard_sqnorm(amgdd_handle_t h, double* out_host);   /* sum of r_0^2 over the owned rows, as computed before stage 1 */
/* The simple alternative of SURVEY.md section 8(e): all-gather x, then amgdd_solve on the shard handle (global residual
 * and restriction redundantly on every rank, AlgFAC on the rank's subdomains).  buf: x at the dofs of a rank, ascending. */
int amgdd_shard_owned_count(amgdd_handle_t h, int32_t rank, int64_t* count);
int amgdd_shard_pack_owned(amgdd_handle_t h, const double* x, double* buf);
int amgdd_shard_unpack_owned(amgdd_handle_t h, int32_t src_rank, const double* buf, double* x);

/* ---- the HBM layout of the matrices, exposed for tests and tools --------------------------------
 * Packs a CSR matrix (HOST; rowptr32 has nrows+1 int32 entries starting at 0, at most 65535
 * entries per row) into the "SELL-32 group" streams the AlgFAC kernel reads with coalesced 128-bit
 * loads (layout: DESIGN.md "Data layout", csrc/amgdd_stream.hpp): rows [0, n_real) and
 * [n_real, nrows) are two row groups (real / ghost rows of a composite A_l); inside
 * windows of `window` rows (multiple of 32 in [32, 1048576]) rows are sorted by descending length
 * and cut into slices of 32 rows, one warp lane per row; a slice is stored as K = max(1,
 * ceil(longest row / 4)) groups of 4 steps (zero padding past the end of a row) and one header of 4 bytes
 * per lane (narrow: row | K << 16 | flag << 31; 0xFFFF: no row) or 8 bytes per lane (wide: row, K | flag << 31);
 * the slices are dealt to AMGDD_NUM_WAYS sub-streams ("ways", one per warp of the kernel).  The l1 diagonal
 * a relaxing step needs is not part of the stream (the kernel fetches it like the other row-local operands).
 *   row_flags  HOST, nrows bytes (0/1) stored in bit 31 of the header word (C-point of the row's level), or NULL
 *   wide     0: uint16 column indices and rows (needs every column < 65536 and at most 65535 rows), 1: uint32
 *   out_ways HOST, AMGDD_NUM_WAYS entries, or NULL
 * With out = NULL only *out_bytes and out_ways are computed.  Returns AMGDD_ERR_INDEX_RANGE for a
 * row with more than 65535 entries, AMGDD_ERR_BAD_ARG on a bad argument or if out_capacity is too
 * small.  Needs no CUDA device. */
#define AMGDD_NUM_WAYS 16
#define AMGDD_GROUP_BYTES_NARROW 1280
#define AMGDD_GROUP_BYTES_WIDE 1536
#define AMGDD_HEADER_BYTES_NARROW 128
#define AMGDD_HEADER_BYTES_WIDE 256
typedef struct amgdd_way {
    uint32_t grp_off128;   /* the way's groups start 128 * grp_off128 bytes from the start of the stream */
    uint32_t hdr_off128;   /* its slice headers start 128 * hdr_off128 bytes from the start of the stream */
    uint32_t ngroups;      /* groups of the way, contiguous */
    uint32_t ngroups_real; /* leading groups that belong to slices of the first row group */
    uint32_t nslices;      /* slices (= headers) of the way */
    uint32_t nslices_real; /* leading slices of the first row group */
    uint32_t reserved[2];
} amgdd_way_t;
int amgdd_pack_stream(int32_t nrows, int32_t n_real, const int32_t* rowptr32, const int32_t* colind, const double* vals,
                      const uint8_t* row_flags, int32_t wide, int32_t window, void* out,
                      int64_t out_capacity, int64_t* out_bytes, amgdd_way_t* out_ways);

/* ---- measurement support ------------------------------------------------------------------
 * Device time (ms, CUDA events on the handle's stream) of the phases of the most recent
 * amgdd_solve that was given a non-NULL resnorm_host, summed over its cycles:
 *   ms[0] global residual + norm (a1, a11)   ms[1] restriction chain (a2)
 *   ms[2] AlgFAC kernel incl. gather and owned update (a3-a10)   ms[3] whole solve
 * launches[0..2]: kernel launches in the same three groups. */
int amgdd_last_solve_profile(amgdd_handle_t h, double ms[4], int64_t launches[3]);

/* Debugging aid.  If the environment variable AMGDD_FAC_PROFILE=1 was set when amgdd_setup ran,
 * the AlgFAC kernel adds SM clock cycles (taken by thread 0 of each CTA) to per-CTA counters; this
 * call sums them over the CTAs into out[16] (HOST) and, with reset != 0, clears them:
 *   [0] CTA barrier waits  [1] fetching a subdomain and its tables  [2] work outside the mat-vec
 *   rows (ghost carry, zeroing, staging)  [3] mat-vec start-up (first groups, first header)
 *   [4] whole kernel  [5] residual gather (a3)  [6] matrix-free first sweep of level 0
 *   [7..11] whole mat-vec steps: relax, A t, restrict, recalculate, interpolate
 *   [12] coarse solve  [13] owned update (a10)  [14] waits for a slice's staged header / operands
 *   [15] waits for a block of the register ring (HBM latency).
 * Returns AMGDD_ERR_BAD_ARG if profiling was not enabled.  Timed runs must not enable it. */
int amgdd_debug_fac_cycles(amgdd_handle_t h, int64_t out[16], int32_t reset);
/* Same switch: SM cycles of every step of the AlgFAC program (thread 0 of each CTA, summed over CTAs and
 * subdomains); out has 4 n entries: out[j] = step j (j < n), out[n + j] = wait at the CTA barrier after it,
 * out[2n + j] = its waits for blocks of the register ring, out[3n + j] = its waits for staged slice operands;
 * kinds_levels[j] (HOST, n entries or NULL) = 256 * kind + level of step j.  Clears the counters. */
int amgdd_debug_fac_op_cycles(amgdd_handle_t h, int64_t* out, int32_t n, int32_t* kinds_levels);

/* Test support for the composite-grid assembly: copies one array of the
 * private block (subdomain p, level) out of the device blob into HOST memory `out`.
 *   which  0 gid (int32[n_bar])   1 dinv (double[n_real])   2 / 3 / 4 the packed A_l / P_l / R_l stream
 *          5 the owned-dof index list of the subdomain (int32[n_owned]; level ignored)
 * *out_bytes receives the size of the array (0 for a level that uses the shared global copy); with out = NULL
 * only the size is returned.  AMGDD_ERR_BAD_ARG on a bad index or if out_capacity is too small. */
int amgdd_debug_read_block(amgdd_handle_t h, int32_t p, int32_t level, int32_t which, void* out, int64_t out_capacity,
                           int64_t* out_bytes);

#ifdef __cplusplus
}
#endif
#endif /* AMGDD_H */
