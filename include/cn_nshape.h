/*
 * cn_nshape.h -- C ABI of the B200-native N-shaped partition Crank-Nicolson stepper.
 *
 * The library advances the 1-D time-dependent Schroedinger equation by the Crank-Nicolson
 * propagator
 *        T psi(t+dt) = T^dagger psi(t),     T = 1 + (i dt / 2) H              PAPER.md:48-52 (Eq. 2)
 * i.e. per step the explicit half-step d = T^dagger psi (Eq. 3) followed by the
 * implicit half-step T psi' = d (Eq. 4), a complex tridiagonal system
 *        b_i psi_{i-1} + a_i psi_i + c_i psi_{i+1} = d_i,  psi_0 = psi_{N+1} = 0   PAPER.md:80-84 (Eq. 5)
 * which is solved by the N-shaped partition method of PAPER.md:78-149 (section 4) and Appendix I
 * (PAPER.md:298-337): the N unknowns are split into P contiguous blocks, every block eliminates
 * locally (stages RD, RU), adds its contributions to its joint lines (JD, JU), a reduced system
 * on the joint lines is solved (RS) and every block substitutes the two support values (SS).
 *
 * Conventions:
 *   H = -1/2 d^2/dx^2 + V(x) in atomic units, 3-point stencil, Dirichlet ends:
 *       (H psi)_j = -(psi_{j-1} - 2 psi_j + psi_{j+1}) / (2 dx^2) + V_j psi_j
 *   so  b = c = -i s,  a_j = 1 + i (2 s + dt V_j / 2),  s = dt / (4 dx^2).   V is real.
 *   Block w (w = 0..P-1) owns rows [floor(w N / P), floor((w+1) N / P)); its LAST row is the joint
 *   line J_w; a virtual joint line "row -1, psi = 0" closes the first block (PAPER.md:92 fixes only
 *   J_0 = first row, J_P = last row and allows unequal blocks).
 *   psi is N interleaved complex128 values (re, im), 16-byte aligned, updated IN PLACE.
 *
 * All functions return a cn_status and never throw.  Pointers are labelled HOST or DEVICE.  No
 * function allocates inside cn_step / cn_batched_sweep.  All work is enqueued on the given CUDA
 * stream (a cudaStream_t passed as void*; NULL = the legacy default stream) and, unless stated,
 * does not synchronise.  There is NO CPU fallback: without a CUDA device every call that needs one
 * returns CN_ECUDA.
 */
#ifndef CN_NSHAPE_H
#define CN_NSHAPE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cn_plan cn_plan; /* opaque, owned by the library */

typedef enum {
    CN_OK = 0,
    CN_EINVAL = 1,         /* bad argument (N < 2, P < 1, P > N, dx <= 0, non-finite dx/dt, dt == 0, NULL, misaligned) */
    CN_ENOMEM = 2,         /* host or device allocation failed / device budget too small */
    CN_ECUDA = 3,          /* a CUDA call failed; see cn_last_cuda_error */
    CN_ENOTFACTORIZED = 4, /* cn_step / cn_batched_sweep before cn_factorize */
    CN_EBREAKDOWN = 5,     /* zero or non-finite pivot met by cn_factorize */
    CN_ETOOLARGE = 6       /* cn_step_static: N exceeds CN_STATIC_NMAX, the size of the library's static device scratch */
} cn_status;

/* Options for cn_plan_set_option (all optional; call before cn_factorize). */
typedef enum {
    CN_OPT_PATH = 1,        /* 0 = auto (default), 1 = force the generic thread-per-block kernels,
                               2 = force the tiled TMA kernels (CN_EINVAL at factorize if the shape does not fit) */
    CN_OPT_TILE_THREADS = 2,/* threads per CTA of the tiled kernels: 0 = auto (64), else 32/64/128/256/512 (8 points per
                               thread; at least one block per tile) */
    CN_OPT_RS_TOPMAX = 3,   /* largest reduced system solved by the single-CTA RS kernel (1..8192, default 4096);
                               a larger one is partitioned again into groups of 256 joint lines (next RS level) */
                            /* 4: not used (CN_EINVAL) */
    CN_OPT_RS_LEVELS = 5,   /* 0 = auto (levels added while the system exceeds RS_TOPMAX), k >= 1 = exactly k nested
                               levels where possible (Eq. 6; CN_EINVAL at factorize if the last
                               level exceeds 8192 rows), -1 = paper-literal serial RS by one thread */
    CN_OPT_PROFILE = 6,     /* 1 = bracket every fused-pass and RS launch of cn_step with CUDA events on the
                               launching stream (read back with cn_plan_get_profile); default 0 */
    CN_OPT_PDL = 7,         /* 1 (default) = launch the per-step kernels with programmatic dependent launch so that
                               each kernel's independent prefetch overlaps the tail of its predecessor; 0 = plain */
    CN_OPT_ONCHIP = 8,      /* 1 (default) = a system of N <= 4096 points whose plan forces neither a path nor an RS
                               structure is stepped by ONE single-CTA launch per cn_step call that keeps psi in
                               registers and loops over the steps on chip (cn_plan_info.path = 3); 0 = never */
                            /* 9: not used (CN_EINVAL) */
    CN_OPT_RS_GROUP = 10,   /* joint lines per group of a nested RS level (2..2^20, default 256): the fan-out
                               n_bl(i) / n_bl(i+1) of PAPER.md:239-247 Eq. 8; any value but 256 selects the
                               paper-shaped kernels in which one thread serves one group */
    CN_OPT_RS_SERIAL_TOP = 11, /* 1 = the LAST level is solved serially by one thread (the beta n_bl term of Eq. 8)
                               whatever the number of nested levels; default 0 = one CTA in parallel */
    CN_OPT_RS_TOP_IN_SUBST = 12, /* 1 (default) = a last level of at most 256 rows is solved inside the substitution
                               kernel of the level below it, redundantly by every CTA (one launch less per step);
                               a value v > 1 sets the row limit to min(v, 1024); 0 = always by its own kernel */
    CN_OPT_BY_COLS = 14,    /* systems per strip of the interleaved-layout kernel of cn_batched_sweep: 0 = auto, 8 = strips
                               128 B wide, 4 = strips 64 B wide (systems of >= 128 rows): twice the rows per CTA, so
                               half the CTAs per cluster for systems of 2048 rows and more */
    CN_OPT_KEEP_P = 13      /* 0 (default) = unless the caller's blocks already have 8 * 2^k <= 256 rows, the tiled path
                               partitions the system itself: blocks of the largest 8 * 2^k <= 256 rows that divides N
                               (cn_plan_info.P_effective; psi does not depend on the partition);
                               1 = the caller's P is the partition: equal blocks of 8 * 2^k <= 4096 rows run on the tiled
                               kernels as given (slower above 256 rows: a block then spans warps), any other shape on
                               the generic thread-per-block kernels */
} cn_option;

typedef struct {
    int64_t N, P;
    int32_t path;            /* 1 generic, 2 tiled, 3 whole system on chip (N <= 4096) */
    int32_t tile_threads;    /* threads per CTA of the pass kernel (tiled path) */
    int64_t tile_points;     /* points per CTA (tiled path) */
    int32_t rs_levels;
    int32_t out_of_core;     /* 1 if a device budget forces host streaming */
    size_t device_bytes;     /* device memory owned by the plan */
    int64_t launches;        /* kernels launched by this plan so far (all entry points) */
    double bytes_per_point_step; /* HBM bytes per point a fused step of the tiled path moves (48: psi 16 + q 16 in, psi 16
                                    out; the formulation that also reads gamma, SURVEY 8d's declared minimum, moves 56) */
    int64_t P_effective;     /* blocks the kernels work with: P, or N / (8 * 2^k) when the tiled path chooses the
                                partition itself (see cn_plan_create, CN_OPT_KEEP_P) */
} cn_plan_info;

/*
 * cn_plan_create -- describe one Hamiltonian / time step.
 *   out : HOST, receives the plan.            N : number of grid points (rows of T), N >= 2.
 *   P   : number of blocks n_bl, 1 <= P <= N.  Blocks need not be equal.  P is the partition the
 *         kernels use ONLY under CN_OPT_PATH = 1 (generic kernels) or CN_OPT_KEEP_P = 1; by default it is a hint:
 *         psi does not depend on the partition (direct solver), so when N is a multiple of 8 the library runs the
 *         tiled kernels on blocks of 8 * 2^k <= 256 rows of its own choosing (the caller's blocks if they already
 *         have that shape) and reports the count as cn_plan_info.P_effective.
 *   dx, dt : grid spacing (> 0) and time step (!= 0, negative = backward propagation).
 *   V   : N real potential values, HOST or DEVICE pointer (detected); copied, caller keeps ownership.
 * Allocates nothing on the device yet except the copy of V.
 */
cn_status cn_plan_create(cn_plan **out, int64_t N, int64_t P, double dx, double dt, const double *V);

/* Cap the device memory the library may own for this plan (config "out-of-core", PAPER.md:94, 161-165:
 * "neither the matrix nor the wavefunction ever need to be placed entirely on a single process").
 * When the factors do not fit, cn_step expects psi in PINNED HOST memory and streams partitions
 * H2D / solve / D2H; factors are recomputed per chunk.  bytes = 0 removes the cap. */
cn_status cn_plan_set_device_budget(cn_plan *plan, size_t bytes);

cn_status cn_plan_set_option(cn_plan *plan, cn_option key, int64_t value);

/*
 * cn_factorize -- everything that does not depend on d, once per (H, dt) (section 5.2.4:
 * "storage of a column of the values of r_i factors"; precomputed 1/a_i).
 * Stores per point the inverse pivot of the block-local downward elimination (RD) and the real
 * diagonal term of T^dagger, per joint line the factored reduced matrix (RS).  Synchronises `stream`
 * once at the end to report CN_EBREAKDOWN.
 */
cn_status cn_factorize(cn_plan *plan, void *stream);

/*
 * cn_step -- nsteps Crank-Nicolson steps of one system, in place.
 *   psi : N complex128.  DEVICE pointer normally; PINNED HOST pointer when the plan is out-of-core.
 * Stages per step: RHS product fused into RD, RU, JD/JU into two slots per joint
 * line, RS, SS fused with the psi write and with RHS+RD/RU of the next step
 * (PAPER.md:27, 201).  Asynchronous on `stream` (the out-of-core mode uses internal streams and
 * returns after the last copy is enqueued; synchronise `stream` to wait).
 */
cn_status cn_step(cn_plan *plan, void *psi, int64_t nsteps, void *stream);

/*
 * Time-dependent Hamiltonian (the propagator of a step uses H(t + dt/2); the laser-driven use
 * case of PAPER.md:70).  H(t) = H0 + f(t) g(x): the potential of step k is V_j + field[k] g_j.
 *   cn_plan_set_td_shape : g, N real values, HOST or DEVICE pointer, copied (e.g. g_j = x_j for a dipole term).
 *   cn_step_td           : nsteps steps in place on the DEVICE vector psi; field = nsteps HOST values
 *                          f(t_k + dt/2), read during the call.  Every step redoes the factorization on the device
 *                          (launches only, no allocation, no synchronisation) and runs
 *                          RHS + RD/RU/JD/JU -> RS -> SS with that step's factors; on return the plan again holds
 *                          the factors of the static H.  Not available for out-of-core plans (CN_EINVAL);
 *                          CN_EINVAL without a shape; a breakdown cannot occur for real V and g (T stays strictly
 *                          diagonally dominant) and is not checked inside the loop.
 */
cn_status cn_plan_set_td_shape(cn_plan *plan, const double *g);
cn_status cn_step_td(cn_plan *plan, void *psi, int64_t nsteps, const double *field, void *stream);

/*
 * cn_batched_sweep -- the same step for nsys independent systems that share the plan's matrix
 * (operator splitting; config C4).  System k, row j lives at
 * psi[k * sys_stride + j * elem_stride] (strides in complex elements).  Supported layouts:
 * elem_stride == 1 (x-sweep, rows contiguous) and sys_stride == 1 (y-sweep, systems interleaved).
 */
cn_status cn_batched_sweep(cn_plan *plan, void *psi, int64_t nsys, int64_t elem_stride, int64_t sys_stride,
                           int64_t nsteps, void *stream);

/*
 * Many systems with a potential of their own each (operator splitting turns an N-D
 * problem into series of 1-D problems, and with a non-separable V(x, y) every line of a sweep has its own matrix).
 *   cn_plan_set_systems : declares, before cn_factorize, that the plan's N rows (its V, and psi alike) are `nsys`
 *       independent systems of N / nsys rows with Dirichlet ends each; row j of system k lives at
 *       [k * sys_stride + j * elem_stride].  Dense layouts only: contiguous systems (elem_stride = 1, sys_stride =
 *       N / nsys) or interleaved systems (elem_stride = nsys, sys_stride = 1).  cn_factorize then stores per-point
 *       factors of every system.  Contiguous systems of 8 * 2^k rows run on the tiled kernels of cn_step -- a system
 *       boundary is a joint line above which "psi = 0", like the top of a single system, so the whole array is one
 *       fused pass: 56 B per point and step (psi 16 + q 16 + gamma 8 in, psi 16 out; 32 B in cn_batched_sweep, whose
 *       systems share one matrix that stays on chip), SS(k) fused with RD/RU(k+1) over the steps of a call.
 *       Any other dense layout runs on one thread per system (correctness path).
 *   cn_batched_sweep_v  : nsteps CN steps of all systems in place (the same call as cn_step on such a plan).
 * Not available for out-of-core, sharded or time-dependent use (CN_EINVAL); cn_batched_sweep refuses such a plan.
 */
cn_status cn_plan_set_systems(cn_plan *plan, int64_t nsys, int64_t elem_stride, int64_t sys_stride);
cn_status cn_batched_sweep_v(cn_plan *plan, void *psi, int64_t nsteps, void *stream);

cn_status cn_destroy(cn_plan *plan);

cn_status cn_plan_get_info(const cn_plan *plan, cn_plan_info *info);

/* Kernel timings gathered since the last call while CN_OPT_PROFILE was on (measurement aid):
 * out[0] = sum of fused-pass kernel durations in ms, out[1] = their count,
 * out[2] = sum of RS kernel durations in ms,        out[3] = their count.
 * HOST pointer to 4 doubles.  Synchronises the recorded events, then resets the counters. */
cn_status cn_plan_get_profile(cn_plan *plan, double *out);
const char *cn_status_string(cn_status s);
/* last CUDA runtime error code seen by this plan (0 = cudaSuccess) */
cn_status cn_last_cuda_error(const cn_plan *plan, int *cuda_err);
const char *cn_version(void);

/*
 * General complex tridiagonal front end (Eq. 5):  b_i x_{i-1} + a_i x_i + c_i x_{i+1} = d_i,
 * i = 1..N, x_0 = x_{N+1} = 0, ARBITRARY complex b, a, c (b_1 and c_N are ignored).  Solved by the same N-shaped
 * partition scheme, nested: blocks of 256 rows, the last row of a block is its joint line.
 *   cn_tridiag_create : b, a, c = N complex128 each, HOST or DEVICE pointers, copied; does all matrix-side work
 *                        on `stream` and synchronises it once.  No pivoting (as in the paper):
 *                       CN_EBREAKDOWN if a zero or non-finite pivot is met; diagonally dominant matrices are safe.
 *   cn_tridiag_solve  : d, x = N complex128 DEVICE vectors (x may alias d); asynchronous on `stream`, no allocation.
 *   cn_tridiag_destroy: frees everything.
 *   cn_tridiag_create_blocks : the same with CALLER-PLACED joint lines ("the blocks may differ in
 *                       size"): joints = P strictly increasing HOST row indices (0-based), joints[P-1] = N - 1; block w =
 *                       rows (joints[w-1], joints[w]], its last row is its joint line, blocks of one row (joint line
 *                       only) and two rows allowed.  Every caller joint line is a joint line of the first level; a
 *                       block of more than 256 rows is partitioned again by the library (further joint lines inside it,
 *                       the same method one level down), so that every block runs on one warp.  The
 *                       reduced system on the joint lines runs on the nested warp-per-group levels.  CN_EINVAL for
 *                       joints that are not increasing or do not end at N - 1.  The solution does not depend on the
 *                       joints.
 */
typedef struct cn_tridiag cn_tridiag;
cn_status cn_tridiag_create(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c, void *stream);
cn_status cn_tridiag_create_blocks(cn_tridiag **out, int64_t N, const void *b, const void *a, const void *c, int64_t P,
                                   const int64_t *joints, void *stream);
cn_status cn_tridiag_solve(cn_tridiag *t, const void *d, void *x, void *stream);
cn_status cn_tridiag_destroy(cn_tridiag *t);

/*
 * Sharded mode: ONE system of N_total rows spread over `nshards` processes / GPUs, the wave function
 * never gathered ("neither the matrix nor the wavefunction ever need to be placed entirely on a
 * single process ... the only data that needs to be gathered is on the joint lines"), one small exchange around the
 * RS stage per step (section 5.2.1; process layout of PAPER.md:282-288 section 6.2).
 *
 * Shard r (0 <= r < nshards, in row order) owns N_local consecutive rows -- the same N_local (a multiple of 256) and
 * the same options on every shard -- with its own factors, slots and nested RS levels over its own joint lines.
 * Its last row is a joint line of every level, so the shard is one block of the partition method applied once more
 * on top (Eq. 6).  What crosses shards, as opaque records of complex128 values that the CALLER
 * all-gathers in rank order (any transport: NCCL, MPI, peer copies; the library never communicates):
 *   - once per (H, dt), the matrix side:  cn_shard_factorize_local writes this shard's record of
 *     `matrix_count` values, cn_shard_factorize_finish reads the nshards records and factors the last RS level of the
 *     whole system, replicated on every shard (no root process; PAPER.md:207 names the alternative);
 *   - per step, the d side: a record of `step_count` = 2 nt values -- the two right-hand-side slots of this shard's
 *     nt last-level rows, written in place by the kernels (nothing is packed), one of them the JU
 *     contribution to the last row of the preceding shard; with nt = 1 these are the two values per process of
 *     PAPER.md:175 for a pre-factored matrix.  The two support values a process gets back
 *      are computed locally from the gathered records;
 *   - once per run, psi^0 on the last row of every shard (1 value; cn_shard_edge), which the first explicit half-step
 *     of the next shard needs (Eq. 3).
 * A run of n steps on one vector:  cn_shard_edge -> gather -> cn_shard_prologue -> [gather -> cn_shard_advance] x (n-1)
 * -> gather -> cn_shard_epilogue.   Stages: prologue = RHS + RD/RU/JD/JU of step 1 and the local reductions; advance =
 * last-level RS + substitutions + SS of step k fused with RHS + RD/RU/JD/JU of step k+1 + local
 * reductions; epilogue = last-level RS + substitutions + SS.  All records are DEVICE pointers, 16-byte aligned; every
 * call is asynchronous on `stream` except the two factorize calls, which synchronise it once.  psi is the shard's
 * N_local complex128 DEVICE vector, updated in place.  nshards = 1 is allowed (records unused).
 * Errors: CN_EINVAL for shapes the sharded mode does not take (N_local not a multiple of 256, forced generic path,
 * device budget, RS options other than CN_OPT_RS_TOPMAX) and for gathered matrix records that are not nshards records
 * of equal-shaped shards in rank order.  cn_factorize / cn_step / cn_step_td on a plan with nshards > 1: CN_EINVAL.
 */
cn_status cn_shard_plan_create(cn_plan **out, int64_t N_local, int64_t P_local, double dx, double dt,
                               const double *V_local, int32_t shard, int32_t nshards);
/* complex128 values per shard record: matrix_count (factorize), step_count (every step) */
cn_status cn_shard_counts(const cn_plan *plan, int64_t *matrix_count, int64_t *step_count);
cn_status cn_shard_factorize_local(cn_plan *plan, void *matrix_send, void *stream);
cn_status cn_shard_factorize_finish(cn_plan *plan, const void *matrix_all, void *stream);
cn_status cn_shard_edge(cn_plan *plan, const void *psi, void *edge_send, void *stream);
cn_status cn_shard_prologue(cn_plan *plan, void *psi, const void *edges_all, void *step_send, void *stream);
cn_status cn_shard_advance(cn_plan *plan, void *psi, const void *step_all, void *step_send, void *stream);
cn_status cn_shard_epilogue(cn_plan *plan, void *psi, const void *step_all, void *stream);

/*
 * The same protocol driven by the library, one shard per process (or thread): the plan owns the records and calls
 * `exchange` wherever a gather is due.  exchange(ctx, send, recv, count, stream) must ENQUEUE on `stream` an all-gather
 * of `count` complex128 values per shard -- send: this shard's record, recv: nshards records in rank order, both DEVICE
 * pointers owned by the plan -- and return CN_OK (e.g. one ncclAllGather of 2 * count doubles); any other status aborts
 * the call and is returned.  It is not called when nshards = 1.
 *   cn_shard_factorize : cn_shard_factorize_local -> exchange -> cn_shard_factorize_finish (synchronises twice).
 *   cn_shard_run       : nsteps steps of this shard's rows: nsteps + 1 exchanges, no synchronisation,
 *                        no allocation after the first call.
 */
typedef cn_status (*cn_exchange_fn)(void *ctx, const void *send, void *recv, int64_t count, void *stream);
cn_status cn_shard_factorize(cn_plan *plan, cn_exchange_fn exchange, void *ctx, void *stream);
cn_status cn_shard_run(cn_plan *plan, void *psi, int64_t nsteps, cn_exchange_fn exchange, void *ctx, void *stream);

/*
 * A stepper that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  No plan: what a plan keeps in device memory it allocated -- gamma and the
 * inverse pivots of the downward elimination of the whole system -- is recomputed by every
 * call into a fixed static device array of the library, CN_STATIC_NMAX rows = 96 KB, which every GPU that loads the
 * library holds until the process exits.  The call makes no cudaMalloc, cudaFree or allocating library call.
 *   cn_step_static : nsteps Crank-Nicolson steps (Eq. 2-3) of ONE system of 2 <= N <= CN_STATIC_NMAX
 *                    points, in place.  V: N doubles, psi: N complex128 (16-byte aligned), both DEVICE pointers owned by
 *                    the caller, on the current device.  Enqueues three launches on `stream` (factor into the scratch,
 *                    the on-chip stepper of cn_step, a check); does not synchronise.  Results are those of
 *                    cn_plan_create(N, .) / cn_factorize / cn_step on its default (on-chip) path, to the last bit.
 *   Errors: CN_ETOOLARGE when N > CN_STATIC_NMAX (use a plan); CN_EINVAL for the other bad arguments of
 *           cn_plan_create / cn_step or a misaligned pointer; CN_ECUDA when a CUDA call fails.  A zero or non-finite
 *           pivot (non-finite V) cannot be returned by an asynchronous call: psi is then filled with NaN.
 *   Sharing: ALL calls on a device share the one array, and it keeps the last call's contents (every call rewrites
 *           what it reads and clears its flag).  Calls that overlap on the GPU -- different streams, or different host
 *           threads without an order between their streams -- RACE on it: the caller serialises them.  The factor
 *           side is a serial recurrence over N rows (about 0.1 ms at N = 4096): amortise it over nsteps.
 */
#define CN_STATIC_NMAX 4096
cn_status cn_step_static(int64_t N, double dx, double dt, const double *V, void *psi, int64_t nsteps, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* CN_NSHAPE_H */
