/*
 * lp.h -- C ABI of the B200-native Lagrangian-Particle (LP) hot path.
 *
 * The library advances N_p macro-particles through one time step of the LP module of
 * arxiv/paper_2602_23434 (/root/reference/PAPER.md, cited below as PAPER.md:<line>):
 *   1. sample the cell-centred fluid state (v, B, rho) at x_LP      PAPER.md:81-85 (Eq. 1 and text)
 *   2. advance x_LP with a two-stage predictor-corrector            PAPER.md:83, 218-227 (Table 1:
 *                                                                    Particles_RK#1/#2, _Boundary)
 *   3. update each particle's spectrum chi(eps) on N_b log bins by   PAPER.md:87-108 (Eq. 2-6),
 *      a conservative upwind, CFL-substepped solve of Eq. 6          218-231 (Particles_Spectra)
 * Every step runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 * The precise arithmetic (and the readings taken where the paper is silent) is in DESIGN.md.
 *
 * Conventions
 *  - All arithmetic is IEEE fp64.  Cell keys are uint32, ids uint64, substep counts int32.
 *  - Grid arrays are cell-centred, [nz][ny][nx] with i (x) fastest.
 *  - chi is particle-major: chi[p*nbins + i], i = 0..nbins-1 (as chi_ of Listing 3).
 *  - Unless a parameter says "host", every pointer is a DEVICE pointer on `device`, BORROWED:
 *    the caller owns it and keeps it alive until the stream it was used on is synchronised.
 *    The library allocates only small tables itself; bulk scratch is the caller's workspace.
 *  - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls only enqueue
 *    work on it and return; lp_get_diag and the *_host call are the ones that synchronise.
 *  - A context is not thread-safe: one host thread at a time per context (several contexts, on one or
 *    several devices, may be used concurrently from different threads: a context shares no mutable state
 *    with another).
 *  - Every function returns an lp_status; nothing aborts, throws or prints.
 *    lp_last_error gives a human-readable detail for the last failure on that context.
 */
#ifndef LP_H
#define LP_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define LP_API __attribute__((visibility("default")))
#else
#define LP_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    LP_OK              =  0,
    LP_ERR_INVALID_ARG = -1,   /* NULL where not allowed, bad size, bad struct_size          */
    LP_ERR_STATE       = -2,   /* call order: fields/particles/workspace not set, stage order */
    LP_ERR_CUDA        = -3,   /* a CUDA runtime/driver call failed (see lp_last_error)      */
    LP_ERR_UNSUPPORTED = -4,   /* nbins not in {16,32,64,128,256,512}; grid > 2^31 cells      */
    LP_ERR_WORKSPACE   = -5    /* workspace missing, misaligned or smaller than required      */
} lp_status;

typedef struct lp_ctx lp_ctx;  /* opaque; owned by the library, released by lp_destroy */

typedef struct {
    uint32_t struct_size;      /* = sizeof(lp_config), checked                                   */
    int32_t  nx, ny, nz;       /* cells per axis                                                  */
    double   xlo[3], xhi[3];   /* domain; cell (i,j,k) covers xlo + [i,i+1)*dx ...                */
    int32_t  periodic[3];      /* 1 periodic, 0 zero-gradient (clamped stencil)     */
    int64_t  np;               /* particles                                                       */
    int32_t  nbins;            /* N_b in {16,32,64,128,256,512}; log-spaced edges on [e_min,e_max] */
    double   e_min, e_max;
    double   kappa, u_rad;     /* c_r = kappa*(|B|^2/2 + u_rad)   (Eq. 4)         */
    double   cfl_e;            /* energy-space CFL number C_E, 0 < C_E <= 1                       */
    int32_t  max_substeps;     /* cap on n_sub (>= 1); capped particles are counted in lp_diag    */
    int32_t  sort_every;       /* lp_step re-sorts by cell every this many steps; 0 = never       */
    int32_t  device;           /* CUDA device ordinal                                             */
} lp_config;

typedef struct {
    int64_t np;
    int64_t sum_substeps;      /* sum over particles of n_sub of the last spectral update        */
    int32_t max_substeps;      /* max over particles                                              */
    int64_t n_capped;          /* particles whose n_sub hit config.max_substeps                   */
    int64_t n_outside;         /* particles outside the box on a non-periodic axis                */
    double  number;            /* sum_p sum_i chi_i dE_i now                                      */
    double  lost;              /* sum_p number that left through the energy ends, last update     */
    int64_t steps;             /* lp_step calls so far                                            */
    int64_t sorts;             /* sorts so far                                                    */
} lp_diag;

/* Create / destroy.  lp_create validates the config, selects the device, builds the bin table
 * (E_k = e_min*(e_max/e_min)^(k/N_b)) and uploads it.  *out is NULL on error
 * except that a context is still returned for LP_ERR_CUDA so lp_last_error can be read. */
LP_API lp_status lp_create(const lp_config *cfg, lp_ctx **out);
LP_API lp_status lp_destroy(lp_ctx *ctx);
LP_API const char *lp_last_error(const lp_ctx *ctx);     /* host string, valid until the next call */

/* Bytes of caller-supplied device scratch the context needs (repacked grid records, stage
 * buffers k1, x_star, rho_old, coefficients, sort buffers and the alternate chi rows used by the
 * re-sort).  Bind a 256-byte aligned device buffer of at least that size before any other call. */
LP_API lp_status lp_workspace_bytes(const lp_config *cfg, size_t *out_bytes /*host*/);
LP_API lp_status lp_bind_workspace(lp_ctx *ctx, void *workspace, size_t bytes);

/* Particle state, advanced in place: positions x,y,z [np], ids [np] (unique), chi [np][nbins]
 * (16-byte aligned).  What a particle carries: PAPER.md:598-613 (Listing 3).  Enqueues nothing: the width
 * of the ids (the number of radix passes a sort makes over them) is measured by the first sort that
 * follows a bind, a raised count or a host copy of the ids -- on that sort's stream, which it synchronises
 * once for it. */
LP_API lp_status lp_bind_particles(lp_ctx *ctx, double *x, double *y, double *z, uint64_t *id, double *chi);

/* Optional per-particle outputs of the spectral update: n_sub [np] (negative = capped) and
 * the number lost through the energy boundaries in that update [np].  NULL = not written. */
LP_API lp_status lp_bind_diag(lp_ctx *ctx, int32_t *nsub, double *lost);

/* Stage the fluid state (7 cell-centred arrays [nz][ny][nx]) for the gathers: repacked into
 * interleaved per-cell records inside the workspace; the inputs are not referenced afterwards.
 * May be called between lp_push stages (time-dependent fields). */
LP_API lp_status lp_set_fields(lp_ctx *ctx, const double *vx, const double *vy, const double *vz,
                        const double *bx, const double *by, const double *bz, const double *rho,
                        void *stream);

/* Trilinear sampling at the current positions: out7 [7][np] in the order
 * vx,vy,vz,bx,by,bz,rho (or NULL) and the containing-cell key (k*ny+j)*nx+i [np] (or NULL). */
LP_API lp_status lp_interpolate(lp_ctx *ctx, double *out7, uint32_t *cell_key, void *stream);

/* The same sampling through shared-memory tiles (the option BASELINE.json's north_star names beside the direct
 * gather): blocks of 64 consecutive particles load the bounding box of their stencils once and gather from
 * shared memory; blocks whose box does not fit (set not sorted by cell, or drifted apart) gather directly.
 * Bit-identical to lp_interpolate.  Kept as a measured alternative: profiles/r02_gather_tile.md has the numbers
 * that decided for the direct gather in the fused kernels. */
LP_API lp_status lp_interpolate_tiled(lp_ctx *ctx, double *out7, void *stream);

/* Reorder all particle arrays ascending by (cell key, id); bound arrays hold the result.  Asynchronous,
 * except for the first sort after the ids may have changed (see lp_bind_particles). */
LP_API lp_status lp_sort(lp_ctx *ctx, void *stream);

/* stage 0: k1 = v(x^n), rho_old = rho(x^n), x* = x^n + dt k1 (kept in the workspace).
 * stage 1: x^{n+1} = x^n + dt/2 (k1 + v(x*)) with the fields set now; periodic wrap.
 * stage 1 without a preceding stage 0 returns LP_ERR_STATE. */
LP_API lp_status lp_push(lp_ctx *ctx, double dt, int stage, void *stream);

/* Third-order pusher, an alternative to lp_push (the paper does not name the
 * variant: the three-stage Shu-Osher scheme is taken), one call per stage, fields may be re-set in between:
 *   stage 0: x0 = x^n (kept in the workspace), rho_old = rho(x^n), x <- x0 + dt v(x0)
 *   stage 1: x <- (3/4) x0 + (1/4) (x + dt v(x))
 *   stage 2: x <- (x0 + 2 (x + dt v(x))) / 3, periodic wrap / outside flag.
 * The bound x, y, z hold the stage positions in between.  Stages out of order return LP_ERR_STATE.
 * lp_spectral_update may follow stage 2 (it uses the rho_old of stage 0). */
LP_API lp_status lp_push_rk3(lp_ctx *ctx, double dt, int stage, void *stream);

/* Spectral update at the current positions with the current fields:
 * coefficients, CFL substep count, n_sub donor-cell upwind substeps of Eq. 6 per particle.
 * Consumes rho_old of the last stage 0 and needs the push finished (lp_push stage 1 or lp_push_rk3 stage 2
 * since that stage 0), so that the bound positions are x^{n+1}; LP_ERR_STATE otherwise. */
LP_API lp_status lp_spectral_update(lp_ctx *ctx, double dt, void *stream);

/* Shock crossing (Eq. 7-8; not part of lp_step): every particle p with r[p] > 1 gets
 *   chi_out,i = C ec_i^(2-q) [ sum_{j<i} chi_j ec_j^(q-3) dE_j + chi_i ec_i^(q-3) dE_i / 2 ],
 *   q = 3 r[p] / (r[p] - 1) + q_r,   ec_i = sqrt(E_i E_{i+1}),
 * with C fixed by number conservation (sum_i chi_i dE_i unchanged); rows with r[p] <= 1 or NaN, and rows
 * whose unnormalised result sums to zero, are left untouched.  r: device array [np] of compression ratios
 * (the paper defines no shock finder: the caller supplies them); q_r: the relativistic correction q_R of
 * Eq. 8 as a scalar, 0 for non-relativistic shocks.  Acts on the bound chi in place. */
LP_API lp_status lp_shock_update(lp_ctx *ctx, const double *r, double q_r, void *stream);

/* Deletion with hole filling (not part of lp_step): the particles with flag[p] != 0 are
 * removed, the survivors stored at p >= N_p - N_del move into the flagged slots below N_p - N_del (k-th hole
 * in ascending order <- k-th such survivor in ascending order), with all their parameters (x, y, z, id, chi
 * row); the context then holds *np_new = N_p - N_del particles in the first *np_new entries of the bound
 * arrays (the arrays and the workspace keep their size).  flag: device int32 [np], or NULL to delete the
 * particles the last lp_push(stage 1) / lp_step marked outside the box on a non-periodic axis (outflow,
 * Particles_Boundary); LP_ERR_STATE if there is no such marking.  Synchronises `stream`. */
LP_API lp_status lp_compact(lp_ctx *ctx, const int32_t *flag, int64_t *np_new /*host*/, void *stream);

/* Particle count within the capacity given to lp_create (config.np at creation): particles are injected by
 * writing them behind the current ones in the bound arrays and raising the count; lp_compact lowers it.
 * The paper sizes its containers in chunks of L = 2^e particles so that growth rarely reallocates
 * (Listing 1: N_c = (N >> e) + (N % L == 0 ? 0 : 1); e = 18 in Listing 3):
 * lp_chunked_capacity returns N_c * L, the capacity to create the context and the arrays with.
 * Per-particle results of earlier calls (n_sub, lost, push stages) are invalidated by lp_set_count. */
LP_API lp_status lp_chunked_capacity(int64_t n, int32_t e, int64_t *capacity /*host*/);
LP_API lp_status lp_set_count(lp_ctx *ctx, int64_t np_new);

/* Exchange of the particles that crossed a rank interface (not part of lp_step), for a
 * domain decomposed into boxes, one direction (axis 0, 1, 2) at a time with a left and a right neighbour per
 * direction.  The library does the steps that touch particle data; sizing buffers and moving them between
 * ranks (NCCL send/recv, a peer copy over NVLink, or a plain pointer between contexts on one GPU) is the
 * caller's.  This rank owns [lo, hi) along `axis`; the global box and its periodicity are the context's.
 *   lp_migrate_count   steps 1: destination of every particle -- 0 stays, 1 left, 2 right; a particle outside
 *                      [lo, hi) goes to the neighbour through whose face the shorter way leads, the other way
 *                      being the one around a periodic axis (positions were wrapped into the global box by the
 *                      pusher) -- and the two totals.  Synchronises `stream` (the totals size the buffers).
 *   lp_migrate_pack    step 4: the leavers' x, y, z, id and chi row, in ascending index order, into the send
 *                      buffers.  A buffer for n particles is n * lp_migrate_record_bytes bytes, 16-byte
 *                      aligned, laid out as arrays  x[n] | y[n] | z[n] | id[n] | chi[n][nbins]  (and, with a
 *                      bound energy grid, | eng[n][nbins+1]);
 *                      NULL is allowed for a buffer whose total is 0.
 *   lp_migrate_unpack  step 8: the n_from_left particles of from_left, then the n_from_right of from_right
 *                      (same layout, written by the neighbours' lp_migrate_pack): the k-th arrival goes into
 *                      the k-th hole (ascending index), arrivals beyond the holes behind the last particle,
 *                      holes beyond the arrivals are closed as lp_compact closes them.  *np_new = the new
 *                      count; LP_ERR_WORKSPACE if it exceeds the capacity (grow with lp_rebind first: the
 *                      paper's step 6).  Synchronises `stream` only when holes are left to compact.
 * Order: count -> pack -> unpack, nothing that moves particles in between (LP_ERR_STATE otherwise); particles
 * outside the global box on a non-periodic axis must have been deleted (lp_compact) before. */
LP_API lp_status lp_migrate_record_bytes(const lp_ctx *ctx, size_t *bytes /*host*/);
LP_API lp_status lp_migrate_count(lp_ctx *ctx, int axis, double lo, double hi, int64_t *n_left /*host*/,
                                  int64_t *n_right /*host*/, void *stream);
LP_API lp_status lp_migrate_pack(lp_ctx *ctx, void *buf_left, void *buf_right, void *stream);
LP_API lp_status lp_migrate_unpack(lp_ctx *ctx, const void *from_left, int64_t n_from_left, const void *from_right,
                                   int64_t n_from_right, int64_t *np_new /*host*/, void *stream);

/* Growing and shrinking the particle storage in whole chunks (Listing 1; Reserve() / Shrink()
 * of Listing 2).  The paper's BlockedContainer appends or frees chunks of L = 2^e elements; here
 * every array is one flat caller-owned allocation (the kernels need contiguous rows), so a change of capacity is:
 * the caller allocates particle arrays and a workspace for the new capacity -- lp_chunked_capacity(N, e) particles,
 * lp_workspace_bytes_for bytes -- and lp_rebind moves the context onto them.  On `stream` it copies the current
 * particles (x, y, z, id, chi rows, from wherever they live: the bound arrays or their ping-pong twins) and the
 * staged cell records (the fields stay set); the old arrays and workspace may be released once the stream has
 * passed the call.  capacity >= the current count (Shrink() only ever drops trailing free chunks).  Afterwards the
 * state is in the new bound arrays, the lp_bind_diag outputs are unbound (they were sized for the old capacity),
 * per-particle results of earlier calls are invalid, and an exchange between lp_migrate_pack and
 * lp_migrate_unpack survives (the paper's step 6: "resize the particle container to accommodate the new
 * particles"). */
LP_API lp_status lp_capacity(const lp_ctx *ctx, int64_t *capacity /*host*/);
LP_API lp_status lp_workspace_bytes_for(const lp_ctx *ctx, int64_t capacity, size_t *out_bytes /*host*/);
LP_API lp_status lp_rebind(lp_ctx *ctx, int64_t capacity, void *workspace, size_t bytes, double *x, double *y,
                           double *z, uint64_t *id, double *chi, void *stream);

/* Per-particle moving energy grid (the eng_ array of Listing 3; the method is deferred to
 * [19] by PAPER.md:122 -- readings E1-E4 of DESIGN.md): an alternative to the fixed log-spaced bins.  Every particle
 * carries its own nbins + 1 bin edges eng[p*(nbins+1) + k]; over a step they follow the characteristics of Eq. 6
 * (PAPER.md:107), eps' = eps e^{-s} / (1 + beta eps) with s = a dtau, beta = c_r dtau (1 - e^{-s})/s, and every bin
 * keeps its number, chi_i' = chi_i dE_i / dE_i': exact for frozen coefficients, no CFL limit, no substeps, no
 * numerical diffusion, nothing lost through the ends.
 *   lp_bind_energy_grid  eng [capacity][nbins+1] (device, caller-owned, updated in place) switches the context to the
 *                        moving grid: lp_spectral_update and lp_step use it (lp_step stays one fused kernel), n_sub reads 1, lp_get_diag's number uses the particle's own widths.  eng_scratch: a
 *                        second array of the same size through which a sort moves the rows (NULL: sorts return
 *                        LP_ERR_STATE).  eng = NULL switches back to the fixed bins.
 *   lp_init_energy_grid  rows [first, first + count) <- the fixed table's edges (the grid every particle starts on).
 *   lp_rebind_energy_grid  after lp_rebind changed the capacity: new arrays of capacity rows; the current particles'
 *                        rows are copied over on `stream`.  Until then every call that uses the grid returns
 *                        LP_ERR_STATE when the capacity has outgrown the bound arrays.
 * The grid rows travel with their particles: lp_sort, lp_compact and lp_migrate_pack / _unpack move them (an
 * exchange buffer then carries eng[n][nbins+1] behind chi[n][nbins]; lp_migrate_record_bytes says so).
 * lp_shock_update takes every row's centres and widths from its own grid.  lp_step_host (no host grid argument)
 * returns LP_ERR_UNSUPPORTED while a grid is bound. */
LP_API lp_status lp_bind_energy_grid(lp_ctx *ctx, double *eng, double *eng_scratch);
LP_API lp_status lp_init_energy_grid(lp_ctx *ctx, int64_t first, int64_t count, void *stream);
LP_API lp_status lp_rebind_energy_grid(lp_ctx *ctx, double *eng, double *eng_scratch, void *stream);
/* Where the grid lives now: with ping-pong buffers (lp_set_pingpong) a re-sort writes the rows in the new order into
 * eng_scratch and the two arrays change roles instead of being copied (in lp_step the permutation is then folded
 * into the fused kernel, as for the fixed bins); without ping-pong it is always the array bound as eng. */
LP_API lp_status lp_current_energy_grid(const lp_ctx *ctx, double **eng);

/* One whole step with frozen fields: [sort every sort_every steps] -> push 0 -> push 1 ->
 * spectral update (order of Table 1, without the fluid stages). */
LP_API lp_status lp_step(lp_ctx *ctx, double dt, void *stream);

/* Ping-pong particle buffers (off by default).  A re-sort cannot run in place: every array is read through
 * the permutation and written in the new order.  By default the library permutes into the workspace and the
 * bound arrays hold the state again when the call returns (one extra pass over every row per sort).  With
 * ping-pong enabled the workspace twins of the bound arrays (same sizes, inside the caller's workspace)
 * become a second home of the state: lp_sort permutes from the current home into the other one, and on a
 * sort step lp_step folds the permutation into the fused kernel (it reads rows, positions and ids through
 * the permutation and writes the other home), so a re-sort costs the permutation itself and nothing else.
 * The price: after a sort the state may live in the workspace -- lp_current_particles says where, and every
 * call of this library follows it (injection through lp_set_count writes behind the current particles of
 * the CURRENT arrays).  Disabling copies the state back into the bound arrays on `stream` if it is not there. */
LP_API lp_status lp_set_pingpong(lp_ctx *ctx, int enable, void *stream);
/* Device pointers of the arrays that hold the particle state now (any may be NULL): the bound arrays, or with
 * ping-pong their workspace twins.  Valid until the next sort. */
LP_API lp_status lp_current_particles(const lp_ctx *ctx, double **x, double **y, double **z, uint64_t **id,
                                      double **chi);

/* The same step on HOST buffers (pinned for overlap; pageable works, serialised): copies x,y,z,id,chi
 * to the bound device arrays, runs lp_step, copies x,y,z,chi (and id on re-sort steps) back and
 * synchronises the stream.  With >= 65536 particles and no re-sort due, the step runs in 16 particle
 * batches so that copy-in, kernels and copy-out overlap (particles are independent); the result is the
 * same as lp_step's.  Work is ordered after what was enqueued on `stream` before the call. */
LP_API lp_status lp_step_host(lp_ctx *ctx, double dt, double *hx, double *hy, double *hz,
                       uint64_t *hid, double *hchi, void *stream);

/* Aggregate diagnostics; synchronises `stream` (the one argument beyond SURVEY.md 8(b)'s signature: the reduction
 * kernels must be ordered behind the caller's work). */
LP_API lp_status lp_get_diag(lp_ctx *ctx, lp_diag *out /*host*/, void *stream);

/* What a hit cap means.  A particle whose CFL-limited substep count exceeds config.max_substeps takes max_substeps
 * substeps instead (n_sub reads negative, lp_diag.n_capped counts it): each of them is longer than the CFL bound
 * allows, the explicit scheme is unstable there and the row is no longer a solution of Eq. 6 to any
 * stated accuracy.  By default that is only reported.  With error_on_cap != 0, lp_get_diag fills *out as usual and
 * returns LP_ERR_UNSUPPORTED when the last spectral update capped any particle, so that a driver loop that checks
 * its diagnostics never carries such rows on unnoticed.  (Kernels run asynchronously: the diagnostics call is the
 * first point where the host can know.) */
LP_API lp_status lp_set_cap_policy(lp_ctx *ctx, int error_on_cap);

/* The particle number  sum_p sum_i chi[p][i] * widths[i]  (the `number` of lp_diag: what Eq. 2 / Eq. 6 conserve,
 * PAPER.md:87, 107) for callers that cannot allocate device memory -- and this call allocates none: no cudaMalloc,
 * no cudaFree, no workspace, no context (lp_create uploads a table with cudaMalloc, and lp_get_diag wants the
 * multi-GB workspace of the whole step).  Meant for a conservation monitor inside a host code that gave all device
 * memory to its own arena at start-up, for a diagnostic fired while other streams run (cudaMalloc / cudaFree
 * stall the whole device), and for code that sits where the allocating runtime calls are forbidden.
 *   device   CUDA ordinal the pointers live on (made current for the call, the previous one restored)
 *   chi      device [np][nbins] doubles, particle-major, 8-byte aligned, read only
 *   widths   device [nbins] doubles: the dE_i of lp_get_bins, copied to the device by the caller
 *   number   device [1] double, written on `stream`; the caller reads it after synchronising (0 for np = 0)
 *   err      host buffer for a one-line reason when the status is not LP_OK (there is no context to hold
 *            one), or NULL; err_len its size
 * The scratch -- one partial sum per 2048 rows -- is a 64 KiB array compiled into the library, resident on every GPU
 * that loads liblp_b200.so for the life of the process.  Hence the limits: np <= LP_NUMBER_STATIC_MAX_NP rows
 * (2^24: workload 4 of BASELINE.json; sum larger sets slice by slice) and nbins <= LP_NUMBER_STATIC_MAX_NBINS;
 * beyond them LP_ERR_UNSUPPORTED with the reason in err, nothing launched.
 * The first call on a device looks the array's address up (cudaGetSymbolAddress, which may make the driver load
 * the library's code on that device): make that first call during set-up, before any stream capture and before
 * the phase in which the device must not be disturbed.  Later calls only enqueue two kernels on `stream`.
 * All calls on one device share the array: two calls whose kernels can overlap on the GPU (different streams, no
 * event between them) race on it and both results are garbage; calls on one stream, or ordered by events, are
 * safe.  Nothing in the array has to start at zero and nothing of a previous call is read.  The sum order
 * depends on (np, nbins) only, so the result is bitwise reproducible across GPUs and runs; it agrees with
 * lp_get_diag's number to rounding, not bit for bit. */
#define LP_NUMBER_STATIC_MAX_NP    ((int64_t)1 << 24)
#define LP_NUMBER_STATIC_MAX_NBINS 512
LP_API lp_status lp_number_static(int device, const double *chi, const double *widths, int32_t nbins, int64_t np,
                                  double *number, void *stream, char *err /*host*/, size_t err_len);

/* Number of kernel launches the library has enqueued so far on this context. */
LP_API lp_status lp_launch_count(const lp_ctx *ctx, int64_t *out /*host*/);

/* Optional device timing of the spectral-update kernel (the dominant kernel): after
 * lp_timing_enable(ctx, n) the next n spectral launches are bracketed by CUDA events on the stream
 * they are launched on; lp_timing_read waits for them, returns the summed kernel time in ms and the
 * number of launches recorded, and re-arms the records.  n = 0 disables. */
LP_API lp_status lp_timing_enable(lp_ctx *ctx, int max_records);
LP_API lp_status lp_timing_read(lp_ctx *ctx, double *spectral_ms_sum /*host*/, int32_t *n_records /*host*/);

/* Copy the library's bin table to host arrays: edges [nbins+1], widths [nbins] (either may be NULL). */
LP_API lp_status lp_get_bins(const lp_ctx *ctx, double *edges /*host*/, double *widths /*host*/);

/* The bins the CFL reduction (step a8) evaluates: on a fixed bin table the maximum outflow rate
 * over all bins is attained, for every (a, c_r >= 0), at a vertex of the convex hull of the bins'
 * coefficient points, found once at lp_create.  bins [*n] on return (capacity >= 24); *n = -1 means
 * every bin is scanned.  Needs no GPU (valid even when lp_create returned LP_ERR_CUDA). */
LP_API lp_status lp_get_cfl_bins(const lp_ctx *ctx, int32_t *bins /*host*/, int32_t *n /*host*/);

#ifdef __cplusplus
}
#endif
#endif /* LP_H */
