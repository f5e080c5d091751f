/* lqcd.h -- C ABI of the B200 staggered-fermion hot path (even/odd Dslash + multi-shift CG).
 *
 * Source of the operations: arxiv/paper_1801_01473, "Portable multi-node LQCD Monte Carlo simulations
 * using OpenACC".  The library implements, for ONE GPU (sm_100a), in double precision (and, through
 * the *_f32 entry points, in single precision: the paper keeps its fields as "double (or float) C99 complex
 * numbers", and runs the MD evolution in single precision):
 *
 *   D_oe, D_eo   the off-diagonal even/odd blocks of the staggered Dirac matrix (the
 *                hopping term between x and x+mu is proportional to U_mu(x); D_oe^dagger = -D_eo), with
 *                the U(1) factors that carry the staggered phases and the antiperiodic time boundary
 *                 computed in registers:
 *                  (D psi)(x) = 1/2 sum_mu [ s_mu(x) U_mu(x) psi(x+mu) - s_mu(x-mu) U_mu(x-mu)^+ psi(x-mu) ]
 *                  s_mu(x) = eta_mu(x) bc_mu(x), eta = (1, (-1)^x, (-1)^(x+y), (-1)^(x+y+z)),
 *                  bc_t(x) = -1 for x_t = Lt-1 when ANTIPERIODIC_T is on, +1 otherwise;
 *   Eq. 2        (m^2 - D_eo D_oe + sigma_i) x_i = b, i = 1..r, solved for all shifts at once by the
 *                shifted ("multimass") conjugate gradient;
 *   link compression  only the first two rows of each SU(3) link are stored and read; the third is
 *                recomputed as r2 = conj(r0 x r1)  [option LQCD_OPT_RECON = 12].
 *
 * Conventions
 *   Sites: lex = x + Lx*(y + Ly*(z + Lz*t)); parity = (x+y+z+t)&1, even = 0.  All extents even, >= 2.
 *   V = Lx*Ly*Lz*Lt, Vh = V/2.  A complex number is two consecutive doubles (re, im).
 *
 *   PARITY VECTOR ("vec3_soa") -- the layout of every in/out/b/x argument:
 *       v[(c*Vh + k)*2 + {0,1}],  c = colour 0..2,  k = lex>>1 of a site of the stated parity.
 *       3*Vh complex doubles = 48*Vh bytes (3 double complex per even site).
 *   CANONICAL GAUGE FIELD -- the argument of lqcd_set_gauge:
 *       links[(((mu*V + lex)*3 + row)*3 + col)*2 + {0,1}],  mu = 0..3 = x,y,z,t;
 *       U_mu(lex) is the link that leaves site lex in direction +mu.  4*V*18 doubles.
 *   SITE FIELD (lqcd_pack_vector / lqcd_unpack_vector only): f[((lex*3) + c)*2 + {0,1}], V*3 complex.
 *
 * Pointers
 *   Unless a parameter is marked HOST, every data pointer is a DEVICE pointer, 16-byte aligned, owned by
 *   the caller; the library reads/writes it on the context's stream and never frees it.  The *_host
 *   entry points take HOST pointers (pinned memory makes the copies asynchronous and faster) and perform
 *   the host<->device copies themselves on the context's stream.
 *   in/out (and b/x[i], x[i]/x[j]) must not alias.
 *
 * Execution
 *   All work is enqueued on the stream set with lqcd_set_stream (default: the legacy default stream).
 *   lqcd_doe / lqcd_deo / lqcd_mdagm / lqcd_pack_vector / lqcd_unpack_vector return after enqueueing.
 *   lqcd_set_gauge and lqcd_mshift_cg (and all *_host calls) return after their work has completed.
 *   A context is not thread-safe; use one per host thread.
 *
 * Errors
 *   Every int-returning call returns LQCD_OK (0) or a negative code; nothing is printed, thrown or
 *   aborted.  lqcd_last_error(ctx) gives a short text for the last failure on that context
 *   (lqcd_last_error(NULL): the last failed lqcd_create).
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx;

/* status codes */
#define LQCD_OK           0
#define LQCD_EINVAL      -1   /* NULL pointer, odd or < 2 extent, nshift < 1, shift < 0, tol <= 0, bad key/value */
#define LQCD_ENOGAUGE    -2   /* operator or solver called before lqcd_set_gauge */
#define LQCD_ENOMEM      -3   /* device allocation failed or caller workspace too small */
#define LQCD_ECUDA       -4   /* a CUDA runtime call or kernel failed (text in lqcd_last_error) */
#define LQCD_ENOCONV     -5   /* MAX_ITER reached; x[] holds the last iterate */
#define LQCD_EBREAKDOWN  -6   /* <p,Ap> <= 0 or non-finite (cannot happen for SU(3) links) */
#define LQCD_ENOTSU3     -7   /* RECON=12 and some link has max|r2 - conj(r0 x r1)| > 1e-12 */
#define LQCD_ECOMM       -8   /* slab context: no transport set, or the transport failed */

/* option keys for lqcd_set_option / lqcd_get_option */
#define LQCD_OPT_MASS            0  /* m of Eq. 2; default 0                               */
#define LQCD_OPT_ANTIPERIODIC_T  1  /* 1 (default): antiperiodic in t; 0: periodic         */
#define LQCD_OPT_RECON           2  /* 18 (default): full links; 12: two-row compression.
                                       Takes effect at the next lqcd_set_gauge.                           */
#define LQCD_OPT_MAX_ITER        3  /* iteration cap of lqcd_mshift_cg; default 100000                    */
#define LQCD_OPT_CHECK_EVERY     4  /* the host looks at the device-side stop flag every this many
                                       iterations; default 0 = chosen from the lattice size                */
#define LQCD_OPT_USE_GRAPH       5  /* 1 (default): replay the CG iteration as a CUDA graph; 0: plain launches */
#define LQCD_OPT_LINK_PRECISIONS 6  /* which copies of the links the next lqcd_set_gauge stores: LQCD_PREC_F64
                                       (default; serves the double entry points), LQCD_PREC_F32 (serves the
                                       *_f32 entry points), or both OR-ed together                         */
#define LQCD_OPT_SHIFT_BLOCK     7  /* m in [1,32]; 0 (default) = chosen by the library (32; 16 on lattices small enough
                                       to live in L2).  The x_i, p_i of the shifted systems (and x_0 of the base
                                       system) are updated once per block of m iterations from the m residuals of the
                                       block (kept in m vectors) instead of once per iteration; same recurrences, same
                                       iteration counts, x_i equal up to rounding.  m = 1: every iteration.
                                       CHECK_EVERY is rounded up to a multiple of m.  lqcd_get_option returns the
                                       value in force.                                                         */
#define LQCD_OPT_PERSISTENT      8  /* -1 (default): lattices whose stored links and solver vectors stay in L2 (links
                                       up to 32 MB) and that give most SMs a block of one site per thread (e.g. 16^4
                                       with two-row links) are solved by ONE cooperative kernel that runs all
                                       iterations with grid-wide barriers between the sweeps (no launch gaps, no
                                       host polling); all others by two operator launches per iteration (+ two
                                       one-block kernels, which small lattices fold into the launches) replayed as
                                       a CUDA graph.
                                       0: never, 1: always the persistent kernel -- a solve it cannot run (slab
                                       context, LQCD_OPT_SHIFT_BLOCK above 16, a device without cooperative launches,
                                       a refused launch) then returns LQCD_EINVAL / LQCD_ECUDA instead of silently
                                       taking the other driver.  With -1 a refused cooperative launch (fewer blocks
                                       resident than expected: another context or MPS client on the GPU) falls back
                                       to the launches.  LQCD_STAT_SOLVER_PATH tells which driver ran.
                                       Same arithmetic per site; the scalar products are added over a different grid,
                                       so results agree to rounding.  Whole-lattice contexts only.            */
#define LQCD_OPT_COMM_TIMEOUT    9  /* seconds (default 120; 0 = for ever) a solve on a slab context over the
                                       peer-memory transport waits for a batch of iterations before it concludes
                                       that a peer rank is gone and returns LQCD_ECOMM (see lqcd_comm_abort)    */
#define LQCD_PREC_F64 1
#define LQCD_PREC_F32 2

/* statistic keys for lqcd_get_stat (about the last lqcd_mshift_cg on this context) */
#define LQCD_STAT_ITERS          0  /* number of iterations performed                                     */
#define LQCD_STAT_REL_RES        1  /* sqrt(|r|^2/|b|^2) of the base recurrence residual at the stop       */
#define LQCD_STAT_FREEZE_ITER    2  /* idx = shift index: iteration after which x[idx] was no longer updated */
#define LQCD_STAT_BASE_SHIFT     3  /* index of the shift used as base system (the smallest)              */
#define LQCD_STAT_GPU_LAUNCHES   4  /* kernels launched by this context since creation                    */
#define LQCD_STAT_SOLVE_MS       5  /* device time of the last solve between CUDA events, milliseconds     */
#define LQCD_STAT_RELIABLE_UPDATES 6 /* lqcd_mshift_cg_mixed: double-precision residual replacements performed */
#define LQCD_STAT_GRAPH_REPLAYS  7  /* CUDA-graph replays of the last solve (0: plain launches or the persistent kernel) */
#define LQCD_STAT_SOLVER_PATH    8  /* which driver ran the iterations of the last lqcd_mshift_cg / lqcd_rational_apply:
                                       0 = plain launches, 1 = CUDA-graph replays, 2 = the persistent kernel        */

/* Create a context for an Lx*Ly*Lz*Lt lattice on the current CUDA device.  NULL on error
 * (extent odd or < 2, volume too large, no device). */
lqcd_ctx* lqcd_create(int Lx, int Ly, int Lz, int Lt);
void      lqcd_destroy(lqcd_ctx* ctx);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
int lqcd_set_stream(lqcd_ctx* ctx, void* cuda_stream);
int lqcd_set_option(lqcd_ctx* ctx, int key, double value);
int lqcd_get_option(const lqcd_ctx* ctx, int key, double* value /*HOST*/);

/* Device memory.  By default the library allocates what it needs with cudaMalloc.  Alternatively the
 * caller provides one arena of at least lqcd_workspace_bytes(ctx, nshift) bytes (256-byte aligned) that
 * then holds the stored links and all solver temporaries for up to nshift shifts; it must stay valid
 * until lqcd_destroy or the next lqcd_set_workspace.  Must be called before lqcd_set_gauge.
 * The size depends on LQCD_OPT_SHIFT_BLOCK and LQCD_OPT_LINK_PRECISIONS: set both BEFORE the query and do not
 * raise them afterwards (lqcd_mshift_cg_mixed needs both precisions).  The device staging copies of the *_host
 * entry points and of lqcd_mshift_cg_mixed (up to nshift + 2 vectors) are not part of the arena: the library
 * allocates them with cudaMalloc on first use. */
size_t lqcd_workspace_bytes(const lqcd_ctx* ctx, int nshift);
int    lqcd_set_workspace(lqcd_ctx* ctx, void* dev, size_t bytes);

/* Store the gauge field (step A1): canonical layout above -> per-parity structure of arrays, 18 or 12
 * reals per link according to LQCD_OPT_RECON.  The input is copied; it may be freed afterwards.
 * With RECON=12 returns LQCD_ENOTSU3 if some third row differs from conj(r0 x r1) by more than 1e-12. */
int lqcd_set_gauge(lqcd_ctx* ctx, const double* links);
int lqcd_set_gauge_host(lqcd_ctx* ctx, const double* links /*HOST*/);

/* General U(1) phase field: "we multiply the pseudofermion fields by u_mu(x) U_mu(x)", with
 * u_mu(x) = exp(i theta_mu(x)) carrying, besides the staggered phases and the boundary sign (which this
 * library computes from the coordinates), an imaginary chemical potential or a background electromagnetic
 * field.  With a field set, every operator and solver of this context uses
 *     (D psi)(x) = 1/2 sum_mu [ s_mu(x) u_mu(x) U_mu(x) psi(x+mu) - s_mu(x-mu) conj(u_mu(x-mu)) U_mu(x-mu)^+ psi(x-mu) ]
 * (D_oe^dagger = -D_eo still holds).  As in the paper, theta is what is stored (8 bytes per link in double,
 * 4 in single) and cos/sin are recomputed in the kernel: +64 bytes per site on 1584.
 *   theta : 4*V doubles, theta[mu*V + lex], radians; copied (into every precision named by
 *           LQCD_OPT_LINK_PRECISIONS at the time of the call).  NULL switches the field off (u = 1).
 * Returns after the copy has completed.  Independent of lqcd_set_gauge (either order). */
int lqcd_set_u1_phases(lqcd_ctx* ctx, const double* theta);
int lqcd_set_u1_phases_host(lqcd_ctx* ctx, const double* theta /*HOST*/);

/* out_odd = D_oe in_even;  out_even = D_eo in_odd.  Parity vectors. */
int lqcd_doe(lqcd_ctx* ctx, double* out_odd, const double* in_even);
int lqcd_deo(lqcd_ctx* ctx, double* out_even, const double* in_odd);
int lqcd_doe_host(lqcd_ctx* ctx, double* out_odd /*HOST*/, const double* in_even /*HOST*/);
int lqcd_deo_host(lqcd_ctx* ctx, double* out_even /*HOST*/, const double* in_odd /*HOST*/);

/* out_even = (m^2 + sigma) in_even - D_eo D_oe in_even: the operator of Eq. 2, the
 * paper's D_oe, D_eo, zaxpy sequence in two launches. */
int lqcd_mdagm(lqcd_ctx* ctx, double* out_even, const double* in_even, double sigma);

/* lqcd_mdagm for callers that are not in a position to allocate device memory.
 *
 * Who that is: code that runs inside an application which has handed all of the GPU's memory to its own pool (an RHMC
 * code that sized its fields for the whole 180 GB, a framework with a caching allocator), where a cudaMalloc from a
 * library fails or fragments the pool; and code on a path that must not stall, since cudaMalloc and cudaFree
 * synchronise the whole device and so stop every other stream of the process.  lqcd_mdagm needs one odd-parity
 * temporary, t = D_oe in (D_oe, D_eo, zaxpy), which it allocates on first use -- from the workspace of
 * lqcd_set_workspace if there is one, else with cudaMalloc -- together with the solver's small state.  This entry
 * point makes the same two launches, with the same kernels and therefore the same bits in out_even, but keeps t in a
 * buffer that is compiled into the library: it calls no cudaMalloc, cudaFree, cudaMallocHost or any other allocating
 * routine, at any call.  (The stored links still have to exist: do lqcd_create and lqcd_set_gauge at start-up, where
 * allocation is allowed, or give the context an arena with lqcd_set_workspace beforehand.)
 *
 * Limit: lattices of at most LQCD_STATIC_MAX_VH = 65536 sites per parity (16^4, 16^3 x 32, 8^3 x 256 ...); larger ones
 * get LQCD_EINVAL with the two numbers in lqcd_last_error.  Double precision, whole-lattice contexts (a slab context
 * gets LQCD_EINVAL).  The buffer is 3 MiB and is held by every GPU on which this library is used, from the moment its
 * code is loaded there until the process ends, also by programs that never call lqcd_mdagm_static.
 *
 * First call on a device: the library asks the runtime where the buffer lives on that device (cudaGetSymbolAddress;
 * the answer is kept per device).  The context's device must be the current one (else LQCD_EINVAL).  Make that first
 * call ahead of any stream capture.  Later calls only check arguments and enqueue the two launches on the context's
 * stream; like lqcd_mdagm the function returns without waiting for them.
 *
 * One buffer per device, shared by all contexts, streams and threads: two calls whose kernels may run on the same GPU
 * at the same time (different streams, or different contexts) overwrite each other's t and both results are garbage.
 * Keep such calls on one stream or order them with events.  The buffer holds whatever the last call left there;
 * nothing needs clearing, because every call rewrites all of t before reading it.
 *   out_even, in_even : parity vectors (even sites), DEVICE, must not alias;  sigma as lqcd_mdagm. */
#define LQCD_STATIC_MAX_VH 65536
int lqcd_mdagm_static(lqcd_ctx* ctx, double* out_even, const double* in_even, double sigma);

/* Single precision: the same operators on float parity vectors (3*Vh complex floats,
 * same index order) with the links stored as floats (LQCD_OPT_LINK_PRECISIONS must include LQCD_PREC_F32 at
 * lqcd_set_gauge time, otherwise LQCD_ENOGAUGE).  Arithmetic is float; only the CG's scalar products and
 * scalar recurrences are kept in double. */
int lqcd_doe_f32(lqcd_ctx* ctx, float* out_odd, const float* in_even);
int lqcd_deo_f32(lqcd_ctx* ctx, float* out_even, const float* in_odd);
int lqcd_doe_f32_host(lqcd_ctx* ctx, float* out_odd /*HOST*/, const float* in_even /*HOST*/);
int lqcd_deo_f32_host(lqcd_ctx* ctx, float* out_even /*HOST*/, const float* in_odd /*HOST*/);
int lqcd_mdagm_f32(lqcd_ctx* ctx, float* out_even, const float* in_even, double sigma);

/* Multi-shift CG for (m^2 - D_eo D_oe + shifts[i]) x[i] = b, i = 0..nshift-1, zero
 * initial guess, base system = smallest shift, stop when |r| <= tol*|b| for the base system, shift i is
 * frozen once zeta_i*|r| <= tol*|b| (readings R5-R7).
 *   b_even : parity vector (even sites);  shifts : HOST array of nshift values >= 0;
 *   x      : HOST array of nshift DEVICE pointers to parity vectors (overwritten).
 * Returns LQCD_OK, LQCD_ENOCONV or LQCD_EBREAKDOWN (or an argument / CUDA error). */
int lqcd_mshift_cg(lqcd_ctx* ctx, const double* b_even, const double* shifts /*HOST*/, int nshift,
                   double tol, double* const* x /*HOST array of DEVICE pointers*/);
/* Same, b and every x[i] in HOST memory; copies are part of the call. */
int lqcd_mshift_cg_host(lqcd_ctx* ctx, const double* b_even /*HOST*/, const double* shifts /*HOST*/,
                        int nshift, double tol, double* const* x /*HOST array of HOST pointers*/);

/* Single-precision multi-shift CG: float vectors and links, float sweeps; the scalar products are summed and
 * the recurrences run in double.  tol is limited by the arithmetic (the recurrence residual of a float CG
 * stops following the true residual around 1e-6..1e-5 relative for these condition numbers). */
int lqcd_mshift_cg_f32(lqcd_ctx* ctx, const float* b_even, const double* shifts /*HOST*/, int nshift,
                       double tol, float* const* x /*HOST array of DEVICE pointers*/);
int lqcd_mshift_cg_f32_host(lqcd_ctx* ctx, const float* b_even /*HOST*/, const double* shifts /*HOST*/,
                            int nshift, double tol, float* const* x /*HOST array of HOST pointers*/);

/* Mixed precision: the systems of lqcd_mshift_cg solved to a DOUBLE-precision tolerance with the iterations in
 * single precision (the paper keeps its fields "double (or float)", and mixes the two at the level of
 * the algorithm; here they are mixed inside one solve).  A float CG iterates on a recurrence residual;
 * whenever that has dropped by a factor 10 since the last time, the float partial solution is added to the double
 * one and the residual is REPLACED by the true residual b - (m^2 - D_eo D_oe + sigma) x computed with the double
 * operator, the search direction being kept ("reliable updates").  The stopping rule is on that true residual:
 * |b - (A + shifts[i]) x[i]| <= tol |b| for every i.  With nshift > 1 a float multi-shift solve first brings all
 * systems to a relative residual ~1e-5, then each system is finished on its own: the shifted systems cannot share
 * residual replacements (they would lose r_i = zeta_i r), so with many light shifts and a tight tol this costs MORE
 * than lqcd_mshift_cg; with one or few systems it is up to ~2x faster.  Measured on a B200 at
 * 48^4, m = 0.0075, tol 1e-10: 16 shifts 1e-5..1 -- 6.9 s (11734 float iterations, 68 residual replacements) against
 * 4.25 s for lqcd_mshift_cg, i.e. 1.6x SLOWER; the lightest system alone -- 2.24 s against 4.18 s.  Use it for single
 * systems (or a few heavy ones), and lqcd_mshift_cg for a whole set of rational-approximation shifts.
 * Needs both link copies (LQCD_OPT_LINK_PRECISIONS = LQCD_PREC_F64 | LQCD_PREC_F32 at lqcd_set_gauge time), else
 * LQCD_ENOGAUGE.  Arguments as lqcd_mshift_cg.  Statistics: LQCD_STAT_ITERS = float iterations in all phases,
 * LQCD_STAT_FREEZE_ITER[i] = float iterations spent finishing system i, LQCD_STAT_REL_RES = the largest final true
 * relative residual, LQCD_STAT_RELIABLE_UPDATES.  Not available on a slab context (LQCD_EINVAL). */
int lqcd_mshift_cg_mixed(lqcd_ctx* ctx, const double* b_even, const double* shifts /*HOST*/, int nshift,
                         double tol, double* const* x /*HOST array of DEVICE pointers*/);

/* Rational function of the Eq. 2 operator applied to b,
 *     y = alpha0 b + sum_i alpha[i] (m^2 - D_eo D_oe + shifts[i])^{-1} b ,
 * the partial-fraction form in which the RHMC uses the solutions of Eq. 2 (the rational approximation of the
 * fractional power of the Dirac matrix with poles sigma_i).  Same solver, stopping and
 * freezing rules as lqcd_mshift_cg, but the sum is accumulated during the solve (y += alpha_i a_i p_i) and
 * the x_i are never stored: 96 instead of 192 bytes per site and active shift in the update sweep, and no
 * memory for nshift solution vectors.
 *   alpha, shifts : HOST arrays of nshift values;  y_even : parity vector (overwritten), must not alias b.
 * Statistics as for lqcd_mshift_cg.  Returns as lqcd_mshift_cg. */
int lqcd_rational_apply(lqcd_ctx* ctx, const double* b_even, double alpha0, const double* alpha /*HOST*/,
                        const double* shifts /*HOST*/, int nshift, double tol, double* y_even);
/* Same, b and y in HOST memory; copies are part of the call. */
int lqcd_rational_apply_host(lqcd_ctx* ctx, const double* b_even /*HOST*/, double alpha0, const double* alpha /*HOST*/,
                             const double* shifts /*HOST*/, int nshift, double tol, double* y_even /*HOST*/);

int lqcd_rational_apply_f32(lqcd_ctx* ctx, const float* b_even, double alpha0, const double* alpha /*HOST*/,
                            const double* shifts /*HOST*/, int nshift, double tol, float* y_even);

/* ---- 1-D slab decomposition over several GPUs (Alg. 1) --------------------------
 * The paper cuts the lattice along one direction, one MPI rank (one GPU) per slab: each application of D_oe / D_eo
 * then needs the faces of the input vector from the two neighbouring ranks ("a pseudofermion border ... 48 bytes
 * per even site"), and each scalar product of the CG a global reduction.  The
 * operator is applied to the interior of the slab while the faces travel and to the two border slices afterwards
 * (Alg. 1).
 *
 * Here: one process per GPU, the cut is along t (the slowest index, so a face is contiguous per colour), rank r of
 * nranks owns the time slices [r*Lt/nranks, (r+1)*Lt/nranks).  Lt/nranks must be even (then local and global site
 * parities agree).  A slab context is used through the SAME calls as a whole-lattice one, on the rank's local
 * data: lqcd_set_gauge takes the links that leave the slab's sites (canonical layout of the local
 * Lx*Ly*Lz*(Lt/nranks) lattice), vectors are parity vectors of the local lattice, lqcd_mshift_cg solves the global
 * system (its statistics are identical on every rank).  Every rank must make the same sequence of calls with the
 * same options, shifts and tol.  The antiperiodic boundary sits on the links that leave the last time slice of the
 * whole lattice.  lqcd_set_u1_phases takes the angles of the slab's own links (4 * V_local) and, like lqcd_set_gauge,
 * needs the transport (the t-links below the slab, and their angles, come from rank-1 once).
 *
 * STATUS: verified on one GPU only (one rank with the ring closed on itself, over NCCL and over peer memory; several
 * ranks sharing the GPU, over peer memory (CUDA IPC) and through a host-staged transport).  Neither NCCL nor the
 * peer-memory transport has been run between two or more GPUs.
 *
 * A transport must be set before lqcd_set_gauge (which exchanges the t-links of the face once, and runs one all-reduce
 * so that the transport's connections exist before any CUDA graph is captured):
 *   lqcd_comm_init_nccl   NCCL send/recv + all-reduce on the GPU (NVLink 5 / NVSwitch between the GPUs of a node),
 *                         enqueued on streams, captured into the CUDA graph of the CG iteration;
 *   lqcd_comm_init_p2p    peer-mapped memory between the GPUs of one node (CUDA IPC): the faces are
 *                         written straight into the neighbours' halo buffers, arrival is a stream memory operation,
 *                         the scalar products are summed through slots in every rank's window; no transport kernel
 *                         on the path of the faces, no CUDA graph (the iteration is launched plainly);
 *   lqcd_set_comm         caller-supplied functions, e.g. on top of MPI or torch.distributed.
 */
lqcd_ctx* lqcd_create_slab(int Lx, int Ly, int Lz, int Lt_global, int rank, int nranks);

/* A transport = the two communication steps of the path.  All ranks call them in the same order.
 *   exchange(user, send_lo, send_hi, recv_lo, recv_hi, bytes, stream)
 *       ring along t: send_lo goes to rank-1, send_hi to rank+1; recv_lo receives what rank-1 sent as its
 *       send_hi, recv_hi what rank+1 sent as its send_lo (with nranks = 1 or 2 both neighbours may be the same
 *       rank, possibly myself).  `bytes` per buffer.
 *   allreduce_sum(user, buf, n, stream)
 *       buf[0..n) <- sum over ranks, in place, the same bits on every rank.
 * host_staged = 0: the buffers are DEVICE memory; the functions enqueue on `stream` (a cudaStream_t) or complete
 *                  before returning, and are ordered after the work already enqueued on `stream`.
 * host_staged = 1: the buffers are pinned HOST memory whose contents are complete on entry and are consumed after
 *                  return (the library does the copies and synchronises); `stream` is NULL.  Blocking.
 * graph_safe  = 1: the functions only enqueue stream work that CUDA graph capture accepts.
 * Return 0 on success; anything else makes the calling lqcd_* function return LQCD_ECOMM. */
typedef struct lqcd_comm_ops {
    void* user;
    int (*exchange)(void* user, const void* send_lo, const void* send_hi, void* recv_lo, void* recv_hi, size_t bytes,
                    void* stream);
    int (*allreduce_sum)(void* user, double* buf, int n, void* stream);
    int host_staged;
    int graph_safe;
} lqcd_comm_ops;
int lqcd_set_comm(lqcd_ctx* ctx, const lqcd_comm_ops* ops /*HOST; copied*/);

/* NCCL transport.  One rank obtains an id (128 bytes, HOST) with lqcd_nccl_unique_id and hands it to the others by
 * any means (e.g. a torch.distributed broadcast); then every rank calls lqcd_comm_init_nccl (collective: it
 * returns once all ranks of the slab context's nranks have joined).  LQCD_ECOMM if NCCL cannot be loaded or fails. */
#define LQCD_NCCL_ID_BYTES 128
int lqcd_nccl_unique_id(void* id /*HOST, 128 bytes*/);
int lqcd_comm_init_nccl(lqcd_ctx* ctx, const void* id /*HOST, 128 bytes*/);

/* Peer-memory transport (GPUs of one node that can map each other's memory; also ranks that share a GPU).
 * Every rank calls lqcd_p2p_export, which allocates its window (header + four face buffers, each the size of the
 * largest face message: 288 bytes x Lx/2*Ly*Lz) and writes LQCD_P2P_HANDLE_BYTES describing it; the caller gathers
 * the handles of all ranks by any means (e.g. torch.distributed.all_gather_object) and hands every rank the table of
 * all of them, in rank order, through lqcd_comm_init_p2p (not collective: it only maps the windows).  At most 16
 * ranks.  The window is allocated with cudaMalloc (CUDA IPC exports whole allocations): it is not part of a caller
 * workspace and is released by lqcd_destroy.  Environment: LQCD_P2P_KERNEL_SIGNAL=1 makes the arrival words of a face be
 * set by a one-thread kernel instead of cuStreamWriteValue32 (the transport switches to that by itself if the driver
 * refuses the stream memory operation on a peer-mapped address).  LQCD_ECOMM if a window cannot be mapped (no peer access, other node) or stream memory operations are
 * unavailable.  STATUS: verified on one GPU (one rank; two and four ranks as processes sharing the GPU over CUDA IPC);
 * not run between two or more GPUs. */
#define LQCD_P2P_HANDLE_BYTES 96
int lqcd_p2p_export(lqcd_ctx* ctx, void* handle /*HOST, LQCD_P2P_HANDLE_BYTES*/);
int lqcd_comm_init_p2p(lqcd_ctx* ctx, const void* handles /*HOST, nranks * LQCD_P2P_HANDLE_BYTES, rank order*/);

/* When a rank cannot go on.  Over the peer-memory transport the ranks wait for each other's faces and partial sums with
 * stream operations on flag words; a rank that stops making the same calls as the others would leave them waiting.
 *   - A rank whose solve fails (transport or CUDA error) marks the flag words of its peers before it returns; the
 *     peers' waits complete, their kernels see the mark, and their lqcd_mshift_cg / lqcd_rational_apply return
 *     LQCD_ECOMM (and pass the mark on, so ranks that were waiting for somebody else are released too).
 *   - A rank that has to leave for a reason of its own (an exception in the caller) calls lqcd_comm_abort first.
 *   - A rank whose process was killed marks nothing: the others give up after LQCD_OPT_COMM_TIMEOUT seconds without
 *     progress and return LQCD_ECOMM.
 * After LQCD_ECOMM (or lqcd_comm_abort) the context's transport is dead: every further solve or operator call on it
 * returns LQCD_ECOMM at once.  The caller must lqcd_destroy the context on EVERY rank (the x[] of the failed solve are
 * undefined), and to continue create new contexts, export new windows and exchange the handles again.  Operator calls
 * (lqcd_doe ...) return after enqueueing and cannot report a peer's mark themselves; the next solve does.
 * The NCCL transport has its own failure handling (NCCL's); a caller-supplied transport reports through its return
 * codes.  lqcd_comm_abort on a slab context without the peer-memory transport does nothing. */
int lqcd_comm_abort(lqcd_ctx* ctx);

/* rank, nranks, first global time slice and global Lt of a context (0, 1, 0, Lt for a whole-lattice one) */
int lqcd_slab_info(const lqcd_ctx* ctx, int* rank, int* nranks, int* t_offset, int* Lt_global /*HOST, may be NULL*/);

/* Statistics of the last solve; *out is HOST. idx is used by LQCD_STAT_FREEZE_ITER only. */
int lqcd_get_stat(const lqcd_ctx* ctx, int key, int idx, double* out /*HOST*/);

/* Convenience: site field (whole lattice, V*3 complex, array of structs) <-> parity vector.
 * pack reads only the sites of `parity`; unpack writes only those sites. */
int lqcd_pack_vector(lqcd_ctx* ctx, int parity, const double* site_field, double* parity_vector);
int lqcd_unpack_vector(lqcd_ctx* ctx, int parity, const double* parity_vector, double* site_field);
int lqcd_pack_vector_f32(lqcd_ctx* ctx, int parity, const float* site_field, float* parity_vector);
int lqcd_unpack_vector_f32(lqcd_ctx* ctx, int parity, const float* parity_vector, float* site_field);

const char* lqcd_last_error(const lqcd_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
