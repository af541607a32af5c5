/*
 * vmg.h -- C-ABI boundary of the B200-native variable-coefficient geometric multigrid library (libvmg.so).
 *
 * Solves, in fp64 on one GPU (sm_100a), the cell-centred finite-volume discretisation of
 *
 *        alpha * a * phi  -  beta * div( b grad phi )  =  f          on a uniform Cartesian box,
 *
 * the "Helmholtz equation form" into which the paper casts every governing equation before handing it to
 * its multigrid solver (sec. 4): the electrostatic Poisson equation Eq. 3, the
 * implicit diffusion part of the species / electron-energy equations Eq. 17 and the
 * photoionisation Helmholtz equations Eq. 9.  Discretisation: second-order central diffusive
 * flux on Cartesian finite-volume cells, implicit in time (sec. 3).  Boundary kinds: fixed
 * potential (Dirichlet) electrodes and homogeneous Neumann walls.  The multigrid
 * components (red-black Gauss-Seidel with face coefficients, residual+restriction, prolongation+correction,
 * coefficient averaging, fixed-sweep bottom solve, V-cycle) are those named by BASELINE.json:north_star; the
 * paper itself only names "multigrid".  All readings are listed in DESIGN.md.
 *
 * All array arguments are DEVICE pointers (fp64, 16-byte aligned) on the device that was current at
 * vmg_create, unless a parameter says "host".  Nothing here takes or returns a torch type.
 *
 * Layout (x fastest).  Cell arrays (a, rhs, phi): idx = i + nx*(j + ny*k).
 *   bx: (nx+1)*ny*nz, bx[i,j,k] is the face at x = i*dx between cells i-1 and i, idx = i + (nx+1)*(j + ny*k);
 *   by: nx*(ny+1)*nz, idx = i + nx*(j + (ny+1)*k);     bz: nx*ny*(nz+1), idx = i + nx*(j + ny*k).
 *   Boundary value planes: x faces idx = j + ny*k; y faces idx = i + nx*k; z faces idx = i + nx*j.
 * nz == 1 selects the 2-D operator: no z coupling; bz, dz and the z-face boundary entries are ignored.
 *
 * Every function returns a status code (below); there are no exceptions, no output on stderr, no abort.
 * After a negative code from vmg_solve the contents of phi are unspecified but the handle stays usable.
 * Calls on one handle must not overlap in time (no internal locking).
 */
#ifndef VMG_H
#define VMG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vmg_s* vmg_handle;

enum { VMG_XLO = 0, VMG_XHI = 1, VMG_YLO = 2, VMG_YHI = 3, VMG_ZLO = 4, VMG_ZHI = 5 };
enum { VMG_BC_DIRICHLET = 0, VMG_BC_NEUMANN = 1 };
enum {
    VMG_OK = 0,              /* converged to rtol                                                       */
    VMG_MAXCYCLES = 1,       /* ran max_vcycles cycles without reaching rtol (always, when rtol <= 0)   */
    VMG_STALLED = 2,         /* residual reduced by less than 10 % in 3 consecutive cycles (fp64 floor) */
    VMG_ERR_ARG = -1,        /* NULL / out-of-range argument, unknown option key                        */
    VMG_ERR_SIZE = -2,       /* grid cannot be coarsened to a bottom grid of <= 512 cells, >= 2^31 cells, ny > 65535 or nz > 32767 */
    VMG_ERR_STATE = -3,      /* vmg_solve before both vmg_set_coeffs and vmg_set_bc                     */
    VMG_ERR_SINGULAR = -4,   /* all active faces Neumann and (a == NULL or alpha == 0)                  */
    VMG_ERR_DIVERGED = -5,   /* residual became NaN or Inf                                              */
    VMG_ERR_CUDA = -6,       /* a CUDA runtime call failed (vmg_last_cuda_error gives the code)         */
    VMG_ERR_ALLOC = -7       /* device or host allocation failed                                        */
};

/* Create a solver for an nx x ny x nz box with cell sizes dx, dy, dz.  The level hierarchy halves every
 * active dimension while all stay even and >= 2 afterwards (256x128x128 -> ... -> 4x2x2); the coarsest grid
 * must have <= 512 cells (VMG_ERR_SIZE otherwise).  cuda_stream is a cudaStream_t; every kernel, copy and graph of this handle is
 * enqueued on it.  NULL: the handle creates a blocking stream of its own (ordered with the legacy default stream, not with
 * non-blocking or per-thread default streams: a caller that produces its inputs there must synchronise first) and
 * vmg_set_coeffs / vmg_set_bc synchronise it before they return.  With a caller-supplied stream those two calls only
 * ENQUEUE: the arrays passed to them must stay valid and unmodified until the stream has passed that point (stream-ordered
 * allocators such as torch's guarantee this for work on the same stream; vmg_solve synchronises the stream anyway).  All device memory the handle
 * needs (about 9.3 fp64 arrays of (nx+2)*ny*nz) is allocated here; vmg_solve allocates nothing on the device. */
int vmg_create(vmg_handle* out, int nx, int ny, int nz, double dx, double dy, double dz, void* cuda_stream);

/* Coefficients.  a: cell array or NULL (a == 0, alpha ignored).  bx, by, bz: face arrays, or all NULL for
 * b == 1 (then the sweeps, the residual + restriction and the residual norm run as kernels that form
 * the face weights from beta/h^2 and the cell's position instead of loading three weight arrays: the same numbers in
 * the same order, bitwise the results of explicit arrays of ones, at 2 instead of 5 doubles of traffic per cell and
 * half-sweep -- the Poisson equation PAPER.md:54 Eq. 3 and Helmholtz equations with a variable a; with a mask set
 * this holds for level 0, whose kernels then read one byte of open-face flags per cell, the averaged coarser levels
 * keep their arrays).  a must be >= 0 with alpha >= 0 and b > 0, beta > 0 (not checked; otherwise undefined behaviour).
 * The arrays are read by the kernels this call enqueues (see vmg_create for when they may be reused): the library
 * averages them to all coarse levels (a: mean of the 8 children, 4 in 2-D; b: mean of the fine faces lying
 * on the coarse face) and converts each level to its internal stencil form.  They are not referenced after
 * that; call again when coefficients change.  Passage: the Helmholtz form every governing equation is cast into,
 * PAPER.md:159 (section 4); Poisson PAPER.md:54 (Eq. 3), implicit diffusion PAPER.md:129-134 (Eq. 17). */
int vmg_set_coeffs(vmg_handle h, const double* a, const double* bx, const double* by, const double* bz,
                   double alpha, double beta);

/* Boundary conditions.  type: HOST array of 6 entries (VMG_BC_DIRICHLET / VMG_BC_NEUMANN), order XLO..ZHI.
 * value: HOST array of 6 DEVICE pointers to value planes, or NULL; a NULL entry (or value == NULL) means
 * homogeneous.  Dirichlet value = phi on the face; Neumann value = outward-normal derivative d(phi)/dn on
 * the face (not the flux b*d(phi)/dn).  The planes are copied (enqueued, see vmg_create).  May be called before
 * or after vmg_set_coeffs, and again at any time.  Passage: fixed-potential electrodes and homogeneous Neumann walls,
 * PAPER.md:230, :266, :284; readings R3-R6 of DESIGN.md section 2 for the discrete form. */
int vmg_set_bc(vmg_handle h, const int type[6], const double* const value[6]);

/* Cell masking ("cell masking for complex geometries").  mask: DEVICE array of
 * nx*ny*nz bytes in the cell layout, 1 = valid cell, 0 = covered cell (inside a solid), or NULL to remove the
 * mask.  kind: what every covered/valid interface face is: VMG_BC_DIRICHLET (phi = the covered cell's value at the
 * face, e.g. an electrode; cval: DEVICE cell array that holds that value in covered cells, NULL = 0) or
 * VMG_BC_NEUMANN (zero flux, e.g. an insulating body; cval ignored).  Covered cells are taken out of the solve: phi
 * comes back 0 there and f is not read there.  Both arrays are copied.  vmg_set_coeffs must be called (again)
 * afterwards -- it applies the mask to the coefficients of every level -- and VMG_ERR_STATE is returned by the
 * solves until then.  A Dirichlet mask with at least one covered cell makes an all-Neumann alpha = 0 problem
 * regular. */
int vmg_set_mask(vmg_handle h, const unsigned char* mask, int kind, const double* cval);

/* Solve.  rhs: f at cell centres (never written).  phi: initial guess in, solution out.
 * Iterates V(nu1,nu2) cycles until ||btilde - A phi||_inf <= rtol * ||btilde||_inf, where btilde is f with
 * the boundary data folded in, or until max_vcycles cycles (rtol <= 0: run exactly max_vcycles cycles).
 * Returns VMG_OK / VMG_MAXCYCLES / VMG_STALLED or a negative error.  Synchronises the stream before
 * returning.  Passage: "The composite multilevel multigrid solver ... is used for each of the governing equations"
 * PAPER.md:159; cycle, smoother, transfers and exit rules are readings C1-C5 / R7-R13 of DESIGN.md section 2. */
int vmg_solve(vmg_handle h, const double* rhs, double* phi, double rtol, int max_vcycles);

/* K handles for K problems on the same grid -- the paper's "multi-component" multigrid solves (section 7:
 * solving several solution components with each multigrid solve "results in more GPU work" per launch).  Same arguments as
 * vmg_create; out: HOST array of k handles.  The members share ONE device allocation (member i's arrays lie a constant
 * stride after member 0's) and one stream (cuda_stream, or one the library creates).  Each member is an ordinary handle for
 * every other call (own coefficients, boundary data, options, vmg_solve, vmg_destroy -- the allocation goes with the last
 * member).  vmg_solve_batch on exactly these k handles advances them with KERNEL-LEVEL batching: level 0 one problem after
 * the other (its consecutive half-sweeps reuse the L2), every coarser level of all k problems in single launches that run
 * over planes x problems, k CTAs in the single-CTA tail, one graph; bitwise the results of k separate vmg_solve calls.
 * That path needs equal smoothing options on all members, piecewise-constant prolongation, blocked = 0 and (for b == NULL)
 * equal beta; otherwise vmg_solve_batch falls back to its stream-level schedule. */
int vmg_create_batch(int k, vmg_handle* out, int nx, int ny, int nz, double dx, double dy, double dz, void* cuda_stream);

/* Batched solve (the paper's "multi-component" optimisation: "simultaneously solving multiple scalar solution
 * components with each multigrid solve results in more GPU work").  n independent
 * problems, one handle each -- same or different grids, coefficients and boundary conditions -- advanced in
 * lock-step: each round enqueues one V-cycle per unfinished handle on that handle's stream, then synchronises and
 * applies the exit rules of vmg_solve to each.  With two or more active handles the level-0 strokes of the handles are
 * run one after the other (token event) and the coarser levels of each handle beside the others' fine levels on a
 * highest-priority stream of its own: same kernels, same order per handle, bitwise the results of vmg_solve.  Create the handles with DISTINCT streams (or cuda_stream = NULL,
 * which gives each its own): the latency-bound coarse levels of one solve then overlap the bandwidth-bound fine
 * level of another.  handles, rhs, phi: HOST arrays of n entries (rhs[i], phi[i]: DEVICE arrays as in vmg_solve);
 * status: HOST array of n ints or NULL, receives what vmg_solve would have returned for problem i.  Every solve
 * performs exactly the operations vmg_solve would: results are bitwise the same.  Returns the most severe status
 * (the smallest negative code if any, else the largest positive, else VMG_OK). */
int vmg_solve_batch(int n, const vmg_handle* handles, const double* const* rhs, double* const* phi, double rtol,
                    int max_vcycles, int* status);

/* Conjugate gradients preconditioned by one symmetric V-cycle -- for the diffusion-dominated,
 * high-contrast regime in which the plain V-cycle iteration of vmg_solve contracts slowly or not at all and for which
 * the paper falls back to HYPRE.  Same arguments, layout, exit rules and status codes as vmg_solve;
 * max_iter counts CG iterations (one V-cycle, one operator application and two dot products each); the history holds
 * ||r||_inf / ||btilde||_inf of the recurrence residual.  The preconditioner is the V-cycle of vmg_solve with the
 * post-smoothing sweeps (and the second half of the bottom sweeps) run black -> red, from a zero guess; it needs
 * nu1 == nu2 (VMG_ERR_ARG otherwise).  Allocates three more level-0 arrays on first use (VMG_ERR_ALLOC). */
int vmg_solve_pcg(vmg_handle h, const double* rhs, double* phi, double rtol, int max_iter);

/* Result of the last vmg_solve.  cycles, relres: HOST scalars (may be NULL).  history: HOST array of at
 * least cycles+1 doubles (relative residual before the first cycle and after each cycle) or NULL. */
int vmg_get_info(vmg_handle h, int* cycles, double* relres, double* history);

/* Options (key is a HOST C string): "nu1", "nu2" (pre/post red-black sweeps, default 3, 0..8),
 * "bottom_sweeps" (default 32), "symmetric" (1: post-smoothing and the second half of the bottom sweeps run black -> red,
 *   which makes one V-cycle from zero a symmetric operator; default 0; vmg_solve_pcg switches it on for itself), "prolong" (0: piecewise-constant prolongation, default; 1: cell-centred trilinear,
 *   weights 3/4 and 1/4 per direction, ghost value -e at Dirichlet and +e at Neumann faces), "graph" (1: replay the V-cycle as a CUDA graph, default; 0: plain launches),
 * "tail" (1: the coarsest levels run in one single-CTA launch, default; 0: one kernel per step),
 * "cluster" (1, default: the level above the single-CTA tail runs distributed over a thread-block cluster of up to 8 CTAs,
 *   resident in their shared memory for its whole down- and up-stroke, halo planes exchanged through distributed shared
 *   memory, barrier.cluster between half-sweeps -- 13 fewer launches per V-cycle, bitwise the same results; needs 3-D,
 *   piecewise-constant prolongation and a level whose slabs fit (vmg_cluster.cuh); 0: one launch per step on that level),
 * "device_loop" (1, default: all V-cycles of a vmg_solve are ONE graph launch -- a conditional WHILE node whose condition
 *   a one-thread kernel sets from the exit rules -- and the residual norm of cycle c is taken by the first half-sweep of
 *   cycle c+1, which writes beside phi so that a converged iterate is returned untouched; bitwise the status, cycle count,
 *   history and phi of the host-driven loop; used when graph = 1, nu1 >= 2, nu2 >= 1, symmetric = 0, blocked = 0,
 *   max_vcycles <= 1000 and level 0 is not in the single-CTA tail; 0: one graph replay and one 8-byte read-back per cycle),
 * "snake" (1: consecutive whole-level kernels walk the level in opposite z-directions so that each starts on
 *   what the previous one left in L2, default; 0: always ascending),
 * "l2_persist" (MB of L2 set aside for the level-0 face weights through a stream access-policy window,
 *   default 24, 0 = none; applied only when those weights exceed half the L2.  NOTE: this raises
 *   cudaLimitPersistingL2CacheSize, a setting of the whole CUDA context, and sets the window on the handle's stream;
 *   vmg_destroy clears the window and puts the limit back to what it was when this handle first changed it),
 * "phi_keep_cells" (levels with at least this many cells read phi in a colour half-sweep (the neighbours) and in the residual norm with the normal
 *   cache policy instead of the streaming one, default 33554432: on a level whose phi is more than twice the L2 the
 *   evict-first lines are gone before the next row and plane ask for them; results do not depend on it),
 * "bottom_matrix" (1, default: the single-CTA tail applies the bottom solve -- bottom_sweeps red-black sweeps from a zero field,
 *   a fixed linear map of the right-hand side -- as that map's matrix, built once per coefficient change by running the sweeps
 *   on the unit vectors, when the bottom grid has at most 64 cells and the cycle is not the symmetric one; 0: run the sweeps.
 *   Same map, another rounding order),
 * "restrict_red_cells" (levels with at least this many cells, default 262144, restrict the residuals of the RED children only
 *   in the down-stroke: pre-smoothing ends with a black half-sweep, after which a black cell's residual is its own rounding
 *   error (~2 ulp of D phi, reading R12 of DESIGN.md), so the pass moves 5 instead of 7 doubles per cell; a very large value
 *   restricts all eight children everywhere, as vmg_step_residual_restrict and the blocked passes always do),
 * "pdl" (1: the V-cycle kernels are launched with programmatic stream serialisation, so each kernel's launch overlaps
 *   the tail of its predecessor, default; 0: plain serialisation),
 * "blocked" (temporally blocked smoother passes with fused transfers: 1 = register-staged (vmg_block2.cuh), 2 = TMA-fed
 *   ring with one split mbarrier per plane, 2 x 2 patch per thread, 3 = the same with one row per thread (vmg_block3.cuh);
 *   0: one kernel per colour half-sweep, default -- the blocked passes are bitwise equal but measure slower on B200),
 * "block_min_cells" (smallest level the blocked passes are used on when blocked = 1, default 4096),
 * "batch_full_mb" (set on member 0 of a vmg_create_batch group: while all members still iterate and k x 56 B x cells stays
 *   below this many MB, vmg_solve_batch runs ALL levels of the group problem-major in one graph, above it only the coarser
 *   levels and level 0 one problem after the other; default 400: measured on B200, k = 8: 64x32x32 4449 solves/s (1292
 *   sequential, 2579 stream-level), 128x64x64 1558 (921, 1636), 256x128x128 278 with level 0 sequential against 266 with
 *   everything batched -- eight 235 MB working sets defeat the L2 reuse of the half-sweeps -- (270, 303)),
 * "const_weights" (1: use the constant-weight kernels when b == NULL, default; 0: always load the weight arrays; takes
 *   effect at the next vmg_set_coeffs, which must follow),
 * "profile" (1: per-kernel-class event timing, see vmg_get_profile; implies plain launches; default 0). */
int vmg_set_option(vmg_handle h, const char* key, double v);

int vmg_destroy(vmg_handle h);

const char* vmg_strerror(int code);       /* static string */
int vmg_last_cuda_error(vmg_handle h);    /* cudaError_t of the last failed runtime call, 0 if none */

/* Self-check: counts the non-zero elements among all pad elements of the handle's internal arrays (the zero pads that
 * stand for the neighbours beyond the domain; no kernel may write them).  compute-sanitizer is not available on every
 * pool; the tests call this after exercising every kernel family (tests/test_gpu_parity.py).  Synchronises the stream. */
int vmg_debug_pad_check(vmg_handle h, long long* nonzero);

/* ---------------------------------------------------------------------------------------------------------
 * Introspection and single-step entry points.  They run the very kernels vmg_solve runs, one step at a
 * time, on caller-owned DEVICE arrays of the level's size, so that tests can compare each kernel with the
 * oracle.  Each synchronises the stream before returning.  Level 0 is the finest.
 * --------------------------------------------------------------------------------------------------------- */
int vmg_num_levels(vmg_handle h);
int vmg_level_dims(vmg_handle h, int level, int dims[3]);                       /* dims: HOST */
/* averaged coefficients of a level in the public layout (any pointer may be NULL) */
int vmg_get_level_coeffs(vmg_handle h, int level, double* a, double* bx, double* by, double* bz);
/* btilde = rhs + boundary terms (level 0) */
int vmg_step_fold_bc(vmg_handle h, const double* rhs, double* btilde);
/* nsweeps red-black Gauss-Seidel sweeps on a level: phi in/out */
int vmg_step_smooth(vmg_handle h, int level, double* phi, const double* rhs, int nsweeps);
/* r = rhs - A phi on a level */
int vmg_step_residual(vmg_handle h, int level, const double* phi, const double* rhs, double* r);
/* rhs_coarse = mean over children of (rhs - A phi) on `level`; coarse array has the size of level+1 */
int vmg_step_residual_restrict(vmg_handle h, int level, const double* phi, const double* rhs, double* rhs_coarse);
/* phi += P e_coarse */
int vmg_step_prolong_correct(vmg_handle h, int level, double* phi, const double* e_coarse);
/* the down-stroke of a level as vmg_solve runs it: nu1 sweeps (phi in/out), then rhs_coarse = mean over children
 * of (rhs - A phi); on levels the blocked smoother covers these are the fused passes */
int vmg_step_down(vmg_handle h, int level, double* phi, const double* rhs, double* rhs_coarse);
/* the up-stroke of a level: phi += P e_coarse, then nu2 sweeps (phi in/out) */
int vmg_step_up(vmg_handle h, int level, double* phi, const double* rhs, const double* e_coarse);
/* one V-cycle from level 0 with an already folded right-hand side: phi in/out */
int vmg_step_vcycle(vmg_handle h, double* phi, const double* btilde);
/* ||v||_inf of a device array of n doubles -> HOST scalar */
int vmg_step_norm_inf(vmg_handle h, const double* v, long long n, double* out);
/* number of kernel launches (graph nodes count individually) issued by the last vmg_solve, and by every
 * vmg_set_coeffs / vmg_solve since vmg_create */
long long vmg_last_launch_count(vmg_handle h);
long long vmg_total_launch_count(vmg_handle h);
/* Per-kernel-class device times.  With option "profile" = 1 the library issues plain launches (no graph)
 * and brackets each group of launches of one class with a CUDA event pair on the handle's stream; the
 * totals accumulate until the option is set again.  ms, launches: HOST arrays of 8 entries, classes:
 * 0 level-0 smoother, 1 level-0 residual+restriction, 2 level-0 prolongation+correction, 3 all coarser
 * levels (incl. bottom), 4 norms, 5 fold_bc, 6 phi copies in/out, 7 vmg_set_coeffs kernels. */
int vmg_get_profile(vmg_handle h, double ms[8], long long launches[8]);

/* ---------------------------------------------------------------------------------------------------------------
 * vmg_norm_inf_static -- the one entry point that ALLOCATES NOTHING (for callers that cannot call cudaMalloc: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  Operation: *out = ||v||_inf = max |v[t]|,
 * t < n, the norm of the exit rules (S6 of SURVEY.md 8(a); relres of 8(c) C5 / R12, BASELINE.json north_star (3)
 * "warp-shuffle and block reductions for the norms"), taken on the bit patterns as vmg_step_norm_inf does: the result
 * is exact and order-independent, a NaN anywhere in v gives a NaN, n == 0 gives 0.
 *   v            DEVICE array of n doubles (8-byte aligned), read only; may be NULL when n == 0
 *   out          DEVICE scalar (8-byte aligned), written by the kernel; valid once the stream has reached this call
 *   cuda_stream  a cudaStream_t of the CURRENT device (NULL = the legacy default stream); the call enqueues one 8-byte
 *                memset and one kernel there and returns without synchronising
 *   why          may be NULL; else receives a static string saying what was wrong ("ok" on success)
 * No handle, no cudaMalloc / cudaFree, no allocating library routine: the kernel's scratch (one partial maximum per
 * 4096 elements and a ticket counter) is a file-scope __device__ array of 262 400 bytes that every GPU which loads
 * libvmg.so holds until the process exits; the first call on a device looks up its address (cudaGetSymbolAddress), so
 * make one call (n = 0 will do) before a stream capture.  Limit: n <= VMG_NORM_INF_STATIC_MAX_N (= 512^3, the largest
 * configuration); beyond it VMG_ERR_SIZE and nothing is enqueued.
 * EVERY call on a device shares that array and it keeps the last call's contents (the call clears what has to start
 * at zero itself): calls that may overlap on the GPU -- different streams, graph branches, host threads -- RACE and
 * return garbage; order them on one stream or with events.  Ownership: caller owns v and out.
 * Errors: VMG_ERR_ARG (out NULL, n < 0, v NULL with n > 0), VMG_ERR_SIZE (n beyond the limit), VMG_ERR_CUDA (symbol
 * look-up, memset or launch refused; the sticky CUDA error is cleared). */
#define VMG_NORM_INF_STATIC_MAX_N 134217728LL
int vmg_norm_inf_static(const double* v, long long n, double* out, void* cuda_stream, const char** why);


/* ---------------------------------------------------------------------------------------------------------------
 * vmg_amr_* -- two-level COMPOSITE solve (second half).  The paper advances all AMR levels with one
 * time step and solves every equation with "the composite multilevel multigrid solver from within AMReX";
 * it gives no formula, so the interface discretisation and the cycle are readings A1-A5 of DESIGN.md (restated in
 * oracle/amr_oracle.c, which this is tested against):
 *   A1  box patches of coarse cells [lo, hi) refined by 2, each at least one coarse cell away from the box boundary and at
 *       least two coarse cells wide in every active direction, two patches at least two coarse cells apart in some
 *       direction (else VMG_ERR_SIZE); the box itself must be a legal vmg grid, a patch may have any such size;
 *   A2  coarse-fine face: flux b_f (g - phi_f) / (1.5 hf) per unit area, g = the coarse field at the point of the adjacent
 *       coarse cell opposite the fine cell centre, interpolated linearly in the tangential directions;
 *   A3  the coarse cell takes the sum of the fine fluxes through its face (conservation);
 *   A4  cycle: composite residual -> ONE V-cycle of the coarse box (options nu1, nu2, ... of the coarse handle) for it,
 *       under the patch for the mean of the children's residuals -> correction added on both levels (piecewise constant)
 *       -> nu_f = 6 red-black sweeps on the patch -> coarse cells under the patch = means of their children;
 *   A5  relres = max(||r_c||_inf over uncovered coarse cells, ||r_f||_inf) / max(||btilde_c||_inf uncovered, ||f_f||_inf);
 *       exit rules, status codes and history as vmg_solve (hist[c] = relres after c cycles).
 * Arrays: DEVICE pointers.  Coarse arrays have the layouts of vmg_set_coeffs / vmg_solve on the nx x ny x nz box; fine
 * arrays the same layouts on the patch as a box of fx x fy x fz = 2 (hi - lo) cells (fz = 1 when nz == 1; vmg_amr_fine_dims).
 * Coefficients are BORROWED on both levels until the next vmg_amr_set_coeffs / vmg_amr_destroy; the coarse coefficients
 * under the patch define the operator of the correction V-cycle there (keep them consistent with the fine ones, e.g.
 * their averages); a_c and a_f are both given or both NULL.  rhs_c under the patch is ignored; phi_c, phi_f: initial guess
 * in, solution out (phi_c under the patch: means of the children).  vmg_set_bc semantics for the box faces.
 * Stream: as vmg_create (NULL: the library creates one).  With one patch both levels run on it; with several, every patch runs
 * on an internal stream forked from and joined to it around each per-patch section.  vmg_amr_solve synchronises it.
 * Options: "nu_f" (1..64); every other key goes to the coarse handle (vmg_set_option).  No mask, no PCG on composite grids. */
typedef struct vmg_amr_s* vmg_amr_handle;
/* npatch >= 1 patches; lo, hi: npatch triples of coarse cell indices, flattened (lo[3 q + d]); HOST arrays */
int vmg_amr_create(vmg_amr_handle* out, int nx, int ny, int nz, double dx, double dy, double dz,
                   int npatch, const int* lo, const int* hi, void* cuda_stream);
int vmg_amr_num_patches(vmg_amr_handle h);
int vmg_amr_fine_dims(vmg_amr_handle h, int patch, int dims[3]);
/* a_f, bx_f, by_f, bz_f: HOST arrays of npatch DEVICE pointers (one set of fine arrays per patch); an array may be NULL
 * altogether or hold NULL entries (a = 0, b = 1 on that patch) */
int vmg_amr_set_coeffs(vmg_amr_handle h, const double* a_c, const double* bx_c, const double* by_c, const double* bz_c,
                       const double* const* a_f, const double* const* bx_f, const double* const* by_f, const double* const* bz_f,
                       double alpha, double beta);
int vmg_amr_set_bc(vmg_amr_handle h, const int type[6], const double* const value[6]);
int vmg_amr_set_option(vmg_amr_handle h, const char* key, double v);
/* rhs_f, phi_f: HOST arrays of npatch DEVICE pointers */
int vmg_amr_solve(vmg_amr_handle h, const double* rhs_c, const double* const* rhs_f, double* phi_c, double* const* phi_f,
                  double rtol, int max_cycles);
int vmg_amr_get_info(vmg_amr_handle h, int* cycles, double* relres, double* history /* >= cycles + 1 or NULL */);
/* vmg_debug_pad_check over the box and the patches: number of non-zero pad entries (0 expected) */
int vmg_amr_debug_pad_check(vmg_amr_handle h, long long* nonzero);
long long vmg_amr_last_launch_count(vmg_amr_handle h);
int vmg_amr_last_cuda_error(vmg_amr_handle h);
int vmg_amr_destroy(vmg_amr_handle h);

#ifdef __cplusplus
}
#endif
#endif /* VMG_H */
