/*
 * pb.h -- C ABI of the B200-native Jacobi-PCG solver for the linear finite-difference
 * Poisson-Boltzmann equation (arxiv 1704.02745; citations are /root/reference/PAPER.md lines).
 *
 * What the library solves (Eq. 3; Eq. 4):
 *
 *      sum over the six faces f of node c of  h^-2 eps_f [phi(c) - phi(nbr_f)]  +  kbar2(c) phi(c)  =  rhs(c)
 *
 * on an nx*ny*nz grid of unknowns (x fastest: idx = (k*ny + j)*nx + i), with Dirichlet
 * values on a ghost layer one node outside the grid (the paper's free-space boundary
 * condition).  The solver is the preconditioned conjugate-gradient iteration
 * of PAPER.md:104-126 (steps 1-8) with the Jacobi preconditioner M = diag(A) of
 * PAPER.md:138-140 and phi_0 = 0.  The library is unit-agnostic: the
 * paper's right-hand side h^-3 q(i,j,k) is whatever the caller passes as `rhs`.
 *
 * All entry points are extern "C", take plain pointers and sizes, never throw or abort,
 * and return a pb_status.  There is no global state: every tunable is per-handle state set with pb_set_option
 * (the only environment variable read is PB_VERBOSE, which turns on diagnostics on stderr).  One handle = one
 * operator on one device and one CUDA stream.  A handle is not thread-safe; distinct handles are independent.
 * There is NO CPU fallback: without a CUDA device every compute call returns PB_ERR_CUDA.
 * Determinism: every reduction has a fixed order for a fixed launch plan, so repeated solves on one handle are
 * bit-identical.  The SpMV plan of a precision is picked by timing candidates when its work arrays are first built
 * (like an FFT plan), so two handles for the same operator may differ in the last bits of the dot products;
 * pb_set_option(h, PB_OPT_AUTOTUNE, 0) pins the static plan, pb_get_plan reports the plan in use.
 *
 * Array layouts (all caller arrays are dense C arrays of fp64 unless stated otherwise):
 *   eps_x [nz][ny][nx+1]  face f lies between node i=f-1 and node i=f; the paper's
 *                         eps_i(i,j,k) (between (i,j,k) and (i+1,j,k)) is eps_x[k][j][i+1];
 *                         f=0 and f=nx touch the ghost layer.
 *   eps_y [nz][ny+1][nx]  likewise along y;   eps_z [nz+1][ny][nx]  likewise along z.
 *   kbar2 [nz][ny][nx]    nodal Boltzmann coefficient ("all the related coefficients ...
 *                         absorbed into kappa^2"), 1/length^2.  NULL = 0.
 *   rhs   [nz][ny][nx]    right-hand side of Eq. 3.  NULL = 0.
 *   bc    ghost Dirichlet values packed x-, x+ ([nz][ny] each), y-, y+ ([nz][nx] each),
 *         z-, z+ ([ny][nx] each): 2*(nz*ny + nz*nx + ny*nx) values.  NULL = 0.
 * `where` says whether the data pointers of THAT call are host (PB_HOST) or device
 * (PB_DEVICE, on the handle's device) pointers.  Scalars out (iters_out, relres_out) are
 * always host pointers.
 */
#ifndef PB_H_
#define PB_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pb_handle pb_handle;

typedef enum {
    PB_OK = 0,
    PB_ERR_INVALID_ARG = 1,
    PB_ERR_ALLOC = 2,
    PB_ERR_CUDA = 3,
    PB_ERR_NOT_SPD = 4,     /* a diagonal entry <= 0 or a non-finite coefficient found at create      */
    PB_ERR_BREAKDOWN = 5,   /* p.Ap <= 0 or NaN/Inf met during the solve; phi = last good iterate     */
    PB_ERR_MAXITER = 6,     /* not converged in maxiter; phi, iters and relres are still returned     */
    PB_ERR_TOO_LARGE = 7    /* pb_residual_noalloc: the grid exceeds the fixed scratch (PB_NOALLOC_MAX_ROWS) */
} pb_status;

typedef enum { PB_F32 = 0, PB_F64 = 1 } pb_precision;
typedef enum { PB_HOST = 0, PB_DEVICE = 1 } pb_memspace;

/*
 * pb_create -- build the operator of Eq. 3 and, if rhs or bc is given,
 * the right-hand side b of Eq. 4 with the ghost Dirichlet terms eps_f*g/h^2 folded in.
 * Inputs are COPIED (the caller may free them on return).  The handle owns all device
 * memory it allocates.  cuda_stream is a cudaStream_t on which every later call of this handle
 * enqueues its work; NULL = the handle creates (and owns) a blocking stream of its own.
 * pb_create only copies the inputs and checks the diagonal; the padded work arrays of a precision
 * (and the launch plan) are built on first use or by pb_prepare.
 * Errors: nx,ny,nz < 1, h <= 0 or non-finite, NULL eps/out pointers -> PB_ERR_INVALID_ARG;
 * a node whose diagonal sum(eps_f)/h^2 + kbar2 is <= 0 or non-finite -> PB_ERR_NOT_SPD;
 * allocation / CUDA failures -> PB_ERR_ALLOC / PB_ERR_CUDA.  On error *out = NULL.
 */
pb_status pb_create(pb_handle **out, int nx, int ny, int nz, double h,
                    const double *eps_x, const double *eps_y, const double *eps_z,
                    const double *kbar2, const double *rhs, const double *bc,
                    pb_memspace where, void *cuda_stream);

/*
 * pb_set_rhs -- same operator, new right-hand side (Eq. 4: b = rhs + ghost fold-in).
 * Used for the many-snapshot workload the paper motivates.  Copies its inputs: the call returns
 * after the copies are complete (host or device), so the caller may free or overwrite them.  Device inputs must be
 * complete when the call is made (the handle's stream is not ordered against the stream that produced them).
 */
pb_status pb_set_rhs(pb_handle *h, const double *rhs, const double *bc, pb_memspace where);

/*
 * pb_apply -- y = A x, the left-hand side of Eq. 3 with x = 0 on the ghost layer, 1/h^2
 * included.  x and y are [nz][ny][nx] arrays of the requested precision (float for
 * PB_F32, double for PB_F64); they must not alias.  Runs the same matrix-free stencil
 * kernel the solver uses.
 */
pb_status pb_apply(pb_handle *h, pb_precision prec, const void *x, void *y, pb_memspace where);

/*
 * pb_solve -- Jacobi-PCG, PAPER.md:104-126 with M = diag(A), phi_0 = 0.
 *   tol         delta of step 3: stop at the first l with ||r_l||_2 / ||b||_2 < tol, r_l the
 *               recurrence residual, b the folded right-hand side of Eq. 4.
 *   maxiter     largest l allowed (>= 0).
 *   prec        storage/arithmetic type of the vectors; every dot product accumulates in fp64.
 *   check_every the host reads the 8-byte on-device {done, iters} latch once per this many
 *               iterations (>= 1); there is no other host<->device traffic during the solve.
 *               The returned iterate is exactly the one at which the test first passed,
 *               whatever check_every is.  (Grids whose working set fits the L2 run the whole loop in
 *               one cooperative kernel and are not polled at all.)
 *   phi_out     [nz][ny][nx] in `prec`, caller-allocated, host or device per `where`.
 *   iters_out   l at exit = number of A*p products (may be NULL).
 *   relres_out  ||r_l||/||b|| at exit (may be NULL).
 * Returns PB_OK, PB_ERR_MAXITER or PB_ERR_BREAKDOWN (phi_out/iters/relres valid in all
 * three), or an argument/CUDA error.  b = 0 gives phi = 0, iters = 0, relres = 0.
 * Blocks until phi_out holds the result.
 */
pb_status pb_solve(pb_handle *h, double tol, int maxiter, pb_precision prec, int check_every,
                   void *phi_out, pb_memspace where, int *iters_out, double *relres_out);

/*
 * pb_solve_from -- pb_solve with a given initial guess phi_0 (step 1 of PAPER.md:108: r_0 = b - A phi_0; the
 * paper's own runs use phi_0 = 0).  phi0 has the layout, precision and memory space of phi_out
 * and may alias it; NULL = 0.  The stopping rule stays ||r_l|| / ||b|| < tol.  Meant for sequences of nearby
 * right-hand sides (MD snapshots): start from the previous potential (NEXT row f2).
 */
pb_status pb_solve_from(pb_handle *h, double tol, int maxiter, pb_precision prec, int check_every,
                        const void *phi0, void *phi_out, pb_memspace where, int *iters_out, double *relres_out);

/*
 * pb_solve_batch -- m right-hand sides on the SAME operator (NEXT row f2 of SURVEY.md 8(f); the paper's motivation is
 * "thousands to millions of snapshots"): the Jacobi-PCG of pb_solve (phi_0 = 0) run
 * for PB_OPT_BATCH_WIDTH members at a time by kernels that stage the operator's coefficient boxes once per plane for
 * all of them (k_spmv_batch) and read Dinv once per node (k_vec_batch).  Every member has its own device-resident
 * scalars and convergence latch; a member that has converged stops being read or written, the group ends when all
 * its members are done.  Per member the arithmetic is that of a single solve (same operations in the same order per
 * node), so its iterates, iteration count and result do not depend on the other members.
 *   rhs [m][nz][ny][nx], bc [m][2*(nz*ny+nz*nx+ny*nx)] (either may be NULL = 0), phi_out [m][nz][ny][nx] in `prec`;
 *   all in the memory space `where`.  iters_out / relres_out / status_out: host arrays of m entries (may be NULL);
 *   status_out[s] is PB_OK, PB_ERR_MAXITER or PB_ERR_BREAKDOWN.
 * Returns the worst member status (BREAKDOWN > MAXITER > OK) or an argument / CUDA error.  Needs the free-space
 * boundary condition (PB_ERR_INVALID_ARG under pb_set_boundary(h, 1)).  The handle's own right-hand side (pb_set_rhs)
 * is left holding the last member's when the members are host arrays.  Face palettes of at most four values are
 * read as 2-bit indices (four nodes per byte), anything else as full words.
 */
pb_status pb_solve_batch(pb_handle *h, int m, const double *rhs, const double *bc, double tol, int maxiter,
                         pb_precision prec, int check_every, void *phi_out, pb_memspace where, int *iters_out,
                         double *relres_out, int *status_out);

/* pb_solve_batch_charges -- the same for a handle made by pb_create_from_atoms: member s is the charge set
 * charges[s][n_atoms] on the stored atoms; its right-hand side and ghost values are built on the device as in
 * pb_set_charges (the handle's rhs / bc end up holding the last member's). */
pb_status pb_solve_batch_charges(pb_handle *h, int m, const double *charges, double tol, int maxiter,
                                 pb_precision prec, int check_every, void *phi_out, pb_memspace where, int *iters_out,
                                 double *relres_out, int *status_out);

/*
 * z-slab decomposition of ONE solve over several GPUs (NEXT row f4; the paper's node had two
 * GPUs).  Rank r owns the planes [z0, z0 + nz) of the global grid; pb_create_slab takes ITS part of the
 * inputs (eps_z with the nz + 1 faces of its planes -- the interface faces are passed to both neighbours --, bc with
 * z-/z+ entries that are ignored across an interface) and says whether a neighbour rank lies below / above; there the
 * neighbouring plane is an unknown of the other rank, not the Dirichlet ghost layer, so nothing is folded into b and
 * the kernels read one ghost plane of r, p and Dinv, refreshed by the caller every iteration.  The library has no
 * communicator of its own: the exchange is the caller's (NCCL through torch.distributed in the Python package,
 * paper_1704_02745_b200/slab.py).  One PCG iteration (steps 4-8) on every rank:
 *     pb_slab_step(h, 0)   K_spmv on the slab; local p.Ap                       -> all-reduce ptrs[2] (1 double)
 *     pb_slab_step(h, 1)   alpha (step 5), K_vec; local r.z, r.r                -> all-reduce ptrs[3] (2 doubles)
 *     pb_slab_step(h, 2)   beta, stopping rule, latch (steps 3, 7) -- identical on every rank
 *     pb_slab_step(h, 4)   pack the boundary planes of r and p into ptrs[0]     -> send halves below / above, receive ptrs[1]
 *     pb_slab_step(h, 5)   unpack ptrs[1] into the ghost planes
 * and once per solve: pb_slab_begin (steps 1-2; local r.r, r.z), all-reduce ptrs[3], pb_slab_step(h, 3) (the step-2
 * finaliser: ||b||^2, beta = 0), the Dinv boundary planes ptrs[4], ptrs[5] sent to the neighbours' ptrs[7], ptrs[6],
 * then pack / exchange / unpack.  Kernels enqueued after the latch is set do nothing, so the loop may run ahead of
 * pb_slab_latch (which synchronises).  pb_slab_result un-pads this rank's planes of phi.  All other solve / apply
 * entry points return PB_ERR_INVALID_ARG for a slab handle.  No periodic boundary.
 */
pb_status pb_create_slab(pb_handle **out, int nx, int ny, int nz, double h,
                         const double *eps_x, const double *eps_y, const double *eps_z,
                         const double *kbar2, const double *rhs, const double *bc,
                         pb_memspace where, void *cuda_stream, int neighbour_below, int neighbour_above);
pb_status pb_slab_begin(pb_handle *h, pb_precision prec, double tol, int maxiter);
pb_status pb_slab_step(pb_handle *h, int which);
/* ptrs[8]: device pointers (valid after pb_slab_begin, until the handle's options change): 0 send buffer, 1 receive
 * buffer (4 planes each: r_lo, p_lo, r_hi, p_hi), 2 p.Ap (1 double), 3 {r.z, r.r} (2 doubles), 4 / 5 Dinv planes 0 and
 * nz-1, 6 / 7 Dinv ghost planes -1 and nz.  *plane_bytes = ny * pitch * sizeof(element). */
pb_status pb_slab_pointers(pb_handle *h, void **ptrs, size_t *plane_bytes);
pb_status pb_slab_latch(pb_handle *h, int *done, int *iters, int *status, double *relres);
pb_status pb_slab_result(pb_handle *h, void *phi_out, pb_memspace where);

/*
 * pb_create_from_atoms -- NEXT row f1, the paper's stated next step "integrated grid stencil setup on GPU"
 * (PAPER.md:11, 283): build the inputs of Eq. 3 on the device from atoms and hand them to pb_create.
 *   centres [n_atoms][3] (x,y,z; node (i,j,k) sits at (i h, j h, k h)), radii [n_atoms], charges [n_atoms]
 *   node is solute iff it lies within some atom sphere (d^2 <= R^2); eps_in there, eps_out elsewhere and on the
 *   ghost layer; face eps = harmonic mean of its two nodes; kbar2 = kbar2_solvent on solvent
 *   nodes, 0 in the solute; charges spread trilinearly, rhs = 4 pi q/h^3; ghost Dirichlet values =
 *   sum_i q_i exp(-kappa r_i)/(eps_out r_i) with kappa^2 = kbar2_solvent/eps_out (free-space boundary).
 * Needs nx,ny,nz >= 2.  The handle keeps the atom positions for pb_set_charges.
 */
pb_status pb_create_from_atoms(pb_handle **out, int nx, int ny, int nz, double h, int n_atoms,
                               const double *centres, const double *radii, const double *charges,
                               double eps_in, double eps_out, double kbar2_solvent,
                               pb_memspace where, void *cuda_stream);

/* pb_set_charges -- same atoms and operator, new charges [n_atoms]: new rhs and ghost values (an MD-snapshot-style
 * batch member).  Only for handles made by pb_create_from_atoms. */
pb_status pb_set_charges(pb_handle *h, const double *charges, pb_memspace where);

/*
 * pb_set_setup_precision -- arithmetic of the Debye-Hueckel boundary sum in later pb_set_charges calls (SURVEY.md 8(f)
 * f1; the sum has n_ghost x n_atoms terms, 5.3e10 at config 5, and is plain-ALU-bound).  PB_F64 (default): every term
 * in fp64, parity with the fp64 setup oracle to rounding.  PB_F32: terms in fp32 (coordinates relative to the box
 * centre, hardware rsqrt / exp2, Kahan-compensated fp32 partial sums per 256 atoms, fp64 across tiles): boundary values
 * within a few 1e-7 of the largest term of the fp64 ones -- enough for an fp32 solve -- at several times the rate.
 * The charge spreading and b stay fp64 either way.
 */
pb_status pb_set_setup_precision(pb_handle *h, pb_precision prec);

/* pb_get_field -- copy one of the handle's dense fp64 input fields to the host (tests of pb_create_from_atoms):
 * which = 0 eps_x, 1 eps_y, 2 eps_z, 3 kbar2, 4 rhs, 5 bc (layouts as in pb_create; a NULL input reads as zeros). */
pb_status pb_get_field(pb_handle *h, int which, double *out_host);

/*
 * pb_set_preconditioner -- kind 1 (default): Jacobi, M = diag(A); kind 0: M = I, i.e. the
 * unpreconditioned CG the paper times as "GPU/CG" (its listing is sign-garbled, so it is run
 * as the PCG recurrence of PAPER.md:104-126 with z = r, DESIGN.md Reading 1).  Applies to later solves.
 */
pb_status pb_set_preconditioner(pb_handle *h, int kind);

/*
 * pb_solve_refined -- mixed-precision iterative refinement ("fp32-inner / fp64-outer"): phi and
 * the true residual r = b - A phi are kept in fp64; each correction A d = r is a Jacobi-PCG solve (PAPER.md:104-126,
 * the kernels of pb_solve) in fp32 to `inner_tol` relative to ||r|| (1e-5 is what fp32 storage delivers; the last
 * correction only closes the remaining gap); phi += d.  Stops when the TRUE relative residual ||b - A phi||/||b||
 * <= tol (written to *relres_out), after `maxiter` inner iterations in total (PB_ERR_MAXITER, phi_out = last
 * iterate) or on a breakdown.  phi_out: [nz][ny][nx] fp64, host or device per `where`.  *outer_out = number of
 * corrections, *iters_out = inner PCG iterations in total.  Builds both the fp32 and the fp64 work arrays.
 */
pb_status pb_solve_refined(pb_handle *h, double tol, int maxiter, double inner_tol, int check_every, double *phi_out,
                           pb_memspace where, int *outer_out, int *iters_out, double *relres_out);

/*
 * pb_residual -- the TRUE relative residual ||b - A phi||_2 / ||b||_2 of a caller-supplied potential ([nz][ny][nx] in
 * `prec`), evaluated with the SpMV kernel in that precision and fp64 sums.  pb_solve tests and returns the recurrence
 * residual (DESIGN.md Reading 5); with fp32 storage the true residual stagnates near 1e-6..1e-5 while
 * the recurrence keeps falling, which is what this call makes visible.
 */
pb_status pb_residual(pb_handle *h, pb_precision prec, const void *phi, pb_memspace where, double *relres_out);

/*
 * pb_set_boundary -- kind 0 (default): the free-space condition, Dirichlet values on the ghost layer; kind 1: the
 * periodic boundary condition the paper also times.  Periodic: the neighbour across
 * a box face is the node on the opposite side; face f = 0 and face f = n of a direction are one physical face (the
 * caller passes equal values); bc is ignored.  In a matrix-free kernel the paper's "6 extra bands" are index wraps.
 */
pb_status pb_set_boundary(pb_handle *h, int kind);

/*
 * Per-handle options ("no global state").  pb_set_option drops the work arrays and the plan of
 * both precisions when the value changes; they are rebuilt on the next use (pb_prepare / pb_solve / ...).
 * Invalid option or value -> PB_ERR_INVALID_ARG.
 */
typedef enum {
    PB_OPT_PERSIST = 0,              /* 1 (default): grids whose working set fits the L2 run the whole loop in one
                                        cooperative kernel; 0: always k_spmv_tma + k_vec                              */
    PB_OPT_PERSIST_MAX_MB = 1,       /* working-set limit of that path in MB (default 100)                           */
    PB_OPT_PERSIST_FUSED_MAX_KNODES = 2, /* below this many thousand padded nodes the two-barrier form (default 600) */
    PB_OPT_PERSIST_BLOCKS_PER_SM = 3,/* cap on co-resident blocks of the cooperative kernel (default 4)              */
    PB_OPT_PALETTE = 4,              /* 1 (default): face dielectrics with few distinct values stored as index bytes */
    PB_OPT_PALETTE_DIAG = 5,         /* 1 (default): k_vec reads Dinv through the diagonal palette                   */
    PB_OPT_PALETTE_DIAG_SPMV = 6,    /* 1 (default): k_spmv_tma too                                                  */
    PB_OPT_AUTOTUNE = 7,             /* 1 (default): time candidate plans; 0: first feasible candidate (static)      */
    PB_OPT_TILE_TXV = 8,             /* k_spmv_tma tile: 16-byte vectors per row (0 = automatic, default)            */
    PB_OPT_TILE_TY = 9,              /*                  rows                                                        */
    PB_OPT_TILE_TZ = 10,             /*                  planes per tile                                             */
    PB_OPT_RING_SLOTS = 11,          /*                  shared-memory ring depth                                    */
    PB_OPT_BLOCKS_PER_SM = 12,       /*                  persistent blocks per SM                                    */
    PB_OPT_VEC_BLOCKS_PER_SM = 13,   /* k_vec blocks per SM (0 = automatic)                                          */
    PB_OPT_GRAPH = 14,               /* 1 (default): check_every iterations are launched as one CUDA graph           */
    PB_OPT_L2_HINTS = 15,            /* bit mask of L2 eviction-priority hints (default 0: none; measured not to help) */
    PB_OPT_BATCH_WIDTH = 16,         /* right-hand sides per kernel pass of pb_solve_batch: 1 (default: one member at a
                                        time through k_pcg_fused, the fastest measured), 2 or 4 (k_spmv_batch + k_vec_batch) */
    PB_OPT_FUSED = 17,               /* 1 (default): pb_solve / pb_solve_batch run ONE kernel per iteration (k_pcg_fused:
                                        K_vec folded into the next K_spmv pass, 34 instead of 41 B per node); 0: K_spmv
                                        + K_vec.  Periodic boundary, warm starts, refinement, slabs and L2-resident
                                        grids always take their own paths                                              */
    PB_OPT_TAIL_POOL = 18,           /* k_pcg_fused: the top ~5 % of the planes are cut into chunks of this many planes
                                        that the blocks fetch from a device-wide counter when they run out of their
                                        static tiles (evens out the blocks' finishing times).  0 (default): chunks of 8
                                        planes when nz >= 64, else off; 1: off; 4..64: on, chunks of that many planes  */
    PB_OPT_COUNT_ = 19
} pb_option;

pb_status pb_set_option(pb_handle *h, pb_option opt, int value);
pb_status pb_get_option(pb_handle *h, pb_option opt, int *value_out);

/* The launch plan of one precision (what bench.py prints and tests pin). */
typedef struct {
    int precision;            /* PB_F32 / PB_F64                                                        */
    int num_sm;               /* multiprocessors of the handle's device                                */
    int persist;              /* 1: pb_solve runs the cooperative kernel (L2-resident grid)            */
    int persist_fused;        /*    its two-barrier form                                               */
    int persist_grid;         /*    its grid                                                           */
    int palette_size;         /* distinct face values (0: more than 256)                               */
    int diag_palette_size;    /* distinct diagonal values (0: none / too many)                         */
    int face_palette;         /* 1: this precision stores face coefficients as index bytes             */
    int diag_palette_vec;     /* 1: k_vec reads Dinv as an index byte                                  */
    int diag_palette_spmv;    /* 1: k_spmv_tma reads Dinv as an index byte                             */
    int txv, ty, tz;          /* k_spmv_tma tile: vectors x rows x planes                              */
    int ring_slots, blocks_per_sm, tiles, grid, threads, smem_bytes;
    int autotuned;            /* 1: picked by timing, 0: static / forced                               */
    int vec_grid, vec_threads;/* k_vec launch                                                          */
    int spmv_bytes_per_node;  /* stored-format bytes per node and launch, as pb_bytes_per_node         */
    int vec_bytes_per_node;
    int pitch;                /* padded row length in elements                                         */
    int fused;                /* 1: pb_solve runs k_pcg_fused (one kernel per iteration); then txv ... smem_bytes
                                 describe ITS plan (ring_slots = vector slots), vec_grid = 0                          */
    int face_quad;            /* fused / batch kernels: faces as 2-bit indices, four nodes per byte                  */
    int coef_slots;           /* fused / batch kernels: depth of the coefficient ring                                */
    int tail_pool;            /* k_pcg_fused: planes per dynamically scheduled chunk of the top of the grid, 0 = none  */
    int reserved[4];
} pb_plan;

/* pb_prepare -- build the work arrays of `prec` (setup row a0: padded coefficients, diagonal, folded b) and pick
 * the launch plan now instead of on first use.  pb_get_plan does the same and reports the plan. */
pb_status pb_prepare(pb_handle *h, pb_precision prec);
pb_status pb_get_plan(pb_handle *h, pb_precision prec, pb_plan *out);

/*
 * pb_iterate -- benchmarking/profiling entry: enqueue exactly `n_iter` PCG iterations
 * (K_spmv + K_vec pairs, PAPER.md:115-126 steps 4-8) with the convergence latch disabled,
 * continuing from the state left by pb_solve_begin.  Does not synchronise.  Used by
 * bench.py to time the steady-state iteration with CUDA events.
 */
pb_status pb_solve_begin(pb_handle *h, pb_precision prec);              /* steps 1-2: x=0, r=b, z=r/D */
pb_status pb_iterate(pb_handle *h, pb_precision prec, int n_iter);

/*
 * pb_profile -- like pb_iterate, but brackets every kernel with a CUDA event on the handle's
 * stream and returns the mean device time (milliseconds) of K_spmv and of K_vec over the
 * n_iter iterations.  Synchronises.  This is the roofline measurement of bench.py.
 */
pb_status pb_profile(pb_handle *h, pb_precision prec, int n_iter, double *ms_spmv, double *ms_vec);

/* Number of CUDA kernels this handle has enqueued so far (those inside launched graphs included). */
long long pb_launch_count(pb_handle *h);

/* Size of the handle's coefficient palette: when the three face-dielectric arrays hold <= 256 distinct values
 * (every molecular map built from eps_in / eps_out and their harmonic mean, does) they are stored
 * exactly as one byte per face plus a table and decoded inside the SpMV; 0 = full-precision face arrays.
 * The index bytes are stored pre-multiplied by the element size (the kernel adds them to the table address without a
 * shift), so a precision uses the palette only when size * sizeof(element) <= 256, i.e. up to 64 values in fp32 and
 * 32 in fp64 (pb_bytes_per_node tells which format a precision got).  PB_OPT_PALETTE = 0 disables the palette. */
int pb_palette_size(pb_handle *h);

/* Size of the diagonal palette: with a face palette and a few-valued salt map the Jacobi diagonal also takes <= 256
 * distinct values, and k_vec then reads one index byte per node instead of a Dinv word (exact: the table holds
 * (T)(1/d)); 0 = Dinv array.  PB_OPT_PALETTE_DIAG = 0 disables it. */
int pb_diag_palette_size(pb_handle *h);

/* Bytes per grid node and launch that kernel `kernel` (0: k_spmv_tma, the PCG step; 1: k_vec) has to move in the
 * storage format this handle uses for `prec` -- the algorithmic bytes of bench.py's roofline:
 * k_spmv_tma reads r, p, x and writes p, x, Ap (6 words) plus Dinv (a word, or one index byte with the diagonal
 * palette; PB_OPT_PALETTE_DIAG_SPMV = 0 keeps the word) plus the three face coefficients (3 words, or 3 index bytes with the
 * palette); k_vec reads r, Ap, writes r (3 words) plus Dinv (word or byte).  Builds the work arrays of `prec` if
 * they do not exist yet; -1 on error. */
int pb_bytes_per_node(pb_handle *h, pb_precision prec, int kernel);

/* pb_destroy(NULL) is a no-op.  Frees every device allocation of the handle. */
pb_status pb_destroy(pb_handle *h);

/* Static, never-NULL description of a status code. */
const char *pb_strerror(pb_status s);

/*
 * pb_residual_noalloc -- the true relative residual ||b - A phi|| / ||b|| (A of Eq. 3, b of Eq. 4 with the ghost
 * Dirichlet terms folded in; the quantity pb_residual reports) for callers that CANNOT ALLOCATE: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  No handle: the call allocates
 * nothing (no cudaMalloc / cudaFree / allocating library routine) and does not synchronise; it enqueues one 256-byte
 * memset and one kernel on `cuda_stream` (a cudaStream_t; NULL = the legacy default stream) of the CURRENT device.
 * Every pointer is a DEVICE pointer on that device, fp64, dense, laid out as for pb_create: eps_x [nz][ny][nx+1],
 * eps_y [nz][ny+1][nx], eps_z [nz+1][ny][nx], kbar2 / rhs / phi [nz][ny][nx], bc = the six ghost faces; kbar2, rhs
 * and bc may be NULL (zeros).  Output, written by the kernel: out3[0] = ||b - A phi|| / ||b|| (0 if b = 0),
 * out3[1] = ||r||^2, out3[2] = ||b||^2 of the h^2-scaled system.  Sums are formed in a fixed order (reproducible).
 * Scratch: a fixed __device__ array of the library (512 KiB + 256 B, held by every GPU that loads the library until
 * exit) sized for PB_NOALLOC_MAX_ROWS = 262 144 grid rows (nz * ny, e.g. 512 x 512; nx is free up to 2e9 nodes):
 * a larger grid -> PB_ERR_TOO_LARGE, nothing enqueued.  Every call on a device SHARES that array: calls that overlap
 * on the GPU (different streams, different host threads) race -- serialise them.  The array keeps the last call's
 * partial sums; the one word that must start at zero is cleared on the stream by every call.  The first call on a
 * device looks the array's device address up (cudaGetSymbolAddress): make it outside stream capture.
 * Errors: sizes < 1, h <= 0 or non-finite, NULL eps / phi / out3 -> PB_ERR_INVALID_ARG; no device, launch or
 * memset failure -> PB_ERR_CUDA.  Asynchronous faults (bad device pointers) surface at the caller's next sync.
 */
#define PB_NOALLOC_MAX_ROWS 262144
pb_status pb_residual_noalloc(int nx, int ny, int nz, double h, const double *eps_x, const double *eps_y,
                              const double *eps_z, const double *kbar2, const double *rhs, const double *bc,
                              const double *phi, double *out3, void *cuda_stream);

/*
 * pb_query -- read back derived quantities for tests (device -> host copies, fp64):
 *   what = 0: diag(A) [nz][ny][nx] (1/h^2 included);  what = 1: folded b of Eq. 4 [nz][ny][nx];
 *   what = 2: the 10 device-resident scalars {r.z, p.Ap, r.r, b.b, alpha, beta, l, done, status, iters}
 *             of the h^2-scaled system as they stand on the stream (diagnostics, out_host[10]);
 *   what = 3..7: the work vectors r, Dinv, p, A'p, x [nz][ny][nx] of the last pb_solve/pb_solve_begin
 *             precision, converted to fp64, in the h^2-scaled system A' = h^2 A (per-kernel parity tests);
 *             x is the stored phi, i.e. without the still-pending alpha*p of the latest iteration.
 */
pb_status pb_query(pb_handle *h, int what, double *out_host);

/* Compile-time facts about the built library (for the bench report). */
int pb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PB_H_ */
