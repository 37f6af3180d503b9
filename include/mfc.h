/*
 * mfc.h -- C ABI of libmfc_b200: the right-hand side of the 5-equation diffuse-interface model
 * (Allaire form, K = 0) with stiffened-gas EOS on a uniform or non-uniform Cartesian grid, as hand-written CUDA for
 * sm_100a (NVIDIA B200), driven by 3-stage TVD Runge-Kutta.
 *
 * Method: arxiv 2305.09163 (Radhakrishnan et al.), cited below as PAPER.md:LINE (section / equation).
 * Readings of passages where the paper is silent or garbled are listed in DESIGN.md ("Readings", B1..B21).
 *
 * Conventions shared by every entry point
 * ---------------------------------------
 * State layout ("flattened multidimensional arrays", Listing 1 index order (j,k,l,i)):
 *   q[eq][z][y][x], x fastest, fp64, padded by ng = 3 cells on both sides of every ACTIVE dimension
 *   (buffers sized by the WENO order); an inactive dimension has extent 1.
 *   Equation order (NEQ = 2*n_fluids + ndim, reading B1):
 *     alpha_i rho_i (i = 1..n_fluids), rho u_d (d = 1..ndim), rho E, alpha_i (i = 1..n_fluids-1).
 *   mfc_layout() returns the padded extents and the element count of one such array.
 * Pointers: names ending in _dev are DEVICE pointers (e.g. a torch tensor's data_ptr()) on the device
 *   given to mfc_init; names ending in _host are HOST pointers.  The caller owns every buffer it passes;
 *   the library owns its scratch (two Runge-Kutta stage arrays, reduction workspace), allocated in mfc_init
 *   and released in mfc_destroy.
 * Boundary conditions: every evaluation of L first fills the ghost cells of its input array in memory
 *   (periodic wrap / zero-gradient copy of the nearest interior cell, corners included).  The ghost cells of q are
 *   therefore OVERWRITTEN by mfc_rhs and mfc_rk3_step (as SURVEY.md 8(b) specifies); their previous contents are never
 *   read.  Ghost entries of rhs are unspecified.
 * Tensor memory: the 3D kernel keeps its z window in tensor memory and allocates ALL 512 TMEM columns of every
 *   multiprocessor for as long as one of its blocks is resident (one block per multiprocessor).  A kernel of another
 *   stream or process that allocates tensor memory on the same device (any tcgen05 GEMM, e.g. a bf16 matmul) is
 *   serialised against it by the hardware allocator: it waits, results are unaffected.
 * Streams: `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work is
 *   enqueued on it.  Only mfc_cfl_dt, mfc_step_cfl, mfc_advance_host, mfc_profile_get and mfc_probe_dfma synchronise.
 * Errors: every function returns MFC_OK (0) or a negative mfc_status; nothing is thrown or printed.
 *   A context is not thread-safe.  State admissibility is not checked on the hot path: non-finite or
 *   inadmissible states propagate as NaN.  There is no CPU fallback: without a CUDA device mfc_init fails
 *   with MFC_ECUDA.
 */
#ifndef MFC_B200_H
#define MFC_B200_H

#ifdef __cplusplus
extern "C" {
#endif

/* Version of this binary interface: bumped whenever a struct below changes its layout or an entry point its signature
 * (3: mfc_grid.inv_dx, mfc_opts.abi_version, mfc_cfl_dt_static; 2: mfc_grid.edges_host, mfc_opts.staging, mfc_rhs takes a
 * non-const q_dev and overwrites its ghost cells).  mfc_abi_version() returns the value the loaded library was built with:
 * a caller compares it with the macro of the header it was compiled against before its first mfc_init (the Python binding
 * does so when it loads the library), and may also store the macro in mfc_opts.abi_version to have mfc_init refuse a
 * mismatch with MFC_EINVAL.
 * ZERO-INITIALISE every struct of this header before setting its fields (`mfc_grid g = {0};`, memset, calloc): fields added
 * by later versions mean "off" when zero, and mfc_init reads every field -- it dereferences edges_host[d] of each active
 * dimension when that pointer is not NULL, so a struct built on the stack without zeroing passes it a garbage pointer. */
#define MFC_ABI_VERSION 3

#define MFC_NG 3         /* ghost layers (WENO5) */
#define MFC_MAX_FLUIDS 3 /* compiled template set: ndim in {1,2,3} x n_fluids in {1,2,3} */

typedef enum {
    MFC_OK = 0,
    MFC_EINVAL = -1,       /* null pointer, bad shape, n_d < 3 in an active dimension, gamma <= 1, bad BC kind or order */
    MFC_EUNSUPPORTED = -2, /* (ndim, n_fluids) outside the compiled template set; kapila with n_fluids != 2; non-uniform
                              spacing with weno_order != 5 or with a non-positive ideal weight */
    MFC_ECUDA = -3,        /* CUDA runtime error (sticky); no device */
    MFC_ENOMEM = -4,       /* device or host allocation failed */
    MFC_ENONFINITE = -5,   /* mfc_advance_host: the CFL time step of the current state is NaN, infinite or zero */
    MFC_ELIMIT = -6        /* mfc_cfl_dt_static: the grid has more interior cells than MFC_STATIC_MAX_CELLS, the most the
                              library's fixed workspace serves; use a context (mfc_init + mfc_cfl_dt) for such a grid */
} mfc_status;

/* Cartesian grid, PAPER.md:105-124 (Eq. 6-9).  Uniform by default: dx_d = (hi_d - lo_d) / n_d.
 * Non-uniform spacing ("structured mesh with non-uniform spacing"; Listing 1's per-index coefficient tables;
 * Eq. 15 stretching): edges_host[d] != NULL gives the n[d] + 1 strictly increasing cell edges of dimension d (host
 * pointer, copied by mfc_init; lo[d], hi[d] are then ignored); dimensions may be mixed.  A ghost cell has the width of the
 * cell its value is copied from (periodic: widths wrap; extrapolation: the boundary cell's width); MFC_BC_HALO sides are
 * not supported in a non-uniform dimension (MFC_EUNSUPPORTED: the ghost widths would be the neighbour's).  WENO5 only
 * (weno_order 5); the ideal weights of every cell must be positive (true for smooth stretching), else MFC_EUNSUPPORTED. */
typedef struct {
    int ndim;        /* 1, 2 or 3 */
    int n[3];        /* interior cells; entries >= ndim are ignored (treated as 1) */
    double lo[3], hi[3];
    const double *edges_host[3]; /* NULL: uniform in that dimension */
    double inv_dx[3]; /* 0: 1 / dx_d = n_d / (hi_d - lo_d).  > 0 (uniform dimensions only): the reciprocal cell width itself.
                         For a block of a decomposed grid (MFC_BC_HALO): pass the GLOBAL n_d / (hi_d - lo_d),
                         so that every block, and the undivided grid, divides a face flux by the identical number; the
                         value recomputed from a block's own lo, hi can differ in the last bits from block to block */
} mfc_grid;

/* stiffened gas, PAPER.md:54-58 (Eq. 1) */
typedef struct {
    double gamma, pi_inf;
} mfc_fluid;

typedef enum {
    MFC_BC_PERIODIC = 0,
    MFC_BC_EXTRAP = 1,
    MFC_BC_HALO = 2 /* the ghost cells of this side belong to the caller: they hold a neighbouring block's cells (domain
                       decomposition) or any fill of the caller's own; the library reads them, never
                       writes them */
} mfc_bc_kind;

/* ghost-cell fills; periodic must be set on both sides of a dimension or on neither */
typedef struct {
    int lo[3], hi[3]; /* mfc_bc_kind per side of each dimension */
} mfc_bc;

typedef struct {
    double weno_eps;   /* WENO-JS epsilon, Eq. 12 / Listing 1; <= 0 selects 1e-16 */
    double cfl;        /* CFL number used by mfc_cfl_dt; <= 0 selects 0.3 */
    int device;        /* CUDA device ordinal; < 0 selects the current device */
    int march_segment; /* planes each block of the fused kernel marches along z (3D); <= 0 selects a heuristic */
    int weno_order;    /* reconstruction: 5 = WENO5-JS (0 selects it), 3 = WENO3-JS, 1 = piecewise
                          constant; the ghost width stays 3 whatever the order */
    int kapila;        /* != 0: Kapila model, the alpha row carries the source K div(u) with the two-fluid K of Eq. 2
                          (PAPER.md:52, 60-62), cell-centred, on the same face-velocity differences as alpha div(u);
                          needs n_fluids == 2 and volume fractions inside (0, 1).  0: Allaire model, K = 0 */
    int staging;       /* which 3D kernel runs: 0 = automatic: the kernel with specialised Z warps (TMA-staged;
                          even padded extent in x (n[0] even) and a 16-byte aligned q_dev), else the one-loop
                          kernel staged by TMA boxes (same layout conditions), else the one-loop kernel staged by per-thread
                          cp.async; 1 = one-loop kernel, TMA only; 2 = one-loop kernel, cp.async only; 3 = specialised Z
                          warps only.  A forced choice fails with MFC_ECUDA where it does not apply.  The one-loop kernels
                          compute the same bits; the kernel with Z warps sums the three directions in another order (last-bit
                          differences) */
    int abi_version;   /* 0 (not checked) or MFC_ABI_VERSION of the header the caller was compiled against: mfc_init returns
                          MFC_EINVAL when it differs from the library's */
} mfc_opts;

typedef struct mfc_ctx mfc_ctx;

/* Creates a context: validates (ndim, n_fluids) against the compiled template set, stores the EOS and BC
 * tables, allocates scratch (2 state-sized stage arrays).  eos: n_fluids entries.  opts may be NULL. */
int mfc_init(mfc_ctx **out, const mfc_grid *grid, int n_fluids, const mfc_fluid *eos, const mfc_bc *bc,
             const mfc_opts *opts);

void mfc_destroy(mfc_ctx *ctx);

/* Layout query: neq, ng, padded extents (x, y, z) and elements of one state array (neq * prod padded).
 * Any out pointer may be NULL. */
int mfc_layout(const mfc_ctx *ctx, int *neq, int *ng, long long padded_n[3], long long *elems);

/* L(q): one evaluation of the spatial operator, PAPER.md:105-130 (Eq. 6-10) with s(q) = 0 (K = 0 unless opts.kapila):
 *   cons->prim with ghost fill -> per direction WENO5-JS (Eq. 12,
 *   Listing 1) -> HLLC flux and face velocity (Eq. 13-14) ->
 *   rhs_k = sum_d (F_{k,-1/2} - F_{k,+1/2})/dx_d  [+ (alpha_i + K) sum_d (u_{+1/2} - u_{-1/2})/dx_d on alpha rows].
 * The ghost cells of q_dev are overwritten with the boundary fill, its interior is read; the interior of rhs_dev is
 * written.  q_dev and rhs_dev must not alias. */
int mfc_rhs(mfc_ctx *ctx, double *q_dev, double *rhs_dev, void *stream);

/* One 3-stage TVD Runge-Kutta step of size dt, in place on the interior of q_dev (ref. [19]):
 *   q1 = q + dt L(q);  q2 = 3/4 q + 1/4 (q1 + dt L(q1));  q <- 1/3 q + 2/3 (q2 + dt L(q2)).
 * On return the ghost cells of q_dev hold the boundary fill of the state the step STARTED from. */
int mfc_rk3_step(mfc_ctx *ctx, double *q_dev, double dt, void *stream);

/* The three stages of mfc_rk3_step one at a time (stage = 0, 1, 2, in this order), for callers that fill ghost cells
 * between the stages (MFC_BC_HALO: halo exchange with neighbouring blocks):
 *   stage 0 evaluates L on q_dev, stage 1 on the library's array q1, stage 2 on q2 (mfc_stage_array), and stage 2
 *   writes the result into q_dev.  The array a stage evaluates L on must have its HALO ghost cells filled first. */
int mfc_rk3_stage(mfc_ctx *ctx, int stage, double *q_dev, double dt, void *stream);
/* Device pointer of the library's stage array k = 1, 2 (q1, q2; `elems` doubles, the layout of q). */
int mfc_stage_array(mfc_ctx *ctx, int k, double **array_dev);

/* CFL-restricted time step: dt = cfl * min over interior cells and directions of
 * dx_d / (|u_d| + c), c the frozen mixture sound speed (dx_d the cell's own width).  Synchronises `stream`; writes one
 * host double.  A cell whose signal speed is not finite (NaN input, negative c^2, zero density) makes the result NaN:
 * the reduction keeps NaN, it does not drop it; the call still returns MFC_OK. */
int mfc_cfl_dt(mfc_ctx *ctx, const double *q_dev, double *dt_host, void *stream);

/* mfc_cfl_dt followed by mfc_rk3_step with that time step, as one call: q_dev advances by the CFL step of the state it
 * holds; *dt_host (may be NULL) receives the step taken.  Same kernels, same bits as the two calls.  The host needs dt before
 * it can launch the first stage, so the call waits once for the reduction; the ghost fill of the first stage (which does not
 * depend on dt) is enqueued before that wait, so the device is busy during the round trip -- at 128^3 the pair of calls
 * leaves it idle for 3 % of a step.  A time step that is NaN, infinite or not positive is not taken: MFC_ENONFINITE, the
 * interior of q_dev untouched (its ghost cells filled), *dt_host holding the offending value. */
int mfc_step_cfl(mfc_ctx *ctx, double *q_dev, double *dt_host, void *stream);

/* The same time step for callers that cannot allocate device memory -- no context, no cudaMalloc, no synchronisation.
 * Meant for: code that runs inside an application whose own memory pool already owns the device (a further cudaMalloc
 * fails or eats into what the application budgeted), time loops with other streams in flight (cudaMalloc / cudaFree
 * stall the whole device), and plug-ins that are given buffers and a stream and may only enqueue work.  Such callers
 * cannot call mfc_init, which allocates the stage arrays and the reduction workspace.
 *   grid, n_fluids, eos: as for mfc_init (host pointers, read during the call); uniform spacing only (edges_host must be
 *     NULL: MFC_EUNSUPPORTED otherwise).  cfl <= 0 selects 0.3.  device < 0 selects the current device.
 *   q_dev: the state, layout above, on `device`; only interior cells are read.  dt_dev: ONE double on `device`, written by
 *     the kernel on `stream`; the call does not wait for it (NaN propagates as for mfc_cfl_dt).  Both belong to the caller.
 * Workspace: one partial maximum per block of MFC_STATIC_CELLS_PER_BLOCK cells plus a counter, in a fixed
 *   `static __device__` array of MFC_STATIC_SCRATCH_BYTES that every device holding the library keeps until the process
 *   exits.  A grid with more than MFC_STATIC_MAX_CELLS interior cells is refused with MFC_ELIMIT before anything is
 *   launched (256^3 and 320^3 fit, 384^3 does not).
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress); make it before any stream capture
 *   begins.  Later calls enqueue one 8-byte memset (the counter starts every launch at zero) and one kernel.
 * Sharing: every call on a device uses the same array, which keeps the previous call's contents.  Calls whose kernels
 *   could run at the same time on one device (different streams without an event between them, or several host threads
 *   doing so) race on it and return garbage; calls ordered on the GPU are safe, from any thread.
 * Returns the same bits as mfc_cfl_dt for the same grid, fluids, cfl and state. */
#define MFC_STATIC_CELLS_PER_BLOCK 4096
#define MFC_STATIC_MAX_BLOCKS 8192
#define MFC_STATIC_MAX_CELLS (MFC_STATIC_CELLS_PER_BLOCK * MFC_STATIC_MAX_BLOCKS) /* 33 554 432 */
#define MFC_STATIC_SCRATCH_BYTES (8 * (32 + MFC_STATIC_MAX_BLOCKS))               /* 65 792 */
int mfc_cfl_dt_static(const mfc_grid *grid, int n_fluids, const mfc_fluid *eos, double cfl, int device,
                      const double *q_dev, double *dt_dev, void *stream);

/* Whole path from HOST memory: copies q_host to the device, takes nsteps RK3 steps (each with
 * dt = dt_fixed if dt_fixed > 0, else the CFL step of the current state), copies the state back into
 * q_host and synchronises.  t_host (may be NULL) receives the sum of the steps taken.
 * q_host: `elems` doubles in the layout above; pinned memory makes the copies asynchronous.
 * With dt_fixed <= 0, a step whose CFL time step is not finite and positive is not taken: MFC_ENONFINITE is returned
 * and q_host is left untouched. */
int mfc_advance_host(mfc_ctx *ctx, double *q_host, int nsteps, double dt_fixed, double *t_host, void *stream);

/* ---- stage outputs, for parity tests of the individual steps of the path ---- */

/* a0 + a1: primitive array w = (alpha_i rho_i, u_d, p, alpha_i) on the whole padded box, ghost cells taken
 * from the wrapped / clamped interior cell of q_dev.  w_dev: `elems` doubles. */
int mfc_cons_to_prim(mfc_ctx *ctx, const double *q_dev, double *w_dev, void *stream);

/* a2 + a3 on one line of primitives with normal direction dir (0,1,2 < ndim), using the same device
 * functions as the sweeps.  w_dev: [neq][n + 6]; vL_dev, vR_dev: [neq][n + 2] (cells -1..n: state at face
 * i+1/2 resp. i-1/2 seen from cell i); F_dev: [neq][n + 1]; uface_dev: [n + 1] (faces -1/2 .. n-1/2).
 * On a non-uniform grid the line is one of the grid's own lines of that direction: n must equal n[dir]. */
int mfc_line_fluxes(mfc_ctx *ctx, int dir, int n, const double *w_dev, double *vL_dev, double *vR_dev,
                    double *F_dev, double *uface_dev, void *stream);

/* ---- measurement hooks ---- */

typedef enum {
    MFC_K_RHS = 0,  /* the fused right-hand side: ghost fill, cons->prim, WENO5 + HLLC in every direction,
                       flux difference and RK stage combine in one launch */
    MFC_K_CFL = 1,  /* CFL reduction */
    MFC_K_PRIM = 2, /* stage output of mfc_cons_to_prim (parity tests only; not on the path) */
    MFC_K_GHOST = 3, /* ghost fill in memory, once before every evaluation of L */
    MFC_K_COUNT = 4
} mfc_kernel_id;

/* With profiling on, every kernel launch is bracketed by CUDA events on its own stream. */
int mfc_profile_enable(mfc_ctx *ctx, int on);
/* Synchronises outstanding event pairs, then returns launches and summed device milliseconds of one kernel
 * family since the last reset.  reset != 0 clears the accumulators of that family afterwards. */
int mfc_profile_get(mfc_ctx *ctx, int kernel_id, long long *launches, double *total_ms, int reset);
/* Number of kernels this context has launched since mfc_init (all families). */
long long mfc_launch_count(const mfc_ctx *ctx);

/* FP64 FMA micro-benchmark (register-resident dependent DFMA chains on every SM) used as the measured
 * ALU roofline denominator.  Returns TFLOP/s (2 flops per DFMA) and the launch time in ms. */
int mfc_probe_dfma(int device, double *tflops_host, double *ms_host);

const char *mfc_strerror(int code);
/* Text of the CUDA runtime error behind the last MFC_ECUDA / MFC_ENOMEM a kernel launch of this context returned. */
const char *mfc_cuda_error(const mfc_ctx *ctx);
const char *mfc_version(void);
/* MFC_ABI_VERSION of the loaded library (see the top of this header). */
int mfc_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MFC_B200_H */
