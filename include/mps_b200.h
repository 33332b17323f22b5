/* mps_b200.h -- C-ABI of libmps_b200.so: the MPS time-step particle-interaction
 * path of arXiv 2105.01677 as hand-written sm_100a CUDA kernels.
 *
 * Citations: "P:n" = line n of the paper text; "Qk" = reading k in
 * DESIGN.md section 3 (where the paper is silent, ambiguous or garbled).
 *
 * Conventions for every entry point
 *  - Returns int: MPS_OK (0) or a negative MPS_ERR_*.  No exception crosses the
 *    ABI, nothing aborts, nothing prints.  mps_last_error() gives a message.
 *  - "device pointer" = address in CUDA global memory of the current device,
 *    owned by the caller (e.g. a torch tensor); "host pointer" = ordinary host
 *    memory.  The library copies what it needs and never keeps a caller pointer.
 *  - All floating point data are IEEE fp64.  Particle arrays passed in or out
 *    with order = MPS_ORDER_ORIGINAL are indexed by the caller's particle index
 *    (the index at mps_init); with MPS_ORDER_SORTED by the library's current
 *    cell-sorted slot (see mps_bin).
 *  - Kernel launches are asynchronous on the ctx's stream.  Device-side error
 *    flags (neighbour overflow, non-finite position) are read and returned by
 *    mps_sync, mps_get_stats, mps_pressure_ppe and mps_step.
 *  - A ctx is not thread-safe.  There is no CPU fallback: every call needs a
 *    CUDA device of compute capability 10.0 (B200).
 *  - Every entry point that launches work opens an NVTX range of its own name.
 *  - Environment variables read at mps_init (development switches; the defaults are what is
 *    measured and tested): MPS_B200_ROWS=lean|warp|cell picks the neighbour-row builder (default: by
 *    size and key_mode; all builders give identical rows), MPS_B200_CG_TEX=0 turns the texture path
 *    of the matrix-free gathers off, MPS_B200_CG_TIMEOUT_CYCLES=<n> sets the spin limit of the
 *    grid barrier inside the persistent CG kernel (default 4e9 SM cycles, 0 = no limit; raise it
 *    or set 0 under compute-sanitizer or a debugger), MPS_B200_CARRY=0 makes mps_step bin twice per
 *    step as if row_skin < 0 (see mps_step), MPS_B200_COND=0 captures the skin bins of mps_step as plain kernel
 *    nodes that return at once instead of conditional graph nodes (the default whenever CUDA_INJECTION64_PATH is
 *    set, i.e. under a profiler: Nsight Compute cannot see kernels of a graph that holds conditional nodes).
 */
#ifndef MPS_B200_H
#define MPS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mps_ctx mps_ctx;

enum {
  MPS_OK = 0,
  MPS_ERR_ARG = -1,                /* null pointer, n <= 0, r_e <= 0, dt <= 0, unsupported option */
  MPS_ERR_CUDA = -2,               /* CUDA runtime error; string in mps_last_error */
  MPS_ERR_NEIGHBOUR_OVERFLOW = -3, /* a particle has more than max_neighbours neighbours */
  MPS_ERR_NOCONV = -4,             /* CG reached cg_maxit; pressures are still written */
  MPS_ERR_NONFINITE = -5,          /* NaN/Inf position, or two coincident particles (Eq. 3 infinite) */
  MPS_ERR_ORDER = -6               /* call made before its prerequisite (e.g. density before bin) */
};

/* particle types ("fluid or boundary p.", "dummy p."; Q3) */
enum { MPS_FLUID = 0, MPS_WALL = 1, MPS_DUMMY = 2, MPS_GHOST = 3 };

enum { MPS_ORDER_ORIGINAL = 0, MPS_ORDER_SORTED = 1 };
enum { MPS_ROUTE_EXPLICIT = 0, MPS_ROUTE_PPE = 1 };
enum { MPS_RADIUS_N = 0, MPS_RADIUS_LAP = 1 };

/* field ids for mps_get_field / mps_set_field.  0..21 are fp64, 32..35 int32. */
enum {
  MPS_F_X = 0, MPS_F_Y = 1, MPS_F_Z = 2,       /* position r */
  MPS_F_U = 3, MPS_F_V = 4, MPS_F_W = 5,       /* velocity u */
  MPS_F_N = 6,                                 /* particle number density n_i (Eq. 5) */
  MPS_F_P = 7,                                 /* pressure */
  MPS_F_AX = 8, MPS_F_AY = 9, MPS_F_AZ = 10,   /* nu lap(u) + g (Eq. 2, Eq. 10) */
  MPS_F_NUT = 11,                              /* Smagorinsky eddy viscosity (Eq. 13, Q10) */
  MPS_F_B = 12,                                /* PPE right-hand side (Eq. 8, Q5) */
  MPS_F_PHAT = 13,                             /* neighbourhood minimum pressure (Eq. 14, Q12) */
  MPS_F_GX = 14, MPS_F_GY = 15, MPS_F_GZ = 16, /* pressure gradient */
  MPS_F_XCG = 17,                              /* CG solution before the clamp (Q4) */
  MPS_F_DNDT = 18,                             /* Dn/Dt of the last mps_dndt (Eq. 15, Q22) */
  MPS_F_NK = 19, MPS_F_DNDTK = 20,             /* n and Dn/Dt kept from the start of the step (Eq. 17) */
  MPS_F_RHOS = 21,                             /* smoothed density <rho> of the multi-density model (Q25) */
  MPS_I_TYPE = 32, MPS_I_PHASE = 33,
  MPS_I_BC = 34,                               /* -1 dummy/ghost, 1 free surface, 0 PPE unknown (Eq. 6) */
  MPS_I_KEY = 35                               /* cell key of the last mps_bin (read only) */
};

/* Parameters: a POD struct copied at mps_init.  Every reading of DESIGN.md
 * section 3 is a field here.  Defaults in parentheses are what the tests use. */
typedef struct mps_params {
  int32_t dim;              /* 3, or 2 (P:292 item 1): d of Eq. 10/14 and the lattice sums of n0, lambda;
                               in 2D the caller keeps z constant, w = 0 and g[2] = 0 */
  int32_t n_phases;         /* 1 or 2 */
  int32_t cg_maxit;         /* (2000) then MPS_ERR_NOCONV; Q15 */
  int32_t grad_variant;     /* 0: (p_j - phat_i) standard [8]; 1: Eq. 14 as printed; 2: (p_i + p_j); Q13;
                               3: multi-density term of the weakly-compressible model, Eq. 11-12; Q25 */
  int32_t clamp_negative_p; /* (1) p < 0 -> 0 after either pressure route; Q4 */
  int32_t rho_pair_mean;    /* 0 arithmetic (default), 1 harmonic; Q6 */
  int32_t nu_pair_mean;     /* 1 harmonic (default), 0 arithmetic; Q9 */
  int32_t key_mode;         /* (0) 0: linear cell key c_x + n_x (c_y + n_y c_z); 1: Morton key, bit k of c_x, c_y, c_z
                               at bits 3k, 3k+1, 3k+2 (3 x 10-bit interleave; at most 512 cells per axis): the key
                               space then has 8^bits entries, bits = ceil(log2(max n_a)), ghosts get 8^bits, and
                               mps_get_grid / mps_get_cell_start report that size */
  int32_t cell_div;         /* (1) cell side h = max(re_n, re_lap) / cell_div; 1..3 */
  int32_t max_neighbours;   /* (300) P:286; capacity of one neighbour row */
  int32_t ppe_source;       /* (0) 0: Eq. 8; 1: higher-order source, Eq. 15 (MPS-HS); 2: HS plus the
                               error-compensating parts, Eq. 17-18 (ECS); Q22 */
  int32_t ppe_laplacian;    /* (0) 0: Eq. 10 form of Listing 2; 1: higher-order Laplacian, Eq. 16 (MPS-HL); Q23 */
  int32_t kernel;           /* (0) 0: w = re/r - 1 (Eq. 3); 1: w = (1 - r/re)^3 (Eq. 4, the paper's
                               recommendation for the explicit route); n0 and lambda follow the kernel */
  int32_t rebin_every;      /* (1) 1: exact neighbour sets at both bins of every step (Q7).  K > 1: the paper's
                               list reuse: mps_step bins once every K steps, at r^k, and every
                               sweep keeps the stored pairs whose current distance is below the radius; Q24 */
  int32_t ppe_operator;     /* (1) how the CG applies A of Listing 2.  0: matrix-free -- rows hold
                               neighbour indices only and every application recomputes c_ij from the positions
                               (inside mps_step with a skin: from an exact index list filtered once per solve);
                               1: assembled -- the coefficients of the rows bc = 0 are computed once per solve
                               (positions are fixed during a solve) into a compact ELL matrix over the unknowns
                               (one 64-bit word per pair: 24-bit column + 40-bit fixed-point coefficient, Q28; the
                               paper's poiss[] of P:272-282 without its N x 300 stride over all particles) and
                               every application streams it.  Same operator, same parity bars; needs n < 2^24. */
  int32_t cg_warm_start;    /* (0) 1: CG starts from the previous step's pressure of the particle (x0 = p^k on
                               the rows bc = 0) instead of x0 = 0 (Q15); one extra operator application per solve */
  double l0;                /* initial particle spacing */
  double re_n;              /* radius for density, p-hat and gradient (2.1 l0) */
  double re_grad;           /* must equal re_n (one list serves both) */
  double re_lap;            /* radius for the Laplacian: viscosity and PPE (3.1 l0); >= re_n */
  double dt;
  double g[3];
  double rho[2];            /* density per phase */
  double nu[2];             /* kinematic viscosity per phase */
  double c0;                /* speed of sound of Eq. 7; Q14 */
  double gamma;             /* (7) Eq. 7 */
  double beta;              /* (0.97) Eq. 6 */
  double compress;          /* (1e-7) diagonal term compress/dt^2, Listing 2; Q5 */
  double ppe_relax;         /* (1.0) factor on the PPE source */
  double cg_rtol;           /* (1e-8) stop at ||r|| <= cg_rtol ||b||; Q15 */
  double cs;                /* Smagorinsky constant, 0 = off; Q10 */
  double domain_min[3];     /* particles outside [domain_min, domain_max) become GHOST; Q11 */
  double domain_max[3];
  double n0_n;              /* 0 => lattice closed form (Q1) */
  double n0_lap;            /* 0 => lattice closed form */
  double lambda;            /* 0 => lattice closed form */
  double row_skin;          /* Verlet skin of mps_step's neighbour rows in units of l0 (Q26): the rows are built
                               with both radii enlarged by row_skin * l0 and serve every sweep -- each re-tests
                               r2 < re^2 with the rounding of Q2, so the sets stay exact -- until some particle has
                               moved by more than 0.45 skins since the build (checked on the device by the predictor
                               and the corrector).  0 => the library chooses: 0.1, and 0.3 while a flow needs more
                               than 0.4 bins per step with 0.1 (looked at over windows of at least 16 steps, between
                               mps_step calls and, with one 4-byte read-back, inside long ones; back to 0.1 below 0.06 bins per step, and above 0.8, where neither
                               skin saves a bin and the thin one has the shorter sweeps); < 0 => no skin: mps_step
                               bins at r^k and at r* in every step, as Q7 is literally stated */
} mps_params;

typedef struct mps_stats {
  int32_t cg_iters;         /* iterations of the last mps_pressure_ppe */
  int32_t cg_converged;
  double cg_relres;         /* sqrt(r.r / b.b) of the recurrence residual at exit */
  int32_t max_neighbours;   /* largest r_lap row of the last mps_bin */
  int32_t n_surface;        /* free-surface particles of the last PPE */
  int32_t n_ghost;          /* particles currently GHOST */
  int32_t n_rows;           /* PPE unknowns (bc == 0) of the last PPE */
  int64_t cg_iters_total;   /* summed over the life of the ctx */
  int64_t steps_total;
  int32_t device_error;     /* sticky MPS_ERR_* raised on the device, 0 if none */
  int32_t cg_noconv_total;  /* solves that hit cg_maxit, summed over the life of the ctx */
  double cg_setup_ms;       /* last solve, timed on the device (%globaltimer, block 0): flags, rhs,
                               compaction and (ppe_operator 1) assembly ... */
  double cg_loop_ms;        /* ... and the CG iterations alone */
  double cg_loop_ms_total;  /* cg_loop_ms summed over the life of the ctx */
  int64_t cg_nnz;           /* ppe_operator 1: off-diagonal entries of the matrix assembled by the last solve */
  int64_t bins_total;       /* bins (sort + neighbour rows) run over the life of the ctx: two per step of mps_step
                               without a skin; with one (row_skin), only when a particle has moved 0.45 skins */
  double row_skin_now;      /* the skin mps_step currently builds its rows with, in units of l0 (-1: none) */
} mps_stats;

/* mps_init: create a ctx and copy n particles in (device pointers, caller's
 * order).  type: MPS_FLUID/WALL/DUMMY/GHOST, phase: 0/1.  Allocates every
 * buffer any later call needs (nothing is allocated after init).  stream is a
 * cudaStream_t (may be NULL = default stream).  Computes n0 and lambda on the
 * ideal cubic lattice unless given (I1-I4 of DESIGN.md section 2; P:134-136,
 * P:170-174). */
int mps_init(mps_ctx** out, const mps_params* prm, int64_t n,
             const double* x, const double* y, const double* z,
             const double* u, const double* v, const double* w,
             const int32_t* type, const int32_t* phase, void* stream);

/* Same, from HOST pointers (pageable or pinned); copies are issued on the stream. */
int mps_init_host(mps_ctx** out, const mps_params* prm, int64_t n,
                  const double* x, const double* y, const double* z,
                  const double* u, const double* v, const double* w,
                  const int32_t* type, const int32_t* phase, void* stream);

int mps_destroy(mps_ctx* ctx);

/* mps_bin: uniform-grid binning (section 4.1).  Cell index
 * c_a = floor((x_a - domain_min_a) * (1/h)); key = c_x + n_x (c_y + n_y c_z);
 * out-of-domain or non-finite particles become GHOST with key = n_cells.
 * Counting sort by key (ties: ascending original index), cell-start table,
 * physical reorder of the particle arrays, and the per-step neighbour rows at
 * re_lap (entries within re_n first) that every later sweep streams (Listing 2's
 * neigh[], without its fixed N x 300 matrix).  Distance test:
 * r2 = (dx*dx + dy*dy) + dz*dz, each operation rounded, r2 < re*re (Q2). */
int mps_bin(mps_ctx* ctx);

/* mps_density: n_i = sum_{j != i, r < re_n} (re_n / r - 1) over non-ghost j
 * (Eq. 5 with P:123 Eq. 3).  Needs mps_bin at the current positions. */
int mps_density(mps_ctx* ctx);

/* mps_viscosity: a_i = (2 d / (n0 lambda)) sum nu_ij (u_j - u_i) w(r) + g for
 * fluid i over r < re_lap (Eq. 10, Eq. 2); if cs > 0 first the
 * Smagorinsky nu_t (Eq. 13; Q9, Q10).  Walls and dummies have u = 0. */
int mps_viscosity(mps_ctx* ctx);

/* mps_predict: u* = u + dt a; r* = r + dt u* for fluid (Q8).
 * Invalidates the bin. */
int mps_predict(mps_ctx* ctx);

/* mps_pressure_explicit: p = rho c0^2 / gamma ((n/n0)^gamma - 1) for fluid and
 * wall, 0 for dummy (Eq. 7; Q4).  Uses the ctx's n field. */
int mps_pressure_explicit(mps_ctx* ctx);

/* mps_pressure_ppe: free-surface flags n < beta n0 (Eq. 6), right-hand
 * side (Eq. 8 divided by -rho; Q5), matrix-free operator with the
 * structure of Listing 2 and conjugate gradients from x0 = 0 to
 * ||r|| <= cg_rtol ||b|| (Eq. 9; Q15).  iters_out / relres_out are
 * HOST pointers (may be NULL), written after a stream synchronisation.
 * Returns MPS_ERR_NOCONV if cg_maxit was reached (pressures still written). */
int mps_pressure_ppe(mps_ctx* ctx, int32_t* iters_out, double* relres_out);

/* mps_smooth_density: <rho>_i = sum_j rho_j w / sum_j w over N(i, re_n) at the current positions
 * ("set for each particle before starting the simulation"; Q25); the value follows its
 * particle through later sorts.  mps_step calls it once, before the first step, when
 * grad_variant = 3.  Needs mps_bin. */
int mps_smooth_density(mps_ctx* ctx);

/* mps_dndt: Dn/Dt_i = -sum_{j in N(i, re_n)} re_n / r^3 (x_ij . u_ij) at the current positions
 * and velocities, every non-ghost i (Eq. 15, the material derivative of Eq. 5; sign:
 * Q22).  keep = 0 writes MPS_F_DNDT; keep = 1 writes MPS_F_DNDTK and copies the ctx's n field to
 * MPS_F_NK (the start-of-step values of Eq. 17).  Needs mps_bin at the current positions. */
int mps_dndt(mps_ctx* ctx, int32_t keep);

/* mps_gradient: p-hat (minimum over i and its non-dummy neighbours within re_n;
 * P:215, Q12) then the pressure gradient of fluid i, variant grad_variant
 * (Eq. 14; Q13).  Variant 3: G_i = rho_i (d/n0) sum ((<rho>_j/<rho>_i) alpha_j - alpha_i)/r^2
 * (r_j - r_i) w, alpha = p/rho (Eq. 11-12; Q25), no p-hat. */
int mps_gradient(mps_ctx* ctx);

/* mps_correct: u = u* - (dt / rho_i) G; r = r* + dt (u - u*) for fluid; walls
 * and dummies do not move (Q8, Q3, Q11).  Invalidates the bin. */
int mps_correct(mps_ctx* ctx);

/* mps_step: nsteps times { bin, [ppe_source 2: density, dndt(keep)], viscosity, predict, bin,
 * density, [ppe_source >= 1: dndt], pressure (route), gradient, correct }.  Every sweep sees the exact
 * neighbour set of the positions it works at (Q7).  How the library gets there (Q26): a bin of mps_step
 * runs on an internal grid with cells of (max re + skin) / cell_div and builds rows with both radii
 * enlarged by the skin (row_skin * l0), and remembers the positions it was made at.  Every sweep re-tests
 * r2 < re^2 with the rounding of Q2, so the sets are exact as long as no particle is further than 0.45
 * skins from its position at the build.  The predictor and the corrector check exactly that for every
 * particle they move (and that none left the domain or became non-finite) and raise a flag ON THE DEVICE;
 * the kernels of the two bins of a step are always launched and return at once unless the flag is up, so
 * the host never waits for the device inside mps_step.  GHOST decisions always use mps_bin's grid.
 * The launches of a step are replayed from CUDA graphs when the ctx has its own stream.  With
 * row_skin < 0 both bins run in every step on mps_bin's grid with the exact radii.
 * Returns the first error met. */
int mps_step(mps_ctx* ctx, int32_t nsteps, int32_t pressure_route);

/* mps_step_host: the end-to-end call on HOST buffers: init from host arrays,
 * nsteps steps, copy x,y,z,u,v,w,p (caller's order) back into the same host
 * arrays (p_out may be NULL), destroy.  All copies are inside the call. */
int mps_step_host(const mps_params* prm, int64_t n, double* x, double* y, double* z,
                  double* u, double* v, double* w, const int32_t* type, const int32_t* phase,
                  double* p_out, int32_t nsteps, int32_t pressure_route, mps_stats* stats_out,
                  void* stream);

/* mps_upload_host / mps_download_host: the per-step host boundary of an existing
 * ctx (no allocation).  upload replaces all n particles from HOST arrays in the
 * caller's order (as mps_init_host does; invalidates the bin); download writes
 * x,y,z,u,v,w and p (caller's order; any pointer may be NULL) to HOST arrays and
 * synchronises the stream.  Pinned buffers make the copies asynchronous. */
int mps_upload_host(mps_ctx* ctx, const double* x, const double* y, const double* z,
                    const double* u, const double* v, const double* w,
                    const int32_t* type, const int32_t* phase);
int mps_download_host(mps_ctx* ctx, double* x, double* y, double* z,
                      double* u, double* v, double* w, double* p);

/* Field access for parity tests and checkpoints.  dst/src are DEVICE pointers
 * to n elements (double for ids < 32, int32_t otherwise).  Positions, velocities, type, phase and the
 * fields an option carries per particle (MPS_F_NK, MPS_F_DNDTK, MPS_F_RHOS) follow their particle
 * through every sort; every other field is the result of the last call that computed it and is only
 * meaningful until the next mps_bin (inside mps_step: MPS_F_AX..AZ and MPS_F_NUT belong to the
 * step's first bin and are not valid after the step). */
int mps_get_field(mps_ctx* ctx, int32_t field, void* dst, int32_t order);
int mps_set_field(mps_ctx* ctx, int32_t field, const void* src, int32_t order);

/* perm[k] = caller's original index of sorted slot k (DEVICE, n x uint32). */
int mps_get_perm(mps_ctx* ctx, uint32_t* dst);
/* grid[0..2] = cells per axis, grid[3] = n_cells (HOST, 4 x int32). */
int mps_get_grid(mps_ctx* ctx, int32_t* grid);
/* cell_start[c] = first sorted slot of cell c, c = 0..n_cells (DEVICE, (n_cells+1) x uint32). */
int mps_get_cell_start(mps_ctx* ctx, uint32_t* dst);
/* Neighbour sets of the last mps_bin as CSR in ORIGINAL numbering, each row
 * ascending: counts[i] (DEVICE, n x uint32) and, if idx != NULL, the first cap
 * entries of the concatenated rows (DEVICE).  *total (HOST) = number of entries.
 * After mps_step with a skin: the sets at the CURRENT positions as the next sweep would see them
 * (the stored rows filtered by the re-test), provided the rows are still valid -- else MPS_ERR_ORDER. */
int mps_get_neighbours(mps_ctx* ctx, int32_t radius_id, uint32_t* counts, uint32_t* idx,
                       int64_t cap, int64_t* total);
/* y = A x with the operator and flags of the last mps_pressure_ppe (DEVICE, n doubles each). */
int mps_ppe_apply(mps_ctx* ctx, const double* x, double* y, int32_t order);
/* out[0..5] = n0_n, n0_lap, lambda, 2d/(n0_lap lambda), h, 1/h (HOST). */
int mps_get_constants(mps_ctx* ctx, double* out);
int mps_get_stats(mps_ctx* ctx, mps_stats* out);
int mps_sync(mps_ctx* ctx);
/* Per-kernel CUDA-event timing for bench.py (the one call that allocates after mps_init: the first
 * mps_timers_enable with a non-zero mask creates a pool of 8192 CUDA events): mps_timers_enable(ctx, mask) with
 * bit k of mask set times every launch of category k with a CUDA-event pair on
 * the ctx's stream (mask 0 switches timing off); mps_timers_read returns the
 * accumulated milliseconds and launch counts (HOST arrays of MPS_NUM_TIMERS). */
enum {
  MPS_T_BIN_SORT = 0, MPS_T_BIN_LIST = 1, MPS_T_VISCOSITY = 2, MPS_T_PREDICT = 3,
  MPS_T_DENSITY = 4, MPS_T_PRESSURE_EXPLICIT = 5, MPS_T_PPE_SETUP = 6, MPS_T_CG_SPMV = 7,
  MPS_T_CG_UPDATE = 8, MPS_T_GRADIENT = 9, MPS_T_CORRECT = 10, MPS_NUM_TIMERS = 11
};
int mps_timers_enable(mps_ctx* ctx, int32_t mask);
int mps_timers_read(mps_ctx* ctx, double* ms, int64_t* launches);
/* Kernels launched by this ctx so far: every __global__ launch issued by the host, plus the kernels of the skin
 * bins that ran as bodies of conditional graph nodes (counted on the device; as of the last mps_step / mps_sync /
 * mps_get_stats, which read the counter).  A bin that did not run is not counted.  While timers are on
 * (mps_timers_enable) mps_step reads the device flag before each of its bins and leaves out the ones not needed. */
int64_t mps_launch_count(mps_ctx* ctx);
/* mps_cell_start_noalloc: the cell-start table of the counting sort (section 4.1; B4 of DESIGN.md section 2)
 * for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * cell_start[c] = number of keys below c, c = 0 .. n_cells -- the same table as mps_get_cell_start after mps_bin.
 * key: DEVICE, n x uint32, the cell keys in any order (a key above n_cells counts as n_cells, the ghost key);
 * cell_start: DEVICE, (n_cells + 1) x uint32, written by the call; stream: cudaStream_t of the current device (may
 * be NULL).  Needs no ctx and calls no cudaMalloc, cudaFree or allocating routine: the histogram and the scan's tile
 * sums live in a file-scope device array of fixed size (1.0 MB, held by every GPU that loads the library until the
 * process exits), which limits n_cells to mps_cell_start_noalloc_max_cells() = 262,144; a larger n_cells returns
 * MPS_ERR_ARG.  Every call shares that array and clears the part it uses on the caller's stream: calls that overlap
 * on the GPU (two streams, two threads) race -- serialise them.  Asynchronous; errors: MPS_ERR_ARG, MPS_ERR_CUDA,
 * message from mps_cell_start_noalloc_error() (valid until the next failing call). */
int mps_cell_start_noalloc(const uint32_t* key, int64_t n, int32_t n_cells, uint32_t* cell_start, void* stream);
int32_t mps_cell_start_noalloc_max_cells(void);
const char* mps_cell_start_noalloc_error(void);
/* Message of the last error of this ctx (owned by the ctx; valid until the
 * next call).  ctx == NULL returns the message of the last failed mps_init. */
const char* mps_last_error(mps_ctx* ctx);
const char* mps_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MPS_B200_H */
