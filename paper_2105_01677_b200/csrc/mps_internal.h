// mps_internal.h -- internal ctx layout and launch helpers of libmps_b200.so.
// Not part of the ABI.  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/mps_b200.h"

// ---- data layout in HBM (all arrays in cell-sorted slot order) ---------------
// pos4[i] = (x, y, z, s): one 32-byte sector per particle, so a neighbour gather
//           is exactly one sector.  s is the scalar the current sweep gathers
//           (pressure for the gradient, CG residual for the PPE operator).
// vel4[i] = (u, v, w, nu_eff): nu_eff < 0 marks WALL/DUMMY (u = 0, nu_ij = nu_i).
// tp[i]   = type | phase << 8.
// oid[i]  = caller's original index of slot i (= perm).
// nbr     = neighbour rows, row-major ELL: row of slot i starts at nbr + i * stride
//           (stride = max_neighbours + 14 rounded up to a multiple of 8, so every
//           row starts on a 32-byte sector and the two parts never share one).
//           Entries with r < re_n fill the row from the front (count cn[i],
//           ascending slot order); entries with re_n <= r < re_lap fill it from the
//           back in whole sectors (count co[i], see back_slot).  The L lanes that
//           share a row read L consecutive entries.  Entry = slot index of j
//           | NB_DUMMY if j is a dummy | NB_PHASE1 if j is of phase 1 | NB_WALL if
//           j is a wall particle.
#define NB_DUMMY 0x80000000u
#define NB_PHASE1 0x40000000u
#define NB_WALL 0x20000000u
#define NB_INDEX 0x1fffffffu
#define ROW_NONE 0xffffffffu     // rowmap: dummy / ghost (bc = -1)
#define ROW_SURFACE 0xfffffffeu  // rowmap: free surface (bc = 1)

// position of back entry kk (0-based) in a row of `stride` entries
__host__ __device__ __forceinline__ uint32_t back_slot(int stride, uint32_t kk) {
  return (uint32_t)stride - 8u * (kk / 8u + 1u) + (kk & 7u);
}

struct CgScalars {  // what the persistent CG kernel reports at exit (block 0)
  double gamma;                 // r.r of the last iteration
  double bb, tol2bb;            // b.b and cg_rtol^2 b.b
  int iters, done, converged, maxit;
  int n_surface, n_rows;
  int noconv_total, pad;        // solves that hit maxit since the ctx was made
  long long iters_total;        // iterations since the ctx was made
  unsigned long long t_setup_ns, t_loop_ns;  // %globaltimer of block 0: setup (+ assembly) and the CG loop
  unsigned long long t_loop_ns_total;
  unsigned long long nnz;       // entries of the assembled operator (ppe_operator 1)
};

// Grid-wide barrier state of the persistent CG kernel (zeroed before every launch).
struct GridBar {
  unsigned int count;    // arrivals since the launch (monotonic; a barrier waits for nb x generation)
  unsigned int timeout;  // a spin exceeded the limit: the kernel drained instead of hanging
};

struct DevFlags {
  int overflow;       // some row exceeded the capacity
  int nonfinite;      // NaN/Inf position or coincident pair
  int max_row;        // largest r_lap row
  int n_ghost;
  // mps_step with a skin (Q26): "the rows in nbr no longer cover the positions" -- raised by the corrector
  // (need_k: read by the predicated bin at the start of the next step, cleared by the predictor) and by the
  // predictor (need_star: read by the predicated bin at r*, cleared by the corrector) when a particle is
  // further than 0.45 skins from its position at the last build, left the domain or is non-finite
  int need_k;
  int need_star;
  int bins;           // predicated bins that actually ran
  int cond_taken;     // ... of which as the body of a conditional graph node (their launches are counted from this)
};

struct KConst {  // by-value kernel parameter
  double re_n, re_n2, re_lap, re_lap2;
  double n0_n, n0_lap, lam, A_lap;
  double dt, g[3];
  double rho[2], nu[2];
  double c0, gamma, beta, compress_dt2, relax_dt2;
  double cs_l0_sq, d_over_n0;
  double inv_rho_pair[2][2];  // 1 / rho_ij by the phases of i and j (arithmetic or harmonic mean, Q6)
  double relax, hl_c;  // ppe_relax; 2 re_lap / n0_lap (Eq. 16)
  double asm_wmax;     // pair weight of the PPE operator at r = 0.5 l0: provisional row scale of the assembly
  int ppe_source, ppe_laplacian;
  int kernel;          // 0: Eq. 3, 1: Eq. 4
  int stale;           // 1 while mps_step walks reused rows: every pair is re-tested (Q24)
  double inv_re_n, inv_re_lap;
  double dmin[3], inv_h;
  int nx, ny, nz, ncells;
  // the grid that decides which particles are GHOST (always the contract's grid, h = max r_e / cell_div;
  // equal to the fields above except in kc_step, whose cells are a little larger)
  double inv_h_dom;
  int nx_dom, ny_dom, nz_dom;
  double carry_d2;  // (0.45 x skin)^2: the distance from the build position up to which the rows stay exact supersets
  int R_lap;  // cells to each side for re_lap
  int R_n;    // ... and for re_n
  int key_mode;  // 0: key = c_x + n_x (c_y + n_y c_z); 1: Morton (3 x 10-bit interleave), ncells = 8^bits
  int cap;    // row capacity (max_neighbours)
  int stride; // row stride in entries (cap + 14 rounded up to a multiple of 8)
  int grad_variant, clamp_negative_p, rho_pair_mean, nu_pair_mean;
  int n;      // particles
  // the current position / velocity buffers as 16-byte texels (0: not used): the first half of a
  // record is fetched through the texture front end, which works in parallel with the LSU
  cudaTextureObject_t pos_tex, vel_tex;
};

// One captured segment of mps_step (a CUDA graph of its kernel launches and memsets) and the host
// state the segment leaves behind, so that a replay can skip the launch code.
struct StepSeg {
  cudaGraphExec_t exec = nullptr;
  int cur_after = 0, stale = 0;
  bool binned = false, ppe_ready = false, posw_is_p = false;
  cudaTextureObject_t pos_tex = 0, vel_tex = 0;
  int64_t launches = 0;
  int64_t bins = 0;
  int64_t t_launches[MPS_NUM_TIMERS] = {0};
};

struct mps_ctx {
  mps_params prm;
  KConst kc;
  KConst kc_step[2];  // kc with the internal grid and the skin radii of mps_step's bins, per skin level (mps_api.cu)
  double skin_l0[2] = {0, 0};  // the two skins in units of l0 (equal when the caller fixed row_skin)
  bool skin_auto = false;      // row_skin = 0: mps_step picks the level from the bins it needed lately
  int skin_level = 0;
  int skin_hold = 0;           // windows during which the thick skin is not tried again
  int64_t win_steps = 0, win_bins = 0, bins_seen = 0, win_forced = 0;  // steps and bins since the level was last looked at
  bool carry_rows = false;   // mps_step builds rows with a skin and rebuilds them only when the device says so
  bool carry_valid = false;  // the rows in nbr are skin rows and the device flags tell whether they still hold
  int rows_mode_built = 0;   // rows_mode of the skin rows in nbr (a route change may need more of them)
  double4* pos_ref = nullptr;  // positions at the last skin build, by slot
  cudaStream_t aux_stream = nullptr;  // captures the body of the conditional graph node that holds a skin bin
  int cond_launches_per_bin = 0;      // kernel launches inside such a body (they happen only when the bin runs)
  bool cond_nodes = true;             // skin bins inside a graph become conditional nodes (else: predicated kernels)
  int64_t n = 0;
  int64_t n_pad = 0;  // n rounded up to 32
  cudaStream_t stream = nullptr;
  double h = 0;
  // double-buffered sorted particle arrays
  double4* pos4[2] = {nullptr, nullptr};
  double4* vel4[2] = {nullptr, nullptr};
  cudaTextureObject_t pos_tex[2] = {0, 0};  // pos4 / vel4 viewed as 16-byte texels
  cudaTextureObject_t vel_tex[2] = {0, 0};
  bool cg_tex = false;
  uint32_t* tp[2] = {nullptr, nullptr};
  uint32_t* oid[2] = {nullptr, nullptr};
  uint32_t* ent = nullptr;         // per slot: own index | NB_* flags (what a neighbour row stores)
  int rows_builder = 0;            // 0: k_build_rows (lanes on candidates, four particles per warp, any key); 1: one
                                   // warp per particle; 2: one warp per cell (MPS_B200_ROWS=lean|warp|cell)
  int cur = 0;
  // bin scratch
  uint32_t* key = nullptr;         // per slot (after bin: key of the slot)
  uint32_t* key_tmp = nullptr;     // per pre-sort slot
  uint32_t* rank = nullptr;
  uint32_t* tmp_src = nullptr;
  uint32_t* tmp_oid = nullptr;
  uint32_t* cell_count = nullptr;  // ncells + 2
  uint32_t* cell_start = nullptr;  // ncells + 2
  uint32_t* scan_tmp = nullptr;
  uint32_t* gbit = nullptr;        // ghosts by original index: bitmap, ones per word, their exclusive scan
  uint32_t* gcnt = nullptr;
  uint32_t* gpre = nullptr;
  // neighbour rows
  uint32_t* nbr = nullptr;
  uint32_t* cn = nullptr;
  uint32_t* co = nullptr;
  // per-particle fields
  double* dens = nullptr;
  double* p = nullptr;
  double4* acc4 = nullptr;
  double* nut = nullptr;
  double* b = nullptr;
  double* phat = nullptr;
  double* dndt = nullptr;
  double* rho_s[2] = {nullptr, nullptr};   // smoothed density (grad_variant 3), carried through the re-sort
  bool rho_s_ready = false;
  double2* keep2[2] = {nullptr, nullptr};  // (n^k, (Dn/Dt)^k) of Eq. 17, carried through the re-sort
  double4* grad4 = nullptr;
  int8_t* bc = nullptr;
  // CG vectors
  double* cg_x = nullptr;
  double* cg_p = nullptr;
  double* cg_s = nullptr;
  double* cg_w = nullptr;
  double* cg_part = nullptr;  // per-block partial sums
  uint32_t* cg_rows = nullptr;   // compacted slot indices of the PPE unknowns (bc == 0)
  // ppe_operator 1: the assembled operator over the compacted rows g = 0..n_rows-1 (ELL, row g at
  // g * kc.stride) and the CG vectors in the same compact numbering
  double* mat_val = nullptr;     // one 64-bit word per stored pair: column (high 24 bits) | coefficient (low 40 bits: fraction
                                 // of the row's largest); holds plain fp64 coefficients while a row is assembled
  uint32_t* mat_col = nullptr;   // assembly scratch: the columns before packing
  double* mat_scale = nullptr;   // row's largest coefficient / (2^40 - 1)
  uint32_t* mat_cnt = nullptr;   // entries of row g
  double* mat_dex = nullptr;     // sum of c_ij over free-surface neighbours + compress / dt^2
  uint32_t* rowmap = nullptr;    // slot -> compact row (ROW_SURFACE / ROW_NONE otherwise)
  double* cg_rc = nullptr;       // residual, compact
  double* cg_xc = nullptr;       // solution, compact (cg_x is its per-slot copy)
  long long cg_timeout_cycles = 4000000000LL;  // grid-barrier spin limit (0: none)
  GridBar* bar_host = nullptr;   // pinned
  int noconv_seen = 0;           // CgScalars.noconv_total at the last read
  uint32_t* cg_bcount = nullptr; // per-block row / surface counts of the setup phase
  GridBar* cg_bar = nullptr;
  int cg_grid = 0;               // co-resident blocks of the persistent CG kernel
  int cg_lanes = 8;              // lanes per row of the operator (power of two)
  bool posw_is_p = false;        // pos4.w currently holds the pressure
  CgScalars* cg = nullptr;    // device
  CgScalars* cg_host = nullptr;  // pinned
  DevFlags* flags = nullptr;
  DevFlags* flags_host = nullptr;  // pinned
  double* io_tmp = nullptr;   // n doubles, staging for get/set
  // state
  bool binned = false;
  int64_t reuse_count = 0;  // steps since the ctx started reusing rows (rebin_every > 1)
  bool ppe_ready = false;
  int sticky_error = 0;
  mps_stats stats{};
  std::string err;
  int64_t launches = 0;
  int64_t bins_run = 0;
  // timers
  uint32_t timer_mask = 0;  // bit k: time category k with CUDA events
  double t_ms[MPS_NUM_TIMERS] = {0};
  int64_t t_launches[MPS_NUM_TIMERS] = {0};
  std::vector<cudaEvent_t> ev_pool;
  std::vector<int> ev_cat;
  size_t ev_used = 0;
  int sm_count = 148;
  // mps_step replays its launch sequence from CUDA graphs (one per route, buffer parity and segment)
  // when the ctx has a capturable stream (not the legacy default stream) and timers are off
  StepSeg seg[2][2][2][4];   // [skin level][route][buffer parity][segment: 0 pre, 1 post]
  bool graphs_ok = true;
};

// ---- launch helper: counts launches, optional CUDA-event timing ------------------
void mps_timer_begin(mps_ctx* c, int cat);
void mps_timer_end(mps_ctx* c, int cat);
void mps_timer_drain(mps_ctx* c);

#define MPS_LAUNCH(c, cat, kern, grid, block, ...)                         \
  do {                                                                     \
    if (((c)->timer_mask >> (cat)) & 1u) mps_timer_begin((c), (cat));                       \
    kern<<<(grid), (block), 0, (c)->stream>>>(__VA_ARGS__);                \
    (c)->launches++;                                                       \
    (c)->t_launches[(cat)]++;                                              \
    if (((c)->timer_mask >> (cat)) & 1u) mps_timer_end((c), (cat));                         \
  } while (0)

static inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// ---- stage launchers (defined in the .cu files) -----------------------------------
// keys, counting sort, reorder, neighbour rows
// rows_mode bit 0: rows of FLUID particles only (all a viscosity sweep needs); bit 1: the re_n part only
// (all the explicit route needs at r*)
#define ROWS_FLUID_ONLY 1
#define ROWS_RN_ONLY 2
#define ROWS_BACK_FLUID 4   // the re_n part of every row, the rest of the re_lap part for FLUID rows only
// go != NULL: the bin of mps_step with a skin -- on the ctx's internal grid, rows with the skin radii
// (kc_step), every kernel returns at once unless *go != 0 (a device flag), and the sorted arrays are
// copied back into the current buffers, so the host state does not depend on whether it ran
int mpsk_bin(mps_ctx* c, int rows_mode = 0, const int* go = nullptr);
void mpsk_exclusive_scan(mps_ctx* c, int cat, const uint32_t* in, uint32_t* out, int64_t n,
                         uint32_t* tmp, const int* go = nullptr);
int mpsk_density(mps_ctx* c);
int mpsk_dndt(mps_ctx* c, int keep);
int mpsk_smooth_density(mps_ctx* c);
int mpsk_viscosity(mps_ctx* c);
int mpsk_predict(mps_ctx* c);
int mpsk_pressure_explicit(mps_ctx* c);
int mpsk_ppe_plan(mps_ctx* c);           // co-resident grid of the persistent CG kernel
int mpsk_pressure_ppe(mps_ctx* c, bool sync = true);  // sync: read the solve's statistics back
int mpsk_ppe_read_stats(mps_ctx* c);
int mpsk_ppe_apply(mps_ctx* c, const double* x, double* y, int order);
int mpsk_gradient(mps_ctx* c);
int mpsk_correct(mps_ctx* c);
int mpsk_get_field(mps_ctx* c, int field, void* dst, int order);
int mpsk_set_field(mps_ctx* c, int field, const void* src, int order);
int mpsk_load_particles(mps_ctx* c, const double* x, const double* y, const double* z,
                        const double* u, const double* v, const double* w, const int32_t* type,
                        const int32_t* phase);
int mpsk_get_neighbours(mps_ctx* c, int radius_id, uint32_t* counts, uint32_t* idx, int64_t cap,
                        int64_t* total);
