// mps_api.cu -- the extern "C" boundary of libmps_b200.so (include/mps_b200.h).
// Host logic only: argument checks, buffer ownership, stage ordering, timers.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>

#include <nvtx3/nvToolsExt.h>  // header-only: ranges show up when a profiler is attached, cost nothing otherwise

#include "mps_internal.h"

static std::string g_init_error;

// one NVTX range per ABI call
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};
#define MPS_RANGE() NvtxRange nvtx_range_(__func__)

#define CK(call)                                                                 \
  do {                                                                           \
    cudaError_t e_ = (call);                                                     \
    if (e_ != cudaSuccess) {                                                     \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);               \
      return MPS_ERR_CUDA;                                                       \
    }                                                                            \
  } while (0)

static int fail(mps_ctx* c, int code, const char* msg) {
  if (c) c->err = msg;
  else g_init_error = msg;
  return code;
}

// ---- lattice closed forms (I2; Eq. 5) -------------------------
// n0 = sum over lattice offsets o != 0 with |o| l0 < re of (re / (|o| l0) - 1),
// lambda = sum |o|^2 l0^2 w / sum w.
static void lattice_sums(int dim, int kernel, double l0, double re, double* n0, double* lam) {
  const int R = (int)ceil(re / l0) + 1;
  double sw = 0.0, sr2w = 0.0;
  const int Rz = dim == 3 ? R : 0;
  for (int a = -Rz; a <= Rz; ++a)
    for (int b = -R; b <= R; ++b)
      for (int k = -R; k <= R; ++k) {
        if (!a && !b && !k) continue;
        const double ex = k * l0, ey = b * l0, ez = a * l0;
        const double r2 = (ex * ex + ey * ey) + ez * ez;
        if (r2 < re * re) {
          const double r = sqrt(r2);
          const double w = kernel == 1 ? (1.0 - r / re) * (1.0 - r / re) * (1.0 - r / re) : re / r - 1.0;
          sw += w;
          sr2w += r2 * w;
        }
      }
  *n0 = sw;
  *lam = sr2w / sw;
}

template <class T>
static cudaError_t dalloc(T** p, size_t count) {
  return cudaMalloc((void**)p, std::max<size_t>(count, 1) * sizeof(T));
}

static void free_all(mps_ctx* c) {
  for (int k = 0; k < 2; ++k) {
    if (c->pos_tex[k]) cudaDestroyTextureObject(c->pos_tex[k]);
    if (c->vel_tex[k]) cudaDestroyTextureObject(c->vel_tex[k]);
    cudaFree(c->pos4[k]); cudaFree(c->vel4[k]); cudaFree(c->tp[k]); cudaFree(c->oid[k]);
  }
  cudaFree(c->ent); cudaFree(c->key); cudaFree(c->key_tmp); cudaFree(c->rank); cudaFree(c->tmp_src);
  cudaFree(c->tmp_oid); cudaFree(c->cell_count); cudaFree(c->cell_start); cudaFree(c->scan_tmp);
  cudaFree(c->gbit); cudaFree(c->gcnt); cudaFree(c->gpre);
  cudaFree(c->nbr); cudaFree(c->cn); cudaFree(c->co); cudaFree(c->pos_ref);
  cudaFree(c->dens); cudaFree(c->p); cudaFree(c->acc4); cudaFree(c->nut); cudaFree(c->b);
  cudaFree(c->phat); cudaFree(c->dndt); cudaFree(c->rho_s[0]); cudaFree(c->rho_s[1]); cudaFree(c->keep2[0]); cudaFree(c->keep2[1]); cudaFree(c->grad4); cudaFree(c->bc);
  cudaFree(c->cg_x); cudaFree(c->cg_p); cudaFree(c->cg_s); cudaFree(c->cg_w); cudaFree(c->cg_part);
  cudaFree(c->cg_rows); cudaFree(c->cg_bcount); cudaFree(c->cg_bar);
  cudaFree(c->mat_val); cudaFree(c->mat_col); cudaFree(c->mat_cnt); cudaFree(c->mat_dex); cudaFree(c->mat_scale); cudaFree(c->rowmap);
  cudaFree(c->cg_rc); cudaFree(c->cg_xc);
  if (c->bar_host) cudaFreeHost(c->bar_host);
  if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
  cudaFree(c->cg); cudaFree(c->flags); cudaFree(c->io_tmp);
  if (c->cg_host) cudaFreeHost(c->cg_host);
  if (c->flags_host) cudaFreeHost(c->flags_host);
  for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
  for (auto& l : c->seg) for (auto& r : l) for (auto& p : r) for (auto& g : p) if (g.exec) cudaGraphExecDestroy(g.exec);
}

static int check_params(const mps_params* p, int64_t n) {
  if (!p) return fail(nullptr, MPS_ERR_ARG, "params is NULL");
  if (n <= 0 || n > (int64_t)NB_INDEX) return fail(nullptr, MPS_ERR_ARG, "n must be in [1, 2^29)");
  if (p->dim != 2 && p->dim != 3) return fail(nullptr, MPS_ERR_ARG, "dim must be 2 or 3");
  if (p->dim == 2 && p->ppe_laplacian == 1)
    return fail(nullptr, MPS_ERR_ARG, "the higher-order Laplacian (Eq. 16) is given for 3D only");
  if (!(p->l0 > 0) || !(p->re_n > 0) || !(p->re_lap > 0) || !(p->dt > 0))
    return fail(nullptr, MPS_ERR_ARG, "l0, re_n, re_lap and dt must be positive");
  if (p->re_grad != p->re_n) return fail(nullptr, MPS_ERR_ARG, "re_grad must equal re_n");
  if (p->re_lap < p->re_n) return fail(nullptr, MPS_ERR_ARG, "re_lap must be >= re_n");
  if (p->key_mode < 0 || p->key_mode > 1) return fail(nullptr, MPS_ERR_ARG, "key_mode must be 0 (linear) or 1 (Morton)");
  if (p->cell_div < 1 || p->cell_div > 3) return fail(nullptr, MPS_ERR_ARG, "cell_div must be 1..3");
  if (p->n_phases < 1 || p->n_phases > 2) return fail(nullptr, MPS_ERR_ARG, "n_phases must be 1 or 2");
  if (p->max_neighbours < 1 || p->max_neighbours > 4096)
    return fail(nullptr, MPS_ERR_ARG, "max_neighbours must be in [1, 4096]");
  if (p->ppe_source < 0 || p->ppe_source > 2) return fail(nullptr, MPS_ERR_ARG, "ppe_source must be 0..2");
  if (p->ppe_laplacian < 0 || p->ppe_laplacian > 1) return fail(nullptr, MPS_ERR_ARG, "ppe_laplacian must be 0 or 1");
  if (p->rebin_every < 1 || p->rebin_every > 1000) return fail(nullptr, MPS_ERR_ARG, "rebin_every must be in [1, 1000]");
  if (p->ppe_operator < 0 || p->ppe_operator > 1) return fail(nullptr, MPS_ERR_ARG, "ppe_operator must be 0 (matrix-free) or 1 (assembled)");
  if (p->ppe_operator == 1 && n >= ((int64_t)1 << 24))
    return fail(nullptr, MPS_ERR_ARG, "ppe_operator 1 stores 24-bit column indices: n must be below 2^24 (use ppe_operator 0)");
  if (p->cg_warm_start < 0 || p->cg_warm_start > 1) return fail(nullptr, MPS_ERR_ARG, "cg_warm_start must be 0 or 1");
  if (p->kernel < 0 || p->kernel > 1) return fail(nullptr, MPS_ERR_ARG, "kernel must be 0 (Eq. 3) or 1 (Eq. 4)");
  if (!(p->row_skin <= 1.0)) return fail(nullptr, MPS_ERR_ARG, "row_skin must be at most 1 (in units of l0); 0 = default, < 0 = off");
  if (p->kernel == 1 && (p->ppe_source != 0 || p->ppe_laplacian != 0))
    return fail(nullptr, MPS_ERR_ARG, "Eq. 15-18 are derived for the Eq. 3 kernel: kernel 1 needs ppe_source = ppe_laplacian = 0");
  if (p->grad_variant < 0 || p->grad_variant > 3) return fail(nullptr, MPS_ERR_ARG, "grad_variant must be 0..3");
  if (!(p->rho[0] > 0) || (p->n_phases == 2 && !(p->rho[1] > 0)))
    return fail(nullptr, MPS_ERR_ARG, "densities must be positive");
  if (!(p->gamma > 0) || !(p->cg_rtol > 0) || p->cg_maxit < 1)
    return fail(nullptr, MPS_ERR_ARG, "gamma, cg_rtol and cg_maxit must be positive");
  for (int a = 0; a < 3; ++a)
    if (!(p->domain_max[a] > p->domain_min[a]))
      return fail(nullptr, MPS_ERR_ARG, "domain_max must exceed domain_min");
  return MPS_OK;
}

static int create_ctx(mps_ctx** out, const mps_params* prm, int64_t n, void* stream) {
  if (!out) return fail(nullptr, MPS_ERR_ARG, "out is NULL");
  *out = nullptr;
  int rc = check_params(prm, n);
  if (rc) return rc;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess)
    return fail(nullptr, MPS_ERR_CUDA, "no CUDA device: libmps_b200 has no CPU fallback");
  if (prop.major < 10)
    return fail(nullptr, MPS_ERR_CUDA, "libmps_b200 is built for sm_100a (B200) only");
  mps_ctx* c = new (std::nothrow) mps_ctx;
  if (!c) return fail(nullptr, MPS_ERR_ARG, "out of host memory");
  c->prm = *prm;
  c->n = n;
  c->n_pad = (n + 31) / 32 * 32;
  c->stream = (cudaStream_t)stream;
  c->sm_count = prop.multiProcessorCount;

  // constants (I1-I4)
  KConst& k = c->kc;
  memset(&k, 0, sizeof(k));
  double n0n, lam_n, n0l, lam_l;
  lattice_sums(prm->dim, prm->kernel, prm->l0, prm->re_n, &n0n, &lam_n);
  lattice_sums(prm->dim, prm->kernel, prm->l0, prm->re_lap, &n0l, &lam_l);
  k.n0_n = prm->n0_n > 0 ? prm->n0_n : n0n;
  k.n0_lap = prm->n0_lap > 0 ? prm->n0_lap : n0l;
  k.lam = prm->lambda > 0 ? prm->lambda : lam_l;
  k.A_lap = 2.0 * prm->dim / (k.n0_lap * k.lam);
  k.re_n = prm->re_n; k.re_n2 = prm->re_n * prm->re_n;
  k.re_lap = prm->re_lap; k.re_lap2 = prm->re_lap * prm->re_lap;
  k.dt = prm->dt;
  for (int a = 0; a < 3; ++a) { k.g[a] = prm->g[a]; k.dmin[a] = prm->domain_min[a]; }
  k.rho[0] = prm->rho[0]; k.rho[1] = prm->n_phases == 2 ? prm->rho[1] : prm->rho[0];
  k.nu[0] = prm->nu[0]; k.nu[1] = prm->n_phases == 2 ? prm->nu[1] : prm->nu[0];
  k.c0 = prm->c0; k.gamma = prm->gamma; k.beta = prm->beta;
  k.compress_dt2 = prm->compress / (prm->dt * prm->dt);
  k.relax_dt2 = prm->ppe_relax / (prm->dt * prm->dt);
  k.cs_l0_sq = (prm->cs * prm->l0) * (prm->cs * prm->l0);
  k.d_over_n0 = (double)prm->dim / k.n0_n;
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) {
      const double ra = k.rho[a], rb = k.rho[b];
      k.inv_rho_pair[a][b] = 1.0 / (prm->rho_pair_mean == 1 ? 2.0 * ra * rb / (ra + rb) : 0.5 * (ra + rb));
    }
  k.relax = prm->ppe_relax;
  k.hl_c = 2.0 * prm->re_lap / k.n0_lap;
  {
    const double r0 = 0.5 * prm->l0;
    k.asm_wmax = prm->ppe_laplacian == 1 ? 1.0 / (r0 * r0 * r0) : prm->kernel == 1 ? 1.0 : prm->re_lap / r0 - 1.0;
  }
  k.ppe_source = prm->ppe_source; k.ppe_laplacian = prm->ppe_laplacian;
  k.kernel = prm->kernel; k.inv_re_n = 1.0 / prm->re_n; k.inv_re_lap = 1.0 / prm->re_lap;
  c->h = std::max(prm->re_n, prm->re_lap) / prm->cell_div;
  k.inv_h = 1.0 / c->h;
  int64_t ncells = 1;
  int nc[3];
  for (int a = 0; a < 3; ++a) {
    nc[a] = (int)ceil((prm->domain_max[a] - prm->domain_min[a]) * k.inv_h);
    if (nc[a] < 1) nc[a] = 1;
    ncells *= nc[a];
  }
  k.key_mode = prm->key_mode;
  if (prm->key_mode == 1) {  // Morton keys live in [0, 8^bits), bits = smallest with 2^bits >= every n_a
    int bits = 0;
    while ((1 << bits) < std::max(nc[0], std::max(nc[1], nc[2]))) ++bits;
    ncells = bits > 10 ? ((int64_t)1 << 31) : ((int64_t)1 << (3 * bits));
  }
  if (ncells >= (int64_t)1 << 30) {
    delete c;
    return fail(nullptr, MPS_ERR_ARG, "grid has 2^30 cells or more (Morton: more than 512 cells along an axis)");
  }
  k.nx = nc[0]; k.ny = nc[1]; k.nz = nc[2]; k.ncells = (int)ncells;
  // cells to scan on each side: ceil(re / h), guarded against re * (1/h) rounding just above an
  // integer (h = re_lap / cell_div gives 3.0000000000000004 for some l0): the scan only needs to be a
  // superset of the radius, and is one with the integer below
  k.R_lap = std::max(1, (int)ceil(prm->re_lap * k.inv_h - 1e-9));
  k.R_n = std::max(1, (int)ceil(prm->re_n * k.inv_h - 1e-9));
  k.cap = prm->max_neighbours;
  k.stride = (k.cap + 14 + 7) / 8 * 8;
  k.grad_variant = prm->grad_variant; k.clamp_negative_p = prm->clamp_negative_p;
  k.rho_pair_mean = prm->rho_pair_mean; k.nu_pair_mean = prm->nu_pair_mean;
  k.n = (int)n;
  k.inv_h_dom = k.inv_h; k.nx_dom = k.nx; k.ny_dom = k.ny; k.nz_dom = k.nz;
  k.carry_d2 = 0.0;
  {
    // mps_step's own bins (Q26): cells of (max re + skin) / cell_div, rows built with both radii enlarged by
    // the skin.  A scan of cell_div cells to each side still finds every pair inside the enlarged radius,
    // and the rows stay exact supersets while no particle is further than 0.45 skins from where it was at
    // the build -- which the predictor and the corrector check.  GHOST decisions stay on the contract's grid.
    // Two skins when the caller leaves the choice to the library (row_skin = 0): 0.1 l0, and 0.3 l0 for a flow
    // that needs more than 0.4 bins per step with the thin one (mps_step switches between calls, see there).
    const char* cr = getenv("MPS_B200_CARRY");
    c->skin_auto = prm->row_skin == 0.0;
    c->carry_rows = prm->rebin_every == 1 && !(prm->row_skin < 0.0) && !(cr && atoi(cr) == 0);
    for (int lv = 0; lv < 2; ++lv) {
      KConst& s = c->kc_step[lv];
      s = k;
      const double skin_l0 = c->skin_auto ? (lv == 0 ? 0.1 : 0.3) : prm->row_skin;
      const double skin = skin_l0 * prm->l0;
      c->skin_l0[lv] = skin_l0;
      const double hs = (std::max(prm->re_n, prm->re_lap) + 1.001 * std::max(skin, 0.0)) / prm->cell_div;
      s.inv_h = 1.0 / hs;
      int64_t ncs = 1;
      int ns[3];
      for (int a = 0; a < 3; ++a) {
        ns[a] = std::max(1, (int)ceil(nc[a] * c->h * s.inv_h));  // covers the contract grid's extent
        ncs *= ns[a];
      }
      s.nx = ns[0]; s.ny = ns[1]; s.nz = ns[2];
      if (prm->key_mode == 1) {
        int bits = 0;
        while ((1 << bits) < std::max(ns[0], std::max(ns[1], ns[2]))) ++bits;
        ncs = (int64_t)1 << (3 * bits);
      }
      s.ncells = (int)ncs;
      s.re_lap2 = (prm->re_lap + skin) * (prm->re_lap + skin);
      s.re_n2 = (prm->re_n + skin) * (prm->re_n + skin);
      s.R_lap = std::max(1, (int)ceil((prm->re_lap + skin) * s.inv_h - 1e-9));
      s.R_n = std::max(1, (int)ceil((prm->re_n + skin) * s.inv_h - 1e-9));
      s.carry_d2 = (0.45 * skin) * (0.45 * skin);
      // off with the paper's list reuse (rebin_every > 1 has its own schedule, Q24) and with row_skin < 0;
      // MPS_B200_CARRY=0 forces the two bins per step of reading Q7 as literally stated
      c->carry_rows = c->carry_rows && skin > 0.0 && ncs <= ncells && s.R_lap == k.R_lap;
    }
    k.carry_d2 = c->kc_step[0].carry_d2;
  }

  // every buffer any later call needs
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  const size_t N = (size_t)c->n_pad;
  for (int b = 0; b < 2; ++b) {
    A(dalloc(&c->pos4[b], N + 32)); A(dalloc(&c->vel4[b], N)); A(dalloc(&c->tp[b], N)); A(dalloc(&c->oid[b], N));
  }
  A(dalloc(&c->ent, N + 32)); A(dalloc(&c->key, N)); A(dalloc(&c->key_tmp, N)); A(dalloc(&c->rank, N));
  A(dalloc(&c->tmp_src, N + 1)); A(dalloc(&c->tmp_oid, N));
  A(dalloc(&c->cell_count, (size_t)ncells + 2)); A(dalloc(&c->cell_start, (size_t)ncells + 2));
  A(dalloc(&c->scan_tmp, std::max<size_t>((size_t)ncells + 2, N) / 2048 + 2));
  A(dalloc(&c->gbit, N / 32 + 2)); A(dalloc(&c->gcnt, N / 32 + 2)); A(dalloc(&c->gpre, N / 32 + 2));
  A(dalloc(&c->nbr, N * (size_t)k.stride)); A(dalloc(&c->cn, N)); A(dalloc(&c->co, N));
  A(dalloc(&c->pos_ref, c->carry_rows ? N : 1));
  if (c->carry_rows) A(cudaStreamCreateWithFlags(&c->aux_stream, cudaStreamNonBlocking));
  {
    // Nsight Compute cannot profile kernel nodes of a graph that holds conditional nodes ("not supported for
    // profiling"): with a CUDA injection library in the process (a profiler is attached), or MPS_B200_COND=0,
    // the skin bins are captured as plain kernel nodes that return at once when not needed
    const char* cn = getenv("MPS_B200_COND");
    const char* inj = getenv("CUDA_INJECTION64_PATH");
    c->cond_nodes = cn ? atoi(cn) != 0 : !(inj && *inj);
  }
  A(dalloc(&c->dens, N)); A(dalloc(&c->p, N)); A(dalloc(&c->acc4, N)); A(dalloc(&c->nut, N));
  A(dalloc(&c->b, N)); A(dalloc(&c->phat, N)); A(dalloc(&c->dndt, N));
  A(dalloc(&c->keep2[0], N)); A(dalloc(&c->keep2[1], N));
  A(dalloc(&c->rho_s[0], N)); A(dalloc(&c->rho_s[1], N)); A(dalloc(&c->grad4, N)); A(dalloc(&c->bc, N));
  A(dalloc(&c->cg_x, N)); A(dalloc(&c->cg_p, N)); A(dalloc(&c->cg_s, N)); A(dalloc(&c->cg_w, N));
  A(dalloc(&c->cg_part, (size_t)2 * (c->sm_count * 8 + 8)));
  A(dalloc(&c->cg_rows, N)); A(dalloc(&c->cg_bcount, (size_t)2 * (c->sm_count * 8 + 8)));
  A(dalloc(&c->cg_bar, 1));
  if (prm->ppe_operator == 1) {  // the assembled operator: 12 bytes per pair of the rows bc = 0
    A(dalloc(&c->mat_val, N * (size_t)k.stride)); A(dalloc(&c->mat_col, N * (size_t)k.stride));
    A(dalloc(&c->mat_cnt, N)); A(dalloc(&c->mat_dex, N)); A(dalloc(&c->mat_scale, N)); A(dalloc(&c->rowmap, N));
    A(dalloc(&c->cg_rc, N)); A(dalloc(&c->cg_xc, N));
  } else if (c->carry_rows) {  // matrix-free on skin rows: the exact list of every unknown row, built once per solve
    A(dalloc(&c->mat_col, N * (size_t)k.stride)); A(dalloc(&c->mat_cnt, N));
  }
  A(cudaMallocHost((void**)&c->bar_host, sizeof(GridBar)));
  A(dalloc(&c->cg, 1)); A(dalloc(&c->flags, 1)); A(dalloc(&c->io_tmp, N));
  A(cudaMallocHost((void**)&c->cg_host, sizeof(CgScalars)));
  A(cudaMallocHost((void**)&c->flags_host, sizeof(DevFlags)));
  if (e != cudaSuccess) {
    g_init_error = std::string("allocation failed: ") + cudaGetErrorString(e);
    free_all(c);
    delete c;
    return MPS_ERR_CUDA;
  }
  {
    // Row builder: 2 = one warp per cell (cell_div 1, large scenes), 1 = one warp per particle (few
    // occupied cells cannot fill the GPU with one warp per cell: measured crossover between 89 k and
    // 438 k particles), 0 = k_build_rows (any key, any cell size; the only one that walks Morton
    // keys).  MPS_B200_ROWS=lean|warp|cell overrides the choice (tests run every builder).
    const char* rw = getenv("MPS_B200_ROWS");
    c->rows_builder = (n >= 200000 && prm->cell_div == 1) ? 2 : 1;
    if (rw) c->rows_builder = !strcmp(rw, "warp") ? 1 : !strcmp(rw, "cell") ? 2 : 0;
    if (prm->key_mode == 1) c->rows_builder = 0;
  }
  {
    // texture views of the two position buffers (MPS_B200_CG_TEX=0 switches them off)
    const char* tx = getenv("MPS_B200_CG_TEX");
    c->cg_tex = (tx ? atoi(tx) != 0 : true) && (2 * (N + 32) <= (size_t)prop.maxTexture1DLinear);
    for (int b = 0; b < 4 && c->cg_tex; ++b) {
      cudaResourceDesc rd;
      memset(&rd, 0, sizeof(rd));
      rd.resType = cudaResourceTypeLinear;
      rd.res.linear.devPtr = b < 2 ? (void*)c->pos4[b] : (void*)c->vel4[b - 2];
      rd.res.linear.desc = cudaCreateChannelDesc<int4>();
      rd.res.linear.sizeInBytes = (b < 2 ? N + 32 : N) * sizeof(double4);
      cudaTextureDesc td;
      memset(&td, 0, sizeof(td));
      td.readMode = cudaReadModeElementType;
      cudaTextureObject_t* dst = b < 2 ? &c->pos_tex[b] : &c->vel_tex[b - 2];
      if (cudaCreateTextureObject(dst, &rd, &td, nullptr) != cudaSuccess) {
        cudaGetLastError();
        c->cg_tex = false;
      }
    }
    c->kc.pos_tex = c->cg_tex ? c->pos_tex[c->cur] : 0;
    c->kc.vel_tex = c->cg_tex ? c->vel_tex[c->cur] : 0;
  }
  if (mpsk_ppe_plan(c) != MPS_OK) {
    g_init_error = "k_ppe_cg cannot be made resident on this device";
    free_all(c);
    delete c;
    return MPS_ERR_CUDA;
  }
  memset(c->cg_host, 0, sizeof(CgScalars));
  memset(c->bar_host, 0, sizeof(GridBar));
  if (prm->ppe_operator == 1) {
    cudaMemsetAsync(c->mat_cnt, 0, N * 4, c->stream);
    cudaMemsetAsync(c->rowmap, 0xff, N * 4, c->stream);
    cudaMemsetAsync(c->cg_rc, 0, N * 8, c->stream);
    cudaMemsetAsync(c->cg_xc, 0, N * 8, c->stream);
  }
  memset(c->flags_host, 0, sizeof(DevFlags));
  cudaStream_t s = c->stream;
  cudaMemsetAsync(c->cg, 0, sizeof(CgScalars), s);
  cudaMemsetAsync(c->cg_bar, 0, sizeof(GridBar), s);
  cudaMemsetAsync(c->cg_rows, 0, N * 4, s);
  cudaMemsetAsync(c->flags, 0, sizeof(DevFlags), s);
  double* zero_d[] = {c->dens, c->p, c->nut, c->b, c->phat, c->dndt, c->cg_x, c->cg_p, c->cg_s, c->cg_w};
  for (int b = 0; b < 2; ++b) {
    cudaMemsetAsync(c->keep2[b], 0, N * sizeof(double2), s);
    cudaMemsetAsync(c->rho_s[b], 0, N * sizeof(double), s);
  }
  for (double* z : zero_d) cudaMemsetAsync(z, 0, N * sizeof(double), s);
  cudaMemsetAsync(c->acc4, 0, N * sizeof(double4), s);
  cudaMemsetAsync(c->grad4, 0, N * sizeof(double4), s);
  cudaMemsetAsync(c->bc, 0, N, s);
  cudaMemsetAsync(c->cn, 0, N * 4, s);
  cudaMemsetAsync(c->co, 0, N * 4, s);
  cudaMemsetAsync(c->key, 0, N * 4, s);
  cudaMemsetAsync(c->ent, 0, (N + 32) * 4, s);
  for (int b = 0; b < 2; ++b) {
    cudaMemsetAsync(c->pos4[b], 0, (N + 32) * sizeof(double4), s);
    cudaMemsetAsync(c->vel4[b], 0, N * sizeof(double4), s);
    cudaMemsetAsync(c->tp[b], 0, N * 4, s);
    cudaMemsetAsync(c->oid[b], 0, N * 4, s);
  }
  *out = c;
  return MPS_OK;
}

// Reads the device-side flags; converts them into a sticky error code.
static int read_flags(mps_ctx* c) {
  CK(cudaMemcpyAsync(c->flags_host, c->flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->stats.max_neighbours = c->flags_host->max_row;
  c->stats.n_ghost = c->flags_host->n_ghost;
  if (c->flags_host->nonfinite) {
    c->sticky_error = MPS_ERR_NONFINITE;
    c->err = "non-finite position or coincident particles";
  } else if (c->flags_host->overflow) {
    c->sticky_error = MPS_ERR_NEIGHBOUR_OVERFLOW;
    c->err = "a particle has more than max_neighbours neighbours";
  }
  c->stats.device_error = c->sticky_error;
  c->stats.bins_total = c->bins_run + c->flags_host->bins;
  c->stats.row_skin_now = c->carry_rows ? c->skin_l0[c->skin_level] : -1.0;
  return c->sticky_error;
}

// ---- timers ---------------------------------------------------------------------
void mps_timer_begin(mps_ctx* c, int cat) {
  if (c->ev_used + 2 > c->ev_pool.size()) mps_timer_drain(c);
  cudaEventRecord(c->ev_pool[c->ev_used], c->stream);
  c->ev_cat[c->ev_used / 2] = cat;
}
void mps_timer_end(mps_ctx* c, int) {
  cudaEventRecord(c->ev_pool[c->ev_used + 1], c->stream);
  c->ev_used += 2;
}
void mps_timer_drain(mps_ctx* c) {
  if (c->ev_used == 0) return;
  cudaStreamSynchronize(c->stream);
  for (size_t k = 0; k < c->ev_used; k += 2) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->ev_pool[k], c->ev_pool[k + 1]) == cudaSuccess)
      c->t_ms[c->ev_cat[k / 2]] += ms;
  }
  c->ev_used = 0;
}

// ---- mps_step segments as CUDA graphs ----------------------------------------------
// The launch sequence of a step is fixed by (route, which of the two particle buffers is
// current, segment), so it is captured once and replayed: a step of a small scene is bound by
// the host's launch rate (about twenty launches and memsets of a few microseconds each), a graph
// launch costs one.  The body runs for real when capture is not possible (legacy default stream,
// timers on) and mutates the same host state either way.
struct HostState {
  int cur, stale; bool binned, ppe_ready, posw_is_p; cudaTextureObject_t pos_tex, vel_tex;
  int64_t launches, bins; int64_t t_launches[MPS_NUM_TIMERS];
};
static HostState save_state(const mps_ctx* c) {
  HostState h{c->cur, c->kc.stale, c->binned, c->ppe_ready, c->posw_is_p, c->kc.pos_tex, c->kc.vel_tex, c->launches, c->bins_run, {0}};
  for (int k = 0; k < MPS_NUM_TIMERS; ++k) h.t_launches[k] = c->t_launches[k];
  return h;
}
static void restore_state(mps_ctx* c, const HostState& h) {
  c->cur = h.cur; c->kc.stale = h.stale; c->binned = h.binned; c->ppe_ready = h.ppe_ready; c->posw_is_p = h.posw_is_p;
  c->kc.pos_tex = h.pos_tex; c->kc.vel_tex = h.vel_tex; c->launches = h.launches; c->bins_run = h.bins;
  for (int k = 0; k < MPS_NUM_TIMERS; ++k) c->t_launches[k] = h.t_launches[k];
}
template <class F>
static void run_segment(mps_ctx* c, int route, int which, F&& body) {
  if (!c->graphs_ok || c->timer_mask != 0 || c->stream == nullptr) { body(); return; }
  StepSeg& g = c->seg[c->skin_level][route][c->cur][which];
  if (!g.exec) {
    const HostState before = save_state(c);
    if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaGetLastError();
      c->graphs_ok = false;
      body();
      return;
    }
    body();
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (e == cudaSuccess && graph) e = cudaGraphInstantiate(&g.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess || !g.exec) {  // not capturable here: run the launches for real from now on
      cudaGetLastError();
      g.exec = nullptr;
      c->graphs_ok = false;
      restore_state(c, before);
      body();
      return;
    }
    g.cur_after = c->cur; g.stale = c->kc.stale; g.binned = c->binned; g.ppe_ready = c->ppe_ready; g.posw_is_p = c->posw_is_p;
    g.pos_tex = c->kc.pos_tex; g.vel_tex = c->kc.vel_tex;
    g.launches = c->launches - before.launches;
    g.bins = c->bins_run - before.bins;
    for (int k = 0; k < MPS_NUM_TIMERS; ++k) g.t_launches[k] = c->t_launches[k] - before.t_launches[k];
  } else {
    c->cur = g.cur_after; c->kc.stale = g.stale; c->binned = g.binned; c->ppe_ready = g.ppe_ready; c->posw_is_p = g.posw_is_p;
    c->kc.pos_tex = g.pos_tex; c->kc.vel_tex = g.vel_tex;
    c->launches += g.launches;
    c->bins_run += g.bins;
    for (int k = 0; k < MPS_NUM_TIMERS; ++k) c->t_launches[k] += g.t_launches[k];
  }
  cudaGraphLaunch(g.exec, c->stream);
}

// The automatic skin (row_skin = 0): looked at after windows of sixteen or more steps, from the bins those steps
// needed (c->flags_host->bins must be fresh; bins forced by new particles or a change of route do not count).  Thin
// skin and more than 0.4 bins per step: rows of 0.3 l0 last three times as long and their longer sweeps cost less
// than the bins saved (measured at 2M in the developed dam break: 5.0 -> 4.1 ms per explicit step); thick skin and
// fewer than 0.06: back (from rest 2.26 vs 2.4 ms).
static void skin_policy(mps_ctx* c, int64_t steps) {
  const int64_t bins_now = c->flags_host->bins;
  c->win_bins += bins_now - c->bins_seen - c->win_forced;
  c->bins_seen = bins_now;
  c->win_forced = 0;
  c->win_steps += steps;
  if (c->win_steps >= 16) {
    const double rate = (double)c->win_bins / (double)c->win_steps;
    int lv = c->skin_level;
    if (lv == 0 && rate >= 0.4 && c->skin_hold == 0) lv = 1;
    else if (lv == 1 && rate <= 0.06) lv = 0;
    else if (lv == 1 && rate >= 0.8) {  // too fast even for the thick skin (one bin per step either way): the thin
      lv = 0;                           // one has the shorter sweeps; do not try again for eight windows
      c->skin_hold = 8;
    } else if (c->skin_hold > 0) --c->skin_hold;
    if (lv != c->skin_level) {
      c->skin_level = lv;
      c->kc.carry_d2 = c->kc_step[lv].carry_d2;
      c->carry_valid = false;  // rows of the other skin: the next step rebuilds (not counted as needed)
    }
    c->win_steps = c->win_bins = 0;
  }
  c->stats.row_skin_now = c->skin_l0[c->skin_level];
}

extern "C" {

const char* mps_version(void) { return "mps_b200 0.1 (sm_100a)"; }

const char* mps_last_error(mps_ctx* c) { return c ? c->err.c_str() : g_init_error.c_str(); }

int mps_init(mps_ctx** out, const mps_params* prm, int64_t n, const double* x, const double* y,
             const double* z, const double* u, const double* v, const double* w, const int32_t* type,
             const int32_t* phase, void* stream) {
  MPS_RANGE();
  if (!x || !y || !z || !u || !v || !w || !type || !phase)
    return fail(nullptr, MPS_ERR_ARG, "a particle array pointer is NULL");
  int rc = create_ctx(out, prm, n, stream);
  if (rc) return rc;
  mps_ctx* c = *out;
  mpsk_load_particles(c, x, y, z, u, v, w, type, phase);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    g_init_error = std::string("mps_init: ") + cudaGetErrorString(e);
    free_all(c);
    delete c;
    *out = nullptr;
    return MPS_ERR_CUDA;
  }
  return MPS_OK;
}

int mps_init_host(mps_ctx** out, const mps_params* prm, int64_t n, const double* x, const double* y,
                  const double* z, const double* u, const double* v, const double* w,
                  const int32_t* type, const int32_t* phase, void* stream) {
  MPS_RANGE();
  if (!x || !y || !z || !u || !v || !w || !type || !phase)
    return fail(nullptr, MPS_ERR_ARG, "a particle array pointer is NULL");
  int rc = create_ctx(out, prm, n, stream);
  if (rc) return rc;
  mps_ctx* c = *out;
  // stage through buffers that are free before the first bin
  double* d[6] = {c->dens, c->p, c->nut, c->b, c->phat, c->cg_x};
  const double* h[6] = {x, y, z, u, v, w};
  for (int k = 0; k < 6; ++k)
    cudaMemcpyAsync(d[k], h[k], n * sizeof(double), cudaMemcpyHostToDevice, c->stream);
  cudaMemcpyAsync(c->key_tmp, type, n * 4, cudaMemcpyHostToDevice, c->stream);
  cudaMemcpyAsync(c->rank, phase, n * 4, cudaMemcpyHostToDevice, c->stream);
  mpsk_load_particles(c, d[0], d[1], d[2], d[3], d[4], d[5], (const int32_t*)c->key_tmp,
                      (const int32_t*)c->rank);
  for (int k = 0; k < 6; ++k) cudaMemsetAsync(d[k], 0, n * sizeof(double), c->stream);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    g_init_error = std::string("mps_init_host: ") + cudaGetErrorString(e);
    free_all(c);
    delete c;
    *out = nullptr;
    return MPS_ERR_CUDA;
  }
  return MPS_OK;
}

int mps_destroy(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  cudaStreamSynchronize(c->stream);
  free_all(c);
  delete c;
  return MPS_OK;
}

int mps_bin(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  mpsk_bin(c);
  CK(cudaGetLastError());
  return MPS_OK;
}

#define NEED_BIN(c)                                                                        \
  do {                                                                                     \
    if (!(c)) return MPS_ERR_ARG;                                                          \
    if (!(c)->binned) return fail((c), MPS_ERR_ORDER, "positions changed since the last mps_bin"); \
  } while (0)

// Skin rows left by mps_step: valid for the current positions unless the last corrector raised need_k.
static bool skin_rows_valid(mps_ctx* c) {
  if (!c->carry_rows || !c->carry_valid) return false;
  if (cudaMemcpyAsync(c->flags_host, c->flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return false;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return false;
  return c->flags_host->need_k == 0;
}

int mps_density(mps_ctx* c) {
  MPS_RANGE();
  NEED_BIN(c);
  mpsk_density(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_smooth_density(mps_ctx* c) {
  MPS_RANGE();
  NEED_BIN(c);
  mpsk_smooth_density(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_dndt(mps_ctx* c, int32_t keep) {
  MPS_RANGE();
  NEED_BIN(c);
  mpsk_dndt(c, keep ? 1 : 0);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_viscosity(mps_ctx* c) {
  MPS_RANGE();
  NEED_BIN(c);
  mpsk_viscosity(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_predict(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  mpsk_predict(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_pressure_explicit(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  mpsk_pressure_explicit(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_pressure_ppe(mps_ctx* c, int32_t* iters_out, double* relres_out) {
  MPS_RANGE();
  NEED_BIN(c);
  int rc = mpsk_pressure_ppe(c);
  if (iters_out) *iters_out = c->stats.cg_iters;
  if (relres_out) *relres_out = c->stats.cg_relres;
  if (rc == MPS_ERR_CUDA) return rc;
  int fl = read_flags(c);
  if (fl) return fl;
  return rc;
}
int mps_gradient(mps_ctx* c) {
  MPS_RANGE();
  NEED_BIN(c);
  mpsk_gradient(c);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_correct(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  mpsk_correct(c);
  CK(cudaGetLastError());
  return MPS_OK;
}

int mps_step(mps_ctx* c, int32_t nsteps, int32_t route) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  if (nsteps < 0 || (route != MPS_ROUTE_EXPLICIT && route != MPS_ROUTE_PPE))
    return fail(c, MPS_ERR_ARG, "bad nsteps or pressure_route");
  int first_err = MPS_OK;
  const bool ecs = route == MPS_ROUTE_PPE && c->prm.ppe_source == 2;
  const bool hs = route == MPS_ROUTE_PPE && c->prm.ppe_source >= 1;
  const int K = c->prm.rebin_every;
  if (nsteps > 0 && c->prm.grad_variant == 3 && !c->rho_s_ready) {
    // the smoothed density is set once, at the initial positions, from rows of every particle
    mpsk_bin(c);
    mpsk_smooth_density(c);
  }
  // rows the route needs from a skin build: the explicit route takes the re_lap part for fluid rows only
  // (viscosity); the PPE operator has rows for walls too, ECS needs n^k and (Dn/Dt)^k of every row
  const bool skin = K == 1 && c->carry_rows;
  const int skin_mode = route == MPS_ROUTE_EXPLICIT && !ecs ? ROWS_BACK_FLUID : 0;
  int64_t since_look = 0;  // steps of this call the skin policy has not seen yet
  for (int s = 0; s < nsteps; ++s) {
    if (K > 1) {
      // list reuse (Q24): bin (all rows, both radii) once every K steps at r^k; every sweep of
      // these steps walks the stored rows and re-tests the current distance
      if (c->reuse_count % K == 0) {
        c->kc.stale = 0;
        mpsk_bin(c);
      }
      c->kc.stale = 1;
      ++c->reuse_count;
    }
    if (skin && (!c->carry_valid || (c->rows_mode_built & ~skin_mode) != 0)) {
      // no skin rows yet (first step, new particles, an API-level stage call in between), or rows that
      // lack a part this route needs: make the predicated bin at r^k run
      const int up[2] = {1, 0};  // need_k, need_star
      CK(cudaMemcpyAsync(&c->flags->need_k, up, sizeof(up), cudaMemcpyHostToDevice, c->stream));
      c->rows_mode_built = skin_mode;
      ++c->win_forced;
    } else if (skin) {
      c->rows_mode_built |= skin_mode;  // a rebuild on the device during this step leaves out what this route skips
    }
    // everything up to the pressure: one replayable segment (list reuse changes the sequence from
    // step to step and runs its launches directly)
    auto pre = [&]() {
      if (skin) {
        // Q26: the rows are supersets, every sweep re-tests the distance (exact); the bin runs only if
        // the last corrector found a particle further than 0.45 skins from its build position
        c->kc.stale = 1;
        mpsk_bin(c, skin_mode, &c->flags->need_k);
      } else if (K == 1) {
        // viscosity and nu_t are computed for fluid i only; ECS also needs n^k and (Dn/Dt)^k of every row
        c->kc.stale = 0;
        mpsk_bin(c, ecs ? 0 : ROWS_FLUID_ONLY);
      }
      if (ecs) {
        mpsk_density(c);
        mpsk_dndt(c, 1);
      }
      mpsk_viscosity(c);
      mpsk_predict(c);
      if (skin) mpsk_bin(c, skin_mode, &c->flags->need_star);  // runs only if the predictor said so
      // without a skin the explicit route needs only the re_n part at r* (density, p-hat, gradient)
      else if (K == 1) mpsk_bin(c, route == MPS_ROUTE_EXPLICIT ? ROWS_RN_ONLY : 0);
      mpsk_density(c);
      if (hs) mpsk_dndt(c, 0);
      if (route == MPS_ROUTE_EXPLICIT) mpsk_pressure_explicit(c);
    };
    auto post = [&]() {
      mpsk_gradient(c);
      mpsk_correct(c);
    };
    if (K > 1) pre(); else run_segment(c, route, 0, pre);
    if (route == MPS_ROUTE_PPE) {
      // the solve is a cooperative launch of its own, between the two segments
      int rc = mpsk_pressure_ppe(c, /*sync=*/false);  // statistics are read once, after the last step
      if (rc == MPS_ERR_CUDA) return rc;
    }
    if (K > 1) post(); else run_segment(c, route, 1, post);
    c->carry_valid = skin;
    c->stats.steps_total++;
    ++since_look;
    if (skin && c->skin_auto && c->win_steps + since_look >= 16 && s + 1 < nsteps) {
      // inside a long call too: one 4-byte read-back per sixteen steps
      CK(cudaMemcpyAsync(&c->flags_host->bins, &c->flags->bins, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
      CK(cudaStreamSynchronize(c->stream));
      skin_policy(c, since_look);
      since_look = 0;
    }
  }
  c->kc.stale = 0;  // API-level sweeps always run on exact rows (they need mps_bin first)
  CK(cudaGetLastError());
  if (route == MPS_ROUTE_PPE && nsteps > 0) {
    int rc = mpsk_ppe_read_stats(c);
    if (rc == MPS_ERR_CUDA) return rc;
    if (rc) first_err = rc;
  }
  int fl = read_flags(c);
  if (skin && c->skin_auto && since_look > 0) skin_policy(c, since_look);
  if (fl) return fl;
  return first_err;
}

int mps_step_host(const mps_params* prm, int64_t n, double* x, double* y, double* z, double* u,
                  double* v, double* w, const int32_t* type, const int32_t* phase, double* p_out,
                  int32_t nsteps, int32_t route, mps_stats* stats_out, void* stream) {
  MPS_RANGE();
  mps_ctx* c = nullptr;
  int rc = mps_init_host(&c, prm, n, x, y, z, u, v, w, type, phase, stream);
  if (rc) return rc;
  rc = mps_step(c, nsteps, route);
  if (rc == MPS_ERR_CUDA || rc == MPS_ERR_ARG) {
    g_init_error = c->err;
    mps_destroy(c);
    return rc;
  }
  double* host[7] = {x, y, z, u, v, w, p_out};
  const int fields[7] = {MPS_F_X, MPS_F_Y, MPS_F_Z, MPS_F_U, MPS_F_V, MPS_F_W, MPS_F_P};
  for (int k = 0; k < 7; ++k) {
    if (!host[k]) continue;
    mpsk_get_field(c, fields[k], c->io_tmp, MPS_ORDER_ORIGINAL);
    cudaMemcpyAsync(host[k], c->io_tmp, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
  }
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (stats_out) *stats_out = c->stats;
  if (e != cudaSuccess) {
    g_init_error = std::string("mps_step_host: ") + cudaGetErrorString(e);
    rc = MPS_ERR_CUDA;
  } else if (rc) {
    g_init_error = c->err;
  }
  mps_destroy(c);
  return rc;
}

int mps_upload_host(mps_ctx* c, const double* x, const double* y, const double* z, const double* u,
                    const double* v, const double* w, const int32_t* type, const int32_t* phase) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  if (!x || !y || !z || !u || !v || !w || !type || !phase)
    return fail(c, MPS_ERR_ARG, "a particle array pointer is NULL");
  const int64_t n = c->n;
  // stage through per-particle fields that every step recomputes before reading
  double* d[6] = {c->dens, c->p, c->nut, c->b, c->phat, c->cg_x};
  const double* h[6] = {x, y, z, u, v, w};
  for (int k = 0; k < 6; ++k)
    CK(cudaMemcpyAsync(d[k], h[k], n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->key_tmp, type, n * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->rank, phase, n * 4, cudaMemcpyHostToDevice, c->stream));
  mpsk_load_particles(c, d[0], d[1], d[2], d[3], d[4], d[5], (const int32_t*)c->key_tmp,
                      (const int32_t*)c->rank);
  for (int k = 0; k < 6; ++k) cudaMemsetAsync(d[k], 0, n * sizeof(double), c->stream);
  CK(cudaGetLastError());
  c->binned = false;
  c->ppe_ready = false;
  c->reuse_count = 0;  // new particle order: the stored rows are void
  c->carry_valid = false;
  c->rho_s_ready = false;
  return MPS_OK;
}

int mps_download_host(mps_ctx* c, double* x, double* y, double* z, double* u, double* v, double* w,
                      double* p) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  double* host[7] = {x, y, z, u, v, w, p};
  const int fields[7] = {MPS_F_X, MPS_F_Y, MPS_F_Z, MPS_F_U, MPS_F_V, MPS_F_W, MPS_F_P};
  for (int k = 0; k < 7; ++k) {
    if (!host[k]) continue;
    mpsk_get_field(c, fields[k], c->io_tmp, MPS_ORDER_ORIGINAL);
    CK(cudaMemcpyAsync(host[k], c->io_tmp, c->n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  }
  CK(cudaStreamSynchronize(c->stream));
  return MPS_OK;
}

int mps_get_field(mps_ctx* c, int32_t field, void* dst, int32_t order) {
  MPS_RANGE();
  if (!c || !dst) return MPS_ERR_ARG;
  if (order != MPS_ORDER_ORIGINAL && order != MPS_ORDER_SORTED) return fail(c, MPS_ERR_ARG, "bad order");
  int rc = mpsk_get_field(c, field, dst, order);
  if (rc) return fail(c, rc, "unknown field id");
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_set_field(mps_ctx* c, int32_t field, const void* src, int32_t order) {
  MPS_RANGE();
  if (!c || !src) return MPS_ERR_ARG;
  if (order != MPS_ORDER_ORIGINAL && order != MPS_ORDER_SORTED) return fail(c, MPS_ERR_ARG, "bad order");
  int rc = mpsk_set_field(c, field, src, order);
  c->carry_valid = false;
  if (rc) return fail(c, rc, "unknown or read-only field id");
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_get_perm(mps_ctx* c, uint32_t* dst) {
  if (!c || !dst) return MPS_ERR_ARG;
  CK(cudaMemcpyAsync(dst, c->oid[c->cur], c->n * 4, cudaMemcpyDeviceToDevice, c->stream));
  return MPS_OK;
}
int mps_get_grid(mps_ctx* c, int32_t* grid) {
  if (!c || !grid) return MPS_ERR_ARG;
  grid[0] = c->kc.nx; grid[1] = c->kc.ny; grid[2] = c->kc.nz; grid[3] = c->kc.ncells;
  return MPS_OK;
}
int mps_get_cell_start(mps_ctx* c, uint32_t* dst) {
  NEED_BIN(c);
  if (!dst) return MPS_ERR_ARG;
  CK(cudaMemcpyAsync(dst, c->cell_start, ((size_t)c->kc.ncells + 1) * 4, cudaMemcpyDeviceToDevice, c->stream));
  return MPS_OK;
}
int mps_get_neighbours(mps_ctx* c, int32_t radius_id, uint32_t* counts, uint32_t* idx, int64_t cap,
                       int64_t* total) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  if (!c->binned && !skin_rows_valid(c)) return fail(c, MPS_ERR_ORDER, "positions changed since the last mps_bin");
  if (!c->binned && radius_id == MPS_RADIUS_LAP && (c->rows_mode_built & ROWS_BACK_FLUID))
    return fail(c, MPS_ERR_ORDER, "the explicit route keeps the re_lap part of fluid rows only");
  if (!counts || (radius_id != MPS_RADIUS_N && radius_id != MPS_RADIUS_LAP)) return MPS_ERR_ARG;
  int rc = mpsk_get_neighbours(c, radius_id, counts, idx, cap, total);
  CK(cudaGetLastError());
  return rc;
}
int mps_ppe_apply(mps_ctx* c, const double* x, double* y, int32_t order) {
  MPS_RANGE();
  NEED_BIN(c);
  if (!x || !y) return MPS_ERR_ARG;
  if (!c->ppe_ready) return fail(c, MPS_ERR_ORDER, "mps_ppe_apply needs mps_pressure_ppe first");
  mpsk_ppe_apply(c, x, y, order);
  CK(cudaGetLastError());
  return MPS_OK;
}
int mps_get_constants(mps_ctx* c, double* out) {
  if (!c || !out) return MPS_ERR_ARG;
  out[0] = c->kc.n0_n; out[1] = c->kc.n0_lap; out[2] = c->kc.lam; out[3] = c->kc.A_lap;
  out[4] = c->h; out[5] = c->kc.inv_h;
  return MPS_OK;
}
int mps_get_stats(mps_ctx* c, mps_stats* out) {
  MPS_RANGE();
  if (!c || !out) return MPS_ERR_ARG;
  int rc = read_flags(c);
  *out = c->stats;
  return rc == MPS_ERR_CUDA ? rc : MPS_OK;
}
int mps_sync(mps_ctx* c) {
  MPS_RANGE();
  if (!c) return MPS_ERR_ARG;
  return read_flags(c);
}
int mps_timers_enable(mps_ctx* c, int32_t on) {  // on = bit mask of categories
  if (!c) return MPS_ERR_ARG;
  if (on && c->ev_pool.empty()) {
    c->ev_pool.resize(8192);
    c->ev_cat.resize(4096);
    for (auto& e : c->ev_pool) CK(cudaEventCreate(&e));
  }
  if (!on) mps_timer_drain(c);
  c->timer_mask = (uint32_t)on;
  if (on) {
    for (int k = 0; k < MPS_NUM_TIMERS; ++k) { c->t_ms[k] = 0; c->t_launches[k] = 0; }
  }
  return MPS_OK;
}
int mps_timers_read(mps_ctx* c, double* ms, int64_t* launches) {
  if (!c) return MPS_ERR_ARG;
  mps_timer_drain(c);
  for (int k = 0; k < MPS_NUM_TIMERS; ++k) {
    if (ms) ms[k] = c->t_ms[k];
    if (launches) launches[k] = c->t_launches[k];
  }
  return MPS_OK;
}
int64_t mps_launch_count(mps_ctx* c) {
  // launches issued by the host, plus those of the skin bins that ran as conditional graph bodies (counted on the
  // device; as of the last read of the device flags: mps_step, mps_sync and mps_get_stats read them)
  return c ? c->launches + (int64_t)c->flags_host->cond_taken * c->cond_launches_per_bin : 0;
}

}  // extern "C"
