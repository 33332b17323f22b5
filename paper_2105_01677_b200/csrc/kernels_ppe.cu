// kernels_ppe.cu -- the semi-implicit pressure route (S8b of DESIGN.md):
// free-surface flags (Eq. 6), right-hand side (Eq. 8; Q5), the
// matrix-free operator with the structure of Listing 2, and the
// conjugate-gradient solve (Eq. 9; Q15).
//
// CG is run in the single-reduction (Chronopoulos-Gear) form: one operator
// kernel per iteration computes w = A r fused with the two dot products r.r and
// r.w (warp shuffles, one partial per block, the last block to finish reduces
// them in a fixed order and derives alpha and beta); one update kernel then
// advances p, s = A p, x and r.  All scalars stay on the device; the host only
// polls a done flag every few iterations.  In exact arithmetic the iterates are
// those of textbook CG; the matrix is never stored.
#include "mps_internal.h"

namespace {

constexpr int TPB = 128;

__device__ __forceinline__ const uint32_t* row_of(const uint32_t* nbr, int cap, int i) {
  return nbr + ((size_t)(i >> 5) * cap) * 32 + (i & 31);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Block-wide sum of two values; result valid in thread 0.
__device__ __forceinline__ void block_sum2(double& a, double& b) {
  __shared__ double sh[2][TPB / 32];
  a = warp_sum(a);
  b = warp_sum(b);
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { sh[0][wid] = a; sh[1][wid] = b; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double sa = 0.0, sb = 0.0;
#pragma unroll
    for (int k = 0; k < TPB / 32; ++k) { sa += sh[0][k]; sb += sh[1][k]; }
    a = sa;
    b = sb;
  }
  __syncthreads();
}

// Publishes this block's partial sums; the last block to arrive adds all
// partials in index order (deterministic) and returns true in its thread 0.
__device__ __forceinline__ bool grid_sum2(double& a, double& b, double* part, unsigned int* counter) {
  __shared__ bool last;
  block_sum2(a, b);
  if (threadIdx.x == 0) {
    part[2 * blockIdx.x] = a;
    part[2 * blockIdx.x + 1] = b;
    __threadfence();
    unsigned int t = atomicAdd(counter, 1u);
    last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!last) return false;
  __threadfence();
  double sa = 0.0, sb = 0.0;
  for (int k = threadIdx.x; k < (int)gridDim.x; k += TPB) {
    sa += __ldcg(&part[2 * k]);
    sb += __ldcg(&part[2 * k + 1]);
  }
  block_sum2(sa, sb);
  a = sa;
  b = sb;
  if (threadIdx.x == 0) *counter = 0;
  return threadIdx.x == 0;
}

// -------------------------------------------------- S8b-1, S8b-2: flags + rhs ---
__global__ void __launch_bounds__(TPB)
k_ppe_setup(KConst kc, double tol2, int maxit, double4* __restrict__ pos4,
            const uint32_t* __restrict__ tp, const double* __restrict__ dens, int8_t* __restrict__ bc,
            double* __restrict__ b, double* __restrict__ x, double* __restrict__ pv,
            double* __restrict__ sv, double* __restrict__ part, CgScalars* __restrict__ cg) {
  double bb = 0.0, cnt = 0.0;
  int n_surf = 0, n_rows = 0;
  for (int i = blockIdx.x * TPB + threadIdx.x; i < kc.n; i += gridDim.x * TPB) {
    uint32_t ty = tp[i] & 0xff;
    int8_t f;
    double bi = 0.0;
    if (ty == MPS_DUMMY || ty == MPS_GHOST) f = -1;
    else if (dens[i] < kc.beta * kc.n0_n) { f = 1; ++n_surf; }
    else {
      f = 0;
      ++n_rows;
      bi = kc.relax_dt2 * (dens[i] - kc.n0_n) / kc.n0_n;
    }
    bc[i] = f;
    b[i] = bi;
    x[i] = 0.0;
    pv[i] = 0.0;
    sv[i] = 0.0;
    pos4[i].w = bi;  // r0 = b
    bb += bi * bi;
  }
  cnt = (double)(n_surf) + 67108864.0 * (double)n_rows;  // two counters in one exact double
  if (grid_sum2(bb, cnt, part, &cg->blocks_done)) {
    double rows = floor(cnt / 67108864.0);
    cg->n_rows = (int)rows;
    cg->n_surface = (int)(cnt - rows * 67108864.0);
    cg->bb = bb;
    cg->tol2bb = tol2 * bb;
    cg->gamma = bb;
    cg->delta = 0.0;
    cg->gamma_old = 1.0;
    cg->alpha_old = 1.0;
    cg->alpha = 0.0;
    cg->beta = 0.0;
    cg->iters = 0;
    cg->maxit = maxit;
    cg->done = (bb == 0.0) ? 1 : 0;
    cg->converged = (bb == 0.0) ? 1 : 0;
  }
}

// ------------------------------------------------------ S8b-3: y = A r (+ dots) ---
// (A r)_i = sum_{j in N(i, re_lap), j not dummy} c_ij (r_i - r_j) + compress/dt^2 r_i
// with c_ij = A_lap w(r_ij) / rho_ij, on rows bc_i = 0.  r_j is read from pos4.w,
// which is 0 on free-surface slots (Dirichlet p = 0) by construction.
template <bool TWO_PHASE, bool REDUCE>
__global__ void __launch_bounds__(TPB)
k_cg_spmv(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ tp,
          const int8_t* __restrict__ bc, const uint32_t* __restrict__ nbr,
          const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co, double* __restrict__ wv,
          double* __restrict__ part, CgScalars* __restrict__ cg) {
  if (REDUCE) {
    if (cg->done) return;
  }
  double gam = 0.0, del = 0.0;
  const double inv_rho0 = 1.0 / kc.rho[0];
  for (int i = blockIdx.x * TPB + threadIdx.x; i < kc.n; i += gridDim.x * TPB) {
    if (bc[i] != 0) {
      if (!REDUCE) wv[i] = 0.0;
      continue;
    }
    const double4 pi = pos4[i];
    const uint32_t* row = row_of(nbr, kc.cap, i);
    const uint32_t nf = cn[i], nb = co[i];
    const double rho_i = TWO_PHASE ? kc.rho[(tp[i] >> 8) & 1] : kc.rho[0];
    double s = 0.0;
    auto term = [&](uint32_t e) {
      if (e & NB_DUMMY) return;
      double4 q = pos4[e & NB_INDEX];
      double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
      double r2 = dx * dx + dy * dy + dz * dz;
      double w = kc.re_lap * rsqrt(r2) - 1.0;
      if (TWO_PHASE) {
        double rho_j = kc.rho[(e & NB_PHASE1) ? 1 : 0];
        double rij = kc.rho_pair_mean == 1 ? 2.0 * rho_i * rho_j / (rho_i + rho_j) : 0.5 * (rho_i + rho_j);
        w = w / rij;
      }
      s += w * (pi.w - q.w);
    };
    for (uint32_t k = 0; k < nf; ++k) term(row[(size_t)k * 32]);
    for (uint32_t k = 0; k < nb; ++k) term(row[(size_t)(kc.cap - 1 - k) * 32]);
    if (!TWO_PHASE) s *= inv_rho0;
    double wi = kc.A_lap * s + kc.compress_dt2 * pi.w;
    wv[i] = wi;
    gam += pi.w * pi.w;
    del += pi.w * wi;
  }
  if (!REDUCE) return;
  if (grid_sum2(gam, del, part, &cg->blocks_done)) {
    cg->gamma = gam;
    cg->delta = del;
    if (gam <= cg->tol2bb) {
      cg->done = 1;
      cg->converged = 1;
    } else if (cg->iters >= cg->maxit) {
      cg->done = 1;
      cg->converged = 0;
    } else {
      double beta, alpha;
      if (cg->iters == 0) {
        beta = 0.0;
        alpha = gam / del;
      } else {
        beta = gam / cg->gamma_old;
        alpha = gam / (del - beta * gam / cg->alpha_old);
      }
      cg->alpha = alpha;
      cg->beta = beta;
      cg->gamma_old = gam;
      cg->alpha_old = alpha;
      cg->iters += 1;
    }
  }
}

// ------------------------------------------------------------ S8b-4: CG update ---
// p = r + beta p; s = w + beta s; x += alpha p; r -= alpha s (rows only).
__global__ void __launch_bounds__(256)
k_cg_update(int n, const int8_t* __restrict__ bc, double4* __restrict__ pos4,
            const double* __restrict__ wv, double* __restrict__ pv, double* __restrict__ sv,
            double* __restrict__ x, const CgScalars* __restrict__ cg) {
  if (cg->done) return;
  const double alpha = cg->alpha, beta = cg->beta;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < n; i += gridDim.x * 256) {
    if (bc[i] != 0) continue;
    double r = pos4[i].w;
    double p = r + beta * pv[i];
    double s = wv[i] + beta * sv[i];
    pv[i] = p;
    sv[i] = s;
    x[i] += alpha * p;
    pos4[i].w = r - alpha * s;
  }
}

// ---------------------------------------------------- S8b-5: pressures from x ---
__global__ void k_ppe_finish(KConst kc, const int8_t* __restrict__ bc, const double* __restrict__ x,
                             double* __restrict__ p) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  double v = (bc[i] == 0) ? x[i] : 0.0;
  if (kc.clamp_negative_p && v < 0.0) v = 0.0;
  p[i] = v;
}

// stage a caller vector into pos4.w (rows only) / read a vector back
__global__ void k_stage_in(int n, int order, const int8_t* __restrict__ bc, const uint32_t* __restrict__ oid,
                           const double* __restrict__ src, double4* __restrict__ pos4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v = src[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i];
  pos4[i].w = (bc[i] == 0) ? v : 0.0;
}
__global__ void k_stage_out(int n, int order, const uint32_t* __restrict__ oid,
                            const double* __restrict__ src, double* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = src[i];
}

int spmv_grid(mps_ctx* c) {
  int need = div_up(c->n, TPB);
  int cap = c->sm_count * 8;
  return need < cap ? need : cap;
}

template <bool REDUCE>
void launch_spmv(mps_ctx* c, int cat) {
  int cur = c->cur;
  int grid = spmv_grid(c);
  if (c->prm.n_phases > 1 && c->prm.rho[0] != c->prm.rho[1]) {
    MPS_LAUNCH(c, cat, (k_cg_spmv<true, REDUCE>), grid, TPB, c->kc, c->pos4[cur], c->tp[cur], c->bc,
               c->nbr, c->cn, c->co, c->cg_w, c->cg_part, c->cg);
  } else {
    MPS_LAUNCH(c, cat, (k_cg_spmv<false, REDUCE>), grid, TPB, c->kc, c->pos4[cur], c->tp[cur], c->bc,
               c->nbr, c->cn, c->co, c->cg_w, c->cg_part, c->cg);
  }
}

}  // namespace

// ============================================================ host launchers ===
int mpsk_pressure_ppe(mps_ctx* c) {
  const int n = (int)c->n;
  const int cur = c->cur;
  const int grid = spmv_grid(c);
  const double tol2 = c->prm.cg_rtol * c->prm.cg_rtol;
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_ppe_setup, grid, TPB, c->kc, tol2, c->prm.cg_maxit, c->pos4[cur],
             c->tp[cur], c->dens, c->bc, c->b, c->cg_x, c->cg_p, c->cg_s, c->cg_part, c->cg);
  c->ppe_ready = true;
  const int POLL = 8;
  const int ugrid = std::min(div_up(n, 256), c->sm_count * 8);
  int batches = 0;
  bool done = false;
  // pipelined polling: batch k is enqueued before the host looks at batch k-1
  while (!done) {
    for (int it = 0; it < POLL; ++it) {
      launch_spmv<true>(c, MPS_T_CG_SPMV);
      MPS_LAUNCH(c, MPS_T_CG_UPDATE, k_cg_update, ugrid, 256, n, c->bc, c->pos4[cur], c->cg_w, c->cg_p,
                 c->cg_s, c->cg_x, c->cg);
    }
    if (batches > 0) {
      cudaEventSynchronize(c->poll_event);
      if (c->cg_host->done) done = true;
    }
    if (!done) {
      cudaMemcpyAsync(c->cg_host, c->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, c->stream);
      cudaEventRecord(c->poll_event, c->stream);
    }
    ++batches;
    if ((int64_t)batches * POLL > (int64_t)c->prm.cg_maxit + 4 * POLL) break;  // safety net
  }
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_ppe_finish, div_up(n, 256), 256, c->kc, c->bc, c->cg_x, c->p);
  cudaMemcpyAsync(c->cg_host, c->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, c->stream);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    c->err = std::string("CUDA error in mps_pressure_ppe: ") + cudaGetErrorString(e);
    return MPS_ERR_CUDA;
  }
  const CgScalars& s = *c->cg_host;
  c->stats.cg_iters = s.iters;
  c->stats.cg_converged = s.converged;
  c->stats.cg_relres = s.bb > 0.0 ? sqrt(s.gamma / s.bb) : 0.0;
  c->stats.n_surface = s.n_surface;
  c->stats.n_rows = s.n_rows;
  c->stats.cg_iters_total += s.iters;
  if (!s.converged) {
    c->err = "CG reached cg_maxit without meeting cg_rtol";
    return MPS_ERR_NOCONV;
  }
  return MPS_OK;
}

int mpsk_ppe_apply(mps_ctx* c, const double* x, double* y, int order) {
  const int n = (int)c->n;
  const int cur = c->cur;
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_in, div_up(n, 256), 256, n, order, c->bc, c->oid[cur], x,
             c->pos4[cur]);
  launch_spmv<false>(c, MPS_T_PPE_SETUP);
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_out, div_up(n, 256), 256, n, order, c->oid[cur], c->cg_w, y);
  return MPS_OK;
}
