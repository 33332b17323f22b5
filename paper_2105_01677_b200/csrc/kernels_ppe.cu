// kernels_ppe.cu -- the semi-implicit pressure route (S8b of DESIGN.md):
// free-surface flags (Eq. 6), right-hand side (Eq. 8; Q5), the
// matrix-free operator with the structure of Listing 2, and the
// conjugate-gradient solve (Eq. 9; Q15).
//
// The whole solve is ONE persistent cooperative kernel (k_ppe_cg): flags and
// right-hand side, ordered compaction of the unknown rows, then the CG loop in its
// single-reduction (Chronopoulos-Gear) form with two grid barriers per iteration:
//   phase A  w = A r fused with the dot products r.r and r.w (L lanes per row,
//            shuffles inside the row group, one partial per block)
//   barrier  every block adds the partials in index order -> identical alpha, beta
//   phase B  p = r + beta p; s = w + beta s; x += alpha p; r -= alpha s
//   barrier  r (kept in pos4.w, so a neighbour gather is one 32-byte sector) is visible
// All scalars stay on the device and the convergence test is taken by every block
// from the same numbers, so there is no host poll.  In exact arithmetic the
// iterates are those of textbook CG; the matrix is never stored.
#include <algorithm>

#include "sweep_common.cuh"

namespace {

#ifdef MPS_CG_PROFILE
#include <cstdio>
#define TICK(slot) do { if (bid == 0 && tid == 0) { long long t_ = clock64(); prof[slot] += t_ - tlast; tlast = t_; } } while (0)
#else
#define TICK(slot) do { } while (0)
#endif

#ifndef MPS_CG_TPB
#define MPS_CG_TPB 1024
#endif
#ifndef MPS_CG_MINB
#define MPS_CG_MINB 1
#endif
constexpr int PPE_ILP = 4;  // independent neighbour gathers in flight per lane
constexpr int CG_TPB = MPS_CG_TPB;
constexpr int CG_MINB = MPS_CG_MINB;  // co-resident blocks per SM the register budget is set for
static_assert(CG_TPB % 256 == 0, "phase A deals rows in super-chunks of 8 warps");

struct PpeArgs {
  double4* pos4;  // .w: CG residual r during the solve, pressure at exit
  cudaTextureObject_t tex;  // pos4 as 16-byte texels (0: not used)
  const uint32_t* tp;
  const double* dens;
  const double* dndt;      // (Dn/Dt)* (ppe_source >= 1)
  const double2* keep2;    // (n^k, (Dn/Dt)^k) (ppe_source == 2)
  int8_t* bc;
  double* b;
  double* x;
  double* pv;
  double* sv;
  double* wv;
  double* p;
  const uint32_t* nbr;
  const uint32_t* cn;
  const uint32_t* co;
  uint32_t* rows;
  uint32_t* bcount;  // 2 per block: rows, surface
  double* part;      // 2 per block
  CgScalars* cg;
  GridBar* bar;
  double tol2;
  int maxit;
};

// ---- block-wide sum of two values, result broadcast to every thread ---------------
// warp shuffles, one partial per warp in shared memory, the first warp folds them in
// a fixed order, the result is broadcast: two block barriers.
template <int NT>
__device__ __forceinline__ void block_sum2(double& a, double& b) {
  __shared__ double sh[2][NT / 32];
  __shared__ double res[2];
  a = warp_sum(a);
  b = warp_sum(b);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) { sh[0][wid] = a; sh[1][wid] = b; }
  __syncthreads();
  if (wid == 0) {
    double sa = lane < NT / 32 ? sh[0][lane] : 0.0;
    double sb = lane < NT / 32 ? sh[1][lane] : 0.0;
    sa = warp_sum(sa);
    sb = warp_sum(sb);
    if (lane == 0) { res[0] = sa; res[1] = sb; }
  }
  __syncthreads();
  a = res[0];
  b = res[1];
  // the next call's writes to sh/res come after its own first barrier at the earliest for
  // sh (written before the barrier by lane 0 of each warp: all reads of sh above are done
  // by warp 0 before the second barrier) and after both barriers for res
}

// ---- grid barrier (all blocks are co-resident: cooperative launch) ----------------
// One monotonically increasing arrival counter: thread 0 of every block adds 1 with
// release semantics and spins (acquire) until the count reaches nb x generation, so
// a barrier costs one L2 round trip for the arrival plus the polls -- there is no
// second "last block flips the flag" hop.  The fence after the spin makes every
// later plain load of the block see the other blocks' writes (it invalidates the
// SM's L1).  A spin that lasts longer than about two seconds raises barrier_timeout
// and lets the kernel drain instead of hanging.
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned int* p, unsigned int v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ bool grid_barrier(GridBar* bar, unsigned int& gen, CgScalars* cg) {
  __shared__ int dead;
  __syncthreads();
  if (threadIdx.x == 0) {
    dead = 0;
    gen += gridDim.x;  // arrivals expected once this barrier is complete
    red_release_add_u32(&bar->count, 1u);
    long long t0 = 0;
    unsigned int polls = 0;
    while ((int)(ld_acquire_u32(&bar->count) - gen) < 0) {
      if ((++polls & 1023u) == 0u) {
        if (t0 == 0) t0 = clock64();
        else if (clock64() - t0 > 4000000000LL) {
          cg->barrier_timeout = 1;
          dead = 1;
          break;
        }
      }
    }
    __threadfence();
  }
  __syncthreads();
  return dead == 0;
}

// ---- one row of y = A r ------------------------------------------------------------
// (A r)_i = sum_{j in N(i, re_lap), j not dummy} c_ij (r_i - r_j) + compress/dt^2 r_i,
// c_ij = A_lap w(r_ij) / rho_ij (Listing 2; Q5, Q6).  r_j is read from
// pos4.w, which is 0 on free-surface slots (Dirichlet p = 0).  The L lanes of the
// group each take every L-th entry; the result is valid in every lane.
template <bool TWO_PHASE, int L, bool TEX>
__device__ __forceinline__ double ppe_row(const KConst& kc, const double4* pos4, cudaTextureObject_t tex,
                                          const uint32_t* tp,
                                          const uint32_t* nbr, const uint32_t* cn, const uint32_t* co,
                                          int i, int sub, bool live, double& ri) {
  // every lane of the warp must come through here (full-mask shuffles below): a
  // group without a row passes live = false and any valid i
  const double4 pi = pos4[i];
  ri = pi.w;
  const uint32_t* row = row_ptr(nbr, kc.stride, i);
  const uint32_t nf = live ? cn[i] : 0u;
  const uint32_t m = live ? nf + co[i] : 0u;
  // 1 / rho_ij for a neighbour of phase 0 and of phase 1 (Q6): two values per row, no division per pair
  const int ph_i = TWO_PHASE ? (int)((tp[i] >> 8) & 1) : 0;
  const double inv_rij0 = kc.inv_rho_pair[ph_i][0], inv_rij1 = kc.inv_rho_pair[ph_i][1];
  const bool hl = kc.ppe_laplacian == 1;
  double s = 0.0;
  // batches of PPE_ILP entries per lane: entry loads, then gathers, then arithmetic, so the
  // L2 round trips of one batch overlap (the L1 is invalidated by every grid barrier).
  // An empty or dummy slot takes a point at distance re_lap on the x axis: its weight is
  // re_lap / re_lap - 1 = 0 exactly.
  for (uint32_t k = sub; k < m; k += PPE_ILP * L) {
    uint32_t e[PPE_ILP];
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const uint32_t kk = k + (uint32_t)(u * L);
      e[u] = kk < m ? row_entry(row, kc.stride, nf, kk) : NB_DUMMY;
    }
    double4 q[PPE_ILP];
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      if (e[u] & NB_DUMMY) q[u] = make_double4(pi.x + kc.re_lap, pi.y, pi.z, pi.w);
      else if (TEX) {
        // (x, y) never change during a solve: fetched through the texture front end, which works
        // in parallel with the LSU; (z, r) -- r changes every iteration -- take the coherent path
        const uint32_t j = e[u] & NB_INDEX;
        const int4 xy = tex1Dfetch<int4>(tex, 2 * (int)j);
        const double2 zr = reinterpret_cast<const double2*>(pos4 + j)[1];
        q[u] = make_double4(__hiloint2double(xy.y, xy.x), __hiloint2double(xy.w, xy.z), zr.x, zr.y);
      } else q[u] = pos4[e[u] & NB_INDEX];
    }
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const double dx = q[u].x - pi.x, dy = q[u].y - pi.y, dz = q[u].z - pi.z;
      const double r2 = pair_r2(dx, dy, dz, kc.stale);
      const double ir = rsqrt_f64(r2);
      // Eq. 10 form: A_lap (re/r - 1); MPS-HL (Eq. 16, Q23): (2 re / n0) / r^3
      double w = hl ? ir * ir * ir : kernel_w(kc.kernel, kc.re_lap, kc.inv_re_lap, r2, ir);
      if (TWO_PHASE) {
        w *= (e[u] & NB_PHASE1) ? inv_rij1 : inv_rij0;
      }
      if ((e[u] & NB_DUMMY) || (kc.stale && !(r2 < kc.re_lap2))) w = 0.0;  // dummy, empty slot, or left the radius
      s = fma(w, pi.w - q[u].w, s);
    }
  }
  s = group_sum<L>(s);
  if (!TWO_PHASE) s *= 1.0 / kc.rho[0];
  return fma(hl ? kc.hl_c : kc.A_lap, s, kc.compress_dt2 * pi.w);
}

// ---- the persistent solve -------------------------------------------------------------
template <bool TWO_PHASE, int L, bool TEX>
__global__ void __launch_bounds__(CG_TPB, CG_MINB)
k_ppe_cg(KConst kc, PpeArgs a) {
  __shared__ uint32_t sh_cnt[2][CG_TPB / 32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int nb = (int)gridDim.x, bid = (int)blockIdx.x;
  unsigned int gen = 0;
#ifdef MPS_CG_PROFILE
  long long prof[8] = {0, 0, 0, 0, 0, 0, 0, 0}, tlast = clock64();
#endif

  // -- S8b-1, S8b-2: flags and right-hand side over this block's contiguous chunk --------
  const int chunk = (kc.n + nb - 1) / nb;
  const int lo = min(bid * chunk, kc.n), hi = min(lo + chunk, kc.n);
  {
    double bb = 0.0, dummy = 0.0;
    uint32_t n_rows = 0, n_surf = 0;
    for (int i = lo + tid; i < hi; i += CG_TPB) {
      const uint32_t ty = a.tp[i] & 0xff;
      int8_t f;
      double bi = 0.0;
      const double ni = a.dens[i];
      if (ty == MPS_DUMMY || ty == MPS_GHOST) f = -1;
      else if (ni < kc.beta * kc.n0_n) { f = 1; ++n_surf; }
      else {
        f = 0;
        ++n_rows;
        if (kc.ppe_source == 0) {         // Eq. 8 divided by -rho (Q5)
          bi = kc.relax_dt2 * (ni - kc.n0_n) / kc.n0_n;
        } else if (kc.ppe_source == 1) {  // MPS-HS, Eq. 15 (Q22)
          bi = kc.relax / (kc.n0_n * kc.dt) * a.dndt[i];
        } else {                          // HS + error-compensating parts, Eq. 17-18 (Q22)
          const double2 kk = a.keep2[i];
          const double alpha = (kk.x - kc.n0_n) / kc.n0_n;
          const double beta = kc.dt / kc.n0_n * kk.y;
          const double ecs = fabs(alpha) * (kk.y / kc.n0_n) + fabs(beta) * (alpha / kc.dt);
          bi = kc.relax / kc.dt * (a.dndt[i] / kc.n0_n + ecs);
        }
      }
      a.bc[i] = f;
      a.b[i] = bi;
      a.x[i] = 0.0;
      a.pv[i] = 0.0;
      a.sv[i] = 0.0;
      a.pos4[i].w = bi;  // r0 = b
      bb += bi * bi;
    }
    block_sum2<CG_TPB>(bb, dummy);
    n_rows = __reduce_add_sync(0xffffffffu, n_rows);
    n_surf = __reduce_add_sync(0xffffffffu, n_surf);
    if (lane == 0) { sh_cnt[0][wid] = n_rows; sh_cnt[1][wid] = n_surf; }
    __syncthreads();
    if (tid == 0) {
      uint32_t r = 0, s = 0;
      for (int k = 0; k < CG_TPB / 32; ++k) { r += sh_cnt[0][k]; s += sh_cnt[1][k]; }
      a.bcount[2 * bid] = r;
      a.bcount[2 * bid + 1] = s;
      a.part[2 * bid] = bb;
      a.part[2 * bid + 1] = 0.0;
    }
  }
  if (!grid_barrier(a.bar, gen, a.cg)) return;

  // -- totals and this block's offset into the compacted row list ------------------------
  double bb = 0.0;
  int n_rows = 0, n_surf = 0, row_off = 0;
  {
    double v = 0.0, dummy = 0.0;
    uint32_t r = 0, s = 0, before = 0;
    for (int k = tid; k < nb; k += CG_TPB) {
      v += __ldcg(&a.part[2 * k]);
      const uint32_t rk = __ldcg(&a.bcount[2 * k]);
      r += rk;
      s += __ldcg(&a.bcount[2 * k + 1]);
      if (k < bid) before += rk;
    }
    block_sum2<CG_TPB>(v, dummy);
    bb = v;
    double fr = (double)r, fs = (double)s;
    block_sum2<CG_TPB>(fr, fs);
    double fb = (double)before;
    block_sum2<CG_TPB>(fb, dummy);
    n_rows = (int)fr;
    n_surf = (int)fs;
    row_off = (int)fb;
  }
  // ordered compaction: rows[] ascending in slot index
  for (int base = lo; base < hi; base += CG_TPB) {
    const int i = base + tid;
    const bool is_row = (i < hi) && (a.bc[i] == 0);
    const uint32_t m = __ballot_sync(0xffffffffu, is_row);
    __syncthreads();
    if (lane == 0) sh_cnt[0][wid] = (uint32_t)__popc(m);
    __syncthreads();
    uint32_t off = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < CG_TPB / 32; ++k) {
      const uint32_t ck = sh_cnt[0][k];
      if (k < wid) off += ck;
      tot += ck;
    }
    if (is_row) a.rows[row_off + off + (uint32_t)__popc(m & ((1u << lane) - 1u))] = (uint32_t)i;
    row_off += (int)tot;
  }
  if (!grid_barrier(a.bar, gen, a.cg)) return;

  TICK(0);
  // -- S8b-3, S8b-4: conjugate gradients ---------------------------------------------------
  const double tol2bb = a.tol2 * bb;
  int iters = 0, converged = (bb == 0.0) ? 1 : 0;
  double gam = bb, gamma_old = 1.0, alpha_old = 1.0;
  const int gthreads = nb * CG_TPB;
  const int gtid = bid * CG_TPB + tid;
  const int sub = tid & (L - 1);
  if (!converged) {
    for (;;) {
      // phase A: w = A r, gamma = r.r, delta = r.w
      double g_part = 0.0, d_part = 0.0;
      // Rows are dealt to the blocks in super-chunks of 8 warps (8 * 32 / L consecutive rows, so
      // the warps that share an SM's L1 work on neighbouring rows) round-robin over the grid:
      // every block gets an even sample of cheap (wall) and expensive (fluid) rows and at most
      // one super-chunk more than any other.  The trip count is warp-uniform.
      constexpr int GPW = 32 / L;        // row groups per warp
      constexpr int SCW = 8;             // warps per super-chunk
      for (int sc = (wid / SCW) * nb + bid; sc * (SCW * GPW) < n_rows; sc += (CG_TPB / 32 / SCW) * nb) {
        const int g = sc * (SCW * GPW) + (wid % SCW) * GPW + (lane / L);
        const bool live = g < n_rows;
        const int i = live ? (int)a.rows[g] : 0;
        double ri;
        const double wi = ppe_row<TWO_PHASE, L, TEX>(kc, a.pos4, a.tex, a.tp, a.nbr, a.cn, a.co, i, sub, live, ri);
        if (live && sub == 0) {
          a.wv[i] = wi;
          g_part = fma(ri, ri, g_part);
          d_part = fma(ri, wi, d_part);
        }
      }
      TICK(1);
      block_sum2<CG_TPB>(g_part, d_part);
      if (tid == 0) {
        a.part[2 * bid] = g_part;
        a.part[2 * bid + 1] = d_part;
      }
      TICK(2);
      if (!grid_barrier(a.bar, gen, a.cg)) return;
      TICK(3);
      double del = 0.0;
      gam = 0.0;
      for (int k = tid; k < nb; k += CG_TPB) {
        gam += __ldcg(&a.part[2 * k]);
        del += __ldcg(&a.part[2 * k + 1]);
      }
      block_sum2<CG_TPB>(gam, del);
      TICK(4);
      if (gam <= tol2bb) { converged = 1; break; }
      if (iters >= a.maxit) break;
      double alpha, beta;
      if (iters == 0) {
        beta = 0.0;
        alpha = gam / del;
      } else {
        beta = gam / gamma_old;
        alpha = gam / (del - beta * gam / alpha_old);
      }
      gamma_old = gam;
      alpha_old = alpha;
      ++iters;
      // phase B: p = r + beta p; s = w + beta s; x += alpha p; r -= alpha s
      for (int g = gtid; g < n_rows; g += gthreads) {
        const int i = (int)a.rows[g];
        const double r = a.pos4[i].w;
        const double pn = fma(beta, a.pv[i], r);
        const double sn = fma(beta, a.sv[i], a.wv[i]);
        a.pv[i] = pn;
        a.sv[i] = sn;
        a.x[i] = fma(alpha, pn, a.x[i]);
        a.pos4[i].w = fma(-alpha, sn, r);
      }
      TICK(5);
      if (!grid_barrier(a.bar, gen, a.cg)) return;
      TICK(6);
    }
  }

  // -- S8b-5: pressures from x (Q4), staged into pos4.w for the gradient ------------------
  for (int i = gtid; i < kc.n; i += gthreads) {
    double v = (a.bc[i] == 0) ? a.x[i] : 0.0;
    if (kc.clamp_negative_p && v < 0.0) v = 0.0;
    a.p[i] = v;
    a.pos4[i].w = v;
  }
#ifdef MPS_CG_PROFILE
  if (bid == 0 && tid == 0)
    printf("cg profile (block 0, kcycles): setup %lld | phaseA %lld | blocksum %lld | barrier1 %lld | reduce %lld | phaseB %lld | barrier2 %lld | iters %d\n",
           prof[0] / 1000, prof[1] / 1000, prof[2] / 1000, prof[3] / 1000, prof[4] / 1000, prof[5] / 1000, prof[6] / 1000, iters);
#endif
  if (bid == 0 && tid == 0) {
    a.cg->gamma = gam;
    a.cg->bb = bb;
    a.cg->tol2bb = tol2bb;
    a.cg->iters = iters;
    a.cg->maxit = a.maxit;
    a.cg->done = 1;
    a.cg->converged = converged;
    a.cg->n_rows = n_rows;
    a.cg->n_surface = n_surf;
  }
}

// ---- y = A x for the tests (mps_ppe_apply): stage, apply, read back ---------------------
__global__ void k_stage_in(int n, int order, const int8_t* __restrict__ bc, const uint32_t* __restrict__ oid,
                           const double* __restrict__ src, double4* __restrict__ pos4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v = src[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i];
  pos4[i].w = (bc[i] == 0) ? v : 0.0;
}
template <bool TWO_PHASE, int L>
__global__ void __launch_bounds__(256)
k_ppe_apply(KConst kc, const double4* pos4, const uint32_t* __restrict__ tp, const int8_t* __restrict__ bc,
            const uint32_t* __restrict__ nbr, const uint32_t* __restrict__ cn,
            const uint32_t* __restrict__ co, double* __restrict__ wv) {
  const int i = (int)((blockIdx.x * 256u + threadIdx.x) / L);
  const int sub = threadIdx.x & (L - 1);
  const bool in = i < kc.n;
  const bool live = in && bc[i] == 0;
  double ri;
  const double wi = ppe_row<TWO_PHASE, L, false>(kc, pos4, 0, tp, nbr, cn, co, in ? i : 0, sub, live, ri);
  if (in && sub == 0) wv[i] = live ? wi : 0.0;
}
__global__ void k_stage_out(int n, int order, const uint32_t* __restrict__ oid,
                            const double* __restrict__ src, double* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = src[i];
}

template <bool TWO_PHASE, int L, bool TEX>
cudaError_t launch_cg(mps_ctx* c, PpeArgs& a, int grid) {
  void* params[] = {(void*)&c->kc, (void*)&a};
  return cudaLaunchCooperativeKernel((const void*)k_ppe_cg<TWO_PHASE, L, TEX>, dim3(grid), dim3(CG_TPB),
                                     params, 0, c->stream);
}
template <bool TWO_PHASE, int L, bool TEX>
int cg_blocks_per_sm() {
  int nb = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_ppe_cg<TWO_PHASE, L, TEX>, CG_TPB, 0);
  return nb;
}

bool two_phase(const mps_ctx* c) { return c->prm.n_phases > 1 && c->prm.rho[0] != c->prm.rho[1]; }

}  // namespace

// ============================================================ host launchers ===
// Number of co-resident blocks of the persistent kernel (called once at init).
int mpsk_ppe_plan(mps_ctx* c) {
  int per_sm = 2;
  const bool tp = two_phase(c);
  c->cg_lanes = 8;  // 4 and 16 lanes per row measured within 5 % of 8
  if (c->cg_tex) per_sm = tp ? cg_blocks_per_sm<true, 8, true>() : cg_blocks_per_sm<false, 8, true>();
  else per_sm = tp ? cg_blocks_per_sm<true, 8, false>() : cg_blocks_per_sm<false, 8, false>();
  if (per_sm < 1) return MPS_ERR_CUDA;
  if (per_sm > CG_MINB) per_sm = CG_MINB;
  c->cg_grid = per_sm * c->sm_count;
  return MPS_OK;
}

int mpsk_pressure_ppe(mps_ctx* c) {
  const int cur = c->cur;
  PpeArgs a;
  a.pos4 = c->pos4[cur]; a.tex = c->cg_tex ? c->pos_tex[cur] : 0; a.tp = c->tp[cur]; a.dens = c->dens; a.dndt = c->dndt; a.keep2 = c->keep2[cur]; a.bc = c->bc; a.b = c->b;
  a.x = c->cg_x; a.pv = c->cg_p; a.sv = c->cg_s; a.wv = c->cg_w; a.p = c->p;
  a.nbr = c->nbr; a.cn = c->cn; a.co = c->co; a.rows = c->cg_rows; a.bcount = c->cg_bcount;
  a.part = c->cg_part; a.cg = c->cg; a.bar = c->cg_bar;
  a.tol2 = c->prm.cg_rtol * c->prm.cg_rtol;
  a.maxit = c->prm.cg_maxit;
  // small problems: no more blocks than there is work for (fewer arrivals per barrier)
  int grid = c->cg_grid;
  const int want = std::max(c->sm_count, div_up((int64_t)c->n * c->cg_lanes, CG_TPB));
  if (grid > want) grid = want;
  cudaMemsetAsync(c->cg_bar, 0, sizeof(GridBar), c->stream);
  if (((c)->timer_mask >> MPS_T_CG_SPMV) & 1u) mps_timer_begin(c, MPS_T_CG_SPMV);
  cudaError_t e;
  const bool tp = two_phase(c);
  if (c->cg_tex) e = tp ? launch_cg<true, 8, true>(c, a, grid) : launch_cg<false, 8, true>(c, a, grid);
  else e = tp ? launch_cg<true, 8, false>(c, a, grid) : launch_cg<false, 8, false>(c, a, grid);
  c->launches++;
  c->t_launches[MPS_T_CG_SPMV]++;
  if (((c)->timer_mask >> MPS_T_CG_SPMV) & 1u) mps_timer_end(c, MPS_T_CG_SPMV);
  if (e != cudaSuccess) {
    c->err = std::string("cooperative launch of k_ppe_cg failed: ") + cudaGetErrorString(e);
    return MPS_ERR_CUDA;
  }
  c->ppe_ready = true;
  c->posw_is_p = true;
  cudaMemcpyAsync(c->cg_host, c->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, c->stream);
  e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    c->err = std::string("CUDA error in mps_pressure_ppe: ") + cudaGetErrorString(e);
    return MPS_ERR_CUDA;
  }
  const CgScalars& s = *c->cg_host;
  if (s.barrier_timeout) {
    c->err = "grid barrier timed out inside k_ppe_cg";
    return MPS_ERR_CUDA;
  }
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
  c->posw_is_p = false;
  const int grid = div_up((int64_t)n * 8, 256);
  if (two_phase(c)) {
    MPS_LAUNCH(c, MPS_T_PPE_SETUP, (k_ppe_apply<true, 8>), grid, 256, c->kc, c->pos4[cur], c->tp[cur],
               c->bc, c->nbr, c->cn, c->co, c->cg_w);
  } else {
    MPS_LAUNCH(c, MPS_T_PPE_SETUP, (k_ppe_apply<false, 8>), grid, 256, c->kc, c->pos4[cur], c->tp[cur],
               c->bc, c->nbr, c->cn, c->co, c->cg_w);
  }
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_out, div_up(n, 256), 256, n, order, c->oid[cur], c->cg_w, y);
  return MPS_OK;
}
