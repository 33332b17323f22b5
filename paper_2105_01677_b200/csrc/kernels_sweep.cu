// kernels_sweep.cu -- the fixed-radius sweeps over the per-step neighbour rows
// (density S4, Smagorinsky S5, viscosity S6, p-hat S9, gradient S10) and the
// streaming updates (predictor S7, equation of state S8a, corrector S11).
// One thread per particle; entry k of the 32 particles of a warp is one
// coalesced 128-byte line; each neighbour costs one 32-byte sector gather.
#include "mps_internal.h"

namespace {

constexpr int TPB = 128;

__device__ __forceinline__ const uint32_t* row_of(const uint32_t* nbr, int cap, int i) {
  return nbr + ((size_t)(i >> 5) * cap) * 32 + (i & 31);
}
// w(r) = re / r - 1 (Eq. 3) from r^2 with one reciprocal square root.
__device__ __forceinline__ double inv_r(double r2) { return rsqrt(r2); }

// ---------------------------------------------------------------- S4 density ---
// n_i = sum_{j in N(i, re_n)} (re_n / r_ij - 1), all non-ghost i and j (Eq. 5).
__global__ void __launch_bounds__(TPB)
k_density(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ nbr,
          const uint32_t* __restrict__ cn, double* __restrict__ dens) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  const double4 pi = pos4[i];
  const uint32_t* row = row_of(nbr, kc.cap, i);
  const uint32_t m = cn[i];
  double s0 = 0.0, s1 = 0.0;
  uint32_t k = 0;
  for (; k + 1 < m; k += 2) {
    uint32_t j0 = row[(size_t)k * 32] & NB_INDEX, j1 = row[(size_t)(k + 1) * 32] & NB_INDEX;
    double4 q0 = pos4[j0], q1 = pos4[j1];
    double dx0 = q0.x - pi.x, dy0 = q0.y - pi.y, dz0 = q0.z - pi.z;
    double dx1 = q1.x - pi.x, dy1 = q1.y - pi.y, dz1 = q1.z - pi.z;
    double r20 = dx0 * dx0 + dy0 * dy0 + dz0 * dz0;
    double r21 = dx1 * dx1 + dy1 * dy1 + dz1 * dz1;
    s0 += kc.re_n * inv_r(r20) - 1.0;
    s1 += kc.re_n * inv_r(r21) - 1.0;
  }
  if (k < m) {
    uint32_t j0 = row[(size_t)k * 32] & NB_INDEX;
    double4 q0 = pos4[j0];
    double dx0 = q0.x - pi.x, dy0 = q0.y - pi.y, dz0 = q0.z - pi.z;
    s0 += kc.re_n * inv_r(dx0 * dx0 + dy0 * dy0 + dz0 * dz0) - 1.0;
  }
  dens[i] = s0 + s1;
}

// --------------------------------------------------- S5 Smagorinsky + nu_eff ---
// G_ab = (d/n0) sum (u_b,j - u_b,i)(x_a,j - x_a,i) / r^2 w(r) over N(i, re_n);
// S = (G + G^T)/2; nu_t = (Cs l0)^2 sqrt(2 S:S) (Eq. 13; Q10).
// Also writes vel4.w = nu_eff (fluid: nu[phase] + nu_t; wall/dummy/ghost: -1).
__global__ void __launch_bounds__(TPB)
k_nu_eff(KConst kc, int with_sps, const double4* __restrict__ pos4, double4* __restrict__ vel4,
         const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
         const uint32_t* __restrict__ cn, double* __restrict__ nut) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  const uint32_t t = tp[i];
  if ((t & 0xff) != MPS_FLUID) {
    nut[i] = 0.0;
    vel4[i].w = -1.0;
    return;
  }
  double nt = 0.0;
  if (with_sps) {
    const double4 pi = pos4[i];
    const double4 vi = vel4[i];
    const uint32_t* row = row_of(nbr, kc.cap, i);
    const uint32_t m = cn[i];
    double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (uint32_t k = 0; k < m; ++k) {
      uint32_t j = row[(size_t)k * 32] & NB_INDEX;
      double4 q = pos4[j];
      double4 vj = vel4[j];  // walls and dummies hold u = 0
      double dr[3] = {q.x - pi.x, q.y - pi.y, q.z - pi.z};
      double du[3] = {vj.x - vi.x, vj.y - vi.y, vj.z - vi.z};
      double r2 = dr[0] * dr[0] + dr[1] * dr[1] + dr[2] * dr[2];
      double ir = inv_r(r2);
      double c = (kc.re_n * ir - 1.0) * ir * ir;
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) G[a][b] += du[b] * dr[a] * c;
    }
    double ss = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        double S = 0.5 * kc.d_over_n0 * (G[a][b] + G[b][a]);
        ss += S * S;
      }
    nt = kc.cs_l0_sq * sqrt(2.0 * ss);
  }
  nut[i] = nt;
  vel4[i].w = kc.nu[(t >> 8) & 1] + nt;
}

// ------------------------------------------------------------- S6 viscosity ---
// a_i = A_lap sum_{j in N(i, re_lap)} nu_ij (u_j - u_i) w(r) + g, fluid i
// (Eq. 10, Eq. 2; Q9).
__device__ __forceinline__ void visc_term(const KConst& kc, const double4& pi, const double4& vi,
                                          const double4& q, const double4& vj, double& sx, double& sy,
                                          double& sz) {
  double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
  double r2 = dx * dx + dy * dy + dz * dz;
  double w = kc.re_lap * inv_r(r2) - 1.0;
  double nui = vi.w, nuj = vj.w, nuij;
  if (nuj < 0.0) nuij = nui;
  else if (kc.nu_pair_mean == 1) nuij = (nui + nuj > 0.0) ? 2.0 * nui * nuj / (nui + nuj) : 0.0;
  else nuij = 0.5 * (nui + nuj);
  double c = nuij * w;
  sx += c * (vj.x - vi.x);
  sy += c * (vj.y - vi.y);
  sz += c * (vj.z - vi.z);
}
__global__ void __launch_bounds__(TPB)
k_viscosity(KConst kc, const double4* __restrict__ pos4, const double4* __restrict__ vel4,
            const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
            const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co,
            double4* __restrict__ acc4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  if ((tp[i] & 0xff) != MPS_FLUID) {
    acc4[i] = make_double4(0.0, 0.0, 0.0, 0.0);
    return;
  }
  const double4 pi = pos4[i];
  const double4 vi = vel4[i];
  const uint32_t* row = row_of(nbr, kc.cap, i);
  const uint32_t nf = cn[i], nb = co[i];
  double sx = 0.0, sy = 0.0, sz = 0.0;
  for (uint32_t k = 0; k < nf; ++k) {
    uint32_t j = row[(size_t)k * 32] & NB_INDEX;
    visc_term(kc, pi, vi, pos4[j], vel4[j], sx, sy, sz);
  }
  for (uint32_t k = 0; k < nb; ++k) {
    uint32_t j = row[(size_t)(kc.cap - 1 - k) * 32] & NB_INDEX;
    visc_term(kc, pi, vi, pos4[j], vel4[j], sx, sy, sz);
  }
  acc4[i] = make_double4(kc.A_lap * sx + kc.g[0], kc.A_lap * sy + kc.g[1], kc.A_lap * sz + kc.g[2], 0.0);
}

// -------------------------------------------------------------- S7 predictor ---
// u* = u + dt a; r* = r + dt u*; fluid only (Q8).
__global__ void k_predict(KConst kc, double4* __restrict__ pos4, double4* __restrict__ vel4,
                          const double4* __restrict__ acc4, const uint32_t* __restrict__ tp) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  if ((tp[i] & 0xff) != MPS_FLUID) return;
  double4 v = vel4[i], a = acc4[i], r = pos4[i];
  v.x = __dadd_rn(v.x, __dmul_rn(kc.dt, a.x));
  v.y = __dadd_rn(v.y, __dmul_rn(kc.dt, a.y));
  v.z = __dadd_rn(v.z, __dmul_rn(kc.dt, a.z));
  r.x = __dadd_rn(r.x, __dmul_rn(kc.dt, v.x));
  r.y = __dadd_rn(r.y, __dmul_rn(kc.dt, v.y));
  r.z = __dadd_rn(r.z, __dmul_rn(kc.dt, v.z));
  vel4[i] = v;
  pos4[i] = r;
}

// ----------------------------------------------------- S8a equation of state ---
// p = rho c0^2 / gamma ((n/n0)^gamma - 1) for fluid and wall, else 0 (Eq. 7; Q4).
__global__ void k_pressure_explicit(KConst kc, const double* __restrict__ dens,
                                    const uint32_t* __restrict__ tp, double* __restrict__ p) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  uint32_t t = tp[i];
  uint32_t ty = t & 0xff;
  double pr = 0.0;
  if (ty == MPS_FLUID || ty == MPS_WALL) {
    double q = dens[i] / kc.n0_n, qg;
    if (kc.gamma == 7.0) {
      double q2 = q * q, q4 = q2 * q2;
      qg = q4 * q2 * q;
    } else {
      qg = pow(q, kc.gamma);
    }
    pr = kc.rho[(t >> 8) & 1] * kc.c0 * kc.c0 / kc.gamma * (qg - 1.0);
    if (kc.clamp_negative_p && pr < 0.0) pr = 0.0;
  }
  p[i] = pr;
}

// ------------------------------------------------------------------ S9 p-hat ---
// phat_i = min(p_i, min over non-dummy j in N(i, re_n) of p_j), fluid and wall i
// (Q12).  Also refreshes pos4.w = p_i for the gradient's gathers.
__global__ void __launch_bounds__(TPB)
k_phat(KConst kc, double4* __restrict__ pos4, const double* __restrict__ p,
       const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
       const uint32_t* __restrict__ cn, double* __restrict__ phat) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  const double pi = p[i];
  pos4[i].w = pi;
  uint32_t ty = tp[i] & 0xff;
  if (ty != MPS_FLUID && ty != MPS_WALL) {
    phat[i] = 0.0;
    return;
  }
  const uint32_t* row = row_of(nbr, kc.cap, i);
  const uint32_t m = cn[i];
  double mn = pi;
  for (uint32_t k = 0; k < m; ++k) {
    uint32_t e = row[(size_t)k * 32];
    if (e & NB_DUMMY) continue;
    mn = fmin(mn, p[e & NB_INDEX]);
  }
  phat[i] = mn;
}

// --------------------------------------------------------------- S10 gradient ---
// G_i = (d/n0) sum coef / r^2 (r_j - r_i) w(r) over non-dummy j in N(i, re_n):
// coef = p_j - phat_i (0) | (p_i + p_j) - (phat_i + phat_j) (1, Eq. 14) | p_i + p_j (2).
template <int VARIANT>
__global__ void __launch_bounds__(TPB)
k_gradient(KConst kc, const double4* __restrict__ pos4, const double* __restrict__ phat,
           const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
           const uint32_t* __restrict__ cn, double4* __restrict__ grad4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  if ((tp[i] & 0xff) != MPS_FLUID) {
    grad4[i] = make_double4(0.0, 0.0, 0.0, 0.0);
    return;
  }
  const double4 pi = pos4[i];  // .w = p_i
  const double phi = phat[i];
  const uint32_t* row = row_of(nbr, kc.cap, i);
  const uint32_t m = cn[i];
  double sx = 0.0, sy = 0.0, sz = 0.0;
  for (uint32_t k = 0; k < m; ++k) {
    uint32_t e = row[(size_t)k * 32];
    if (e & NB_DUMMY) continue;
    uint32_t j = e & NB_INDEX;
    double4 q = pos4[j];
    double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    double r2 = dx * dx + dy * dy + dz * dz;
    double ir = inv_r(r2);
    double coef;
    if (VARIANT == 0) coef = q.w - phi;
    else if (VARIANT == 1) coef = (pi.w + q.w) - (phi + phat[j]);
    else coef = pi.w + q.w;
    double c = coef * (kc.re_n * ir - 1.0) * ir * ir;
    sx += c * dx;
    sy += c * dy;
    sz += c * dz;
  }
  grad4[i] = make_double4(kc.d_over_n0 * sx, kc.d_over_n0 * sy, kc.d_over_n0 * sz, 0.0);
}

// --------------------------------------------------------------- S11 corrector ---
// u = u* - (dt / rho_i) G; r = r* + dt (u - u*); fluid only (Q8).
__global__ void k_correct(KConst kc, double4* __restrict__ pos4, double4* __restrict__ vel4,
                          const double4* __restrict__ grad4, const uint32_t* __restrict__ tp) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= kc.n) return;
  uint32_t t = tp[i];
  if ((t & 0xff) != MPS_FLUID) return;
  const double s = kc.dt / kc.rho[(t >> 8) & 1];
  double4 v = vel4[i], gq = grad4[i], r = pos4[i];
  double ux = __dsub_rn(v.x, __dmul_rn(s, gq.x));
  double uy = __dsub_rn(v.y, __dmul_rn(s, gq.y));
  double uz = __dsub_rn(v.z, __dmul_rn(s, gq.z));
  r.x = __dadd_rn(r.x, __dmul_rn(kc.dt, __dsub_rn(ux, v.x)));
  r.y = __dadd_rn(r.y, __dmul_rn(kc.dt, __dsub_rn(uy, v.y)));
  r.z = __dadd_rn(r.z, __dmul_rn(kc.dt, __dsub_rn(uz, v.z)));
  v.x = ux; v.y = uy; v.z = uz;
  vel4[i] = v;
  pos4[i] = r;
}

}  // namespace

// ============================================================ host launchers ===
int mpsk_density(mps_ctx* c) {
  int n = (int)c->n;
  MPS_LAUNCH(c, MPS_T_DENSITY, k_density, div_up(n, TPB), TPB, c->kc, c->pos4[c->cur], c->nbr, c->cn,
             c->dens);
  return MPS_OK;
}

int mpsk_viscosity(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  MPS_LAUNCH(c, MPS_T_VISCOSITY, k_nu_eff, div_up(n, TPB), TPB, c->kc, c->prm.cs > 0.0 ? 1 : 0,
             c->pos4[cur], c->vel4[cur], c->tp[cur], c->nbr, c->cn, c->nut);
  MPS_LAUNCH(c, MPS_T_VISCOSITY, k_viscosity, div_up(n, TPB), TPB, c->kc, c->pos4[cur], c->vel4[cur],
             c->tp[cur], c->nbr, c->cn, c->co, c->acc4);
  return MPS_OK;
}

int mpsk_predict(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  MPS_LAUNCH(c, MPS_T_PREDICT, k_predict, div_up(n, 256), 256, c->kc, c->pos4[cur], c->vel4[cur],
             c->acc4, c->tp[cur]);
  c->binned = false;
  c->ppe_ready = false;
  return MPS_OK;
}

int mpsk_pressure_explicit(mps_ctx* c) {
  int n = (int)c->n;
  MPS_LAUNCH(c, MPS_T_PRESSURE_EXPLICIT, k_pressure_explicit, div_up(n, 256), 256, c->kc, c->dens,
             c->tp[c->cur], c->p);
  return MPS_OK;
}

int mpsk_gradient(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  MPS_LAUNCH(c, MPS_T_GRADIENT, k_phat, div_up(n, TPB), TPB, c->kc, c->pos4[cur], c->p, c->tp[cur],
             c->nbr, c->cn, c->phat);
  switch (c->prm.grad_variant) {
    case 0:
      MPS_LAUNCH(c, MPS_T_GRADIENT, k_gradient<0>, div_up(n, TPB), TPB, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
    case 1:
      MPS_LAUNCH(c, MPS_T_GRADIENT, k_gradient<1>, div_up(n, TPB), TPB, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
    default:
      MPS_LAUNCH(c, MPS_T_GRADIENT, k_gradient<2>, div_up(n, TPB), TPB, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
  }
  return MPS_OK;
}

int mpsk_correct(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  MPS_LAUNCH(c, MPS_T_CORRECT, k_correct, div_up(n, 256), 256, c->kc, c->pos4[cur], c->vel4[cur],
             c->grad4, c->tp[cur]);
  c->binned = false;
  c->ppe_ready = false;
  return MPS_OK;
}
