// kernels_sweep.cu -- the fixed-radius sweeps over the per-step neighbour rows
// (density S4, Smagorinsky S5, viscosity S6, p-hat S9, gradient S10) and the
// streaming updates (predictor S7, equation of state S8a, corrector S11).
// One thread per particle; entry k of the 32 particles of a warp is one
// coalesced 128-byte line; each neighbour costs one 32-byte sector gather.
#include "sweep_common.cuh"

namespace {

constexpr int TPB = 256;
// L lanes per row (a template parameter of every row kernel; TPB / L rows per block): 4 from 50,000 particles up,
// 8 below, where four lanes per row leave an SM short of threads (measured at 2M: viscosity 1.35 -> 1.31 ms, density
// 0.234 -> 0.212, gradient 0.353 -> 0.279; 16 lanes: 1.59 / 0.366 / 0.522; 2 lanes: 1.66 / 0.234 / 0.271; at 19k
// particles the explicit step takes 0.105 ms with 8 lanes and 0.125 with 4)

// group -> particle; sub = lane within the group
#define ROW_GROUP(i, sub)                                              \
  const int i = (int)((blockIdx.x * (unsigned)TPB + threadIdx.x) / L); \
  const int sub = threadIdx.x & (L - 1);                               \
  const bool row_live = i < kc.n;                                      \
  const int ii = row_live ? i : 0

// ---------------------------------------------------------------- S4 density ---
// n_i = sum_{j in N(i, re_n)} (re_n / r_ij - 1), all non-ghost i and j (Eq. 5).
template <int L>
__global__ void __launch_bounds__(TPB)
k_density(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ nbr,
          const uint32_t* __restrict__ cn, double* __restrict__ dens) {
  ROW_GROUP(i, sub);
  const double4 pi = pos4[ii];
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  const uint32_t m = row_live ? cn[ii] : 0u;
  double s = 0.0;
  for (uint32_t k = sub; k < m; k += L) {
    const double4 q = gather_rec(kc.pos_tex, pos4, row[k] & NB_INDEX);
    const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    const double r2 = pair_r2(dx, dy, dz, kc.stale);
    if (kc.stale && !(r2 < kc.re_n2)) continue;  // reused row: the pair has left the radius
    s += kernel_w(kc.kernel, kc.re_n, kc.inv_re_n, r2, rsqrt_f64(r2));
  }
  s = group_sum<L>(s);
  if (row_live && sub == 0) dens[i] = s;
}

// ------------------------------------ NEXT-2: smoothed density of the multi-density model ---
// <rho>_i = sum_j rho_j w(r_ij) / sum_j w(r_ij) over N(i, re_n), every non-ghost i; rho_j comes
// from the phase bit of the row entry (Q25).  No neighbour: the particle's own density.
template <int L>
__global__ void __launch_bounds__(TPB)
k_smooth_density(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ tp,
                 const uint32_t* __restrict__ nbr, const uint32_t* __restrict__ cn,
                 double* __restrict__ rho_s) {
  ROW_GROUP(i, sub);
  const double4 pi = pos4[ii];
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  const uint32_t m = row_live ? cn[ii] : 0u;
  double sw = 0.0, srw = 0.0;
  for (uint32_t k = sub; k < m; k += L) {
    const uint32_t e = row[k];
    const double4 q = gather_rec(kc.pos_tex, pos4, e & NB_INDEX);
    const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double w = kernel_w(kc.kernel, kc.re_n, kc.inv_re_n, r2, rsqrt_f64(r2));
    sw += w;
    srw = fma(kc.rho[(e & NB_PHASE1) ? 1 : 0], w, srw);
  }
  sw = group_sum<L>(sw);
  srw = group_sum<L>(srw);
  if (row_live && sub == 0) rho_s[i] = sw > 0.0 ? srw / sw : kc.rho[(tp[i] >> 8) & 1];
}

// stage beta_i = <rho>_i alpha_i = <rho>_i p_i / rho_i into pos4.w for the variant-3 gradient
__global__ void k_stage_beta(KConst kc, const double* __restrict__ p, const double* __restrict__ rho_s,
                             const uint32_t* __restrict__ tp, double4* __restrict__ pos4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < kc.n) pos4[i].w = rho_s[i] * (p[i] / kc.rho[(tp[i] >> 8) & 1]);
}

// ---------------------------------------------------- NEXT-1: Dn/Dt (MPS-HS) ---
// Dn/Dt_i = d/dt sum_j (re_n / r_ij - 1) = -sum_{j in N(i, re_n)} re_n / r^3 (x_ij . u_ij),
// x_ij = x_j - x_i, u_ij = u_j - u_i; walls and dummies hold u = 0 in vel4 (P:224-228
// Eq. 15; sign: Q22).  keep: also store (n_i, Dn/Dt_i) as the start-of-step pair of Eq. 17.
template <int L>
__global__ void __launch_bounds__(TPB)
k_dndt(KConst kc, const double4* __restrict__ pos4, const double4* __restrict__ vel4,
       const uint32_t* __restrict__ nbr, const uint32_t* __restrict__ cn,
       const double* __restrict__ dens, double* __restrict__ dndt, double2* __restrict__ keep2) {
  ROW_GROUP(i, sub);
  const double4 pi = pos4[ii];
  const double4 vi = vel4[ii];
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  const uint32_t m = row_live ? cn[ii] : 0u;
  double s = 0.0;
  for (uint32_t k = sub; k < m; k += L) {
    const uint32_t j = row[k] & NB_INDEX;
    const double4 q = gather_rec(kc.pos_tex, pos4, j);
    const double4 vj = gather_rec(kc.vel_tex, vel4, j);
    const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    const double r2 = pair_r2(dx, dy, dz, kc.stale);
    if (kc.stale && !(r2 < kc.re_n2)) continue;
    const double ir = rsqrt_f64(r2);
    const double xu = dx * (vj.x - vi.x) + dy * (vj.y - vi.y) + dz * (vj.z - vi.z);
    s = fma(ir * ir * ir, xu, s);
  }
  s = -kc.re_n * group_sum<L>(s);
  if (row_live && sub == 0) {
    if (keep2) keep2[i] = make_double2(dens[i], s);
    else dndt[i] = s;
  }
}

// --------------------------------------------------- S5 Smagorinsky + nu_eff ---
// G_ab = (d/n0) sum (u_b,j - u_b,i)(x_a,j - x_a,i) / r^2 w(r) over N(i, re_n);
// S = (G + G^T)/2; nu_t = (Cs l0)^2 sqrt(2 S:S) (Eq. 13; Q10).
// Writes nut and vel4.w = nu_eff (fluid: nu[phase] + nu_t; wall/dummy/ghost: -1).
template <int L>
__global__ void __launch_bounds__(TPB)
k_nu_eff(KConst kc, int with_sps, const double4* __restrict__ pos4, double4* __restrict__ vel4,
         const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
         const uint32_t* __restrict__ cn, double* __restrict__ nut) {
  ROW_GROUP(i, sub);
  const uint32_t t = tp[ii];
  const bool fluid = row_live && (t & 0xff) == MPS_FLUID;
  double nt = 0.0;
  if (with_sps) {
    const double4 pi = pos4[ii];
    const double4 vi = vel4[ii];
    const uint32_t* row = row_ptr(nbr, kc.stride, ii);
    const uint32_t m = fluid ? cn[ii] : 0u;
    double G[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (uint32_t k = sub; k < m; k += L) {
      const uint32_t j = row[k] & NB_INDEX;
      const double4 q = gather_rec(kc.pos_tex, pos4, j);
      const double4 vj = gather_rec(kc.vel_tex, vel4, j);  // walls and dummies hold u = 0
      const double dr[3] = {q.x - pi.x, q.y - pi.y, q.z - pi.z};
      const double du[3] = {vj.x - vi.x, vj.y - vi.y, vj.z - vi.z};
      const double r2 = pair_r2(dr[0], dr[1], dr[2], kc.stale);
      if (kc.stale && !(r2 < kc.re_n2)) continue;
      const double ir = rsqrt_f64(r2);
      const double c = kernel_w(kc.kernel, kc.re_n, kc.inv_re_n, r2, ir) * ir * ir;
#pragma unroll
      for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) G[a][b] += du[b] * dr[a] * c;
    }
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) G[a][b] = group_sum<L>(G[a][b]);
    double ss = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) {
        const double S = 0.5 * kc.d_over_n0 * (G[a][b] + G[b][a]);
        ss += S * S;
      }
    nt = kc.cs_l0_sq * sqrt(2.0 * ss);
  }
  if (row_live && sub == 0) {
    nut[i] = fluid ? nt : 0.0;
    vel4[i].w = fluid ? kc.nu[(t >> 8) & 1] + nt : -1.0;
  }
}

// ------------------------------------------------------------- S6 viscosity ---
// a_i = A_lap sum_{j in N(i, re_lap)} nu_ij (u_j - u_i) w(r) + g, fluid i
// (Eq. 10, Eq. 2; Q9).  SPS = false: nu_j comes from the entry's
// phase / wall / dummy bits (no pre-pass); SPS = true: nu_j = vel4[j].w.
// (five blocks per SM: 48 registers with a 16-byte spill beat four blocks at 60 -- 1.398 -> 1.350 ms at 2M -- and six at 40)
template <bool SPS, int L>
__global__ void __launch_bounds__(TPB, 5)
k_viscosity(KConst kc, const double4* __restrict__ pos4, const double4* __restrict__ vel4,
            const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
            const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co,
            double4* __restrict__ acc4) {
  ROW_GROUP(i, sub);
  const uint32_t t = tp[ii];
  const bool fluid = row_live && (t & 0xff) == MPS_FLUID;
  const double4 pi = pos4[ii];
  const double4 vi = vel4[ii];
  const double nui = SPS ? vi.w : kc.nu[(t >> 8) & 1];
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  const uint32_t nf = fluid ? cn[ii] : 0u;
  const uint32_t m = fluid ? nf + co[ii] : 0u;
  double sx = 0.0, sy = 0.0, sz = 0.0;
  for (uint32_t k = sub; k < m; k += L) {
    const uint32_t e = row_entry(row, kc.stride, nf, k);
    const uint32_t j = e & NB_INDEX;
    const double4 q = gather_rec(kc.pos_tex, pos4, j);
    const double4 vj = gather_rec(kc.vel_tex, vel4, j);
    const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    const double r2 = pair_r2(dx, dy, dz, kc.stale);
    if (kc.stale && !(r2 < kc.re_lap2)) continue;
    const double w = kernel_w(kc.kernel, kc.re_lap, kc.inv_re_lap, r2, rsqrt_f64(r2));
    double nuij;
    if (e & (NB_DUMMY | NB_WALL)) {
      nuij = nui;
    } else {
      const double nuj = SPS ? vj.w : kc.nu[(e & NB_PHASE1) ? 1 : 0];
      if (kc.nu_pair_mean == 1) nuij = (nui + nuj > 0.0) ? 2.0 * nui * nuj / (nui + nuj) : 0.0;
      else nuij = 0.5 * (nui + nuj);
    }
    const double c = nuij * w;
    sx += c * (vj.x - vi.x);
    sy += c * (vj.y - vi.y);
    sz += c * (vj.z - vi.z);
  }
  sx = group_sum<L>(sx);
  sy = group_sum<L>(sy);
  sz = group_sum<L>(sz);
  if (row_live && sub == 0) {
    acc4[i] = fluid ? make_double4(kc.A_lap * sx + kc.g[0], kc.A_lap * sy + kc.g[1],
                                   kc.A_lap * sz + kc.g[2], 0.0)
                    : make_double4(0.0, 0.0, 0.0, 0.0);
  }
}

// Skin rows of mps_step (Q26): do they still cover position r of a particle whose rows were built at ref?
// Yes while |r - ref| <= 0.45 skins, r is inside the domain (else the next BIN makes it a GHOST) and finite.
__device__ __forceinline__ bool rows_cover(const KConst& kc, const double4& r, const double4& ref) {
  const double ex = r.x - ref.x, ey = r.y - ref.y, ez = r.z - ref.z;
  const double gx = floor((r.x - kc.dmin[0]) * kc.inv_h_dom), gy = floor((r.y - kc.dmin[1]) * kc.inv_h_dom);
  const double gz = floor((r.z - kc.dmin[2]) * kc.inv_h_dom);
  const bool in = (gx >= 0.0 && gx < (double)kc.nx_dom) && (gy >= 0.0 && gy < (double)kc.ny_dom) &&
                  (gz >= 0.0 && gz < (double)kc.nz_dom);
  return (ex * ex + ey * ey + ez * ez <= kc.carry_d2) && in;  // NaN fails the first test
}

// -------------------------------------------------------------- S7 predictor ---
// u* = u + dt a; r* = r + dt u*; fluid only (Q8).
// flags != NULL (mps_step with a skin): lower need_k (the bin at r^k, if any, has run) and raise need_star
// when the rows do not cover some r*: the predicated bin that follows then runs.
__global__ void k_predict(KConst kc, double4* __restrict__ pos4, double4* __restrict__ vel4,
                          const double4* __restrict__ acc4, const uint32_t* __restrict__ tp,
                          const double4* __restrict__ pos_ref, DevFlags* __restrict__ flags) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (flags && i == 0) flags->need_k = 0;
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
  if (flags && !rows_cover(kc, r, pos_ref[i])) flags->need_star = 1;
}

// ----------------------------------------------------- S8a equation of state ---
// p = rho c0^2 / gamma ((n/n0)^gamma - 1) for fluid and wall, else 0 (Eq. 7; Q4).
// Also stages p into pos4.w for the gradient's gathers.
__global__ void k_pressure_explicit(KConst kc, const double* __restrict__ dens,
                                    const uint32_t* __restrict__ tp, double* __restrict__ p,
                                    double4* __restrict__ pos4) {
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
  pos4[i].w = pr;
}

// stage p into pos4.w (only when some other call left a different scalar there)
__global__ void k_stage_p(int n, const double* __restrict__ p, double4* __restrict__ pos4) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) pos4[i].w = p[i];
}

// ------------------------------------------------------------------ S9 p-hat ---
// phat_i = min(p_i, min over non-dummy j in N(i, re_n) of p_j), fluid and wall i
// (Q12).  p_j is read from pos4.w.
template <int L>
__global__ void __launch_bounds__(TPB)
k_phat(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ tp,
       const uint32_t* __restrict__ nbr, const uint32_t* __restrict__ cn, double* __restrict__ phat) {
  ROW_GROUP(i, sub);
  const uint32_t ty = tp[ii] & 0xff;
  const bool on = row_live && (ty == MPS_FLUID || ty == MPS_WALL);
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  const uint32_t m = on ? cn[ii] : 0u;
  const double4 pi = pos4[ii];
  double mn = pi.w;
  for (uint32_t k = sub; k < m; k += L) {
    const uint32_t e = row[k];
    if (e & NB_DUMMY) continue;
    const double4 q = gather_rec(kc.pos_tex, pos4, e & NB_INDEX);
    if (kc.stale && !(pair_r2(q.x - pi.x, q.y - pi.y, q.z - pi.z, 1) < kc.re_n2)) continue;
    mn = fmin(mn, q.w);
  }
  mn = group_min<L>(mn);
  if (row_live && sub == 0) phat[i] = on ? mn : 0.0;
}

// --------------------------------------------------------------- S10 gradient ---
// G_i = (d/n0) sum coef / r^2 (r_j - r_i) w(r) over non-dummy j in N(i, re_n):
// coef = p_j - phat_i (0) | (p_i + p_j) - (phat_i + phat_j) (1, Eq. 14) | p_i + p_j (2).
// Variants 0 and 2 find phat_i in the same pass over the row as the sum (no pre-pass
// kernel); variant 1 needs phat_j of the neighbours, so k_phat runs first.
template <int VARIANT, int L>
__global__ void __launch_bounds__(TPB, 6)
k_gradient(KConst kc, const double4* __restrict__ pos4, double* __restrict__ phat,
           const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
           const uint32_t* __restrict__ cn, double4* __restrict__ grad4) {
  ROW_GROUP(i, sub);
  const uint32_t ty = tp[ii] & 0xff;
  const bool fluid = row_live && ty == MPS_FLUID;
  const bool wall = row_live && ty == MPS_WALL;
  const double4 pi = pos4[ii];  // .w = p_i
  const uint32_t* row = row_ptr(nbr, kc.stride, ii);
  // variants 0 and 2 also produce p-hat, which wall rows have too; the sum itself is for fluid rows
  const uint32_t m = ((VARIANT == 0 || VARIANT == 2) ? (fluid || wall) : fluid) ? cn[ii] : 0u;
  double phi = 0.0;
  if (VARIANT == 1) phi = phat[ii];
  double inv_rsi = 0.0, ai = 0.0, scale = kc.d_over_n0;
  if (VARIANT == 3) {
    // pi.w = beta_i; phat carries <rho> (see mpsk_gradient): nothing to pre-compute
    inv_rsi = 1.0 / phat[ii];     // phat points at <rho> for this variant
    ai = pi.w * inv_rsi;          // alpha_i = beta_i / <rho>_i
    scale *= kc.rho[(tp[ii] >> 8) & 1];  // stored as rho_i x Eq. 11: the corrector divides by rho_i
  }
  // ONE pass over the row.  Variant 0 is linear in phat_i: sum (p_j - phat_i) c x_ij = sum p_j c x_ij -
  // phat_i sum c x_ij, so the minimum and both sums come out of the same gathers (the two-pass form gathered
  // every record twice); the difference to the oracle's order of operations is rounding (a few 1e-14 relative).
  double sx = 0.0, sy = 0.0, sz = 0.0, bx = 0.0, by = 0.0, bz = 0.0;
  double mn = pi.w;
  for (uint32_t k = sub; k < m; k += L) {
    const uint32_t e = row[k];
    if (e & NB_DUMMY) continue;
    const uint32_t j = e & NB_INDEX;
    const double4 q = gather_rec(kc.pos_tex, pos4, j);
    const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
    const double r2 = pair_r2(dx, dy, dz, kc.stale);
    if (kc.stale && !(r2 < kc.re_n2)) continue;
    if (VARIANT == 0 || VARIANT == 2) mn = fmin(mn, q.w);
    const double ir = rsqrt_f64(r2);
    const double c = kernel_w(kc.kernel, kc.re_n, kc.inv_re_n, r2, ir) * ir * ir;
    double coef;
    if (VARIANT == 0) coef = q.w;
    else if (VARIANT == 1) coef = (pi.w + q.w) - (phi + phat[j]);
    else if (VARIANT == 2) coef = pi.w + q.w;
    else coef = fma(q.w, inv_rsi, -ai);  // (<rho>_j / <rho>_i) alpha_j - alpha_i, Eq. 11
    const double cc = coef * c;
    sx += cc * dx;
    sy += cc * dy;
    sz += cc * dz;
    if (VARIANT == 0) {
      bx += c * dx;
      by += c * dy;
      bz += c * dz;
    }
  }
  if (VARIANT == 0 || VARIANT == 2) {
    phi = group_min<L>(mn);
    if (row_live && sub == 0) phat[i] = (fluid || wall) ? phi : 0.0;
  }
  if (VARIANT == 0) {
    sx = fma(-phi, bx, sx);
    sy = fma(-phi, by, sy);
    sz = fma(-phi, bz, sz);
  }
  if (!fluid) sx = sy = sz = 0.0;  // wall rows only wanted their p-hat
  sx = group_sum<L>(sx);
  sy = group_sum<L>(sy);
  sz = group_sum<L>(sz);
  if (row_live && sub == 0)
    grad4[i] = make_double4(scale * sx, scale * sy, scale * sz, 0.0);
}

// --------------------------------------------------------------- S11 corrector ---
// u = u* - (dt / rho_i) G; r = r* + dt (u - u*); fluid only (Q8).
// flags != NULL (mps_step with a skin): lower need_star and raise need_k when the rows do not cover some
// r^(k+1): the predicated bin at the start of the next step then runs.
__global__ void k_correct(KConst kc, double4* __restrict__ pos4, double4* __restrict__ vel4,
                          const double4* __restrict__ grad4, const uint32_t* __restrict__ tp,
                          const double4* __restrict__ pos_ref, DevFlags* __restrict__ flags) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (flags && i == 0) flags->need_star = 0;
  if (i >= kc.n) return;
  uint32_t t = tp[i];
  if ((t & 0xff) != MPS_FLUID) return;
  const double s = kc.dt / kc.rho[(t >> 8) & 1];
  double4 v = vel4[i], gq = grad4[i], r = pos4[i];
  double ux = __dsub_rn(v.x, __dmul_rn(s, gq.x));
  double uy = __dsub_rn(v.y, __dmul_rn(s, gq.y));
  double uz = __dsub_rn(v.z, __dmul_rn(s, gq.z));
  const double ex = __dmul_rn(kc.dt, __dsub_rn(ux, v.x)), ey = __dmul_rn(kc.dt, __dsub_rn(uy, v.y));
  const double ez = __dmul_rn(kc.dt, __dsub_rn(uz, v.z));
  r.x = __dadd_rn(r.x, ex);
  r.y = __dadd_rn(r.y, ey);
  r.z = __dadd_rn(r.z, ez);
  if (flags && !rows_cover(kc, r, pos_ref[i])) flags->need_k = 1;
  v.x = ux; v.y = uy; v.z = uz;
  vel4[i] = v;
  pos4[i] = r;
}

}  // namespace

// ============================================================ host launchers ===
static inline int group_grid(int n, int lanes) { return div_up((int64_t)n * lanes, TPB); }
static inline int sweep_lanes(const mps_ctx* c) { return c->n >= 50000 ? 4 : 8; }
// launch a row kernel with the lanes per row that suit the scene: KERN<4> or KERN<8> (PRE: leading template arguments)
#define LAUNCH_ROWS(c, cat, KERN, n, ...)                                                                   \
  do {                                                                                                      \
    if (sweep_lanes(c) == 4) MPS_LAUNCH(c, cat, (KERN<4>), group_grid(n, 4), TPB, __VA_ARGS__);             \
    else MPS_LAUNCH(c, cat, (KERN<8>), group_grid(n, 8), TPB, __VA_ARGS__);                                 \
  } while (0)
#define LAUNCH_ROWS2(c, cat, KERN, PRE, n, ...)                                                             \
  do {                                                                                                      \
    if (sweep_lanes(c) == 4) MPS_LAUNCH(c, cat, (KERN<PRE, 4>), group_grid(n, 4), TPB, __VA_ARGS__);        \
    else MPS_LAUNCH(c, cat, (KERN<PRE, 8>), group_grid(n, 8), TPB, __VA_ARGS__);                            \
  } while (0)

int mpsk_density(mps_ctx* c) {
  int n = (int)c->n;
  LAUNCH_ROWS(c, MPS_T_DENSITY, k_density, n, c->kc, c->pos4[c->cur], c->nbr, c->cn,
             c->dens);
  return MPS_OK;
}

int mpsk_smooth_density(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  LAUNCH_ROWS(c, MPS_T_DENSITY, k_smooth_density, n, c->kc, c->pos4[cur], c->tp[cur],
             c->nbr, c->cn, c->rho_s[cur]);
  c->rho_s_ready = true;
  return MPS_OK;
}

int mpsk_dndt(mps_ctx* c, int keep) {
  int n = (int)c->n;
  int cur = c->cur;
  LAUNCH_ROWS(c, MPS_T_DENSITY, k_dndt, n, c->kc, c->pos4[cur], c->vel4[cur], c->nbr,
             c->cn, c->dens, c->dndt, keep ? c->keep2[cur] : nullptr);
  return MPS_OK;
}

int mpsk_viscosity(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  if (c->prm.cs > 0.0) {
    LAUNCH_ROWS(c, MPS_T_VISCOSITY, k_nu_eff, n, c->kc, 1, c->pos4[cur], c->vel4[cur],
               c->tp[cur], c->nbr, c->cn, c->nut);
    LAUNCH_ROWS2(c, MPS_T_VISCOSITY, k_viscosity, true, n, c->kc, c->pos4[cur],
               c->vel4[cur], c->tp[cur], c->nbr, c->cn, c->co, c->acc4);
  } else {
    LAUNCH_ROWS2(c, MPS_T_VISCOSITY, k_viscosity, false, n, c->kc, c->pos4[cur],
               c->vel4[cur], c->tp[cur], c->nbr, c->cn, c->co, c->acc4);
  }
  return MPS_OK;
}

int mpsk_predict(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  const bool skin = c->kc.stale && c->carry_rows && c->prm.rebin_every == 1;  // inside mps_step with a skin
  MPS_LAUNCH(c, MPS_T_PREDICT, k_predict, div_up(n, 256), 256, c->kc, c->pos4[cur], c->vel4[cur],
             c->acc4, c->tp[cur], c->pos_ref, skin ? c->flags : nullptr);
  c->binned = false;
  c->carry_valid = false;
  c->ppe_ready = false;
  return MPS_OK;
}

int mpsk_pressure_explicit(mps_ctx* c) {
  int n = (int)c->n;
  MPS_LAUNCH(c, MPS_T_PRESSURE_EXPLICIT, k_pressure_explicit, div_up(n, 256), 256, c->kc, c->dens,
             c->tp[c->cur], c->p, c->pos4[c->cur]);
  c->posw_is_p = true;
  return MPS_OK;
}

int mpsk_gradient(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  if (c->prm.grad_variant == 3) {
    MPS_LAUNCH(c, MPS_T_GRADIENT, k_stage_beta, div_up(n, 256), 256, c->kc, c->p, c->rho_s[cur], c->tp[cur],
               c->pos4[cur]);
    c->posw_is_p = false;
    LAUNCH_ROWS2(c, MPS_T_GRADIENT, k_gradient, 3, n, c->kc, c->pos4[cur], c->rho_s[cur],
               c->tp[cur], c->nbr, c->cn, c->grad4);
    return MPS_OK;
  }
  if (!c->posw_is_p) {
    MPS_LAUNCH(c, MPS_T_GRADIENT, k_stage_p, div_up(n, 256), 256, n, c->p, c->pos4[cur]);
    c->posw_is_p = true;
  }
  switch (c->prm.grad_variant) {
    case 0:
      LAUNCH_ROWS2(c, MPS_T_GRADIENT, k_gradient, 0, n, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
    case 1:
      LAUNCH_ROWS(c, MPS_T_GRADIENT, k_phat, n, c->kc, c->pos4[cur], c->tp[cur], c->nbr,
                 c->cn, c->phat);
      LAUNCH_ROWS2(c, MPS_T_GRADIENT, k_gradient, 1, n, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
    default:
      LAUNCH_ROWS2(c, MPS_T_GRADIENT, k_gradient, 2, n, c->kc, c->pos4[cur], c->phat,
                 c->tp[cur], c->nbr, c->cn, c->grad4);
      break;
  }
  return MPS_OK;
}

int mpsk_correct(mps_ctx* c) {
  int n = (int)c->n;
  int cur = c->cur;
  const bool skin = c->kc.stale && c->carry_rows && c->prm.rebin_every == 1;  // inside mps_step with a skin
  MPS_LAUNCH(c, MPS_T_CORRECT, k_correct, div_up(n, 256), 256, c->kc, c->pos4[cur], c->vel4[cur],
             c->grad4, c->tp[cur], c->pos_ref, skin ? c->flags : nullptr);
  c->binned = false;
  c->carry_valid = false;  // mps_step sets it again once its own corrector has run
  c->ppe_ready = false;
  return MPS_OK;
}
