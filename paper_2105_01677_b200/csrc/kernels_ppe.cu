// kernels_ppe.cu -- the semi-implicit pressure route (S8b of DESIGN.md):
// free-surface flags (Eq. 6), right-hand side (Eq. 8; Q5), the
// operator with the structure of Listing 2, and the
// conjugate-gradient solve (Eq. 9; Q15).
//
// The whole solve is ONE persistent cooperative kernel (k_ppe_cg): flags and
// right-hand side, ordered compaction of the unknown rows, (ppe_operator 1) assembly of
// the coefficients, then the CG loop in its single-reduction (Chronopoulos-Gear) form
// with two grid barriers per iteration:
//   phase A  w = A r fused with the dot products r.r and r.w (8 lanes per row,
//            shuffles inside the row group, one partial per block)
//   barrier  every block adds the partials in index order -> identical alpha, beta
//   phase B  p = r + beta p; s = w + beta s; x += alpha p; r -= alpha s
//   barrier  r is visible to every block
// All scalars stay on the device and the convergence test is taken by every block
// from the same numbers, so there is no host poll.  In exact arithmetic the
// iterates are those of textbook CG.
//
// Two forms of the operator (mps_params.ppe_operator), same numbers up to rounding:
//   0  matrix-free: r lives in pos4.w (a neighbour gather is one 32-byte record) and
//      c_ij = A_lap w(r_ij) / rho_ij is recomputed at every application;
//   1  assembled: positions are fixed during a solve, so the c_ij of the rows bc = 0 are
//      computed once into a compact ELL matrix in the numbering of the compacted rows
//      (neighbours on the free surface fold into a per-row diagonal term, dummies drop out).
//      One stored pair is ONE 64-bit word: the column in the high 24 bits and c_ij as a 40-bit
//      fixed-point fraction of the row's largest coefficient in the low 40 (absolute error
//      <= 2^-41 of that coefficient: 1e-12 of an operator row, far inside the 1e-10 bar).  An
//      application streams 8 bytes per pair, coalesced, and gathers 8 bytes from a dense
//      vector in which neighbouring rows share cache lines.
#include <algorithm>
#include <stdlib.h>

#include "sweep_common.cuh"

namespace {

constexpr int PPE_ILP = 4;   // independent neighbour gathers in flight per lane
// Streamed entries of the assembled operator in flight per lane: the loop is bound by HBM latency x
// bandwidth, so one 1024-thread block per SM keeps 1024 x 8 x 12 B = 96 KB of matrix in flight
// (measured at 1.44M rows: 315 ps per row per iteration with 4, 265 with 8; two blocks per SM at 32
// registers spill and are slower, 303-330)
constexpr int ASM_ILP = 8;
#ifndef MPS_ASM_L
#define MPS_ASM_L 8
#endif
// lanes per row in the CG loop's operator application (assembled form); measured at 1.44M rows: 4 lanes 229 ps
// per row per iteration, 8 lanes 216, 16 lanes 243 (260k rows: 259 / 221 / 239)
constexpr int ASM_L = MPS_ASM_L;
#ifndef MPS_ASM_RUN_LOG2
#define MPS_ASM_RUN_LOG2 3
#endif
#ifndef MPS_ASM_MINRUNS
#define MPS_ASM_MINRUNS 8
#endif
constexpr int ASM_RUN_LOG2 = MPS_ASM_RUN_LOG2;  // log2 of the consecutive super-chunks a warp group works through before it jumps
constexpr double PACK_QMAX = 1099511627775.0;  // 2^40 - 1: a stored coefficient is q / QMAX of the row's largest
constexpr int CG_TPB = 1024;
constexpr int L = 8;         // lanes per row
constexpr int GPW = 32 / L;  // row groups per warp
#ifndef MPS_SCW
#define MPS_SCW 32
#endif
constexpr int SCW = MPS_SCW;  // warps per super-chunk of consecutive rows (measured 8 vs 32: 219 vs 215 ps at 260k rows, 207 vs 205 at 5.8M)
static_assert(CG_TPB % (32 * SCW) == 0, "phase A deals rows in super-chunks of SCW warps");

struct PpeArgs {
  double4* pos4;  // matrix-free: .w is the CG residual r during the solve; pressure at exit
  cudaTextureObject_t tex;  // pos4 as 16-byte texels (0: not used)
  const uint32_t* tp;
  const double* dens;
  const double* dndt;      // (Dn/Dt)* (ppe_source >= 1)
  const double2* keep2;    // (n^k, (Dn/Dt)^k) (ppe_source == 2)
  int8_t* bc;
  double* b;
  double* x;               // per slot: the solution (matrix-free: the CG iterate itself)
  double* pv;              // p, s, w: per slot (matrix-free) or compact (assembled)
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
  // assembled operator
  uint32_t* rowmap;
  double* mval;
  uint32_t* mcol;
  uint32_t* mcnt;
  double* mdex;
  double* mscale;  // row's largest coefficient / (2^40 - 1)
  double* rc;
  double* xc;
  double tol2;
  long long timeout_cycles;
  int maxit;
  int warm;
  int compact;  // matrix-free on skin rows: walk the exact lists built once per solve (compact_row)
};

__device__ __forceinline__ void prefetch_l2(const void* p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

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
  // the next call's writes to sh come before its first barrier (lane 0 of each warp) and every
  // read of sh above is done by warp 0 before the second barrier; res is rewritten only
  // between the next call's two barriers
}

// ---- grid barrier (all blocks are co-resident: cooperative launch) ----------------
// One monotonically increasing arrival counter: thread 0 of every block adds 1 with
// release semantics and spins (acquire) until the count reaches nb x generation, so
// a barrier costs one L2 round trip for the arrival plus the polls.  The fence after
// the spin makes every later plain load of the block see the other blocks' writes.
// A spin longer than timeout_cycles (0: no limit) raises bar->timeout and lets the
// kernel drain instead of hanging.
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned int* p, unsigned int v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ bool grid_barrier(GridBar* bar, unsigned int& gen, long long timeout_cycles) {
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
        if (ld_acquire_u32(&bar->timeout)) { dead = 1; break; }  // some block gave up: follow it
        if (timeout_cycles > 0) {
          if (t0 == 0) t0 = clock64();
          else if (clock64() - t0 > timeout_cycles) {
            bar->timeout = 1u;
            dead = 1;
            break;
          }
        }
      }
    }
    __threadfence();
  }
  __syncthreads();
  return dead == 0;
}

// ---- pair coefficient before the row's common factor ---------------------------------
// Eq. 10 form (Listing 2): w(r) (then times A_lap); MPS-HL (Eq. 16; Q23): 1 / r^3 (then
// times 2 re / n0); both times 1 / rho_ij (Q6).
template <bool TWO_PHASE>
__device__ __forceinline__ double pair_coef(const KConst& kc, bool hl, double r2, uint32_t e,
                                            double inv_rij0, double inv_rij1) {
  const double ir = rsqrt_f64(r2);
  double w = hl ? ir * ir * ir : kernel_w(kc.kernel, kc.re_lap, kc.inv_re_lap, r2, ir);
  if (TWO_PHASE) w *= (e & NB_PHASE1) ? inv_rij1 : inv_rij0;
  return w;
}

// ---- one row of y = A r, matrix-free ---------------------------------------------------
// (A r)_i = sum_{j in N(i, re_lap), j not dummy} c_ij (r_i - r_j) + compress/dt^2 r_i,
// c_ij = A_lap w(r_ij) / rho_ij (Listing 2; Q5, Q6).  r_j is read from
// pos4.w, which is 0 on free-surface slots (Dirichlet p = 0).  The L lanes of the
// group each take every L-th entry; the result is valid in every lane.
// row / nf / m: the entries to walk (a neighbour row with its front and back parts, or -- nf = m -- a plain list);
// stale: re-test every pair against re_lap (skin rows, reused lists).
template <bool TWO_PHASE, bool TEX>
__device__ __forceinline__ double ppe_row_core(const KConst& kc, const double4* pos4, cudaTextureObject_t tex,
                                               const uint32_t* tp, const uint32_t* row, uint32_t nf, uint32_t m,
                                               int stale, int i, int sub, double& ri) {
  // every lane of the warp must come through here (full-mask shuffles below): a
  // group without a row passes m = 0 and any valid i
  const double4 pi = pos4[i];
  ri = pi.w;
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
      const double r2 = pair_r2(dx, dy, dz, stale);
      double w = pair_coef<TWO_PHASE>(kc, hl, r2, e[u], inv_rij0, inv_rij1);
      if ((e[u] & NB_DUMMY) || (stale && !(r2 < kc.re_lap2))) w = 0.0;  // dummy, empty slot, or left the radius
      s = fma(w, pi.w - q[u].w, s);
    }
  }
  s = group_sum<L>(s);
  if (!TWO_PHASE) s *= 1.0 / kc.rho[0];
  return fma(hl ? kc.hl_c : kc.A_lap, s, kc.compress_dt2 * pi.w);
}
template <bool TWO_PHASE, bool TEX>
__device__ __forceinline__ double ppe_row(const KConst& kc, const double4* pos4, cudaTextureObject_t tex,
                                          const uint32_t* tp,
                                          const uint32_t* nbr, const uint32_t* cn, const uint32_t* co,
                                          int i, int sub, bool live, double& ri) {
  const uint32_t nf = live ? cn[i] : 0u;
  const uint32_t m = live ? nf + co[i] : 0u;
  return ppe_row_core<TWO_PHASE, TEX>(kc, pos4, tex, tp, row_ptr(nbr, kc.stride, i), nf, m, kc.stale, i, sub, ri);
}

// ---- matrix-free solve on skin rows: the exact list of row g, once per solve -----------------------------
// Positions are fixed during a solve, so the re-test of a skin row (and the skipping of its dummies) need not be
// repeated in every application: the entries that pass go to a plain list (a.mcol row g, count a.mcnt[g]) in the
// row's order, and the CG loop walks that (10 % fewer gathers, no test).  Every lane of the warp comes through
// here with a warp-uniform trip count m_max.
__device__ __forceinline__ void compact_row(const KConst& kc, const PpeArgs& a, int g, int i, int sub, int grp,
                                            bool live, uint32_t m_max) {
  const double4 pi = a.pos4[i];
  const uint32_t* row = row_ptr(a.nbr, kc.stride, i);
  const uint32_t nf = live ? a.cn[i] : 0u;
  const uint32_t m = live ? nf + a.co[i] : 0u;
  uint32_t* crow = a.mcol + (size_t)g * (size_t)kc.stride;
  const uint32_t lt = (1u << sub) - 1u;
  uint32_t cnt = 0;
  for (uint32_t k0 = 0; k0 < m_max; k0 += PPE_ILP * L) {
    uint32_t e[PPE_ILP];
    double4 q[PPE_ILP];
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const uint32_t kk = k0 + (uint32_t)(u * L + sub);
      e[u] = kk < m ? row_entry(row, kc.stride, nf, kk) : NB_DUMMY;
    }
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u)
      q[u] = (e[u] & NB_DUMMY) ? make_double4(pi.x + 2.0 * kc.re_lap, pi.y, pi.z, 0.0) : a.pos4[e[u] & NB_INDEX];
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const double r2 = pair_r2(q[u].x - pi.x, q[u].y - pi.y, q[u].z - pi.z, 1);
      const bool keep = !(e[u] & NB_DUMMY) && r2 < kc.re_lap2;
      const uint32_t m8 = (__ballot_sync(0xffffffffu, keep) >> (grp * L)) & ((1u << L) - 1u);
      if (keep) crow[cnt + (uint32_t)__popc(m8 & lt)] = e[u];
      cnt += (uint32_t)__popc(m8);
    }
  }
  if (live && sub == 0) a.mcnt[g] = cnt;
}

// ---- assembly of one row (ppe_operator 1) ----------------------------------------------
// Walks the neighbour row of slot i once, computes c_ij as ppe_row does and writes the pairs
// whose j is an unknown too as (value, compact column), in the row's order, at the start of
// ELL row g; neighbours on the free surface (p = 0) only add to the diagonal term.
// Every lane of the warp must come through here with a warp-uniform trip count m_max.
// The word needs the row's scale before its first coefficient is known.  EXACT = false: one pass with a
// provisional scale -- the coefficient of a pair at 0.5 l0 (kc.asm_wmax), within a bit or two of the true
// largest one of a row -- packing as it goes; if some pair of the row is closer than that (redo), the caller
// runs the row again with EXACT = true: coefficients to scratch, their true maximum, then the packing pass.
template <bool TWO_PHASE, bool EXACT>
__device__ __forceinline__ uint32_t assemble_row(const KConst& kc, const PpeArgs& a, int g, int i, int sub,
                                                 int grp, bool live, uint32_t m_max, bool& redo) {
  const double4 pi = a.pos4[i];
  const uint32_t* row = row_ptr(a.nbr, kc.stride, i);
  const uint32_t nf = live ? a.cn[i] : 0u;
  const uint32_t m = live ? nf + a.co[i] : 0u;
  const int ph_i = TWO_PHASE ? (int)((a.tp[i] >> 8) & 1) : 0;
  const double inv_rij0 = kc.inv_rho_pair[ph_i][0], inv_rij1 = kc.inv_rho_pair[ph_i][1];
  const bool hl = kc.ppe_laplacian == 1;
  const double scale = (hl ? kc.hl_c : kc.A_lap) * (TWO_PHASE ? 1.0 : 1.0 / kc.rho[0]);
  double* vrow = a.mval + (size_t)g * (size_t)kc.stride;
  uint32_t* crow = a.mcol + (size_t)g * (size_t)kc.stride;
  unsigned long long* prow = reinterpret_cast<unsigned long long*>(vrow);
  const double cprov = scale * kc.asm_wmax * (TWO_PHASE ? fmax(inv_rij0, inv_rij1) : 1.0);
  const double invp = PACK_QMAX / cprov;
  const uint32_t lt = (1u << sub) - 1u;
  uint32_t cnt = 0;
  double dex = 0.0, cmax = 0.0;
  for (uint32_t k0 = 0; k0 < m_max; k0 += PPE_ILP * L) {
    uint32_t e[PPE_ILP], rm[PPE_ILP];
    double4 q[PPE_ILP];
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const uint32_t kk = k0 + (uint32_t)(u * L + sub);
      e[u] = kk < m ? row_entry(row, kc.stride, nf, kk) : NB_DUMMY;
    }
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const bool use = !(e[u] & NB_DUMMY);
      const uint32_t j = e[u] & NB_INDEX;
      q[u] = use ? a.pos4[j] : make_double4(pi.x + kc.re_lap, pi.y, pi.z, -2.0);
    }
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u)  // the neighbour's row code from its record: -2 none, -1 free surface, else its row
      rm[u] = q[u].w >= 0.0 ? (uint32_t)q[u].w : (q[u].w == -1.0 ? ROW_SURFACE : ROW_NONE);
#pragma unroll
    for (int u = 0; u < PPE_ILP; ++u) {
      const double dx = q[u].x - pi.x, dy = q[u].y - pi.y, dz = q[u].z - pi.z;
      const double r2 = pair_r2(dx, dy, dz, kc.stale);
      double c = scale * pair_coef<TWO_PHASE>(kc, hl, r2, e[u], inv_rij0, inv_rij1);
      if (kc.stale && !(r2 < kc.re_lap2)) rm[u] = ROW_NONE;  // reused row: the pair has left the radius
      const bool off = rm[u] < ROW_SURFACE;
      if (rm[u] == ROW_SURFACE) dex += c;
      const uint32_t m8 = (__ballot_sync(0xffffffffu, off) >> (grp * L)) & ((1u << L) - 1u);
      if (off) {
        const uint32_t at = cnt + (uint32_t)__popc(m8 & lt);
        if (EXACT) {
          vrow[at] = c;
          crow[at] = rm[u];
        } else {
          prow[at] = ((unsigned long long)rm[u] << 40) | __double2ull_rn(fmin(c, cprov) * invp);
        }
        cmax = fmax(cmax, c);
      }
      cnt += (uint32_t)__popc(m8);
    }
  }
  dex = group_sum<L>(dex);
  cmax = group_max<L>(cmax);
  redo = !EXACT && cmax > cprov;
  if (EXACT) {
    // second pass over the row just written (L1 / L2 hot): pack (coefficient, column) into one word
    __syncwarp();
    const double inv = cmax > 0.0 ? PACK_QMAX / cmax : 0.0;
    for (uint32_t k = sub; k < cnt; k += L) {
      const unsigned long long q = __double2ull_rn(vrow[k] * inv);
      prow[k] = ((unsigned long long)crow[k] << 40) | q;
    }
  }
  if (live && sub == 0) {
    a.mcnt[g] = cnt;
    a.mdex[g] = dex + kc.compress_dt2;
    a.mscale[g] = (EXACT ? cmax : cprov) / PACK_QMAX;
  }
  return cnt;
}

// ---- one row of y = A v with the assembled operator -------------------------------------
// y_g = sum_k val_k (v_g - v_col_k) + dex_g v_g: the same sum as ppe_row, pair by pair.
// Matrix entries are read once per application: streaming loads; v is gathered through L1.
// a packed word: compact column in the high 24 bits, q = round(c / c_max (2^40 - 1)) in the low 40.  q as a double
// without a conversion or a 64-bit shift: 2^52 + q is the word's low 40 bits under the exponent of 2^52
// (two instructions per word instead of the four of the column-low layout: 219 -> 213 ps per row per iteration).
__device__ __forceinline__ double word_coef(uint32_t hi, uint32_t lo) {
  return __hiloint2double((int)((hi & 0xffu) | 0x43300000u), (int)lo) - 4503599627370496.0;
}
template <int LL = L>
__device__ __forceinline__ double asm_row(const KConst& kc, const PpeArgs& a, const double* __restrict__ v,
                                          int g, int sub, bool live, double& vg) {
  vg = v[g];
  const uint32_t n = live ? a.mcnt[g] : 0u;
  const unsigned long long* prow = reinterpret_cast<const unsigned long long*>(a.mval) + (size_t)g * (size_t)kc.stride;
  double s0 = 0.0, s1 = 0.0;
  for (uint32_t k = sub; k < n; k += ASM_ILP * LL) {
    unsigned long long w[ASM_ILP];
#pragma unroll
    for (int u = 0; u < ASM_ILP; ++u) {
      const uint32_t kk = k + (uint32_t)(u * LL);
      w[u] = kk < n ? __ldcs(prow + kk) : ((unsigned long long)(uint32_t)g << 40);  // q = 0, column g
    }
    double vj[ASM_ILP];
#pragma unroll
    for (int u = 0; u < ASM_ILP; ++u) vj[u] = v[(uint32_t)(w[u] >> 40)];
#pragma unroll
    for (int u = 0; u < ASM_ILP; u += 2) {
      const double c0 = word_coef((uint32_t)(w[u] >> 32), (uint32_t)w[u]);
      const double c1 = word_coef((uint32_t)(w[u + 1] >> 32), (uint32_t)w[u + 1]);
      s0 = fma(c0, vg - vj[u], s0);
      s1 = fma(c1, vg - vj[u + 1], s1);
    }
  }
  const double s = group_sum<LL>(s0 + s1);
  return live ? fma(a.mdex[g], vg, a.mscale[g] * s) : 0.0;
}

// ---- the persistent solve -------------------------------------------------------------
template <bool TWO_PHASE, bool ASM, bool TEX>
__global__ void __launch_bounds__(CG_TPB, 1)
k_ppe_cg(KConst kc, PpeArgs a) {
  __shared__ uint32_t sh_cnt[2][CG_TPB / 32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int nb = (int)gridDim.x, bid = (int)blockIdx.x;
  unsigned int gen = 0;
  unsigned long long t_start = 0, t_loop = 0;
  if (bid == 0 && tid == 0) { t_start = global_ns(); a.cg->nnz = 0ull; }

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
      // warm start (Q15 option): the particle's previous pressure, carried in pos4.w by the sort
      const double x0 = (a.warm && f == 0) ? a.pos4[i].w : 0.0;
      a.bc[i] = f;
      a.b[i] = bi;
      a.x[i] = x0;
      if (ASM) {
        // rows get their index in the compaction below.  The code also rides in pos4.w (free during an assembled
        // solve) as a double, so that the assembly finds it in the position record it gathers anyway
        a.rowmap[i] = f == 1 ? ROW_SURFACE : ROW_NONE;
        a.pos4[i].w = f == 1 ? -1.0 : -2.0;
      } else {
        a.pv[i] = 0.0;
        a.sv[i] = 0.0;
        a.pos4[i].w = a.warm ? x0 : bi;  // r0 = b (the warm start applies A to x0 first)
      }
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
  if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;

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
    if (is_row) {
      const uint32_t g = (uint32_t)row_off + off + (uint32_t)__popc(m & ((1u << lane) - 1u));
      a.rows[g] = (uint32_t)i;
      if (ASM) {
        a.rowmap[i] = g;
        a.pos4[i].w = (double)g;  // exact: g < 2^24
      }
    }
    row_off += (int)tot;
  }
  if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;

  const int gthreads = nb * CG_TPB;
  const int gtid = bid * CG_TPB + tid;
  const int sub = tid & (L - 1);
  const int grp = lane / L;
  // Rows are dealt to the blocks in super-chunks of SCW warps (SCW * 32 / L consecutive rows, so
  // the warps that share an SM's L1 work on neighbouring rows) round-robin over the grid:
  // every block gets an even sample of cheap (wall) and expensive (fluid) rows and at most
  // one super-chunk more than any other.  The trip count is warp-uniform.
  const int sc_first = (wid / SCW) * nb + bid;
  const int sc_step = (CG_TPB / 32 / SCW) * nb;
  const int g_in_sc = (wid % SCW) * GPW + grp;

  // -- ppe_operator 1: assemble the rows, set up the compact vectors ------------------------
  if (ASM) {
    uint32_t nnz = 0;
    for (int sc = sc_first; sc * (SCW * GPW) < n_rows; sc += sc_step) {
      const int g = sc * (SCW * GPW) + g_in_sc;
      const bool live = g < n_rows;
      const int i = live ? (int)a.rows[g] : 0;
      uint32_t m = live ? a.cn[i] + a.co[i] : 0u;
      m = __reduce_max_sync(0xffffffffu, m);
      bool redo;
      uint32_t cnt = assemble_row<TWO_PHASE, false>(kc, a, live ? g : 0, i, sub, grp, live, m, redo);
      if (__any_sync(0xffffffffu, redo))  // a pair closer than 0.5 l0 in one of the warp's rows: the two-pass form
        cnt = assemble_row<TWO_PHASE, true>(kc, a, live ? g : 0, i, sub, grp, live, m, redo);
      if (live && sub == 0) {
        nnz += cnt;
        a.xc[g] = a.x[i];
        a.rc[g] = a.b[i];
        a.pv[g] = 0.0;
        a.sv[g] = 0.0;
      }
    }
    nnz = __reduce_add_sync(0xffffffffu, nnz);
    if (lane == 0 && nnz) atomicAdd(&a.cg->nnz, (unsigned long long)nnz);
    if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
  }
  // -- matrix-free on skin rows: the exact list of every unknown row, once ------------------------------
  if (!ASM && a.compact) {
    for (int sc = sc_first; sc * (SCW * GPW) < n_rows; sc += sc_step) {
      const int g = sc * (SCW * GPW) + g_in_sc;
      const bool live = g < n_rows;
      const int i = live ? (int)a.rows[g] : 0;
      uint32_t m = live ? a.cn[i] + a.co[i] : 0u;
      m = __reduce_max_sync(0xffffffffu, m);
      compact_row(kc, a, live ? g : 0, i, sub, grp, live, m);
    }
    if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
  }
  // one row of the matrix-free operator, from the exact list when there is one
  auto mf_row = [&](int g, int i, bool live, double& ri) {
    if (a.compact) {
      const uint32_t m = live ? a.mcnt[g] : 0u;
      return ppe_row_core<TWO_PHASE, TEX>(kc, a.pos4, a.tex, a.tp, a.mcol + (size_t)g * (size_t)kc.stride, m, m, 0, i, sub, ri);
    }
    return ppe_row<TWO_PHASE, TEX>(kc, a.pos4, a.tex, a.tp, a.nbr, a.cn, a.co, i, sub, live, ri);
  };
  // -- warm start: r0 = b - A x0 ---------------------------------------------------------------
  if (a.warm) {
    for (int sc = sc_first; sc * (SCW * GPW) < n_rows; sc += sc_step) {
      const int g = sc * (SCW * GPW) + g_in_sc;
      const bool live = g < n_rows;
      double xi;
      if (ASM) {
        const double t = asm_row(kc, a, a.xc, live ? g : 0, sub, live, xi);
        if (live && sub == 0) a.rc[g] = a.rc[g] - t;
      } else {
        const int i = live ? (int)a.rows[g] : 0;
        const double t = mf_row(live ? g : 0, i, live, xi);
        if (live && sub == 0) a.wv[i] = t;
      }
    }
    if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
    if (!ASM) {  // every gather of x0 is done: pos4.w <- r0
      for (int g = gtid; g < n_rows; g += gthreads) {
        const int i = (int)a.rows[g];
        a.pos4[i].w = a.b[i] - a.wv[i];
      }
      if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
    }
  }
  if (bid == 0 && tid == 0) t_loop = global_ns();

  // -- S8b-3, S8b-4: conjugate gradients ---------------------------------------------------
  const double tol2bb = a.tol2 * bb;
  int iters = 0, converged = (bb == 0.0) ? 1 : 0;
  double gam = bb, gamma_old = 1.0, alpha_old = 1.0;
  if (!converged) {
    for (;;) {
      // phase A: w = A r, gamma = r.r, delta = r.w
      double g_part = 0.0, d_part = 0.0;
      // assembled operator: the loop is bound by HBM latency x bytes in flight, so each group asks
      // the L2 for the words of its NEXT row (one 128-byte line per lane, as many as that row has)
      // while it works on this one; the row counts run one more row ahead
      if (ASM) {
        // LA lanes per row: a batch of ASM_ILP words per lane covers 8 LA entries of the row
        constexpr int LA = ASM_L, GPWA = 32 / LA;
        const int subA = lane & (LA - 1);
        const int g_in_scA = (wid % SCW) * GPWA + lane / LA;
        // super-chunks are dealt in runs of ASM_RUN consecutive ones (round-robin over the grid between runs): the
        // next trip of a warp then works on the rows next to the ones it just did, whose neighbours it has just
        // gathered into this SM's L1
        // (runs of 2^ASM_RUN_LOG2 super-chunks; single ones when a warp group would get fewer than eight runs --
        // load balance: 260k rows measured 221 ps per row per iteration with single super-chunks, 227 with runs of 8)
        constexpr int RPS = SCW * GPWA;  // rows per super-chunk
        const int rs = n_rows >= RPS * sc_step * MPS_ASM_MINRUNS * (1 << ASM_RUN_LOG2) ? ASM_RUN_LOG2 : 0;
        auto row_of = [&](int t) { return ((((sc_first + (t >> rs) * sc_step) << rs) + (t & ((1 << rs) - 1))) * RPS) + g_in_scA; };
        auto trips_left = [&](int t) { return ((sc_first + (t >> rs) * sc_step) << rs) * RPS < n_rows; };
        // (prefetch distance 1 / 2 / 3 trips measured: 208 / 210 / 215 ps per row per iteration at 1.44M rows,
        // 216 / 227 / 240 at 260k)
        uint32_t n_ahead = 0;
        {
          const int g1 = row_of(1);
          n_ahead = g1 < n_rows ? a.mcnt[g1] : 0u;
        }
        for (int t = 0; trips_left(t); ++t) {
          const int g = row_of(t);
          const bool live = g < n_rows;
          double ri;
          const int g1 = row_of(t + 1), g2 = row_of(t + 2);
          for (uint32_t k = (uint32_t)subA * 16u; k < n_ahead; k += 16u * LA)
            prefetch_l2(reinterpret_cast<const unsigned long long*>(a.mval) + (size_t)g1 * (size_t)kc.stride + k);
          n_ahead = g2 < n_rows ? a.mcnt[g2] : 0u;
          const double wi = asm_row<LA>(kc, a, a.rc, live ? g : 0, subA, live, ri);
          if (live && subA == 0) {
            a.wv[g] = wi;
            g_part = fma(ri, ri, g_part);
            d_part = fma(ri, wi, d_part);
          }
        }
      } else {
        for (int sc = sc_first; sc * (SCW * GPW) < n_rows; sc += sc_step) {
          const int g = sc * (SCW * GPW) + g_in_sc;
          const bool live = g < n_rows;
          double ri;
          const int i = live ? (int)a.rows[g] : 0;
          const double wi = mf_row(live ? g : 0, i, live, ri);
          if (live && sub == 0) {
            a.wv[i] = wi;
            g_part = fma(ri, ri, g_part);
            d_part = fma(ri, wi, d_part);
          }
        }
      }
      block_sum2<CG_TPB>(g_part, d_part);
      if (tid == 0) {
        a.part[2 * bid] = g_part;
        a.part[2 * bid + 1] = d_part;
      }
      if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
      double del = 0.0;
      gam = 0.0;
      for (int k = tid; k < nb; k += CG_TPB) {
        gam += __ldcg(&a.part[2 * k]);
        del += __ldcg(&a.part[2 * k + 1]);
      }
      block_sum2<CG_TPB>(gam, del);
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
      if (ASM) {
        for (int g = gtid; g < n_rows; g += gthreads) {
          const double r = a.rc[g];
          const double pn = fma(beta, a.pv[g], r);
          const double sn = fma(beta, a.sv[g], a.wv[g]);
          a.pv[g] = pn;
          a.sv[g] = sn;
          a.xc[g] = fma(alpha, pn, a.xc[g]);
          a.rc[g] = fma(-alpha, sn, r);
        }
      } else {
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
      }
      if (!grid_barrier(a.bar, gen, a.timeout_cycles)) return;
    }
  }
  const unsigned long long t_end = (bid == 0 && tid == 0) ? global_ns() : 0ull;

  // -- S8b-5: pressures from x (Q4), staged into pos4.w for the gradient ------------------
  for (int i = gtid; i < kc.n; i += gthreads) {
    double v;
    if (ASM) {
      const uint32_t g = a.rowmap[i];
      v = g < ROW_SURFACE ? a.xc[g] : 0.0;
      a.x[i] = v;
    } else {
      v = (a.bc[i] == 0) ? a.x[i] : 0.0;
    }
    if (bb == 0.0) v = 0.0;  // b = 0: the solution is 0 whatever the start
    if (kc.clamp_negative_p && v < 0.0) v = 0.0;
    a.p[i] = v;
    a.pos4[i].w = v;
  }
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
    a.cg->iters_total += iters;
    a.cg->noconv_total += converged ? 0 : 1;
    a.cg->t_setup_ns = t_loop - t_start;
    a.cg->t_loop_ns = t_end - t_loop;
    a.cg->t_loop_ns_total += t_end - t_loop;
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
template <bool TWO_PHASE>
__global__ void __launch_bounds__(256)
k_ppe_apply(KConst kc, const double4* pos4, const uint32_t* __restrict__ tp, const int8_t* __restrict__ bc,
            const uint32_t* __restrict__ nbr, const uint32_t* __restrict__ cn,
            const uint32_t* __restrict__ co, double* __restrict__ wv) {
  const int i = (int)((blockIdx.x * 256u + threadIdx.x) / L);
  const int sub = threadIdx.x & (L - 1);
  const bool in = i < kc.n;
  const bool live = in && bc[i] == 0;
  double ri;
  const double wi = ppe_row<TWO_PHASE, false>(kc, pos4, 0, tp, nbr, cn, co, in ? i : 0, sub, live, ri);
  if (in && sub == 0) wv[i] = live ? wi : 0.0;
}
__global__ void k_stage_out(int n, int order, const uint32_t* __restrict__ oid,
                            const double* __restrict__ src, double* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = src[i];
}
// the same through the matrix assembled by the last solve (compact numbering)
__global__ void k_stage_in_c(int n_rows, int order, const uint32_t* __restrict__ rows,
                             const uint32_t* __restrict__ oid, const double* __restrict__ src,
                             double* __restrict__ vc) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n_rows) return;
  const uint32_t i = rows[g];
  vc[g] = src[order == MPS_ORDER_ORIGINAL ? oid[i] : i];
}
__global__ void __launch_bounds__(256)
k_ppe_apply_c(KConst kc, PpeArgs a, int n_rows, const double* __restrict__ vc, double* __restrict__ yc) {
  const int g = (int)((blockIdx.x * 256u + threadIdx.x) / L);
  const int sub = threadIdx.x & (L - 1);
  const bool live = g < n_rows;
  double vg;
  const double y = asm_row(kc, a, vc, live ? g : 0, sub, live, vg);
  if (live && sub == 0) yc[g] = y;
}
__global__ void k_stage_out_c(int n, int order, const uint32_t* __restrict__ rowmap,
                              const uint32_t* __restrict__ oid, const double* __restrict__ yc,
                              double* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t g = rowmap[i];
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = g < ROW_SURFACE ? yc[g] : 0.0;
}

template <bool TWO_PHASE, bool ASM, bool TEX>
cudaError_t launch_cg(mps_ctx* c, PpeArgs& a, int grid) {
  void* params[] = {(void*)&c->kc, (void*)&a};
  return cudaLaunchCooperativeKernel((const void*)k_ppe_cg<TWO_PHASE, ASM, TEX>, dim3(grid), dim3(CG_TPB),
                                     params, 0, c->stream);
}
template <bool TWO_PHASE, bool ASM, bool TEX>
int cg_blocks_per_sm() {
  int nb = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_ppe_cg<TWO_PHASE, ASM, TEX>, CG_TPB, 0);
  return nb;
}

bool two_phase(const mps_ctx* c) { return c->prm.n_phases > 1 && c->prm.rho[0] != c->prm.rho[1]; }

PpeArgs make_args(mps_ctx* c) {
  const int cur = c->cur;
  PpeArgs a;
  a.pos4 = c->pos4[cur]; a.tex = c->cg_tex ? c->pos_tex[cur] : 0; a.tp = c->tp[cur]; a.dens = c->dens;
  a.dndt = c->dndt; a.keep2 = c->keep2[cur]; a.bc = c->bc; a.b = c->b;
  a.x = c->cg_x; a.pv = c->cg_p; a.sv = c->cg_s; a.wv = c->cg_w; a.p = c->p;
  a.nbr = c->nbr; a.cn = c->cn; a.co = c->co; a.rows = c->cg_rows; a.bcount = c->cg_bcount;
  a.part = c->cg_part; a.cg = c->cg; a.bar = c->cg_bar;
  a.rowmap = c->rowmap; a.mval = c->mat_val; a.mcol = c->mat_col; a.mcnt = c->mat_cnt; a.mdex = c->mat_dex; a.mscale = c->mat_scale;
  a.rc = c->cg_rc; a.xc = c->cg_xc;
  a.tol2 = c->prm.cg_rtol * c->prm.cg_rtol;
  a.timeout_cycles = c->cg_timeout_cycles;
  a.maxit = c->prm.cg_maxit;
  a.warm = c->prm.cg_warm_start ? 1 : 0;
  a.compact = (c->prm.ppe_operator == 0 && c->kc.stale && c->mat_col && c->mat_cnt) ? 1 : 0;
  return a;
}

}  // namespace

// ============================================================ host launchers ===
// Number of co-resident blocks of the persistent kernel (called once at init).
int mpsk_ppe_plan(mps_ctx* c) {
  int per_sm;
  const bool tp = two_phase(c);
  const bool as = c->prm.ppe_operator == 1;
  if (as) per_sm = tp ? cg_blocks_per_sm<true, true, false>() : cg_blocks_per_sm<false, true, false>();
  else if (c->cg_tex) per_sm = tp ? cg_blocks_per_sm<true, false, true>() : cg_blocks_per_sm<false, false, true>();
  else per_sm = tp ? cg_blocks_per_sm<true, false, false>() : cg_blocks_per_sm<false, false, false>();
  if (per_sm < 1) return MPS_ERR_CUDA;
  c->cg_grid = c->sm_count;  // one 1024-thread block per SM
  c->cg_lanes = L;
  const char* to = getenv("MPS_B200_CG_TIMEOUT_CYCLES");  // documented in include/mps_b200.h
  if (to) c->cg_timeout_cycles = atoll(to);
  return MPS_OK;
}

// Reads the solve statistics back (one small copy and a stream synchronisation).
int mpsk_ppe_read_stats(mps_ctx* c) {
  cudaMemcpyAsync(c->cg_host, c->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, c->stream);
  cudaMemcpyAsync(c->bar_host, c->cg_bar, sizeof(GridBar), cudaMemcpyDeviceToHost, c->stream);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) {
    c->err = std::string("CUDA error in the PPE solve: ") + cudaGetErrorString(e);
    return MPS_ERR_CUDA;
  }
  const CgScalars& s = *c->cg_host;
  if (c->bar_host->timeout) {
    c->err = "grid barrier timed out inside k_ppe_cg";
    return MPS_ERR_CUDA;
  }
  c->stats.cg_iters = s.iters;
  c->stats.cg_converged = s.converged;
  c->stats.cg_relres = s.bb > 0.0 ? sqrt(s.gamma / s.bb) : 0.0;
  c->stats.n_surface = s.n_surface;
  c->stats.n_rows = s.n_rows;
  c->stats.cg_iters_total = s.iters_total;
  c->stats.cg_noconv_total = s.noconv_total;
  c->stats.cg_setup_ms = 1e-6 * (double)s.t_setup_ns;
  c->stats.cg_loop_ms = 1e-6 * (double)s.t_loop_ns;
  c->stats.cg_loop_ms_total = 1e-6 * (double)s.t_loop_ns_total;
  c->stats.cg_nnz = (int64_t)s.nnz;
  const bool noconv = s.noconv_total > c->noconv_seen;
  c->noconv_seen = s.noconv_total;
  if (noconv) {
    c->err = "CG reached cg_maxit without meeting cg_rtol";
    return MPS_ERR_NOCONV;
  }
  return MPS_OK;
}

int mpsk_pressure_ppe(mps_ctx* c, bool sync) {
  PpeArgs a = make_args(c);
  // small problems: no more blocks than there is work for (fewer arrivals per barrier)
  int grid = c->cg_grid;
  const int want = std::max(1, div_up((int64_t)c->n * L, CG_TPB));
  if (grid > want) grid = want;
  cudaMemsetAsync(c->cg_bar, 0, sizeof(GridBar), c->stream);
  if (((c)->timer_mask >> MPS_T_CG_SPMV) & 1u) mps_timer_begin(c, MPS_T_CG_SPMV);
  cudaError_t e;
  const bool tp = two_phase(c);
  if (c->prm.ppe_operator == 1) e = tp ? launch_cg<true, true, false>(c, a, grid) : launch_cg<false, true, false>(c, a, grid);
  else if (c->cg_tex) e = tp ? launch_cg<true, false, true>(c, a, grid) : launch_cg<false, false, true>(c, a, grid);
  else e = tp ? launch_cg<true, false, false>(c, a, grid) : launch_cg<false, false, false>(c, a, grid);
  c->launches++;
  c->t_launches[MPS_T_CG_SPMV]++;
  if (((c)->timer_mask >> MPS_T_CG_SPMV) & 1u) mps_timer_end(c, MPS_T_CG_SPMV);
  if (e != cudaSuccess) {
    c->err = std::string("cooperative launch of k_ppe_cg failed: ") + cudaGetErrorString(e);
    return MPS_ERR_CUDA;
  }
  c->ppe_ready = true;
  c->posw_is_p = true;
  return sync ? mpsk_ppe_read_stats(c) : MPS_OK;
}

int mpsk_ppe_apply(mps_ctx* c, const double* x, double* y, int order) {
  const int n = (int)c->n;
  const int cur = c->cur;
  if (c->prm.ppe_operator == 1) {
    // the matrix assembled by the last solve; cg_w / cg_s serve as compact staging vectors
    const int nr = c->stats.n_rows;
    PpeArgs a = make_args(c);
    if (nr > 0) {
      MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_in_c, div_up(nr, 256), 256, nr, order, c->cg_rows, c->oid[cur], x,
                 c->cg_s);
      MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_ppe_apply_c, div_up((int64_t)nr * L, 256), 256, c->kc, a, nr, c->cg_s,
                 c->cg_w);
    }
    MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_out_c, div_up(n, 256), 256, n, order, c->rowmap, c->oid[cur], c->cg_w,
               y);
    return MPS_OK;
  }
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_in, div_up(n, 256), 256, n, order, c->bc, c->oid[cur], x,
             c->pos4[cur]);
  c->posw_is_p = false;
  const int grid = div_up((int64_t)n * L, 256);
  if (two_phase(c)) {
    MPS_LAUNCH(c, MPS_T_PPE_SETUP, (k_ppe_apply<true>), grid, 256, c->kc, c->pos4[cur], c->tp[cur],
               c->bc, c->nbr, c->cn, c->co, c->cg_w);
  } else {
    MPS_LAUNCH(c, MPS_T_PPE_SETUP, (k_ppe_apply<false>), grid, 256, c->kc, c->pos4[cur], c->tp[cur],
               c->bc, c->nbr, c->cn, c->co, c->cg_w);
  }
  MPS_LAUNCH(c, MPS_T_PPE_SETUP, k_stage_out, div_up(n, 256), 256, n, order, c->oid[cur], c->cg_w, y);
  return MPS_OK;
}
