// kernels_bin.cu -- uniform-grid binning (S1-S3 of DESIGN.md): cell key,
// counting sort with a device-side scan, canonical (stable) order inside each
// cell, physical reorder, and the per-step neighbour rows.
// Paper: section 4.1 (cell-linked list), P:288, P:273-274 (neigh[] rows).
#include <algorithm>
#include <string.h>

#include "mps_internal.h"

namespace {

constexpr int TPB = 256;

// A bin of mps_step with a skin is launched in every step and runs only when the device flag *go is up
// (raised by the predictor or the corrector); go == NULL: run.  Uniform over the grid.
__device__ __forceinline__ bool skipped(const int* go) { return go != nullptr && *(const volatile int*)go == 0; }

// ---------------------------------------------------------------- load / io ---
__global__ void k_load(int n, const double* __restrict__ x, const double* __restrict__ y,
                       const double* __restrict__ z, const double* __restrict__ u,
                       const double* __restrict__ v, const double* __restrict__ w,
                       const int32_t* __restrict__ type, const int32_t* __restrict__ phase,
                       double4* __restrict__ pos4, double4* __restrict__ vel4,
                       uint32_t* __restrict__ tp, uint32_t* __restrict__ oid) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  pos4[i] = make_double4(x[i], y[i], z[i], 0.0);
  int t = type[i];
  bool solid = (t == MPS_WALL || t == MPS_DUMMY);
  vel4[i] = make_double4(solid ? 0.0 : u[i], solid ? 0.0 : v[i], solid ? 0.0 : w[i], 0.0);
  tp[i] = (uint32_t)(t & 0xff) | ((uint32_t)(phase[i] & 1) << 8);
  oid[i] = (uint32_t)i;
}

// ------------------------------------------------------- Morton key (key_mode 1) ---
// bit k of c_x -> bit 3k, c_y -> bit 3k+1, c_z -> bit 3k+2, k = 0..9 (the "3 x 10-bit interleave").
__device__ __forceinline__ uint32_t dilate3(uint32_t v) {
  v &= 0x3ffu;
  v = (v | (v << 16)) & 0x030000ffu;
  v = (v | (v << 8)) & 0x0300f00fu;
  v = (v | (v << 4)) & 0x030c30c3u;
  v = (v | (v << 2)) & 0x09249249u;
  return v;
}
__device__ __forceinline__ uint32_t compact3(uint32_t v) {
  v &= 0x09249249u;
  v = (v | (v >> 2)) & 0x030c30c3u;
  v = (v | (v >> 4)) & 0x0300f00fu;
  v = (v | (v >> 8)) & 0x030000ffu;
  v = (v | (v >> 16)) & 0x3ffu;
  return v;
}
__device__ __forceinline__ uint32_t cell_key(const KConst& kc, int cx, int cy, int cz) {
  if (kc.key_mode == 1) return dilate3((uint32_t)cx) | (dilate3((uint32_t)cy) << 1) | (dilate3((uint32_t)cz) << 2);
  return (uint32_t)(cx + kc.nx * (cy + kc.ny * cz));
}
__device__ __forceinline__ void key_cell(const KConst& kc, uint32_t k, int& cx, int& cy, int& cz) {
  if (kc.key_mode == 1) {
    cx = (int)compact3(k); cy = (int)compact3(k >> 1); cz = (int)compact3(k >> 2);
  } else {
    cx = (int)(k % (uint32_t)kc.nx);
    cy = (int)((k / (uint32_t)kc.nx) % (uint32_t)kc.ny);
    cz = (int)(k / ((uint32_t)kc.nx * (uint32_t)kc.ny));
  }
}

// ---------------------------------------------------------------- S1: keys ---
// c_a = floor((x_a - min_a) * inv_h); key = c_x + n_x (c_y + n_y c_z); particles
// outside the grid (or non-finite) become GHOST with key = n_cells.  The rank
// inside the cell comes from a warp-aggregated atomic on the cell counter; the
// canonical order (ascending original index) is restored in k_reorder.
__global__ void k_keys(KConst kc, const double4* __restrict__ pos4, uint32_t* __restrict__ tp,
                       uint32_t* __restrict__ key_tmp, uint32_t* __restrict__ rank,
                       uint32_t* __restrict__ cell_count, DevFlags* __restrict__ flags, const uint32_t* __restrict__ oid,
                       uint32_t* __restrict__ gbit, const int* go) {
  if (skipped(go)) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (go && i == 0) atomicAdd(&flags->bins, 1);
  bool live = i < kc.n;
  uint32_t key = 0xffffffffu;
  if (live) {
    double4 q = pos4[i];
    uint32_t t = tp[i];
    bool ghost = (t & 0xff) == MPS_GHOST;
    // (x - min) * inv_h: a subtraction then a multiplication, each rounded (no FMA possible)
    const double sx = __dsub_rn(q.x, kc.dmin[0]), sy = __dsub_rn(q.y, kc.dmin[1]), sz = __dsub_rn(q.z, kc.dmin[2]);
    // in or out of the domain: always on the contract's grid (B1)
    const double gx = floor(__dmul_rn(sx, kc.inv_h_dom)), gy = floor(__dmul_rn(sy, kc.inv_h_dom));
    const double gz = floor(__dmul_rn(sz, kc.inv_h_dom));
    bool in = (gx >= 0.0 && gx < (double)kc.nx_dom) && (gy >= 0.0 && gy < (double)kc.ny_dom) &&
              (gz >= 0.0 && gz < (double)kc.nz_dom);
    // the cell that holds the particle (the same grid, except for the internal bin of mps_step)
    double fx = floor(__dmul_rn(sx, kc.inv_h)), fy = floor(__dmul_rn(sy, kc.inv_h)), fz = floor(__dmul_rn(sz, kc.inv_h));
    fx = fmin(fx, (double)(kc.nx - 1)); fy = fmin(fy, (double)(kc.ny - 1)); fz = fmin(fz, (double)(kc.nz - 1));
    if (!ghost && !(isfinite(q.x) && isfinite(q.y) && isfinite(q.z))) flags->nonfinite = 1;
    if (ghost || !in) {
      if (!ghost) tp[i] = (t & ~0xffu) | MPS_GHOST;
      key = (uint32_t)kc.ncells;
      const uint32_t o = oid[i];  // ghosts by original index: k_reorder ranks them from this bitmap
      atomicOr(&gbit[o >> 5], 1u << (o & 31u));
    } else {
      key = cell_key(kc, (int)fx, (int)fy, (int)fz);
    }
    key_tmp[i] = key;
  }
  // warp-aggregated atomic: one atomicAdd per distinct key in the warp
  unsigned peers = __match_any_sync(0xffffffffu, key);
  int lane = threadIdx.x & 31;
  int leader = __ffs(peers) - 1;
  uint32_t base = 0;
  if (live && lane == leader) base = atomicAdd(&cell_count[key], (uint32_t)__popc(peers));
  base = __shfl_sync(0xffffffffu, base, leader);
  if (live) rank[i] = base + (uint32_t)__popc(peers & ((1u << lane) - 1u));
}

// ones per word of the ghost bitmap (scanned into gpre: ghosts with a smaller original index, word by word)
__global__ void k_ghost_popc(int nwords, const uint32_t* __restrict__ gbit, uint32_t* __restrict__ gcnt, const int* go) {
  if (skipped(go)) return;
  int w = blockIdx.x * blockDim.x + threadIdx.x;
  if (w < nwords) gcnt[w] = (uint32_t)__popc(gbit[w]);
}

// ------------------------------------------------- device-side exclusive scan ---
// Three small kernels (reduce per tile, scan the tile sums in one block, scan
// each tile with its offset).  Tile = 256 threads x 8 items.
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = TPB * SCAN_ITEMS;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
  __shared__ uint32_t warp_sums[TPB / 32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t s = lane < TPB / 32 ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < TPB / 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += t;
    }
    if (lane < TPB / 32) warp_sums[lane] = s;
  }
  __syncthreads();
  uint32_t off = wid ? warp_sums[wid - 1] : 0;
  *total = warp_sums[TPB / 32 - 1];
  __syncthreads();
  return off + inc - v;
}

__global__ void k_scan_reduce(const uint32_t* __restrict__ in, int64_t n, uint32_t* __restrict__ tile_sum,
                              const int* go) {
  if (skipped(go)) return;
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    int64_t i = base + k * TPB + threadIdx.x;
    if (i < n) s += in[i];
  }
  uint32_t tot;
  block_exclusive_scan(s, &tot);
  if (threadIdx.x == 0) tile_sum[blockIdx.x] = tot;
}
__global__ void k_scan_spine(uint32_t* __restrict__ tile_sum, int ntiles, const int* go) {
  if (skipped(go)) return;
  uint32_t carry = 0;
  for (int base = 0; base < ntiles; base += TPB) {
    int i = base + threadIdx.x;
    uint32_t v = i < ntiles ? tile_sum[i] : 0;
    uint32_t tot;
    uint32_t ex = block_exclusive_scan(v, &tot);
    if (i < ntiles) tile_sum[i] = carry + ex;
    carry += tot;
  }
}
__global__ void k_scan_apply(const uint32_t* __restrict__ in, uint32_t* __restrict__ out, int64_t n,
                             const uint32_t* __restrict__ tile_off, const int* go) {
  if (skipped(go)) return;
  int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS];
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0;
    s += v[k];
  }
  uint32_t tot;
  uint32_t ex = block_exclusive_scan(s, &tot) + tile_off[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k < n) out[base + k] = ex;
    ex += v[k];
  }
}

// Small inputs (a few tiles): the whole scan in ONE block, tile after tile with a running carry
// -- one launch instead of three.
__global__ void __launch_bounds__(TPB) k_scan_small(const uint32_t* __restrict__ in,
                                                    uint32_t* __restrict__ out, int64_t n, const int* go) {
  if (skipped(go)) return;
  uint32_t carry = 0;
  for (int64_t tile = 0; tile < n; tile += SCAN_TILE) {
    const int64_t base = tile + (int64_t)threadIdx.x * SCAN_ITEMS;
    uint32_t v[SCAN_ITEMS];
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
      v[k] = (base + k < n) ? in[base + k] : 0;
      s += v[k];
    }
    uint32_t tot;
    uint32_t ex = block_exclusive_scan(s, &tot) + carry;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
      if (base + k < n) out[base + k] = ex;
      ex += v[k];
    }
    carry += tot;
  }
}

// ------------------------------------------------------- S2: scatter + reorder ---
__global__ void k_scatter(int n, const uint32_t* __restrict__ key_tmp, const uint32_t* __restrict__ rank,
                          const uint32_t* __restrict__ cell_start, const uint32_t* __restrict__ oid,
                          uint32_t* __restrict__ tmp_src, uint32_t* __restrict__ tmp_oid,
                          uint32_t* __restrict__ key, int ncells, DevFlags* __restrict__ flags, const int* go) {
  if (skipped(go)) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    flags->n_ghost = n - (int)cell_start[ncells];  // ghosts sit behind the last cell
    if (go) flags->max_row = 0;                    // the row builder of this bin raises it again
  }
  if (i >= n) return;
  uint32_t k = key_tmp[i];
  uint32_t dst = cell_start[k] + rank[i];
  tmp_src[dst] = (uint32_t)i;
  tmp_oid[dst] = oid[i];
  key[dst] = k;
}

// Final slot of s inside its cell = number of cell mates with a smaller original
// index (ties impossible): this makes the sort the unique stable one whatever
// order the atomics handed out.  Then move the payload.
__global__ void k_reorder(int n, int ncells, const uint32_t* __restrict__ key,
                          const uint32_t* __restrict__ cell_start, const uint32_t* __restrict__ tmp_src,
                          const uint32_t* __restrict__ tmp_oid, const double4* __restrict__ pos_in,
                          const double4* __restrict__ vel_in, const uint32_t* __restrict__ tp_in,
                          double4* __restrict__ pos_out, double4* __restrict__ vel_out,
                          uint32_t* __restrict__ tp_out, uint32_t* __restrict__ oid_out,
                          uint32_t* __restrict__ ent_out, const double2* __restrict__ keep_in,
                          double2* __restrict__ keep_out, const double* __restrict__ rs_in,
                          double* __restrict__ rs_out, int carry_w, const uint32_t* __restrict__ gbit,
                          const uint32_t* __restrict__ gpre, const int* go) {
  if (skipped(go)) return;
  int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= n) return;
  uint32_t c = key[s];
  uint32_t lo = cell_start[c];
  uint32_t me = tmp_oid[s];
  uint32_t f = lo;
  if (c == (uint32_t)ncells) {
    // the ghost pseudo-cell can hold any number of particles (everything that ever left the domain): rank by
    // original index from the bitmap and its scanned word counts instead of a loop over the cell mates
    f += gpre[me >> 5] + (uint32_t)__popc(gbit[me >> 5] & ((1u << (me & 31u)) - 1u));
  } else {
    const uint32_t hi = cell_start[c + 1];
    for (uint32_t t = lo; t < hi; ++t) f += (tmp_oid[t] < me) ? 1u : 0u;
  }
  uint32_t src = tmp_src[s];
  double4 q = pos_in[src];
  if (!carry_w) q.w = 0.0;  // cg_warm_start: the previous pressure follows its particle
  pos_out[f] = q;
  vel_out[f] = vel_in[src];
  const uint32_t tj = tp_in[src];
  const uint32_t ty = tj & 0xff;
  tp_out[f] = tj;
  oid_out[f] = me;
  if (keep_in) keep_out[f] = keep_in[src];  // (n^k, (Dn/Dt)^k) of Eq. 17 follow their particle
  if (rs_in) rs_out[f] = rs_in[src];        // so does the smoothed density of Eq. 11
  // the neighbour-row entry that names this particle (flags of mps_internal.h)
  ent_out[f] = f | (ty == MPS_DUMMY ? NB_DUMMY : 0u) | (ty == MPS_WALL ? NB_WALL : 0u) |
               ((tj & 0x100) ? NB_PHASE1 : 0u);
}

// Inside a CUDA graph the skin bin is the body of a conditional node (cudaGraphCondTypeIf): this one-thread
// kernel, placed just before the node, hands the device flag to the node, so a bin that is not needed costs
// one graph node instead of eight launches that return at once.
__global__ void k_set_cond(cudaGraphConditionalHandle h, const int* go, DevFlags* flags) {
  const int on = *(const volatile int*)go != 0;
  if (on) flags->cond_taken += 1;
  cudaGraphSetConditional(h, on ? 1u : 0u);
}

// The bin of mps_step with a skin leaves the sorted particles in the buffers they came from (so that no
// pointer on the host depends on whether the bin ran) and records the positions the rows are built at.
__global__ void k_commit(int n, const double4* __restrict__ pos_s, const double4* __restrict__ vel_s,
                         const uint32_t* __restrict__ tp_s, const uint32_t* __restrict__ oid_s,
                         const double2* __restrict__ keep_s, const double* __restrict__ rs_s,
                         double4* __restrict__ pos, double4* __restrict__ vel, uint32_t* __restrict__ tp,
                         uint32_t* __restrict__ oid, double2* __restrict__ keep, double* __restrict__ rs,
                         double4* __restrict__ pos_ref, const int* go) {
  if (skipped(go)) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double4 q = pos_s[i];
  pos[i] = q;
  pos_ref[i] = q;
  vel[i] = vel_s[i];
  tp[i] = tp_s[i];
  oid[i] = oid_s[i];
  if (keep) keep[i] = keep_s[i];
  if (rs) rs[i] = rs_s[i];
}

// ------------------------------------------------ S3: neighbour rows (the sweep) ---
// One warp per particle i, the 32 lanes test 32 candidates j at a time.  For every
// (dy, dz) row of cells the candidates are one contiguous slot range (x-fastest
// key), read as coalesced 32-byte records.  Decision: r2 = (dx*dx + dy*dy) + dz*dz
// with every operation rounded separately, r2 < re*re (strict, Eq. 3; Q2).  Hits
// are compacted with a ballot and written as contiguous runs: inside re_n to the
// front of the row, the others to the back; entries come out in ascending slot
// order, so every later sum has a fixed order.
constexpr int ROWS_TPB = 256;
constexpr int ROWS_PPW = 4;  // particles per warp (consecutive slots: almost always one cell)

// Append the hits of one 32-candidate trip to the row of one particle: ballot compaction,
// front part upwards, back part downwards (back_slot).  On overflow keep what fits, in order.
__device__ __forceinline__ void row_append(uint32_t* row, int stride, uint32_t cap, uint32_t lt_mask,
                                           bool in_n, bool in_o, uint32_t e, uint32_t& nf,
                                           uint32_t& nb, bool& overflow) {
  const uint32_t m_n = __ballot_sync(0xffffffffu, in_n);
  const uint32_t m_o = __ballot_sync(0xffffffffu, in_o);
  if ((m_n | m_o) == 0u) return;
  const uint32_t add_n = (uint32_t)__popc(m_n), add_o = (uint32_t)__popc(m_o);
  const uint32_t pn = (uint32_t)__popc(m_n & lt_mask), po = (uint32_t)__popc(m_o & lt_mask);
  if (nf + nb + add_n + add_o <= cap) {
    if (in_n) row[nf + pn] = e;
    else if (in_o) row[back_slot(stride, nb + po)] = e;
    nf += add_n;
    nb += add_o;
  } else {
    overflow = true;
    const uint32_t room = cap - (nf + nb);
    if (in_n && pn < room) row[nf + pn] = e;
    const uint32_t took_n = add_n < room ? add_n : room;
    const uint32_t room_o = room - took_n;
    if (in_o && po < room_o) row[back_slot(stride, nb + po)] = e;
    nf += took_n;
    nb += add_o < room_o ? add_o : room_o;
  }
}

// exact squared distance of reading Q2
__device__ __forceinline__ double r2_exact(const double4& q, const double4& p) {
  const double dx = __dsub_rn(q.x, p.x), dy = __dsub_rn(q.y, p.y), dz = __dsub_rn(q.z, p.z);
  return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

__global__ void __launch_bounds__(ROWS_TPB)
k_build_rows_warp(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ tp,
             const uint32_t* __restrict__ ent, const uint32_t* __restrict__ key,
             const uint32_t* __restrict__ cell_start, uint32_t* __restrict__ nbr,
             uint32_t* __restrict__ cn, uint32_t* __restrict__ co, DevFlags* __restrict__ flags,
             int mode, const int* go) {
  if (skipped(go)) return;
  const int fluid_only = mode & ROWS_FLUID_ONLY;
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * ROWS_TPB + threadIdx.x) >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const int R = kc.R_lap, S = kc.stride;
  const uint32_t cap = (uint32_t)kc.cap;
  const int i0 = warp * ROWS_PPW;
  if (i0 >= kc.n) return;
  int warp_max = 0;
  bool coincident = false, overflow = false;
  // which of the warp's particles want a row, and do they share one cell?
  bool want[ROWS_PPW];
  uint32_t kk[ROWS_PPW];
  bool same = true;
#pragma unroll
  for (int t = 0; t < ROWS_PPW; ++t) {
    const int i = i0 + t;
    kk[t] = i < kc.n ? key[i] : 0xffffffffu;
    want[t] = i < kc.n && kk[t] < (uint32_t)kc.ncells && !(fluid_only && (tp[i] & 0xff) != MPS_FLUID);
    if (i < kc.n && !want[t] && lane == 0) { cn[i] = 0; co[i] = 0; }  // ghost, or not needed by this bin
    same = same && (kk[t] == kk[0]);
  }
  if (same && kk[0] < (uint32_t)kc.ncells) {
    // ---- one candidate load per trip serves all ROWS_PPW particles -----------------------
    const uint32_t k = kk[0];
    const int cx = (int)(k % (uint32_t)kc.nx);
    const int cy = (int)((k / (uint32_t)kc.nx) % (uint32_t)kc.ny);
    const int cz = (int)(k / ((uint32_t)kc.nx * (uint32_t)kc.ny));
    const int x_lo = max(cx - R, 0), x_hi = min(cx + R, kc.nx - 1);
    double4 pi[ROWS_PPW];
    uint32_t nf[ROWS_PPW], nb[ROWS_PPW];
#pragma unroll
    for (int t = 0; t < ROWS_PPW; ++t) { pi[t] = pos4[i0 + t]; nf[t] = 0; nb[t] = 0; }
    for (int dz = -R; dz <= R; ++dz) {
      const int z2 = cz + dz;
      if (z2 < 0 || z2 >= kc.nz) continue;
      for (int dy = -R; dy <= R; ++dy) {
        const int y2 = cy + dy;
        if (y2 < 0 || y2 >= kc.ny) continue;
        const int cbase = kc.nx * (y2 + kc.ny * z2);
        const uint32_t js = cell_start[cbase + x_lo];
        const uint32_t je = cell_start[cbase + x_hi + 1];
        for (uint32_t j0 = js; j0 < je; j0 += 32) {
          const uint32_t j = j0 + (uint32_t)lane;
          const bool valid = j < je;
          double4 q = make_double4(0.0, 0.0, 0.0, 0.0);
          uint32_t e = 0;
          if (valid) { q = pos4[j]; e = ent[j]; }
#pragma unroll
          for (int t = 0; t < ROWS_PPW; ++t) {
            if (!want[t]) continue;  // warp-uniform
            const double r2 = r2_exact(q, pi[t]);
            const bool in_lap = valid && (r2 < kc.re_lap2) && (j != (uint32_t)(i0 + t));
            const bool in_n = in_lap && (r2 < kc.re_n2);
            if (in_lap && r2 == 0.0) coincident = true;
            row_append(nbr + (size_t)(i0 + t) * (size_t)S, S, cap, lt_mask, in_n, in_lap && !in_n, e, nf[t],
                       nb[t], overflow);
          }
        }
      }
    }
#pragma unroll
    for (int t = 0; t < ROWS_PPW; ++t) {
      if (!want[t]) continue;
      if (lane == 0) { cn[i0 + t] = nf[t]; co[i0 + t] = nb[t]; }
      warp_max = max(warp_max, (int)(nf[t] + nb[t]));
    }
  } else {
    // ---- the warp straddles cells (or holds ghosts): one particle after the other ----------
    for (int t = 0; t < ROWS_PPW; ++t) {
      if (!want[t]) continue;
      const int i = i0 + t;
      const uint32_t k = kk[t];
      const double4 pi = pos4[i];
      const int cx = (int)(k % (uint32_t)kc.nx);
      const int cy = (int)((k / (uint32_t)kc.nx) % (uint32_t)kc.ny);
      const int cz = (int)(k / ((uint32_t)kc.nx * (uint32_t)kc.ny));
      const int x_lo = max(cx - R, 0), x_hi = min(cx + R, kc.nx - 1);
      uint32_t* row = nbr + (size_t)i * (size_t)S;
      uint32_t nf = 0, nb = 0;  // warp-uniform
      for (int dz = -R; dz <= R; ++dz) {
        const int z2 = cz + dz;
        if (z2 < 0 || z2 >= kc.nz) continue;
        for (int dy = -R; dy <= R; ++dy) {
          const int y2 = cy + dy;
          if (y2 < 0 || y2 >= kc.ny) continue;
          const int cbase = kc.nx * (y2 + kc.ny * z2);
          const uint32_t js = cell_start[cbase + x_lo];
          const uint32_t je = cell_start[cbase + x_hi + 1];
          for (uint32_t j0 = js; j0 < je; j0 += 32) {
            const uint32_t j = j0 + (uint32_t)lane;
            bool in_lap = false, in_n = false;
            uint32_t e = 0;
            if (j < je) {
              const double r2 = r2_exact(pos4[j], pi);
              in_lap = (r2 < kc.re_lap2) && (j != (uint32_t)i);
              in_n = in_lap && (r2 < kc.re_n2);
              if (in_lap && r2 == 0.0) coincident = true;
              e = ent[j];
            }
            row_append(row, S, cap, lt_mask, in_n, in_lap && !in_n, e, nf, nb, overflow);
          }
        }
      }
      if (lane == 0) { cn[i] = nf; co[i] = nb; }
      warp_max = max(warp_max, (int)(nf + nb));
    }
  }
  coincident = __any_sync(0xffffffffu, coincident);
  if (lane == 0) {
    if (overflow) flags->overflow = 1;
    if (coincident) flags->nonfinite = 1;
    if (warp_max > 0) atomicMax(&flags->max_row, warp_max);
  }
}


// --------------------------------- S3: the row builder (lanes on candidates) ---
// One warp builds the rows of four consecutive slots (almost always one cell): the 32 lanes load 32
// candidates j of a cell run as coalesced records and test them against each of the four particles,
// so one candidate load serves four rows.  A trip costs, per particle, the exact test of reading Q2
// (8 fp64 operations + 2 compares), two ballots and the stores of the hits: the lane that holds hit
// number k of the trip writes entry nf + k of the front part (r < re_n) or entry nb + k of the back
// part (back_slot), so rows come out in ascending slot order with no per-hit loop.  Linear key: the
// candidates of a (dy, dz) row of cells are one contiguous range; Morton key: one range per cell.
// mode: ROWS_FLUID_ONLY (rows of fluid particles only), ROWS_RN_ONLY (front part only, R_n cells).
constexpr int LEAN_TPB = 256;
constexpr int LEAN_PPW = 4;

// rare path: the trip's hits do not all fit; keep what fits, in order
__device__ __noinline__ void row_append_overflow(uint32_t* row, int stride, uint32_t cap, uint32_t lt_mask,
                                                 bool in_n, bool in_o, uint32_t e, uint32_t& nf, uint32_t& nb) {
  const uint32_t m_n = __ballot_sync(0xffffffffu, in_n);
  const uint32_t m_o = __ballot_sync(0xffffffffu, in_o);
  const uint32_t add_n = (uint32_t)__popc(m_n), add_o = (uint32_t)__popc(m_o);
  const uint32_t pn = (uint32_t)__popc(m_n & lt_mask), po = (uint32_t)__popc(m_o & lt_mask);
  const uint32_t room = cap - (nf + nb);
  if (in_n && pn < room) row[nf + pn] = e;
  const uint32_t took_n = add_n < room ? add_n : room;
  const uint32_t room_o = room - took_n;
  if (in_o && po < room_o) row[back_slot(stride, nb + po)] = e;
  nf += took_n;
  nb += add_o < room_o ? add_o : room_o;
}

__global__ void __launch_bounds__(LEAN_TPB)
k_build_rows(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ ent,
             const uint32_t* __restrict__ key, const uint32_t* __restrict__ cell_start,
             uint32_t* __restrict__ nbr, uint32_t* __restrict__ cn, uint32_t* __restrict__ co,
             DevFlags* __restrict__ flags, int mode, const int* go) {
  if (skipped(go)) return;
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * LEAN_TPB + threadIdx.x) >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  const int i0 = warp * LEAN_PPW;
  if (i0 >= kc.n) return;
  const bool rn_only = (mode & ROWS_RN_ONLY) != 0;
  const int R = rn_only ? kc.R_n : kc.R_lap, S = kc.stride;
  const double re_out2 = rn_only ? kc.re_n2 : kc.re_lap2;
  const uint32_t cap = (uint32_t)kc.cap;
  // the four particles: key, wanted?, position, row
  uint32_t kk[LEAN_PPW], nf[LEAN_PPW], nb[LEAN_PPW];
  bool want[LEAN_PPW], back_skip[LEAN_PPW];
  double px[LEAN_PPW], py[LEAN_PPW], pz[LEAN_PPW];
#pragma unroll
  for (int t = 0; t < LEAN_PPW; ++t) {
    const int i = i0 + t;
    const bool in = i < kc.n;
    kk[t] = in ? key[i] : 0xffffffffu;
    const bool solid = in && (ent[i] & (NB_DUMMY | NB_WALL));
    want[t] = in && kk[t] < (uint32_t)kc.ncells && !((mode & ROWS_FLUID_ONLY) && solid);
    back_skip[t] = (mode & ROWS_BACK_FLUID) && solid;
    const double4 q = pos4[in ? i : i0];
    px[t] = q.x; py[t] = q.y; pz[t] = q.z;
    nf[t] = 0; nb[t] = 0;
  }
  bool coincident = false, overflow = false;
  // particles of one cell share the candidate scan; a warp that straddles cells takes them in turns
  for (int t0 = 0; t0 < LEAN_PPW;) {
    int t1 = t0 + 1;
    while (t1 < LEAN_PPW && kk[t1] == kk[t0]) ++t1;
    bool act[LEAN_PPW];
    bool any = false;
#pragma unroll
    for (int t = 0; t < LEAN_PPW; ++t) { act[t] = t >= t0 && t < t1 && want[t]; any = any || act[t]; }
    if (any) {
      int cx, cy, cz;
      key_cell(kc, kk[t0], cx, cy, cz);
      const int x_lo = max(cx - R, 0), x_hi = min(cx + R, kc.nx - 1);
      const int seg = kc.key_mode == 1 ? 1 : x_hi - x_lo + 1;  // cells per contiguous candidate range
      for (int dz = -R; dz <= R; ++dz) {
        const int z2 = cz + dz;
        if (z2 < 0 || z2 >= kc.nz) continue;
        for (int dy = -R; dy <= R; ++dy) {
          const int y2 = cy + dy;
          if (y2 < 0 || y2 >= kc.ny) continue;
          for (int x2 = x_lo; x2 <= x_hi; x2 += seg) {
            const uint32_t js = cell_start[cell_key(kc, x2, y2, z2)];
            const uint32_t je = cell_start[cell_key(kc, x2 + seg - 1, y2, z2) + 1u];
            for (uint32_t j0 = js; j0 < je; j0 += 32) {
              const uint32_t j = j0 + (uint32_t)lane;
              const bool valid = j < je;
              const double4 q = pos4[valid ? j : js];
              const uint32_t e = ent[valid ? j : js];
#pragma unroll
              for (int t = 0; t < LEAN_PPW; ++t) {
                if (!act[t]) continue;  // warp-uniform
                const double dx = __dsub_rn(q.x, px[t]), dy_ = __dsub_rn(q.y, py[t]), dz_ = __dsub_rn(q.z, pz[t]);
                const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy_, dy_)), __dmul_rn(dz_, dz_));
                const bool in_lap = valid && (r2 < re_out2);
                uint32_t m_lap = __ballot_sync(0xffffffffu, in_lap);
                // the particle itself (r2 = 0) sits in lane i - j0 of its own trip
                const uint32_t self = (uint32_t)(i0 + t) - j0;
                if (self < 32u) m_lap &= ~(1u << self);
                if (m_lap == 0u) continue;
                bool hit = (m_lap >> lane) & 1u;
                const bool in_n = hit && (rn_only || r2 < kc.re_n2);
                if (hit && __double2hiint(r2) == 0) coincident = true;  // r = 0 (or denormal): Eq. 3 is infinite
                const uint32_t m_n = __ballot_sync(0xffffffffu, in_n);
                if (back_skip[t]) {  // ROWS_BACK_FLUID: a wall or dummy row keeps its re_n part only (warp-uniform)
                  m_lap = m_n;
                  hit = in_n;
                  if (m_lap == 0u) continue;
                }
                const uint32_t m_o = m_lap & ~m_n;
                uint32_t* row = nbr + (size_t)(i0 + t) * (size_t)S;
                if (nf[t] + nb[t] + (uint32_t)__popc(m_lap) <= cap) {
                  if (in_n) row[nf[t] + (uint32_t)__popc(m_n & lt_mask)] = e;
                  else if (hit) row[back_slot(S, nb[t] + (uint32_t)__popc(m_o & lt_mask))] = e;
                  nf[t] += (uint32_t)__popc(m_n);
                  nb[t] += (uint32_t)__popc(m_o);
                } else {
                  overflow = true;
                  row_append_overflow(row, S, cap, lt_mask, in_n, hit && !in_n, e, nf[t], nb[t]);
                }
              }
            }
          }
        }
      }
    }
    t0 = t1;
  }
  int warp_max = 0;
#pragma unroll
  for (int t = 0; t < LEAN_PPW; ++t) {
    if (i0 + t < kc.n && lane == 0) { cn[i0 + t] = nf[t]; co[i0 + t] = nb[t]; }
    warp_max = max(warp_max, (int)(nf[t] + nb[t]));
  }
  coincident = __any_sync(0xffffffffu, coincident);
  if (lane == 0) {
    if (overflow) flags->overflow = 1;
    if (coincident) flags->nonfinite = 1;
    if (warp_max > *(volatile int*)&flags->max_row) atomicMax(&flags->max_row, warp_max);
  }
}

// ------------------------------------ S3, cell_div = 1: one warp per cell ---
// The 32 lanes hold up to 32 particles i of one cell and walk the candidates j of
// the (2R+1)^2 cell runs in lock-step, so every candidate is ONE broadcast load
// for the whole warp (no gathers) and the exact test costs 8 fp64 operations per
// lane.  Hits are collected per lane in a shared-memory buffer of 8 entries and
// written as whole 32-byte sectors (two 128-bit stores), front part upwards, back
// part downwards (back_slot).  Entries come out in ascending slot order, as above.
// Measured and rejected in round 2: whole rows staged in shared memory
// and copied out coalesced (fewer instructions but 12 instead of 20 warps per SM: 6.1 vs 4.9 ms
// per step at 2M particles), 16-entry rings drained once per 32-candidate chunk (4.7 vs 4.2 ms),
// cells handed out through an atomic counter, grid-wide (2.2 vs 1.2 ms at 438k: the warps of a
// block share the candidates of neighbouring cells in L1) or per block of 24 cells (1.4 vs 1.05 ms
// at 438k, no change at 2M), and a tests-only kernel writing hit masks followed by a warp-per-row
// expansion (1.7 + 1.8 ms per bin at 2M against 2.5 ms: the tests alone take 1.7 ms at 58 % of the
// fp64 pipe, so the appends cost about a third of this kernel, not the half their instruction
// count suggests).  Round 2, later: one loop over both parts of a row with the target chosen per hit (3.67 vs
// 3.51 ms for the two exact bins of a step at 2M: the select costs more than the second loop's overhead).
constexpr int CELL_TPB = 256;
constexpr int CELL_WARPS = CELL_TPB / 32;
constexpr int CELL_BATCH = 8;  // candidates tested per lane before the hits are appended

__device__ __forceinline__ void flush_sector(uint32_t* dst, const uint32_t (*b)[32], int lane) {
  uint4 lo = make_uint4(b[0][lane], b[1][lane], b[2][lane], b[3][lane]);
  uint4 hi = make_uint4(b[4][lane], b[5][lane], b[6][lane], b[7][lane]);
  reinterpret_cast<uint4*>(dst)[0] = lo;
  reinterpret_cast<uint4*>(dst)[1] = hi;
}

// EXACT: the distance test with the rounding of reading Q2 (mps_bin: the rows ARE the sets).  A skin build
// (mps_step) only needs a superset of radius re + 0.9 skin, every sweep re-tests exactly: fused arithmetic,
// two fp64 instructions fewer per candidate.
template <bool EXACT>
__global__ void __launch_bounds__(CELL_TPB, 4)
k_build_rows_cell(KConst kc, const double4* __restrict__ pos4, const uint32_t* __restrict__ ent,
                  const uint32_t* __restrict__ cell_start, uint32_t* __restrict__ nbr,
                  uint32_t* __restrict__ cn, uint32_t* __restrict__ co, DevFlags* __restrict__ flags,
                  int mode, const int* go) {
  if (skipped(go)) return;
  const bool fluid_only = (mode & ROWS_FLUID_ONLY) != 0, rn_only = (mode & ROWS_RN_ONLY) != 0;
  __shared__ uint32_t buf[2][CELL_WARPS][8][32];
  // the 32 candidates of a chunk, loaded once (coalesced, one record per lane) and then read by every lane as
  // shared-memory broadcasts: a warp-uniform LDG.128 costs the L1 a pass per quarter warp, 8 per candidate
  // (ncu: l1tex 72 %, the busiest unit of this kernel), an LDS broadcast one
  __shared__ double2 cand_xy[CELL_WARPS][32];
  __shared__ double cand_z[CELL_WARPS][32];
  __shared__ uint32_t cand_e[CELL_WARPS][32];  // and their row entries
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int gwarp = blockIdx.x * CELL_WARPS + wid;
  const int nwarps = gridDim.x * CELL_WARPS;
  uint32_t (*bn)[32] = buf[0][wid];
  uint32_t (*bo)[32] = buf[1][wid];
  // ghosts sit behind the last cell and have no neighbours
  for (uint32_t i = cell_start[kc.ncells] + (uint32_t)(gwarp * 32 + lane); i < (uint32_t)kc.n;
       i += (uint32_t)nwarps * 32u) {
    cn[i] = 0;
    co[i] = 0;
  }
  const int R = kc.R_lap, S = kc.stride;
  const uint32_t cap = (uint32_t)kc.cap;
  int lane_max = 0;
  int coincident = 0, overflow = 0;
  for (int c = gwarp; c < kc.ncells; c += nwarps) {
    const uint32_t ps = cell_start[c], pe = cell_start[c + 1];
    if (ps == pe) continue;
    const int cx = c % kc.nx, cy = (c / kc.nx) % kc.ny, cz = c / (kc.nx * kc.ny);
    const int x_lo = max(cx - R, 0), x_hi = min(cx + R, kc.nx - 1);
    for (uint32_t base = ps; base < pe; base += 32) {
      const uint32_t i = base + (uint32_t)lane;
      bool act = i < pe;
      if (fluid_only) {  // the first bin of a step serves viscosity: fluid rows only
        if (act && (ent[i] & (NB_DUMMY | NB_WALL))) {
          act = false;
          cn[i] = 0;
          co[i] = 0;
        }
        if (!__any_sync(0xffffffffu, act)) continue;
      }
      const uint32_t ii = act ? i : ps;
      const double4 pi = pos4[ii];
      uint32_t* row = nbr + (size_t)ii * (size_t)S;
      const bool back_skip = (mode & ROWS_BACK_FLUID) && (ent[ii] & (NB_DUMMY | NB_WALL));
      uint32_t nf = 0, nb = 0;
      for (int dz = -R; dz <= R; ++dz) {
        const int z2 = cz + dz;
        if (z2 < 0 || z2 >= kc.nz) continue;
        for (int dy = -R; dy <= R; ++dy) {
          const int y2 = cy + dy;
          if (y2 < 0 || y2 >= kc.ny) continue;
          const int cbase = kc.nx * (y2 + kc.ny * z2);
          const uint32_t js = cell_start[cbase + x_lo];
          const uint32_t je = cell_start[cbase + x_hi + 1];
          for (uint32_t j0 = js; j0 < je; j0 += 32) {
            // phase 1: up to 32 independent exact tests per lane; every load is a warp-uniform
            // broadcast.  Slots past je (at most 31, inside the padded arrays) are masked off.
            const uint32_t cnt = min(32u, je - j0);
            uint32_t m_lap = 0, m_n = 0;
            {
              const double4 mine = pos4[j0 + (uint32_t)lane];  // past je: inside the padded array, masked below
              __syncwarp();                                    // the previous chunk has been read by every lane
              cand_xy[wid][lane] = make_double2(mine.x, mine.y);
              cand_z[wid][lane] = mine.z;
              cand_e[wid][lane] = ent[j0 + (uint32_t)lane];
              __syncwarp();
            }
            const double2* qxy = cand_xy[wid];
            const double* qz = cand_z[wid];
            for (uint32_t g = 0; g < cnt; g += CELL_BATCH, qxy += CELL_BATCH, qz += CELL_BATCH) {
              uint32_t b_lap = 0, b_n = 0;
#pragma unroll
              for (int t = 0; t < CELL_BATCH; ++t) {
                const double2 qa = qxy[t];
                const double dx = __dsub_rn(qa.x, pi.x), dy_ = __dsub_rn(qa.y, pi.y), dz_ = __dsub_rn(qz[t], pi.z);
                const double r2 =
                    EXACT ? __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy_, dy_)), __dmul_rn(dz_, dz_))
                          : fma(dz_, dz_, fma(dy_, dy_, dx * dx));
                if (r2 < kc.re_lap2) b_lap |= 1u << t;
                if (r2 < kc.re_n2) b_n |= 1u << t;
              }
              m_lap |= b_lap << g;
              m_n |= b_n << g;
            }
            uint32_t keep = cnt == 32u ? 0xffffffffu : ((1u << cnt) - 1u);
            if (i - j0 < 32u) keep &= ~(1u << (i - j0));  // j == i
            m_lap = act ? (m_lap & keep) : 0u;
            if (rn_only || back_skip) m_lap &= m_n;  // only the re_n part is wanted (for this row)
            // capacity: keep the first hits that fit (ascending j), flag the rest
            if (nf + nb + (uint32_t)__popc(m_lap) > cap) {
              overflow = 1;
              while (nf + nb + (uint32_t)__popc(m_lap) > cap) m_lap &= ~(0x80000000u >> __clz((int)m_lap));
            }
            m_n &= m_lap;
            uint32_t m_o = m_lap & ~m_n;
            // phase 2: every lane appends its own hits in ascending j.  The entries come from shared memory (word
            // `bit`: distinct bits are distinct banks, equal bits a broadcast), so the loops need no vote and no
            // shuffle and each lane simply runs as long as it has hits
            const uint32_t* ce = cand_e[wid];
            while (m_n) {
              const int bit = __ffs((int)m_n) - 1;
              m_n &= m_n - 1u;
              bn[nf & 7u][lane] = ce[bit];
              ++nf;
              if ((nf & 7u) == 0u) flush_sector(row + (nf - 8u), bn, lane);
            }
            while (m_o) {
              const int bit = __ffs((int)m_o) - 1;
              m_o &= m_o - 1u;
              bo[nb & 7u][lane] = ce[bit];
              ++nb;
              if ((nb & 7u) == 0u) flush_sector(row + ((uint32_t)S - nb), bo, lane);
            }
          }
        }
      }
      // coincident particles (r = 0 makes Eq. 3 infinite) can only be cell mates
      for (uint32_t j = ps; j < pe; ++j) {
        const double4 q = pos4[j];
        if (act && j != i && q.x == pi.x && q.y == pi.y && q.z == pi.z) coincident = 1;
      }
      if (act) {
        if (nf & 7u) flush_sector(row + (nf & ~7u), bn, lane);
        if (nb & 7u) flush_sector(row + ((uint32_t)S - 8u * (nb / 8u + 1u)), bo, lane);
        cn[i] = nf;
        co[i] = nb;
        lane_max = max(lane_max, (int)(nf + nb));
      }
    }
  }
  coincident = __any_sync(0xffffffffu, coincident != 0);
  overflow = __any_sync(0xffffffffu, overflow != 0);
  const int warp_max = __reduce_max_sync(0xffffffffu, lane_max);
  if (lane == 0) {
    if (overflow) flags->overflow = 1;
    if (coincident) flags->nonfinite = 1;
    if (warp_max > 0) atomicMax(&flags->max_row, warp_max);
  }
}

// ---------------------------------------------------------- field get / set ---
__global__ void k_get_f64(int n, int field, int order, const double4* __restrict__ pos4,
                          const double4* __restrict__ vel4, const double4* __restrict__ acc4,
                          const double4* __restrict__ grad4, const double* __restrict__ scalar,
                          const double2* __restrict__ keep2, const uint32_t* __restrict__ oid,
                          double* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v;
  switch (field) {
    case MPS_F_X: v = pos4[i].x; break;
    case MPS_F_Y: v = pos4[i].y; break;
    case MPS_F_Z: v = pos4[i].z; break;
    case MPS_F_U: v = vel4[i].x; break;
    case MPS_F_V: v = vel4[i].y; break;
    case MPS_F_W: v = vel4[i].z; break;
    case MPS_F_AX: v = acc4[i].x; break;
    case MPS_F_AY: v = acc4[i].y; break;
    case MPS_F_AZ: v = acc4[i].z; break;
    case MPS_F_GX: v = grad4[i].x; break;
    case MPS_F_GY: v = grad4[i].y; break;
    case MPS_F_GZ: v = grad4[i].z; break;
    case MPS_F_NK: v = keep2[i].x; break;
    case MPS_F_DNDTK: v = keep2[i].y; break;
    default: v = scalar[i]; break;
  }
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = v;
}
__global__ void k_set_f64(int n, int field, int order, double4* __restrict__ pos4,
                          double4* __restrict__ vel4, double4* __restrict__ acc4,
                          double4* __restrict__ grad4, double* __restrict__ scalar,
                          double2* __restrict__ keep2, const uint32_t* __restrict__ oid,
                          const double* __restrict__ src) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v = src[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i];
  switch (field) {
    case MPS_F_X: pos4[i].x = v; break;
    case MPS_F_Y: pos4[i].y = v; break;
    case MPS_F_Z: pos4[i].z = v; break;
    case MPS_F_U: vel4[i].x = v; break;
    case MPS_F_V: vel4[i].y = v; break;
    case MPS_F_W: vel4[i].z = v; break;
    case MPS_F_AX: acc4[i].x = v; break;
    case MPS_F_AY: acc4[i].y = v; break;
    case MPS_F_AZ: acc4[i].z = v; break;
    case MPS_F_GX: grad4[i].x = v; break;
    case MPS_F_GY: grad4[i].y = v; break;
    case MPS_F_GZ: grad4[i].z = v; break;
    case MPS_F_NK: keep2[i].x = v; break;
    case MPS_F_DNDTK: keep2[i].y = v; break;
    default: scalar[i] = v; break;
  }
}
__global__ void k_get_i32(int n, int field, int order, const uint32_t* __restrict__ tp,
                          const int8_t* __restrict__ bc, const uint32_t* __restrict__ key,
                          const uint32_t* __restrict__ oid, int32_t* __restrict__ dst) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t v;
  switch (field) {
    case MPS_I_TYPE: v = (int32_t)(tp[i] & 0xff); break;
    case MPS_I_PHASE: v = (int32_t)((tp[i] >> 8) & 1); break;
    case MPS_I_BC: v = (int32_t)bc[i]; break;
    default: v = (int32_t)key[i]; break;
  }
  dst[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i] = v;
}
__global__ void k_set_i32(int n, int field, int order, uint32_t* __restrict__ tp, int8_t* __restrict__ bc,
                          const uint32_t* __restrict__ oid, const int32_t* __restrict__ src) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t v = src[order == MPS_ORDER_ORIGINAL ? oid[i] : (uint32_t)i];
  switch (field) {
    case MPS_I_TYPE: tp[i] = (tp[i] & ~0xffu) | (uint32_t)(v & 0xff); break;
    case MPS_I_PHASE: tp[i] = (tp[i] & ~0x100u) | ((uint32_t)(v & 1) << 8); break;
    case MPS_I_BC: bc[i] = (int8_t)v; break;
    default: break;
  }
}

// ------------------------------------------------ neighbour sets for the tests ---
__global__ void k_nb_counts(int n, int radius_id, const uint32_t* __restrict__ cn,
                            const uint32_t* __restrict__ co, const uint32_t* __restrict__ oid,
                            uint32_t* __restrict__ counts) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  counts[oid[i]] = cn[i] + (radius_id == MPS_RADIUS_LAP ? co[i] : 0u);
}
// Skin rows (mps_step): the set a sweep sees is the stored row filtered by the re-test at the current
// positions.  GHOST rows are empty.
__device__ __forceinline__ bool nb_keep(const double4* pos4, int i, uint32_t e, double re2) {
  return r2_exact(pos4[e & NB_INDEX], pos4[i]) < re2;
}
__global__ void k_nb_counts_skin(int n, int cap_row, double re2, int lap, const double4* __restrict__ pos4,
                                 const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
                                 const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co,
                                 const uint32_t* __restrict__ oid, uint32_t* __restrict__ counts) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t* row = nbr + (size_t)i * (size_t)cap_row;
  const uint32_t nf = cn[i], m = nf + (lap ? co[i] : 0u);
  uint32_t k_ = 0;
  if ((tp[i] & 0xff) != MPS_GHOST)
    for (uint32_t k = 0; k < m; ++k) {
      const uint32_t e = (k < nf) ? row[k] : row[back_slot(cap_row, k - nf)];
      if (nb_keep(pos4, i, e, re2)) ++k_;
    }
  counts[oid[i]] = k_;
}
__global__ void k_nb_fill_skin(int n, int cap_row, double re2, int lap, const double4* __restrict__ pos4,
                               const uint32_t* __restrict__ tp, const uint32_t* __restrict__ nbr,
                               const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co,
                               const uint32_t* __restrict__ oid, const uint32_t* __restrict__ offs,
                               uint32_t* __restrict__ idx, int64_t cap) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n || (tp[i] & 0xff) == MPS_GHOST) return;
  const uint32_t* row = nbr + (size_t)i * (size_t)cap_row;
  const uint32_t nf = cn[i], m = nf + (lap ? co[i] : 0u);
  const int64_t base = offs[oid[i]];
  int64_t w = base;
  for (uint32_t k = 0; k < m; ++k) {
    const uint32_t e = (k < nf) ? row[k] : row[back_slot(cap_row, k - nf)];
    if (!nb_keep(pos4, i, e, re2)) continue;
    if (w >= cap) return;  // caller's buffer too small: the row is cut
    const uint32_t v = oid[e & NB_INDEX];
    int64_t t = w++;
    while (t > base && idx[t - 1] > v) { idx[t] = idx[t - 1]; --t; }
    idx[t] = v;
  }
}
__global__ void k_nb_fill(int n, int cap_row, int radius_id, const uint32_t* __restrict__ nbr,
                          const uint32_t* __restrict__ cn, const uint32_t* __restrict__ co,
                          const uint32_t* __restrict__ oid, const uint32_t* __restrict__ offs,
                          uint32_t* __restrict__ idx, int64_t cap) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t* row = nbr + (size_t)i * (size_t)cap_row;
  int64_t base = offs[oid[i]];
  uint32_t nf = cn[i], nb = (radius_id == MPS_RADIUS_LAP) ? co[i] : 0u;
  uint32_t m = nf + nb;
  if (base + m > cap) return;  // caller's buffer too small for this row: skip it
  // insertion sort by original index while writing
  for (uint32_t k = 0; k < m; ++k) {
    uint32_t e = (k < nf) ? row[k] : row[back_slot(cap_row, k - nf)];
    uint32_t v = oid[e & NB_INDEX];
    int64_t t = base + k;
    while (t > base && idx[t - 1] > v) { idx[t] = idx[t - 1]; --t; }
    idx[t] = v;
  }
}

}  // namespace

// ============================================================ host launchers ===
void mpsk_exclusive_scan(mps_ctx* c, int cat, const uint32_t* in, uint32_t* out, int64_t n,
                         uint32_t* tmp, const int* go) {
  int ntiles = div_up(n, SCAN_TILE);
  if (ntiles <= 16) {  // up to 32k entries: one block is faster than three launches
    MPS_LAUNCH(c, cat, k_scan_small, 1, TPB, in, out, n, go);
    return;
  }
  MPS_LAUNCH(c, cat, k_scan_reduce, ntiles, TPB, in, n, tmp, go);
  MPS_LAUNCH(c, cat, k_scan_spine, 1, TPB, tmp, ntiles, go);
  MPS_LAUNCH(c, cat, k_scan_apply, ntiles, TPB, in, out, n, tmp, go);
}

int mpsk_load_particles(mps_ctx* c, const double* x, const double* y, const double* z,
                        const double* u, const double* v, const double* w, const int32_t* type,
                        const int32_t* phase) {
  int n = (int)c->n;
  MPS_LAUNCH(c, MPS_T_BIN_SORT, k_load, div_up(n, TPB), TPB, n, x, y, z, u, v, w, type, phase,
             c->pos4[c->cur], c->vel4[c->cur], c->tp[c->cur], c->oid[c->cur]);
  return MPS_OK;
}

int mpsk_bin(mps_ctx* c, int rows_mode, const int* go) {
  const int n = (int)c->n;
  const KConst& kg = go ? c->kc_step[c->skin_level] : c->kc;
  const int nc = kg.ncells;
  const int cur = c->cur, nxt = cur ^ 1;
  if (go && c->timer_mask != 0) {
    // per-kernel timers are on (bench.py's instrumented replay; launches go out one by one, each between two
    // events): read the flag and leave out a bin that is not needed, as the conditional graph node does
    int up = 1;
    if (cudaMemcpyAsync(&up, go, sizeof(int), cudaMemcpyDeviceToHost, c->stream) == cudaSuccess &&
        cudaStreamSynchronize(c->stream) == cudaSuccess && up == 0) {
      c->ppe_ready = false;
      c->posw_is_p = false;
      return MPS_OK;
    }
  }
  // A skin bin captured into a graph becomes the body of an IF node keyed on the device flag
  cudaStream_t outer = c->stream;
  bool cond = false;
  int64_t launches_before = 0, t_before[MPS_NUM_TIMERS];
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (go && c->cond_nodes && c->aux_stream && c->stream && cudaStreamIsCapturing(c->stream, &cap) == cudaSuccess &&
      cap == cudaStreamCaptureStatusActive) {
    cudaGraph_t graph = nullptr, body = nullptr;
    const cudaGraphNode_t* deps = nullptr;
    size_t ndeps = 0;
    unsigned long long id = 0;
    cudaGraphConditionalHandle handle;
    cudaGraphNode_t node;
    cudaGraphNodeParams np = {};
    bool ok = cudaStreamGetCaptureInfo_v2(outer, &cap, &id, &graph, &deps, &ndeps) == cudaSuccess &&
              cudaGraphConditionalHandleCreate(&handle, graph, 0, cudaGraphCondAssignDefault) == cudaSuccess;
    if (ok) {
      MPS_LAUNCH(c, MPS_T_BIN_SORT, k_set_cond, 1, 1, handle, go, c->flags);
      np.type = cudaGraphNodeTypeConditional;
      np.conditional.handle = handle;
      np.conditional.type = cudaGraphCondTypeIf;
      np.conditional.size = 1;
      ok = cudaStreamGetCaptureInfo_v2(outer, &cap, &id, &graph, &deps, &ndeps) == cudaSuccess &&
           cudaGraphAddNode(&node, graph, deps, ndeps, &np) == cudaSuccess &&
           cudaStreamUpdateCaptureDependencies(outer, &node, 1, cudaStreamSetCaptureDependencies) == cudaSuccess;
      if (ok) {
        body = np.conditional.phGraph_out[0];
        ok = cudaStreamBeginCaptureToGraph(c->aux_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
      }
      if (ok) {
        cond = true;
        c->stream = c->aux_stream;  // the launches below go into the body
        launches_before = c->launches;
        for (int k = 0; k < MPS_NUM_TIMERS; ++k) t_before[k] = c->t_launches[k];
      } else {
        cudaGetLastError();  // the capture is broken: run_segment sees EndCapture fail and falls back to launches
      }
    } else {
      cudaGetLastError();
    }
  }
  const int gwords = n / 32 + 1;
  cudaMemsetAsync(c->cell_count, 0, sizeof(uint32_t) * (nc + 2), c->stream);
  cudaMemsetAsync(c->gbit, 0, sizeof(uint32_t) * gwords, c->stream);
  if (!go) cudaMemsetAsync(&c->flags->max_row, 0, sizeof(int), c->stream);  // predicated: k_scatter does it
  MPS_LAUNCH(c, MPS_T_BIN_SORT, k_keys, div_up(n, TPB), TPB, kg, c->pos4[cur], c->tp[cur],
             c->key_tmp, c->rank, c->cell_count, c->flags, c->oid[cur], c->gbit, go);
  mpsk_exclusive_scan(c, MPS_T_BIN_SORT, c->cell_count, c->cell_start, nc + 2, c->scan_tmp, go);
  MPS_LAUNCH(c, MPS_T_BIN_SORT, k_ghost_popc, div_up(gwords, TPB), TPB, gwords, c->gbit, c->gcnt, go);
  mpsk_exclusive_scan(c, MPS_T_BIN_SORT, c->gcnt, c->gpre, gwords, c->scan_tmp, go);
  MPS_LAUNCH(c, MPS_T_BIN_SORT, k_scatter, div_up(n, TPB), TPB, n, c->key_tmp, c->rank,
             c->cell_start, c->oid[cur], c->tmp_src, c->tmp_oid, c->key, nc, c->flags, go);
  const bool keep = c->prm.ppe_source == 2, rs = c->prm.grad_variant == 3;
  MPS_LAUNCH(c, MPS_T_BIN_SORT, k_reorder, div_up(n, TPB), TPB, n, nc, c->key, c->cell_start,
             c->tmp_src, c->tmp_oid, c->pos4[cur], c->vel4[cur], c->tp[cur], c->pos4[nxt],
             c->vel4[nxt], c->tp[nxt], c->oid[nxt], c->ent,
             keep ? c->keep2[cur] : nullptr, c->keep2[nxt],
             rs ? c->rho_s[cur] : nullptr, c->rho_s[nxt], go ? 1 : c->prm.cg_warm_start, c->gbit, c->gpre, go);
  int at = nxt;
  if (go) {
    // back into the current buffers (the host cannot know whether this bin ran) + the build positions
    MPS_LAUNCH(c, MPS_T_BIN_SORT, k_commit, div_up(n, TPB), TPB, n, c->pos4[nxt], c->vel4[nxt], c->tp[nxt],
               c->oid[nxt], c->keep2[nxt], c->rho_s[nxt], c->pos4[cur], c->vel4[cur], c->tp[cur], c->oid[cur],
               keep ? c->keep2[cur] : nullptr, rs ? c->rho_s[cur] : nullptr, c->pos_ref, go);
    at = cur;
  } else {
    c->cur = nxt;
    c->kc.pos_tex = c->cg_tex ? c->pos_tex[nxt] : 0;
    c->kc.vel_tex = c->cg_tex ? c->vel_tex[nxt] : 0;
    c->carry_valid = false;
  }
  if (c->rows_builder == 0) {
    MPS_LAUNCH(c, MPS_T_BIN_LIST, k_build_rows, div_up(n, (LEAN_TPB / 32) * LEAN_PPW), LEAN_TPB, kg, c->pos4[at],
               c->ent, c->key, c->cell_start, c->nbr, c->cn, c->co, c->flags, rows_mode, go);
  } else if (c->prm.cell_div == 1 && c->rows_builder == 2) {
    if (go)
      MPS_LAUNCH(c, MPS_T_BIN_LIST, k_build_rows_cell<false>, div_up(nc, CELL_WARPS), CELL_TPB, kg, c->pos4[at],
                 c->ent, c->cell_start, c->nbr, c->cn, c->co, c->flags, rows_mode, go);
    else
      MPS_LAUNCH(c, MPS_T_BIN_LIST, k_build_rows_cell<true>, div_up(nc, CELL_WARPS), CELL_TPB, kg, c->pos4[at],
                 c->ent, c->cell_start, c->nbr, c->cn, c->co, c->flags, rows_mode, go);
  } else {
    // small cells hold only a few particles each: one warp per particle, lanes on candidates
    MPS_LAUNCH(c, MPS_T_BIN_LIST, k_build_rows_warp, div_up(n, (ROWS_TPB / 32) * ROWS_PPW), ROWS_TPB, kg,
               c->pos4[at], c->tp[at], c->ent, c->key, c->cell_start, c->nbr, c->cn, c->co, c->flags, rows_mode, go);
  }
  if (cond) {
    cudaGraph_t body_out = nullptr;
    cudaStreamEndCapture(c->aux_stream, &body_out);
    c->stream = outer;
    // the body's launches happen only when the bin runs: mps_launch_count adds them from the device counter
    c->cond_launches_per_bin = (int)(c->launches - launches_before);
    c->launches = launches_before;
    for (int k = 0; k < MPS_NUM_TIMERS; ++k) c->t_launches[k] = t_before[k];
  }
  if (!go) {
    c->binned = true;
    c->bins_run++;
  }
  c->ppe_ready = false;
  c->posw_is_p = false;
  return MPS_OK;
}

static const double* scalar_field(mps_ctx* c, int field) {
  switch (field) {
    case MPS_F_N: return c->dens;
    case MPS_F_P: return c->p;
    case MPS_F_NUT: return c->nut;
    case MPS_F_B: return c->b;
    case MPS_F_PHAT: return c->phat;
    case MPS_F_XCG: return c->cg_x;
    case MPS_F_DNDT: return c->dndt;
    case MPS_F_RHOS: return c->rho_s[c->cur];
  }
  return nullptr;
}

int mpsk_get_field(mps_ctx* c, int field, void* dst, int order) {
  int n = (int)c->n;
  int cur = c->cur;
  if (field >= 0 && field <= MPS_F_RHOS) {
    MPS_LAUNCH(c, MPS_T_BIN_SORT, k_get_f64, div_up(n, TPB), TPB, n, field, order, c->pos4[cur],
               c->vel4[cur], c->acc4, c->grad4, scalar_field(c, field), c->keep2[cur], c->oid[cur],
               (double*)dst);
    return MPS_OK;
  }
  if (field >= MPS_I_TYPE && field <= MPS_I_KEY) {
    MPS_LAUNCH(c, MPS_T_BIN_SORT, k_get_i32, div_up(n, TPB), TPB, n, field, order, c->tp[cur], c->bc,
               c->key, c->oid[cur], (int32_t*)dst);
    return MPS_OK;
  }
  return MPS_ERR_ARG;
}

int mpsk_set_field(mps_ctx* c, int field, const void* src, int order) {
  int n = (int)c->n;
  int cur = c->cur;
  if (field >= 0 && field <= MPS_F_RHOS) {
    if (field == MPS_F_RHOS) c->rho_s_ready = true;
    MPS_LAUNCH(c, MPS_T_BIN_SORT, k_set_f64, div_up(n, TPB), TPB, n, field, order, c->pos4[cur],
               c->vel4[cur], c->acc4, c->grad4, (double*)scalar_field(c, field), c->keep2[cur],
               c->oid[cur], (const double*)src);
    if (field <= MPS_F_Z) { c->binned = false; c->ppe_ready = false; }
    if (field == MPS_F_P) c->posw_is_p = false;
    return MPS_OK;
  }
  if (field >= MPS_I_TYPE && field <= MPS_I_BC) {
    MPS_LAUNCH(c, MPS_T_BIN_SORT, k_set_i32, div_up(n, TPB), TPB, n, field, order, c->tp[cur], c->bc,
               c->oid[cur], (const int32_t*)src);
    if (field != MPS_I_BC) { c->binned = false; c->ppe_ready = false; }
    return MPS_OK;
  }
  return MPS_ERR_ARG;
}

int mpsk_get_neighbours(mps_ctx* c, int radius_id, uint32_t* counts, uint32_t* idx, int64_t cap,
                        int64_t* total) {
  int n = (int)c->n;
  int cur = c->cur;
  const bool skin = !c->binned;  // the caller has checked that the skin rows are valid
  const double re2 = radius_id == MPS_RADIUS_LAP ? c->kc.re_lap2 : c->kc.re_n2;
  const int lap = radius_id == MPS_RADIUS_LAP;
  if (skin)
    MPS_LAUNCH(c, MPS_T_BIN_LIST, k_nb_counts_skin, div_up(n, TPB), TPB, n, c->kc.stride, re2, lap, c->pos4[cur],
               c->tp[cur], c->nbr, c->cn, c->co, c->oid[cur], counts);
  else
  MPS_LAUNCH(c, MPS_T_BIN_LIST, k_nb_counts, div_up(n, TPB), TPB, n, radius_id, c->cn, c->co,
             c->oid[cur], counts);
  // offsets in original order: scan into tmp_src (n entries; free between bins)
  mpsk_exclusive_scan(c, MPS_T_BIN_LIST, counts, c->tmp_src, n, c->scan_tmp);
  uint32_t last_off = 0, last_cnt = 0;
  cudaMemcpyAsync(&last_off, c->tmp_src + (n - 1), 4, cudaMemcpyDeviceToHost, c->stream);
  cudaMemcpyAsync(&last_cnt, counts + (n - 1), 4, cudaMemcpyDeviceToHost, c->stream);
  cudaStreamSynchronize(c->stream);
  if (total) *total = (int64_t)last_off + last_cnt;
  if (idx && skin) {
    MPS_LAUNCH(c, MPS_T_BIN_LIST, k_nb_fill_skin, div_up(n, TPB), TPB, n, c->kc.stride, re2, lap, c->pos4[cur],
               c->tp[cur], c->nbr, c->cn, c->co, c->oid[cur], c->tmp_src, idx, cap);
  } else if (idx) {
    MPS_LAUNCH(c, MPS_T_BIN_LIST, k_nb_fill, div_up(n, TPB), TPB, n, c->kc.stride, radius_id, c->nbr,
               c->cn, c->co, c->oid[cur], c->tmp_src, idx, cap);
  }
  return MPS_OK;
}
