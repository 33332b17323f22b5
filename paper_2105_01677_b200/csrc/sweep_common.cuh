// sweep_common.cuh -- device helpers shared by the list-driven sweeps.
// Not part of the ABI.  Shares nothing with oracle/.
#pragma once
#include "mps_internal.h"

// ---- neighbour rows (row-major ELL, see mps_internal.h) ---------------------------
__device__ __forceinline__ const uint32_t* row_ptr(const uint32_t* nbr, int stride, int i) {
  return nbr + (size_t)i * (size_t)stride;
}
// Entry k of a row with nf front entries: the re_n part grows from the front,
// the re_n <= r < re_lap part from the back in whole 32-byte sectors (8 entries),
// ascending inside each sector: back entry kk sits at stride - 8 (kk/8 + 1) + kk % 8.
__device__ __forceinline__ uint32_t row_entry(const uint32_t* row, int stride, uint32_t nf, uint32_t k) {
  return k < nf ? row[k] : row[back_slot(stride, k - nf)];
}

// ---- 1/sqrt(x) in fp64: hardware seed (about 2^-22) plus one cubically convergent
// correction y (1 + e/2 + 3e^2/8), e = 1 - x y^2: five fp64 operations, error a
// few 1e-16 relative.  x must be positive, finite and normal (r^2 of two distinct
// particles).  No bit-exact quantity depends on it (reading Q2).
__device__ __forceinline__ double rsqrt_f64(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = x * y;
  double e = fma(-t, y, 1.0);
  double q = fma(e, 0.375, 0.5);
  double c = q * e;
  return fma(y, c, y);
}

// ---- kernel function w(r), 0 <= r < re, from r^2 and ir = 1/r: Eq. 3 re/r - 1, or
// Eq. 4 (1 - r/re)^3 when kernel == 1 (a warp-uniform switch).
__device__ __forceinline__ double kernel_w(int kernel, double re, double inv_re, double r2, double ir) {
  if (kernel == 1) {
    const double t = fma(-(r2 * ir), inv_re, 1.0);
    return t * t * t;
  }
  return fma(re, ir, -1.0);
}

// ---- squared distance of a pair: fused arithmetic, or -- while rows are reused (Q24) -- the
// rounding of reading Q2, so that the re-test r2 < re^2 decides exactly as the oracle's does.
__device__ __forceinline__ double pair_r2(double dx, double dy, double dz, int stale) {
  if (stale) return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return dx * dx + dy * dy + dz * dz;
}

// ---- neighbour record gathers ------------------------------------------------------
// A sweep is bound by the rate at which the LSU serves one 32-byte record per lane per pair
// (profiles/r01_ceilings_microbench.md).  When the texture view exists, the first 16 bytes come
// through the texture front end and the second 16 through the LSU: the two work in parallel
// (measured 1.2x).  Only data that no thread writes during the kernel may take the texture path.
__device__ __forceinline__ double4 gather_rec(cudaTextureObject_t tex, const double4* __restrict__ a, uint32_t j) {
  if (tex) {
    const int4 lo = tex1Dfetch<int4>(tex, 2 * (int)j);
    const double2 hi = reinterpret_cast<const double2*>(a + j)[1];
    return make_double4(__hiloint2double(lo.y, lo.x), __hiloint2double(lo.w, lo.z), hi.x, hi.y);
  }
  return a[j];
}

// ---- reductions over the L lanes that share a row (L a power of two <= 32) -----------
template <int L>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
  for (int o = L / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
template <int L>
__device__ __forceinline__ double group_min(double v) {
#pragma unroll
  for (int o = L / 2; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
template <int L>
__device__ __forceinline__ double group_max(double v) {
#pragma unroll
  for (int o = L / 2; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_sum(double v) { return group_sum<32>(v); }
