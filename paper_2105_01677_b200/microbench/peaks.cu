// peaks.cu -- stand-alone micro-benchmarks of the two on-chip ceilings the MPS sweeps meet
// on B200: the fp64 pipe, and the L1 serving one 32-byte particle
// record per lane per neighbour pair.  Not part of libmps_b200.so; built by
//   python -m paper_2105_01677_b200.build --peaks     ->  paper_2105_01677_b200/mps_peaks
// and run as  paper_2105_01677_b200/mps_peaks  (prints one line per measurement).
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <cstdlib>
#include <vector>

#define CK(x)                                                        \
  do {                                                               \
    cudaError_t e_ = (x);                                            \
    if (e_ != cudaSuccess) {                                         \
      printf("%s: %s\n", #x, cudaGetErrorString(e_));                \
      return 1;                                                      \
    }                                                                \
  } while (0)

// ---- fp64 pipe: 8 independent register-resident chains per thread ---------------------
template <int MODE>
__global__ void __launch_bounds__(512) k_fp64(double* out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) x[k] = threadIdx.x * 1e-3 + k;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (MODE == 0) x[k] = fma(x[k], a, b);
      if (MODE == 1) x[k] = (k & 1) ? __dmul_rn(x[k], a) : __dadd_rn(x[k], b);
      if (MODE == 2) asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(x[k]));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- list-driven sweep: rows of NE neighbour indices, L lanes per row, one double4 gather
// and the PPE pair arithmetic per entry (the shape of k_ppe_cg's phase A) -----------------
__device__ __forceinline__ double rsqrt_f64(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = x * y, e = fma(-t, y, 1.0), q = fma(e, 0.375, 0.5);
  return fma(y, q * e, y);
}
// SPLIT: first 16 bytes of the record through the texture unit, second 16 through the LSU
template <int L, bool MATH, bool SPLIT>
__global__ void __launch_bounds__(1024)
k_gather(const double4* __restrict__ pos, cudaTextureObject_t tex, const uint32_t* __restrict__ list,
         int NE, int nrows, double* __restrict__ y) {
  const int sub = threadIdx.x & (L - 1);
  const int gstride = gridDim.x * blockDim.x / L;
  for (int r = (blockIdx.x * blockDim.x + threadIdx.x) / L; r < nrows; r += gstride) {
    const uint32_t* row = list + (size_t)r * NE;
    const double4 pi = pos[r];
    double s = 0.0;
#pragma unroll 4
    for (int k = sub; k < NE; k += L) {
      double4 q;
      if (SPLIT) {
        const uint32_t j = row[k];
        const int4 lo = tex1Dfetch<int4>(tex, 2 * (int)j);
        const double2 hi = reinterpret_cast<const double2*>(pos + j)[1];
        q = make_double4(__hiloint2double(lo.y, lo.x), __hiloint2double(lo.w, lo.z), hi.x, hi.y);
      } else {
        q = pos[row[k]];
      }
      if (MATH) {
        const double dx = q.x - pi.x, dy = q.y - pi.y, dz = q.z - pi.z;
        const double r2 = dx * dx + dy * dy + dz * dz;
        s = fma(fma(3.1, rsqrt_f64(r2), -1.0), pi.w - q.w, s);
      } else {
        s += (q.x + q.y) + (q.z + q.w);
      }
    }
    for (int o = L / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (sub == 0) y[r] = s;
  }
}

int main() {
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, 0));
  const int sms = prop.multiProcessorCount;
  const double ghz = prop.clockRate * 1e-6;
  printf("device %s, %d SMs, max clock %.3f GHz\n", prop.name, sms, ghz);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float ms;
  {
    double* out;
    CK(cudaMalloc(&out, (size_t)sms * 4 * 512 * 8));
    const int iters = 20000;
    auto run = [&](auto kern, const char* name) {
      kern<<<sms * 4, 512>>>(out, 100, 1.0000001, 1e-9);
      cudaDeviceSynchronize();
      cudaEventRecord(e0);
      kern<<<sms * 4, 512>>>(out, iters, 1.0000001, 1e-9);
      cudaEventRecord(e1);
      cudaDeviceSynchronize();
      cudaEventElapsedTime(&ms, e0, e1);
      const double ops = (double)sms * 4 * 512 * 8.0 * iters;
      printf("fp64 %-18s %.3e thread-instructions/s = %.1f per SM per clock\n", name, ops / (ms * 1e-3),
             ops / (ms * 1e-3) / sms / (ghz * 1e9));
    };
    run(k_fp64<0>, "DFMA");
    run(k_fp64<1>, "DADD/DMUL");
    run(k_fp64<2>, "rsqrt.approx.f64");
    cudaFree(out);
  }
  {
    // rows shaped like an MPS neighbour row in cell-sorted order: 9 runs of ~90 consecutive
    // slots (x-runs of three cells), ~14 hits per run, ascending; adjacent rows nearly agree
    const int N = 1 << 19, NE = 128;
    std::vector<double4> hp(N);
    for (int i = 0; i < N; ++i) hp[i] = make_double4(drand48(), drand48(), drand48() + 2.0, drand48());
    std::vector<uint32_t> hl((size_t)N * NE);
    for (int r = 0; r < N; ++r) {
      int k = 0;
      for (int run = 0; run < 9; ++run) {
        const long base = (long)r - 45 + (run - 4) * 6000L;
        for (int t = 0; t < 14 && k < NE; ++t) {
          long j = base + t * 6 + (lrand48() % 6);
          j = ((j % N) + N) % N;
          hl[(size_t)r * NE + k++] = (uint32_t)j;
        }
      }
      const int filled = k;
      while (k < NE) { hl[(size_t)r * NE + k] = hl[(size_t)r * NE + (k % filled)]; ++k; }
    }
    double4* dp;
    uint32_t* dl;
    double* dy;
    CK(cudaMalloc(&dp, (size_t)N * 32));
    CK(cudaMalloc(&dl, hl.size() * 4));
    CK(cudaMalloc(&dy, (size_t)N * 8));
    CK(cudaMemcpy(dp, hp.data(), (size_t)N * 32, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(dl, hl.data(), hl.size() * 4, cudaMemcpyHostToDevice));
    cudaResourceDesc rd = {};
    rd.resType = cudaResourceTypeLinear;
    rd.res.linear.devPtr = dp;
    rd.res.linear.desc = cudaCreateChannelDesc<int4>();
    rd.res.linear.sizeInBytes = (size_t)N * 32;
    cudaTextureDesc td = {};
    td.readMode = cudaReadModeElementType;
    cudaTextureObject_t tex;
    CK(cudaCreateTextureObject(&tex, &rd, &td, nullptr));
    auto run = [&](auto kern, const char* name) {
      kern<<<sms, 1024>>>(dp, tex, dl, NE, N, dy);
      cudaDeviceSynchronize();
      cudaEventRecord(e0);
      for (int r = 0; r < 5; ++r) kern<<<sms, 1024>>>(dp, tex, dl, NE, N, dy);
      cudaEventRecord(e1);
      cudaDeviceSynchronize();
      cudaEventElapsedTime(&ms, e0, e1);
      ms /= 5;
      printf("gather %-28s %6.0f ps per row of %d pairs = %.1f SM-cycles per 32 pairs; list + row bytes at %.0f GB/s\n",
             name, ms * 1e9 / N, NE, ms * 1e-3 * ghz * 1e9 * sms / ((double)N * NE) * 32,
             (double)N * (NE * 4 + 41) / (ms * 1e-3) / 1e9);
    };
    run(k_gather<8, true, false>, "L=8, pair arithmetic");
    run(k_gather<8, false, false>, "L=8, loads only");
    run(k_gather<16, true, false>, "L=16, pair arithmetic");
    run(k_gather<32, true, false>, "L=32, pair arithmetic");
    run(k_gather<8, true, true>, "L=8, TEX+LSU split, arith.");
    run(k_gather<8, false, true>, "L=8, TEX+LSU split, loads");
  }
  return 0;
}
