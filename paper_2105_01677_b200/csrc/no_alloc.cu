// no_alloc.cu -- mps_cell_start_noalloc: the cell-start table of the counting sort (S2 of DESIGN.md; P:252
// section 4.1) for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses
// that forbid cudaMalloc.  The same result as mps_bin's table (mps_get_cell_start), from the caller's keys, with
// the histogram and the scan's tile sums in a file-scope device array instead of ctx buffers.
//
// The array is one per device and process: every call shares it and it keeps the last call's contents.  Each
// call clears the part it uses (on the caller's stream) before it counts.  Calls that overlap on the GPU (two
// streams, two host threads) race on it: serialise them.  Nothing here calls cudaMalloc, cudaFree or a library
// routine that allocates; the kernels are this file's own (no existing code path is touched).
#include <mutex>
#include <string>

#include "mps_internal.h"

namespace {

constexpr int NA_TPB = 256;
constexpr int NA_ITEMS = 8;
constexpr int NA_TILE = NA_TPB * NA_ITEMS;                 // entries one block scans
constexpr int NA_MAX_CELLS = 1 << 18;                      // 262,144 cells: the 2M-particle scene has 216k
constexpr int NA_COUNTS = NA_MAX_CELLS + 64;               // n_cells + 1 counters (the ghost cell is the last), padded
constexpr int NA_MAX_TILES = NA_COUNTS / NA_TILE + 1;
constexpr int NA_WORDS = NA_COUNTS + NA_MAX_TILES + 63;

// 1.0 MB per GPU that loads the library, held until the process exits: [0, NA_COUNTS) counters, then tile sums
static __device__ __align__(256) uint32_t g_na_scratch[NA_WORDS];

// In host code g_na_scratch is only a stand-in for the symbol, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current.
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
uint32_t* g_na_ptr[NA_MAX_DEVICES] = {nullptr};
std::string g_na_error;

int na_fail(int code, const std::string& msg) {
  std::lock_guard<std::mutex> lock(g_na_mutex);
  g_na_error = msg;
  return code;
}

// keys above n_cells count as ghosts (n_cells), as mps_bin's out-of-domain particles do
__global__ void k_na_hist(int64_t n, uint32_t ncells, const uint32_t* __restrict__ key, uint32_t* __restrict__ counts) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  uint32_t k = 0xffffffffu;
  if (i < n) k = min(key[i], ncells);
  // one atomic per distinct key of the warp
  const unsigned peers = __match_any_sync(0xffffffffu, k);
  const int lane = threadIdx.x & 31;
  if (i < n && lane == __ffs(peers) - 1) atomicAdd(&counts[k], (uint32_t)__popc(peers));
}

__device__ __forceinline__ uint32_t na_block_scan(uint32_t v, uint32_t* total) {
  __shared__ uint32_t ws[NA_TPB / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) ws[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t s = lane < NA_TPB / 32 ? ws[lane] : 0;
#pragma unroll
    for (int o = 1; o < NA_TPB / 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += t;
    }
    if (lane < NA_TPB / 32) ws[lane] = s;
  }
  __syncthreads();
  const uint32_t off = wid ? ws[wid - 1] : 0;
  *total = ws[NA_TPB / 32 - 1];
  __syncthreads();
  return off + inc - v;
}

__global__ void __launch_bounds__(NA_TPB) k_na_tile_sums(int m, const uint32_t* __restrict__ counts, uint32_t* __restrict__ tiles) {
  const int base = blockIdx.x * NA_TILE;
  uint32_t s = 0;
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k) {
    const int i = base + k * NA_TPB + threadIdx.x;
    if (i < m) s += counts[i];
  }
  uint32_t tot;
  na_block_scan(s, &tot);
  if (threadIdx.x == 0) tiles[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(NA_TPB) k_na_spine(int ntiles, uint32_t* __restrict__ tiles) {
  uint32_t carry = 0;
  for (int base = 0; base < ntiles; base += NA_TPB) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < ntiles ? tiles[i] : 0;
    uint32_t tot;
    const uint32_t ex = na_block_scan(v, &tot);
    if (i < ntiles) tiles[i] = carry + ex;
    carry += tot;
  }
}
__global__ void __launch_bounds__(NA_TPB) k_na_apply(int m, const uint32_t* __restrict__ counts, const uint32_t* __restrict__ tiles,
                                                     uint32_t* __restrict__ out) {
  const int base = blockIdx.x * NA_TILE + threadIdx.x * NA_ITEMS;
  uint32_t v[NA_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k) {
    v[k] = base + k < m ? counts[base + k] : 0;
    s += v[k];
  }
  uint32_t tot;
  uint32_t ex = na_block_scan(s, &tot) + tiles[blockIdx.x];
#pragma unroll
  for (int k = 0; k < NA_ITEMS; ++k) {
    if (base + k < m) out[base + k] = ex;
    ex += v[k];
  }
}

}  // namespace

extern "C" {

int32_t mps_cell_start_noalloc_max_cells(void) { return NA_MAX_CELLS; }

const char* mps_cell_start_noalloc_error(void) {
  std::lock_guard<std::mutex> lock(g_na_mutex);
  return g_na_error.c_str();
}

int mps_cell_start_noalloc(const uint32_t* key, int64_t n, int32_t n_cells, uint32_t* cell_start, void* stream) {
  if (!key && n > 0) return na_fail(MPS_ERR_ARG, "mps_cell_start_noalloc: key is NULL");
  if (!cell_start) return na_fail(MPS_ERR_ARG, "mps_cell_start_noalloc: cell_start is NULL");
  if (n < 0 || n >= ((int64_t)1 << 32)) return na_fail(MPS_ERR_ARG, "mps_cell_start_noalloc: n must be in [0, 2^32)");
  if (n_cells < 1) return na_fail(MPS_ERR_ARG, "mps_cell_start_noalloc: n_cells must be at least 1");
  if (n_cells > NA_MAX_CELLS)
    return na_fail(MPS_ERR_ARG, "mps_cell_start_noalloc: n_cells = " + std::to_string(n_cells) + " exceeds the fixed scratch of " +
                                    std::to_string(NA_MAX_CELLS) + " cells (use mps_bin / mps_get_cell_start, which allocate at mps_init)");
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES)
    return na_fail(MPS_ERR_CUDA, std::string("mps_cell_start_noalloc: no usable current device: ") + cudaGetErrorString(e));
  uint32_t* scratch = nullptr;
  {
    // set-up, once per device, with that device current: the device address of the file-scope array
    std::lock_guard<std::mutex> lock(g_na_mutex);
    if (!g_na_ptr[dev]) {
      uint32_t* p = nullptr;
      e = cudaGetSymbolAddress((void**)&p, g_na_scratch);
      if (e != cudaSuccess || !p) {
        g_na_error = std::string("mps_cell_start_noalloc: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e);
        return MPS_ERR_CUDA;
      }
      g_na_ptr[dev] = p;
    }
    scratch = g_na_ptr[dev];
  }
  cudaStream_t s = (cudaStream_t)stream;
  const int m = n_cells + 1;  // counters 0 .. n_cells (ghosts), cell_start has as many entries
  const int ntiles = (m + NA_TILE - 1) / NA_TILE;
  uint32_t* counts = scratch;
  uint32_t* tiles = scratch + NA_COUNTS;
  // the array keeps the last call's counts: clear the part this call uses
  e = cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)m, s);
  if (e != cudaSuccess) return na_fail(MPS_ERR_CUDA, std::string("mps_cell_start_noalloc: ") + cudaGetErrorString(e));
  if (n > 0) k_na_hist<<<(unsigned)((n + NA_TPB - 1) / NA_TPB), NA_TPB, 0, s>>>(n, (uint32_t)n_cells, key, counts);
  k_na_tile_sums<<<ntiles, NA_TPB, 0, s>>>(m, counts, tiles);
  k_na_spine<<<1, NA_TPB, 0, s>>>(ntiles, tiles);
  k_na_apply<<<ntiles, NA_TPB, 0, s>>>(m, counts, tiles, cell_start);
  e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(MPS_ERR_CUDA, std::string("mps_cell_start_noalloc: launch failed: ") + cudaGetErrorString(e));
  return MPS_OK;
}

}  // extern "C"
