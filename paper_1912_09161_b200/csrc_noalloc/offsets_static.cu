// allen_velo_offsets_noalloc (include/allen_velo_noalloc.h): the output-compaction scan of the path (A9 of SURVEY.md
// §8(a)) for callers that cannot allocate.  Same method as scan_kernel of csrc/velo_scan.cu — single-pass
// exclusive prefix sum, tiles claimed by an atomic ticket, aggregates / inclusive prefixes published through one 64-bit
// status word per tile, decoupled look-back by the first warp — but the scratch words are a file-scope static device
// array of this file instead of a slice of the caller's workspace, and there is no handle.  Nothing here is called by
// allen_velo_reconstruct; this file shares no code with the rest of the library.
//
// The array's name is a device symbol: in HOST code it is a stand-in, not a device address.  The host gets the address
// once per device with cudaGetSymbolAddress (with that device current) and passes it to cudaMemsetAsync and the kernel.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/allen_velo_noalloc.h"

namespace {

constexpr uint32_t kThreads = 256, kItems = 8, kTile = kThreads * kItems;  // 2048 counts per CTA
constexpr uint32_t kMaxTiles = ALLEN_VELO_NOALLOC_MAX_COUNTS / kTile;      // 2048
constexpr uint32_t kStateWords = 1 + kMaxTiles;                            // [0] ticket, [1 + t] status of tile t
static_assert(ALLEN_VELO_NOALLOC_MAX_COUNTS % kTile == 0, "whole tiles");

// 16 392 bytes on every GPU that loads the library, until the process exits.  Shared by all calls on the device.
static __device__ __align__(256) unsigned long long g_offsets_state[kStateWords];

constexpr unsigned long long kAggregate = 1ull << 62, kInclusive = 2ull << 62, kValue = (1ull << 62) - 1;
constexpr unsigned kAll = 0xFFFFFFFFu;

__device__ __forceinline__ unsigned long long load_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void store_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__global__ void __launch_bounds__(kThreads) offsets_static_kernel(const uint32_t* __restrict__ counts,
                                                                   uint32_t* __restrict__ offsets, uint32_t n,
                                                                   unsigned long long* state) {
  __shared__ unsigned long long warp_total[kThreads / 32];
  __shared__ unsigned long long before_tile;
  __shared__ uint32_t my_tile;
  // a ticket, not blockIdx: every tile before a running tile is then running or done, whatever the block schedule
  if (threadIdx.x == 0) my_tile = (uint32_t)atomicAdd(state, 1ull);
  __syncthreads();
  const uint32_t tile = my_tile, lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  unsigned long long* status = state + 1;
  const uint32_t first = tile * kTile + threadIdx.x * kItems;

  unsigned long long c[kItems], mine = 0;
#pragma unroll
  for (uint32_t k = 0; k < kItems; ++k) {
    c[k] = first + k < n ? (unsigned long long)counts[first + k] : 0ull;
    mine += c[k];
  }
  unsigned long long incl = mine;  // inclusive scan of the threads' sums inside the warp
#pragma unroll
  for (uint32_t d = 1; d < 32; d <<= 1) {
    const unsigned long long up = __shfl_up_sync(kAll, incl, d);
    if (lane >= d) incl += up;
  }
  if (lane == 31) warp_total[warp] = incl;
  __syncthreads();
  unsigned long long before_warp = 0, tile_total = 0;
#pragma unroll
  for (uint32_t w = 0; w < kThreads / 32; ++w) {
    if (w < warp) before_warp += warp_total[w];
    tile_total += warp_total[w];
  }

  if (warp == 0) {
    if (lane == 0) store_status(status + tile, (tile == 0 ? kInclusive : kAggregate) | tile_total);
    unsigned long long sum = 0;
    if (tile > 0) {
      // look back 32 tiles at a time until one of them has published its inclusive prefix
      for (int newest = (int)tile - 1;; newest -= 32) {
        const int t = newest - (int)lane;
        unsigned long long s = kInclusive;  // "tile -1": inclusive prefix 0
        if (t >= 0) {
          do { s = load_status(status + t); } while ((s >> 62) == 0);
        }
        const uint32_t has_prefix = __ballot_sync(kAll, (s >> 62) == 2);
        const int stop = has_prefix ? __ffs(has_prefix) - 1 : 32;  // nearest tile with an inclusive prefix
        unsigned long long part = (int)lane <= stop ? (s & kValue) : 0ull;
#pragma unroll
        for (uint32_t d = 16; d; d >>= 1) part += __shfl_xor_sync(kAll, part, d);
        sum += part;
        if (has_prefix) break;
      }
      if (lane == 0) store_status(status + tile, kInclusive | (sum + tile_total));
    }
    if (lane == 0) before_tile = sum;
  }
  __syncthreads();
  unsigned long long run = before_tile + before_warp + (incl - mine);
#pragma unroll
  for (uint32_t k = 0; k < kItems; ++k) {
    const uint32_t i = first + k;
    if (i < n) offsets[i] = (uint32_t)run;
    run += c[k];
    if (i + 1 == n) offsets[n] = (uint32_t)run;
  }
}

// Device address of the array, per device: looked up once, with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_lock;
unsigned long long* g_state_address[kMaxDevices] = {};

int fail(char* text, size_t bytes, int code, const char* what, cudaError_t err) {
  if (text && bytes) {
    if (err != cudaSuccess) snprintf(text, bytes, "allen_velo_offsets_noalloc: %s failed: %s", what, cudaGetErrorString(err));
    else snprintf(text, bytes, "allen_velo_offsets_noalloc: %s", what);
  }
  return code;
}

}  // namespace

extern "C" int allen_velo_offsets_noalloc(const uint32_t* counts, uint32_t n, uint32_t* offsets, void* cuda_stream,
                                          char* error_text, size_t error_text_bytes) {
  if (error_text && error_text_bytes) error_text[0] = 0;
  if (!offsets || (n > 0 && !counts))
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_INVALID, "null pointer (counts with n > 0, or offsets)", cudaSuccess);
  if (n > ALLEN_VELO_NOALLOC_MAX_COUNTS) {
    char msg[160];
    snprintf(msg, sizeof msg, "n = %u exceeds ALLEN_VELO_NOALLOC_MAX_COUNTS = %u (the static scratch array holds one "
             "status word per %u counts); nothing was enqueued", n, ALLEN_VELO_NOALLOC_MAX_COUNTS, kTile);
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_TOO_LARGE, msg, cudaSuccess);
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t err;
  if (n == 0) {  // offsets[0] = 0; no scratch needed
    err = cudaMemsetAsync(offsets, 0, sizeof(uint32_t), stream);
    return err == cudaSuccess ? ALLEN_VELO_OK : fail(error_text, error_text_bytes, ALLEN_VELO_ERR_CUDA, "cudaMemsetAsync(offsets)", err);
  }
  int device = -1;
  if ((err = cudaGetDevice(&device)) != cudaSuccess)
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_CUDA, "cudaGetDevice", err);
  if (device < 0 || device >= kMaxDevices)
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_INVALID, "device ordinal beyond 63", cudaSuccess);
  unsigned long long* state = nullptr;
  {
    std::lock_guard<std::mutex> guard(g_lock);
    if (!g_state_address[device]) {
      void* address = nullptr;
      if ((err = cudaGetSymbolAddress(&address, g_offsets_state)) != cudaSuccess || !address)
        return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_CUDA, "cudaGetSymbolAddress(g_offsets_state)", err);
      g_state_address[device] = static_cast<unsigned long long*>(address);
    }
    state = g_state_address[device];
  }
  const uint32_t tiles = (n + kTile - 1) / kTile;
  // the array keeps the last call's contents: the ticket and the status words of this call's tiles start at zero
  if ((err = cudaMemsetAsync(state, 0, (1 + (size_t)tiles) * sizeof(unsigned long long), stream)) != cudaSuccess)
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_CUDA, "cudaMemsetAsync(scratch)", err);
  offsets_static_kernel<<<tiles, kThreads, 0, stream>>>(counts, offsets, n, state);
  if ((err = cudaGetLastError()) != cudaSuccess)
    return fail(error_text, error_text_bytes, ALLEN_VELO_ERR_CUDA, "kernel launch", err);
  return ALLEN_VELO_OK;
}
