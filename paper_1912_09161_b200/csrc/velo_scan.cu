// Prefix-sum output compaction of the tracks (A9 of SURVEY.md §8(a); only quantities that size later work ever
// need to leave the device — here nothing does, the offsets are produced and consumed on the device).
//
//  * scan_kernel: single-pass exclusive prefix sum with decoupled look-back (tile aggregates / inclusive prefixes
//    published through one 64-bit status word per tile; tiles are claimed by an atomic ticket so that every
//    predecessor of a running tile is itself running or finished).  Used for the cluster counts per
//    (event, layer) -> layer_offsets / event_offsets and for the (tracks, hits) counts per event.  The data moves are
//    fused into the track kernel (clusters) and compact_tracks_kernel (tracks).
#include "velo_common.cuh"

namespace velo {
namespace {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr uint32_t kTile = kScanThreads * kScanItems;
constexpr unsigned long long kFlagAggregate = 1ull << 62, kFlagInclusive = 2ull << 62, kValueMask = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// state[0] = ticket counter, state[1 + t] = status of tile t.
template <typename TIn, typename TOut>
__global__ void __launch_bounds__(kScanThreads) scan_kernel(const TIn* __restrict__ in, TOut* __restrict__ out,
                                                            uint32_t n, unsigned long long* state,
                                                            uint32_t* __restrict__ aux_out, uint32_t aux_stride) {
  __shared__ unsigned long long warp_sums[kScanThreads / 32];
  __shared__ unsigned long long tile_exclusive;
  __shared__ uint32_t tile_id;
  if (threadIdx.x == 0) tile_id = (uint32_t)atomicAdd(state, 1ull);
  __syncthreads();
  const uint32_t tile = tile_id;
  unsigned long long* status = state + 1;
  const uint32_t base = tile * kTile + threadIdx.x * kScanItems;

  unsigned long long v[kScanItems], sum = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    v[i] = base + i < n ? (unsigned long long)in[base + i] : 0ull;
    sum += v[i];
  }
  // block exclusive scan of the per-thread sums
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
  unsigned long long incl = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned long long t = __shfl_up_sync(kFull, incl, d);
    if (lane >= (uint32_t)d) incl += t;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  unsigned long long warp_off = 0, tile_total = 0;
#pragma unroll
  for (int w = 0; w < kScanThreads / 32; ++w) {
    if (w < (int)warp) warp_off += warp_sums[w];
    tile_total += warp_sums[w];
  }

  if (warp == 0) {
    if (lane == 0) st_status(status + tile, (tile == 0 ? kFlagInclusive : kFlagAggregate) | tile_total);
    unsigned long long exclusive = 0;
    if (tile > 0) {
      int look = (int)tile - 1;
      for (;;) {
        const int idx = look - (int)lane;
        unsigned long long s = kFlagInclusive;  // tiles before the first count as an inclusive prefix of 0
        if (idx >= 0) {
          do { s = ld_status(status + idx); } while ((s >> 62) == 0);
        }
        const uint32_t incl_mask = __ballot_sync(kFull, (s >> 62) == 2);
        const int first = incl_mask ? __ffs(incl_mask) - 1 : 32;
        unsigned long long part = (int)lane <= first ? (s & kValueMask) : 0ull;
#pragma unroll
        for (int d = 16; d; d >>= 1) part += __shfl_xor_sync(kFull, part, d);
        exclusive += part;
        if (incl_mask) break;
        look -= 32;
      }
      if (lane == 0) st_status(status + tile, kFlagInclusive | (exclusive + tile_total));
    }
    if (lane == 0) tile_exclusive = exclusive;
  }
  __syncthreads();
  unsigned long long run = tile_exclusive + warp_off + (incl - sum);
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    const uint32_t idx = base + i;
    if (idx < n) {
      out[idx] = (TOut)run;
      if (aux_out && idx % aux_stride == 0) aux_out[idx / aux_stride] = (uint32_t)run;
    }
    run += v[i];
    if (idx + 1 == n) {
      out[n] = (TOut)run;
      if (aux_out && n % aux_stride == 0) aux_out[n / aux_stride] = (uint32_t)run;
    }
  }
}

template <typename TIn, typename TOut>
cudaError_t run_scan(const TIn* in, TOut* out, uint32_t n, unsigned long long* state, uint32_t* aux_out,
                     uint32_t aux_stride, cudaStream_t stream) {
  const uint32_t tiles = (n + kTile - 1) / kTile;
  cudaError_t err = cudaMemsetAsync(state, 0, scan_state_words(n) * sizeof(unsigned long long), stream);
  if (err != cudaSuccess) return err;
  if (n == 0) return cudaMemsetAsync(out, 0, sizeof(TOut), stream);
  scan_kernel<TIn, TOut><<<tiles, kScanThreads, 0, stream>>>(in, out, n, state, aux_out, aux_stride);
  return cudaGetLastError();
}

}  // namespace

size_t scan_state_words(uint32_t n) { return 1 + (size_t)(n + kTile - 1) / kTile; }

cudaError_t launch_scan_u32(const uint32_t* in, uint32_t* out, uint32_t n, unsigned long long* tile_state,
                            uint32_t* aux_out, uint32_t aux_stride, cudaStream_t stream) {
  return run_scan<uint32_t, uint32_t>(in, out, n, tile_state, aux_out, aux_stride ? aux_stride : 1, stream);
}

cudaError_t launch_scan_u64(const unsigned long long* in, unsigned long long* out, uint32_t n,
                            unsigned long long* tile_state, cudaStream_t stream) {
  return run_scan<unsigned long long, unsigned long long>(in, out, n, tile_state, nullptr, 1, stream);
}

}  // namespace velo
