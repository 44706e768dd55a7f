// Definitions shared by the two implementations of the track search (velo_track_flat.cu: four warps per event, flattened phases, the common
// case; velo_track.cu: one CTA per event with larger staging capacities).  Not part of the ABI, not used by oracle/.
#pragma once
#include "velo_common.cuh"

namespace velo {

constexpr unsigned long long kNoClaim = ~0ull;
constexpr uint32_t kUsedBit = 0x10000u;

// Hit record of the search in shared memory; the cluster kernel writes the same 16 bytes to the slab.
struct __align__(16) Hit {
  float x, y, z;
  uint32_t w;  // phi16 (low 16 bits, two's complement) | used << 16
};

__device__ __forceinline__ int phi_of(uint32_t w) { return (int)(int16_t)(uint16_t)(w & 0xFFFFu); }
__device__ __forceinline__ int wrap16(int v) { return (int)(int16_t)(uint16_t)v; }

// class of an event (TrackLaunch::level), set by classify_events_kernel
constexpr uint8_t kClsFlat = 0;    // searched by velo_track_flat_kernel (busiest layer <= kFlatCap hits)
constexpr uint8_t kClsMid = 1;     // the flat kernel's instance with 512 hits per layer
constexpr uint8_t kClsLarge = 2;   // the flat kernel's instance with 1024 hits per layer
constexpr uint8_t kClsSkip = 255;  // nothing to do (no clusters, or the output cannot hold them)
constexpr uint8_t kClsCopy = 254;  // clusters are moved to the output, no tracking (incomplete or > 65535 clusters)

constexpr int kFlatCap = 256;      // hits of one layer the flat kernel stages

// Final state of a track (tstate layout of both kernels): newest hit (event-local) << 16 | weak_ok << 15 | n_hits << 8.
__device__ __forceinline__ uint32_t track_n_hits(uint32_t st) { return (st >> 8) & 0x7Fu; }

cudaError_t track_flat_prepare();
cudaError_t launch_track_flat(const TrackLaunch& a, cudaStream_t stream);
cudaError_t launch_track_flat_list(const TrackLaunch& a, uint32_t which, uint32_t grid, cudaStream_t stream);

}  // namespace velo
