// Definitions shared by the kernels of the track search (velo_seed.cu + velo_follow.cu: the two-kernel path every event
// takes first; velo_track.cu: one CTA per event, for the events that path hands on).  Not part of the ABI, not used by oracle/.
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
constexpr uint8_t kClsFlat = 0;    // busiest layer <= kFlatCap hits
constexpr uint8_t kClsMid = 1;     // <= 512 hits per layer
constexpr uint8_t kClsLarge = 2;   // <= 1024 hits per layer
constexpr uint8_t kClsSkip = 255;  // nothing to do (no clusters, or the output cannot hold them)
constexpr uint8_t kClsCopy = 254;  // clusters are moved to the output, no tracking (incomplete or > 65535 clusters)

constexpr int kFlatCap = 256;      // hits per layer of the first instance of velo_follow.cu

constexpr uint32_t kEvRedo = 1u;   // TrackLaunch::ev_flags: velo_seed.cu could not list the event's seed candidates
constexpr uint32_t kEvFinal = 2u;  // velo_follow.cu has left the event's tracks as final states (trk_final) and links; the
                                   // number of tracks created is in bits 8 and up (compact_tracks_kernel does T5 and the fit)

// TrackLaunch::counters
constexpr uint32_t kCtrFollow = 0;         // [3] events of class 0 / 1 / 2
constexpr uint32_t kCtrFollowCursor = 4;   // [3]
constexpr uint32_t kCtrRedo = 12;          // [2] events in redo_list
constexpr uint32_t kCtrRedoCursor = 14;    // [2]
constexpr uint32_t kCtrCount = 16;

// Final state of a track (tstate layout of both kernels): newest hit (event-local) << 16 | weak_ok << 15 | n_hits << 8.
__device__ __forceinline__ uint32_t track_n_hits(uint32_t st) { return (st >> 8) & 0x7Fu; }

cudaError_t seed_prepare();
cudaError_t launch_seed(const TrackLaunch& a, cudaStream_t stream);
cudaError_t follow_prepare();
cudaError_t launch_follow(const TrackLaunch& a, uint32_t level, uint32_t n_sms, cudaStream_t stream);

}  // namespace velo
