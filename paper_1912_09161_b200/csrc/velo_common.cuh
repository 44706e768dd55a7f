// Internal definitions shared by the CUDA kernels of the VELO hot path (not part of the ABI, not used by oracle/).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/allen_velo.h"

namespace velo {

constexpr uint32_t kMagic = 0x56454C4Fu;
constexpr int kMaxSensorsPerLayer = 8;
constexpr int kMaxLayers = 64;
constexpr uint32_t kFull = 0xFFFFFFFFu;

// Device view of the geometry (pointers into the handle's constant block).
struct DeviceGeometry {
  uint32_t n_sensors, n_layers, n_cols, n_rows, sp_cols, sp_rows;
  uint32_t table_words;  // bank table incl. padding, in u32 words
  uint32_t region_shift_c, region_shift_r;  // local clustering variant (R11): log2 of the region size in SPs; 31 = exact CCL
  uint32_t* debug_fault;  // one word in the handle's device block: highest VELO_CHECK code that failed (VELO_DEBUG builds)
  float pitch;
  const uint16_t* sensor_layer;     // [n_sensors]
  const uint16_t* layer_sensors;    // [n_layers][kMaxSensorsPerLayer]
  const uint8_t* layer_n_sensors;   // [n_layers]
  const float* ltg;                 // [n_sensors][9]
  allen_velo_params_t params;
};

// Slab the cluster kernel writes: two arrays of 16-byte records with `capacity` entries; the region of (event, layer)
// starts at slab_base[item] and holds counts[item] clusters in the normative order.  The track kernel stages a layer with
// one 128-bit load per hit and moves it to the output.
//   rec[i]  = { x, y, z (fp32 bit patterns), phi16 as u16 in the low half (high half zero) }  = the search's hit record
//   info[i] = { key, n_pixels, sum_col, sum_row }
// Entries [0, dense) are placed from the bank tables alone (one entry per raw SP word: the region of a layer starts at
// the position of its first SP word); a layer with more clusters than SP words (super-pixels holding two clusters)
// takes its region from [dense, capacity) with a cursor instead.
struct ClusterSlab {
  uint32_t capacity, dense;
  uint4 *rec, *info;
  uint32_t* checksum;
  uint32_t* spill_cursor;  // entries handed out of [dense, capacity), zeroed by the launcher
  uint16_t* phi_tab;       // [n_events*n_layers][kPhiTabStride] first cluster of every 256-unit slice of phi16 (+ total), per layer
};
constexpr uint32_t kPhiSlices = 256;      // the buckets of the cluster kernel's counting sort on the top byte of phi16
constexpr uint32_t kPhiTabStride = 264;   // u16 per (event, layer): kPhiSlices + 1 entries, padded to 16 bytes

// ---- bounds checks of the debug build (compute-sanitizer is closed on this pool) ---------------------------------------
// Built with -DVELO_DEBUG (paper_1912_09161_b200/build.py --debug -> _allen_velo_debug.so) every index into a shared-memory
// or workspace capacity is tested where it is formed; a failing test records its code in DeviceGeometry::debug_fault
// (read and cleared with allen_velo_debug_fault) and the access is still made, so that results show the damage too.
// Codes: 1xx velo_cluster.cu, 2xx velo_seed.cu, 3xx velo_follow.cu, 4xx velo_track.cu.
#ifdef VELO_DEBUG
#define VELO_CHECK(geo, cond, code) do { if (!(cond)) atomicMax((geo).debug_fault, (uint32_t)(code)); } while (0)
#else
#define VELO_CHECK(geo, cond, code) ((void)0)
#endif

// ---- small device helpers -------------------------------------------------------------------
__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// mix32 of DESIGN.md R2 (membership checksum term of one pixel)
__device__ __forceinline__ uint32_t mix32(uint32_t v) {
  uint32_t m = (v + 1u) * 2654435761u;
  m ^= m >> 15;
  m *= 2246822519u;
  m ^= m >> 13;
  return m;
}

// Normative fp32 position of a cluster (R3): every operation a single IEEE RN op, fma fused, no contraction.
// Two halves: local coordinates (u, v) from the integer sums, then the sensor's local-to-global transform.
__device__ __forceinline__ void cluster_local(uint32_t n, uint32_t sum_col, uint32_t sum_row, float pitch, float& u,
                                              float& v) {
  const float fn = __uint2float_rn(n);
  const float fc = __fadd_rn(__fdiv_rn(__uint2float_rn(sum_col), fn), 0.5f);
  const float fr = __fadd_rn(__fdiv_rn(__uint2float_rn(sum_row), fn), 0.5f);
  u = __fmul_rn(fc, pitch);
  v = __fmul_rn(fr, pitch);
}
__device__ __forceinline__ void local_to_global(float u, float v, const float* __restrict__ M, float& x, float& y,
                                                float& z) {
  x = __fmaf_rn(u, __ldg(M + 0), __fmaf_rn(v, __ldg(M + 1), __ldg(M + 2)));
  y = __fmaf_rn(u, __ldg(M + 3), __fmaf_rn(v, __ldg(M + 4), __ldg(M + 5)));
  z = __fmaf_rn(u, __ldg(M + 6), __fmaf_rn(v, __ldg(M + 7), __ldg(M + 8)));
}
__device__ __forceinline__ void cluster_position(uint32_t n, uint32_t sum_col, uint32_t sum_row, float pitch,
                                                 const float* __restrict__ M, float& x, float& y, float& z) {
  float u, v;
  cluster_local(n, sum_col, sum_row, pitch, u, v);
  local_to_global(u, v, M, x, y, z);
}

// Normative phi16 (R3): Abramowitz & Stegun 4.4.49 polynomial, Horner with fma, round-half-even, wrap.
__device__ __forceinline__ int16_t phi16_of(float x, float y) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = ax > ay ? ax : ay, mn = ax > ay ? ay : ax;
  const float t = mx == 0.0f ? 0.0f : __fdiv_rn(mn, mx);
  const float s = __fmul_rn(t, t);
  float p = 0.0028662257f;
  p = __fmaf_rn(p, s, -0.0161657367f);
  p = __fmaf_rn(p, s, 0.0429096138f);
  p = __fmaf_rn(p, s, -0.0752896400f);
  p = __fmaf_rn(p, s, 0.1065626393f);
  p = __fmaf_rn(p, s, -0.1420889944f);
  p = __fmaf_rn(p, s, 0.1999355085f);
  p = __fmaf_rn(p, s, -0.3333314528f);
  p = __fmaf_rn(p, s, 1.0f);
  p = __fmul_rn(p, t);
  if (ay > ax) p = __fsub_rn(1.5707964f, p);
  if (x < 0.0f) p = __fsub_rn(3.1415927f, p);
  if (y < 0.0f) p = -p;
  const int r = __float2int_rn(__fmul_rn(p, 10430.378f));
  return (int16_t)(uint16_t)(r & 0xFFFF);
}

// Normative scatter (R5) of c after a (older) then b (newer).
__device__ __forceinline__ float scatter(float xa, float ya, float za, float xb, float yb, float zb, float xc,
                                         float yc, float zc) {
  const float dz_ab = __fsub_rn(zb, za);
  const float tx = __fdiv_rn(__fsub_rn(xb, xa), dz_ab);
  const float ty = __fdiv_rn(__fsub_rn(yb, ya), dz_ab);
  const float dz = __fsub_rn(zc, zb);
  const float ex = __fsub_rn(__fmaf_rn(tx, dz, xb), xc);
  const float ey = __fsub_rn(__fmaf_rn(ty, dz, yb), yc);
  return __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
}

__device__ __forceinline__ int dphi16(int16_t a, int16_t b) { return (int16_t)(uint16_t)((uint16_t)a - (uint16_t)b); }

// ---- kernel launchers (defined in the .cu files) -----------------------------------------------
// Cluster kernel: one warp per (event, layer); writes the layer, sorted, to its slab region.  Layers that exceed the
// warp's shared memory use slots of the two pools.
struct ClusterLaunch {
  DeviceGeometry geo;
  const uint32_t* raw;
  const uint32_t* event_offsets;
  uint32_t n_events;
  ClusterSlab slab;
  uint32_t* counts;           // [n_events*n_layers] clusters per (event, layer)
  uint32_t* slab_base;        // [n_events*n_layers] first slab entry of the (event, layer) region
  uint32_t* desc;             // [n_events*n_layers][18] bank ranges of the layer (velo_prepare_kernel)
  uint32_t* status;           // [n_events], zeroed before
  uint32_t* defer_list[2];    // [n_events*n_layers] each: items left to the 256-entry / the 512-entry instance
  uint32_t* defer_count;      // [2][2] list size, cursor; zeroed before
  uint32_t* big_mask;         // [(n_big_slots + 31) / 32] busy bits of the big slots, zeroed before
  uint32_t* mid_mask;         // [n_mid_sms] busy bits of the mid slots of every SM, zeroed before
  unsigned char* mid_pool;    // [32 * n_mid_sms] slots
  unsigned char* big_pool;    // [n_big_slots] slots
  uint32_t n_mid_sms, n_big_slots;
  bool with_checksum;
};
cudaError_t launch_cluster(const ClusterLaunch& a, bool big_layers, uint32_t n_sms, uint32_t* n_launches,
                           cudaStream_t stream);
size_t cluster_mid_slot_bytes();
size_t cluster_big_slot_bytes();

// Exclusive prefix sum of `in[n]` into `out[n+1]` (out[n] = total), single pass with decoupled look-back.
// `tile_state` needs scan_state_words(n) u64 words, zeroed by the launcher.
size_t scan_state_words(uint32_t n);
cudaError_t launch_scan_u32(const uint32_t* in, uint32_t* out, uint32_t n, unsigned long long* tile_state,
                            uint32_t* aux_out, uint32_t aux_stride, cudaStream_t stream);
cudaError_t launch_scan_u64(const unsigned long long* in, unsigned long long* out, uint32_t n,
                            unsigned long long* tile_state, cudaStream_t stream);

// Search by triplet + fit, one CTA per event.  Per-event slabs are addressed from the cluster offsets: an event
// with clusters [co, co+n) owns hits_slab[co, co+n) (a hit belongs to at most one track) and track slots
// [co/3, (co+n)/3) (a track has at least three hits).
struct TrackLaunch {
  DeviceGeometry geo;
  uint32_t n_events;
  allen_velo_clusters_t clusters;  // compacted cluster output: offsets final; the arrays are filled by this kernel
  ClusterSlab slab;                // sorted layers as the cluster kernel left them
  const uint32_t* slab_base;       // [n_events*n_layers]
  uint16_t* link;                  // [cluster capacity] scratch: previous (older) hit of the same track, per hit
  uint16_t* hits_slab;             // [cluster capacity] hit lists of the event's output tracks, back to back
  uint32_t* trk_hitoff;            // [capacity/3+1] event-local first entry in hits_slab of every output track
  float4* trk_fit;                 // [capacity/3+1] x0, y0, tx, ty
  uint32_t* trk_final;             // [capacity/3+1] final state of every track by order of creation
  unsigned long long* counts;      // [n_events] (n_tracks << 32) | n_track_hits
  uint8_t* level;                  // [n_events] class of the event (velo_track.cuh): hits per layer 256 / 512 / 1024, copy only, nothing
  uint2* fwd_win;                  // [cluster capacity] velo_seed.cu: forwarding phi windows of every hit (layer below, the one below that)
  unsigned long long* trip;        // [cluster capacity] velo_seed.cu: seed candidates of every (event, layer B), at the layer's hits
  uint32_t* trip_count;            // [n_events*n_layers] entries in the list of every (event, layer)
  uint32_t* ev_flags;              // [n_events] kEvRedo: the event goes to the CTA-per-event kernel
  uint32_t* flw_list[3];           // [n_events] each: events of class 0 / 1 / 2 (velo_follow.cu)
  uint32_t* redo_list[2];          // [n_events] each: events for the CTA-per-event kernel with 512 / 1024 hits per layer
  uint32_t* counters;              // [kCtrCount] list sizes and cursors (velo_track.cuh), zeroed by the launcher
};
cudaError_t launch_track_seed(const TrackLaunch& a, cudaStream_t stream, uint32_t* n_launches);
cudaError_t launch_track_follow(const TrackLaunch& a, cudaStream_t stream, cudaStream_t* side, cudaEvent_t* ev,
                                uint32_t n_sms, uint32_t* n_launches);
cudaError_t track_prepare();    // once per process: dynamic shared-memory limits of the track kernels
cudaError_t cluster_prepare();  // likewise for the cluster kernels

struct CompactTracksLaunch {
  uint32_t n_events;
  uint32_t n_layers;
  float pitch;  // pixel pitch, mm (measurement error of the Kalman fit)
  allen_velo_clusters_t clusters;
  const uint16_t* hits_slab;
  const uint32_t* trk_hitoff;
  const float4* trk_fit;
  const unsigned long long* offsets;  // [n_events+1] exclusive scan of counts
  const uint32_t* ev_flags;           // [n_events] kEvFinal: tracks as final states + links (velo_follow.cu), else as slabs
  const uint32_t* trk_final;
  const uint16_t* link;
  float s_weak;
  allen_velo_tracks_t out;
};
cudaError_t launch_compact_tracks(const CompactTracksLaunch& a, cudaStream_t stream);

// Primary-vertex finding, one warp per event, after the tracks are compacted (velo_pv.cu).
struct PvLaunch {
  uint32_t n_events;
  allen_velo_tracks_t tracks;  // compacted tracks incl. the Kalman states
  allen_velo_vertices_t out;
  uint32_t* status;            // [n_events]
};
cudaError_t launch_pv(const PvLaunch& a, cudaStream_t stream);

}  // namespace velo
