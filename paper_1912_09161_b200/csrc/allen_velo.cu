// Host side of the C ABI declared in include/allen_velo.h: argument checks, workspace carving and the launch
// sequence of the hot path.  No host<->device synchronisation happens in allen_velo_reconstruct.
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "velo_common.cuh"
#include "../../include/allen_velo_debug.h"

using namespace velo;

struct allen_velo {
  allen_velo_geometry_t geo{};  // pointers nulled: host copies live in the vectors below
  DeviceGeometry dev{};
  void* dev_block = nullptr;    // handle-owned device constants
  void* ws = nullptr;
  size_t ws_bytes = 0;
  uint32_t last_launches = 0;
  const uint32_t* last_track_counters = nullptr;  // device: list sizes of the last call (workspace memory)
  uint32_t n_mid_sms = 0;      // SM ids the mid-slot pool of the cluster kernel covers
  uint32_t n_sms = 0;
  uint32_t sp_words_per_layer = 0;  // caller's hint (0: none)
  allen_velo_vertices_t vertices{};  // optional primary-vertex output (vertices == nullptr: off)
  cudaStream_t side[2] = {nullptr, nullptr};  // the larger track-kernel instances run beside the first one
  cudaEvent_t fork_join[3] = {nullptr, nullptr, nullptr};
  std::string last_error;
  // optional per-kernel timing: a ring of (kKernels + 1) events per call
  std::vector<cudaEvent_t> events;
  uint32_t timing_calls = 0;   // ring size in calls (0 = timing off)
  uint64_t call_index = 0;     // reconstruct() calls since timing was enabled
};

namespace {

// timed segments: velo_cluster = prepare + the chain of cluster instances; velo_seed = classification + velo_seed_kernel;
// velo_follow = the three instances of velo_follow_kernel + the second pass
constexpr uint32_t kKernels = 6;
const char* const kKernelNames[kKernels] = {"velo_cluster", "scan_clusters", "velo_seed", "velo_follow", "scan_tracks",
                                            "compact_tracks"};
constexpr size_t kAlign = 256;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

// bytes per slab entry (two 16-byte records + checksum), tracking scratch per cluster (link, hits_slab, fwd_win, trip) and per track
// slot (trk_hitoff, trk_fit, trk_final; one slot per 3 clusters)
constexpr size_t kSlabEntryBytes = 16 + 16 + 4;
constexpr size_t kTrackScratchBytes = 2 + 2 + 8 + 8;  // link, hits_slab, forwarding windows, seed candidates
constexpr size_t kTrackSlotBytes = 4 + 16 + 4;

struct Carve {
  unsigned char* base;
  size_t used = 0;
  template <typename T>
  T* take(size_t count) {
    T* p = reinterpret_cast<T*>(base + used);
    used = align_up(used + count * sizeof(T));
    return p;
  }
};

// Pool slots for layers that exceed the cluster kernel's shared memory (velo_cluster.cu): sized with the batch.
uint32_t big_slots(uint32_t items) { return 16 + items / 4096; }

size_t fixed_bytes(uint32_t n_events, uint32_t n_layers, uint32_t n_mid_sms) {
  const uint32_t items = n_events * n_layers;
  size_t b = 0;
  b += align_up((size_t)items * 4) * 2 + align_up((size_t)items * 18 * 4);  // counts, slab_base, layer descriptors
  b += align_up(scan_state_words(items) * 8);                     // scan state (clusters)
  b += align_up(32 + (size_t)n_mid_sms * 4 + (size_t)(big_slots(items) + 31) / 32 * 4);  // slab spill cursor, deferred-item counters, mid and big masks
  b += align_up((size_t)items * 4) * 2;                           // deferred items of the cluster kernel (two lists)
  b += align_up((size_t)n_mid_sms * 32 * cluster_mid_slot_bytes());
  b += align_up((size_t)big_slots(items) * cluster_big_slot_bytes());
  b += align_up((size_t)n_events * 8) + align_up(((size_t)n_events + 1) * 8);  // track counts, offsets
  b += align_up(scan_state_words(n_events) * 8);                  // scan state (tracks)
  b += align_up(n_events);                                        // class of every event
  b += align_up((size_t)n_events * 4) * 6 + align_up(16 * 4);     // event lists of the track kernels, event flags, counters
  b += align_up((size_t)items * 4);                               // seed candidates per (event, layer)
  b += align_up((size_t)items * kPhiTabStride * 2);               // phi look-up table per (event, layer)
  return b + 16 * kAlign;
}

// Per raw SP word: THREE slab entries (one in the dense part, placed from the bank table; two behind it, because a layer
// with more clusters than SP words moves there as a whole and a super-pixel holds up to two clusters) and the tracking
// scratch of TWO clusters.
size_t per_word_bytes() { return 3 * kSlabEntryBytes + 2 * (kTrackScratchBytes + (kTrackSlotBytes + 2) / 3); }

int fail(allen_velo* h, int code, const char* what, cudaError_t err = cudaSuccess) {
  if (h) {
    h->last_error = what;
    if (err != cudaSuccess) { h->last_error += ": "; h->last_error += cudaGetErrorString(err); }
  }
  return code;
}

}  // namespace

extern "C" {

void allen_velo_default_params(allen_velo_params_t* p) {
  if (!p) return;
  p->w_seed_phi16 = 512;
  p->w_fwd_phi16 = 512;
  p->max_slope = 0.4f;
  p->s_seed = 0.015625f;   // 2^-6 mm^2
  p->s_fwd = 0.0625f;      // 2^-4
  p->s_weak = 0.0078125f;  // 2^-7
  p->max_skipped = 1;
}

int allen_velo_create(const allen_velo_geometry_t* geo, allen_velo_t** out) {
  if (!geo || !out) return ALLEN_VELO_ERR_INVALID;
  *out = nullptr;
  if (!geo->sensor_module || !geo->module_layer || !geo->sensor_ltg) return ALLEN_VELO_ERR_INVALID;
  if (geo->n_sensors == 0 || geo->n_sensors > 4096 || geo->n_modules == 0 || geo->n_layers < 3 ||
      geo->n_layers > (uint32_t)kMaxLayers)
    return ALLEN_VELO_ERR_INVALID;
  if (geo->n_cols == 0 || geo->n_cols > 1024 || (geo->n_cols & 1) || geo->n_rows == 0 || geo->n_rows > 256 ||
      (geo->n_rows & 3) || (uint64_t)geo->n_cols * geo->n_rows > (1u << 18))
    return ALLEN_VELO_ERR_INVALID;
  const allen_velo_params_t& P = geo->params;
  if (P.w_seed_phi16 < 0 || P.w_seed_phi16 > 16383 || P.w_fwd_phi16 < 0 || P.w_fwd_phi16 > 16383 ||
      P.max_skipped < 0 || P.max_skipped > 200 || !(P.max_slope >= 0) || !(P.s_seed >= 0) || !(P.s_fwd >= 0) ||
      !(P.s_weak >= 0))
    return ALLEN_VELO_ERR_INVALID;

  const uint32_t S = geo->n_sensors, L = geo->n_layers;
  std::vector<uint16_t> sensor_layer(S), layer_sensors((size_t)L * kMaxSensorsPerLayer, 0);
  std::vector<uint8_t> layer_n(L, 0);
  for (uint32_t s = 0; s < S; ++s) {
    const uint32_t m = geo->sensor_module[s];
    if (m >= geo->n_modules) return ALLEN_VELO_ERR_INVALID;
    const uint32_t l = geo->module_layer[m];
    if (l >= L) return ALLEN_VELO_ERR_INVALID;
    if (layer_n[l] >= kMaxSensorsPerLayer) return ALLEN_VELO_ERR_INVALID;
    sensor_layer[s] = (uint16_t)l;
    layer_sensors[(size_t)l * kMaxSensorsPerLayer + layer_n[l]++] = (uint16_t)s;
  }

  allen_velo* h = new (std::nothrow) allen_velo();
  if (!h) return ALLEN_VELO_ERR_INVALID;
  h->geo = *geo;
  h->geo.sensor_module = nullptr; h->geo.module_layer = nullptr; h->geo.sensor_ltg = nullptr;

  // one device block: ltg | sensor_layer | layer_sensors | layer_n_sensors
  const size_t b_ltg = align_up((size_t)S * 9 * 4), b_sl = align_up((size_t)S * 2),
               b_ls = align_up(layer_sensors.size() * 2), b_ln = align_up(L);
  cudaError_t err = cudaMalloc(&h->dev_block, b_ltg + b_sl + b_ls + b_ln + kAlign);
  if (err == cudaSuccess) err = cudaMemset(static_cast<unsigned char*>(h->dev_block) + b_ltg + b_sl + b_ls + b_ln, 0, kAlign);
  if (err != cudaSuccess) { delete h; return ALLEN_VELO_ERR_CUDA; }
  unsigned char* d = static_cast<unsigned char*>(h->dev_block);
  err = cudaMemcpy(d, geo->sensor_ltg, (size_t)S * 9 * 4, cudaMemcpyHostToDevice);
  if (err == cudaSuccess) err = cudaMemcpy(d + b_ltg, sensor_layer.data(), (size_t)S * 2, cudaMemcpyHostToDevice);
  if (err == cudaSuccess)
    err = cudaMemcpy(d + b_ltg + b_sl, layer_sensors.data(), layer_sensors.size() * 2, cudaMemcpyHostToDevice);
  if (err == cudaSuccess) err = cudaMemcpy(d + b_ltg + b_sl + b_ls, layer_n.data(), L, cudaMemcpyHostToDevice);
  if (err != cudaSuccess) { cudaFree(h->dev_block); delete h; return ALLEN_VELO_ERR_CUDA; }

  int dev = 0, n_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm <= 0) {
    cudaFree(h->dev_block); delete h; return ALLEN_VELO_ERR_CUDA;
  }
  h->n_sms = (uint32_t)n_sm;
  if (cluster_prepare() != cudaSuccess || track_prepare() != cudaSuccess) { cudaFree(h->dev_block); delete h; return ALLEN_VELO_ERR_CUDA; }
  h->n_mid_sms = (uint32_t)n_sm + 16;  // %smid is below the SM count on the parts seen; margin for gaps in the numbering
  for (int i = 0; i < 2; ++i)
    if (cudaStreamCreateWithFlags(&h->side[i], cudaStreamNonBlocking) != cudaSuccess) { allen_velo_destroy(h); return ALLEN_VELO_ERR_CUDA; }
  for (int i = 0; i < 3; ++i)
    if (cudaEventCreateWithFlags(&h->fork_join[i], cudaEventDisableTiming) != cudaSuccess) { allen_velo_destroy(h); return ALLEN_VELO_ERR_CUDA; }
  DeviceGeometry& g = h->dev;
  g.n_sensors = S; g.n_layers = L; g.n_cols = geo->n_cols; g.n_rows = geo->n_rows;
  g.sp_cols = geo->n_cols / 2; g.sp_rows = geo->n_rows / 4;
  g.table_words = (S + 1 + 3) / 4 * 4;
  g.region_shift_c = g.region_shift_r = 31;
  g.pitch = geo->pitch_mm;
  g.ltg = reinterpret_cast<const float*>(d);
  g.sensor_layer = reinterpret_cast<const uint16_t*>(d + b_ltg);
  g.layer_sensors = reinterpret_cast<const uint16_t*>(d + b_ltg + b_sl);
  g.layer_n_sensors = reinterpret_cast<const uint8_t*>(d + b_ltg + b_sl + b_ls);
  g.params = geo->params;
  g.debug_fault = reinterpret_cast<uint32_t*>(d + b_ltg + b_sl + b_ls + b_ln);
  *out = h;
  return ALLEN_VELO_OK;
}

size_t allen_velo_workspace_bytes(const allen_velo_t* h, uint32_t n_events, size_t raw_bytes) {
  if (!h) return 0;
  if ((uint64_t)n_events * h->dev.n_layers >= (1ull << 31)) return 0;  // reconstruct() refuses such a batch
  // slab and tracking scratch per raw word (per_word_bytes): a super-pixel holds at most two clusters: one in the dense
  // part of the slab, one behind it for layers with more clusters than SP words
  const size_t words = raw_bytes / 4 + 2048;
  return fixed_bytes(n_events, h->dev.n_layers, h->n_mid_sms) + words * per_word_bytes() + 16 * kAlign;
}

int allen_velo_set_occupancy_hint(allen_velo_t* h, uint32_t sp_words_per_layer) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  h->sp_words_per_layer = sp_words_per_layer;
  return ALLEN_VELO_OK;
}

int allen_velo_set_cluster_regions(allen_velo_t* h, uint32_t sp_cols, uint32_t sp_rows) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  if (sp_cols == 0 || sp_rows == 0) { h->dev.region_shift_c = h->dev.region_shift_r = 31; return ALLEN_VELO_OK; }
  if ((sp_cols & (sp_cols - 1)) || (sp_rows & (sp_rows - 1))) return fail(h, ALLEN_VELO_ERR_INVALID, "region size not a power of two");
  uint32_t sc = 0, sr = 0;
  while ((1u << sc) < sp_cols) ++sc;
  while ((1u << sr) < sp_rows) ++sr;
  h->dev.region_shift_c = sc;
  h->dev.region_shift_r = sr;
  return ALLEN_VELO_OK;
}

int allen_velo_set_vertex_output(allen_velo_t* h, const allen_velo_vertices_t* out) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  if (!out) { h->vertices = allen_velo_vertices_t{}; return ALLEN_VELO_OK; }
  if (!out->n_vertices || !out->vertices || out->max_per_event == 0) return fail(h, ALLEN_VELO_ERR_INVALID, "null vertex output");
  h->vertices = *out;
  return ALLEN_VELO_OK;
}

int allen_velo_set_workspace(allen_velo_t* h, void* dev_ptr, size_t bytes) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  if (dev_ptr && (reinterpret_cast<uintptr_t>(dev_ptr) % kAlign)) return fail(h, ALLEN_VELO_ERR_INVALID, "workspace misaligned");
  h->ws = dev_ptr;
  h->ws_bytes = dev_ptr ? bytes : 0;
  return ALLEN_VELO_OK;
}

int allen_velo_reconstruct(allen_velo_t* h, const void* raw_banks, const uint32_t* event_offsets, uint32_t n_events,
                           void* cuda_stream, const allen_velo_clusters_t* oc, const allen_velo_tracks_t* ot) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  h->last_launches = 0;
  if (!event_offsets || !oc || !ot || (!raw_banks && n_events)) return fail(h, ALLEN_VELO_ERR_INVALID, "null argument");
  if (reinterpret_cast<uintptr_t>(raw_banks) % 16) return fail(h, ALLEN_VELO_ERR_INVALID, "raw_banks not 16-byte aligned");
  if (!oc->event_offsets || !oc->layer_offsets || !oc->status || !ot->event_offsets || !ot->hit_offsets)
    return fail(h, ALLEN_VELO_ERR_INVALID, "null output offsets");
  if (oc->capacity && (!oc->key || !oc->n_pixels || !oc->sum_col || !oc->sum_row || !oc->x || !oc->y || !oc->z || !oc->phi16))
    return fail(h, ALLEN_VELO_ERR_INVALID, "null cluster array");
  if (ot->capacity_tracks && (!ot->x0 || !ot->y0 || !ot->tx || !ot->ty)) return fail(h, ALLEN_VELO_ERR_INVALID, "null track array");
  if (ot->capacity_hits && !ot->hits) return fail(h, ALLEN_VELO_ERR_INVALID, "null hits array");
  if (h->vertices.vertices && !ot->kalman) return fail(h, ALLEN_VELO_ERR_INVALID, "vertex output needs tracks.kalman");
  const uint32_t L = h->dev.n_layers;
  if ((uint64_t)n_events * L >= (1ull << 31)) return fail(h, ALLEN_VELO_ERR_INVALID, "too many events");
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t err;

  if (n_events == 0) {
    err = cudaMemsetAsync(oc->event_offsets, 0, 4, stream);
    if (err == cudaSuccess) err = cudaMemsetAsync(oc->layer_offsets, 0, 4, stream);
    if (err == cudaSuccess) err = cudaMemsetAsync(ot->event_offsets, 0, 4, stream);
    if (err == cudaSuccess) err = cudaMemsetAsync(ot->hit_offsets, 0, 4, stream);
    return err == cudaSuccess ? ALLEN_VELO_OK : fail(h, ALLEN_VELO_ERR_CUDA, "memset", err);
  }

  // ---- carve the workspace
  const size_t fixed = fixed_bytes(n_events, L, h->n_mid_sms);
  if (!h->ws || h->ws_bytes < fixed + 512 * per_word_bytes() + 16 * kAlign) return fail(h, ALLEN_VELO_ERR_WORKSPACE, "workspace too small");
  const uint32_t items = n_events * L;
  Carve cv{static_cast<unsigned char*>(h->ws)};
  uint32_t* counts = cv.take<uint32_t>(items);
  uint32_t* slab_base = cv.take<uint32_t>(items);
  uint32_t* desc = cv.take<uint32_t>((size_t)items * 18);
  unsigned long long* scan_state = cv.take<unsigned long long>(scan_state_words(items));
  // slab spill cursor, deferred-item counts and cursors, then the mid and big masks: zeroed by one memset
  const size_t state_bytes = 32 + (size_t)h->n_mid_sms * 4 + (size_t)(big_slots(items) + 31) / 32 * 4;
  unsigned long long* state = reinterpret_cast<unsigned long long*>(cv.take<unsigned char>(state_bytes));
  uint32_t* defer_list = cv.take<uint32_t>(items);
  uint32_t* defer_list2 = cv.take<uint32_t>(items);
  const uint32_t n_big = big_slots(items);
  unsigned char* mid_pool = cv.take<unsigned char>((size_t)h->n_mid_sms * 32 * cluster_mid_slot_bytes());
  unsigned char* big_pool = cv.take<unsigned char>((size_t)n_big * cluster_big_slot_bytes());
  unsigned long long* trk_counts = cv.take<unsigned long long>(n_events);
  unsigned long long* trk_offsets = cv.take<unsigned long long>((size_t)n_events + 1);
  unsigned long long* trk_scan_state = cv.take<unsigned long long>(scan_state_words(n_events));
  uint8_t* trk_level = cv.take<uint8_t>(n_events);
  uint32_t* trk_lists[6];
  for (uint32_t*& p : trk_lists) p = cv.take<uint32_t>(n_events);
  uint32_t* trk_counters = cv.take<uint32_t>(16);
  uint32_t* trip_count = cv.take<uint32_t>(items);
  uint16_t* phi_tab = cv.take<uint16_t>((size_t)items * kPhiTabStride);
  size_t words = (h->ws_bytes - cv.used - 16 * kAlign) / per_word_bytes();
  if (words > 0x2AAAAAA0u) words = 0x2AAAAAA0u;
  const size_t slab_entries = 3 * words;
  const size_t entries = 2 * words;  // clusters the tracking scratch (indexed by output cluster) can hold
  ClusterSlab slab{};
  slab.capacity = (uint32_t)slab_entries;
  slab.dense = (uint32_t)words;
  slab.rec = cv.take<uint4>(slab_entries);
  slab.info = cv.take<uint4>(slab_entries);
  slab.checksum = cv.take<uint32_t>(slab_entries);
  slab.spill_cursor = reinterpret_cast<uint32_t*>(state) + 1;
  slab.phi_tab = phi_tab;
  // tracking scratch is addressed by output cluster index; it shares the entry count with the slab
  uint16_t* link = cv.take<uint16_t>(entries);
  uint16_t* hits_slab = cv.take<uint16_t>(entries);
  uint2* fwd_win = cv.take<uint2>(entries);
  unsigned long long* trip = cv.take<unsigned long long>(entries);
  uint32_t* trk_hitoff = cv.take<uint32_t>(entries / 3 + 1);
  float4* trk_fit = cv.take<float4>(entries / 3 + 1);
  uint32_t* trk_final = cv.take<uint32_t>(entries / 3 + 1);
  if (cv.used > h->ws_bytes) return fail(h, ALLEN_VELO_ERR_WORKSPACE, "workspace carve overflow");

  // ---- launch sequence
  err = cudaMemsetAsync(oc->status, 0, (size_t)n_events * 4, stream);
  if (err == cudaSuccess) err = cudaMemsetAsync(state, 0, state_bytes, stream);
  if (err != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "memset", err);
  cudaEvent_t* ev = nullptr;
  if (h->timing_calls) ev = h->events.data() + (h->call_index++ % h->timing_calls) * (kKernels + 1);
  auto mark = [&](uint32_t i) { if (ev) cudaEventRecord(ev[i], stream); };
  mark(0);

  ClusterLaunch cl{};
  cl.geo = h->dev;
  cl.raw = static_cast<const uint32_t*>(raw_banks);
  cl.event_offsets = event_offsets;
  cl.n_events = n_events;
  cl.slab = slab;
  cl.counts = counts;
  cl.slab_base = slab_base;
  cl.desc = desc;
  cl.status = oc->status;
  cl.big_mask = reinterpret_cast<uint32_t*>(state + 4) + h->n_mid_sms;
  cl.defer_count = reinterpret_cast<uint32_t*>(state) + 2;
  cl.defer_list[0] = defer_list;
  cl.defer_list[1] = defer_list2;
  cl.mid_mask = reinterpret_cast<uint32_t*>(state + 4);
  cl.mid_pool = mid_pool;
  cl.big_pool = big_pool;
  cl.n_mid_sms = h->n_mid_sms;
  cl.n_big_slots = n_big;
  cl.with_checksum = oc->checksum != nullptr;
  const bool big_layers = h->sp_words_per_layer > 192;  // the larger shared-memory instance keeps such layers on chip
  uint32_t n_cluster_launches = 0;
  if ((err = launch_cluster(cl, big_layers, h->n_sms, &n_cluster_launches, stream)) != cudaSuccess)
    return fail(h, ALLEN_VELO_ERR_CUDA, "cluster kernel", err);
  h->last_launches += n_cluster_launches;
  mark(1);

  if ((err = launch_scan_u32(counts, oc->layer_offsets, items, scan_state, oc->event_offsets, L, stream)) != cudaSuccess)
    return fail(h, ALLEN_VELO_ERR_CUDA, "cluster scan", err);
  h->last_launches++;
  mark(2);

  TrackLaunch tl{};
  tl.geo = h->dev;
  tl.n_events = n_events;
  tl.clusters = *oc;
  tl.slab = slab;
  tl.slab_base = slab_base;
  if (tl.clusters.capacity > entries) tl.clusters.capacity = (uint32_t)entries;  // scratch is indexed by cluster
  tl.link = link;
  tl.hits_slab = hits_slab;
  tl.trk_hitoff = trk_hitoff;
  tl.trk_fit = trk_fit;
  tl.trk_final = trk_final;
  tl.counts = trk_counts;
  tl.level = trk_level;
  tl.flw_list[0] = trk_lists[0]; tl.flw_list[1] = trk_lists[1]; tl.flw_list[2] = trk_lists[2];
  tl.redo_list[0] = trk_lists[3]; tl.redo_list[1] = trk_lists[4];
  tl.ev_flags = trk_lists[5];
  tl.fwd_win = fwd_win;
  tl.trip = trip;
  tl.trip_count = trip_count;
  tl.counters = trk_counters;
  h->last_track_counters = trk_counters;
  uint32_t n_track_launches = 0;
  if ((err = launch_track_seed(tl, stream, &n_track_launches)) != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "seed kernel", err);
  h->last_launches += n_track_launches;
  mark(3);
  if ((err = launch_track_follow(tl, stream, h->side, h->fork_join, h->n_sms, &n_track_launches)) != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "follow kernel", err);
  h->last_launches += n_track_launches;
  mark(4);

  if ((err = launch_scan_u64(trk_counts, trk_offsets, n_events, trk_scan_state, stream)) != cudaSuccess)
    return fail(h, ALLEN_VELO_ERR_CUDA, "track scan", err);
  h->last_launches++;
  mark(5);

  CompactTracksLaunch ct{};
  ct.n_events = n_events;
  ct.n_layers = h->dev.n_layers;
  ct.pitch = h->dev.pitch;
  ct.clusters = *oc;
  ct.hits_slab = hits_slab;
  ct.trk_hitoff = trk_hitoff;
  ct.trk_fit = trk_fit;
  ct.offsets = trk_offsets;
  ct.ev_flags = tl.ev_flags;
  ct.trk_final = trk_final;
  ct.link = link;
  ct.s_weak = h->dev.params.s_weak;
  ct.out = *ot;
  if ((err = launch_compact_tracks(ct, stream)) != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "track compaction", err);
  h->last_launches++;
  mark(6);
  if (h->vertices.vertices) {  // beyond the timed segments of the headline path
    PvLaunch pv{};
    pv.n_events = n_events;
    pv.tracks = *ot;
    pv.out = h->vertices;
    pv.status = oc->status;
    if ((err = launch_pv(pv, stream)) != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "vertex kernel", err);
    h->last_launches++;
  }
  return ALLEN_VELO_OK;
}

int allen_velo_enable_timing(allen_velo_t* h, uint32_t n_calls) {
  if (!h) return ALLEN_VELO_ERR_INVALID;
  for (cudaEvent_t e : h->events) cudaEventDestroy(e);
  h->events.clear();
  h->timing_calls = 0;
  h->call_index = 0;
  if (n_calls == 0) return ALLEN_VELO_OK;
  h->events.resize((size_t)n_calls * (kKernels + 1));
  for (cudaEvent_t& e : h->events)
    if (cudaEventCreate(&e) != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "cudaEventCreate");
  h->timing_calls = n_calls;
  return ALLEN_VELO_OK;
}

uint32_t allen_velo_kernel_count(void) { return kKernels; }

const char* allen_velo_kernel_name(uint32_t i) { return i < kKernels ? kKernelNames[i] : ""; }

int allen_velo_kernel_times(allen_velo_t* h, uint32_t call, float* out_ms) {
  if (!h || !out_ms || !h->timing_calls || call >= h->timing_calls) return ALLEN_VELO_ERR_INVALID;
  cudaEvent_t* ev = h->events.data() + (size_t)call * (kKernels + 1);
  for (uint32_t i = 0; i < kKernels; ++i) {
    cudaError_t err = cudaEventElapsedTime(out_ms + i, ev[i], ev[i + 1]);
    if (err != cudaSuccess) return fail(h, ALLEN_VELO_ERR_CUDA, "cudaEventElapsedTime", err);
  }
  return ALLEN_VELO_OK;
}

uint32_t allen_velo_last_launch_count(const allen_velo_t* h) { return h ? h->last_launches : 0; }

int allen_velo_debug_fault(allen_velo_t* h, uint32_t* out) {
  if (!h || !out) return ALLEN_VELO_ERR_INVALID;
  cudaError_t err = cudaMemcpy(out, h->dev.debug_fault, sizeof(uint32_t), cudaMemcpyDeviceToHost);
  if (err == cudaSuccess) err = cudaMemset(h->dev.debug_fault, 0, sizeof(uint32_t));
  return err == cudaSuccess ? ALLEN_VELO_OK : fail(h, ALLEN_VELO_ERR_CUDA, "cudaMemcpy", err);
}

int allen_velo_debug_checks_compiled(void) {
#ifdef VELO_DEBUG
  return 1;
#else
  return 0;
#endif
}

int allen_velo_debug_track_counters(allen_velo_t* h, uint32_t* out) {
  if (!h || !out || !h->last_track_counters) return ALLEN_VELO_ERR_INVALID;
  const cudaError_t err = cudaMemcpy(out, h->last_track_counters, 16 * sizeof(uint32_t), cudaMemcpyDeviceToHost);
  return err == cudaSuccess ? ALLEN_VELO_OK : fail(h, ALLEN_VELO_ERR_CUDA, "cudaMemcpy", err);
}

const char* allen_velo_last_error(const allen_velo_t* h) { return h ? h->last_error.c_str() : "null handle"; }

void allen_velo_destroy(allen_velo_t* h) {
  if (!h) return;
  for (cudaEvent_t e : h->events) cudaEventDestroy(e);
  for (cudaStream_t st : h->side) if (st) cudaStreamDestroy(st);
  for (cudaEvent_t e : h->fork_join) if (e) cudaEventDestroy(e);
  if (h->dev_block) cudaFree(h->dev_block);
  delete h;
}

}  // extern "C"
