// Kernel 1 of the VELO hot path: raw decode (A1), exact connected-component clustering (A2), centroid -> global
// position and phi16 (A3) and the per-layer phi sort (A4) — SURVEY.md §8(a); definitions DESIGN.md R1-R4; paper
// P:153 (decoding), P:179 (clustering as connected component labelling), P:183 (sort hits on every layer by phi).
//
// Work decomposition: ONE WARP per (event, layer).  Clustering is independent per sensor (R2) and the sort is
// independent per layer (R4), so a warp needs no block-level barrier: everything below synchronises with
// __syncwarp / warp votes only, and the warps of a CTA are fully decoupled.
//
// Clustering without a pixel grid: the nodes of the graph are "SP components" — a 2x4 super-pixel holds at most two
// 8-connected components (pixels in adjacent rows of a 2-wide block always touch, so components are runs of occupied
// rows).  Super-pixels of one sensor are put into a small open-addressing hash table in shared memory keyed by
// (sp_col, sp_row); each SP looks up only its four "forward" neighbours (col+1: row-1,row,row+1; col: row+1), and only
// those its border pixels can touch (about one probe per SP on minimum-bias occupancy).  Touching components become
// edges; labels (node ids) are propagated over the edge list to the minimum until nothing changes, which is exact for
// any cluster size.  Roots get cluster slots by warp ballot (no atomics); non-root components add their integer sums
// to the root's slot with shared-memory atomics (commutative integer adds/min: deterministic).
//
// The layer's clusters are then ranked by (phi16, key) with a 256-bucket counting sort on the top byte of phi plus an
// exact in-bucket rank, and written in the normative order, coalesced, to the (event, layer) region of the slab.
#include "velo_common.cuh"

namespace velo {
namespace {

constexpr int kWarps = 4;            // warps per CTA (independent work items)
constexpr int kHashBits = 9;
constexpr uint32_t kH = 1u << kHashBits;  // hash slots per sensor
constexpr uint32_t kSpCap = 320;     // SP words per sensor the table takes (load factor <= 0.625)
constexpr uint32_t kEdgeCap = kH;    // edges per sensor
constexpr uint32_t kClCap = 768;     // clusters per (event, layer) staged in shared memory

// per-warp shared memory (bytes)
constexpr uint32_t kScratchBytes = 12 * kH;  // tab u32[H] | lab u16[2H] | edges u32[H] (aliased: cidmap u16[2H])
static_assert(1024 + 6 * kClCap <= kScratchBytes, "sort scratch must fit in the CCL scratch it aliases");

template <bool kChecksum>
struct WarpSmem {
  uint32_t scratch[kScratchBytes / 4];
  uint32_t ckey[kClCap], cn[kClCap], ccol[kClCap], crow[kClCap];
  uint32_t ccks[kChecksum ? kClCap : 1];
  uint32_t n_edges;
};

__device__ __forceinline__ uint32_t hash_slot(uint32_t key) { return (key * 0x9E3779B1u) >> (32 - kHashBits); }

// Slot of `key` in the table, or -1.  Entries are (key << 8) | hitmap, 0 = empty.
__device__ __forceinline__ int lookup(const uint32_t* tab, uint32_t key) {
  uint32_t s = hash_slot(key);
  for (;;) {
    const uint32_t e = tab[s];
    if (e == 0) return -1;
    if ((e >> 8) == key) return (int)s;
    s = (s + 1) & (kH - 1);
  }
}

struct Comps {
  uint32_t rA, rB;  // occupied-row masks (4 bits) of the lowest run and of the rest
};
__device__ __forceinline__ Comps split_rows(uint32_t hitmap) {
  const uint32_t r4 = (hitmap | (hitmap >> 4)) & 0xFu;
  const uint32_t low = r4 & (0u - r4);
  Comps c;
  c.rA = r4 & ~(r4 + low);
  c.rB = r4 ^ c.rA;
  return c;
}

struct Stats {
  uint32_t n, sum_col, sum_row, minpix, cks;
};
template <bool kChecksum>
__device__ __forceinline__ Stats comp_stats(uint32_t m, uint32_t C, uint32_t R, uint32_t n_cols) {
  Stats s;
  s.n = __popc(m);
  s.sum_col = 2 * C * s.n + __popc(m >> 4);
  s.sum_row = 4 * R * s.n + __popc(m & 0x22u) + 2 * __popc(m & 0x44u) + 3 * __popc(m & 0x88u);
  const uint32_t rm = (m | (m >> 4)) & 0xFu;
  const uint32_t r_low = __ffs(rm) - 1;
  const uint32_t dc_low = ((m >> r_low) & 1u) ? 0u : 1u;
  s.minpix = (4 * R + r_low) * n_cols + 2 * C + dc_low;
  s.cks = 0;
  if (kChecksum) {
    uint32_t mm = m;
    while (mm) {
      const uint32_t b = __ffs(mm) - 1;
      mm &= mm - 1;
      s.cks += mix32((4 * R + (b & 3u)) * n_cols + 2 * C + (b >> 2));
    }
  }
  return s;
}

template <bool kChecksum>
__global__ void __launch_bounds__(kWarps * 32) velo_cluster_kernel(const ClusterLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using WS = WarpSmem<kChecksum>;
  WS& ws = reinterpret_cast<WS*>(smem_raw)[threadIdx.x >> 5];
  const DeviceGeometry& g = a.geo;
  const uint32_t lane = lane_id();
  const uint32_t L = g.n_layers;
  const uint32_t item = blockIdx.x * kWarps + (threadIdx.x >> 5);
  if (item >= a.n_events * L) return;
  const uint32_t e = item / L, layer = item % L;

  // ---------------- A1: header, bank table (raw format v1, R1) ----------------
  const uint32_t byte0 = __ldg(a.event_offsets + e), byte1 = __ldg(a.event_offsets + e + 1);
  const uint32_t* ev = a.raw + (byte0 >> 2);
  bool bad = byte1 < byte0 || (byte1 - byte0) < 16 || ((byte1 - byte0) & 15u) || (byte0 & 15u);
  uint32_t n_sp_total = 0;
  if (!bad) {
    const uint32_t n_words = (byte1 - byte0) >> 2;
    bad = __ldg(ev) != kMagic || __ldg(ev + 1) != g.n_sensors;
    n_sp_total = __ldg(ev + 2);
    const unsigned long long need = 4ull + g.table_words + (((unsigned long long)n_sp_total + 3ull) & ~3ull);
    bad = bad || need != n_words;
  }
  const uint32_t* tbl = ev + 4;
  uint32_t before = 0;  // SP words of this event in layers below `layer` (slab placement)
  if (!bad) {
    for (uint32_t j = lane; j < g.n_sensors; j += 32) {
      const uint32_t o0 = __ldg(tbl + j), o1 = __ldg(tbl + j + 1);
      bad = bad || o0 > o1 || (j == 0 && o0 != 0) || (j + 1 == g.n_sensors && o1 != n_sp_total);
      if (__ldg(g.sensor_layer + j) < layer) before += o1 - o0;
    }
  }
  bad = __any_sync(kFull, bad);
  if (bad) {
    if (lane == 0) {
      if (layer == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_BAD_HEADER);
      a.counts[item] = 0;
      a.slab_base[item] = 0;
    }
    return;
  }
  before = __reduce_add_sync(kFull, before);
  const uint32_t* sp = tbl + g.table_words;
  const uint32_t slab0 = 2u * ((byte0 >> 2) + 4u + g.table_words + before);

  // sensors of this layer: lane k < K holds sensor k's bank range
  const uint32_t K = __ldg(g.layer_n_sensors + layer);
  uint32_t my_sensor = 0, my_off = 0, my_cnt = 0;
  if (lane < K) {
    my_sensor = __ldg(g.layer_sensors + layer * kMaxSensorsPerLayer + lane);
    my_off = __ldg(tbl + my_sensor);
    my_cnt = __ldg(tbl + my_sensor + 1) - my_off;
  }
  const uint32_t n_sp_layer = __reduce_add_sync(kFull, my_cnt);
  bool overflow = (unsigned long long)slab0 + 2ull * n_sp_layer > a.slab.capacity;

  uint32_t* tab = ws.scratch;
  uint16_t* lab = reinterpret_cast<uint16_t*>(ws.scratch + kH);
  uint32_t* edges = ws.scratch + 2 * kH;
  uint16_t* cidmap = reinterpret_cast<uint16_t*>(ws.scratch + 2 * kH);

  uint32_t n_cl = 0;  // clusters of this layer so far (warp-uniform)
  bool bad_sp = false;

  // ---------------- A2: clustering, sensor by sensor ----------------
  for (uint32_t k = 0; k < K && !overflow; ++k) {
    const uint32_t sensor = __shfl_sync(kFull, my_sensor, k);
    const uint32_t off = __shfl_sync(kFull, my_off, k);
    const uint32_t cnt = __shfl_sync(kFull, my_cnt, k);
    if (cnt == 0) continue;
    if (cnt > kSpCap) { overflow = true; break; }
    for (uint32_t s = lane; s < kH; s += 32) tab[s] = 0;
    if (lane == 0) ws.n_edges = 0;
    __syncwarp();

    // Phase A: insert SP words (entry = key << 8 | hitmap, key = sp_col << 6 | sp_row); a repeated address merges.
    uint32_t absorbed = 0;  // bit per chunk: this lane's word needs no processing (invalid, empty or merged)
    for (uint32_t i = lane, chunk = 0; i < cnt; i += 32, ++chunk) {
      const uint32_t w = __ldg(sp + off + i);
      const uint32_t h = w & 0xFFu, R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
      if (C >= g.sp_cols || R >= g.sp_rows) { bad_sp = true; absorbed |= 1u << chunk; continue; }
      if (h == 0) { absorbed |= 1u << chunk; continue; }
      const uint32_t key = (C << 6) | R;
      uint32_t s = hash_slot(key);
      for (;;) {
        const uint32_t old = atomicCAS(tab + s, 0u, (key << 8) | h);
        if (old == 0) break;
        if ((old >> 8) == key) { atomicOr(tab + s, h); absorbed |= 1u << chunk; break; }
        s = (s + 1) & (kH - 1);
      }
    }
    __syncwarp();

    // Phase B: every SP initialises its node labels and pushes edges to touching forward neighbours.
    for (uint32_t i = lane, chunk = 0; i < cnt; i += 32, ++chunk) {
      if (absorbed >> chunk & 1u) continue;
      const uint32_t w = __ldg(sp + off + i);
      const uint32_t R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
      const uint32_t key = (C << 6) | R;
      const uint32_t slot = (uint32_t)lookup(tab, key);
      const uint32_t h = tab[slot] & 0xFFu;
      const Comps mine = split_rows(h);
      const uint32_t nA = 2 * slot, nB = 2 * slot + 1;
      lab[nA] = (uint16_t)nA;
      lab[nB] = (uint16_t)nB;
      auto push = [&](uint32_t u, uint32_t v) {
        const uint32_t idx = atomicAdd(&ws.n_edges, 1u);
        if (idx < kEdgeCap) edges[idx] = u | (v << 16);
      };
      const uint32_t r4 = mine.rA | mine.rB;
      const uint32_t n_row3 = (mine.rA & 8u) ? nA : nB;  // our component holding row 3
      // (C, R+1): our row 3 touches their row 0 whatever the columns
      if ((r4 & 8u) && R + 1 < g.sp_rows) {
        const int t = lookup(tab, key + 1);
        if (t >= 0) {
          const uint32_t q = tab[t] & 0xFFu;
          if ((q | (q >> 4)) & 1u) push(n_row3, 2 * t);
        }
      }
      if (C + 1 < g.sp_cols) {
        // (C+1, R): our column-1 pixels touch their column-0 pixels within one row
        if (h & 0xF0u) {
          const int t = lookup(tab, key + 64);
          if (t >= 0) {
            const uint32_t q = tab[t] & 0xFFu;
            const Comps theirs = split_rows(q);
            const uint32_t gl = q & 0xFu;
            const uint32_t hA = (h >> 4) & mine.rA, hB = (h >> 4) & mine.rB;
            const uint32_t adjA = (hA | (hA << 1) | (hA >> 1)) & gl, adjB = (hB | (hB << 1) | (hB >> 1)) & gl;
            if (adjA & theirs.rA) push(nA, 2 * t);
            if (adjA & theirs.rB) push(nA, 2 * t + 1);
            if (adjB & theirs.rA) push(nB, 2 * t);
            if (adjB & theirs.rB) push(nB, 2 * t + 1);
          }
        }
        // (C+1, R+1): our pixel (dc=1, dr=3) touches their pixel (dc=0, dr=0)
        if ((h & 0x80u) && R + 1 < g.sp_rows) {
          const int t = lookup(tab, key + 65);
          if (t >= 0 && (tab[t] & 1u)) push(n_row3, 2 * t);
        }
        // (C+1, R-1): our pixel (dc=1, dr=0) touches their pixel (dc=0, dr=3)
        if ((h & 0x10u) && R >= 1) {
          const int t = lookup(tab, key + 63);
          if (t >= 0 && (tab[t] & 8u)) {
            const Comps theirs = split_rows(tab[t] & 0xFFu);
            push(nA, (theirs.rA & 8u) ? 2 * t : 2 * t + 1);
          }
        }
      }
    }
    __syncwarp();
    const uint32_t n_edges = ws.n_edges;
    if (n_edges > kEdgeCap) { overflow = true; break; }

    // Phase C: propagate the minimum node id over the edges until nothing changes (exact for any cluster size).
    if (n_edges) {
      for (;;) {
        bool changed = false;
        for (uint32_t j = lane; j < n_edges; j += 32) {
          const uint32_t uv = edges[j];
          const uint32_t u = uv & 0xFFFFu, v = uv >> 16;
          const uint16_t lu = lab[u], lv = lab[v];
          if (lu < lv) { lab[v] = lu; changed = true; }
          else if (lv < lu) { lab[u] = lv; changed = true; }
        }
        __syncwarp();
        if (!__any_sync(kFull, changed)) break;
      }
    }

    // Phase D1: roots take cluster slots (ballot order) and store their own sums; cidmap[node] = slot.
    const uint32_t n_cl_before = n_cl;
    uint32_t has_child = 0;  // chunks in which this lane's SP has a non-root component
    for (uint32_t i0 = 0, chunk = 0; i0 < cnt; i0 += 32, ++chunk) {
      const uint32_t i = i0 + lane;
      const bool live = i < cnt && !(absorbed >> chunk & 1u);
      uint32_t slot = 0, h = 0, C = 0, R = 0;
      Comps mine{0, 0};
      if (live) {
        const uint32_t w = __ldg(sp + off + i);
        R = (w >> 8) & 0x3Fu; C = (w >> 14) & 0x1FFu;
        slot = (uint32_t)lookup(tab, (C << 6) | R);
        h = tab[slot] & 0xFFu;
        mine = split_rows(h);
      }
      const bool rootA = live && lab[2 * slot] == 2 * slot;
      const bool rootB = live && mine.rB && lab[2 * slot + 1] == 2 * slot + 1;
      const uint32_t ballotA = __ballot_sync(kFull, rootA), ballotB = __ballot_sync(kFull, rootB);
      const uint32_t cidA = n_cl + __popc(ballotA & lanemask_lt());
      const uint32_t cidB = n_cl + __popc(ballotA) + __popc(ballotB & lanemask_lt());
      n_cl += __popc(ballotA) + __popc(ballotB);
      if (live && (!rootA || (mine.rB && !rootB))) has_child |= 1u << chunk;
      if (n_cl > kClCap) { overflow = true; break; }
      if (rootA) {
        const Stats s = comp_stats<kChecksum>(h & (mine.rA | (mine.rA << 4)), C, R, g.n_cols);
        ws.ckey[cidA] = (sensor << 18) | s.minpix; ws.cn[cidA] = s.n; ws.ccol[cidA] = s.sum_col; ws.crow[cidA] = s.sum_row;
        if (kChecksum) ws.ccks[cidA] = s.cks;
        cidmap[2 * slot] = (uint16_t)cidA;
      }
      if (rootB) {
        const Stats s = comp_stats<kChecksum>(h & (mine.rB | (mine.rB << 4)), C, R, g.n_cols);
        ws.ckey[cidB] = (sensor << 18) | s.minpix; ws.cn[cidB] = s.n; ws.ccol[cidB] = s.sum_col; ws.crow[cidB] = s.sum_row;
        if (kChecksum) ws.ccks[cidB] = s.cks;
        cidmap[2 * slot + 1] = (uint16_t)cidB;
      }
    }
    if (overflow) break;
    __syncwarp();
    // Phase D2: non-root components add their sums to the root's slot.
    const uint32_t any_child = __reduce_or_sync(kFull, has_child);
    for (uint32_t i = lane, chunk = 0; i < cnt && (any_child >> chunk); i += 32, ++chunk) {
      if (!(has_child >> chunk & 1u)) continue;
      const uint32_t w = __ldg(sp + off + i);
      const uint32_t R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
      const uint32_t slot = (uint32_t)lookup(tab, (C << 6) | R);
      const uint32_t h = tab[slot] & 0xFFu;
      const Comps mine = split_rows(h);
#pragma unroll
      for (int comp = 0; comp < 2; ++comp) {
        const uint32_t rows = comp ? mine.rB : mine.rA;
        const uint32_t node = 2 * slot + comp;
        if (!rows || lab[node] == node) continue;
        const uint32_t cid = cidmap[lab[node]];
        const Stats s = comp_stats<kChecksum>(h & (rows | (rows << 4)), C, R, g.n_cols);
        atomicMin(&ws.ckey[cid], (sensor << 18) | s.minpix);
        atomicAdd(&ws.cn[cid], s.n);
        atomicAdd(&ws.ccol[cid], s.sum_col);
        atomicAdd(&ws.crow[cid], s.sum_row);
        if (kChecksum) atomicAdd(&ws.ccks[cid], s.cks);
      }
    }
    __syncwarp();
    (void)n_cl_before;
  }

  if (__any_sync(kFull, bad_sp) && lane == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_BAD_SP);
  if (overflow) {
    if (lane == 0) {
      atomicOr(a.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
      a.counts[item] = 0;
      a.slab_base[item] = slab0;
    }
    return;
  }

  // ---------------- A3 + A4: position, phi16, rank by (phi16, key) ----------------
  uint32_t* cnt256 = ws.scratch;                                            // u32[256]
  uint16_t* tmp = reinterpret_cast<uint16_t*>(ws.scratch + 256);            // u16[kClCap]
  uint16_t* order = tmp + kClCap;                                           // u16[kClCap]
  uint16_t* phis = order + kClCap;                                          // u16[kClCap] phi16 + 32768
  for (uint32_t s = lane; s < 256; s += 32) cnt256[s] = 0;
  __syncwarp();
  for (uint32_t c = lane; c < n_cl; c += 32) {
    float x, y, z;
    cluster_position(ws.cn[c], ws.ccol[c], ws.crow[c], g.pitch, g.ltg + 9 * (ws.ckey[c] >> 18), x, y, z);
    const uint16_t p = (uint16_t)((uint16_t)phi16_of(x, y) ^ 0x8000u);
    phis[c] = p;
    atomicAdd(&cnt256[p >> 8], 1u);
  }
  __syncwarp();
  {  // exclusive scan of the 256 bucket counts: 8 per lane + warp scan
    uint32_t v[8], sum = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { v[q] = cnt256[lane * 8 + q]; sum += v[q]; }
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(kFull, incl, d);
      if (lane >= (uint32_t)d) incl += t;
    }
    uint32_t run = incl - sum;
#pragma unroll
    for (int q = 0; q < 8; ++q) { cnt256[lane * 8 + q] = run; run += v[q]; }
  }
  __syncwarp();
  for (uint32_t c = lane; c < n_cl; c += 32) tmp[atomicAdd(&cnt256[phis[c] >> 8], 1u)] = (uint16_t)c;
  __syncwarp();
  for (uint32_t j = lane; j < n_cl; j += 32) {
    const uint32_t c = tmp[j];
    const uint32_t b = phis[c] >> 8;
    const uint32_t start = b ? cnt256[b - 1] : 0, end = cnt256[b];
    const unsigned long long mine = ((unsigned long long)phis[c] << 32) | ws.ckey[c];
    uint32_t rank = 0;
    for (uint32_t q = start; q < end; ++q) {
      const uint32_t o = tmp[q];
      rank += (((unsigned long long)phis[o] << 32) | ws.ckey[o]) < mine;
    }
    order[start + rank] = (uint16_t)c;
  }
  __syncwarp();

  // ---------------- write the layer in the normative order (coalesced) ----------------
  for (uint32_t j = lane; j < n_cl; j += 32) {
    const uint32_t c = order[j];
    const uint32_t key = ws.ckey[c], n = ws.cn[c], sc = ws.ccol[c], sr = ws.crow[c];
    float x, y, z;
    cluster_position(n, sc, sr, g.pitch, g.ltg + 9 * (key >> 18), x, y, z);
    const uint32_t o = slab0 + j;
    a.slab.key[o] = key;
    a.slab.n_pixels[o] = n;
    a.slab.sum_col[o] = sc;
    a.slab.sum_row[o] = sr;
    a.slab.x[o] = x;
    a.slab.y[o] = y;
    a.slab.z[o] = z;
    a.slab.phi16[o] = (int16_t)(phis[c] ^ 0x8000u);
    if (kChecksum) a.slab.checksum[o] = ws.ccks[c];
  }
  if (lane == 0) {
    a.counts[item] = n_cl;
    a.slab_base[item] = slab0;
  }
}

}  // namespace

cudaError_t launch_cluster(const ClusterLaunch& a, cudaStream_t stream) {
  const uint32_t items = a.n_events * a.geo.n_layers;
  if (items == 0) return cudaSuccess;
  const uint32_t grid = (items + kWarps - 1) / kWarps;
  cudaError_t err;
  if (a.with_checksum) {
    const size_t smem = sizeof(WarpSmem<true>) * kWarps;
    err = cudaFuncSetAttribute(velo_cluster_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    velo_cluster_kernel<true><<<grid, kWarps * 32, smem, stream>>>(a);
  } else {
    const size_t smem = sizeof(WarpSmem<false>) * kWarps;
    err = cudaFuncSetAttribute(velo_cluster_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    velo_cluster_kernel<false><<<grid, kWarps * 32, smem, stream>>>(a);
  }
  return cudaGetLastError();
}

}  // namespace velo
