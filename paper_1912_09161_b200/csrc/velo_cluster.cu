// Kernel 1 of the VELO hot path: raw decode (A1), exact connected-component clustering (A2), centroid -> global
// position and phi16 (A3), the per-layer phi sort (A4) and the placement of the layer in the compacted output (A9) —
// SURVEY.md §8(a); definitions DESIGN.md R1-R4; paper P:153 (decoding), P:179 (clustering as connected component
// labelling), P:183 (sort hits on every layer by phi), P:136 (sizes stay on the device).
//
// Work decomposition: ONE WARP per (event, layer).  Clustering is independent per sensor (R2) and the sort is
// independent per layer (R4), so a warp needs no block-level barrier: everything below synchronises with
// __syncwarp / warp votes only, and the warps of a CTA are fully decoupled.
//
// Clustering without a pixel grid: the nodes of the graph are "SP components" — a 2x4 super-pixel holds at most two
// 8-connected components (pixels in adjacent rows of a 2-wide block always touch, so components are runs of occupied
// rows).  The super-pixels of the layer's sensors are staged in shared memory and put into one open-addressing hash
// table keyed by (sensor, sp_col, sp_row); each SP looks up only its four "forward" neighbours (col+1: row-1, row,
// row+1; col: row+1), and only those its border pixels can touch.  Touching components become edges; labels (node
// ids) are propagated over the edge list to the minimum until nothing changes, which is exact for any cluster size.
// Roots get cluster slots by warp ballot (no atomics); non-root components add their integer sums to the root's slot
// with shared-memory atomics (commutative integer adds / min: deterministic).
//
// The layer's clusters are ranked by (phi16, key) with a 256-bucket counting sort on the top byte of phi plus an exact
// in-bucket rank and written, coalesced and in the normative order, as two 16-byte records per cluster, to the layer's
// region of a slab whose position depends only on the event's bank table (the position of the layer's first SP word;
// the rare layer with more clusters than SP words takes a region behind that dense part): warps never wait for one another.
// (A decoupled look-back over the 260 k (event, layer) items that wrote the compacted output directly was measured
// first: in-order publication made every warp wait for its slowest predecessor — 66 % of the issued instructions
// were the spin — so compaction moved into the track kernel, which reads every hit anyway; profiles/README.md.)
//
// Capacities.  The kernel is instantiated for 128, 256 and 512 SP words / clusters / edges per layer in shared memory
// (4.6 / 9.2 / 18 kB per warp).  Every layer is clustered by the smallest instance that holds it (FAST): an instance
// appends the layers that are too large for it to a list, and the next larger one takes that list with resident warps.
// Beyond 512: MID — every sensor of the layer fits: one pass per sensor group in shared memory, cluster records and
// sort scratch in a pool slot in global memory; BIG — everything in a (larger) pool slot in global memory.  Same code,
// same results, decreasing speed; a layer is flagged STAGE_OVERFLOW only if it
// holds more than 8192 SP words.  MID slots belong to resident warps (per-SM bit masks), so they never run out and
// nobody waits for one; BIG slots are taken from a bit mask for the time of one item and given back (a warp that finds
// none free waits for one), so their number bounds concurrency, not the batch.
#include "velo_common.cuh"

namespace velo {
namespace {

constexpr int kWarps = 4;  // warps per CTA (independent work items) of the 128-entry instance
// (the 256-entry instance over ALL items, which busy batches start with, is 2 % faster with two warps per CTA: 4.11 against
// 4.19 ms at nu = 12; the list instances and the 128-entry instance are faster with four)
template <uint32_t kCap> struct WarpsOf { static constexpr int v = kCap <= 128 ? kWarps : 2; };
constexpr uint32_t kDescWords = 18;  // per (event, layer) descriptor written by velo_prepare_kernel
// per-warp shared memory
// kCap SP words / clusters / edges per layer, 2 * kCap hash slots; two instances: 256 (nu ~ 6) and 512 (busier batches)
template <uint32_t kCap>
struct Caps {
  static constexpr uint32_t kHashBits = kCap == 128 ? 8 : kCap == 256 ? 9 : 10;
  static constexpr uint32_t kLevel = kCap == 128 ? 0 : 1;  // deferral list an instance with kDefer appends to
  static_assert(kCap == 128 || kCap == 256 || kCap == 512, "hash bits");
};
// pool slots in global memory
constexpr uint32_t kMidCl = 1024;
constexpr uint32_t kBigSp = 8192, kBigHashBits = 14, kBigEdges = 7 * kBigSp, kBigCl = 2 * kBigSp;

// Storage of one clustering pass.  Staged SP word: hitmap | sp_row << 8 | sp_col << 14 | local sensor << 23; 0 = dead.
struct Pass {
  uint32_t* sp;     // [cap_sp]
  uint32_t* tab;    // [1 << hash_bits] entries (key << 14) | (index + 1), 0 = empty; key = staged word bits 25:8
  uint16_t* lab;    // [2 * cap_sp] label of node 2 * index + component
  uint32_t* edges;  // [cap_edges] u | v << 16; reused as cidmap u16[2 * cap_sp] once the labels are final
  uint32_t hash_bits, cap_sp, cap_edges;
};
struct ClusterStore {  // cluster records of the whole layer
  uint32_t *key, *n, *col, *row, *cks;
  uint32_t cap;
};
struct SortStore {
  uint32_t* cnt256;             // [256]
  uint16_t *tmp, *order, *phis; // [cap] each; phis = phi16 + 32768
  float* uv;                    // [2][cap] local coordinates kept between ranking and writing, or nullptr (recompute)
  uint32_t cap;
};

__device__ __forceinline__ uint32_t hash_slot(uint32_t key, uint32_t bits) { return (key * 0x9E3779B1u) >> (32 - bits); }

// Index of the staged SP with `key`, or -1.
__device__ __forceinline__ int lookup(const uint32_t* tab, uint32_t bits, uint32_t key) {
  const uint32_t mask = (1u << bits) - 1u;
  uint32_t s = hash_slot(key, bits);
#pragma unroll 1
  for (;;) {
    const uint32_t e = tab[s];
    if (e == 0) return -1;
    if ((e >> 14) == key) return (int)(e & 0x3FFFu) - 1;
    s = (s + 1) & mask;
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
#pragma unroll 1
    while (mm) {
      const uint32_t b = __ffs(mm) - 1;
      mm &= mm - 1;
      s.cks += mix32((4 * R + (b & 3u)) * n_cols + 2 * C + (b >> 2));
    }
  }
  return s;
}

// One clustering pass over the sensors [k0, k1) of the layer (lane k holds sensor k's id and bank range): stage,
// insert, find edges, propagate labels, give roots cluster ids from n_cl upwards and accumulate the cluster records.
// Returns false if a capacity of `p` or `cs` is exceeded (the caller retries with larger storage).
template <bool kChecksum>
__device__ __forceinline__ bool ccl_pass(const Pass& p, const ClusterStore& cs, const DeviceGeometry& g,
                                         const uint32_t* __restrict__ spw, uint32_t my_sensor, uint32_t my_off,
                                         uint32_t my_cnt, uint32_t k0, uint32_t k1, uint32_t& n_cl, bool& bad_sp,
                                         uint32_t* n_edges_ctr, bool sparse) {
  const uint32_t lane = lane_id();
  const uint32_t bits = p.hash_bits;
  // ---- stage the SP words of the group (R1: addresses outside the sensor are ignored and flagged).  The group is
  //      one flat index range; four loads per lane are in flight before the first is used.
  const uint32_t in_group = (lane >= k0 && lane < k1) ? my_cnt : 0u;
  uint32_t incl = in_group;
#pragma unroll
  for (int d = 1; d < 8; d <<= 1) {  // at most kMaxSensorsPerLayer = 8 lanes carry counts
    const uint32_t t = __shfl_up_sync(kFull, incl, d);
    if (lane >= (uint32_t)d) incl += t;
  }
  const uint32_t my_start = incl - in_group;                 // first staged index of sensor `lane`
  const uint32_t n = __shfl_sync(kFull, incl, (k1 - 1) & 31);  // staged words of the group
  uint32_t start_of[kMaxSensorsPerLayer];  // first staged index of every sensor of the group; "never" outside it
#pragma unroll
  for (int kk = 0; kk < kMaxSensorsPerLayer; ++kk) {
    const uint32_t st = __shfl_sync(kFull, my_start, kk);
    start_of[kk] = ((uint32_t)kk > k0 && (uint32_t)kk < k1) ? st : 0xFFFFFFFFu;
  }
  auto stage_word = [&](uint32_t i, uint32_t w) {  // staged index i (< n), raw word w
    uint32_t k = k0;
#pragma unroll
    for (int kk = 1; kk < kMaxSensorsPerLayer; ++kk) k += i >= start_of[kk];
    const uint32_t R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
    uint32_t staged = (w & 0x7FFFFFu) | (k << 23);
    if ((w & 0xFFu) == 0) staged = 0;
    if (C >= g.sp_cols || R >= g.sp_rows) { bad_sp = true; staged = 0; }
    p.sp[i] = staged;
  };
  // The banks of a layer's sensors usually follow one another in the raw event (G0: sensors 4k .. 4k+3): the group is
  // then ONE range of SP words, read with 128-bit loads (ld.global.nc.v4: the SP area of an event starts on a 16-byte
  // boundary and is padded to one, R1), two loads per lane in flight.  Otherwise word by word.
  const uint32_t has = __ballot_sync(kFull, in_group != 0);
  const uint32_t rel = my_off - my_start;  // raw position of staged index 0, if the group is one range
  const uint32_t g0 = __shfl_sync(kFull, rel, has ? __ffs(has) - 1 : 0);
  if (__all_sync(kFull, in_group == 0 || rel == g0)) {
    const uint32_t a0 = g0 & ~3u;
    const uint4* __restrict__ v4 = reinterpret_cast<const uint4*>(spw + a0);
    const uint32_t nv = n ? ((g0 + n + 3u) >> 2) - (a0 >> 2) : 0u;
    const int skew = (int)(a0 - g0);  // staged index of the first word of vector 0 (<= 0)
#pragma unroll 1
    for (uint32_t v0 = 0; v0 < nv; v0 += 64) {
      const uint32_t va = v0 + lane, vb = v0 + 32 + lane;
      uint4 wa = make_uint4(0, 0, 0, 0), wb = wa;
      if (va < nv) wa = __ldg(v4 + va);
      if (vb < nv) wb = __ldg(v4 + vb);
      const uint32_t ua[4] = {wa.x, wa.y, wa.z, wa.w}, ub[4] = {wb.x, wb.y, wb.z, wb.w};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int ia = skew + (int)(4 * va) + u, ib = skew + (int)(4 * vb) + u;
        if (va < nv && ia >= 0 && ia < (int)n) stage_word((uint32_t)ia, ua[u]);
        if (vb < nv && ib >= 0 && ib < (int)n) stage_word((uint32_t)ib, ub[u]);
      }
    }
  } else {
#pragma unroll 1
    for (uint32_t i0 = 0; i0 < n; i0 += 128) {
      uint32_t w[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const uint32_t i = i0 + 32 * u + lane;
        uint32_t k = k0;
#pragma unroll
        for (int kk = 1; kk < kMaxSensorsPerLayer; ++kk) k += i >= start_of[kk];
        const uint32_t src = __shfl_sync(kFull, my_off, k) + (i - __shfl_sync(kFull, my_start, k));
        w[u] = i < n ? __ldg(spw + src) : 0u;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const uint32_t i = i0 + 32 * u + lane;
        if (i < n) stage_word(i, w[u]);
      }
    }
  }
  {
    uint4* tab4 = reinterpret_cast<uint4*>(p.tab);  // 16-byte aligned in every storage
#pragma unroll 1
    for (uint32_t s = lane; s < (1u << bits) / 4; s += 32) tab4[s] = make_uint4(0, 0, 0, 0);
  }
  if (lane == 0) *n_edges_ctr = 0;
  __syncwarp();

  // ---- isolated super-pixels (most of them at nu = 6: two thirds of the fired pixels are noise).  A super-pixel with no
  //      other super-pixel in the coarse cells around it (1 SP column x 32 SP rows per cell; a bit map of the occupied
  //      cells and one of the cells holding more than one SP, in the cluster-record arrays, which are free until the
  //      roots are numbered) has no neighbour: it needs no hash entry and no look-up, its components are roots.  Only the
  //      others are listed (ballot) and go through insert and edges below: two rounds of 32 instead of five for a typical
  //      layer.  The test is conservative (cells are folded modulo kOccCells; a far SP in a neighbouring cell only costs
  //      the slow path), and symmetric for true neighbours, so every neighbour of a listed SP is listed too.
  constexpr uint32_t kOccCells = 4096, kOccWords = kOccCells / 32;
  uint16_t* nz = nullptr;
  uint32_t n_nz = n;
  if (sparse) {
    uint32_t* occ = cs.key;              // (sparse: the caller's records are in shared memory and n_cl == 0)
    uint32_t* multi = cs.key + kOccWords;
    nz = reinterpret_cast<uint16_t*>(cs.key + 2 * kOccWords);
#pragma unroll 1
    for (uint32_t s = lane; s < 2 * kOccWords; s += 32) occ[s] = 0;
    __syncwarp();
    // cell of (sensor k, SP column C, band = SP row / 32) = bit 2 * (k * sp_cols + C) + band: the six cells around an SP
    // (columns C-1 .. C+1, two bands) are six consecutive bits.  (Column -1 / sp_cols of a sensor is a column of its
    // neighbour in the numbering, and the numbering is folded modulo kOccCells: both only ever add occupied cells.)
    auto base_of = [&](uint32_t w) { return 2u * ((w >> 23) * g.sp_cols + ((w >> 14) & 0x1FFu)); };
#pragma unroll 1
    for (uint32_t i = lane; i < n; i += 32) {
      const uint32_t w = p.sp[i];
      if (!w) continue;
      const uint32_t cell = (base_of(w) + (((w >> 8) & 0x3Fu) >> 5)) & (kOccCells - 1u);
      const uint32_t bit = 1u << (cell & 31u);
      if (atomicOr(&occ[cell >> 5], bit) & bit) atomicOr(&multi[cell >> 5], bit);
    }
    __syncwarp();
    n_nz = 0;
#pragma unroll 1
    for (uint32_t i0 = 0; i0 < n; i0 += 32) {
      const uint32_t i = i0 + lane;
      const uint32_t w = i < n ? p.sp[i] : 0u;
      bool listed = false;
      if (w) {
        const uint32_t R = (w >> 8) & 0x3Fu, band = R >> 5;
        const uint32_t own = (base_of(w) + band) & (kOccCells - 1u);
        const uint32_t first = (base_of(w) - 2u) & (kOccCells - 1u);  // cell (C-1, band 0); even
        const uint32_t wi = first >> 5, sh = first & 31u;
        const uint32_t win = __funnelshift_r(occ[wi], occ[(wi + 1) & (kOccWords - 1u)], sh) & 0x3Fu;
        // neighbours in the same band: columns C-1 and C+1; in the other band (only if row R-1 or R+1 lies there): all three
        const bool crosses = (R >= 1 && ((R - 1) >> 5) != band) || (R + 1 < g.sp_rows && ((R + 1) >> 5) != band);
        const uint32_t near = (0x11u << band) | (crosses ? (0x15u << (1u - band)) : 0u);
        listed = (win & near) != 0 || ((multi[own >> 5] >> (own & 31u)) & 1u) != 0;
      }
      const uint32_t bal = __ballot_sync(kFull, listed);
      if (listed) nz[n_nz + __popc(bal & lanemask_lt())] = (uint16_t)i;
      n_nz += __popc(bal);
    }
    VELO_CHECK(g, n_nz <= n && 4 * (2 * kOccWords) + 2 * n <= 16 * cs.cap, 106);  // bit maps + list fit the record arrays
    __syncwarp();
  }

  // ---- insert: entry = key << 14 | (index + 1); a repeated address merges its hitmap into the first one (R1)
  const uint32_t mask = (1u << bits) - 1u;
#pragma unroll 1
  for (uint32_t j = lane; j < n_nz; j += 32) {
    const uint32_t i = nz ? nz[j] : j;
    const uint32_t w = p.sp[i];
    if (!w) continue;
    const uint32_t key = (w >> 8) & 0x3FFFFu;
    uint32_t s = hash_slot(key, bits);
    [[maybe_unused]] uint32_t probes = 0;
#pragma unroll 1
    for (;;) {
      VELO_CHECK(g, ++probes <= (1u << bits), 101);  // the table has twice as many slots as entries: a free one exists
      const uint32_t old = atomicCAS(p.tab + s, 0u, (key << 14) | (i + 1));
      if (old == 0) break;
      if ((old >> 14) == key) {
        atomicOr(p.sp + (old & 0x3FFFu) - 1, w & 0xFFu);
        p.sp[i] = 0;
        break;
      }
      s = (s + 1) & mask;
    }
  }
  __syncwarp();

  // ---- edges to touching forward neighbours; node = 2 * index + component
#pragma unroll 1
  for (uint32_t x = lane; x < 2 * n; x += 32) p.lab[x] = (uint16_t)x;  // (dead entries too: the pointer-jumping pass reads every label)
#pragma unroll 1
  for (uint32_t j = lane; j < n_nz; j += 32) {
    const uint32_t i = nz ? nz[j] : j;
    const uint32_t w = p.sp[i];
    const uint32_t nA = 2 * i, nB = 2 * i + 1;
    if (!w) continue;
    const uint32_t h = w & 0xFFu, R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
    const uint32_t key = (w >> 8) & 0x3FFFFu;
    const Comps mine = split_rows(h);
    auto push = [&](uint32_t u, uint32_t v) {
      const uint32_t idx = atomicAdd(n_edges_ctr, 1u);
      if (idx < p.cap_edges) p.edges[idx] = u | (v << 16);
    };
    const uint32_t r4 = mine.rA | mine.rB;
    const uint32_t n_row3 = (mine.rA & 8u) ? nA : nB;  // our component holding row 3
    // local clustering variant (R11; "locally in small regions"): edges stay inside a region of
    // 2^shift super-pixels; shift 31 (the default) puts the whole sensor in one region = exact components
    const bool same_c = ((C + 1) >> g.region_shift_c) == (C >> g.region_shift_c);
    const bool same_up = ((R + 1) >> g.region_shift_r) == (R >> g.region_shift_r);
    const bool same_dn = R >= 1 && ((R - 1) >> g.region_shift_r) == (R >> g.region_shift_r);
    // (C, R+1): our row 3 touches their row 0 whatever the columns
    if ((r4 & 8u) && R + 1 < g.sp_rows && same_up) {
      const int t = lookup(p.tab, bits, key + 1);
      if (t >= 0) {
        const uint32_t q = p.sp[t] & 0xFFu;
        if ((q | (q >> 4)) & 1u) push(n_row3, 2 * t);
      }
    }
    if (C + 1 < g.sp_cols && same_c) {
      // (C+1, R): our column-1 pixels touch their column-0 pixels within one row
      if (h & 0xF0u) {
        const int t = lookup(p.tab, bits, key + 64);
        if (t >= 0) {
          const uint32_t q = p.sp[t] & 0xFFu;
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
      if ((h & 0x80u) && R + 1 < g.sp_rows && same_up) {
        const int t = lookup(p.tab, bits, key + 65);
        if (t >= 0 && (p.sp[t] & 1u)) push(n_row3, 2 * t);
      }
      // (C+1, R-1): our pixel (dc=1, dr=0) touches their pixel (dc=0, dr=3)
      if ((h & 0x10u) && same_dn) {
        const int t = lookup(p.tab, bits, key + 63);
        if (t >= 0 && (p.sp[t] & 8u)) {
          const Comps theirs = split_rows(p.sp[t] & 0xFFu);
          push(nA, (theirs.rA & 8u) ? 2 * t : 2 * t + 1);
        }
      }
    }
  }
  __syncwarp();
  const uint32_t n_edges = *n_edges_ctr;
  if (n_edges > p.cap_edges) return false;
  VELO_CHECK(g, n <= p.cap_sp && 2 * n <= 0x10000u, 102);  // staged words fit the pass, node ids fit 16 bits

  // ---- propagate the minimum node id over the edges until nothing changes (exact for any cluster size)
  //      A label is always the id of a node of the same component and only ever decreases, so the fix point (every edge
  //      joins equal labels) gives every node the smallest id of its component.  From the third pass on every node also
  //      takes the label of its label (pointer jumping): a long thin cluster then needs O(log diameter) passes, not one
  //      pass per hop.
  if (n_edges) {
#pragma unroll 1
    for (uint32_t pass = 0;; ++pass) {
      bool changed = false;
#pragma unroll 1
      for (uint32_t j = lane; j < n_edges; j += 32) {
        const uint32_t uv = p.edges[j];
        const uint32_t u = uv & 0xFFFFu, v = uv >> 16;
        const uint16_t lu = p.lab[u], lv = p.lab[v];
        if (lu < lv) { p.lab[v] = lu; changed = true; }
        else if (lv < lu) { p.lab[u] = lv; changed = true; }
      }
      __syncwarp();
      if (!__any_sync(kFull, changed)) break;
      if (pass >= 2) {
#pragma unroll 1
        for (uint32_t x = lane; x < 2 * n; x += 32) {
          const uint16_t l = p.lab[x];
          const uint16_t ll = p.lab[l];
          if (ll < l) p.lab[x] = ll;
        }
        __syncwarp();
      }
    }
  }

  // ---- roots take cluster ids (ballot order) and store their own sums; cidmap[node] = id
  uint16_t* cidmap = reinterpret_cast<uint16_t*>(p.edges);
  bool any_child = false;
#pragma unroll 1
  for (uint32_t i0 = 0; i0 < n; i0 += 32) {
    const uint32_t i = i0 + lane;
    const uint32_t w = i < n ? p.sp[i] : 0u;
    const bool live = w != 0;
    const uint32_t h = w & 0xFFu, R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
    const uint32_t sensor = __shfl_sync(kFull, my_sensor, (w >> 23) & 7u);
    const Comps mine = split_rows(h);
    const bool rootA = live && p.lab[2 * i] == 2 * i;
    const bool rootB = live && mine.rB && p.lab[2 * i + 1] == 2 * i + 1;
    const uint32_t ballotA = __ballot_sync(kFull, rootA), ballotB = __ballot_sync(kFull, rootB);
    const uint32_t cidA = n_cl + __popc(ballotA & lanemask_lt());
    const uint32_t cidB = n_cl + __popc(ballotA) + __popc(ballotB & lanemask_lt());
    n_cl += __popc(ballotA) + __popc(ballotB);
    any_child = any_child || (live && (!rootA || (mine.rB && !rootB)));
    if (n_cl > cs.cap) return false;  // warp-uniform
    if (rootA) {
      const Stats s = comp_stats<kChecksum>(h & (mine.rA | (mine.rA << 4)), C, R, g.n_cols);
      cs.key[cidA] = (sensor << 18) | s.minpix; cs.n[cidA] = s.n; cs.col[cidA] = s.sum_col; cs.row[cidA] = s.sum_row;
      if (kChecksum) cs.cks[cidA] = s.cks;
      cidmap[2 * i] = (uint16_t)cidA;
    }
    if (rootB) {
      const Stats s = comp_stats<kChecksum>(h & (mine.rB | (mine.rB << 4)), C, R, g.n_cols);
      cs.key[cidB] = (sensor << 18) | s.minpix; cs.n[cidB] = s.n; cs.col[cidB] = s.sum_col; cs.row[cidB] = s.sum_row;
      if (kChecksum) cs.cks[cidB] = s.cks;
      cidmap[2 * i + 1] = (uint16_t)cidB;
    }
  }
  __syncwarp();
  // ---- non-root components add their sums to the root's record
  if (__any_sync(kFull, any_child)) {
#pragma unroll 1
    for (uint32_t i = lane; i < n; i += 32) {
      const uint32_t w = p.sp[i];
      if (!w) continue;
      const uint32_t h = w & 0xFFu, R = (w >> 8) & 0x3Fu, C = (w >> 14) & 0x1FFu;
      const Comps mine = split_rows(h);
#pragma unroll
      for (int comp = 0; comp < 2; ++comp) {
        const uint32_t rows = comp ? mine.rB : mine.rA;
        const uint32_t node = 2 * i + comp;
        if (!rows || p.lab[node] == node) continue;
        const uint32_t cid = cidmap[p.lab[node]];
        VELO_CHECK(g, p.lab[node] < 2 * n && cid < n_cl, 103);
        const Stats s = comp_stats<kChecksum>(h & (rows | (rows << 4)), C, R, g.n_cols);
        atomicMin(&cs.key[cid], (cs.key[cid] & ~0x3FFFFu) | s.minpix);
        atomicAdd(&cs.n[cid], s.n);
        atomicAdd(&cs.col[cid], s.sum_col);
        atomicAdd(&cs.row[cid], s.sum_row);
        if (kChecksum) atomicAdd(&cs.cks[cid], s.cks);
      }
    }
    __syncwarp();
  }
  return true;
}

// A3 + A4 for one layer whose n_cl cluster records are in `cs`: position and phi16, rank by (phi16, key), coalesced
// write in the normative order to the slab region [slab0, slab0 + n_cl).
template <bool kChecksum>
__device__ __forceinline__ void finish_layer(const ClusterLaunch& a, const ClusterStore& cs, const SortStore& ss,
                                             uint32_t item, uint32_t slab0, uint32_t region, uint32_t n_cl) {
  const DeviceGeometry& g = a.geo;
  const uint32_t lane = lane_id();
  if (n_cl > region) {  // warp-uniform: more clusters than SP words -> a region behind the dense part of the slab
    uint32_t s = 0;
    if (lane == 0) s = atomicAdd(a.slab.spill_cursor, n_cl);
    s = __shfl_sync(kFull, s, 0);
    if ((unsigned long long)a.slab.dense + s + n_cl > a.slab.capacity) {  // workspace smaller than workspace_bytes()
      if (lane == 0) atomicOr(a.status + item / g.n_layers, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
      n_cl = 0;
    } else {
      slab0 = a.slab.dense + s;
      if (lane == 0) a.slab_base[item] = slab0;  // otherwise the value velo_prepare_kernel wrote stands
    }
  }
  if (lane == 0) a.counts[item] = n_cl;
  // the phi look-up table of the layer for the track search (velo_seed.cu): first cluster of every slice of phi16
  uint4* tab = reinterpret_cast<uint4*>(a.slab.phi_tab + (size_t)item * kPhiTabStride);
  if (n_cl == 0) {
    tab[lane] = make_uint4(0, 0, 0, 0);
    if (lane == 0) tab[32] = make_uint4(0, 0, 0, 0);
    return;
  }
#pragma unroll 1
  for (uint32_t s = lane; s < 256; s += 32) ss.cnt256[s] = 0;
  __syncwarp();
#pragma unroll 1
  for (uint32_t c = lane; c < n_cl; c += 32) {
    float u, v, x, y, z;
    cluster_local(cs.n[c], cs.col[c], cs.row[c], g.pitch, u, v);
    local_to_global(u, v, g.ltg + 9 * (cs.key[c] >> 18), x, y, z);
    if (ss.uv) { ss.uv[c] = u; ss.uv[ss.cap + c] = v; }
    const uint16_t p = (uint16_t)((uint16_t)phi16_of(x, y) ^ 0x8000u);
    ss.phis[c] = p;
    atomicAdd(&ss.cnt256[p >> 8], 1u);
  }
  __syncwarp();
  {  // exclusive scan of the 256 bucket counts: 8 per lane + warp scan
    uint32_t v[8], sum = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { v[q] = ss.cnt256[lane * 8 + q]; sum += v[q]; }
    uint32_t incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(kFull, incl, d);
      if (lane >= (uint32_t)d) incl += t;
    }
    uint32_t run = incl - sum;
    uint32_t st[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { ss.cnt256[lane * 8 + q] = run; st[q] = run; run += v[q]; }
    // the exclusive sums are the table (the by-product of this sort that the track search wants): 8 entries per lane
    tab[lane] = make_uint4(st[0] | (st[1] << 16), st[2] | (st[3] << 16), st[4] | (st[5] << 16), st[6] | (st[7] << 16));
    if (lane == 0) tab[32] = make_uint4(n_cl, 0, 0, 0);
  }
  __syncwarp();
#pragma unroll 1
  for (uint32_t c = lane; c < n_cl; c += 32) ss.tmp[atomicAdd(&ss.cnt256[ss.phis[c] >> 8], 1u)] = (uint16_t)c;
  __syncwarp();
#pragma unroll 1
  for (uint32_t j = lane; j < n_cl; j += 32) {
    const uint32_t c = ss.tmp[j];
    const uint32_t b = ss.phis[c] >> 8;
    const uint32_t start = b ? ss.cnt256[b - 1] : 0, end = ss.cnt256[b];
    const unsigned long long mine = ((unsigned long long)ss.phis[c] << 32) | cs.key[c];
    uint32_t rank = 0;
#pragma unroll 1
    for (uint32_t q = start; q < end; ++q) {
      const uint32_t o = ss.tmp[q];
      rank += (((unsigned long long)ss.phis[o] << 32) | cs.key[o]) < mine;
    }
    VELO_CHECK(g, start + rank < n_cl && c < n_cl && end <= n_cl, 104);
    ss.order[start + rank] = (uint16_t)c;
  }
  __syncwarp();
#pragma unroll 1
  for (uint32_t j = lane; j < n_cl; j += 32) {
    const uint32_t c = ss.order[j];
    const uint32_t key = cs.key[c], n = cs.n[c], sc = cs.col[c], sr = cs.row[c];
    float u, v, x, y, z;
    if (ss.uv) { u = ss.uv[c]; v = ss.uv[ss.cap + c]; }
    else cluster_local(n, sc, sr, g.pitch, u, v);
    local_to_global(u, v, g.ltg + 9 * (key >> 18), x, y, z);
    const uint32_t o = slab0 + j;
    VELO_CHECK(g, o < a.slab.capacity && c < n_cl, 105);
    a.slab.rec[o] = make_uint4(__float_as_uint(x), __float_as_uint(y), __float_as_uint(z), (uint32_t)(ss.phis[c] ^ 0x8000u));
    a.slab.info[o] = make_uint4(key, n, sc, sr);
    if (kChecksum) a.slab.checksum[o] = cs.cks[c];
  }
}

// Out-of-line instances for storage in global memory (MID and BIG): generic pointers, rarely executed.
template <bool kChecksum>
__device__ __noinline__ bool ccl_pass_generic(const Pass& p, const ClusterStore& cs, const DeviceGeometry& g,
                                              const uint32_t* __restrict__ spw, uint32_t my_sensor, uint32_t my_off,
                                              uint32_t my_cnt, uint32_t k0, uint32_t k1, uint32_t& n_cl, bool& bad_sp,
                                              uint32_t* n_edges_ctr) {
  return ccl_pass<kChecksum>(p, cs, g, spw, my_sensor, my_off, my_cnt, k0, k1, n_cl, bad_sp, n_edges_ctr, false);
}
template <bool kChecksum>
__device__ __noinline__ void finish_layer_generic(const ClusterLaunch& a, const ClusterStore& cs, const SortStore& ss,
                                                  uint32_t item, uint32_t slab0, uint32_t region, uint32_t n_cl) {
  finish_layer<kChecksum>(a, cs, ss, item, slab0, region, n_cl);
}

template <bool kChecksum, uint32_t kCap>
struct alignas(16) WarpSmem {
  static constexpr uint32_t kCapSp = kCap, kCapEdges = kCap, kCapCl = kCap, kHashBits = Caps<kCap>::kHashBits;
  uint32_t sp[kCapSp];
  uint32_t tab[1u << kHashBits];
  uint16_t lab[2 * kCapSp];
  uint32_t edges[kCapEdges];
  uint32_t ckey[kCapCl], cn[kCapCl], ccol[kCapCl], crow[kCapCl];
  uint32_t ccks[kChecksum ? kCapCl : 1];
  uint32_t n_edges;
};
// sort scratch (1 kB of bucket counts, then tmp / order / phis) aliases sp + tab, for 128 entries also lab
static_assert(1024 + 6 * 128 <= 4 * 128 + 4 * (1u << 8) + 4 * 128 && 1024 + 6 * 256 <= 4 * 256 + 4 * (1u << 9) &&
                  1024 + 6 * 512 <= 4 * 512 + 4 * (1u << 10),
              "sort scratch aliases sp + tab (+ lab)");

// Layout of the pool slots (bytes from the slot base).
struct MidSlot {
  static constexpr size_t kStats = 0;                              // 5 x u32[kMidCl]
  static constexpr size_t kCnt = kStats + 5 * 4 * (size_t)kMidCl;  // u32[256]
  static constexpr size_t kSort = kCnt + 1024;                     // 3 x u16[kMidCl]
  static constexpr size_t kBytes = (kSort + 3 * 2 * (size_t)kMidCl + 255) / 256 * 256;
};
struct BigSlot {
  static constexpr size_t kSp = 0;
  static constexpr size_t kTab = kSp + 4 * (size_t)kBigSp;
  static constexpr size_t kLab = kTab + 4 * ((size_t)1 << kBigHashBits);
  static constexpr size_t kEdges = kLab + 2 * 2 * (size_t)kBigSp;
  static constexpr size_t kStats = kEdges + 4 * (size_t)kBigEdges;
  static constexpr size_t kCnt = kStats + 5 * 4 * (size_t)kBigCl;
  static constexpr size_t kSort = kCnt + 1024;
  static constexpr size_t kCtr = kSort + 3 * 2 * (size_t)kBigCl;   // u32 edge counter
  static constexpr size_t kBytes = (kCtr + 4 + 255) / 256 * 256;
};

__device__ __forceinline__ void stores_at(unsigned char* base, size_t stats, size_t cnt, size_t sort, uint32_t cap,
                                          ClusterStore& cs, SortStore& ss) {
  uint32_t* s = reinterpret_cast<uint32_t*>(base + stats);
  cs.key = s; cs.n = s + cap; cs.col = s + 2 * cap; cs.row = s + 3 * cap; cs.cks = s + 4 * cap; cs.cap = cap;
  ss.cnt256 = reinterpret_cast<uint32_t*>(base + cnt);
  uint16_t* t = reinterpret_cast<uint16_t*>(base + sort);
  ss.tmp = t; ss.order = t + cap; ss.phis = t + 2 * cap;
  ss.uv = nullptr; ss.cap = cap;
}

// Everything for one (event, layer) item, by one warp.  kDefer: layers that do not fit this instance's shared memory
// are put on a list for the instance with 512 entries (launched next) instead of taking the pool paths here.
template <bool kChecksum, uint32_t kCap, bool kDefer>
__device__ __forceinline__ void cluster_item(const ClusterLaunch& a, WarpSmem<kChecksum, kCap>& ws, uint32_t item) {
  constexpr uint32_t kCapSp = kCap, kCapEdges = kCap, kCapCl = kCap, kHashBits = Caps<kCap>::kHashBits;
  const DeviceGeometry& g = a.geo;
  const uint32_t lane = lane_id();
  const uint32_t L = g.n_layers;
  const uint32_t e = item / L, layer = item % L;

  ClusterStore cs;
  cs.key = ws.ckey; cs.n = ws.cn; cs.col = ws.ccol; cs.row = ws.crow; cs.cks = ws.ccks; cs.cap = kCapCl;
  SortStore ss;
  ss.cnt256 = ws.sp;
  ss.tmp = reinterpret_cast<uint16_t*>(ws.sp + 256);  // sp, tab, lab, edges are contiguous
  ss.order = ss.tmp + kCapCl;
  ss.phis = ss.order + kCapCl;
  // lab + edges: 2 * kCapCl floats, dead once the cluster records exist (128 entries: the sort scratch reaches into lab)
  ss.uv = kCap == 128 ? nullptr : reinterpret_cast<float*>(ws.lab);
  ss.cap = kCapCl;

  // ---------------- A1: the layer's bank ranges, validated and laid out by velo_prepare_kernel ----------------
  const uint32_t* d = a.desc + (size_t)item * kDescWords;
  const uint32_t dv = lane < kDescWords ? __ldg(d + lane) : 0u;
  const uint32_t my_off = dv;                                        // lanes 0..7: first SP word (index into raw)
  const uint32_t my_cnt = __shfl_sync(kFull, dv, (lane & 7u) + 8u);  // lanes 0..7: SP words of sensor k
  const uint32_t slab0 = __shfl_sync(kFull, dv, 16);
  if (__shfl_sync(kFull, dv, 17) & 1u) {  // malformed event (BAD_HEADER set by the prepare kernel): no clusters
    finish_layer<kChecksum>(a, cs, ss, item, 0, 0, 0);
    return;
  }
  const uint32_t* spw = a.raw;
  const uint32_t K = __ldg(g.layer_n_sensors + layer);
  const uint32_t my_sensor = lane < K ? __ldg(g.layer_sensors + layer * kMaxSensorsPerLayer + lane) : 0u;
  const uint32_t cnt_k = lane < K ? my_cnt : 0u;
  const uint32_t n_sp_layer = __reduce_add_sync(kFull, cnt_k);
  const uint32_t max_cnt = __reduce_max_sync(kFull, cnt_k);
  if ((unsigned long long)slab0 + n_sp_layer > a.slab.dense) {  // workspace smaller than workspace_bytes()
    if (lane == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
    finish_layer<kChecksum>(a, cs, ss, item, 0, 0, 0);
    return;
  }

  Pass fast;
  fast.sp = ws.sp; fast.tab = ws.tab; fast.lab = ws.lab; fast.edges = ws.edges;
  fast.hash_bits = kHashBits; fast.cap_sp = kCapSp; fast.cap_edges = kCapEdges;

  uint32_t n_cl = 0;
  bool bad_sp = false, overflow = false;
  int mode = n_sp_layer <= kCapSp ? 0 : (max_cnt <= kCapSp && n_sp_layer <= kMidCl) ? 1 : 2;
  if (kDefer && mode != 0) {
    if (lane == 0) a.defer_list[Caps<kCap>::kLevel][atomicAdd(a.defer_count + 2 * Caps<kCap>::kLevel, 1u)] = item;
    return;
  }
  if (mode == 0) {
    if (ccl_pass<kChecksum>(fast, cs, g, spw, my_sensor, my_off, cnt_k, 0, K, n_cl, bad_sp, &ws.n_edges, true)) {
      if (__any_sync(kFull, bad_sp) && lane == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_BAD_SP);
      finish_layer<kChecksum>(a, cs, ss, item, slab0, n_sp_layer, n_cl);
      return;
    }
    // more clusters or edges than the warp's shared memory holds (not seen on physics-like input): the next larger
    // instance takes the layer; the last one uses a slot of the big pool
    if (kDefer) {
      if (lane == 0) a.defer_list[Caps<kCap>::kLevel][atomicAdd(a.defer_count + 2 * Caps<kCap>::kLevel, 1u)] = item;
      return;
    }
    mode = 2;
  }
  uint32_t held = 0xFFFFFFFFu;  // mid slot of this warp (released at the end)
  if (mode == 1) {
    // one slot per resident warp: bit b of mid_mask[sm] <-> slot 32 * sm + b.  A kernel with at most 32 resident warps
    // per SM always finds a free bit, so nobody ever waits for a slot.
    uint32_t slot = 0xFFFFFFFFu;
    if (lane == 0) {
      uint32_t sm;
      asm volatile("mov.u32 %0, %%smid;" : "=r"(sm));
      if (sm < a.n_mid_sms) {
#pragma unroll 1
        for (;;) {
          const uint32_t free_bits = ~*reinterpret_cast<volatile uint32_t*>(a.mid_mask + sm);
          if (!free_bits) break;
          const uint32_t b = __ffs(free_bits) - 1;
          if (!(atomicOr(a.mid_mask + sm, 1u << b) >> b & 1u)) { slot = 32 * sm + b; break; }
        }
      }
    }
    slot = __shfl_sync(kFull, slot, 0);
    if (slot == 0xFFFFFFFFu) {
      mode = 2;
    } else {
      held = slot;
      unsigned char* base = a.mid_pool + (size_t)slot * MidSlot::kBytes;
      stores_at(base, MidSlot::kStats, MidSlot::kCnt, MidSlot::kSort, kMidCl, cs, ss);
      n_cl = 0;
      bad_sp = false;
      bool ok = true;
#pragma unroll 1
      for (uint32_t k0 = 0; k0 < K && ok;) {  // greedy groups of consecutive sensors that fit the shared memory
        uint32_t k1 = k0, sum = 0;
#pragma unroll 1
        while (k1 < K) {
          const uint32_t cnt = __shfl_sync(kFull, cnt_k, k1);
          if (sum + cnt > kCapSp) break;
          sum += cnt;
          ++k1;
        }
        ok = ccl_pass_generic<kChecksum>(fast, cs, g, spw, my_sensor, my_off, cnt_k, k0, k1, n_cl, bad_sp, &ws.n_edges);
        k0 = k1;
      }
      if (!ok) mode = 2;
    }
  }
  uint32_t held_big = 0xFFFFFFFFu;  // big slot of this warp (released at the end)
  if (mode == 2) {
    // a slot of the big pool: bit b of big_mask[w] <-> slot 32 * w + b, taken for the time of this item.  If all are
    // taken the warp waits: holders never wait for anything, so a slot always comes back.
    uint32_t slot = 0xFFFFFFFFu;
    if (lane == 0 && n_sp_layer <= kBigSp) {
      const uint32_t words = (a.n_big_slots + 31) / 32;
#pragma unroll 1
      while (slot == 0xFFFFFFFFu) {
#pragma unroll 1
        for (uint32_t w = 0; w < words && slot == 0xFFFFFFFFu; ++w) {
          const uint32_t valid = (w + 1) * 32 <= a.n_big_slots ? 0xFFFFFFFFu : (1u << (a.n_big_slots & 31u)) - 1u;
          const uint32_t free_bits = ~*reinterpret_cast<volatile uint32_t*>(a.big_mask + w) & valid;
          if (!free_bits) continue;
          const uint32_t b = __ffs(free_bits) - 1;
          if (!(atomicOr(a.big_mask + w, 1u << b) >> b & 1u)) slot = 32 * w + b;
        }
        if (slot == 0xFFFFFFFFu) __nanosleep(500);
      }
    }
    slot = __shfl_sync(kFull, slot, 0);
    if (slot == 0xFFFFFFFFu) {  // beyond kBigSp super-pixels in one layer
      overflow = true;
    } else {
      held_big = slot;
      unsigned char* base = a.big_pool + (size_t)slot * BigSlot::kBytes;
      Pass big;
      big.sp = reinterpret_cast<uint32_t*>(base + BigSlot::kSp);
      big.tab = reinterpret_cast<uint32_t*>(base + BigSlot::kTab);
      big.lab = reinterpret_cast<uint16_t*>(base + BigSlot::kLab);
      big.edges = reinterpret_cast<uint32_t*>(base + BigSlot::kEdges);
      big.hash_bits = kBigHashBits; big.cap_sp = kBigSp; big.cap_edges = kBigEdges;
      stores_at(base, BigSlot::kStats, BigSlot::kCnt, BigSlot::kSort, kBigCl, cs, ss);
      n_cl = 0;
      bad_sp = false;
      overflow = !ccl_pass_generic<kChecksum>(big, cs, g, spw, my_sensor, my_off, cnt_k, 0, K, n_cl, bad_sp,
                                              reinterpret_cast<uint32_t*>(base + BigSlot::kCtr));
    }
  }
  if (overflow) {
    if (lane == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
    n_cl = 0;
  } else if (__any_sync(kFull, bad_sp) && lane == 0) {
    atomicOr(a.status + e, ALLEN_VELO_STATUS_BAD_SP);
  }
  finish_layer_generic<kChecksum>(a, cs, ss, item, slab0, n_sp_layer, n_cl);
  __syncwarp();
  if (held != 0xFFFFFFFFu && lane == 0) atomicAnd(a.mid_mask + (held >> 5), ~(1u << (held & 31u)));
  if (held_big != 0xFFFFFFFFu && lane == 0) {
    __threadfence();  // this warp is done with the slot's memory before the next holder starts
    atomicAnd(a.big_mask + (held_big >> 5), ~(1u << (held_big & 31u)));
  }
}


// Every warp takes kItemsPerWarp items of the batch, in grid order (more than one item per warp, or resident warps
// taking items from a counter, was measured: no gain at 10 000 events, a loss at 1 000).
constexpr uint32_t kItemsPerWarp = 1;
template <bool kChecksum, uint32_t kCap, bool kDefer>
__global__ void __launch_bounds__(WarpsOf<kCap>::v * 32, kCap <= 128 ? 11 : 1) velo_cluster_kernel(const __grid_constant__ ClusterLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using WS = WarpSmem<kChecksum, kCap>;
  WS& ws = reinterpret_cast<WS*>(smem_raw)[threadIdx.x >> 5];
  const uint32_t n = a.n_events * a.geo.n_layers;
#pragma unroll 1
  for (uint32_t r = 0; r < kItemsPerWarp; ++r) {
    constexpr uint32_t w = WarpsOf<kCap>::v;
    const uint32_t item = (blockIdx.x * kItemsPerWarp + r) * w + (threadIdx.x >> 5);
    if (item >= n) return;
    cluster_item<kChecksum, kCap, kDefer>(a, ws, item);
    __syncwarp();
  }
}

// Resident warps take the deferred items of list `kFrom` (a few per cent of the layers at most for the last list).
template <bool kChecksum, uint32_t kCap, bool kDefer, uint32_t kFrom>
__global__ void __launch_bounds__(kWarps * 32) velo_cluster_list_kernel(const __grid_constant__ ClusterLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  using WS = WarpSmem<kChecksum, kCap>;
  WS& ws = reinterpret_cast<WS*>(smem_raw)[threadIdx.x >> 5];
  const uint32_t n = a.defer_count[2 * kFrom];
#pragma unroll 1
  for (;;) {
    uint32_t idx = 0;
    if (lane_id() == 0) idx = atomicAdd(a.defer_count + 2 * kFrom + 1, 1u);
    idx = __shfl_sync(kFull, idx, 0);
    if (idx >= n) return;
    cluster_item<kChecksum, kCap, kDefer>(a, ws, a.defer_list[kFrom][idx]);
    __syncwarp();
  }
}

// One warp per event: validate header and bank table once (R1), and lay out for every layer of the event what its
// cluster warp needs: desc[item] = { first SP word of each of its sensors (index into raw) [8], SP words of each [8],
// slab base, flags (bit 0: malformed event) }.  26 warps per event used to redo this validation each.
__global__ void __launch_bounds__(128) velo_prepare_kernel(const __grid_constant__ ClusterLaunch a) {
  const DeviceGeometry& g = a.geo;
  const uint32_t lane = lane_id(), L = g.n_layers;
  const uint32_t e = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (e >= a.n_events) return;
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
  if (!bad) {
#pragma unroll 1
    for (uint32_t j = lane; j < g.n_sensors; j += 32) {
      const uint32_t o0 = __ldg(tbl + j), o1 = __ldg(tbl + j + 1);
      bad = bad || o0 > o1 || (j == 0 && o0 != 0) || (j + 1 == g.n_sensors && o1 != n_sp_total);
    }
  }
  bad = __any_sync(kFull, bad);
  if (bad && lane == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_BAD_HEADER);
  const uint32_t words0 = (byte0 >> 2) + 4u + g.table_words;  // first SP word of the event in raw
  uint32_t carry = 0;                                          // SP words of the layers handled in earlier rounds
#pragma unroll 1
  for (uint32_t l0 = 0; l0 < L; l0 += 32) {
    const uint32_t l = l0 + lane;
    uint32_t off[kMaxSensorsPerLayer], cnt[kMaxSensorsPerLayer], total = 0;
    const uint32_t K = (l < L && !bad) ? __ldg(g.layer_n_sensors + l) : 0u;
#pragma unroll
    for (int k = 0; k < kMaxSensorsPerLayer; ++k) {
      off[k] = 0; cnt[k] = 0;
      if ((uint32_t)k < K) {
        const uint32_t sns = __ldg(g.layer_sensors + l * kMaxSensorsPerLayer + k);
        const uint32_t o0 = __ldg(tbl + sns), o1 = __ldg(tbl + sns + 1);
        off[k] = words0 + o0; cnt[k] = o1 - o0; total += o1 - o0;
      }
    }
    uint32_t incl = total;
#pragma unroll
    for (int dd = 1; dd < 32; dd <<= 1) {
      const uint32_t t = __shfl_up_sync(kFull, incl, dd);
      if (lane >= (uint32_t)dd) incl += t;
    }
    const uint32_t before = carry + incl - total;  // SP words of this event in the layers below l
    carry += __shfl_sync(kFull, incl, 31);
    if (l < L) {
      const uint32_t item = e * L + l;
      // one slab entry per SP word, placed by the raw position: the layers of the batch tile the dense part of the
      // slab without gaps (a layer with more clusters than SP words moves behind it, finish_layer)
      const uint32_t slab0 = bad ? 0u : words0 + before;
      uint32_t* d = a.desc + (size_t)item * kDescWords;
#pragma unroll
      for (int k = 0; k < kMaxSensorsPerLayer; ++k) { d[k] = off[k]; d[8 + k] = cnt[k]; }
      d[16] = slab0;
      d[17] = bad ? 1u : 0u;
      a.slab_base[item] = slab0;
    }
  }
}

}  // namespace

size_t cluster_mid_slot_bytes() { return MidSlot::kBytes; }
size_t cluster_big_slot_bytes() { return BigSlot::kBytes; }

template <bool kChecksum, uint32_t kCap, bool kDefer>
cudaError_t launch_cluster_instance(const ClusterLaunch& a, uint32_t grid, cudaStream_t stream) {
  constexpr uint32_t w = WarpsOf<kCap>::v;
  const size_t smem = sizeof(WarpSmem<kChecksum, kCap>) * w;
  grid = (grid * kWarps + w - 1) / w;  // (the caller counts CTAs of kWarps warps)
  velo_cluster_kernel<kChecksum, kCap, kDefer><<<grid, w * 32, smem, stream>>>(a);
  return cudaGetLastError();
}

template <bool kChecksum, uint32_t kCap, bool kDefer, uint32_t kFrom>
cudaError_t launch_cluster_list(const ClusterLaunch& a, uint32_t grid, cudaStream_t stream) {
  const size_t smem = sizeof(WarpSmem<kChecksum, kCap>) * kWarps;
  velo_cluster_list_kernel<kChecksum, kCap, kDefer, kFrom><<<grid, kWarps * 32, smem, stream>>>(a);
  return cudaGetLastError();
}

template <bool kChecksum>
cudaError_t prepare_cluster_kernels() {
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  cudaError_t err = cudaFuncSetAttribute(velo_cluster_kernel<kChecksum, 128, true>, attr, (int)sizeof(WarpSmem<kChecksum, 128>) * WarpsOf<128>::v);
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_cluster_kernel<kChecksum, 256, true>, attr, (int)sizeof(WarpSmem<kChecksum, 256>) * WarpsOf<256>::v);
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_cluster_list_kernel<kChecksum, 256, true, 0>, attr, (int)sizeof(WarpSmem<kChecksum, 256>) * kWarps);
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_cluster_list_kernel<kChecksum, 512, false, 1>, attr, (int)sizeof(WarpSmem<kChecksum, 512>) * kWarps);
  return err;
}

template <bool kChecksum>
cudaError_t launch_cluster_chain(const ClusterLaunch& a, uint32_t grid, uint32_t n_sms, uint32_t* n_launches,
                                 cudaStream_t stream) {
  cudaError_t err = launch_cluster_instance<kChecksum, 128, true>(a, (grid + kItemsPerWarp - 1) / kItemsPerWarp, stream);
  if (err != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_cluster_list<kChecksum, 256, true, 0>(a, min(grid, 6 * n_sms), stream)) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_cluster_list<kChecksum, 512, false, 1>(a, min(grid, 3 * n_sms), stream)) != cudaSuccess) return err;
  ++*n_launches;
  return cudaSuccess;
}

cudaError_t cluster_prepare() {
  cudaError_t err = prepare_cluster_kernels<true>();
  return err == cudaSuccess ? prepare_cluster_kernels<false>() : err;
}

// prepare -> cluster kernel with 128 entries per layer over all (event, layer) items -> the 256-entry instance over
// the layers that one deferred -> the 512-entry instance over the layers the second deferred.  Small layers run at
// twice the occupancy of the 256-entry instance (4.6 instead of 9.2 kB of shared memory per warp).
// `big_layers`: the batch averages more than 192 SP words per layer (caller's hint): the chain starts at 256 entries.
cudaError_t launch_cluster(const ClusterLaunch& a, bool big_layers, uint32_t n_sms, uint32_t* n_launches,
                           cudaStream_t stream) {
  *n_launches = 0;
  const uint32_t items = a.n_events * a.geo.n_layers;
  if (items == 0) return cudaSuccess;
  velo_prepare_kernel<<<(a.n_events + 3) / 4, 128, 0, stream>>>(a);
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess) return err;
  ++*n_launches;
  const uint32_t grid = (items + kWarps - 1) / kWarps;
  if (big_layers) {  // 256 -> 512
    err = a.with_checksum ? launch_cluster_instance<true, 256, true>(a, (grid + kItemsPerWarp - 1) / kItemsPerWarp, stream)
                          : launch_cluster_instance<false, 256, true>(a, (grid + kItemsPerWarp - 1) / kItemsPerWarp, stream);
    if (err != cudaSuccess) return err;
    ++*n_launches;
    const uint32_t lg = min(grid, 3 * n_sms);
    err = a.with_checksum ? launch_cluster_list<true, 512, false, 1>(a, lg, stream)
                          : launch_cluster_list<false, 512, false, 1>(a, lg, stream);
    ++*n_launches;
    return err;
  }
  return a.with_checksum ? launch_cluster_chain<true>(a, grid, n_sms, n_launches, stream)
                         : launch_cluster_chain<false>(a, grid, n_sms, n_launches, stream);
}

}  // namespace velo
