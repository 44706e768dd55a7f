// Search by triplet (A5 seeding, A6 forwarding, A7 clone/ghost killing), straight-line fit (A8) and the cluster half of
// the output compaction (A9) for the common case (busiest layer <= 256 hits): one small CTA of four warps per event
// ("a single event is assigned to one block, while intra-event parallelism is mapped to the threads within one
// block") — SURVEY.md §8(a); the algorithm is DESIGN.md reading R5 (T1..T5) of P:181-183 ("forming seeds of three hits
// from consecutive layers ('triplets'), and then extending these to the other layers"; "sort hits on every layer by phi
// for fast look-up") and R6 of P:149.
//
// What the ncu captures decided (profiles/README.md).  Round 1 gave every thread a phi window to walk: 16 of 32 lanes
// active, 154 k warp instructions per event, barrier stalls on top.  Here the work of a phase is FLATTENED:
//  * a phi window is an index range of the sorted layer (256-bucket table + a walk of 0-2 hits for each end), never
//    walked hit by hit by one thread;
//  * the candidates of up to 32 windows are laid end to end (warp scan of the window lengths) and taken 32 at a time,
//    one lane per candidate; the window a candidate belongs to is found from a 32-bit mask of the window starts inside
//    the current group of 32 (one warp OR-reduction + a population count), the window's data come from a slot in shared
//    memory;
//  * seeding is two such expansions, nested: middle hits b -> (b, a) doublets (slopes, slope cut) -> (b, a, c)
//    candidates (scatter); forwarding is one: active tracks -> (track, c) candidates.  Both end in a 64-bit
//    shared-memory atomicMin on the packed key (bits(S) << 32 | indices), so the result is the oracle's whatever the order.
// One warp per event with this scheme was exact but bound by its own latency (27 % issue utilisation at the ten warps per
// SM the shared memory allows); the four warps of a CTA therefore split every phase: each owns a quarter of the middle
// hits or a segment of the active tracks (its own slots, so a warp synchronises with __syncwarp inside a phase), and
// they meet at block barriers between the phases of an iteration: [T1 forward (two warps carry the active tracks; a
// third lists the unused middle hits)] [T2 resolve] [T3 seed: the unused middle hits in equal shares] [T4 resolve by
// warp 0 | the other three warps stage the next layer and move it to the compacted output].
//
// Three instances by staging capacity (256 / 512 / 1024 hits per layer; 27 / 53 / 103 kB of shared memory); every event
// is taken by the smallest one that holds its busiest layer (classify_events_kernel).  An event that runs out of
// active-track or triplet slots is redone by the second pass of velo_track.cu.  Same results in every case
// (tests/test_gpu_parity.py).
#include "velo_track.cuh"

namespace velo {
namespace {

constexpr int kWBuckets = 256;  // phi look-up table per layer: first hit of every 256-unit slice of phi16
constexpr uint32_t kNone16 = 0xFFFFu;

// Staging capacity (hits per layer), warps per event, warps that carry active tracks (T1, T2), active tracks per track
// warp, triplets (one per middle hit) per iteration.  The warps per event grow with the shared memory an event needs, so
// that an SM keeps about 32 warps whatever the instance.
template <int kCap_, int kW_, int kTW_, int kSeg_, int kTrip_, int kLevel_>
struct FlatCfg {
  static constexpr int kCap = kCap_, kW = kW_, kTW = kTW_, kSeg = kSeg_, kTrip = kTrip_, kLevel = kLevel_;
  static constexpr int kThreads = 32 * kW_;
};
using Flat256 = FlatCfg<256, 4, 4, 64, 96, 0>;
using Flat512 = FlatCfg<512, 8, 8, 64, 192, 1>;
using Flat1024 = FlatCfg<1024, 16, 8, 128, 384, 2>;

struct __align__(16) WarpScratch {
  uint4 bslot[32];              // T3: middle hits of the current group that have doublets
  uint4 dslot[32];              // scorer: base segments (tracks or doublets) of the current group
  unsigned long long best[32];  // scorer: argmin per track / per middle hit of the current group
};

template <class C>
struct __align__(16) FlatSmem {
  static constexpr int kCap = C::kCap, kSeg = C::kSeg, kTrip = C::kTrip;
  Hit rec[3 * kCap];                    // ring of three layers: layer l lives in rec[(l % 3) * kCap ...]
  unsigned long long claim[kCap];       // T1/T2: forward claims on the hits of layer C; T3/T4: triplet of every unused b
  WarpScratch ws[C::kW];
  unsigned long long trip_key[kTrip];   // T4: bits(S) << 32 | a_local << 16 | c_local, ascending b
  float ttx[C::kTW][kSeg], tty[C::kTW][kSeg]; // active tracks: slopes of the last segment (older -> newest hit)
  uint32_t tstate[C::kTW][kSeg];           // newest hit (event-local) << 16 | weak_ok << 15 | n_hits << 8 | missed
  uint16_t tseed[C::kTW][kSeg];            // track_key: event-local index of the seed's middle hit
  uint16_t tcid[C::kTW][kSeg];             // order of creation within the event
  uint16_t fsel[C::kTW][kSeg];             // hit of layer C chosen in T1 (kNone16: none)
  uint16_t trip_b[kTrip];
  uint16_t ub[kCap];                    // layer-local indices of the unused hits of layer B, ascending
  uint16_t bucket[3][kWBuckets + 2];
  uint32_t lo[kMaxLayers + 1];          // first cluster of every layer, relative to the event
  uint32_t src[kMaxLayers];             // first slab entry of every layer
  uint32_t n_seg[C::kTW];                  // active tracks of every track warp
  uint32_t n_ub;                        // unused hits of layer B
  uint32_t n_created;                   // tracks created so far
  uint32_t overflow;                    // out of track slots / triplet slots: the event is redone elsewhere
  uint32_t scan_tot[C::kW];
  uint32_t next_event;
};
static_assert(sizeof(FlatSmem<Flat256>) + 1024 <= 227 * 1024 / 8, "eight events per SM");
static_assert(sizeof(FlatSmem<Flat512>) + 1024 <= 227 * 1024 / 4, "four events per SM");
static_assert(sizeof(FlatSmem<Flat1024>) + 1024 <= 227 * 1024 / 2, "two events per SM");

__device__ __forceinline__ uint32_t lanemask_le() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
  return m;
}

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(kFull, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}

// First index in [0, n) of the layer (sorted by signed phi16) with phi >= target, or n.
__device__ __forceinline__ uint32_t lower_bound_phi(const uint16_t* __restrict__ bucket, const Hit* __restrict__ rec,
                                                    uint32_t n, int target) {
  uint32_t idx = bucket[(uint32_t)(target + 32768) >> 8];
#pragma unroll 1
  while (idx < n && phi_of(rec[idx].w) < target) ++idx;
  return idx;
}

// The hits of a layer with |dphi16(hit, ph)| <= w as a circular index range: `first`, then `count` hits (indices modulo
// n).  w <= 16383 (checked at create), so the window is shorter than the circle and wraps at most once.
__device__ __forceinline__ void phi_window(const uint16_t* __restrict__ bucket, const Hit* __restrict__ rec, uint32_t n,
                                           int ph, int w, uint32_t& first, uint32_t& count) {
  const int tl = ph - w, th = ph + w;
  const bool wrapped = tl < -32768 || th > 32767;
  const uint32_t lo = lower_bound_phi(bucket, rec, n, wrap16(tl));
  const int thw = wrap16(th);
  const uint32_t hi = thw == 32767 ? n : lower_bound_phi(bucket, rec, n, thw + 1);
  first = lo;
  count = wrapped ? n - lo + hi : hi - lo;
}

template <class C>
struct Ctx {
  const TrackLaunch& a;
  FlatSmem<C>& sm;
  uint32_t lane, warp;
};

// Hit q (event-local index) that has left the ring (only tracks that skipped more than one layer): from the slab.
template <class C>
__device__ __forceinline__ Hit far_hit(const Ctx<C>& c, uint32_t q, uint32_t first_layer) {
  uint32_t l = first_layer;
#pragma unroll 1
  while (q >= c.sm.lo[l + 1]) ++l;
  const uint4 r = __ldg(c.a.slab.rec + c.sm.src[l] + (q - c.sm.lo[l]));
  Hit h;
  h.x = __uint_as_float(r.x); h.y = __uint_as_float(r.y); h.z = __uint_as_float(r.z); h.w = r.w;
  return h;
}

// Layer l: slab -> ring slot l % 3 (with its phi table) and -> its final place in the compacted cluster output, by a
// team of `n_team` warps of which this one is number `member` (groups of 32 hits in turn).
template <bool kStage, class C>
__device__ __forceinline__ void stage_and_copy_layer(const Ctx<C>& c, uint32_t l, uint32_t co, uint32_t member,
                                                     uint32_t n_team) {
  const TrackLaunch& a = c.a;
  FlatSmem<C>& sm = c.sm;
  const uint32_t lane = c.lane;
  const uint32_t base = sm.src[l], n = sm.lo[l + 1] - sm.lo[l], dst = co + sm.lo[l];
  Hit* rec = sm.rec + (l % 3) * C::kCap;
  uint16_t* bucket = sm.bucket[l % 3];
  if (n == 0) {
    if (kStage && member == 0)
#pragma unroll 1
      for (uint32_t b = lane; b <= (uint32_t)kWBuckets; b += 32) bucket[b] = 0;
    return;
  }
#pragma unroll 1
  for (uint32_t k0 = member * 32; k0 < n; k0 += 32 * n_team) {
    const uint32_t k = k0 + lane;
    int bk = kWBuckets;
    if (k < n) {
      const uint4 r = __ldg(a.slab.rec + base + k), q = __ldg(a.slab.info + base + k);
      if (kStage) *reinterpret_cast<uint4*>(&rec[k]) = r;
      const uint32_t d = dst + k;
      a.clusters.key[d] = q.x; a.clusters.n_pixels[d] = q.y; a.clusters.sum_col[d] = q.z; a.clusters.sum_row[d] = q.w;
      a.clusters.x[d] = __uint_as_float(r.x); a.clusters.y[d] = __uint_as_float(r.y); a.clusters.z[d] = __uint_as_float(r.z);
      a.clusters.phi16[d] = (int16_t)(uint16_t)r.w;
      if (a.clusters.checksum) a.clusters.checksum[d] = __ldg(a.slab.checksum + base + k);
      bk = (int)(((r.w & 0xFFFFu) ^ 0x8000u) >> 8);
    }
    if (kStage) {  // bucket[b] = first hit whose phi slice is >= b: every hit fills the slices since its predecessor's
      int bp = __shfl_up_sync(kFull, bk, 1);
      if (lane == 0) bp = k0 ? (int)(((__ldg(reinterpret_cast<const uint32_t*>(a.slab.rec + base + k0 - 1) + 3) & 0xFFFFu) ^ 0x8000u) >> 8) : -1;
      if (k < n)
#pragma unroll 1
        for (int b = bp + 1; b <= bk; ++b) bucket[b] = (uint16_t)k;
      if (k0 + 32 >= n) {  // the group with the last hit also fills the slices behind it
        const int last_bk = __shfl_sync(kFull, bk, n - 1u - k0);
#pragma unroll 1
        for (int b = last_bk + 1 + (int)lane; b <= kWBuckets; b += 32) bucket[b] = (uint16_t)n;
      }
    }
  }
}

// Ask the L2 for the slab lines of layer l (staged one iteration later).
template <class C>
__device__ __forceinline__ void prefetch_layer(const Ctx<C>& c, uint32_t l) {
  const uint32_t base = c.sm.src[l], n = c.sm.lo[l + 1] - c.sm.lo[l];
  const char* r = reinterpret_cast<const char*>(c.a.slab.rec + base);
  const char* q = reinterpret_cast<const char*>(c.a.slab.info + base);
#pragma unroll 1
  for (uint32_t o = threadIdx.x * 128u; o < n * 16u; o += (uint32_t)C::kThreads * 128u) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(r + o));
    asm volatile("prefetch.global.L2 [%0];" ::"l"(q + o));
  }
}

// The scorer.  Every lane brings one base segment (a track's last segment in T1, an (a, b) doublet in T3): slopes tx, ty,
// the ring position `qref` of the newer hit, its window on layer C as (c_first, n) — n = 0 for a lane without a segment —
// the high key bits `idbits` (low 16 bits clear) and the slot of best[] its result goes to.  The n candidates of all
// lanes are laid end to end and taken 32 at a time, one lane per candidate: normative scatter (R5), cut, and
// the packed key bits(S) << 32 | idbits | c_local into best[slot] by atomicMin.  The whole warp must call it.
template <bool kCheckUsed>
__device__ __forceinline__ void score_windows(const Hit* __restrict__ ring, WarpScratch& ws, uint32_t lane,
                                              const Hit* __restrict__ recC, uint32_t nC, float cut, uint32_t n,
                                              uint32_t c_first, float tx, float ty, uint32_t qref, uint32_t idbits,
                                              uint32_t slot) {
  const uint32_t incl = warp_incl_scan(n, lane);
  const uint32_t total = __shfl_sync(kFull, incl, 31);
  if (total == 0) return;
  const uint32_t p = incl - n;  // position of this lane's first candidate
  const uint32_t nonempty = __ballot_sync(kFull, n != 0);
  if (n)
    ws.dslot[__popc(nonempty & lanemask_lt())] =
        make_uint4(__float_as_uint(tx), __float_as_uint(ty), idbits | qref, c_first | (slot << 10) | (p << 15));
  __syncwarp();
  uint32_t before = 0;  // segments that start before the current group of 32 candidates
#pragma unroll 1
  for (uint32_t j0 = 0; j0 < total; j0 += 32) {
    const uint32_t rel = p - j0;  // < 32 iff this lane's window starts inside the group
    const uint32_t starts = __reduce_or_sync(kFull, (n != 0 && rel < 32u) ? (1u << rel) : 0u);
    const uint32_t owner = before + __popc(starts & lanemask_le()) - 1u;
    before += __popc(starts);
    const uint32_t j = j0 + lane;
    if (j < total) {
      const uint4 d = ws.dslot[owner];
      uint32_t ic = (d.w & 0x3FFu) + (j - (d.w >> 15));
      if (ic >= nC) ic -= nC;
      const Hit hc = recC[ic];
      if (!kCheckUsed || !(hc.w & kUsedBit)) {
        const Hit hq = ring[d.z & 0xFFFFu];
        const float dz = __fsub_rn(hc.z, hq.z);
        const float ex = __fsub_rn(__fmaf_rn(__uint_as_float(d.x), dz, hq.x), hc.x);
        const float ey = __fsub_rn(__fmaf_rn(__uint_as_float(d.y), dz, hq.y), hc.y);
        const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
        if (S <= cut)
          atomicMin(&ws.best[(d.w >> 10) & 31u], ((unsigned long long)__float_as_uint(S) << 32) | (d.z & 0xFFFF0000u) | ic);
      }
    }
  }
  __syncwarp();  // the slots are free again, best[] is final for this call
}

template <class C>
__device__ __forceinline__ void load_offsets(const Ctx<C>& c, uint32_t e, uint32_t co) {
  const uint32_t L = c.a.geo.n_layers;
#pragma unroll 1
  for (uint32_t l = threadIdx.x; l <= L; l += C::kThreads) c.sm.lo[l] = c.a.clusters.layer_offsets[e * L + l] - co;
#pragma unroll 1
  for (uint32_t l = threadIdx.x; l < L; l += C::kThreads) c.sm.src[l] = c.a.slab_base[e * L + l];
  __syncthreads();
}

template <class C>
__device__ __forceinline__ void track_event_flat(const TrackLaunch& a, uint32_t e, FlatSmem<C>& sm) {
  constexpr uint32_t kCap = C::kCap, kSeg = C::kSeg, kTrip = C::kTrip;
  const DeviceGeometry& g = a.geo;
  const allen_velo_params_t& P = g.params;
  const uint32_t L = g.n_layers, lane = lane_id(), warp = threadIdx.x >> 5;
  const uint32_t co = a.clusters.event_offsets[e];
  const Ctx<C> c{a, sm, lane, warp};
  WarpScratch& ws = sm.ws[warp];
  if (threadIdx.x < (uint32_t)C::kTW) sm.n_seg[threadIdx.x] = 0;
  if (threadIdx.x == 0) { sm.n_created = 0; sm.overflow = 0; sm.n_ub = 0; }
  load_offsets(c, e, co);
  uint16_t* link = a.link + co;
  const uint32_t trk0 = co / 3;

  stage_and_copy_layer<true>(c, L - 1, co, warp, C::kW);
  stage_and_copy_layer<true>(c, L - 2, co, warp, C::kW);
  stage_and_copy_layer<true>(c, L - 3, co, warp, C::kW);
  if (L >= 4) prefetch_layer(c, L - 4);
  __syncthreads();

#pragma unroll 1
  for (int i = (int)L - 1; i >= 2; --i) {
    const uint32_t A0 = sm.lo[i], A1 = sm.lo[i + 1], B0 = sm.lo[i - 1], C0 = sm.lo[i - 2];
    const uint32_t nA = A1 - A0, nB = A0 - B0, nC = B0 - C0;
    const uint32_t refA = (i % 3) * kCap, refB = ((i - 1) % 3) * kCap, refC = ((i - 2) % 3) * kCap;
    Hit* recA = sm.rec + refA;
    Hit* recB = sm.rec + refB;
    Hit* recC = sm.rec + refC;
    const uint16_t* bucketA = sm.bucket[i % 3];
    const uint16_t* bucketC = sm.bucket[(i - 2) % 3];
    if (i >= 4) prefetch_layer(c, (uint32_t)i - 4);
    const bool seeding = nA != 0 && nB != 0 && nC != 0 && sm.overflow == 0;  // block-uniform: written before the last barrier
    const uint32_t n_mine = warp < (uint32_t)C::kTW ? sm.n_seg[warp] : 0u;
    uint32_t all_tracks = 0;
#pragma unroll
    for (int w = 0; w < C::kTW; ++w) all_tracks |= sm.n_seg[w];
    const bool any_track = all_tracks != 0;

    // ---- T1 forward (track warps): best hit of layer C per active track (nothing of C is used yet; claim[] is clear);
    //      claim it with (bits(S), track_key)
    if (nC) {
#pragma unroll 1
      for (uint32_t t0 = 0; t0 < n_mine; t0 += 32) {
        const uint32_t t = t0 + lane;
        uint32_t n = 0, c_first = 0, qref = 0;
        float tx = 0.f, ty = 0.f;
        bool far = false;
        Hit hq;
        if (t < n_mine) {
          const uint32_t q = sm.tstate[warp][t] >> 16;
          far = q >= A1;
          qref = q >= A0 ? refA + (q - A0) : refB + (q - B0);
          hq = far ? far_hit(c, q, (uint32_t)i + 1) : sm.rec[qref];
          tx = sm.ttx[warp][t]; ty = sm.tty[warp][t];
          phi_window(bucketC, recC, nC, phi_of(hq.w), P.w_fwd_phi16, c_first, n);
        }
        ws.best[lane] = kNoClaim;
        if (far) {  // (max_skipped >= 2 only) the last hit is not in the ring: this thread walks its window itself
          unsigned long long best = kNoClaim;
#pragma unroll 1
          for (uint32_t k = 0, ic = c_first; k < n; ++k, ++ic) {
            if (ic >= nC) ic -= nC;
            const Hit hc = recC[ic];
            const float dz = __fsub_rn(hc.z, hq.z);
            const float ex = __fsub_rn(__fmaf_rn(tx, dz, hq.x), hc.x);
            const float ey = __fsub_rn(__fmaf_rn(ty, dz, hq.y), hc.y);
            const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
            if (S <= P.s_fwd) best = min(best, ((unsigned long long)__float_as_uint(S) << 32) | ic);
          }
          ws.best[lane] = best;
          n = 0;
        }
        score_windows<false>(sm.rec, ws, lane, recC, nC, P.s_fwd, n, c_first, tx, ty, qref, 0u, lane);
        if (t < n_mine) {
          const unsigned long long bk = ws.best[lane];
          uint32_t sel = kNone16;
          if (bk != kNoClaim) {
            sel = (uint32_t)bk & 0xFFFFu;
            atomicMin(&sm.claim[sel], (bk & 0xFFFFFFFF00000000ull) | sm.tseed[warp][t]);
          }
          sm.fsel[warp][t] = (uint16_t)sel;
        }
      }
    }
    // ---- (last warp, beside T1) the unused hits of layer B, in order: its used flags are final since the last barrier
    if (warp == (uint32_t)C::kW - 1 && seeding) {
      uint32_t n_ub = 0;
#pragma unroll 1
      for (uint32_t k0 = 0; k0 < nB; k0 += 32) {
        const uint32_t k = k0 + lane;
        const bool un = k < nB && !(recB[k].w & kUsedBit);
        const uint32_t bal = __ballot_sync(kFull, un);
        if (un) sm.ub[n_ub + __popc(bal & lanemask_lt())] = (uint16_t)k;
        n_ub += __popc(bal);
      }
      if (lane == 0) sm.n_ub = n_ub;
    }
    __syncthreads();  // B1: all claims are in; ub[] is complete
    if (any_track) {
      // ---- T2 resolve (track warps): the minimal claim wins the hit (track keys are unique: the low half of the claim
      //      names the winner); everyone else counts a miss; closed tracks leave the segment, the others move up
      uint32_t kept = 0;
#pragma unroll 1
      for (uint32_t t0 = 0; t0 < n_mine; t0 += 32) {
        const uint32_t t = t0 + lane;
        bool keep = false;
        uint32_t st = 0, seed = 0, cid = 0;
        float tx = 0.f, ty = 0.f;
        if (t < n_mine) {
          st = sm.tstate[warp][t]; seed = sm.tseed[warp][t]; cid = sm.tcid[warp][t];
          tx = sm.ttx[warp][t]; ty = sm.tty[warp][t];
          const uint32_t fc = nC ? sm.fsel[warp][t] : kNone16;
          if (fc != kNone16 && ((uint32_t)sm.claim[fc] & 0xFFFFu) == seed) {
            const uint32_t q = st >> 16;
            const Hit hq = q >= A1 ? far_hit(c, q, (uint32_t)i + 1) : q >= A0 ? recA[q - A0] : recB[q - B0];
            const Hit hc = recC[fc];
            const float dz = __fsub_rn(hc.z, hq.z);
            tx = __fdiv_rn(__fsub_rn(hc.x, hq.x), dz);
            ty = __fdiv_rn(__fsub_rn(hc.y, hq.y), dz);
            recC[fc].w = hc.w | kUsedBit;
            link[C0 + fc] = (uint16_t)q;
            st = ((C0 + fc) << 16) | (st & 0x8000u) | ((track_n_hits(st) + 1u) << 8);
            keep = true;
          } else {
            const uint32_t m = (st & 0xFFu) + 1u;
            if (m > (uint32_t)P.max_skipped) {
              a.trk_final[trk0 + cid] = st;
            } else {
              st = (st & 0xFFFFFF00u) | m;
              keep = true;
            }
          }
        }
        const uint32_t bal = __ballot_sync(kFull, keep);
        __syncwarp();  // every lane of the group has read its state: positions <= t0 + 31 may be overwritten
        if (keep) {
          const uint32_t pos = kept + __popc(bal & lanemask_lt());
          sm.tstate[warp][pos] = st; sm.tseed[warp][pos] = (uint16_t)seed; sm.tcid[warp][pos] = (uint16_t)cid;
          sm.ttx[warp][pos] = tx; sm.tty[warp][pos] = ty;
        }
        kept += __popc(bal);
      }
      if (lane == 0 && warp < (uint32_t)C::kTW) sm.n_seg[warp] = kept;
      __syncthreads();  // B2: used flags of layer C are final for the seeding
    }

    // ---- T3 seed: every unused middle hit b of layer B: argmin over unused a in A and c in C inside b's phi windows
    //      of (bits(S), a, c), subject to the slope cut on a -> b and S <= s_seed.  The warps take equal shares of ub[] and
    //      leave the triplet of ub[u] (or "none") in claim[u].
    const uint32_t n_ub = seeding ? sm.n_ub : 0u;
    if (n_ub) {
      const uint32_t passes = (n_ub + 32 * C::kW - 1) / (32 * C::kW), per = (n_ub + passes * C::kW - 1) / (passes * C::kW);
#pragma unroll 1
      for (uint32_t chunk = warp; chunk < passes * C::kW; chunk += C::kW) {
        const uint32_t u = chunk * per + lane, u_end = min(n_ub, (chunk + 1) * per);
        uint32_t kb = 0, nd = 0, a_first = 0, c_first = 0, c_n = 0;
        if (u < u_end) {
          kb = sm.ub[u];
          const int phb = phi_of(recB[kb].w);
          phi_window(bucketC, recC, nC, phb, P.w_seed_phi16, c_first, c_n);
          if (c_n) phi_window(bucketA, recA, nA, phb, P.w_seed_phi16, a_first, nd);
        }
        ws.best[lane] = kNoClaim;
        // (b, a) doublets of the group, laid end to end; one lane per doublet
        const uint32_t incl = warp_incl_scan(nd, lane);
        const uint32_t total = __shfl_sync(kFull, incl, 31);
        if (total) {
          const uint32_t p = incl - nd;
          const uint32_t nonempty = __ballot_sync(kFull, nd != 0);
          if (nd) ws.bslot[__popc(nonempty & lanemask_lt())] = make_uint4(kb | (lane << 16), a_first, c_first | (c_n << 16), p);
          __syncwarp();
          uint32_t before = 0;
#pragma unroll 1
          for (uint32_t j0 = 0; j0 < total; j0 += 32) {
            const uint32_t rel = p - j0;
            const uint32_t starts = __reduce_or_sync(kFull, (nd != 0 && rel < 32u) ? (1u << rel) : 0u);
            const uint32_t owner = before + __popc(starts & lanemask_le()) - 1u;
            before += __popc(starts);
            const uint32_t j = j0 + lane;
            uint32_t n = 0, cf = 0, idbits = 0, slot = 0, qref = 0;
            float tx = 0.f, ty = 0.f;
            if (j < total) {
              const uint4 bs = ws.bslot[owner];
              uint32_t ia = bs.y + (j - bs.w);
              if (ia >= nA) ia -= nA;
              const Hit ha = recA[ia];
              if (!(ha.w & kUsedBit)) {
                qref = refB + (bs.x & 0xFFFFu);
                const Hit hb = sm.rec[qref];
                const float dz_ab = __fsub_rn(hb.z, ha.z);
                tx = __fdiv_rn(__fsub_rn(hb.x, ha.x), dz_ab);
                ty = __fdiv_rn(__fsub_rn(hb.y, ha.y), dz_ab);
                if (fabsf(tx) <= P.max_slope && fabsf(ty) <= P.max_slope) {
                  n = bs.z >> 16; cf = bs.z & 0xFFFFu; idbits = ia << 16; slot = bs.x >> 16;
                }
              }
            }
            score_windows<true>(sm.rec, ws, lane, recC, nC, P.s_seed, n, cf, tx, ty, qref, idbits, slot);
          }
        }
        __syncwarp();
        if (u < u_end) sm.claim[u] = ws.best[lane];
      }
    }
    __syncthreads();  // B3: the triplets of all middle hits are in claim[]

    if (warp == 0) {
      // ---- T4 resolve (warp 0): a triplet is accepted iff it holds the minimal key (bits(S), b) among the triplets
      //      that contain its a, and likewise its c; accepted -> new active track [a, b, c], in ascending b
      uint32_t n_trip = 0;
#pragma unroll 1
      for (uint32_t u0 = 0; u0 < n_ub; u0 += 32) {
        const uint32_t u = u0 + lane;
        const unsigned long long bk = u < n_ub ? sm.claim[u] : kNoClaim;
        const bool found = bk != kNoClaim;
        const uint32_t bal = __ballot_sync(kFull, found);
        if (found) {
          const uint32_t pos = n_trip + __popc(bal & lanemask_lt());
          if (pos < kTrip) { sm.trip_key[pos] = bk; sm.trip_b[pos] = sm.ub[u]; }
        }
        n_trip += __popc(bal);
      }
      __syncwarp();
      if (n_trip > kTrip) {
        if (lane == 0) sm.overflow = 1;
        n_trip = 0;
      }
      uint32_t n_created = sm.n_created;
#pragma unroll 1
      for (uint32_t c0 = 0; c0 < n_trip; c0 += 32) {
        const uint32_t ti = c0 + lane;
        const bool valid = ti < n_trip;
        const unsigned long long key = valid ? sm.trip_key[ti] : 0ull;
        const uint32_t kb = valid ? sm.trip_b[ti] : 0u;
        const uint32_t ia = ((uint32_t)key >> 16) & 0xFFFFu, ic = (uint32_t)key & 0xFFFFu;
        const unsigned long long tkey = (key & 0xFFFFFFFF00000000ull) | (B0 + kb);
        bool acc = valid;
        bool conflicts = n_trip > 1;
        if (n_trip <= 32) {  // one group: does any triplet share its a or its c with another one?
          const uint32_t act = __ballot_sync(kFull, valid);
          uint32_t others = 0;
          if (valid) others = (__match_any_sync(act, ia) | __match_any_sync(act, ic)) & ~(1u << lane);
          conflicts = __any_sync(kFull, others != 0);
        }
        if (conflicts) {
#pragma unroll 1
          for (uint32_t j = 0; j < n_trip; ++j) {
            const unsigned long long kj = sm.trip_key[j];
            const uint32_t aj = ((uint32_t)kj >> 16) & 0xFFFFu, cj = (uint32_t)kj & 0xFFFFu;
            const unsigned long long okey = (kj & 0xFFFFFFFF00000000ull) | (B0 + sm.trip_b[j]);
            if (j != ti && (aj == ia || cj == ic) && okey < tkey) acc = false;
          }
        }
        const uint32_t bal = __ballot_sync(kFull, acc);
        const uint32_t n_acc = __popc(bal);
        if (acc) {
          // tracks are dealt to the track warps' segments in turn, by order of creation
          const uint32_t r = __popc(bal & lanemask_lt()), cid = n_created + r;
          const uint32_t seg = cid % C::kTW, first_r = (seg + C::kTW - n_created % C::kTW) % C::kTW;
          const uint32_t slot = sm.n_seg[seg] + (r - first_r) / C::kTW;
          if (slot < kSeg) {
            const Hit hb = recB[kb], hc = recC[ic];
            const float dz = __fsub_rn(hc.z, hb.z);
            sm.ttx[seg][slot] = __fdiv_rn(__fsub_rn(hc.x, hb.x), dz);
            sm.tty[seg][slot] = __fdiv_rn(__fsub_rn(hc.y, hb.y), dz);
            const float S = __uint_as_float((uint32_t)(key >> 32));
            sm.tstate[seg][slot] = ((C0 + ic) << 16) | (S <= P.s_weak ? 0x8000u : 0u) | (3u << 8);
            sm.tseed[seg][slot] = (uint16_t)(B0 + kb);
            sm.tcid[seg][slot] = (uint16_t)cid;
            link[B0 + kb] = (uint16_t)(A0 + ia);
            link[C0 + ic] = (uint16_t)(B0 + kb);
            // layer A leaves the ring after this iteration: its used flags are never read again
            recB[kb].w = hb.w | kUsedBit;
            recC[ic].w = hc.w | kUsedBit;
          } else {
            sm.overflow = 1;  // out of track slots: redone by the second pass
          }
        }
        __syncwarp();
        if (lane < (uint32_t)C::kTW && n_acc) {  // lane s: tracks that went to segment s
          const uint32_t first_r = (lane + C::kTW - n_created % C::kTW) % C::kTW;
          if (first_r < n_acc) sm.n_seg[lane] = min(sm.n_seg[lane] + (n_acc - first_r + C::kTW - 1) / C::kTW, kSeg);
        }
        n_created += n_acc;
        __syncwarp();
      }
      if (lane == 0) sm.n_created = n_created;
      // claim[] for the next T1
      const uint32_t nC_next = i >= 3 ? sm.lo[i - 2] - sm.lo[i - 3] : 0u;
#pragma unroll 1
      for (uint32_t k = lane; k < nC_next; k += 32) sm.claim[k] = kNoClaim;
    } else if (i >= 3) {
      // ---- (warps 1-3) layer A leaves; its ring slot takes the layer the next iteration needs as C
      stage_and_copy_layer<true>(c, (uint32_t)i - 3, co, warp - 1, C::kW - 1);
    }
    __syncthreads();  // B4
  }

  if (sm.overflow) {  // the second pass of velo_track.cu redoes the event (its clusters are in the output now)
    if (threadIdx.x == 0) {
      constexpr int which = C::kLevel == 2 ? 1 : 0;
      a.redo_list[which][atomicAdd(a.counters + 2 + which, 1u)] = e;
    }
    return;
  }

  // ---- the tracks still active are closed
  if (warp < (uint32_t)C::kTW) {
    const uint32_t n_mine = sm.n_seg[warp];
#pragma unroll 1
    for (uint32_t t = lane; t < n_mine; t += 32) a.trk_final[trk0 + sm.tcid[warp][t]] = sm.tstate[warp][t];
  }
  __syncthreads();

  // ---- T5 finalise + A8 fit, in order of creation: keep >= 4 hits, or 3 hits with S_seed <= s_weak
  const uint32_t n_created = sm.n_created;
  uint32_t out_tracks = 0, out_hits = 0;
#pragma unroll 1
  for (uint32_t base = 0; base < n_created; base += C::kThreads) {
    const uint32_t t = base + threadIdx.x;
    uint32_t n = 0, st = 0;
    if (t < n_created) {
      st = __ldcg(a.trk_final + trk0 + t);
      n = track_n_hits(st);
      if (n == 3 && !(st & 0x8000u)) n = 0;
    }
    const uint32_t v = n ? ((1u << 20) | n) : 0u;
    const uint32_t incl = warp_incl_scan(v, lane);
    if (lane == 31) sm.scan_tot[warp] = incl;
    __syncthreads();
    uint32_t off = incl - v, total = 0;
#pragma unroll
    for (int w = 0; w < C::kW; ++w) {
      const uint32_t u = sm.scan_tot[w];
      if (w < (int)warp) off += u;
      total += u;
    }
    __syncthreads();
    if (n) {
      const uint32_t ot = out_tracks + (off >> 20), oh = out_hits + (off & 0xFFFFFu);
      // hits in order of addition: walk the links from the newest hit backwards
      uint16_t* out_h = a.hits_slab + co + oh;
      uint32_t h = st >> 16;
#pragma unroll 1
      for (int k = (int)n - 1; k >= 0; --k) {
        out_h[k] = (uint16_t)h;
        if (k) h = link[h];
      }
      // A8: the oracle's operations in the oracle's order (R6: fp64 means, then centred sums, over the hits
      // in order of addition, from the fp32 coordinates) -> bit-identical parameters.  Coordinates from the slab records
      // (one 16-byte load per hit); the hits go down in layers, so the layer of a hit is found by walking down.
      const double dn = (double)n;
      double zm = 0, xm = 0, ym = 0;
      uint32_t l = L - 1;
#pragma unroll 1
      for (uint32_t k = 0; k < n; ++k) {
        h = out_h[k];
#pragma unroll 1
        while (h < sm.lo[l]) --l;
        const uint4 r = __ldg(a.slab.rec + sm.src[l] + (h - sm.lo[l]));
        zm += (double)__uint_as_float(r.z); xm += (double)__uint_as_float(r.x); ym += (double)__uint_as_float(r.y);
      }
      zm /= dn; xm /= dn; ym /= dn;
      double szz = 0, szx = 0, szy = 0;
      l = L - 1;
#pragma unroll 1
      for (uint32_t k = 0; k < n; ++k) {
        h = out_h[k];
#pragma unroll 1
        while (h < sm.lo[l]) --l;
        const uint4 r = __ldg(a.slab.rec + sm.src[l] + (h - sm.lo[l]));
        const double dz = (double)__uint_as_float(r.z) - zm;
        szz += dz * dz;
        szx += dz * ((double)__uint_as_float(r.x) - xm);
        szy += dz * ((double)__uint_as_float(r.y) - ym);
      }
      const double tx = szx / szz, ty = szy / szz;
      a.trk_hitoff[trk0 + ot] = oh;
      a.trk_fit[trk0 + ot] = make_float4((float)(xm - tx * zm), (float)(ym - ty * zm), (float)tx, (float)ty);
    }
    out_tracks += total >> 20;
    out_hits += total & 0xFFFFFu;
  }
  if (threadIdx.x == 0) a.counts[e] = ((unsigned long long)out_tracks << 32) | out_hits;
}

// One CTA of four warps per event of class kClsFlat, in four size bins, largest first; it also moves the clusters of
// copy-only events.
template <class C>
__global__ void __launch_bounds__(C::kThreads, 1024 / C::kThreads) velo_track_flat_kernel(const __grid_constant__ TrackLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FlatSmem<C>& sm = *reinterpret_cast<FlatSmem<C>*>(smem_raw);
  uint32_t j = blockIdx.x, bin = 0;
#pragma unroll 1
  for (; bin < 4; ++bin) {
    const uint32_t n = a.counters[8 + bin];
    if (j < n) break;
    j -= n;
  }
  if (bin == 4) return;
  const uint32_t e = a.order[(size_t)bin * a.n_events + j];
  const uint8_t cls = a.level[e];
  if (cls == kClsCopy) {
    const uint32_t co = a.clusters.event_offsets[e], L = a.geo.n_layers;
    const Ctx<C> c{a, sm, lane_id(), threadIdx.x >> 5};
    load_offsets(c, e, co);
#pragma unroll 1
    for (uint32_t l = 0; l < L; ++l) stage_and_copy_layer<false>(c, l, co, threadIdx.x >> 5, C::kW);
    return;
  }
  if (cls != kClsFlat) return;
  track_event_flat<C>(a, e, sm);
}

// Larger instances: a few resident CTAs take events from a list (most nu = 6 batches have few of them).
template <class C>
__global__ void __launch_bounds__(C::kThreads, 1024 / C::kThreads) velo_track_flat_list_kernel(const __grid_constant__ TrackLaunch a,
                                                                        const uint32_t* __restrict__ list,
                                                                        const uint32_t* __restrict__ count,
                                                                        uint32_t* cursor) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FlatSmem<C>& sm = *reinterpret_cast<FlatSmem<C>*>(smem_raw);
  const uint32_t n = *count;
#pragma unroll 1
  for (;;) {
    if (threadIdx.x == 0) sm.next_event = atomicAdd(cursor, 1u);
    __syncthreads();
    const uint32_t idx = sm.next_event;
    if (idx >= n) return;
    track_event_flat<C>(a, list[idx], sm);
    __syncthreads();
  }
}

}  // namespace

cudaError_t track_flat_prepare() {
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  cudaError_t err = cudaFuncSetAttribute(velo_track_flat_kernel<Flat256>, attr, (int)sizeof(FlatSmem<Flat256>));
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_track_flat_list_kernel<Flat512>, attr, (int)sizeof(FlatSmem<Flat512>));
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_track_flat_list_kernel<Flat1024>, attr, (int)sizeof(FlatSmem<Flat1024>));
  return err;
}

// Events of class kClsFlat (and copy-only events): one CTA each.
cudaError_t launch_track_flat(const TrackLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  velo_track_flat_kernel<Flat256><<<a.n_events, Flat256::kThreads, sizeof(FlatSmem<Flat256>), stream>>>(a);
  return cudaGetLastError();
}

// Events of class kClsMid (which = 0) / kClsLarge (which = 1), from their lists.
cudaError_t launch_track_flat_list(const TrackLaunch& a, uint32_t which, uint32_t grid, cudaStream_t stream) {
  if (a.n_events == 0 || grid == 0) return cudaSuccess;
  if (which == 0)
    velo_track_flat_list_kernel<Flat512><<<grid, Flat512::kThreads, sizeof(FlatSmem<Flat512>), stream>>>(a, a.ev_list[0], a.counters + 0, a.counters + 4);
  else
    velo_track_flat_list_kernel<Flat1024><<<grid, Flat1024::kThreads, sizeof(FlatSmem<Flat1024>), stream>>>(a, a.ev_list[1], a.counters + 1, a.counters + 5);
  return cudaGetLastError();
}

}  // namespace velo
