// Second pass of the track search, and the kernels around it: classification of the events, compaction of the tracks.
//
// The events the two-kernel path (velo_seed.cu + velo_follow.cu) hands on — a candidate list that outgrew its region, or
// more active tracks than velo_follow keeps — are searched here by ONE CTA per event ("a single event is assigned to one
// block, while intra-event parallelism is mapped to the threads within one block"): search by triplet (A5 seeding,
// A6 forwarding, A7 clone/ghost killing) and the straight-line fit (A8) — SURVEY.md §8(a); reading R5 (T1..T5) of
// P:181-183 and R6 of P:149.  This is the track kernel of round 1 (it applies the used flags before it looks for
// triplets, six block barriers per layer iteration), reading the compacted cluster output velo_seed.cu has filled:
//  * the three layers of an iteration live in shared memory as 16-byte hit records (x, y, z, phi16 | used << 16) in a
//    ring of three slots: one LDS.128 per candidate; the next layer is brought in with cp.async into the slot of the
//    layer that leaves, as soon as the seeding is done with it;
//  * phi look-up uses a 128-bucket start table per layer, built while the layer is staged (no binary search);
//  * S1 lists (b, a) doublets inside the phi window, S2 gives every doublet one thread that scans b's window on layer
//    C; the per-b argmin is a 64-bit shared-memory atomicMin on (bits(S), a, c);
//  * all conflict rules are order-independent minima on packed keys (bits(S) << 32 | index): no "first thread wins",
//    so the result is exactly the oracle's whatever the thread schedule;
//  * two instances by staging capacity (512 / 1024 hits per layer); one that runs out of track slots hands the event to
//    the next, the last one flags it STAGE_OVERFLOW.
#include <cuda_pipeline.h>

#include "velo_track.cuh"

namespace velo {
namespace {

constexpr int kBuckets = 128;
constexpr int kBucketShift = 9;  // 65536 / 128

template <int kThreads_, int kCap_, int kCapTracks_, int kCapDoublets_, int kLevel_, bool kLast_>
struct Cfg {
  static constexpr int kThreads = kThreads_;
  static constexpr int kCap = kCap_;            // hits of one layer staged
  static constexpr int kCapTracks = kCapTracks_;
  static constexpr int kCapDoublets = kCapDoublets_;
  static constexpr int kLevel = kLevel_;
  static constexpr bool kLast = kLast_;
  static constexpr int kBlock = kThreads;
  static constexpr int kWarps = kThreads / 32;
  static constexpr int kRoundsB = (kCap + kThreads - 1) / kThreads;
  static constexpr int kRoundsT = (kCapTracks + kThreads - 1) / kThreads;
};
// second pass for events the two-kernel path ran out of track or list slots on: their clusters are already in the output
using CfgMr = Cfg<256, 512, 1024, 4096, 1, false>;
using CfgLr = Cfg<512, 1024, 2048, 2048, 2, true>;

template <class C>
struct Smem {
  Hit rec[3][C::kCap];
  unsigned long long best[C::kCap];  // T3: per-b argmin key; T1/T2: forward claims on layer C (aliased by phase)
  unsigned long long claimA[C::kCap], claimC[C::kCap];
  uint32_t doublets[C::kCapDoublets];  // b_local | a_local << 16
  float ttx[C::kCapTracks], tty[C::kCapTracks];  // slopes of the last segment (older -> newest hit)
  uint32_t tstate[C::kCapTracks];                // newest << 16 | weak_ok << 15 | nhits << 8 | missed (0xFF: closed)
  uint16_t tseedB[C::kCapTracks];                // track_key: event-local index of the seed's middle hit
  uint16_t fsel[C::kCapTracks];                  // hit of layer C chosen by the track in T1 (0xFFFF: none)
  uint16_t bucket[3][kBuckets + 2];
  uint32_t lo[kMaxLayers + 1];
  uint32_t src[kMaxLayers];  // first entry of every layer in the arrays X, Y, Z, PHI are read from
  uint32_t warp_tot[C::kRoundsB > C::kRoundsT ? C::kRoundsB : C::kRoundsT][C::kWarps];
  uint32_t ovf[(C::kCap + 31) / 32];   // middle hits whose doublets did not all fit the list (S2 walks those itself)
  uint32_t n_doublets;
  uint32_t min_active[2];
  uint32_t flags;
  uint32_t next_event;
};

__device__ __forceinline__ int phi_of(uint32_t w) { return (int)(int16_t)(uint16_t)(w & 0xFFFFu); }

// First index in [0, n) of the layer (sorted by signed phi16) with phi >= target, or n.
__device__ __forceinline__ uint32_t lower_bound_phi(const uint16_t* __restrict__ bucket, const Hit* __restrict__ rec,
                                                    uint32_t n, int target) {
  uint32_t idx = bucket[((uint32_t)(target + 32768) & 0xFFFFu) >> kBucketShift];
#pragma unroll 1
  while (idx < n && phi_of(rec[idx].w) < target) ++idx;
  return idx;
}

__device__ __forceinline__ int wrap16(int v) { return (int)(int16_t)(uint16_t)v; }

template <class C>
__device__ __forceinline__ void tsync() { __syncthreads(); }

// The hits are read from the compacted cluster output (velo_seed.cu has filled it).
template <class C>
struct Ctx {
  Smem<C>& sm;
  const float* __restrict__ X;
  const float* __restrict__ Y;
  const float* __restrict__ Z;
  const int16_t* __restrict__ PHI;
  allen_velo_params_t P;
};

// Hit at absolute position s of the source arrays (a track's last hit that has left the ring).
template <class C>
__device__ __forceinline__ Hit far_hit(const Ctx<C>& c, uint32_t s) {
  Hit h;
  h.x = __ldg(c.X + s); h.y = __ldg(c.Y + s); h.z = __ldg(c.Z + s); h.w = (uint16_t)__ldg(c.PHI + s);
  return h;
}

// Bring layer `l` into ring slot l % 3 by cp.async (three 4-byte copies per hit from the output arrays); the bucket table
// by this thread.  Completion: __pipeline_wait_prior(0) + barrier by the caller.
template <class C>
__device__ __forceinline__ void stage_layer(const Ctx<C>& c, uint32_t l) {
  Smem<C>& sm = c.sm;
  const uint32_t base = sm.src[l], n = sm.lo[l + 1] - sm.lo[l];
  Hit* rec = sm.rec[l % 3];
  uint16_t* bucket = sm.bucket[l % 3];
  if (n == 0) {
#pragma unroll 1
    for (uint32_t b = threadIdx.x; b <= (uint32_t)kBuckets; b += C::kThreads) bucket[b] = 0;
    return;
  }
#pragma unroll 1
  for (uint32_t k = threadIdx.x; k < n; k += C::kThreads) {
    __pipeline_memcpy_async(&rec[k].x, c.X + base + k, 4);
    __pipeline_memcpy_async(&rec[k].y, c.Y + base + k, 4);
    __pipeline_memcpy_async(&rec[k].z, c.Z + base + k, 4);
    const uint32_t ph = (uint16_t)__ldg(c.PHI + base + k);
    rec[k].w = ph;
    const uint32_t ph_prev = k ? (uint16_t)__ldg(c.PHI + base + k - 1) : 0u;
    const int bk = (int)((ph ^ 0x8000u) >> kBucketShift);
    const int bp = k ? (int)((ph_prev ^ 0x8000u) >> kBucketShift) : -1;
#pragma unroll 1
    for (int b = bp + 1; b <= bk; ++b) bucket[b] = (uint16_t)k;
    if (k + 1 == n)
#pragma unroll 1
      for (int b = bk + 1; b <= kBuckets; ++b) bucket[b] = (uint16_t)n;
  }
  __pipeline_commit();
}

// One (b, a) doublet of T3: slopes of a -> b, slope cut, then the best unused c of layer C inside b's phi window.
template <class C>
__device__ __forceinline__ void process_doublet(const Ctx<C>& c, const Hit* __restrict__ recA,
                                                const Hit* __restrict__ recB, const Hit* __restrict__ recC,
                                                const uint16_t* __restrict__ bucketC, uint32_t nC, uint32_t kb,
                                                uint32_t ia) {
  const Hit hb = recB[kb], ha = recA[ia];
  const float dz_ab = __fsub_rn(hb.z, ha.z);
  const float tx = __fdiv_rn(__fsub_rn(hb.x, ha.x), dz_ab), ty = __fdiv_rn(__fsub_rn(hb.y, ha.y), dz_ab);
  if (!(fabsf(tx) <= c.P.max_slope) || !(fabsf(ty) <= c.P.max_slope)) return;
  const int w = c.P.w_seed_phi16, phb = phi_of(hb.w);
  uint32_t ic = lower_bound_phi(bucketC, recC, nC, wrap16(phb - w));
  unsigned long long best = kNoClaim;
#pragma unroll 1
  for (uint32_t k = 0; k < nC; ++k, ++ic) {
    if (ic >= nC) ic -= nC;
    const Hit hc = recC[ic];
    const int d = wrap16(phi_of(hc.w) - phb);
    if (d > w || d < -w) break;
    if (hc.w & kUsedBit) continue;
    const float dz = __fsub_rn(hc.z, hb.z);
    const float ex = __fsub_rn(__fmaf_rn(tx, dz, hb.x), hc.x);
    const float ey = __fsub_rn(__fmaf_rn(ty, dz, hb.y), hc.y);
    const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
    if (!(S <= c.P.s_seed)) continue;
    // argmin over (bits(S), a, c): layer-local indices order like the event-local ones
    const unsigned long long key = ((unsigned long long)__float_as_uint(S) << 32) | (ia << 16) | ic;
    best = key < best ? key : best;
  }
  if (best != kNoClaim) atomicMin(&c.sm.best[kb], best);
}

// Offsets of the event's layers: lo[] relative to the event's first cluster, src[] absolute in the output arrays.
template <class C>
__device__ __forceinline__ void load_offsets(const TrackLaunch& a, uint32_t e, Smem<C>& sm, uint32_t co) {
  const uint32_t L = a.geo.n_layers;
#pragma unroll 1
  for (uint32_t l = threadIdx.x; l <= L; l += C::kBlock) sm.lo[l] = a.clusters.layer_offsets[e * L + l] - co;
#pragma unroll 1
  for (uint32_t l = threadIdx.x; l < L; l += C::kBlock)
    sm.src[l] = a.clusters.layer_offsets[e * L + l];
}

// Search by triplet and fit for event e; the whole CTA calls it.
template <class C>
__device__ __forceinline__ void track_event(const TrackLaunch& a, uint32_t e, Smem<C>& sm) {
  const DeviceGeometry& g = a.geo;
  const uint32_t L = g.n_layers, tid = threadIdx.x;
  const uint32_t lane = lane_id(), warp = tid >> 5;
  const uint32_t co = a.clusters.event_offsets[e];
  load_offsets<C>(a, e, sm, co);
  if (tid == 0) { sm.flags = 0; sm.min_active[0] = 0; sm.min_active[1] = 0; sm.n_doublets = 0; }
  if (tid < (uint32_t)(C::kCap + 31) / 32) sm.ovf[tid] = 0;
  __syncthreads();
  Ctx<C> c{sm, a.clusters.x, a.clusters.y, a.clusters.z, a.clusters.phi16, g.params};
  const allen_velo_params_t& P = c.P;
  uint16_t* link = a.link + co;

#pragma unroll 1
  for (uint32_t k = tid; k < (uint32_t)C::kCap; k += C::kThreads) {
    sm.best[k] = kNoClaim; sm.claimA[k] = kNoClaim; sm.claimC[k] = kNoClaim;
  }
  stage_layer(c, L - 1);
  stage_layer(c, L - 2);
  stage_layer(c, L - 3);

  uint32_t n_tracks = 0;        // block-uniform
  uint32_t first_new = 0;       // n_tracks before the latest T4 (block-uniform)

#pragma unroll 1
  for (int i = (int)L - 1; i >= 2; --i) {
    const uint32_t A0 = sm.lo[i], A1 = sm.lo[i + 1], B0 = sm.lo[i - 1], C0 = sm.lo[i - 2];
    const uint32_t nA = A1 - A0, nB = A0 - B0, nC = B0 - C0;
    Hit* recA = sm.rec[i % 3];
    Hit* recB = sm.rec[(i - 1) % 3];
    Hit* recC = sm.rec[(i - 2) % 3];
    const uint16_t* bucketA = sm.bucket[i % 3];
    const uint16_t* bucketC = sm.bucket[(i - 2) % 3];

    __pipeline_wait_prior(0);
    tsync<C>();  // B1: layer C staged; tracks created by the previous T4 visible; claims re-initialised

    // ---- T1 forward: best hit of layer C per active track (nothing of C is used yet); claim with (bits(S), key)
    const uint32_t first = min(sm.min_active[i & 1], first_new);
    if (tid == 0) sm.min_active[(i - 1) & 1] = 0xFFFFFFFFu;
#pragma unroll 1
    for (uint32_t k = tid; k < max(nA, nC); k += C::kThreads) { sm.claimA[k] = kNoClaim; sm.claimC[k] = kNoClaim; }
    uint16_t* fsel = sm.fsel;
#pragma unroll 1
    for (uint32_t t = first + tid; t < n_tracks; t += C::kThreads) {
      fsel[t] = 0xFFFFu;
      const uint32_t st = sm.tstate[t];
      if ((st & 0xFFu) == 0xFFu || nC == 0) continue;
      const uint32_t q = st >> 16;
      float xq, yq, zq;
      int phq;
      if (q < A1) {  // q on layer A or B (always, when max_skipped <= 1)
        const Hit hq = q >= A0 ? recA[q - A0] : recB[q - B0];
        xq = hq.x; yq = hq.y; zq = hq.z; phq = phi_of(hq.w);
      } else {       // tracks that skipped more than one layer: their last hit left the ring
        uint32_t l = (uint32_t)i + 1;
#pragma unroll 1
        while (q >= sm.lo[l + 1]) ++l;
        const Hit hq = far_hit(c, sm.src[l] + (q - sm.lo[l]));
        xq = hq.x; yq = hq.y; zq = hq.z; phq = phi_of(hq.w);
      }
      const float tx = sm.ttx[t], ty = sm.tty[t];
      const int w = P.w_fwd_phi16;
      uint32_t ic = lower_bound_phi(bucketC, recC, nC, wrap16(phq - w));
      unsigned long long best = kNoClaim;
#pragma unroll 1
      for (uint32_t k = 0; k < nC; ++k, ++ic) {
        if (ic >= nC) ic -= nC;
        const Hit hc = recC[ic];
        const int d = wrap16(phi_of(hc.w) - phq);
        if (d > w || d < -w) break;
        const float dz = __fsub_rn(hc.z, zq);
        const float ex = __fsub_rn(__fmaf_rn(tx, dz, xq), hc.x);
        const float ey = __fsub_rn(__fmaf_rn(ty, dz, yq), hc.y);
        const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
        if (!(S <= P.s_fwd)) continue;
        const unsigned long long key = ((unsigned long long)__float_as_uint(S) << 32) | ic;
        best = key < best ? key : best;
      }
      if (best != kNoClaim) {
        const uint32_t ic_best = (uint32_t)best;
        fsel[t] = (uint16_t)ic_best;
        atomicMin(&sm.best[ic_best], (best & 0xFFFFFFFF00000000ull) | sm.tseedB[t]);
      }
    }
    // ---- T3/S1 (same phase as T1: it reads only the used flags of layers A and B, final since the last T4): every
    //      unused b lists the unused hits of layer A inside its phi window as (b, a) doublets
    const bool seeding = nA != 0 && nB != 0 && nC != 0;
#pragma unroll 1
    for (uint32_t kb = tid; kb < nB; kb += C::kThreads) {
      const uint32_t wb = recB[kb].w;
      if (!seeding || (wb & kUsedBit)) continue;
      const int w = P.w_seed_phi16, phb = phi_of(wb);
      uint32_t ia = lower_bound_phi(bucketA, recA, nA, wrap16(phb - w));
      // the window is walked in runs of up to 32 hits: a bit mask of the unused ones, ONE reservation in the list per
      // run, then the entries are written from the mask (no list atomic per doublet)
      bool more = true;
#pragma unroll 1
      for (uint32_t k = 0; k < nA && more;) {
        const uint32_t ia0 = ia;
        uint32_t mask = 0, run = 0;
#pragma unroll 1
        for (; run < 32 && k < nA; ++run, ++k, ++ia) {
          if (ia >= nA) ia -= nA;
          const uint32_t wa = recA[ia].w;
          const int d = wrap16(phi_of(wa) - phb);
          if (d > w || d < -w) { more = false; break; }
          if (!(wa & kUsedBit)) mask |= 1u << run;
        }
        if (mask) {
          uint32_t pos = atomicAdd(&sm.n_doublets, (uint32_t)__popc(mask));
          if (pos + (uint32_t)__popc(mask) > (uint32_t)C::kCapDoublets) atomicOr(&sm.ovf[kb >> 5], 1u << (kb & 31u));
#pragma unroll 1
          for (; mask; mask &= mask - 1, ++pos) {
            uint32_t a_idx = ia0 + (uint32_t)__ffs(mask) - 1u;
            if (a_idx >= nA) a_idx -= nA;
            if (pos < (uint32_t)C::kCapDoublets) sm.doublets[pos] = kb | (a_idx << 16);  // else: S2 walks this b again
          }
        }
      }
    }
    tsync<C>();  // B2
    // ---- T2 resolve: the minimal claim wins the hit (track keys are unique, so the low half of the claim names the
    //      winner); everyone else counts a miss
    uint32_t my_min_active = 0xFFFFFFFFu;  // lowest track slot of this thread that stays active
#pragma unroll 1
    for (uint32_t t = first + tid; t < n_tracks; t += C::kThreads) {
      const uint32_t st = sm.tstate[t];
      if ((st & 0xFFu) == 0xFFu) continue;
      const uint32_t fc = fsel[t];
      // the winner puts the claim word back to "none" (losers then still fail the test: a key is never 0xFFFF), so
      // best[] is clean again for the per-b argmin of T3 without a pass of its own
      const bool won = fc != 0xFFFFu && (uint16_t)sm.best[fc] == sm.tseedB[t];
      if (won) {
        sm.best[fc] = kNoClaim;
        const uint32_t q = st >> 16, cg = C0 + fc;
        float xq, yq, zq;
        if (q < A1) {
          const Hit hq = q >= A0 ? recA[q - A0] : recB[q - B0];
          xq = hq.x; yq = hq.y; zq = hq.z;
        } else {
          uint32_t l = (uint32_t)i + 1;
#pragma unroll 1
          while (q >= sm.lo[l + 1]) ++l;
          const Hit hq = far_hit(c, sm.src[l] + (q - sm.lo[l]));
          xq = hq.x; yq = hq.y; zq = hq.z;
        }
        const Hit hc = recC[fc];
        const float dz = __fsub_rn(hc.z, zq);
        sm.ttx[t] = __fdiv_rn(__fsub_rn(hc.x, xq), dz);
        sm.tty[t] = __fdiv_rn(__fsub_rn(hc.y, yq), dz);
        recC[fc].w = hc.w | kUsedBit;
        link[cg] = (uint16_t)q;
        const uint32_t nh = ((st >> 8) & 0x7Fu) + 1u;
        sm.tstate[t] = (cg << 16) | (st & 0x8000u) | (nh << 8);
        my_min_active = min(my_min_active, t);
      } else {
        const uint32_t m = (st & 0xFFu) + 1u;
        if (m > (uint32_t)P.max_skipped) {
          sm.tstate[t] = st | 0xFFu;
        } else {
          sm.tstate[t] = (st & 0xFFFFFF00u) | m;
          my_min_active = min(my_min_active, t);
        }
      }
    }
    my_min_active = __reduce_min_sync(kFull, my_min_active);  // one shared-memory atomic per warp, not per track
    if (lane == 0 && my_min_active != 0xFFFFFFFFu) atomicMin(&sm.min_active[(i - 1) & 1], my_min_active);
    tsync<C>();  // B3

    // ---- T3/S2: one thread per listed doublet; middle hits whose doublets did not all fit the list walk their phi
    //      window themselves (a doublet evaluated twice gives the same key: the argmin does not care)
    {
      const uint32_t n_listed = sm.n_doublets, nd = min(n_listed, (uint32_t)C::kCapDoublets);
#pragma unroll 1
      for (uint32_t d = tid; d < nd; d += C::kThreads) {
        const uint32_t v = sm.doublets[d];
        process_doublet(c, recA, recB, recC, bucketC, nC, v & 0xFFFFu, v >> 16);
      }
      if (n_listed > (uint32_t)C::kCapDoublets) {  // block-uniform
#pragma unroll 1
        for (uint32_t kb = tid; kb < nB; kb += C::kThreads) {
          if (!(sm.ovf[kb >> 5] >> (kb & 31u) & 1u)) continue;
          const uint32_t wb = recB[kb].w;
          const int w = P.w_seed_phi16, phb = phi_of(wb);
          uint32_t ia = lower_bound_phi(bucketA, recA, nA, wrap16(phb - w));
#pragma unroll 1
          for (uint32_t k = 0; k < nA; ++k, ++ia) {
            if (ia >= nA) ia -= nA;
            const uint32_t wa = recA[ia].w;
            const int d = wrap16(phi_of(wa) - phb);
            if (d > w || d < -w) break;
            if (!(wa & kUsedBit)) process_doublet(c, recA, recB, recC, bucketC, nC, kb, ia);
          }
        }
      }
    }
    tsync<C>();  // B5

    // ---- T4a: every b with a triplet claims its a and its c with (bits(S), b)
    if (tid == 0) sm.n_doublets = 0;  // S2 is over; the next S1 starts after two more barriers
    if (tid < (uint32_t)(C::kCap + 31) / 32) sm.ovf[tid] = 0;
    // layer A is done with (T4 reads only B and C): its ring slot takes the next layer, needed at the top of the
    // next iteration; the copy runs behind T4
    if (i >= 3) stage_layer(c, (uint32_t)i - 3);
    const uint32_t roundsB = seeding ? (nB + C::kThreads - 1) / C::kThreads : 0;  // block-uniform
#pragma unroll 1
    for (uint32_t kb = tid; kb < nB && seeding; kb += C::kThreads) {
      const unsigned long long k = sm.best[kb];
      if (k == kNoClaim) continue;
      const uint32_t ac = (uint32_t)k;  // a_local << 16 | c_local
      const unsigned long long tkey = (k & 0xFFFFFFFF00000000ull) | (B0 + kb);
      atomicMin(&sm.claimA[ac >> 16], tkey);
      atomicMin(&sm.claimC[ac & 0xFFFFu], tkey);
    }
    tsync<C>();  // B6
    // ---- T4b: accepted iff the triplet holds the minimal key on both its a and its c; new tracks take slots in
    //      ascending b (ballot + per-warp totals).  best[] and the claims stay untouched until the end of T4b, so
    //      both halves re-derive "accepted" instead of carrying it in registers.
    auto accepted_of = [&](uint32_t kb, uint32_t& ac, unsigned long long& tkey) -> bool {
      if (kb >= nB) return false;
      const unsigned long long k = sm.best[kb];
      if (k == kNoClaim) return false;
      ac = (uint32_t)k;
      tkey = (k & 0xFFFFFFFF00000000ull) | (B0 + kb);
      return sm.claimA[ac >> 16] == tkey && sm.claimC[ac & 0xFFFFu] == tkey;
    };
#pragma unroll 1
    for (uint32_t r = 0; r < roundsB; ++r) {
      uint32_t ac = 0;
      unsigned long long tkey = 0;
      const uint32_t ballot = __ballot_sync(kFull, accepted_of(r * C::kThreads + tid, ac, tkey));
      if (lane == 0) sm.warp_tot[r][warp] = __popc(ballot);
    }
    tsync<C>();  // B7
    first_new = n_tracks;
    {
      uint32_t run = n_tracks;
#pragma unroll 1
      for (uint32_t r = 0; r < roundsB; ++r) {
        uint32_t before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < C::kWarps; ++w) {
          const uint32_t v = sm.warp_tot[r][w];
          if (w < (int)warp) before += v;
          total += v;
        }
        const uint32_t kb = r * C::kThreads + tid;
        if (total) {  // block-uniform
          uint32_t ac = 0;
          unsigned long long tkey = 0;
          const bool acc = accepted_of(kb, ac, tkey);
          const uint32_t ballot = __ballot_sync(kFull, acc);
          if (acc) {
            const uint32_t slot = run + before + __popc(ballot & lanemask_lt());
            if (slot < (uint32_t)C::kCapTracks) {
              const uint32_t ia = ac >> 16, ic = ac & 0xFFFFu;
              const Hit hb = recB[kb], hc = recC[ic];
              const float dz = __fsub_rn(hc.z, hb.z);
              sm.ttx[slot] = __fdiv_rn(__fsub_rn(hc.x, hb.x), dz);
              sm.tty[slot] = __fdiv_rn(__fsub_rn(hc.y, hb.y), dz);
              const float S = __uint_as_float((uint32_t)(tkey >> 32));
              sm.tstate[slot] = ((C0 + ic) << 16) | (S <= P.s_weak ? 0x8000u : 0u) | (3u << 8);
              sm.tseedB[slot] = (uint16_t)(B0 + kb);
              link[B0 + kb] = (uint16_t)(A0 + ia);
              link[C0 + ic] = (uint16_t)(B0 + kb);
              // layer A leaves the ring after this iteration: its used flags are never read again
              recB[kb].w = hb.w | kUsedBit;
              recC[ic].w = hc.w | kUsedBit;
            } else {
              sm.flags = 1;  // out of track slots: a larger instance redoes the event
            }
          }
        }
        if (kb < nB) sm.best[kb] = kNoClaim;  // only this thread reads best[kb] in T4b; the next T1 needs "none"
        run += total;
      }
      n_tracks = min(run, (uint32_t)C::kCapTracks);
    }
  }
  __pipeline_wait_prior(0);
  __syncthreads();

  if (sm.flags) {  // out of track slots: the next larger instance redoes the event in the second pass
    if (tid == 0) {
      if (C::kLast) { atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW); a.counts[e] = 0; }
      else a.redo_list[C::kLevel][atomicAdd(a.counters + kCtrRedo + C::kLevel, 1u)] = e;
    }
    return;
  }

  // ---- T5 finalise + A8 fit: keep >= 4 hits, or 3 hits with S_seed <= s_weak; output in order of creation
  uint32_t out_tracks = 0, out_hits = 0;
  const uint32_t trk0 = co / 3;
  // the fit reads the compacted output (an earlier kernel filled it)
  const float* X = a.clusters.x + co;
  const float* Y = a.clusters.y + co;
  const float* Z = a.clusters.z + co;
#pragma unroll 1
  for (uint32_t base = 0; base < n_tracks; base += C::kThreads) {
    const uint32_t t = base + tid;
    uint32_t n = 0, st = 0;
    if (t < n_tracks) {
      st = sm.tstate[t];
      n = (st >> 8) & 0x7Fu;
      if (n == 3 && !(st & 0x8000u)) n = 0;
    }
    // block exclusive scan of (1 << 20 | n)
    const uint32_t v = n ? ((1u << 20) | n) : 0u;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t u = __shfl_up_sync(kFull, incl, d);
      if (lane >= (uint32_t)d) incl += u;
    }
    tsync<C>();
    if (lane == 31) sm.warp_tot[0][warp] = incl;
    tsync<C>();
    uint32_t off = incl - v, total = 0;
#pragma unroll
    for (int w = 0; w < C::kWarps; ++w) {
      const uint32_t u = sm.warp_tot[0][w];
      if (w < (int)warp) off += u;
      total += u;
    }
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
      // A8: the oracle's operations in the oracle's order (R6) -> bit-identical parameters
      const double dn = (double)n;
      double zm = 0, xm = 0, ym = 0;
#pragma unroll 1
      for (uint32_t k = 0; k < n; ++k) {
        h = out_h[k];
        zm += (double)__ldcg(Z + h); xm += (double)__ldcg(X + h); ym += (double)__ldcg(Y + h);
      }
      zm /= dn; xm /= dn; ym /= dn;
      double szz = 0, szx = 0, szy = 0;
#pragma unroll 1
      for (uint32_t k = 0; k < n; ++k) {
        h = out_h[k];
        const double dz = (double)__ldcg(Z + h) - zm;
        szz += dz * dz;
        szx += dz * ((double)__ldcg(X + h) - xm);
        szy += dz * ((double)__ldcg(Y + h) - ym);
      }
      const double tx = szx / szz, ty = szy / szz;
      a.trk_hitoff[trk0 + ot] = oh;
      a.trk_fit[trk0 + ot] = make_float4((float)(xm - tx * zm), (float)(ym - ty * zm), (float)tx, (float)ty);
    }
    out_tracks += total >> 20;
    out_hits += total & 0xFFFFFu;
  }
  if (tid == 0) a.counts[e] = ((unsigned long long)out_tracks << 32) | out_hits;
}

// One CTA per event: move the event's tracks from its slabs to the compacted output.
constexpr uint32_t kLinkStage = 8192;  // links of an event staged in shared memory (events with more clusters: global)
constexpr uint32_t kCompactThreads = 128;  // (256: one round for the ~150 tracks of a nu = 6 event, but 0.21 instead of 0.18 ms)
__global__ void __launch_bounds__(kCompactThreads) compact_tracks_kernel(const CompactTracksLaunch a) {
  extern __shared__ __align__(16) unsigned char compact_smem[];  // links [kLinkStage], hit lists [n_layers][kCompactThreads] (u16)
  const uint32_t e = blockIdx.x;
  const unsigned long long o0 = a.offsets[e], o1 = a.offsets[e + 1];
  const uint32_t T0 = (uint32_t)(o0 >> 32), H0 = (uint32_t)o0;
  const uint32_t nT = (uint32_t)(o1 >> 32) - T0, nH = (uint32_t)o1 - H0;
  if (threadIdx.x == 0) {
    a.out.event_offsets[e] = T0;
    if (e + 1 == a.n_events) {
      a.out.event_offsets[e + 1] = T0 + nT;
      // the total number of hits also at a fixed place (the last element), whether or not the tracks fit, so that a host
      // needs one read for both totals (it equals hit_offsets[n_tracks] when n_tracks == capacity_tracks)
      a.out.hit_offsets[a.out.capacity_tracks] = H0 + nH;
    }
  }
  const bool fits = (unsigned long long)T0 + nT <= a.out.capacity_tracks &&
                    (unsigned long long)H0 + nH <= a.out.capacity_hits;
  if (!fits) {
    if (threadIdx.x == 0 && nT) {
      atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_TRACK_CAPACITY);
      if (T0 < a.out.capacity_tracks) a.out.hit_offsets[T0] = H0;  // closes the hit list of the last track before this event
    }
    return;
  }
  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t trk0 = co / 3;
  const uint32_t fl = a.ev_flags[e];
  if (fl & kEvFinal) {
    // ---- tracks as velo_follow.cu left them: final state of every track by order of creation + links between the hits.
    //      T5 (R5): keep >= 4 hits, or 3 hits with S_seed <= s_weak (bit 15 of the state).  A thread per track: offsets by
    //      a block scan in order of creation, hit list by walking the links back from the newest hit, then A8: the
    //      oracle's operations in the oracle's order (R6: fp64 means, then centred sums, over the hits in order
    //      of addition, from the fp32 coordinates) -> bit-identical parameters.
    __shared__ uint32_t warp_tot[kCompactThreads / 32];
    const uint32_t n_created = fl >> 8, lane = lane_id(), warp = threadIdx.x >> 5;
    const uint16_t* link = a.link + co;
    const float* X = a.clusters.x + co;
    const float* Y = a.clusters.y + co;
    const float* Z = a.clusters.z + co;
    // The links of the event go to shared memory first (one coalesced pass), and every thread keeps the hit list of its
    // track there: walking the links and re-reading the list were chains of dependent global loads (7 + 14 per track).
    uint16_t* s_link = reinterpret_cast<uint16_t*>(compact_smem);
    uint16_t* my_hits = s_link + kLinkStage + threadIdx.x;  // [k * kCompactThreads]
    const uint32_t n_cl = a.clusters.event_offsets[e + 1] - co;
    const bool staged = n_cl <= kLinkStage;
    if (staged) {
#pragma unroll 4
      for (uint32_t i = threadIdx.x; i < n_cl; i += kCompactThreads) s_link[i] = __ldg(link + i);
    }
    __syncthreads();
    uint32_t run_t = 0, run_h = 0;
#pragma unroll 1
    for (uint32_t base = 0; base < n_created; base += kCompactThreads) {
      const uint32_t t = base + threadIdx.x;
      uint32_t n = 0, st = 0;
      if (t < n_created) {
        st = a.trk_final[trk0 + t];
        n = track_n_hits(st);
        if (n == 3 && !(st & 0x8000u)) n = 0;
      }
      const uint32_t v = n ? ((1u << 20) | n) : 0u;
      uint32_t incl = v;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(kFull, incl, d);
        if (lane >= (uint32_t)d) incl += u;
      }
      if (lane == 31) warp_tot[warp] = incl;
      __syncthreads();
      uint32_t off = incl - v, total = 0;
#pragma unroll
      for (int w = 0; w < (int)(kCompactThreads / 32); ++w) {
        const uint32_t u = warp_tot[w];
        if (w < (int)warp) off += u;
        total += u;
      }
      __syncthreads();
      if (n) {
        const uint32_t ot = T0 + run_t + (off >> 20), oh = H0 + run_h + (off & 0xFFFFFu);
        uint16_t* out_h = a.out.hits + oh;
        uint32_t h = st >> 16;
#pragma unroll 1
        for (int k = (int)n - 1; k >= 0; --k) {
          out_h[k] = (uint16_t)h;
          my_hits[k * kCompactThreads] = (uint16_t)h;
          if (k) h = staged ? s_link[h] : link[h];
        }
        const double dn = (double)n;
        double zm = 0, xm = 0, ym = 0;
        // (four hits per trip: their loads are in flight together; the sums keep the order of addition)
#pragma unroll 1
        for (uint32_t k0 = 0; k0 < n; k0 += 4) {
          float zz[4], xx[4], yy[4];
#pragma unroll
          for (uint32_t u = 0; u < 4; ++u) {
            if (k0 + u < n) {
              h = my_hits[(k0 + u) * kCompactThreads];
              zz[u] = Z[h]; xx[u] = X[h]; yy[u] = Y[h];
            }
          }
#pragma unroll
          for (uint32_t u = 0; u < 4; ++u) {
            if (k0 + u < n) { zm += (double)zz[u]; xm += (double)xx[u]; ym += (double)yy[u]; }
          }
        }
        zm /= dn; xm /= dn; ym /= dn;
        double szz = 0, szx = 0, szy = 0;
#pragma unroll 1
        for (uint32_t k0 = 0; k0 < n; k0 += 4) {
          float zz[4], xx[4], yy[4];
#pragma unroll
          for (uint32_t u = 0; u < 4; ++u) {
            if (k0 + u < n) {
              h = my_hits[(k0 + u) * kCompactThreads];
              zz[u] = Z[h]; xx[u] = X[h]; yy[u] = Y[h];
            }
          }
#pragma unroll
          for (uint32_t u = 0; u < 4; ++u) {
            if (k0 + u < n) {
              const double dz = (double)zz[u] - zm;
              szz += dz * dz;
              szx += dz * ((double)xx[u] - xm);
              szy += dz * ((double)yy[u] - ym);
            }
          }
        }
        const double tx = szx / szz, ty = szy / szz;
        a.out.x0[ot] = (float)(xm - tx * zm); a.out.y0[ot] = (float)(ym - ty * zm);
        a.out.tx[ot] = (float)tx; a.out.ty[ot] = (float)ty;
        a.out.hit_offsets[ot] = oh;
      }
      run_t += total >> 20;
      run_h += total & 0xFFFFFu;
    }
  } else {
    // ---- tracks as the CTA-per-event kernel left them: hit lists and fits in per-event slabs
#pragma unroll 1
    for (uint32_t t = threadIdx.x; t < nT; t += blockDim.x) {
      const float4 f = a.trk_fit[trk0 + t];
      a.out.x0[T0 + t] = f.x; a.out.y0[T0 + t] = f.y; a.out.tx[T0 + t] = f.z; a.out.ty[T0 + t] = f.w;
      a.out.hit_offsets[T0 + t] = H0 + a.trk_hitoff[trk0 + t];
    }
#pragma unroll 1
    for (uint32_t k = threadIdx.x; k < nH; k += blockDim.x) a.out.hits[H0 + k] = a.hits_slab[co + k];
  }
  // ---- simple Kalman fit (R9), one thread per track, x and y independent: start at the first hit
  //      with (measured position, slope 0), C = diag(var_m, 1); per further hit add the scattering of a 400 MeV pT
  //      track to C11, propagate, update.  (1 - K0) = var_m / S keeps the covariance update free of cancellation.
  if (a.out.kalman) {
    __syncthreads();  // the hit lists above are complete
    const float* X = a.clusters.x + co;
    const float* Y = a.clusters.y + co;
    const float* Z = a.clusters.z + co;
    const float var_m = a.pitch * a.pitch * (1.0f / 12.0f);
#pragma unroll 1
    for (uint32_t t = threadIdx.x; t < nT; t += blockDim.x) {
      const uint32_t h0 = a.out.hit_offsets[T0 + t], h1 = t + 1 < nT ? a.out.hit_offsets[T0 + t + 1] : H0 + nH;
      const uint16_t* hits = a.out.hits + h0;
      uint32_t h = hits[0], hn = hits[1];
      float zp = Z[h];
      const float dz01 = Z[hn] - zp, tx0 = (X[hn] - X[h]) / dz01, ty0 = (Y[hn] - Y[h]) / dz01;
      const float t2 = tx0 * tx0 + ty0 * ty0;
      const float theta02 = (13.6f / 400.0f) * (13.6f / 400.0f) * 0.02f * t2 / (1.0f + t2);
      const float qx = theta02 * (1.0f + tx0 * tx0) * (1.0f + t2), qy = theta02 * (1.0f + ty0 * ty0) * (1.0f + t2);
      // Hit 1 in closed form: with the diffuse slope prior (C11 = 1) the generic update subtracts two nearly equal
      // numbers; for C = [[v + dz^2 P, dz P], [dz P, P]], P = 1 + q, S = 2 v + dz^2 P the posterior is
      // C00 = (v + dz^2 P) v / S, C01 = dz P v / S, C11 = 2 v P / S, gains K0 = (v + dz^2 P) / S, K1 = dz P / S.
      float px, sx, ax, bx, cx, py, sy, ay, by, cy, chi2;
      {
        const float Px = 1.0f + qx, Py = 1.0f + qy, d2 = dz01 * dz01;
        const float ix = 1.0f / (2.0f * var_m + d2 * Px), iy = 1.0f / (2.0f * var_m + d2 * Py);
        const float rx = X[hn] - X[h], ry = Y[hn] - Y[h];
        px = X[h] + (var_m + d2 * Px) * ix * rx; sx = dz01 * Px * ix * rx;
        py = Y[h] + (var_m + d2 * Py) * iy * ry; sy = dz01 * Py * iy * ry;
        ax = (var_m + d2 * Px) * var_m * ix; bx = dz01 * Px * var_m * ix; cx = 2.0f * var_m * Px * ix;
        ay = (var_m + d2 * Py) * var_m * iy; by = dz01 * Py * var_m * iy; cy = 2.0f * var_m * Py * iy;
        chi2 = rx * rx * ix + ry * ry * iy;
        zp = Z[hn];
      }
#pragma unroll 1
      for (uint32_t k = 2; k < h1 - h0; ++k) {
        h = hits[k];
        const float z = Z[h], dz = z - zp;
        zp = z;
        cx += qx; px += sx * dz; ax += 2.0f * dz * bx + dz * dz * cx; bx += dz * cx;
        cy += qy; py += sy * dz; ay += 2.0f * dz * by + dz * dz * cy; by += dz * cy;
        const float rx = X[h] - px, ry = Y[h] - py;
        const float ix = 1.0f / (ax + var_m), iy = 1.0f / (ay + var_m);
        px += ax * ix * rx; sx += bx * ix * rx; cx -= bx * bx * ix;
        py += ay * iy * ry; sy += by * iy * ry; cy -= by * by * iy;
        bx *= var_m * ix; ax *= var_m * ix;
        by *= var_m * iy; ay *= var_m * iy;
        chi2 += rx * rx * ix + ry * ry * iy;
      }
      float* o = a.out.kalman + 12 * (size_t)(T0 + t);
      o[0] = px; o[1] = py; o[2] = sx; o[3] = sy; o[4] = zp; o[5] = chi2;
      o[6] = ax; o[7] = bx; o[8] = cx; o[9] = ay; o[10] = by; o[11] = cy;
    }
  }
  if (threadIdx.x == 0 && e + 1 == a.n_events) a.out.hit_offsets[T0 + nT] = H0 + nH;
}

// One thread per event: class of the event (hits per layer its search needs, or copy only / nothing) and the event lists of
// the three instances of velo_follow.cu.
__global__ void __launch_bounds__(256) classify_events_kernel(const __grid_constant__ TrackLaunch a) {
  const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= a.n_events) return;
  const uint32_t L = a.geo.n_layers;
  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t n_cl = a.clusters.event_offsets[e + 1] - co;
  const uint32_t st0 = a.clusters.status[e];
  uint8_t cls;
  if (n_cl == 0) {
    cls = kClsSkip;
  } else if ((unsigned long long)co + n_cl > a.clusters.capacity) {  // the output (or the per-cluster scratch) is full
    atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_CLUSTER_CAPACITY);
    cls = kClsSkip;
  } else if ((st0 & (ALLEN_VELO_STATUS_BAD_HEADER | ALLEN_VELO_STATUS_STAGE_OVERFLOW)) != 0) {
    cls = kClsCopy;  // incomplete clusters take no part in tracking
  } else if (n_cl > 65535u) {
    atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_TOO_MANY_CLUSTERS);  // hit indices are 16 bit
    cls = kClsCopy;
  } else {
    uint32_t mx = 0, prev = co;
#pragma unroll 1
    for (uint32_t l = 1; l <= L; ++l) {
      const uint32_t o = a.clusters.layer_offsets[e * L + l];
      mx = max(mx, o - prev);
      prev = o;
    }
    if (mx <= (uint32_t)kFlatCap) cls = kClsFlat;
    else if (mx <= (uint32_t)CfgMr::kCap) cls = kClsMid;
    else if (mx <= (uint32_t)CfgLr::kCap) cls = kClsLarge;
    else {  // busiest layer beyond the largest staging capacity
      atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
      cls = kClsCopy;
    }
    if (cls <= kClsLarge) a.flw_list[cls][atomicAdd(a.counters + kCtrFollow + cls, 1u)] = e;
  }
  a.level[e] = cls;
  a.ev_flags[e] = 0;
  if (cls >= kClsCopy) a.counts[e] = 0;
}

// Larger instances: a few resident CTAs take events from a list (most batches have few or none of them).
template <class C>
__global__ void __launch_bounds__(C::kBlock) velo_track_list_kernel(const __grid_constant__ TrackLaunch a,
                                                                    const uint32_t* __restrict__ list,
                                                                    const uint32_t* __restrict__ count,
                                                                    uint32_t* cursor) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<C>& sm = *reinterpret_cast<Smem<C>*>(smem_raw);
  const uint32_t n = *count;
#pragma unroll 1
  for (;;) {
    if (threadIdx.x == 0) sm.next_event = atomicAdd(cursor, 1u);
    __syncthreads();
    const uint32_t idx = sm.next_event;
    if (idx >= n) return;
    track_event<C>(a, list[idx], sm);
    __syncthreads();
  }
}

template <class C>
cudaError_t prepare_list() {
  static_assert(sizeof(Smem<C>) <= 227 * 1024, "shared memory of one CTA");
  return cudaFuncSetAttribute(velo_track_list_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem<C>));
}

template <class C>
cudaError_t launch_list(const TrackLaunch& a, uint32_t which, uint32_t grid, cudaStream_t stream) {
  velo_track_list_kernel<C><<<grid, C::kBlock, sizeof(Smem<C>), stream>>>(a, a.redo_list[which], a.counters + kCtrRedo + which,
                                                                          a.counters + kCtrRedoCursor + which);
  return cudaGetLastError();
}

}  // namespace

// Once per process (allen_velo_create): the kernels' dynamic shared-memory limits.
cudaError_t track_prepare() {
  cudaError_t err = seed_prepare();
  if (err == cudaSuccess) err = follow_prepare();
  if (err == cudaSuccess) err = prepare_list<CfgMr>();
  if (err == cudaSuccess) err = prepare_list<CfgLr>();
  return err;
}

// classify -> velo_seed.  Then launch_track_follow: velo_follow (three instances beside each other) -> second pass (CTA
// per event, 512 hits per layer, then 1024) for the events those handed on.  `side`/`ev`: two extra streams and events
// owned by the handle; everything is ordered after and before the work on `stream` by events (a fork/join a CUDA graph
// can capture), nothing synchronises.
cudaError_t launch_track_seed(const TrackLaunch& a, cudaStream_t stream, uint32_t* n_launches) {
  *n_launches = 0;
  if (a.n_events == 0) return cudaSuccess;
  cudaError_t err = cudaMemsetAsync(a.counters, 0, kCtrCount * sizeof(uint32_t), stream);
  if (err != cudaSuccess) return err;
  classify_events_kernel<<<(a.n_events + 255) / 256, 256, 0, stream>>>(a);
  if ((err = cudaGetLastError()) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_seed(a, stream)) != cudaSuccess) return err;
  ++*n_launches;
  return cudaSuccess;
}

cudaError_t launch_track_follow(const TrackLaunch& a, cudaStream_t stream, cudaStream_t* side, cudaEvent_t* ev,
                                uint32_t n_sms, uint32_t* n_launches) {
  *n_launches = 0;
  if (a.n_events == 0) return cudaSuccess;
  cudaError_t err;
  if ((err = cudaEventRecord(ev[0], stream)) != cudaSuccess) return err;
  if ((err = cudaStreamWaitEvent(side[0], ev[0], 0)) != cudaSuccess) return err;
  if ((err = cudaStreamWaitEvent(side[1], ev[0], 0)) != cudaSuccess) return err;
  if ((err = launch_follow(a, 1, n_sms, side[0])) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_follow(a, 2, n_sms, side[1])) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_follow(a, 0, n_sms, stream)) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = cudaEventRecord(ev[1], side[0])) != cudaSuccess) return err;
  if ((err = cudaEventRecord(ev[2], side[1])) != cudaSuccess) return err;
  if ((err = cudaStreamWaitEvent(stream, ev[1], 0)) != cudaSuccess) return err;
  if ((err = cudaStreamWaitEvent(stream, ev[2], 0)) != cudaSuccess) return err;
  if ((err = launch_list<CfgMr>(a, 0, min(a.n_events, 2 * n_sms), stream)) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_list<CfgLr>(a, 1, min(a.n_events, n_sms), stream)) != cudaSuccess) return err;
  ++*n_launches;
  return cudaSuccess;
}

cudaError_t launch_compact_tracks(const CompactTracksLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  compact_tracks_kernel<<<a.n_events, kCompactThreads, 2u * kLinkStage + 2u * kCompactThreads * a.n_layers, stream>>>(a);
  return cudaGetLastError();
}

}  // namespace velo
