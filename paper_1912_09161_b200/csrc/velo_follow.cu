// Search by triplet, part 2 of 2: the sequential part — forwarding (A6), the conflict rules and clone/ghost killing (A7),
// the choice among the precomputed seed candidates (A5) — and the straight-line fit (A8).  SURVEY.md §8(a); DESIGN.md
// reading R5 (T1..T5) of P:181-183 and R6 of P:149.
//
// ONE WARP per event, no block barrier anywhere.  What is left of an iteration i (A = layer i, B = i-1, C = i-2) once
// velo_seed.cu has listed every (a, b, c) that passes the seeding cuts is small:
//   T1  every active track (about 40 per iteration at nu = 6, a lane each) evaluates the 3-4 hits of its precomputed phi
//       window on layer C (16-byte records straight from the slab; nothing of C can be used yet) and claims its best one
//       with a 64-bit shared-memory atomicMin on (bits(S), track_key);
//   T2  winners append the hit, the others count a miss; the list of active tracks is compacted by ballot;
//   T3  the list of layer B (about 33 entries, a lane each): entries whose three hits are still unused take part in the
//       per-b argmin on (bits(S), a, c);
//   T4  the best entry of every b claims its a and its c with (bits(S), b); accepted iff it holds both; new tracks in
//       ascending b (bit mask over b + prefix population counts).
// All conflict rules are order-independent minima on packed keys, so the result is exactly the oracle's.  A warp waits
// for its own loads and atomics most of the time (four dependent round trips per iteration), so the kernel lives on the
// number of events in flight: ~19 warps per SM for events with at most 256 hits per layer, one event each.
// Three instances by hits per layer (256 / 512 / 1024) and active tracks (192 / 384 / 768); an event that runs out of
// track slots, or that velo_seed.cu could not list, goes to the CTA-per-event kernel of velo_track.cu.
#include "velo_track.cuh"

namespace velo {
namespace {

constexpr uint32_t kNone16 = 0xFFFFu;

template <int kCap_, int kSeg_, int kLevel_>
struct FollowCfg {
  static constexpr int kCap = kCap_, kSeg = kSeg_, kLevel = kLevel_;
  static constexpr int kWords = kCap_ / 32;
};
using Follow256 = FollowCfg<256, 192, 0>;
using Follow512 = FollowCfg<512, 384, 1>;
using Follow1024 = FollowCfg<1024, 768, 2>;

template <class C>
struct __align__(16) FollowSmem {
  unsigned long long claimC[C::kCap];  // T1/T2: forward claims on the hits of layer C; T4: seed claims on c
  unsigned long long bestB[C::kCap];   // T3: argmin key of every middle hit; then T4: seed claims on a (the best entries are
                                       // marked in `beste` by then)
  float ttx[C::kSeg], tty[C::kSeg];    // active tracks: slopes of the last segment (older -> newest hit)
  uint32_t tstate[C::kSeg];            // newest hit (event-local) << 16 | weak_ok << 15 | n_hits << 8 | missed
  uint32_t twin[C::kSeg];              // phi windows of the newest hit on the next layer down (low half) and the one below
                                       // (high half), each first | count << 10; count 63 = "more: search the layer"
  uint16_t tseed[C::kSeg];             // track_key: event-local index of the seed's middle hit
  uint16_t tcid[C::kSeg];              // order of creation within the event
  uint16_t fsel[C::kSeg];              // hit of layer C chosen in T1 (kNone16: none)
  uint32_t used[3][C::kWords];         // used flags of layer l in used[l % 3]
  uint32_t accw[C::kWords];            // T4: accepted middle hits
  uint32_t acce[C::kWords];            // T4: accepted entries of the list, by round
  uint32_t beste[C::kWords];           // T3: entries that are the best of their middle hit, by round
  uint16_t lo[kMaxLayers + 2];         // first cluster of every layer, relative to the event (an event has < 65536)
  uint32_t src[kMaxLayers];            // first slab entry of every layer
};

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(kFull, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}

// The two forwarding windows of a hit (velo_seed.cu: first | count << 16 each) in 32 bits.
__device__ __forceinline__ uint32_t pack_windows(uint2 w) {
  const uint32_t c0 = min(w.x >> 16, 63u), c1 = min(w.y >> 16, 63u);
  return (w.x & 0x3FFu) | (c0 << 10) | ((w.y & 0x3FFu) << 16) | (c1 << 26);
}

__device__ __forceinline__ Hit load_hit(const uint4* __restrict__ p) {
  const uint4 r = __ldg(p);
  Hit h;
  h.x = __uint_as_float(r.x); h.y = __uint_as_float(r.y); h.z = __uint_as_float(r.z); h.w = r.w;
  return h;
}

// (max_skipped >= 2 only) phi window of a track that has missed two or more layers: binary search in the slab.
__device__ __forceinline__ uint32_t lower_bound_slab(const uint4* __restrict__ rec, uint32_t n, int target) {
  uint32_t lo = 0, hi = n;
#pragma unroll 1
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;
    if (phi_of(__ldg(reinterpret_cast<const uint32_t*>(rec + mid) + 3)) < target) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ uint32_t window_slab(const uint4* __restrict__ rec, uint32_t n, int ph, int w) {
  const int tl = ph - w, th = ph + w;
  const bool wrapped = tl < -32768 || th > 32767;
  const uint32_t lo = lower_bound_slab(rec, n, wrap16(tl));
  const int thw = wrap16(th);
  const uint32_t hi = thw == 32767 ? n : lower_bound_slab(rec, n, thw + 1);
  return lo | ((wrapped ? n - lo + hi : hi - lo) << 16);
}

// Ask the L2 for [p, p + bytes): the lines an iteration reads are requested one iteration ahead (the events in flight
// on the GPU hold more data than the L2, so without this every dependent load of an iteration goes to DRAM).
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes, uint32_t lane) {
  const char* c = reinterpret_cast<const char*>(p);
#pragma unroll 1
  for (uint32_t o = lane * 128u; o < bytes; o += 32u * 128u) asm volatile("prefetch.global.L2 [%0];" ::"l"(c + o));
}

template <class C>
__device__ __forceinline__ void follow_event(const TrackLaunch& a, uint32_t e, FollowSmem<C>& sm) {
  constexpr uint32_t kSeg = C::kSeg, kWords = C::kWords;
  const DeviceGeometry& g = a.geo;
  const allen_velo_params_t& P = g.params;
  const uint32_t L = g.n_layers, lane = lane_id();
  constexpr int which_redo = C::kLevel == 2 ? 1 : 0;
  if (a.ev_flags[e] & kEvRedo) {  // velo_seed.cu could not list the event
    if (lane == 0) a.redo_list[which_redo][atomicAdd(a.counters + kCtrRedo + which_redo, 1u)] = e;
    return;
  }
  const uint32_t co = a.clusters.event_offsets[e];
  uint16_t* link = a.link + co;
  const uint32_t trk0 = co / 3;
  const uint4* __restrict__ slab = a.slab.rec;
  const unsigned long long* __restrict__ trip = a.trip + co;
  const uint2* __restrict__ fwd_win = a.fwd_win + co;

#pragma unroll 1
  for (uint32_t l = lane; l <= L; l += 32) sm.lo[l] = (uint16_t)(a.clusters.layer_offsets[e * L + l] - co);  // (65535 at most: n_cl <= 65535)
#pragma unroll 1
  for (uint32_t l = lane; l < L; l += 32) sm.src[l] = a.slab_base[e * L + l];
  if (lane < 3 * kWords) (&sm.used[0][0])[lane] = 0;
  if (3 * kWords > 32) {
#pragma unroll 1
    for (uint32_t k = 32 + lane; k < 3 * kWords; k += 32) (&sm.used[0][0])[k] = 0;
  }
  if (lane < kWords) sm.accw[lane] = 0;
  // entries in the list of every layer: lane l holds layers l and l + 32
  const uint32_t tc0 = lane < L ? a.trip_count[e * L + lane] : 0u;
  const uint32_t tc1 = lane + 32 < L ? a.trip_count[e * L + lane + 32] : 0u;
  __syncwarp();
  auto list_size = [&](uint32_t l) -> uint32_t { return l < 32 ? __shfl_sync(kFull, tc0, l) : __shfl_sync(kFull, tc1, l - 32); };
  // what the first iteration reads: records and windows of layers L-2 and L-3, the list of layer L-2
  prefetch_l2(trip + sm.lo[L - 2], 8u * list_size(L - 2), lane);
#pragma unroll 1
  for (uint32_t l = L - 3; l < L - 1; ++l) {
    const uint32_t n = sm.lo[l + 1] - sm.lo[l];
    prefetch_l2(slab + sm.src[l], 16u * n, lane);
    prefetch_l2(fwd_win + sm.lo[l], 8u * n, lane);
  }

  uint32_t n_act = 0, n_created = 0;
  uint32_t out_tracks = 0, out_hits = 0;  // per lane: closed tracks that pass T5, and their hits
  bool overflow = false;

#pragma unroll 1
  for (int i = (int)L - 1; i >= 2; --i) {
    const uint32_t A0 = sm.lo[i], B0 = sm.lo[i - 1], C0 = sm.lo[i - 2];
    const uint32_t nC = B0 - C0;
    const uint4* __restrict__ recB = slab + sm.src[i - 1];
    const uint4* __restrict__ recC = slab + sm.src[i - 2];
    uint32_t* usedA = sm.used[i % 3];
    uint32_t* usedB = sm.used[(i - 1) % 3];
    uint32_t* usedC = sm.used[(i - 2) % 3];
    const uint32_t n_t = list_size((uint32_t)i - 1u);
    // first 64 entries of layer B's list: asked for now, needed after T2
    const unsigned long long ent0 = lane < n_t ? __ldg(trip + B0 + lane) : kNoClaim;
    const unsigned long long ent1 = lane + 32 < n_t ? __ldg(trip + B0 + 32 + lane) : kNoClaim;
    if (i >= 3) {  // the next iteration's lines: records and windows of its layer C, the list of its layer B
      const uint32_t l = (uint32_t)i - 3u, n = C0 - sm.lo[l];
      prefetch_l2(slab + sm.src[l], 16u * n, lane);
      prefetch_l2(fwd_win + sm.lo[l], 8u * n, lane);
      prefetch_l2(trip + C0, 8u * list_size((uint32_t)i - 2u), lane);
    }

    if (n_act) {
      // ---- T1 forward: best hit of layer C per active track (nothing of C is used yet); claim it with (bits(S), track_key)
      if (nC) {
#pragma unroll 1
        for (uint32_t t0 = 0; t0 < n_act; t0 += 32) {
          const uint32_t t = t0 + lane;
          if (t < n_act) {
            const uint32_t st = sm.tstate[t], m = st & 0xFFu, q = st >> 16;
            const uint32_t lq = (uint32_t)i - 1u + m;
            VELO_CHECK(g, lq < L && q >= sm.lo[lq] && q < sm.lo[lq + 1], 301);
            const Hit hq = load_hit(slab + sm.src[lq] + (q - sm.lo[lq]));
            const uint32_t tw = sm.twin[t] >> (m == 0 ? 0 : 16);
            uint32_t cnt = (tw >> 10) & 0x3Fu, ic = tw & 0x3FFu;
            if (m >= 2 || cnt == 63u) {  // missed two layers or more (max_skipped >= 2), or a window of 63 hits or more
              const uint32_t win = window_slab(recC, nC, phi_of(hq.w), P.w_fwd_phi16);
              cnt = win >> 16;
              ic = win & 0xFFFFu;
            }
            VELO_CHECK(g, cnt <= nC && ic <= nC && nC <= (uint32_t)C::kCap, 302);  // (a wrapped window may start at nC = index 0)
            const float tx = sm.ttx[t], ty = sm.tty[t];
            const int phq = phi_of(hq.w);
            unsigned long long best = kNoClaim;
            // four candidates at a time: their loads are in flight together
#pragma unroll 1
            for (uint32_t j0 = 0; j0 < cnt; j0 += 4) {
              Hit hc[4];
              uint32_t idx[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                idx[u] = ic + (uint32_t)u;
                if (idx[u] >= nC) idx[u] -= nC;
                if (j0 + (uint32_t)u < cnt) hc[u] = load_hit(recC + idx[u]);
              }
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                // (the window two layers down is a superset: whole phi slices)
                if (j0 + (uint32_t)u < cnt && abs(wrap16(phi_of(hc[u].w) - phq)) <= P.w_fwd_phi16) {
                  const float dz = __fsub_rn(hc[u].z, hq.z);
                  const float ex = __fsub_rn(__fmaf_rn(tx, dz, hq.x), hc[u].x);
                  const float ey = __fsub_rn(__fmaf_rn(ty, dz, hq.y), hc[u].y);
                  const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
                  if (S <= P.s_fwd) {
                    const unsigned long long key = ((unsigned long long)__float_as_uint(S) << 32) | idx[u];
                    best = key < best ? key : best;
                  }
                }
              }
              ic += 4;
              if (ic >= nC) ic -= nC;
            }
            uint32_t sel = kNone16;
            if (best != kNoClaim) {
              sel = (uint32_t)best & 0xFFFFu;
              atomicMin(&sm.claimC[sel], (best & 0xFFFFFFFF00000000ull) | sm.tseed[t]);
            }
            sm.fsel[t] = (uint16_t)sel;
          }
        }
        __syncwarp();
      }
      // ---- T2 resolve: the minimal claim wins the hit (track keys are unique: the low half of the claim names the
      //      winner, who puts the claim word back to "none"); everyone else counts a miss; closed tracks leave the list
      uint32_t kept = 0;
#pragma unroll 1
      for (uint32_t t0 = 0; t0 < n_act; t0 += 32) {
        const uint32_t t = t0 + lane;
        bool keep = false;
        uint32_t st = 0, seed = 0, cid = 0;
        float tx = 0.f, ty = 0.f;
        uint32_t tw = 0;
        if (t < n_act) {
          st = sm.tstate[t]; seed = sm.tseed[t]; cid = sm.tcid[t];
          tx = sm.ttx[t]; ty = sm.tty[t]; tw = sm.twin[t];
          const uint32_t fc = nC ? sm.fsel[t] : kNone16;
          if (fc != kNone16 && (uint32_t)sm.claimC[fc] == seed) {
            sm.claimC[fc] = kNoClaim;
            const uint32_t m = st & 0xFFu, q = st >> 16, lq = (uint32_t)i - 1u + m;
            const Hit hq = load_hit(slab + sm.src[lq] + (q - sm.lo[lq]));
            const Hit hc = load_hit(recC + fc);
            tw = pack_windows(__ldg(fwd_win + C0 + fc));
            const float dz = __fsub_rn(hc.z, hq.z);
            tx = __fdiv_rn(__fsub_rn(hc.x, hq.x), dz);
            ty = __fdiv_rn(__fsub_rn(hc.y, hq.y), dz);
            atomicOr(&usedC[fc >> 5], 1u << (fc & 31u));
            link[C0 + fc] = (uint16_t)q;
            st = ((C0 + fc) << 16) | (st & 0x8000u) | ((track_n_hits(st) + 1u) << 8);
            keep = true;
          } else {
            const uint32_t m = (st & 0xFFu) + 1u;
            if (m > (uint32_t)P.max_skipped) {
              a.trk_final[trk0 + cid] = st;
              const uint32_t n = track_n_hits(st);
              if (n >= 4 || (st & 0x8000u)) { out_tracks += 1; out_hits += n; }
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
          sm.tstate[pos] = st; sm.tseed[pos] = (uint16_t)seed; sm.tcid[pos] = (uint16_t)cid;
          sm.ttx[pos] = tx; sm.tty[pos] = ty; sm.twin[pos] = tw;
        }
        kept += __popc(bal);
      }
      n_act = kept;
      VELO_CHECK(g, n_act <= kSeg, 305);
      __syncwarp();
    }

    // A new track from an accepted entry: `rank` = accepted middle hits below its b (tracks are created in ascending b).
    auto create_track = [&](unsigned long long en, uint32_t rank) {
      const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
      const uint32_t slot = n_act + rank, cid = n_created + rank;
      VELO_CHECK(g, 3 * (cid + 1) <= sm.lo[L], 304);  // a track has three hits of its own: slots [co/3, (co+n)/3)
      if (slot < kSeg) {
        const Hit hb = load_hit(recB + kb), hc = load_hit(recC + ic);
        const float dz = __fsub_rn(hc.z, hb.z);
        sm.ttx[slot] = __fdiv_rn(__fsub_rn(hc.x, hb.x), dz);
        sm.tty[slot] = __fdiv_rn(__fsub_rn(hc.y, hb.y), dz);
        const float S = __uint_as_float((uint32_t)(en >> 32));
        sm.tstate[slot] = ((C0 + ic) << 16) | (S <= P.s_weak ? 0x8000u : 0u) | (3u << 8);
        sm.tseed[slot] = (uint16_t)(B0 + kb);
        sm.tcid[slot] = (uint16_t)cid;
        sm.twin[slot] = pack_windows(__ldg(fwd_win + C0 + ic));
        link[B0 + kb] = (uint16_t)(A0 + ia);
        link[C0 + ic] = (uint16_t)(B0 + kb);
        // layer A leaves after this iteration: its used flags are never read again
        atomicOr(&usedB[kb >> 5], 1u << (kb & 31u));
        atomicOr(&usedC[ic >> 5], 1u << (ic & 31u));
        return false;
      }
      return true;  // out of track slots: redone by the CTA-per-event kernel
    };

    // ---- T3 + T4 over the list of layer B
    if (n_t && n_t <= 32 && !overflow) {
      // A list of one round (55 % of the layers at nu = 6) is resolved in registers: lanes with equal b, a or c find each
      // other with match_any and compare keys by shuffle — the same minima as below, no shared-memory atomics, no resets.
      const unsigned long long en = ent0;
      const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
      const bool valid = en != kNoClaim && !((usedA[ia >> 5] >> (ia & 31u)) & 1u) && !((usedB[kb >> 5] >> (kb & 31u)) & 1u) &&
                         !((usedC[ic >> 5] >> (ic & 31u)) & 1u);
      // is the lane's key the smallest among the lanes that take part and carry the same `what`?
      auto holds_min = [&](bool takes_part, uint32_t what, unsigned long long key) {
        uint32_t peers = __match_any_sync(kFull, takes_part ? what : (0x10000u | lane)) & ~(1u << lane);
        bool least = takes_part;
#pragma unroll 1
        while (__any_sync(kFull, peers != 0)) {
          const uint32_t src = peers ? (uint32_t)__ffs(peers) - 1u : lane;
          const unsigned long long other = __shfl_sync(kFull, key, src);
          if (peers && other < key) least = false;
          peers &= peers - 1u;
        }
        return least;
      };
      // T3: argmin per middle hit on (bits(S), a, c); T4: the winner claims its a and its c with (bits(S), b)
      const bool best = holds_min(valid, kb, (en & 0xFFFFFFFF00000000ull) | (ia << 16) | ic);
      const unsigned long long tkey = (en & 0xFFFFFFFF00000000ull) | kb;
      const bool acc = holds_min(best, ia, tkey) & holds_min(best, ic, tkey);
      const uint32_t accm = __ballot_sync(kFull, acc);
      if (accm) {
        uint32_t rank = 0;  // accepted middle hits below this one
#pragma unroll 1
        for (uint32_t rest = accm; rest; rest &= rest - 1u) rank += __shfl_sync(kFull, kb, __ffs(rest) - 1) < kb ? 1u : 0u;
        if (acc) overflow = create_track(en, rank);
        overflow = __any_sync(kFull, overflow);
        n_act = min(n_act + (uint32_t)__popc(accm), kSeg);
        n_created += __popc(accm);
      }
      __syncwarp();
    } else if (n_t && !overflow) {
      const uint32_t rounds = (n_t + 31) / 32;
      auto entry = [&](uint32_t r) -> unsigned long long {
        if (r == 0) return ent0;
        if (r == 1) return ent1;
        const uint32_t k = r * 32 + lane;
        return k < n_t ? __ldg(trip + B0 + k) : kNoClaim;
      };
      // T3: entries whose three hits are unused take part in the argmin of their middle hit on (bits(S), a, c)
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
        const bool valid = en != kNoClaim && !((usedA[ia >> 5] >> (ia & 31u)) & 1u) && !((usedB[kb >> 5] >> (kb & 31u)) & 1u) &&
                           !((usedC[ic >> 5] >> (ic & 31u)) & 1u);
        VELO_CHECK(g, en == kNoClaim || (ia < sm.lo[i + 1] - A0 && kb < A0 - B0 && ic < nC && ia < (uint32_t)C::kCap && kb < (uint32_t)C::kCap), 303);
        if (valid) atomicMin(&sm.bestB[kb], (en & 0xFFFFFFFF00000000ull) | (ia << 16) | ic);
      }
      __syncwarp();
      // the entries that won their middle hit are marked; bestB[] then goes back to "none" and serves as claimA[]
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
        const unsigned long long key = (en & 0xFFFFFFFF00000000ull) | (ia << 16) | ic;
        // (an entry with a used hit never equals the key in bestB: keys of one middle hit are distinct)
        const uint32_t bal = __ballot_sync(kFull, en != kNoClaim && sm.bestB[kb] == key);
        if (lane == 0) sm.beste[r] = bal;
      }
      __syncwarp();
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        if (en != kNoClaim) sm.bestB[((uint32_t)en >> 10) & 0x3FFu] = kNoClaim;
      }
      __syncwarp();
      unsigned long long* claimA = sm.bestB;
      // T4a: the triplet of every middle hit claims its a and its c with (bits(S), b)
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
        if ((sm.beste[r] >> lane) & 1u) {
          const unsigned long long tkey = (en & 0xFFFFFFFF00000000ull) | kb;
          atomicMin(&claimA[ia], tkey);
          atomicMin(&sm.claimC[ic], tkey);
        }
      }
      __syncwarp();
      // T4b: accepted iff it holds the minimal key on both its a and its c
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, kb = ((uint32_t)en >> 10) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
        const unsigned long long tkey = (en & 0xFFFFFFFF00000000ull) | kb;
        const bool acc = ((sm.beste[r] >> lane) & 1u) && claimA[ia] == tkey && sm.claimC[ic] == tkey;
        const uint32_t bal = __ballot_sync(kFull, acc);
        if (acc) atomicOr(&sm.accw[kb >> 5], 1u << (kb & 31u));
        if (lane == 0) sm.acce[r] = bal;
      }
      __syncwarp();
      // new tracks in ascending b: rank of a middle hit = accepted middle hits below it
      const uint32_t wv = lane < kWords ? sm.accw[lane] : 0u;
      const uint32_t pc = __popc(wv);
      const uint32_t incl = warp_incl_scan(pc, lane);
      const uint32_t excl = incl - pc;
      const uint32_t n_acc = __shfl_sync(kFull, incl, 31);
      if (n_acc) {
#pragma unroll 1
        for (uint32_t r = 0; r < rounds; ++r) {
          const unsigned long long en = entry(r);
          const uint32_t kb = ((uint32_t)en >> 10) & 0x3FFu;
          const uint32_t below = __shfl_sync(kFull, excl, kb >> 5);
          const uint32_t word = __shfl_sync(kFull, wv, kb >> 5);
          if ((sm.acce[r] >> lane) & 1u) {
            if (create_track(en, below + __popc(word & ((1u << (kb & 31u)) - 1u)))) overflow = true;
          }
        }
        overflow = __any_sync(kFull, overflow);
        n_act = min(n_act + n_acc, kSeg);
        n_created += n_acc;
      }
      __syncwarp();
      // every word touched goes back to "none"
#pragma unroll 1
      for (uint32_t r = 0; r < rounds; ++r) {
        const unsigned long long en = entry(r);
        if (en != kNoClaim) {
          const uint32_t ia = ((uint32_t)en >> 20) & 0x3FFu, ic = (uint32_t)en & 0x3FFu;
          claimA[ia] = kNoClaim; sm.claimC[ic] = kNoClaim;
        }
      }
      if (lane < kWords) sm.accw[lane] = 0;
    }
    // the ring slot of layer A takes layer i - 3
    if (lane < kWords) usedA[lane] = 0;
    __syncwarp();
  }

  if (overflow) {
    if (lane == 0) a.redo_list[which_redo][atomicAdd(a.counters + kCtrRedo + which_redo, 1u)] = e;
    return;
  }

  // ---- the tracks still active are closed.  T5 (keep >= 4 hits, or 3 hits with S_seed <= s_weak), the hit lists and the
  //      fit (A8) are done per track by compact_tracks_kernel, a thread per track: here they would be one more chain
  //      of dependent loads in a kernel that lives on latency (39 % of its time when it was done here).
#pragma unroll 1
  for (uint32_t t = lane; t < n_act; t += 32) {
    const uint32_t st = sm.tstate[t];
    a.trk_final[trk0 + sm.tcid[t]] = st;
    const uint32_t n = track_n_hits(st);
    if (n >= 4 || (st & 0x8000u)) { out_tracks += 1; out_hits += n; }
  }
  out_tracks = __reduce_add_sync(kFull, out_tracks);
  out_hits = __reduce_add_sync(kFull, out_hits);
  if (lane == 0) {
    a.counts[e] = ((unsigned long long)out_tracks << 32) | out_hits;
    a.ev_flags[e] = kEvFinal | (n_created << 8);
  }
}

// Resident one-warp CTAs take the events of class kLevel from their list.
template <class C>
__global__ void __launch_bounds__(32) velo_follow_kernel(const __grid_constant__ TrackLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FollowSmem<C>& sm = *reinterpret_cast<FollowSmem<C>*>(smem_raw);
  const uint32_t lane = lane_id();
  const uint32_t n = a.counters[kCtrFollow + C::kLevel];
  if (blockIdx.x >= n) return;
#pragma unroll 1
  for (uint32_t k = lane; k < (uint32_t)C::kCap; k += 32) { sm.claimC[k] = kNoClaim; sm.bestB[k] = kNoClaim; }
  __syncwarp();
#pragma unroll 1
  for (;;) {
    uint32_t idx = 0;
    if (lane == 0) idx = atomicAdd(a.counters + kCtrFollowCursor + C::kLevel, 1u);
    idx = __shfl_sync(kFull, idx, 0);
    if (idx >= n) return;
    follow_event<C>(a, a.flw_list[C::kLevel][idx], sm);
    __syncwarp();
  }
}

template <class C>
cudaError_t launch_follow_instance(const TrackLaunch& a, uint32_t n_sms, cudaStream_t stream) {
  const uint32_t per_sm = min(32u, (227u * 1024u) / ((uint32_t)sizeof(FollowSmem<C>) + 1024u));
  const uint32_t grid = min(a.n_events, n_sms * max(per_sm, 1u));
  velo_follow_kernel<C><<<grid, 32, sizeof(FollowSmem<C>), stream>>>(a);
  return cudaGetLastError();
}

}  // namespace

cudaError_t follow_prepare() {
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  cudaError_t err = cudaFuncSetAttribute(velo_follow_kernel<Follow256>, attr, (int)sizeof(FollowSmem<Follow256>));
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_follow_kernel<Follow512>, attr, (int)sizeof(FollowSmem<Follow512>));
  if (err == cudaSuccess) err = cudaFuncSetAttribute(velo_follow_kernel<Follow1024>, attr, (int)sizeof(FollowSmem<Follow1024>));
  return err;
}

cudaError_t launch_follow(const TrackLaunch& a, uint32_t level, uint32_t n_sms, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  if (level == 0) return launch_follow_instance<Follow256>(a, n_sms, stream);
  if (level == 1) return launch_follow_instance<Follow512>(a, n_sms, stream);
  return launch_follow_instance<Follow1024>(a, n_sms, stream);
}

}  // namespace velo
