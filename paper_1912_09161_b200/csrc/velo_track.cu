// Kernel 2 of the VELO hot path: search by triplet (A5 seeding, A6 forwarding, A7 clone/ghost killing) and the
// straight-line fit (A8) — SURVEY.md §8(a); the algorithm is DESIGN.md reading R5 (T1..T5) of P:181-183 ("forming
// seeds of three hits from consecutive layers ('triplets'), and then extending these to the other layers"; "sort hits
// on every layer by phi for fast look-up") and R6 of P:149 (straight lines).
//
// One CTA per event ("a single event is assigned to one block, while intra-event parallelism is mapped to the threads
// within one block").  The 24 layer iterations are sequential; inside an iteration tracks (T1/T2) and middle
// hits (T3/T4) are processed one per thread.  All conflict rules are order-independent minima, implemented as 64-bit
// atomicMin on shared-memory claim words keyed (bits(S) << 32 | index): no "first thread wins" anywhere, so the
// result is exactly the oracle's.  Track slots and output positions come from block-wide ballot/prefix scans, which
// makes the output order deterministic (order of creation).
#include "velo_common.cuh"

namespace velo {
namespace {

constexpr int kThreads = 128;
constexpr uint32_t kCapLayer = 768;    // hits of one layer staged (claims, used flags, triplets)
constexpr uint32_t kCapTracks = 1024;  // tracks of one event kept in shared memory
constexpr unsigned long long kNoClaim = ~0ull;

struct Smem {
  unsigned long long claimA[kCapLayer], claimC[kCapLayer];
  uint32_t tripS[kCapLayer];
  uint16_t tripA[kCapLayer], tripC[kCapLayer];
  float seedS[kCapTracks];
  uint32_t choiceS[kCapTracks];
  uint16_t choiceC[kCapTracks];
  uint16_t newest[kCapTracks], previous[kCapTracks], seedB[kCapTracks];
  uint8_t nhits[kCapTracks], missed[kCapTracks];  // missed == 0xFF: closed
  uint8_t used[3][kCapLayer];
  uint32_t lo[kMaxLayers + 1];
  uint32_t warp_tot[kThreads / 32];
  uint32_t overflow;
};

// Exclusive prefix of `v` over the block in thread order; returns the block total in `total`.
__device__ __forceinline__ uint32_t block_scan(uint32_t v, uint32_t* warp_tot, uint32_t& total) {
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(kFull, incl, d);
    if (lane >= (uint32_t)d) incl += t;
  }
  __syncthreads();  // protects warp_tot against the previous use
  if (lane == 31) warp_tot[warp] = incl;
  __syncthreads();
  uint32_t off = 0;
  total = 0;
#pragma unroll
  for (int w = 0; w < kThreads / 32; ++w) {
    if (w < (int)warp) off += warp_tot[w];
    total += warp_tot[w];
  }
  return off + incl - v;
}

// First index in [0, n) of the sorted (signed) phi array with phi >= target, or n.
__device__ __forceinline__ uint32_t lower_bound_phi(const int16_t* __restrict__ phi, uint32_t n, int target) {
  uint32_t a = 0, b = n;
  while (a < b) {
    const uint32_t mid = (a + b) >> 1;
    if ((int)__ldg(phi + mid) < target) a = mid + 1; else b = mid;
  }
  return a;
}

__global__ void __launch_bounds__(kThreads) velo_track_kernel(const TrackLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  const DeviceGeometry& g = a.geo;
  const allen_velo_params_t P = g.params;
  const uint32_t e = blockIdx.x, L = g.n_layers, tid = threadIdx.x;

  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t n_cl = a.clusters.event_offsets[e + 1] - co;
  const uint32_t st = a.clusters.status[e];
  // events whose clusters were not produced or not written take no part in tracking
  const bool skip = (st & (ALLEN_VELO_STATUS_BAD_HEADER | ALLEN_VELO_STATUS_TOO_MANY_CLUSTERS |
                           ALLEN_VELO_STATUS_CLUSTER_CAPACITY | ALLEN_VELO_STATUS_STAGE_OVERFLOW)) != 0;
  if (skip || n_cl == 0) {
    if (tid == 0) a.counts[e] = 0;
    return;
  }
  if ((unsigned long long)co + n_cl > a.clusters.capacity) {  // tracking scratch is indexed by cluster
    if (tid == 0) { atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW); a.counts[e] = 0; }
    return;
  }
  for (uint32_t l = tid; l <= L; l += kThreads) sm.lo[l] = a.clusters.layer_offsets[e * L + l] - co;
  if (tid == 0) sm.overflow = 0;
  __syncthreads();
  for (uint32_t l = tid; l < L; l += kThreads)
    if (sm.lo[l + 1] - sm.lo[l] > kCapLayer) sm.overflow = 1;
  for (uint32_t i = tid; i < 3 * kCapLayer; i += kThreads) (&sm.used[0][0])[i] = 0;
  for (uint32_t i = tid; i < kCapLayer; i += kThreads) { sm.claimA[i] = kNoClaim; sm.claimC[i] = kNoClaim; }
  __syncthreads();
  if (sm.overflow) {
    if (tid == 0) { atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW); a.counts[e] = 0; }
    return;
  }

  const float* __restrict__ X = a.clusters.x + co;
  const float* __restrict__ Y = a.clusters.y + co;
  const float* __restrict__ Z = a.clusters.z + co;
  const int16_t* __restrict__ PHI = a.clusters.phi16 + co;
  uint16_t* link = a.link + co;

  uint32_t n_tracks = 0;  // block-uniform

  for (int i = (int)L - 1; i >= 2; --i) {
    const uint32_t A0 = sm.lo[i], A1 = sm.lo[i + 1], B0 = sm.lo[i - 1], C0 = sm.lo[i - 2];
    const uint32_t nA = A1 - A0, nB = A0 - B0, nC = B0 - C0;
    uint8_t* usedA = sm.used[i % 3];
    uint8_t* usedB = sm.used[(i - 1) % 3];
    uint8_t* usedC = sm.used[(i - 2) % 3];
    if (i != (int)L - 1) {  // layer C enters the window: nothing of it is used yet
      for (uint32_t k = tid; k < nC; k += kThreads) usedC[k] = 0;
      __syncthreads();
    }

    // ---- T1 forward: best unused hit of layer C per active track, claim it with (bits(S), track_key)
    for (uint32_t t = tid; t < n_tracks; t += kThreads) {
      sm.choiceC[t] = 0xFFFF;
      if (sm.missed[t] == 0xFF || nC == 0) continue;
      const uint32_t p = sm.previous[t], q = sm.newest[t];
      const float xp = __ldg(X + p), yp = __ldg(Y + p), zp = __ldg(Z + p);
      const float xq = __ldg(X + q), yq = __ldg(Y + q), zq = __ldg(Z + q);
      const int16_t phq = __ldg(PHI + q);
      const int w = P.w_fwd_phi16;
      const uint32_t s0 = lower_bound_phi(PHI + C0, nC, (int)(int16_t)(uint16_t)((int)phq - w));
      unsigned long long best = kNoClaim;
      for (uint32_t k = 0; k < nC; ++k) {
        uint32_t idx = s0 + k;
        if (idx >= nC) idx -= nC;
        const uint32_t c = C0 + idx;
        const int d = dphi16(__ldg(PHI + c), phq);
        if (d > w || d < -w) break;
        if (usedC[idx]) continue;
        const float S = scatter(xp, yp, zp, xq, yq, zq, __ldg(X + c), __ldg(Y + c), __ldg(Z + c));
        if (!(S <= P.s_fwd)) continue;
        const unsigned long long key = ((unsigned long long)__float_as_uint(S) << 32) | c;
        best = key < best ? key : best;
      }
      if (best != kNoClaim) {
        const uint32_t c = (uint32_t)best, sb = (uint32_t)(best >> 32);
        sm.choiceC[t] = (uint16_t)c;
        sm.choiceS[t] = sb;
        atomicMin(&sm.claimC[c - C0], ((unsigned long long)sb << 32) | sm.seedB[t]);
      }
    }
    __syncthreads();
    // ---- T2 resolve: the minimal claim wins the hit; everyone else counts a miss
    for (uint32_t t = tid; t < n_tracks; t += kThreads) {
      if (sm.missed[t] == 0xFF) continue;
      const uint32_t c = sm.choiceC[t];
      bool won = false;
      if (c != 0xFFFF) won = sm.claimC[c - C0] == (((unsigned long long)sm.choiceS[t] << 32) | sm.seedB[t]);
      if (won) {
        link[c] = sm.newest[t];
        sm.previous[t] = sm.newest[t];
        sm.newest[t] = (uint16_t)c;
        sm.nhits[t] += 1;
        sm.missed[t] = 0;
        usedC[c - C0] = 1;
      } else {
        const uint32_t m = sm.missed[t] + 1u;
        sm.missed[t] = m > (uint32_t)P.max_skipped ? 0xFF : (uint8_t)m;
      }
    }
    __syncthreads();
    for (uint32_t k = tid; k < nC; k += kThreads) sm.claimC[k] = kNoClaim;
    __syncthreads();

    // ---- T3 seed: best (a, c) per unused middle hit b; claim a and c with (bits(S), b)
    for (uint32_t kb = tid; kb < nB; kb += kThreads) {
      sm.tripS[kb] = 0xFFFFFFFFu;
      if (usedB[kb] || nA == 0 || nC == 0) continue;
      const uint32_t b = B0 + kb;
      const float xb = __ldg(X + b), yb = __ldg(Y + b), zb = __ldg(Z + b);
      const int16_t phb = __ldg(PHI + b);
      const int w = P.w_seed_phi16;
      const int target = (int)(int16_t)(uint16_t)((int)phb - w);
      const uint32_t sA = lower_bound_phi(PHI + A0, nA, target);
      const uint32_t sC = lower_bound_phi(PHI + C0, nC, target);
      uint32_t bestS = 0xFFFFFFFFu, bestA = 0, bestC = 0;
      bool found = false;
      for (uint32_t ka = 0; ka < nA; ++ka) {
        uint32_t ia = sA + ka;
        if (ia >= nA) ia -= nA;
        const uint32_t ha = A0 + ia;
        const int da = dphi16(__ldg(PHI + ha), phb);
        if (da > w || da < -w) break;
        if (usedA[ia]) continue;
        const float xa = __ldg(X + ha), ya = __ldg(Y + ha), za = __ldg(Z + ha);
        const float dz_ab = __fsub_rn(zb, za);
        const float tx = __fdiv_rn(__fsub_rn(xb, xa), dz_ab), ty = __fdiv_rn(__fsub_rn(yb, ya), dz_ab);
        if (!(fabsf(tx) <= P.max_slope) || !(fabsf(ty) <= P.max_slope)) continue;
        for (uint32_t kc = 0; kc < nC; ++kc) {
          uint32_t ic = sC + kc;
          if (ic >= nC) ic -= nC;
          const uint32_t hc = C0 + ic;
          const int dc = dphi16(__ldg(PHI + hc), phb);
          if (dc > w || dc < -w) break;
          if (usedC[ic]) continue;
          const float dz = __fsub_rn(__ldg(Z + hc), zb);
          const float ex = __fsub_rn(__fmaf_rn(tx, dz, xb), __ldg(X + hc));
          const float ey = __fsub_rn(__fmaf_rn(ty, dz, yb), __ldg(Y + hc));
          const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
          if (!(S <= P.s_seed)) continue;
          const uint32_t sb = __float_as_uint(S);
          // argmin over (bits(S), a, c)
          const bool better = !found || sb < bestS || (sb == bestS && (ha < bestA || (ha == bestA && hc < bestC)));
          if (better) { bestS = sb; bestA = ha; bestC = hc; found = true; }
        }
      }
      if (found) {
        sm.tripS[kb] = bestS;
        sm.tripA[kb] = (uint16_t)bestA;
        sm.tripC[kb] = (uint16_t)bestC;
        const unsigned long long key = ((unsigned long long)bestS << 32) | b;
        atomicMin(&sm.claimA[bestA - A0], key);
        atomicMin(&sm.claimC[bestC - C0], key);
      }
    }
    __syncthreads();
    // ---- T4 resolve: accepted iff the triplet holds the minimal key on both its a and its c; new tracks take
    //      slots in ascending b (block prefix scan)
    for (uint32_t base = 0; base < nB; base += kThreads) {
      const uint32_t kb = base + tid;
      bool accepted = false;
      uint32_t ha = 0, hc = 0, sb = 0;
      if (kb < nB && sm.tripS[kb] != 0xFFFFFFFFu) {
        ha = sm.tripA[kb]; hc = sm.tripC[kb]; sb = sm.tripS[kb];
        const unsigned long long key = ((unsigned long long)sb << 32) | (B0 + kb);
        accepted = sm.claimA[ha - A0] == key && sm.claimC[hc - C0] == key;
      }
      uint32_t total;
      const uint32_t slot = n_tracks + block_scan(accepted ? 1u : 0u, sm.warp_tot, total);
      if (accepted) {
        if (slot < kCapTracks) {
          const uint32_t b = B0 + kb;
          sm.newest[slot] = (uint16_t)hc;
          sm.previous[slot] = (uint16_t)b;
          sm.seedB[slot] = (uint16_t)b;
          sm.seedS[slot] = __uint_as_float(sb);
          sm.nhits[slot] = 3;
          sm.missed[slot] = 0;
          link[b] = (uint16_t)ha;
          link[hc] = (uint16_t)b;
          usedA[ha - A0] = 1;
          usedB[kb] = 1;
          usedC[hc - C0] = 1;
        } else {
          sm.overflow = 1;
        }
      }
      n_tracks += total;
      if (n_tracks > kCapTracks) n_tracks = kCapTracks;
    }
    __syncthreads();
    for (uint32_t k = tid; k < nA; k += kThreads) sm.claimA[k] = kNoClaim;
    for (uint32_t k = tid; k < nC; k += kThreads) sm.claimC[k] = kNoClaim;
    __syncthreads();
  }

  if (sm.overflow) {
    if (tid == 0) { atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW); a.counts[e] = 0; }
    return;
  }

  // ---- T5 finalise + A8 fit: keep >= 4 hits, or 3 hits with S_seed <= s_weak; compact in order of creation
  uint32_t out_tracks = 0, out_hits = 0;
  const uint32_t trk0 = co / 3;
  for (uint32_t base = 0; base < n_tracks; base += kThreads) {
    const uint32_t t = base + tid;
    uint32_t n = 0;
    if (t < n_tracks) {
      n = sm.nhits[t];
      if (n == 3 && !(sm.seedS[t] <= P.s_weak)) n = 0;
    }
    uint32_t total;
    const uint32_t off = block_scan(n ? ((1u << 20) | n) : 0u, sm.warp_tot, total);
    if (n) {
      const uint32_t ot = out_tracks + (off >> 20), oh = out_hits + (off & 0xFFFFFu);
      // hits in order of addition: walk the links from the newest hit backwards
      double sz = 0, sx = 0, sy = 0;
      uint32_t h = sm.newest[t];
      for (int k = (int)n - 1; k >= 0; --k) {
        a.hits_slab[co + oh + k] = (uint16_t)h;
        sz += (double)__ldg(Z + h); sx += (double)__ldg(X + h); sy += (double)__ldg(Y + h);
        if (k) h = link[h];
      }
      const double inv = 1.0 / (double)n;
      const double zm = sz * inv, xm = sx * inv, ym = sy * inv;
      double szz = 0, szx = 0, szy = 0;
      h = sm.newest[t];
      for (int k = (int)n - 1; k >= 0; --k) {
        const double dz = (double)__ldg(Z + h) - zm;
        szz += dz * dz;
        szx += dz * ((double)__ldg(X + h) - xm);
        szy += dz * ((double)__ldg(Y + h) - ym);
        if (k) h = link[h];
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
__global__ void __launch_bounds__(128) compact_tracks_kernel(const CompactTracksLaunch a) {
  const uint32_t e = blockIdx.x;
  const unsigned long long o0 = a.offsets[e], o1 = a.offsets[e + 1];
  const uint32_t T0 = (uint32_t)(o0 >> 32), H0 = (uint32_t)o0;
  const uint32_t nT = (uint32_t)(o1 >> 32) - T0, nH = (uint32_t)o1 - H0;
  if (threadIdx.x == 0) {
    a.out.event_offsets[e] = T0;
    if (e + 1 == a.n_events) a.out.event_offsets[e + 1] = T0 + nT;
  }
  const bool fits = (unsigned long long)T0 + nT <= a.out.capacity_tracks &&
                    (unsigned long long)H0 + nH <= a.out.capacity_hits;
  if (!fits) {
    if (threadIdx.x == 0 && nT) atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_TRACK_CAPACITY);
    return;
  }
  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t trk0 = co / 3;
  for (uint32_t t = threadIdx.x; t < nT; t += blockDim.x) {
    const float4 f = a.trk_fit[trk0 + t];
    a.out.x0[T0 + t] = f.x; a.out.y0[T0 + t] = f.y; a.out.tx[T0 + t] = f.z; a.out.ty[T0 + t] = f.w;
    a.out.hit_offsets[T0 + t] = H0 + a.trk_hitoff[trk0 + t];
  }
  for (uint32_t k = threadIdx.x; k < nH; k += blockDim.x) a.out.hits[H0 + k] = a.hits_slab[co + k];
  if (threadIdx.x == 0 && e + 1 == a.n_events) a.out.hit_offsets[T0 + nT] = H0 + nH;
}

}  // namespace

cudaError_t launch_track(const TrackLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  cudaError_t err = cudaFuncSetAttribute(velo_track_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(Smem));
  if (err != cudaSuccess) return err;
  velo_track_kernel<<<a.n_events, kThreads, sizeof(Smem), stream>>>(a);
  return cudaGetLastError();
}

cudaError_t launch_compact_tracks(const CompactTracksLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  compact_tracks_kernel<<<a.n_events, 128, 0, stream>>>(a);
  return cudaGetLastError();
}

}  // namespace velo
