// Kernel 2 of the VELO hot path: search by triplet (A5 seeding, A6 forwarding, A7 clone/ghost killing) and the
// straight-line fit (A8) — SURVEY.md §8(a); the algorithm is DESIGN.md reading R5 (T1..T5) of P:181-183 ("forming
// seeds of three hits from consecutive layers ('triplets'), and then extending these to the other layers"; "sort hits
// on every layer by phi for fast look-up") and R6 of P:149 (straight lines).
//
// One CTA per event ("a single event is assigned to one block, while intra-event parallelism is mapped to the threads
// within one block").  The L-2 layer iterations are sequential.  Design for sm_100a:
//  * the three layers of an iteration (plus the one being prefetched) live in shared memory as 16-byte hit records
//    (x, y, z, phi16 | used << 16) in a ring of four slots: one LDS.128 per candidate; the next layer is brought in
//    with cp.async one iteration ahead, so its DRAM latency hides behind the current iteration;
//  * phi look-up uses a 128-bucket start table per layer, built while the layer is staged (no binary search);
//  * seeding is flattened: S1 lists (b, a) doublets inside the phi window, S2 gives every doublet one thread that
//    scans b's window on layer C; the per-b argmin is a 64-bit shared-memory atomicMin on (bits(S), a, c);
//  * all conflict rules are order-independent minima on packed keys (bits(S) << 32 | index): no "first thread wins",
//    so the result is exactly the oracle's whatever the thread schedule;
//  * compaction of the clusters (A9) rides along: in the first instance a fifth warp copies the event's layers from
//    the cluster kernel's slab to their final place while the four tracking warps (own named barrier) search;
//  * the kernel is instantiated for three staging capacities (256 / 512 / 1024 hits per layer); every event is taken
//    by the smallest instance it fits, and an instance that runs out of track slots hands the event to the next one.
#include <cuda_pipeline.h>

#include "velo_common.cuh"

namespace velo {
namespace {

constexpr unsigned long long kNoClaim = ~0ull;
constexpr int kBuckets = 128;
constexpr int kBucketShift = 9;  // 65536 / 128
constexpr uint32_t kUsedBit = 0x10000u;

struct __align__(16) Hit {
  float x, y, z;
  uint32_t w;  // phi16 (low 16 bits, two's complement) | used << 16
};

template <int kThreads_, int kCap_, int kCapTracks_, int kCapDoublets_, int kLevel_, bool kLast_, bool kCopier_>
struct Cfg {
  static constexpr int kThreads = kThreads_;
  static constexpr int kCap = kCap_;            // hits of one layer staged
  static constexpr int kCapTracks = kCapTracks_;
  static constexpr int kCapDoublets = kCapDoublets_;
  static constexpr int kLevel = kLevel_;
  static constexpr bool kLast = kLast_;
  static constexpr bool kCopier = kCopier_;      // an extra warp moves the event's clusters from the slab to the output
  static constexpr int kBlock = kThreads + (kCopier ? 32 : 0);
  static constexpr int kWarps = kThreads / 32;
  static constexpr int kRoundsB = (kCap + kThreads - 1) / kThreads;
  static constexpr int kRoundsT = (kCapTracks + kThreads - 1) / kThreads;
};
#ifndef VELO_TRK_S_THREADS
#define VELO_TRK_S_THREADS 128
#endif
#ifndef VELO_TRK_S_TRACKS
#define VELO_TRK_S_TRACKS 384
#endif
#ifndef VELO_TRK_S_DOUBLETS
#define VELO_TRK_S_DOUBLETS 256
#endif
using CfgS = Cfg<VELO_TRK_S_THREADS, 256, VELO_TRK_S_TRACKS, VELO_TRK_S_DOUBLETS, 0, false, true>;
using CfgM = Cfg<256, 512, 1024, 1024, 1, false, false>;
using CfgL = Cfg<512, 1024, 2048, 2048, 2, true, false>;

template <class C>
struct Smem {
  Hit rec[4][C::kCap];
  unsigned long long best[C::kCap];  // T3: per-b argmin key; T1/T2: forward claims on layer C (aliased by phase)
  unsigned long long claimA[C::kCap], claimC[C::kCap];
  uint32_t doublets[C::kCapDoublets];  // b_local | a_local << 16
  float ttx[C::kCapTracks], tty[C::kCapTracks];  // slopes of the last segment (older -> newest hit)
  uint32_t tstate[C::kCapTracks];                // newest << 16 | weak_ok << 15 | nhits << 8 | missed (0xFF: closed)
  uint16_t tseedB[C::kCapTracks];                // track_key: event-local index of the seed's middle hit
  uint16_t bucket[4][kBuckets + 2];
  uint32_t lo[kMaxLayers + 1];
  uint32_t src[kMaxLayers];  // first entry of every layer in the arrays X, Y, Z, PHI are read from
  uint32_t warp_tot[C::kRoundsB > C::kRoundsT ? C::kRoundsB : C::kRoundsT][C::kWarps];
  uint32_t n_doublets;
  uint32_t min_active[2];
  uint32_t flags;
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

// Barrier over the tracking threads only (the copier warp, if any, runs on its own).
template <class C>
__device__ __forceinline__ void tsync() {
  if (C::kCopier) asm volatile("bar.sync 1, %0;" ::"n"(C::kThreads) : "memory");
  else __syncthreads();
}

template <class C>
struct Ctx {
  Smem<C>& sm;
  const float* __restrict__ X;
  const float* __restrict__ Y;
  const float* __restrict__ Z;
  const int16_t* __restrict__ PHI;
  allen_velo_params_t P;
};

// Bring layer `l` into ring slot l & 3: x, y, z by cp.async (4-byte copies into the 16-byte records), the phi word and
// the bucket table by this thread.  Completion: __pipeline_wait_prior(0) + __syncthreads() by the caller.
template <class C>
__device__ __forceinline__ void stage_layer(const Ctx<C>& c, uint32_t l) {
  Smem<C>& sm = c.sm;
  const uint32_t base = sm.src[l], n = sm.lo[l + 1] - sm.lo[l];
  Hit* rec = sm.rec[l & 3];
  uint16_t* bucket = sm.bucket[l & 3];
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
    const int bk = (int)((ph ^ 0x8000u) >> kBucketShift);
    const int bp = k ? (int)((((uint32_t)(uint16_t)__ldg(c.PHI + base + k - 1)) ^ 0x8000u) >> kBucketShift) : -1;
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

// Copy clusters [k0, k1) of layer l (layer-local indices) from the slab to the compacted output.
__device__ __forceinline__ void copy_clusters(const TrackLaunch& a, uint32_t src, uint32_t dst, uint32_t n,
                                              uint32_t first, uint32_t step) {
#pragma unroll 1
  for (uint32_t k = first; k < n; k += step) {
    const uint32_t s = src + k, d = dst + k;
    const uint32_t key = __ldg(a.slab.key + s), np = __ldg(a.slab.n_pixels + s);
    const uint32_t sc = __ldg(a.slab.sum_col + s), sr = __ldg(a.slab.sum_row + s);
    const float x = __ldg(a.slab.x + s), y = __ldg(a.slab.y + s), z = __ldg(a.slab.z + s);
    const int16_t ph = __ldg(a.slab.phi16 + s);
    a.clusters.key[d] = key; a.clusters.n_pixels[d] = np; a.clusters.sum_col[d] = sc; a.clusters.sum_row[d] = sr;
    a.clusters.x[d] = x; a.clusters.y[d] = y; a.clusters.z[d] = z; a.clusters.phi16[d] = ph;
    if (a.clusters.checksum) a.clusters.checksum[d] = __ldg(a.slab.checksum + s);
  }
}

template <class C>
__global__ void __launch_bounds__(C::kBlock) velo_track_kernel(const __grid_constant__ TrackLaunch a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<C>& sm = *reinterpret_cast<Smem<C>*>(smem_raw);
  const DeviceGeometry& g = a.geo;
  const uint32_t e = blockIdx.x, L = g.n_layers, tid = threadIdx.x;
  const uint32_t lane = lane_id(), warp = tid >> 5;

  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t n_cl = a.clusters.event_offsets[e + 1] - co;
  const uint32_t st0 = a.clusters.status[e];
  if (n_cl == 0) {
    if (C::kLevel == 0 && tid == 0) a.counts[e] = 0;
    return;
  }
  if ((unsigned long long)co + n_cl > a.clusters.capacity) {  // the output (or the per-cluster scratch) cannot hold it
    if (C::kLevel == 0 && tid == 0) {
      atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_CLUSTER_CAPACITY);
      a.counts[e] = 0;
    }
    return;
  }
  // events whose clusters are incomplete, or too many for 16-bit hit indices, take no part in tracking
  const bool skip = (st0 & (ALLEN_VELO_STATUS_BAD_HEADER | ALLEN_VELO_STATUS_STAGE_OVERFLOW)) != 0 || n_cl > 65535u;
  // ---- which instance takes this event: the smallest whose staging capacity holds its busiest layer, unless a
  //      smaller instance ran out of track slots and passed it on (level[e])
  if (tid == 0) sm.flags = 0;
#pragma unroll 1
  for (uint32_t l = tid; l <= L; l += C::kBlock) sm.lo[l] = a.clusters.layer_offsets[e * L + l] - co;
  // the instance with the copier reads the slab the cluster kernel wrote; the others the output it has filled
#pragma unroll 1
  for (uint32_t l = tid; l < L; l += C::kBlock)
    sm.src[l] = C::kCopier ? a.slab_base[e * L + l] : a.clusters.layer_offsets[e * L + l];
  __syncthreads();
  {
    uint32_t mx = 0;
#pragma unroll 1
    for (uint32_t l = tid; l < L; l += C::kBlock) mx = max(mx, sm.lo[l + 1] - sm.lo[l]);
    if (mx) atomicMax(&sm.flags, mx);
  }
  __syncthreads();
  const uint32_t max_layer = sm.flags;
  const uint32_t natural = max_layer <= (uint32_t)CfgS::kCap ? 0u : max_layer <= (uint32_t)CfgM::kCap ? 1u : 2u;
  const uint32_t level = max(natural, (uint32_t)a.level[e]);  // level[e]: 0 unless raised by a smaller instance
  const bool fits = max_layer <= (uint32_t)C::kCap;
  const bool take = !skip && level == (uint32_t)C::kLevel && fits;
  __syncthreads();  // everyone has read sm.flags
  if (!take) {
    if (C::kCopier)  // the output is still to be filled: the whole CTA moves the event
#pragma unroll 1
      for (uint32_t l = 0; l < L; ++l)
        copy_clusters(a, sm.src[l], co + sm.lo[l], sm.lo[l + 1] - sm.lo[l], tid, C::kBlock);
    if (tid == 0) {
      if (C::kLevel == 0 && n_cl > 65535u) atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_TOO_MANY_CLUSTERS);
      if (C::kLevel == 0 && skip) a.counts[e] = 0;
      if (C::kLast && !skip && !fits) {  // busiest layer beyond the largest staging capacity
        atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);
        a.counts[e] = 0;
      }
    }
    return;
  }
  if (C::kCopier && tid >= (uint32_t)C::kThreads) {
    // copier warp: layers in the order the search stages them (their slab lines are then in L2 for both readers)
#pragma unroll 1
    for (int l = (int)L - 1; l >= 0; --l)
      copy_clusters(a, sm.src[l], co + sm.lo[l], sm.lo[l + 1] - sm.lo[l], lane, 32);
    __syncthreads();  // pairs with the barrier before the fit: the output arrays are complete
    return;
  }
  if (tid == 0) { sm.flags = 0; sm.min_active[0] = 0; sm.min_active[1] = 0; }

  Ctx<C> c{sm,
           C::kCopier ? a.slab.x : a.clusters.x, C::kCopier ? a.slab.y : a.clusters.y,
           C::kCopier ? a.slab.z : a.clusters.z, C::kCopier ? a.slab.phi16 : a.clusters.phi16, g.params};
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
    Hit* recA = sm.rec[i & 3];
    Hit* recB = sm.rec[(i - 1) & 3];
    Hit* recC = sm.rec[(i - 2) & 3];
    const uint16_t* bucketA = sm.bucket[i & 3];
    const uint16_t* bucketC = sm.bucket[(i - 2) & 3];

    __pipeline_wait_prior(0);
    tsync<C>();  // B1: layer C staged; tracks created by the previous T4 visible; claims re-initialised
    if (i >= 3) stage_layer(c, (uint32_t)i - 3);  // prefetch: needed at the top of the next iteration

    // ---- T1 forward: best hit of layer C per active track (nothing of C is used yet); claim with (bits(S), key)
    const uint32_t first = min(sm.min_active[i & 1], first_new);
    if (tid == 0) { sm.min_active[(i - 1) & 1] = 0xFFFFFFFFu; sm.n_doublets = 0; }
#pragma unroll 1
    for (uint32_t k = tid; k < max(nA, nC); k += C::kThreads) { sm.claimA[k] = kNoClaim; sm.claimC[k] = kNoClaim; }
    uint16_t* fsel = reinterpret_cast<uint16_t*>(sm.doublets);  // hit of layer C chosen by every track (T1 -> T2)
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
        const uint32_t s = sm.src[l] + (q - sm.lo[l]);
        xq = __ldg(c.X + s); yq = __ldg(c.Y + s); zq = __ldg(c.Z + s); phq = (int)__ldg(c.PHI + s);
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
    tsync<C>();  // B2
    // ---- T2 resolve: the minimal claim wins the hit (track keys are unique, so the low half of the claim names the
    //      winner); everyone else counts a miss
#pragma unroll 1
    for (uint32_t t = first + tid; t < n_tracks; t += C::kThreads) {
      const uint32_t st = sm.tstate[t];
      if ((st & 0xFFu) == 0xFFu) continue;
      const uint32_t fc = fsel[t];
      const bool won = fc != 0xFFFFu && (uint16_t)sm.best[fc] == sm.tseedB[t];
      if (won) {
        const uint32_t q = st >> 16, cg = C0 + fc;
        float xq, yq, zq;
        if (q < A1) {
          const Hit hq = q >= A0 ? recA[q - A0] : recB[q - B0];
          xq = hq.x; yq = hq.y; zq = hq.z;
        } else {
          uint32_t l = (uint32_t)i + 1;
#pragma unroll 1
          while (q >= sm.lo[l + 1]) ++l;
          const uint32_t s = sm.src[l] + (q - sm.lo[l]);
          xq = __ldg(c.X + s); yq = __ldg(c.Y + s); zq = __ldg(c.Z + s);
        }
        const Hit hc = recC[fc];
        const float dz = __fsub_rn(hc.z, zq);
        sm.ttx[t] = __fdiv_rn(__fsub_rn(hc.x, xq), dz);
        sm.tty[t] = __fdiv_rn(__fsub_rn(hc.y, yq), dz);
        recC[fc].w = hc.w | kUsedBit;
        link[cg] = (uint16_t)q;
        const uint32_t nh = ((st >> 8) & 0x7Fu) + 1u;
        sm.tstate[t] = (cg << 16) | (st & 0x8000u) | (nh << 8);
        atomicMin(&sm.min_active[(i - 1) & 1], t);
      } else {
        const uint32_t m = (st & 0xFFu) + 1u;
        if (m > (uint32_t)P.max_skipped) {
          sm.tstate[t] = st | 0xFFu;
        } else {
          sm.tstate[t] = (st & 0xFFFFFF00u) | m;
          atomicMin(&sm.min_active[(i - 1) & 1], t);
        }
      }
    }
    tsync<C>();  // B3

    // ---- T3/S1: every unused b lists the unused hits of layer A inside its phi window as (b, a) doublets
    const bool seeding = nA != 0 && nB != 0 && nC != 0;
#pragma unroll 1
    for (uint32_t k = nB + tid; k < nC; k += C::kThreads) sm.best[k] = kNoClaim;  // forward claims beyond layer B's size
#pragma unroll 1
    for (uint32_t kb = tid; kb < nB; kb += C::kThreads) {
      sm.best[kb] = kNoClaim;  // forward claims are done with; from here on: per-b argmin
      const uint32_t wb = recB[kb].w;
      if (!seeding || (wb & kUsedBit)) continue;
      const int w = P.w_seed_phi16, phb = phi_of(wb);
      uint32_t ia = lower_bound_phi(bucketA, recA, nA, wrap16(phb - w));
#pragma unroll 1
      for (uint32_t k = 0; k < nA; ++k, ++ia) {
        if (ia >= nA) ia -= nA;
        const uint32_t wa = recA[ia].w;
        const int d = wrap16(phi_of(wa) - phb);
        if (d > w || d < -w) break;
        if (wa & kUsedBit) continue;
        const uint32_t pos = atomicAdd(&sm.n_doublets, 1u);
        if (pos < (uint32_t)C::kCapDoublets) sm.doublets[pos] = kb | (ia << 16);
        else process_doublet(c, recA, recB, recC, bucketC, nC, kb, ia);  // list full: do it here (same result)
      }
    }
    tsync<C>();  // B4
    // ---- T3/S2: one thread per doublet
    {
      const uint32_t nd = min(sm.n_doublets, (uint32_t)C::kCapDoublets);
#pragma unroll 1
      for (uint32_t d = tid; d < nd; d += C::kThreads) {
        const uint32_t v = sm.doublets[d];
        process_doublet(c, recA, recB, recC, bucketC, nC, v & 0xFFFFu, v >> 16);
      }
    }
    tsync<C>();  // B5

    // ---- T4a: every b with a triplet claims its a and its c with (bits(S), b)
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

  if (sm.flags) {
    if (tid == 0) {
      if (C::kLast) { atomicOr(a.clusters.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW); a.counts[e] = 0; }
      else a.level[e] = (uint8_t)(C::kLevel + 1);
    }
    return;
  }

  // ---- T5 finalise + A8 fit: keep >= 4 hits, or 3 hits with S_seed <= s_weak; output in order of creation
  uint32_t out_tracks = 0, out_hits = 0;
  const uint32_t trk0 = co / 3;
  // the fit reads the compacted output (complete: the copier warp passed the barrier above, or an earlier kernel
  // filled it); __ldcg because these lines may have been written during this kernel
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
      double sz = 0, sx = 0, sy = 0;
      uint32_t h = st >> 16;
#pragma unroll 1
      for (int k = (int)n - 1; k >= 0; --k) {
        a.hits_slab[co + oh + k] = (uint16_t)h;
        sz += (double)__ldcg(Z + h); sx += (double)__ldcg(X + h); sy += (double)__ldcg(Y + h);
        if (k) h = link[h];
      }
      const double inv = 1.0 / (double)n;
      const double zm = sz * inv, xm = sx * inv, ym = sy * inv;
      double szz = 0, szx = 0, szy = 0;
      h = st >> 16;
#pragma unroll 1
      for (int k = (int)n - 1; k >= 0; --k) {
        const double dz = (double)__ldcg(Z + h) - zm;
        szz += dz * dz;
        szx += dz * ((double)__ldcg(X + h) - xm);
        szy += dz * ((double)__ldcg(Y + h) - ym);
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
#pragma unroll 1
  for (uint32_t t = threadIdx.x; t < nT; t += blockDim.x) {
    const float4 f = a.trk_fit[trk0 + t];
    a.out.x0[T0 + t] = f.x; a.out.y0[T0 + t] = f.y; a.out.tx[T0 + t] = f.z; a.out.ty[T0 + t] = f.w;
    a.out.hit_offsets[T0 + t] = H0 + a.trk_hitoff[trk0 + t];
  }
#pragma unroll 1
  for (uint32_t k = threadIdx.x; k < nH; k += blockDim.x) a.out.hits[H0 + k] = a.hits_slab[co + k];
  if (threadIdx.x == 0 && e + 1 == a.n_events) a.out.hit_offsets[T0 + nT] = H0 + nH;
}

template <class C>
cudaError_t launch_instance(const TrackLaunch& a, cudaStream_t stream) {
  cudaError_t err = cudaFuncSetAttribute(velo_track_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(Smem<C>));
  static_assert(sizeof(Smem<C>) <= 227 * 1024, "shared memory of one CTA");
  if (err != cudaSuccess) return err;
  velo_track_kernel<C><<<a.n_events, C::kBlock, sizeof(Smem<C>), stream>>>(a);
  return cudaGetLastError();
}

}  // namespace

// Three launches over all events: each CTA first decides whether its event belongs to this instance (see the header
// comment); events of other instances cost one small read and an exit.
cudaError_t launch_track(const TrackLaunch& a, cudaStream_t stream, uint32_t* n_launches) {
  *n_launches = 0;
  if (a.n_events == 0) return cudaSuccess;
  cudaError_t err = cudaMemsetAsync(a.level, 0, a.n_events, stream);
  if (err != cudaSuccess) return err;
  if ((err = launch_instance<CfgS>(a, stream)) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_instance<CfgM>(a, stream)) != cudaSuccess) return err;
  ++*n_launches;
  if ((err = launch_instance<CfgL>(a, stream)) != cudaSuccess) return err;
  ++*n_launches;
  return cudaSuccess;
}

cudaError_t launch_compact_tracks(const CompactTracksLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  compact_tracks_kernel<<<a.n_events, 128, 0, stream>>>(a);
  return cudaGetLastError();
}

}  // namespace velo
