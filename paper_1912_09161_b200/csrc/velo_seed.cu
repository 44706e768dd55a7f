// Search by triplet, part 1 of 2: everything of the seeding (A5) that does not depend on which hits are already used,
// for all layers of an event at once, and the cluster half of the output compaction (A9).  SURVEY.md §8(a); the
// algorithm is DESIGN.md reading R5 (T3) of P:181 ("forming seeds of three hits from consecutive layers ('triplets')")
// with the phi windows of P:183 ("sort hits on every layer by phi for fast look-up").
//
// Why two kernels.  R5 is sequential over the layers only through the `used` flags and the list of active tracks.  The
// expensive part of an iteration — every middle hit b of layer B against the hits a of layer A and c of layer C inside
// its phi windows, slopes and slope cut of a -> b, scatter S(a, b, c) <= s_seed — reads hit coordinates and nothing
// else.  This kernel therefore evaluates it for ALL (a, b, c) of ALL layer triples of an event in one go, whatever
// will be used later, and writes the few combinations that pass (about 800 of 24 000 per nu = 6 event) to a list per
// (event, layer B).  The second kernel (velo_follow.cu) walks the layers in order, one warp per event, and takes the
// argmin of R5 T3 over the entries of the list whose three hits are still unused: the minimum over the unused
// candidates of a set equals the minimum of R5 as long as the set holds every candidate that passes the cuts, which it
// does.  The price is about 3x more candidate evaluations than with the used flags applied first; what it buys is
// 260 000 independent (event, layer) work units per batch instead of 24 dependent rounds of block barriers per event
// (round 1: 154 k warp instructions per event at 16 of 32 lanes, barrier stalls on top; profiles/README.md).
//
// Mapping (sm_100a): ONE WARP per (event, middle layer B), like the cluster kernel; the warps of a CTA take the
// consecutive layers of an event, share nothing and never meet at a barrier.  Nothing is staged: the hit records
// {x, y, z, phi16} (16 bytes, as the cluster kernel left them) are read with ld.global.nc.v4 and live in the L1 — a warp
// walks its layer in phi order, so its windows on the neighbouring layers slide over a few lines that the warps of the
// same CTA touch as well; the kernel's own shared memory is 3 kB per warp, which leaves the L1 nearly whole.  The phi
// look-up tables (first hit of every 256-unit slice of phi16) are the prefix sums of the cluster kernel's counting sort.
// Per chunk of 32 consecutive hits of the layer:
//   0. the hits go to their final place in the compacted cluster output (A9; every hit is in exactly one chunk);
//   1. lane = middle hit: its phi windows on A and C as index ranges; the forwarding windows of the hit (layers B-1 and
//      B-2, w_fwd) go to global memory for the second kernel, which then never searches a layer;
//   2. the (b, a) doublets of the 32 windows laid end to end, one lane per doublet: slopes (the normative divisions),
//      slope cut; survivors are compacted (ballot) into a ring of 64 doublets that lives across the chunks;
//   3. whenever the ring holds 32 doublets: one lane per doublet walks b's window on C (neighbouring lanes have
//      neighbouring b, hence windows of similar length) and evaluates the normative scatter; a pass appends
//      bits(S) << 32 | a << 20 | b << 10 | c (layer-local indices) to the list of the layer, which this warp owns.
// A list that outgrows its region (one entry per hit of the layer) flags the event for the CTA-per-event kernel of
// velo_track.cu.
#include "velo_track.cuh"

namespace velo {
namespace {

constexpr int kSeedWarps = 4;   // warps per CTA (independent work units)
constexpr uint32_t kRing = 64;  // doublets a warp holds between stages 2 and 3

struct __align__(16) SeedWarp {
  uint4 ring[kRing][2];  // {tx, ty, x_b, y_b}, {z_b, b | a << 16 (layer-local), c_first | c_n << 16, -}
  uint4 bslot[32][2];    // stage 2: the middle hits of the chunk that have doublets: record, {b, a_first, c window, first doublet}
  uint32_t n_trip;       // entries appended to the list of the unit's layer
  uint32_t pad[3];
};

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, uint32_t lane) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(kFull, v, d);
    if (lane >= (uint32_t)d) v += t;
  }
  return v;
}
__device__ __forceinline__ uint32_t lanemask_le() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
  return m;
}

// One layer as the search reads it: slab records, its phi table, number of hits.
struct LayerView {
  const uint4* __restrict__ rec;
  const uint16_t* __restrict__ tab;
  uint32_t n;
};
__device__ __forceinline__ int phi_at(const LayerView& v, uint32_t idx) {
  return phi_of(__ldg(reinterpret_cast<const uint32_t*>(v.rec + idx) + 3));
}

// First index in [0, n) of the layer (sorted by signed phi16) with phi >= target, or n.  From the slice's first hit
// onwards, four hits at a time: the loads of a group are in flight together, and one group is nearly always enough.
__device__ __forceinline__ uint32_t lower_bound_phi(const LayerView& v, int target) {
  uint32_t idx = __ldg(v.tab + ((uint32_t)(target + 32768) >> 8));
#pragma unroll 1
  for (;;) {
    uint32_t below = 0;
#pragma unroll
    for (uint32_t u = 0; u < 4; ++u) below += (idx + u < v.n && phi_at(v, idx + u) < target) ? 1u : 0u;
    idx += below;
    if (below < 4) break;
  }
  return idx;
}

// The hits of a layer with |dphi16(hit, ph)| <= w as a circular index range: `first`, then `count` hits (indices modulo
// n).  w <= 16383 (checked at create), so the window is shorter than the circle and wraps at most once.
__device__ __forceinline__ void phi_window(const LayerView& v, int ph, int w, uint32_t& first, uint32_t& count) {
  const int tl = ph - w, th = ph + w;
  const bool wrapped = tl < -32768 || th > 32767;
  const uint32_t lo = lower_bound_phi(v, wrap16(tl));
  const int thw = wrap16(th);
  const uint32_t hi = thw == 32767 ? v.n : lower_bound_phi(v, thw + 1);
  first = lo;
  count = wrapped ? v.n - lo + hi : hi - lo;
}

// A superset of that window from the table alone (whole slices): for the forwarding window two layers down, which few
// tracks ever use; velo_follow.cu tests |dphi| of every candidate itself.
__device__ __forceinline__ void phi_window_slices(const LayerView& v, int ph, int w, uint32_t& first, uint32_t& count) {
  const int tl = ph - w, th = ph + w;
  const bool wrapped = tl < -32768 || th > 32767;
  const uint32_t lo = __ldg(v.tab + ((uint32_t)(wrap16(tl) + 32768) >> 8));
  const uint32_t hi = __ldg(v.tab + ((uint32_t)(wrap16(th) + 32768) >> 8) + 1);
  first = lo;
  count = wrapped ? v.n - lo + hi : hi - lo;
}

struct SeedCtx {
  const TrackLaunch& a;
  SeedWarp& ws;
  LayerView C;                 // the layer below the unit's
  unsigned long long* trip;    // list of the unit's layer
  uint32_t nB, lane;
  uint32_t ring_head, ring_n;  // warp-uniform
};

// Stage 3 for the 32 oldest doublets of the ring (or the `n_valid` < 32 left at the end): one lane per doublet.  A lane
// keeps its first passing candidate in registers and the lanes of the round append theirs together (positions by
// ballot); further passes of the same doublet are rare and go out one by one.
__device__ __forceinline__ void score_doublets(SeedCtx& c, uint32_t n_valid) {
  const float s_seed = c.a.geo.params.s_seed;
  const uint32_t nC = c.C.n;
  bool have = false;
  uint32_t first_lo = 0, first_s = 0;
  if (c.lane < n_valid) {
    const uint32_t slot = (c.ring_head + c.lane) & (kRing - 1);
    const uint4 d0 = c.ws.ring[slot][0], d1 = c.ws.ring[slot][1];
    const float tx = __uint_as_float(d0.x), ty = __uint_as_float(d0.y), xb = __uint_as_float(d0.z), yb = __uint_as_float(d0.w);
    const float zb = __uint_as_float(d1.x);
    const uint32_t ab = ((d1.y >> 16) << 20) | ((d1.y & 0xFFFFu) << 10);
    uint32_t ic = d1.z & 0xFFFFu;
    const uint32_t c_n = d1.z >> 16;
#pragma unroll 1
    for (uint32_t j = 0; j < c_n; ++j, ++ic) {
      if (ic >= nC) ic -= nC;
      VELO_CHECK(c.a.geo, ic < nC, 201);
      const uint4 r = __ldg(c.C.rec + ic);
      const float dz = __fsub_rn(__uint_as_float(r.z), zb);
      const float ex = __fsub_rn(__fmaf_rn(tx, dz, xb), __uint_as_float(r.x));
      const float ey = __fsub_rn(__fmaf_rn(ty, dz, yb), __uint_as_float(r.y));
      const float S = __fmaf_rn(ex, ex, __fmul_rn(ey, ey));
      if (S <= s_seed) {
        if (!have) {
          have = true; first_s = __float_as_uint(S); first_lo = ab | ic;
        } else {
          const uint32_t pos = atomicAdd(&c.ws.n_trip, 1u);
          if (pos < c.nB) c.trip[pos] = ((unsigned long long)__float_as_uint(S) << 32) | ab | ic;
        }
      }
    }
  }
  __syncwarp();
  const uint32_t bal = __ballot_sync(kFull, have);
  if (bal) {
    uint32_t base = 0;
    if (c.lane == 0) base = atomicAdd(&c.ws.n_trip, (uint32_t)__popc(bal));
    base = __shfl_sync(kFull, base, 0);
    if (have) {
      const uint32_t pos = base + __popc(bal & lanemask_lt());
      if (pos < c.nB) c.trip[pos] = ((unsigned long long)first_s << 32) | first_lo;
    }
  }
  const uint32_t taken = n_valid < 32u ? n_valid : 32u;
  c.ring_head = (c.ring_head + taken) & (kRing - 1);
  c.ring_n -= taken;
}

// Everything for the hits of layer l of event e, by one warp.
__device__ __forceinline__ void seed_unit(const TrackLaunch& a, SeedWarp& ws, uint32_t e, uint32_t l) {
  const allen_velo_params_t& P = a.geo.params;
  const uint32_t L = a.geo.n_layers, lane = lane_id();
  const uint8_t cls = a.level[e];
  if (cls == kClsSkip) return;
  const uint32_t co = a.clusters.event_offsets[e];
  const uint32_t item = e * L + l;
  // layer offsets l-2 .. l+2 of the event (lanes 0..4), clamped to the event
  uint32_t lo_v = 0;
  if (lane < 5) {
    const int ll = (int)l - 2 + (int)lane;
    const uint32_t idx = ll < 0 ? 0u : ll > (int)L ? L : (uint32_t)ll;
    lo_v = a.clusters.layer_offsets[e * L + idx] - co;
  }
  const uint32_t D0 = __shfl_sync(kFull, lo_v, 0), C0 = __shfl_sync(kFull, lo_v, 1), B0 = __shfl_sync(kFull, lo_v, 2),
                 A0 = __shfl_sync(kFull, lo_v, 3), A1 = __shfl_sync(kFull, lo_v, 4);
  const uint32_t nB = A0 - B0;
  if (nB == 0) {
    if (lane == 0) a.trip_count[item] = 0;
    return;
  }
  const uint32_t srcB = a.slab_base[item];
  const uint4* __restrict__ recB = a.slab.rec + srcB;
  const uint4* __restrict__ infoB = a.slab.info + srcB;
  const bool search = cls <= kClsLarge;
  const bool middle = search && l >= 1 && l + 1 < L;
  LayerView A{nullptr, nullptr, 0}, Cv{nullptr, nullptr, 0}, D{nullptr, nullptr, 0};
  if (search && l >= 1) {
    Cv.rec = a.slab.rec + a.slab_base[item - 1];
    Cv.tab = a.slab.phi_tab + (size_t)(item - 1) * kPhiTabStride;
    Cv.n = B0 - C0;
  }
  if (search && l >= 2) {
    D.rec = a.slab.rec + a.slab_base[item - 2];
    D.tab = a.slab.phi_tab + (size_t)(item - 2) * kPhiTabStride;
    D.n = C0 - D0;
  }
  if (middle) {
    A.rec = a.slab.rec + a.slab_base[item + 1];
    A.tab = a.slab.phi_tab + (size_t)(item + 1) * kPhiTabStride;
    A.n = A1 - A0;
  }
  if (lane == 0) ws.n_trip = 0;
  // Ask for everything the unit will read before the first dependent load needs it: its own records, the records and
  // phi tables of the neighbouring layers (the cluster kernel's output is long gone from the L2 for a batch this size).
  {
    auto prefetch = [&](const void* ptr, uint32_t bytes) {
      const char* q = reinterpret_cast<const char*>(ptr);
#pragma unroll 1
      for (uint32_t o = lane * 128u; o < bytes; o += 32u * 128u) asm volatile("prefetch.global.L1 [%0];" ::"l"(q + o));
    };
    prefetch(recB, 16u * nB);
    prefetch(infoB, 16u * nB);
    if (Cv.n) { prefetch(Cv.rec, 16u * Cv.n); prefetch(Cv.tab, 2u * (kPhiSlices + 1)); }
    if (A.n) { prefetch(A.rec, 16u * A.n); prefetch(A.tab, 2u * (kPhiSlices + 1)); }
    if (D.n) prefetch(D.tab, 2u * (kPhiSlices + 1));
  }
  __syncwarp();
  SeedCtx c{a, ws, Cv, a.trip + co + B0, nB, lane, 0u, 0u};
  const uint32_t dst = co + B0;

#pragma unroll 1
  for (uint32_t k0 = 0; k0 < nB; k0 += 32) {
    const uint32_t kb = k0 + lane;
    // ---- stage 0: the chunk's hits to the compacted output; stage 1: windows of the middle hit
    uint32_t nd = 0, a_first = 0, c_first = 0, c_n = 0;
    uint4 r = make_uint4(0, 0, 0, 0);
    if (kb < nB) {
      r = __ldg(recB + kb);
      const uint4 q = __ldg(infoB + kb);
      const uint32_t d = dst + kb;
      a.clusters.key[d] = q.x; a.clusters.n_pixels[d] = q.y; a.clusters.sum_col[d] = q.z; a.clusters.sum_row[d] = q.w;
      a.clusters.x[d] = __uint_as_float(r.x); a.clusters.y[d] = __uint_as_float(r.y); a.clusters.z[d] = __uint_as_float(r.z);
      a.clusters.phi16[d] = (int16_t)(uint16_t)r.w;
      if (a.clusters.checksum) a.clusters.checksum[d] = __ldg(a.slab.checksum + srcB + kb);
      if (search && l >= 1) {
        const int phb = phi_of(r.w);
        phi_window(Cv, phb, P.w_seed_phi16, c_first, c_n);
        uint32_t f1 = c_first, n1 = c_n, f2 = 0, n2 = 0;
        if (P.w_fwd_phi16 != P.w_seed_phi16) phi_window(Cv, phb, P.w_fwd_phi16, f1, n1);
        if (l >= 2) phi_window_slices(D, phb, P.w_fwd_phi16, f2, n2);
        if (f1 >= Cv.n) f1 = 0;  // (a wrapped window may start "behind the last hit" = at hit 0)
        if (f2 >= D.n) f2 = 0;
        a.fwd_win[dst + kb] = make_uint2(f1 | (n1 << 16), f2 | (n2 << 16));
        if (middle && c_n) phi_window(A, phb, P.w_seed_phi16, a_first, nd);
      }
    }
    if (!middle) continue;

    // ---- stage 2: the (b, a) doublets of the chunk laid end to end, one lane per doublet
    const uint32_t incl = warp_incl_scan(nd, lane);
    const uint32_t total = __shfl_sync(kFull, incl, 31);
    if (total == 0) continue;
    const uint32_t p = incl - nd;  // position of this lane's first doublet
    {
      const uint32_t nonempty = __ballot_sync(kFull, nd != 0);
      if (nd) {
        const uint32_t s = __popc(nonempty & lanemask_lt());
        VELO_CHECK(a.geo, s < 32 && a_first <= A.n && c_first <= Cv.n && nd <= A.n && c_n <= Cv.n && kb < 1024, 202);
        ws.bslot[s][0] = r;
        ws.bslot[s][1] = make_uint4(kb, a_first, c_first | (c_n << 16), p);
      }
    }
    __syncwarp();
    uint32_t before = 0;  // middle hits whose doublets start before the current group of 32
#pragma unroll 1
    for (uint32_t j0 = 0; j0 < total; j0 += 32) {
      const uint32_t rel = p - j0;  // < 32 iff this lane's window starts inside the group
      const uint32_t starts = __reduce_or_sync(kFull, (nd != 0 && rel < 32u) ? (1u << rel) : 0u);
      const uint32_t owner = before + __popc(starts & lanemask_le()) - 1u;
      before += __popc(starts);
      const uint32_t j = j0 + lane;
      bool pass = false;
      uint4 o0 = make_uint4(0, 0, 0, 0), o1 = o0;
      if (j < total) {
        const uint4 hb = ws.bslot[owner][0], bs = ws.bslot[owner][1];
        uint32_t ia = bs.y + (j - bs.w);
        if (ia >= A.n) ia -= A.n;
        VELO_CHECK(a.geo, owner < 32 && ia < A.n && j - bs.w < A.n, 203);
        const uint4 ha = __ldg(A.rec + ia);
        const float dz_ab = __fsub_rn(__uint_as_float(hb.z), __uint_as_float(ha.z));
        const float tx = __fdiv_rn(__fsub_rn(__uint_as_float(hb.x), __uint_as_float(ha.x)), dz_ab);
        const float ty = __fdiv_rn(__fsub_rn(__uint_as_float(hb.y), __uint_as_float(ha.y)), dz_ab);
        pass = fabsf(tx) <= P.max_slope && fabsf(ty) <= P.max_slope;
        o0 = make_uint4(__float_as_uint(tx), __float_as_uint(ty), hb.x, hb.y);
        o1 = make_uint4(hb.z, bs.x | (ia << 16), bs.z, 0u);
      }
      const uint32_t bal = __ballot_sync(kFull, pass);
      if (pass) {
        const uint32_t slot = (c.ring_head + c.ring_n + __popc(bal & lanemask_lt())) & (kRing - 1);
        ws.ring[slot][0] = o0;
        ws.ring[slot][1] = o1;
      }
      c.ring_n += __popc(bal);
      VELO_CHECK(a.geo, c.ring_n <= kRing, 204);
      __syncwarp();
      if (c.ring_n >= 32) score_doublets(c, 32);
    }
    __syncwarp();  // bslot is free for the next chunk
  }
  if (c.ring_n) score_doublets(c, c.ring_n);
  __syncwarp();
  if (lane == 0) {
    const uint32_t n_trip = ws.n_trip;
    a.trip_count[item] = min(n_trip, nB);
    if (n_trip > nB) atomicOr(a.ev_flags + e, kEvRedo);  // the list outgrew its region
  }
}

// One warp per (event, layer); the warps of a CTA take consecutive layers of one event (their windows overlap in the L1).
__global__ void __launch_bounds__(kSeedWarps * 32, 10) velo_seed_kernel(const __grid_constant__ TrackLaunch a) {
  __shared__ SeedWarp ws[kSeedWarps];
  const uint32_t unit = blockIdx.x * kSeedWarps + (threadIdx.x >> 5);
  const uint32_t L = a.geo.n_layers;
  if (unit >= a.n_events * L) return;
  seed_unit(a, ws[threadIdx.x >> 5], unit / L, unit % L);
}

}  // namespace

cudaError_t seed_prepare() { return cudaSuccess; }

cudaError_t launch_seed(const TrackLaunch& a, cudaStream_t stream) {
  const uint32_t units = a.n_events * a.geo.n_layers;
  if (units == 0) return cudaSuccess;
  velo_seed_kernel<<<(units + kSeedWarps - 1) / kSeedWarps, kSeedWarps * 32, 0, stream>>>(a);
  return cudaGetLastError();
}

}  // namespace velo
