// Primary-vertex finding (beyond the headline path; "we search for PVs in a histogram of the
// point of closest approach of tracks to the beamline, where a cluster indicates a PV candidate ... every track is
// assigned to every vertex based on a weight, so that all candidates can be fitted in parallel"; R10).
//
// One CTA of four warps per event; the warps share the histogram and take the candidates in turn.  Seeding is integer work on fp32 values that are bit-identical to the oracle's (normative
// operations on the straight-line fit), so the candidates are exactly the oracle's; the weighted fits (all tracks to
// every candidate, 8 passes of Tukey-weighted least squares on the Kalman states) run in fp32, lanes over tracks,
// sums by warp shuffles.
#include "velo_common.cuh"

namespace velo {
namespace {

constexpr int kPvWarps = 4;
constexpr int kPvBins = 600;
constexpr int kPvCand = 96;   // candidates staged per event
constexpr int kPvMax = 32;    // vertices written per event
constexpr float kChi2Max = 12.0f;

struct PvSmem {
  uint32_t h[kPvBins + 4];  // h[b + 2] = bin b, two guard bins on either side
  float seed[kPvCand];
  float vx[kPvCand], vy[kPvCand], vz[kPvCand], sw[kPvCand], chi2[kPvCand];
  uint32_t nw[kPvCand];     // tracks with w > 0; 0xFFFFFFFF: fit failed
  uint32_t n_cand, b_lo, b_hi;
};

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
  return v;
}

__global__ void __launch_bounds__(kPvWarps * 32) velo_pv_kernel(const __grid_constant__ PvLaunch a) {
  __shared__ PvSmem sm;
  const uint32_t lane = lane_id(), warp = threadIdx.x >> 5, tid = threadIdx.x;
  const uint32_t e = blockIdx.x;
  const uint32_t t0 = a.tracks.event_offsets[e], n = a.tracks.event_offsets[e + 1] - t0;
  const bool fits = (unsigned long long)t0 + n <= a.tracks.capacity_tracks;  // else the tracks were not written
  float* out = a.out.vertices + (size_t)e * a.out.max_per_event * 8;

  // ---- 1, 2: histogram of the z of closest approach to the beam line (normative fp32 operations)
#pragma unroll 1
  for (uint32_t b = tid; b < kPvBins + 4; b += kPvWarps * 32) sm.h[b] = 0;
  if (tid == 0) { sm.n_cand = 0; sm.b_lo = kPvBins; sm.b_hi = 0; }
  __syncthreads();
  uint32_t b_lo = kPvBins, b_hi = 0;  // occupied bin range: candidates can only be within one bin of it
#pragma unroll 1
  for (uint32_t i = tid; i < n && fits; i += kPvWarps * 32) {
    const float x0 = a.tracks.x0[t0 + i], y0 = a.tracks.y0[t0 + i], tx = a.tracks.tx[t0 + i], ty = a.tracks.ty[t0 + i];
    const float t2 = __fmaf_rn(tx, tx, __fmul_rn(ty, ty));
    if (!(t2 >= 1e-8f)) continue;
    const float zp = __fdiv_rn(-__fmaf_rn(x0, tx, __fmul_rn(y0, ty)), t2);
    const float u = __fadd_rn(zp, 300.0f);
    if (!(u >= 0.0f) || !(u < (float)kPvBins)) continue;
    const int bin = (int)floorf(u);
    atomicAdd(&sm.h[bin + 2], 1u);
    b_lo = min(b_lo, (uint32_t)bin);
    b_hi = max(b_hi, (uint32_t)bin);
  }
  b_lo = __reduce_min_sync(kFull, b_lo);
  b_hi = __reduce_max_sync(kFull, b_hi);
  if (lane == 0 && b_lo <= b_hi) { atomicMin(&sm.b_lo, b_lo); atomicMax(&sm.b_hi, b_hi); }
  __syncthreads();
  b_lo = sm.b_lo;
  b_hi = sm.b_hi;
  // ---- candidates: local maxima of (s, h), s = three-bin sum >= 4; ascending bin order by ballot
  const uint32_t scan_lo = b_lo > 0 ? b_lo - 1 : 0, scan_hi = min(b_hi + 2, (uint32_t)kPvBins);
#pragma unroll 1
  for (uint32_t b0 = scan_lo; b0 < scan_hi && b_lo <= b_hi && warp == 0; b0 += 32) {  // warp 0 lists the candidates
    const uint32_t b = b0 + lane;
    bool cand = false;
    float seed = 0.0f;
    if (b < scan_hi) {
      const int hmm = sm.h[b], hm = sm.h[b + 1], hc = sm.h[b + 2], hp = sm.h[b + 3], hpp = sm.h[b + 4];
      const int s = hm + hc + hp, sl = hmm + hm + hc, sr = hc + hp + hpp;
      const bool above_left = s > sl || (s == sl && hc > hm), not_below_right = s > sr || (s == sr && hc >= hp);
      cand = s >= 4 && above_left && not_below_right;
      if (cand) seed = -300.0f + (float)b + 0.5f + (float)(hp - hm) / (float)s;
    }
    const uint32_t ballot = __ballot_sync(kFull, cand);
    const uint32_t base = sm.n_cand;
    if (cand) {
      const uint32_t pos = base + __popc(ballot & lanemask_lt());
      if (pos < kPvCand) sm.seed[pos] = seed;
    }
    __syncwarp();
    if (lane == 0) sm.n_cand = base + __popc(ballot);
    __syncwarp();
  }
  __syncthreads();
  const uint32_t n_cand = min(sm.n_cand, (uint32_t)kPvCand);
  if (sm.n_cand > (uint32_t)kPvCand && tid == 0) atomicOr(a.status + e, ALLEN_VELO_STATUS_STAGE_OVERFLOW);

  // ---- 3: every candidate is fitted with all tracks (lanes over tracks)
  const float* K = a.tracks.kalman + 12 * (size_t)t0;
#pragma unroll 1
  for (uint32_t c = warp; c < n_cand; c += kPvWarps) {  // the warps take the candidates in turn
    float vx = 0.0f, vy = 0.0f, vz = sm.seed[c], sw = 0.0f, chi2 = 0.0f;
    uint32_t nw = 0;
    bool ok = true;
#pragma unroll 1
    for (int it = 0; it < 8 && ok; ++it) {
      float a00 = 0, a11 = 0, a02 = 0, a12 = 0, a22 = 0, b0 = 0, b1 = 0, b2 = 0, s_w = 0, s_c = 0;
      uint32_t cnt = 0;
#pragma unroll 1
      for (uint32_t i = lane; i < n; i += 32) {
        const float4 k0 = __ldg(reinterpret_cast<const float4*>(K + 12 * (size_t)i));      // x, y, tx, ty
        const float4 k1 = __ldg(reinterpret_cast<const float4*>(K + 12 * (size_t)i) + 1);  // z, chi2, C00x, C01x
        const float4 k2 = __ldg(reinterpret_cast<const float4*>(K + 12 * (size_t)i) + 2);  // C11x, C00y, C01y, C11y
        const float d = vz - k1.x;
        const float dx = k0.x + k0.z * d - vx, dy = k0.y + k0.w * d - vy;
        const float var_x = k1.z + 2.0f * d * k1.w + d * d * k2.x, var_y = k2.y + 2.0f * d * k2.z + d * d * k2.w;
        // most tracks belong to other vertices: reject them before the two divisions (same cut, cross-multiplied)
        if (!(dx * dx * var_y + dy * dy * var_x < kChi2Max * var_x * var_y)) continue;
        const float ix = 1.0f / var_x, iy = 1.0f / var_y;
        const float c2 = dx * dx * ix + dy * dy * iy;
        if (!(c2 < kChi2Max)) continue;
        const float q = 1.0f - c2 * (1.0f / kChi2Max), w = q * q;
        const float wx = w * ix, wy = w * iy;
        a00 += wx; a11 += wy; a02 -= wx * k0.z; a12 -= wy * k0.w; a22 += wx * k0.z * k0.z + wy * k0.w * k0.w;
        b0 += wx * dx; b1 += wy * dy; b2 -= wx * k0.z * dx + wy * k0.w * dy;
        s_w += w; s_c += w * c2; cnt += 1;
      }
      a00 = warp_sum(a00); a11 = warp_sum(a11); a02 = warp_sum(a02); a12 = warp_sum(a12); a22 = warp_sum(a22);
      b0 = warp_sum(b0); b1 = warp_sum(b1); b2 = warp_sum(b2);
      sw = warp_sum(s_w); chi2 = warp_sum(s_c); nw = __reduce_add_sync(kFull, cnt);
      if (it == 7) break;
      if (!(a00 > 0.0f) || !(a11 > 0.0f)) { ok = false; break; }
      const float den = a22 - a02 * a02 / a00 - a12 * a12 / a11;
      if (!(den > 0.0f)) { ok = false; break; }
      const float dz = (b2 - a02 * b0 / a00 - a12 * b1 / a11) / den;
      vx += (b0 - a02 * dz) / a00;
      vy += (b1 - a12 * dz) / a11;
      vz += dz;
    }
    if (lane == 0) {
      sm.vx[c] = vx; sm.vy[c] = vy; sm.vz[c] = vz; sm.sw[c] = sw; sm.chi2[c] = chi2;
      sm.nw[c] = (ok && sw >= 3.0f) ? nw : 0xFFFFFFFFu;
    }
  }
  __syncthreads();
  if (warp != 0) return;
  // ---- 4: drop duplicates (another accepted vertex within 1 mm in z with a sum w more than 0.1 % larger; within
  //         0.1 %, i.e. two candidates that converged to the same vertex: the earlier wins),
  //         write in candidate order
  uint32_t n_out = 0;
#pragma unroll 1
  for (uint32_t c0 = 0; c0 < n_cand; c0 += 32) {
    const uint32_t c = c0 + lane;
    bool keep = c < n_cand && sm.nw[c] != 0xFFFFFFFFu;
    if (keep) {
#pragma unroll 1
      for (uint32_t j = 0; j < n_cand && keep; ++j)
        if (j != c && sm.nw[j] != 0xFFFFFFFFu && fabsf(sm.vz[j] - sm.vz[c]) < 1.0f) {
          const bool j_larger = sm.sw[j] > sm.sw[c] * 1.001f, c_larger = sm.sw[c] > sm.sw[j] * 1.001f;
          if (j_larger || (!c_larger && j < c)) keep = false;
        }
    }
    const uint32_t ballot = __ballot_sync(kFull, keep);
    const uint32_t pos = n_out + __popc(ballot & lanemask_lt());
    if (keep && pos < min((uint32_t)kPvMax, a.out.max_per_event)) {
      float* o = out + 8 * (size_t)pos;
      o[0] = sm.vx[c]; o[1] = sm.vy[c]; o[2] = sm.vz[c]; o[3] = sm.sw[c];
      o[4] = (float)sm.nw[c]; o[5] = sm.chi2[c]; o[6] = sm.seed[c]; o[7] = 0.0f;
    }
    n_out += __popc(ballot);
  }
  if (lane == 0) a.out.n_vertices[e] = min(n_out, min((uint32_t)kPvMax, a.out.max_per_event));
}

}  // namespace

cudaError_t launch_pv(const PvLaunch& a, cudaStream_t stream) {
  if (a.n_events == 0) return cudaSuccess;
  velo_pv_kernel<<<a.n_events, kPvWarps * 32, 0, stream>>>(a);
  return cudaGetLastError();
}

}  // namespace velo
