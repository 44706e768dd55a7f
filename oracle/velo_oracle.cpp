// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded-per-event CPU implementation of the VELO pixel hot path of Allen's HLT1
// (arXiv:1912.09161), written from the paper's statements and the readings listed in DESIGN.md.  It is the
// parity reference for the CUDA path and the timed CPU baseline of bench.py.  It shares NO code, header,
// table or helper with paper_1912_09161_b200/csrc: only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load it.
//
// Citations: "P:n" = /root/reference/PAPER.md line n; "D:Rk" = reading k in DESIGN.md §3 (points on which the
// paper is silent).  Pins for every function below are in tests/test_oracle_*.py (DESIGN.md §4 lists them).
//   O1 decode            P:153 "Decoding the raw input into coordinates"; raw format v1 D:R1
//   O2 clustering        P:179 "connected component labeling" -> exact 8-connected components (D:R2), flood fill
//   O3 centroid/global   P:153 "coordinates in the LHCb global coordinate system"; phi P:183 (D:R3)
//   O4 phi sort          P:183 "sort hits on every layer by phi" (D:R4)
//   O5 search by triplet P:181-183 "seeds of three hits from consecutive layers ... extending these to the other
//                        layers" (D:R5 step-by-step reading T1..T5)
//   O6 straight-line fit P:149 "tracks in the Velo detector form straight lines" -> unweighted LSQ (D:R6)
//   O7 simple Kalman fit P:185 "simple Kalman filter ... x- and y-components are independent ... constant average
//                        transverse momentum of 400 MeV ... noise contribution from multiple scattering" (D:R9)
//   O8 PV finding        P:187 "histogram of the point of closest approach of tracks to the beamline, where a cluster
//                        indicates a PV candidate ... every track is assigned to every vertex based on a weight, so
//                        that all candidates can be fitted in parallel" (D:R10)
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off (no fast-math) -shared -fPIC -pthread.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

// ------------------------------------------------------------------------------------------------
// Inputs
// ------------------------------------------------------------------------------------------------
struct Params {  // D:R5 cut values
  int32_t w_seed_phi16, w_fwd_phi16;
  float max_slope;
  float s_seed, s_fwd, s_weak;
  int32_t max_skipped;
};

struct Geometry {
  uint32_t n_sensors, n_modules, n_layers, n_cols, n_rows;
  float pitch_mm;
  const uint16_t* sensor_module;
  const uint16_t* module_layer;
  const float* sensor_ltg;  // [n_sensors][9]
  Params params;
};

enum : uint32_t {
  STATUS_BAD_HEADER = 1u << 0,
  STATUS_BAD_SP = 1u << 1,
  STATUS_TOO_MANY_CLUSTERS = 1u << 2,
};

// ------------------------------------------------------------------------------------------------
// O2-local (D:R11): region size in super-pixels, 0 = off.  Set by oracle_set_cluster_regions before a run.
static uint32_t region_sp_cols = 0, region_sp_rows = 0;

// O2 helper: membership checksum (D:R2) — sum over the cluster's pixels of mix32(row*n_cols+col), mod 2^32.
// ------------------------------------------------------------------------------------------------
uint32_t mix32(uint32_t v) {
  uint32_t m = (v + 1u) * 2654435761u;
  m ^= m >> 15;
  m *= 2246822519u;
  m ^= m >> 13;
  return m;
}

// ------------------------------------------------------------------------------------------------
// O3: phi as a 16-bit angle.  D:R3 fixes the expression tree: every operation one IEEE-754 binary32
// round-to-nearest operation, fma = fused.  Polynomial: Abramowitz & Stegun 4.4.49,
// arctan(t) = t * sum_{k=0..8} a_{2k} t^{2k}, 0 <= t <= 1.
// ------------------------------------------------------------------------------------------------
float atan2_poly(float x, float y) {
  const float a0 = 1.0f, a1 = -0.3333314528f, a2 = 0.1999355085f, a3 = -0.1420889944f, a4 = 0.1065626393f,
              a5 = -0.0752896400f, a6 = 0.0429096138f, a7 = -0.0161657367f, a8 = 0.0028662257f;
  float ax = std::fabs(x), ay = std::fabs(y);
  float mx = ax > ay ? ax : ay, mn = ax > ay ? ay : ax;
  float t = mx == 0.0f ? 0.0f : mn / mx;
  float s = t * t;
  float poly = a8;
  poly = std::fmaf(poly, s, a7);
  poly = std::fmaf(poly, s, a6);
  poly = std::fmaf(poly, s, a5);
  poly = std::fmaf(poly, s, a4);
  poly = std::fmaf(poly, s, a3);
  poly = std::fmaf(poly, s, a2);
  poly = std::fmaf(poly, s, a1);
  poly = std::fmaf(poly, s, a0);
  float p = poly * t;
  if (ay > ax) p = 1.5707964f - p;
  if (x < 0.0f) p = 3.1415927f - p;
  if (y < 0.0f) p = -p;
  return p;
}

int16_t phi16_of(float x, float y) {
  float p = atan2_poly(x, y);
  float scaled = p * 10430.378f;            // 32768/pi
  int32_t r = (int32_t)std::nearbyintf(scaled);  // round-half-even (default rounding mode)
  return (int16_t)(uint16_t)(r & 0xFFFF);   // +32768 wraps to -32768
}

inline int dphi(int16_t a, int16_t b) { return (int16_t)(uint16_t)((uint16_t)a - (uint16_t)b); }

// ------------------------------------------------------------------------------------------------
// O5 helper: scatter of candidate c after hits a (older) then b (newer), D:R5.
// ------------------------------------------------------------------------------------------------
struct Hit {
  float x, y, z;
  int16_t phi;
};

float scatter(const Hit& a, const Hit& b, const Hit& c) {
  float dz_ab = b.z - a.z;
  float tx = (b.x - a.x) / dz_ab;
  float ty = (b.y - a.y) / dz_ab;
  float dz = c.z - b.z;
  float ex = std::fmaf(tx, dz, b.x) - c.x;
  float ey = std::fmaf(ty, dz, b.y) - c.y;
  return std::fmaf(ex, ex, ey * ey);
}

inline uint32_t fbits(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  return u;
}

// ------------------------------------------------------------------------------------------------
// Per-event result
// ------------------------------------------------------------------------------------------------
struct Cluster {
  uint32_t key, n, sum_col, sum_row, checksum;
  float x, y, z;
  int16_t phi;
  uint32_t layer;
};

struct Track {
  std::vector<uint32_t> hits;  // event-local cluster indices in the normative order, in order of addition
  uint32_t seed_key;           // normative index of the seed's middle hit
  float s_seed;
  int missed;
  bool active;
  float x0, y0, tx, ty;
};

struct EventResult {
  uint32_t status = 0;
  std::vector<Cluster> clusters;             // normative order (layer, phi16, key)
  std::vector<uint32_t> layer_offsets;       // [n_layers+1]
  std::vector<uint32_t> pix_key;             // (sensor<<18)|(row*n_cols+col) for every decoded pixel
  std::vector<uint32_t> pix_cluster;         // its cluster (normative index)
  std::vector<Track> tracks;                 // accepted tracks, in order of creation
  uint32_t near_cut = 0;                     // number of decisions within 1e-4 of a cut (D:R7)
  std::vector<uint32_t> near_cut_hits;       // hits touched by such decisions
};

struct Scratch {
  std::vector<int32_t> grid;  // n_cols*n_rows, -1 = empty, -2 = fired/unlabelled, >=0 = cluster id
};

// ------------------------------------------------------------------------------------------------
// O1 + O2 + O3 + O4
// ------------------------------------------------------------------------------------------------
void cluster_event(const Geometry& g, const uint8_t* raw, size_t bytes, EventResult& out, Scratch& sc) {
  const uint32_t L = g.n_layers;
  out.layer_offsets.assign(L + 1, 0);
  // ---- O1: header and bank table (raw format v1, D:R1)
  if (bytes < 16 || bytes % 16) { out.status |= STATUS_BAD_HEADER; return; }
  const uint32_t* w = reinterpret_cast<const uint32_t*>(raw);
  const size_t n_words = bytes / 4;
  if (w[0] != 0x56454C4Fu || w[1] != g.n_sensors) { out.status |= STATUS_BAD_HEADER; return; }
  const uint32_t n_banks = w[1], n_sp_total = w[2];
  const size_t table_words = ((size_t)n_banks + 1 + 3) / 4 * 4;
  const size_t sp_words = ((size_t)n_sp_total + 3) / 4 * 4;
  if (4 + table_words + sp_words != n_words) { out.status |= STATUS_BAD_HEADER; return; }
  const uint32_t* bank_offset = w + 4;
  const uint32_t* sp = w + 4 + table_words;
  if (bank_offset[0] != 0 || bank_offset[n_banks] != n_sp_total) { out.status |= STATUS_BAD_HEADER; return; }
  for (uint32_t j = 0; j < n_banks; ++j)
    if (bank_offset[j] > bank_offset[j + 1]) { out.status |= STATUS_BAD_HEADER; return; }

  if (sc.grid.size() != (size_t)g.n_cols * g.n_rows) sc.grid.assign((size_t)g.n_cols * g.n_rows, -1);
  std::vector<Cluster> clusters;
  std::vector<uint32_t> pix_key, pix_cluster_unsorted;
  std::vector<uint32_t> fired;  // pixel indices row*n_cols+col of the current sensor
  std::vector<uint32_t> stack;
  for (uint32_t s = 0; s < n_banks; ++s) {
    // O1: expand every SP word of bank s (= sensor s) into fired pixels.
    fired.clear();
    for (uint32_t i = bank_offset[s]; i < bank_offset[s + 1]; ++i) {
      uint32_t word = sp[i];
      uint32_t hitmap = word & 0xFF, sp_row = (word >> 8) & 0x3F, sp_col = (word >> 14) & 0x1FF;
      if (2 * sp_col + 1 >= g.n_cols || 4 * sp_row + 3 >= g.n_rows) { out.status |= STATUS_BAD_SP; continue; }
      for (uint32_t bit = 0; bit < 8; ++bit) {
        if (!(hitmap >> bit & 1)) continue;
        uint32_t col = 2 * sp_col + (bit >> 2), row = 4 * sp_row + (bit & 3);
        uint32_t idx = row * g.n_cols + col;
        if (sc.grid[idx] == -1) { sc.grid[idx] = -2; fired.push_back(idx); }  // set semantics: duplicates merge
      }
    }
    // O2: maximal 8-connected components by flood fill.
    for (uint32_t start : fired) {
      if (sc.grid[start] != -2) continue;
      int32_t id = (int32_t)clusters.size();
      Cluster c{};
      c.key = 0xFFFFFFFFu;
      stack.assign(1, start);
      sc.grid[start] = id;
      while (!stack.empty()) {
        uint32_t idx = stack.back();
        stack.pop_back();
        uint32_t row = idx / g.n_cols, col = idx % g.n_cols;
        c.n += 1;
        c.sum_col += col;
        c.sum_row += row;
        c.checksum += mix32(idx);
        uint32_t k = (s << 18) | idx;
        if (k < c.key) c.key = k;
        pix_key.push_back(k);
        pix_cluster_unsorted.push_back((uint32_t)id);
        for (int dr = -1; dr <= 1; ++dr)
          for (int dc = -1; dc <= 1; ++dc) {
            int r2 = (int)row + dr, c2 = (int)col + dc;
            if (r2 < 0 || c2 < 0 || r2 >= (int)g.n_rows || c2 >= (int)g.n_cols) continue;
            uint32_t j = (uint32_t)r2 * g.n_cols + (uint32_t)c2;
            // O2-local ("searches for clusters locally in small regions. Every region can be treated
            // independently"; D:R11): with regions switched on, a cluster never leaves its region of
            // region_sp_cols x region_sp_rows super-pixels.  Off (0, 0) = the exact definition above.
            if (region_sp_cols && ((uint32_t)c2 / 2 / region_sp_cols != col / 2 / region_sp_cols ||
                                   (uint32_t)r2 / 4 / region_sp_rows != row / 4 / region_sp_rows))
              continue;
            if (sc.grid[j] == -2) { sc.grid[j] = id; stack.push_back(j); }
          }
      }
      // O3: centroid -> local mm -> global (x,y,z), then phi16 (normative fp32 tree, D:R3).
      const float* M = g.sensor_ltg + 9 * s;
      float fc = (float)c.sum_col / (float)c.n + 0.5f;
      float fr = (float)c.sum_row / (float)c.n + 0.5f;
      float u = fc * g.pitch_mm, v = fr * g.pitch_mm;
      c.x = std::fmaf(u, M[0], std::fmaf(v, M[1], M[2]));
      c.y = std::fmaf(u, M[3], std::fmaf(v, M[4], M[5]));
      c.z = std::fmaf(u, M[6], std::fmaf(v, M[7], M[8]));
      c.phi = phi16_of(c.x, c.y);
      c.layer = g.module_layer[g.sensor_module[s]];
      clusters.push_back(c);
    }
    for (uint32_t idx : fired) sc.grid[idx] = -1;
  }
  // O4: normative order = ascending (layer, phi16 signed, key)  (D:R4).
  std::vector<uint32_t> order(clusters.size());
  for (uint32_t i = 0; i < order.size(); ++i) order[i] = i;
  std::sort(order.begin(), order.end(), [&](uint32_t a, uint32_t b) {
    const Cluster &ca = clusters[a], &cb = clusters[b];
    if (ca.layer != cb.layer) return ca.layer < cb.layer;
    if (ca.phi != cb.phi) return ca.phi < cb.phi;
    return ca.key < cb.key;
  });
  std::vector<uint32_t> new_index(clusters.size());
  out.clusters.resize(clusters.size());
  for (uint32_t i = 0; i < order.size(); ++i) {
    out.clusters[i] = clusters[order[i]];
    new_index[order[i]] = i;
    out.layer_offsets[out.clusters[i].layer + 1] += 1;
  }
  for (uint32_t l = 0; l < L; ++l) out.layer_offsets[l + 1] += out.layer_offsets[l];
  out.pix_key = pix_key;
  out.pix_cluster.resize(pix_key.size());
  for (size_t i = 0; i < pix_key.size(); ++i) out.pix_cluster[i] = new_index[pix_cluster_unsorted[i]];
  if (out.clusters.size() > 65535) out.status |= STATUS_TOO_MANY_CLUSTERS;
}

// ------------------------------------------------------------------------------------------------
// O5: search by triplet (D:R5, steps T1..T5), linear window scans.
// ------------------------------------------------------------------------------------------------
struct NearCut {
  EventResult& out;
  void touch(uint32_t h) { out.near_cut_hits.push_back(h); }
  // value against an upper cut: near if |v - cut| <= 1e-4 * cut
  void cut(float v, float cut, uint32_t h) {
    if (std::fabs((double)v - (double)cut) <= 1e-4 * std::fabs((double)cut)) { out.near_cut++; touch(h); }
  }
  void window(int d, int w, uint32_t h) {
    int a = std::abs(d);
    if (a == w || a == w + 1) { out.near_cut++; touch(h); }
  }
  // two competing scatter values: near if they differ by <= 1e-4 relative
  void tie(float s1, float s2, uint32_t h) {
    double a = s1, b = s2;
    if (std::fabs(a - b) <= 1e-4 * std::max(a, b)) { out.near_cut++; touch(h); }
  }
};

void search_by_triplet(const std::vector<Hit>& hits, const std::vector<uint32_t>& lo, const Params& P,
                       EventResult& out) {
  const int L = (int)lo.size() - 1;
  std::vector<uint8_t> used(hits.size(), 0);
  std::vector<Track> tracks;  // every track ever created (active or closed), in order of creation
  NearCut nc{out};
  struct Choice { bool any; float S; uint32_t c; };

  for (int i = L - 1; i >= 2; --i) {
    const uint32_t A0 = lo[i], A1 = lo[i + 1], B0 = lo[i - 1], B1 = lo[i], C0 = lo[i - 2], C1 = lo[i - 1];

    // ---- T1 forward: every active track takes best = min (bits(S), c) over the unused hits c of layer C
    //      inside its phi window and scatter cut.  `used` is not modified until T2 (snapshot).
    std::vector<Choice> choice(tracks.size(), Choice{false, 0.0f, 0});
    for (size_t t = 0; t < tracks.size(); ++t) {
      const Track& T = tracks[t];
      if (!T.active) continue;
      const Hit& p = hits[T.hits[T.hits.size() - 2]];  // older
      const Hit& q = hits[T.hits[T.hits.size() - 1]];  // newest
      std::vector<float> all_S;
      for (uint32_t c = C0; c < C1; ++c) {
        if (used[c]) continue;
        int d = dphi(hits[c].phi, q.phi);
        nc.window(d, P.w_fwd_phi16, c);
        if (std::abs(d) > P.w_fwd_phi16) continue;
        float S = scatter(p, q, hits[c]);
        nc.cut(S, P.s_fwd, c);
        if (!(S <= P.s_fwd)) continue;
        all_S.push_back(S);
        Choice& best = choice[t];
        if (!best.any || fbits(S) < fbits(best.S) || (fbits(S) == fbits(best.S) && c < best.c)) best = {true, S, c};
      }
      if (all_S.size() > 1) {  // near-cut bookkeeping only: runner-up within 1e-4 of the winner
        std::sort(all_S.begin(), all_S.end());
        nc.tie(all_S[0], all_S[1], choice[t].c);
      }
    }

    // ---- T2 resolve: for every hit c chosen by >= 1 track the winner is the track with the minimal
    //      (bits(S), track_key), track_key = normative index of the seed's middle hit.  The winner appends c;
    //      every other active track counts a miss and is closed after more than max_skipped misses in a row.
    std::vector<uint8_t> extended(tracks.size(), 0);
    for (uint32_t c = C0; c < C1; ++c) {
      bool any = false;
      size_t winner = 0;
      std::vector<float> all_S;
      for (size_t t = 0; t < tracks.size(); ++t) {
        if (!tracks[t].active || !choice[t].any || choice[t].c != c) continue;
        all_S.push_back(choice[t].S);
        if (!any || fbits(choice[t].S) < fbits(choice[winner].S) ||
            (fbits(choice[t].S) == fbits(choice[winner].S) && tracks[t].seed_key < tracks[winner].seed_key)) {
          any = true;
          winner = t;
        }
      }
      if (!any) continue;
      if (all_S.size() > 1) { std::sort(all_S.begin(), all_S.end()); nc.tie(all_S[0], all_S[1], c); }
      tracks[winner].hits.push_back(c);
      extended[winner] = 1;
      used[c] = 1;
    }
    for (size_t t = 0; t < tracks.size(); ++t) {
      Track& T = tracks[t];
      if (!T.active) continue;
      if (extended[t]) { T.missed = 0; continue; }
      T.missed += 1;
      if (T.missed > P.max_skipped) T.active = false;
    }

    // ---- T3 seed: for every unused middle hit b of layer B, the triplet of b is the argmin over (a, c) of
    //      (bits(S(a,b,c)), a, c) with a in A, c in C unused, inside the phi windows around b, |slopes(a->b)| <=
    //      max_slope and S <= s_seed.
    struct Triplet { uint32_t a, b, c; float S; };
    std::vector<Triplet> triplets;
    for (uint32_t b = B0; b < B1; ++b) {
      if (used[b]) continue;
      const Hit& hb = hits[b];
      bool found = false;
      Triplet best{};
      std::vector<float> all_S;
      for (uint32_t a = A0; a < A1; ++a) {
        if (used[a]) continue;
        const Hit& ha = hits[a];
        int da = dphi(ha.phi, hb.phi);
        nc.window(da, P.w_seed_phi16, a);
        if (std::abs(da) > P.w_seed_phi16) continue;
        float dz_ab = hb.z - ha.z;
        float tx = (hb.x - ha.x) / dz_ab, ty = (hb.y - ha.y) / dz_ab;
        nc.cut(std::fabs(tx), P.max_slope, a);
        nc.cut(std::fabs(ty), P.max_slope, a);
        if (!(std::fabs(tx) <= P.max_slope) || !(std::fabs(ty) <= P.max_slope)) continue;
        for (uint32_t c = C0; c < C1; ++c) {
          if (used[c]) continue;
          int dc = dphi(hits[c].phi, hb.phi);
          nc.window(dc, P.w_seed_phi16, c);
          if (std::abs(dc) > P.w_seed_phi16) continue;
          float S = scatter(ha, hb, hits[c]);
          nc.cut(S, P.s_seed, b);
          if (!(S <= P.s_seed)) continue;
          all_S.push_back(S);
          bool better = !found || fbits(S) < fbits(best.S) ||
                        (fbits(S) == fbits(best.S) && (a < best.a || (a == best.a && c < best.c)));
          if (better) { best = {a, b, c, S}; found = true; }
        }
      }
      if (!found) continue;
      if (all_S.size() > 1) { std::sort(all_S.begin(), all_S.end()); nc.tie(all_S[0], all_S[1], b); }
      triplets.push_back(best);
    }

    // ---- T4 resolve: a triplet is accepted iff it holds the minimal key (bits(S), b) among all triplets (one
    //      per b) that contain its a, and likewise among all that contain its c.  Accepted -> new active track
    //      [a, b, c]; rejected triplets vanish and their hits stay free.  (Acceptance depends only on the list
    //      of triplets, not on `used`, so marking hits here does not make the result order dependent.)
    for (const Triplet& t : triplets) {
      const uint64_t key = ((uint64_t)fbits(t.S) << 32) | t.b;
      bool accepted = true;
      for (const Triplet& o : triplets) {
        if (o.b == t.b || (o.a != t.a && o.c != t.c)) continue;
        nc.tie(t.S, o.S, t.b);
        const uint64_t okey = ((uint64_t)fbits(o.S) << 32) | o.b;
        if (okey < key) accepted = false;
      }
      if (!accepted) continue;
      Track T;
      T.hits = {t.a, t.b, t.c};
      T.seed_key = t.b;
      T.s_seed = t.S;
      T.missed = 0;
      T.active = true;
      T.x0 = T.y0 = T.tx = T.ty = 0;
      tracks.push_back(T);
      used[t.a] = used[t.b] = used[t.c] = 1;
    }
  }

  // ---- T5 finalise: all tracks are closed; >= 4 hits -> output; exactly 3 hits -> output iff S_seed <= s_weak
  //      (dropped 3-hit tracks keep their hits consumed, which no longer matters after the last iteration).
  for (Track& T : tracks) {
    T.active = false;
    if (T.hits.size() == 3) {
      nc.cut(T.s_seed, P.s_weak, T.hits[1]);
      if (!(T.s_seed <= P.s_weak)) continue;
    }
    out.tracks.push_back(T);
  }
}

// ------------------------------------------------------------------------------------------------
// O6: unweighted least-squares straight line, x and y separately, reference plane z = 0; fp64 from the fp32 hit
// coordinates, rounded to fp32 (D:R6).
// ------------------------------------------------------------------------------------------------
void fit_line(const std::vector<Hit>& hits, Track& T) {
  const double n = (double)T.hits.size();
  double zm = 0, xm = 0, ym = 0;
  for (uint32_t h : T.hits) { zm += hits[h].z; xm += hits[h].x; ym += hits[h].y; }
  zm /= n; xm /= n; ym /= n;
  double szz = 0, szx = 0, szy = 0;
  for (uint32_t h : T.hits) {
    double dz = hits[h].z - zm;
    szz += dz * dz;
    szx += dz * (hits[h].x - xm);
    szy += dz * (hits[h].y - ym);
  }
  double tx = szx / szz, ty = szy / szz;
  T.tx = (float)tx;
  T.ty = (float)ty;
  T.x0 = (float)(xm - tx * zm);
  T.y0 = (float)(ym - ty * zm);
}

// ------------------------------------------------------------------------------------------------
// O7: simple Kalman filter over the hits of a track in the order they were added (downstream -> upstream), x and y
// independent, state (pos, slope) per projection (D:R9 step by step).  fp64 from the fp32 hit coordinates.
//   measurement variance  var_m = pitch^2 / 12
//   scattering per plane  theta0^2 = (13.6 MeV / p)^2 * X,  p = pT / sin(theta),  pT = 400 MeV,  X = 0.02;
//                         sin^2(theta) = (tx^2 + ty^2) / (1 + tx^2 + ty^2) with the slopes of the first two hits;
//                         q_x = theta0^2 (1 + tx^2)(1 + tx^2 + ty^2), q_y likewise with ty
//   start at hit 0:       pos = measured, slope = 0, C = diag(var_m, 1)
//   for hit k = 1..n-1:   C11 += q; propagate by dz = z_k - z_{k-1}; update with the measured position
// out12 = x, y, tx, ty, z (of the last hit), chi2 (x + y), C00x, C01x, C11x, C00y, C01y, C11y.
// ------------------------------------------------------------------------------------------------
void kalman_track(uint32_t n, const float* x, const float* y, const float* z, double pitch, double* out12) {
  const double var_m = pitch * pitch / 12.0;
  const double tx0 = ((double)x[1] - x[0]) / ((double)z[1] - z[0]);
  const double ty0 = ((double)y[1] - y[0]) / ((double)z[1] - z[0]);
  const double t2 = tx0 * tx0 + ty0 * ty0;
  const double theta02 = (13.6 / 400.0) * (13.6 / 400.0) * 0.02 * t2 / (1.0 + t2);
  const double q[2] = {theta02 * (1.0 + tx0 * tx0) * (1.0 + t2), theta02 * (1.0 + ty0 * ty0) * (1.0 + t2)};
  const float* m[2] = {x, y};
  double chi2 = 0;
  for (int pr = 0; pr < 2; ++pr) {
    double pos = m[pr][0], slope = 0, c00 = var_m, c01 = 0, c11 = 1.0;
    for (uint32_t k = 1; k < n; ++k) {
      const double dz = (double)z[k] - z[k - 1];
      c11 += q[pr];                                // scattering in the plane just left
      pos += slope * dz;                           // straight-line propagation
      c00 += 2.0 * dz * c01 + dz * dz * c11;
      c01 += dz * c11;
      const double r = m[pr][k] - pos, S = c00 + var_m;
      const double k0 = c00 / S, k1 = c01 / S;     // gain
      pos += k0 * r;
      slope += k1 * r;
      c11 -= k1 * c01;
      c01 -= k0 * c01;
      c00 -= k0 * c00;
      chi2 += r * r / S;
    }
    out12[pr] = pos; out12[2 + pr] = slope;
    out12[6 + 3 * pr] = c00; out12[7 + 3 * pr] = c01; out12[8 + 3 * pr] = c11;
  }
  out12[4] = z[n - 1];
  out12[5] = chi2;
}

// ------------------------------------------------------------------------------------------------
// O8: primary vertices of one event (D:R10 step by step).
//   1. z of closest approach to the beam line (x = y = 0) from the straight-line fit (O6, fp32, normative ops):
//      t2 = tx*tx + ty*ty (fma), zp = -(x0*tx + y0*ty) / t2; tracks with t2 < 1e-8 or zp outside [-300, 300) are left out
//   2. histogram h of zp in 600 bins of 1 mm; s[b] = h[b-1] + h[b] + h[b+1]; bin b is a candidate iff s[b] >= 4 and
//      (s[b], h[b]) > (s[b-1], h[b-1]) and (s[b], h[b]) >= (s[b+1], h[b+1]) in lexicographic order;
//      z_seed = -300 + b + 0.5 + (h[b+1] - h[b-1]) / s[b]
//   3. every candidate is fitted with ALL tracks, 8 iterations from (0, 0, z_seed): track position and variance at the
//      vertex z from its Kalman state (O7); chi2_t = dx^2/var_x + dy^2/var_y; Tukey weight w = (1 - chi2_t/12)^2 below
//      12, else 0; one exact weighted least-squares step for (vx, vy, vz) per iteration
//   4. accepted iff sum w >= 3 after the last iteration; a vertex is dropped if another accepted one lies within 1 mm
//      in z and has a sum w more than 0.1 % larger (within 0.1 %: the earlier candidate wins)
// kal: [n][12] from O7; out rows: x, y, z, sum_w, n_tracks (w > 0), chi2 (sum w chi2_t), z_seed, 0.  fp64 except step 1.
// ------------------------------------------------------------------------------------------------
constexpr int kPvBins = 600;
constexpr int kPvMax = 32;

// cand_out (optional, pins only): every candidate as it stands after step 3, before the duplicate removal of step 4:
// rows of z_seed, x, y, z, sum_w, ok (1 = fit converged and sum w >= 3), at most cand_cap rows.
uint32_t find_pvs(uint32_t n, const float* x0, const float* y0, const float* tx, const float* ty, const double* kal,
                  double* out /* [kPvMax][8] */, uint32_t* n_candidates, int n_iter = 8, double* cand_out = nullptr,
                  uint32_t cand_cap = 0) {
  int h[kPvBins + 2] = {0};  // h[b + 1] = bin b; guard bins at both ends
  for (uint32_t i = 0; i < n; ++i) {
    const float t2 = std::fmaf(tx[i], tx[i], ty[i] * ty[i]);
    if (!(t2 >= 1e-8f)) continue;
    const float zp = -std::fmaf(x0[i], tx[i], y0[i] * ty[i]) / t2;
    const float u = zp + 300.0f;
    if (!(u >= 0.0f) || !(u < (float)kPvBins)) continue;
    h[(int)std::floor(u) + 1] += 1;
  }
  struct Cand { double z_seed, v[3], sw, chi2; int nw; bool ok; };
  std::vector<Cand> cands;
  for (int b = 0; b < kPvBins; ++b) {
    const int hm = h[b], hc = h[b + 1], hp = h[b + 2];
    const int s = hm + hc + hp;
    const int sl = (b > 0 ? h[b - 1] : 0) + hm + hc, sr = hc + hp + (b + 3 < kPvBins + 2 ? h[b + 3] : 0);
    // local maximum of (s, h) in lexicographic order: strictly above the left neighbour, not below the right one
    const bool above_left = s > sl || (s == sl && hc > hm), not_below_right = s > sr || (s == sr && hc >= hp);
    if (s >= 4 && above_left && not_below_right) {
      Cand c{};
      c.z_seed = -300.0 + b + 0.5 + (double)(hp - hm) / s;
      cands.push_back(c);
    }
  }
  *n_candidates = (uint32_t)cands.size();
  for (Cand& c : cands) {
    double vx = 0, vy = 0, vz = c.z_seed;
    c.ok = true;
    for (int it = 0; it < n_iter && c.ok; ++it) {
      double a00 = 0, a11 = 0, a02 = 0, a12 = 0, a22 = 0, b0 = 0, b1 = 0, b2 = 0, sw = 0, chi2 = 0;
      int nw = 0;
      for (uint32_t i = 0; i < n; ++i) {
        const double* k = kal + 12 * (size_t)i;
        const double d = vz - k[4];
        const double dx = k[0] + k[2] * d - vx, dy = k[1] + k[3] * d - vy;
        const double var_x = k[6] + 2 * d * k[7] + d * d * k[8], var_y = k[9] + 2 * d * k[10] + d * d * k[11];
        const double c2 = dx * dx / var_x + dy * dy / var_y;
        if (!(c2 < 12.0)) continue;
        const double w = (1 - c2 / 12.0) * (1 - c2 / 12.0);
        const double wx = w / var_x, wy = w / var_y;
        a00 += wx; a11 += wy; a02 -= wx * k[2]; a12 -= wy * k[3]; a22 += wx * k[2] * k[2] + wy * k[3] * k[3];
        b0 += wx * dx; b1 += wy * dy; b2 -= wx * k[2] * dx + wy * k[3] * dy;
        sw += w; chi2 += w * c2; nw += 1;
      }
      c.sw = sw; c.chi2 = chi2; c.nw = nw;
      if (it == n_iter - 1) break;  // the sums of the last pass describe the final position
      // solve [[a00, 0, a02], [0, a11, a12], [a02, a12, a22]] delta = b by eliminating the first two unknowns
      if (!(a00 > 0) || !(a11 > 0)) { c.ok = false; break; }
      const double den = a22 - a02 * a02 / a00 - a12 * a12 / a11;
      if (!(den > 0)) { c.ok = false; break; }
      const double dz = (b2 - a02 * b0 / a00 - a12 * b1 / a11) / den;
      vx += (b0 - a02 * dz) / a00;
      vy += (b1 - a12 * dz) / a11;
      vz += dz;
    }
    c.v[0] = vx; c.v[1] = vy; c.v[2] = vz;
    c.ok = c.ok && c.sw >= 3.0;
  }
  for (size_t i = 0; cand_out && i < cands.size() && i < cand_cap; ++i) {
    double* o = cand_out + 6 * i;
    o[0] = cands[i].z_seed; o[1] = cands[i].v[0]; o[2] = cands[i].v[1]; o[3] = cands[i].v[2]; o[4] = cands[i].sw;
    o[5] = cands[i].ok ? 1.0 : 0.0;
  }
  uint32_t n_out = 0;
  for (size_t i = 0; i < cands.size(); ++i) {
    if (!cands[i].ok) continue;
    bool dropped = false;
    for (size_t j = 0; j < cands.size() && !dropped; ++j)
      if (j != i && cands[j].ok && std::fabs(cands[j].v[2] - cands[i].v[2]) < 1.0) {
        // candidates that converged to the same vertex have the same sum w up to rounding: within 0.1 % is a tie
        const bool j_larger = cands[j].sw > cands[i].sw * 1.001, i_larger = cands[i].sw > cands[j].sw * 1.001;
        if (j_larger || (!i_larger && j < i)) dropped = true;
      }
    if (dropped || n_out >= (uint32_t)kPvMax) continue;
    double* o = out + 8 * (size_t)n_out++;
    o[0] = cands[i].v[0]; o[1] = cands[i].v[1]; o[2] = cands[i].v[2]; o[3] = cands[i].sw;
    o[4] = cands[i].nw; o[5] = cands[i].chi2; o[6] = cands[i].z_seed; o[7] = 0;
  }
  return n_out;
}

void reconstruct_event(const Geometry& g, const uint8_t* raw, size_t bytes, EventResult& out, Scratch& sc) {
  cluster_event(g, raw, bytes, out, sc);
  if (out.status & (STATUS_BAD_HEADER | STATUS_TOO_MANY_CLUSTERS)) return;
  std::vector<Hit> hits(out.clusters.size());
  for (size_t i = 0; i < hits.size(); ++i) hits[i] = {out.clusters[i].x, out.clusters[i].y, out.clusters[i].z, out.clusters[i].phi};
  search_by_triplet(hits, out.layer_offsets, g.params, out);
  for (Track& T : out.tracks) fit_line(hits, T);
}

struct Run {
  std::vector<EventResult> events;
};

}  // namespace

// ------------------------------------------------------------------------------------------------
// C interface for ctypes (tests / bench cpu_baseline only)
// ------------------------------------------------------------------------------------------------
extern "C" {

uint32_t oracle_mix32(uint32_t v) { return mix32(v); }
float oracle_atan2_poly(float x, float y) { return atan2_poly(x, y); }
int32_t oracle_phi16(float x, float y) { return phi16_of(x, y); }
float oracle_scatter(const float* a, const float* b, const float* c) {
  Hit ha{a[0], a[1], a[2], 0}, hb{b[0], b[1], b[2], 0}, hc{c[0], c[1], c[2], 0};
  return scatter(ha, hb, hc);
}

// Fit one track given its hit coordinates; out = x0, y0, tx, ty.
void oracle_fit(uint32_t n, const float* x, const float* y, const float* z, float* out4) {
  std::vector<Hit> hits(n);
  Track T;
  for (uint32_t i = 0; i < n; ++i) { hits[i] = {x[i], y[i], z[i], 0}; T.hits.push_back(i); }
  fit_line(hits, T);
  out4[0] = T.x0; out4[1] = T.y0; out4[2] = T.tx; out4[3] = T.ty;
}

// O7 for a batch of tracks: track t has hits abs_hits[hit_offsets[t] .. hit_offsets[t+1]) (indices into x, y, z).
void oracle_kalman(uint32_t n_tracks, const uint32_t* hit_offsets, const uint32_t* abs_hits, const float* x,
                   const float* y, const float* z, double pitch, double* out12) {
  std::vector<float> hx, hy, hz;
  for (uint32_t t = 0; t < n_tracks; ++t) {
    const uint32_t n = hit_offsets[t + 1] - hit_offsets[t];
    hx.resize(n); hy.resize(n); hz.resize(n);
    for (uint32_t k = 0; k < n; ++k) {
      const uint32_t h = abs_hits[hit_offsets[t] + k];
      hx[k] = x[h]; hy[k] = y[h]; hz[k] = z[h];
    }
    kalman_track(n, hx.data(), hy.data(), hz.data(), pitch, out12 + 12 * (size_t)t);
  }
}

// O8 for a batch: tracks of event e are [track_offsets[e], track_offsets[e+1]); out [n_events][32][8], counts [n_events],
// candidates [n_events] (histogram peaks before the fit).
void oracle_pvs(uint32_t n_events, const uint32_t* track_offsets, const float* x0, const float* y0, const float* tx,
                const float* ty, const double* kal, double* out, uint32_t* counts, uint32_t* candidates,
                int n_iter /* 8 in the method; other values only for the pins */) {
  for (uint32_t e = 0; e < n_events; ++e) {
    const uint32_t t0 = track_offsets[e], n = track_offsets[e + 1] - t0;
    counts[e] = find_pvs(n, x0 + t0, y0 + t0, tx + t0, ty + t0, kal + 12 * (size_t)t0, out + (size_t)e * kPvMax * 8,
                         candidates + e, n_iter);
  }
}

// O8 for ONE event, also returning every candidate before step 4 (cand [cand_cap][6]: z_seed, x, y, z, sum_w, ok).
// Returns the number of vertices; *n_candidates = histogram peaks.  Used by the pins of step 4 and by the parity test's
// near-cut accounting.
uint32_t oracle_pv_candidates(uint32_t n, const float* x0, const float* y0, const float* tx, const float* ty,
                              const double* kal, double* out /* [32][8] */, uint32_t* n_candidates, double* cand,
                              uint32_t cand_cap) {
  return find_pvs(n, x0, y0, tx, ty, kal, out, n_candidates, 8, cand, cand_cap);
}

// O2-local: region size in super-pixels for the runs that follow (0, 0 = exact connected components).
void oracle_set_cluster_regions(uint32_t sp_cols, uint32_t sp_rows) {
  region_sp_cols = sp_cols && sp_rows ? sp_cols : 0;
  region_sp_rows = sp_cols && sp_rows ? sp_rows : 0;
}

void* oracle_run(const Geometry* g, const uint8_t* raw, const uint32_t* event_offsets, uint32_t n_events,
                 uint32_t n_threads) {
  Run* run = new Run();
  run->events.resize(n_events);
  if (n_threads <= 1) {
    Scratch sc;
    for (uint32_t e = 0; e < n_events; ++e)
      reconstruct_event(*g, raw + event_offsets[e], event_offsets[e + 1] - event_offsets[e], run->events[e], sc);
  } else {
    // Contiguous event ranges per thread; every thread runs the unchanged single-threaded code.
    std::vector<std::thread> pool;
    for (uint32_t t = 0; t < n_threads; ++t) {
      uint32_t e0 = (uint64_t)n_events * t / n_threads, e1 = (uint64_t)n_events * (t + 1) / n_threads;
      pool.emplace_back([=]() {
        Scratch sc;
        for (uint32_t e = e0; e < e1; ++e)
          reconstruct_event(*g, raw + event_offsets[e], event_offsets[e + 1] - event_offsets[e], run->events[e], sc);
      });
    }
    for (auto& th : pool) th.join();
  }
  return run;
}

// Search-by-triplet + fit on caller-given hits of ONE event (already in normative order).
void* oracle_run_hits(const Params* P, uint32_t n_hits, const float* x, const float* y, const float* z,
                      const int16_t* phi, uint32_t n_layers, const uint32_t* layer_offsets) {
  Run* run = new Run();
  run->events.resize(1);
  EventResult& out = run->events[0];
  std::vector<Hit> hits(n_hits);
  for (uint32_t i = 0; i < n_hits; ++i) hits[i] = {x[i], y[i], z[i], phi[i]};
  out.layer_offsets.assign(layer_offsets, layer_offsets + n_layers + 1);
  out.clusters.resize(n_hits);
  for (uint32_t i = 0; i < n_hits; ++i) {
    out.clusters[i] = Cluster{};
    out.clusters[i].x = x[i]; out.clusters[i].y = y[i]; out.clusters[i].z = z[i]; out.clusters[i].phi = phi[i];
  }
  search_by_triplet(hits, out.layer_offsets, *P, out);
  for (Track& T : out.tracks) fit_line(hits, T);
  return run;
}

void oracle_free(void* h) { delete (Run*)h; }

// Totals: what = 0 clusters, 1 tracks, 2 track hits, 3 pixels, 4 near-cut hits
uint64_t oracle_total(void* h, int what) {
  Run* run = (Run*)h;
  uint64_t n = 0;
  for (const EventResult& ev : run->events) {
    switch (what) {
      case 0: n += ev.clusters.size(); break;
      case 1: n += ev.tracks.size(); break;
      case 2: for (const Track& T : ev.tracks) n += T.hits.size(); break;
      case 3: n += ev.pix_key.size(); break;
      case 4: n += ev.near_cut_hits.size(); break;
    }
  }
  return n;
}

// Flattened, compacted outputs in the layout of the C ABI (include/allen_velo.h), plus oracle-only extras.
void oracle_export_clusters(void* h, uint32_t n_layers, uint32_t* event_offsets, uint32_t* layer_offsets,
                            uint32_t* key, uint32_t* n_pixels, uint32_t* sum_col, uint32_t* sum_row, float* x,
                            float* y, float* z, int16_t* phi16, uint32_t* checksum, uint32_t* status) {
  Run* run = (Run*)h;
  uint32_t pos = 0;
  for (size_t e = 0; e < run->events.size(); ++e) {
    const EventResult& ev = run->events[e];
    event_offsets[e] = pos;
    status[e] = ev.status;
    for (uint32_t l = 0; l < n_layers; ++l) layer_offsets[e * n_layers + l] = pos + ev.layer_offsets[l];
    for (const Cluster& c : ev.clusters) {
      key[pos] = c.key; n_pixels[pos] = c.n; sum_col[pos] = c.sum_col; sum_row[pos] = c.sum_row;
      x[pos] = c.x; y[pos] = c.y; z[pos] = c.z; phi16[pos] = c.phi; checksum[pos] = c.checksum;
      ++pos;
    }
  }
  event_offsets[run->events.size()] = pos;
  layer_offsets[run->events.size() * n_layers] = pos;
}

void oracle_export_tracks(void* h, uint32_t* event_offsets, uint32_t* hit_offsets, uint16_t* hits, float* x0,
                          float* y0, float* tx, float* ty) {
  Run* run = (Run*)h;
  uint32_t t = 0, hpos = 0;
  for (size_t e = 0; e < run->events.size(); ++e) {
    event_offsets[e] = t;
    for (const Track& T : run->events[e].tracks) {
      hit_offsets[t] = hpos;
      for (uint32_t hh : T.hits) hits[hpos++] = (uint16_t)hh;
      x0[t] = T.x0; y0[t] = T.y0; tx[t] = T.tx; ty[t] = T.ty;
      ++t;
    }
  }
  event_offsets[run->events.size()] = t;
  hit_offsets[t] = hpos;
}

// Pixel membership: for every decoded pixel its key (sensor<<18 | row*n_cols+col), event and cluster (event-local).
void oracle_export_pixels(void* h, uint32_t* pix_event, uint32_t* pix_key, uint32_t* pix_cluster) {
  Run* run = (Run*)h;
  size_t pos = 0;
  for (size_t e = 0; e < run->events.size(); ++e) {
    const EventResult& ev = run->events[e];
    for (size_t i = 0; i < ev.pix_key.size(); ++i) {
      pix_event[pos] = (uint32_t)e; pix_key[pos] = ev.pix_key[i]; pix_cluster[pos] = ev.pix_cluster[i];
      ++pos;
    }
  }
}

void oracle_export_near_cut(void* h, uint32_t* per_event_count, uint32_t* hit_event, uint32_t* hit_index) {
  Run* run = (Run*)h;
  size_t pos = 0;
  for (size_t e = 0; e < run->events.size(); ++e) {
    const EventResult& ev = run->events[e];
    per_event_count[e] = ev.near_cut;
    for (uint32_t hh : ev.near_cut_hits) { hit_event[pos] = (uint32_t)e; hit_index[pos] = hh; ++pos; }
  }
}

}  // extern "C"
