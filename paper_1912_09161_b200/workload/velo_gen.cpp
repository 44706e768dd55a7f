// Synthetic VELO-like event generator and raw-bank packer (input generation only).
//
// This file holds NONE of the reconstruction method's arithmetic: it draws particles, propagates
// straight lines through a pixel geometry, digitises crossings to fired pixels and packs them into
// the raw format v1 of include/allen_velo.h (the inverse of the decoder).  It serves both the CPU
// oracle (oracle/) and the CUDA path as the single source of seeded inputs; neither of them shares
// any code with it.  Recipe: DESIGN.md "Input recipe", after SURVEY.md §8(d) and BASELINE.json configs
// (paper context: ~6 pp collisions per crossing PAPER.md:96; 26 Velo planes PAPER.md:165; 2<eta<5
// PAPER.md:240; batches of >=1000 events PAPER.md:135).
//
// RNG: Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11), keyed by the
// 64-bit seed, counter = (draw index lo, draw index hi, event index lo, event index hi), so every event
// has its own stream and its content does not depend on the batch it is generated in.
//
// Build: g++ -O2 -shared -fPIC (see paper_1912_09161_b200/workload/__init__.py).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Philox {
  uint32_t key[2];
  uint32_t ctr[4];
  uint32_t out[4];
  int have = 0;
  Philox(uint64_t seed, uint64_t stream) {
    key[0] = (uint32_t)seed;
    key[1] = (uint32_t)(seed >> 32);
    ctr[0] = ctr[1] = 0;
    ctr[2] = (uint32_t)stream;
    ctr[3] = (uint32_t)(stream >> 32);
  }
  static inline void mulhilo(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
    uint64_t p = (uint64_t)a * b;
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
  }
  void block() {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
      uint32_t hi0, lo0, hi1, lo1;
      mulhilo(0xD2511F53u, c0, hi0, lo0);
      mulhilo(0xCD9E8D57u, c2, hi1, lo1);
      uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
      c0 = n0; c1 = n1; c2 = n2; c3 = n3;
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
    if (++ctr[0] == 0) ++ctr[1];
    have = 4;
  }
  uint32_t u32() {
    if (!have) block();
    return out[4 - have--];
  }
  double uniform() {  // [0,1) with 53 bits
    uint32_t a = u32() >> 5, b = u32() >> 6;
    return (a * 67108864.0 + b) * (1.0 / 9007199254740992.0);
  }
  double uniform_open() {  // (0,1]
    return 1.0 - uniform();
  }
  double normal() {  // Box-Muller, one value per call (second discarded for a fixed draw count)
    double u1 = uniform_open(), u2 = uniform();
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586 * u2);
  }
  int poisson(double mean) {  // Knuth multiplication; mean <= ~30 here
    double L = std::exp(-mean), p = 1.0;
    int k = 0;
    do { ++k; p *= uniform(); } while (p > L);
    return k - 1;
  }
  double exponential(double mean) { return -mean * std::log(uniform_open()); }
  uint32_t below(uint32_t n) { return (uint32_t)(uniform() * n); }
};

struct Sensor {
  double ox, oy, ecx, ecy, erx, ery, z;
};

struct Config {
  uint64_t seed;
  uint64_t first_event;
  uint32_t n_events;
  int32_t fixed_pv;       // >0: exactly this many PVs; else Poisson(nu)
  double nu;
  int32_t fixed_tracks;   // >0: exactly this many tracks per PV; else Poisson(mean_tracks)
  double mean_tracks;
  double noise_occ;
  double hit_eff;
  int32_t charge_sharing;
  double scatter_sigma;
  double displaced_frac;
  double displaced_mean;
  int32_t isolate;
  int32_t shuffle_sp;
  // geometry
  uint32_t n_sensors, n_modules, n_cols, n_rows;
  double pitch;
};

struct Gen {
  Config cfg;
  std::vector<Sensor> sensors;
  std::vector<uint16_t> sensor_module;  // module index of every sensor
  std::vector<double> module_z;         // z of every module (sensors of a module share z)
  std::vector<uint32_t> module_order;   // modules by increasing z
  std::vector<std::vector<uint32_t>> module_sensors;
  // outputs
  std::vector<uint8_t> raw;
  std::vector<uint32_t> event_offsets;
  // particle truth
  std::vector<uint32_t> p_event;
  std::vector<int32_t> p_pv;
  std::vector<uint8_t> p_displaced;
  std::vector<double> p_ox, p_oy, p_oz, p_tx, p_ty;
  std::vector<uint32_t> p_n_crossings, p_n_hits;
  // pixel truth (one entry per (pixel, source)); particle = -1 for noise
  std::vector<uint32_t> x_event;
  std::vector<uint16_t> x_sensor, x_col, x_row;
  std::vector<int32_t> x_particle;
  std::vector<uint8_t> x_main;  // 1 = pixel containing the crossing point, 0 = charge-sharing neighbour / noise
  // PV truth
  std::vector<uint32_t> v_event;
  std::vector<double> v_x, v_y, v_z;
};

struct Pix {
  uint16_t sensor, col, row;
  uint8_t main;
};

// Propagate one particle; returns fired pixels (after efficiency and charge sharing).
void propagate(const Gen& g, Philox& rng, double ox, double oy, double oz, double tx, double ty,
               std::vector<Pix>& pix, uint32_t& n_cross, uint32_t& n_hit) {
  const Config& c = g.cfg;
  double x = ox, y = oy, z = oz;
  const double len_u = c.n_cols * c.pitch, len_v = c.n_rows * c.pitch;
  n_cross = n_hit = 0;
  for (uint32_t m : g.module_order) {
    double zm = g.module_z[m];
    if (zm <= oz) continue;
    x += tx * (zm - z);
    y += ty * (zm - z);
    z = zm;
    bool crossed = false;
    for (uint32_t s : g.module_sensors[m]) {
      const Sensor& S = g.sensors[s];
      double u = (x - S.ox) * S.ecx + (y - S.oy) * S.ecy;
      double v = (x - S.ox) * S.erx + (y - S.oy) * S.ery;
      if (u < 0.0 || u >= len_u || v < 0.0 || v >= len_v) continue;
      crossed = true;
      ++n_cross;
      bool eff = (c.hit_eff >= 1.0) ? true : (rng.uniform() < c.hit_eff);
      if (!eff) break;
      ++n_hit;
      double fu = u / c.pitch, fv = v / c.pitch;
      int col = (int)std::floor(fu), row = (int)std::floor(fv);
      if (col >= (int)c.n_cols) col = c.n_cols - 1;
      if (row >= (int)c.n_rows) row = c.n_rows - 1;
      pix.push_back({(uint16_t)s, (uint16_t)col, (uint16_t)row, 1});
      if (c.charge_sharing) {
        double du = fu - col, dv = fv - row;
        int nc = du < 0.2 ? col - 1 : (du > 0.8 ? col + 1 : col);
        int nr = dv < 0.2 ? row - 1 : (dv > 0.8 ? row + 1 : row);
        if (nc != col && nc >= 0 && nc < (int)c.n_cols) pix.push_back({(uint16_t)s, (uint16_t)nc, (uint16_t)row, 0});
        if (nr != row && nr >= 0 && nr < (int)c.n_rows) pix.push_back({(uint16_t)s, (uint16_t)col, (uint16_t)nr, 0});
      }
      break;  // sensors of one module do not overlap
    }
    if (crossed && c.scatter_sigma > 0.0) {
      tx += c.scatter_sigma * rng.normal();
      ty += c.scatter_sigma * rng.normal();
    }
  }
}

void draw_direction(Philox& rng, double& tx, double& ty) {
  double eta = 2.0 + 3.0 * rng.uniform();
  double phi = 6.283185307179586 * rng.uniform();
  double theta = 2.0 * std::atan(std::exp(-eta));
  double t = std::tan(theta);
  tx = t * std::cos(phi);
  ty = t * std::sin(phi);
}

bool touches(const std::vector<Pix>& a, const std::vector<Pix>& b) {
  for (const Pix& p : a)
    for (const Pix& q : b)
      if (p.sensor == q.sensor && std::abs((int)p.col - (int)q.col) <= 1 && std::abs((int)p.row - (int)q.row) <= 1)
        return true;
  return false;
}

void generate_event(Gen& g, uint64_t event_index, uint32_t local_event) {
  const Config& c = g.cfg;
  Philox rng(c.seed, event_index);
  std::vector<std::vector<Pix>> accepted;  // for isolation (config 0)
  struct EvPix { uint16_t sensor, col, row; };
  std::vector<EvPix> fired;

  int n_pv = c.fixed_pv > 0 ? c.fixed_pv : rng.poisson(c.nu);
  for (int ipv = 0; ipv < n_pv; ++ipv) {
    double vx = 0.04 * rng.normal(), vy = 0.04 * rng.normal(), vz = 45.0 * rng.normal();
    g.v_event.push_back(local_event);
    g.v_x.push_back(vx); g.v_y.push_back(vy); g.v_z.push_back(vz);
    int n_trk = c.fixed_tracks > 0 ? c.fixed_tracks : rng.poisson(c.mean_tracks);
    for (int it = 0; it < n_trk; ++it) {
      std::vector<Pix> pix;
      double ox, oy, oz, tx, ty;
      uint32_t n_cross = 0, n_hit = 0;
      bool displaced = false;
      for (int attempt = 0; attempt < 1000; ++attempt) {
        pix.clear();
        ox = vx; oy = vy; oz = vz;
        displaced = c.displaced_frac > 0.0 && rng.uniform() < c.displaced_frac;
        if (displaced) {
          double L = rng.exponential(c.displaced_mean);
          double dx, dy;
          draw_direction(rng, dx, dy);
          double norm = std::sqrt(1.0 + dx * dx + dy * dy);
          ox += L * dx / norm; oy += L * dy / norm; oz += L / norm;
        }
        draw_direction(rng, tx, ty);
        propagate(g, rng, ox, oy, oz, tx, ty, pix, n_cross, n_hit);
        if (!c.isolate) break;
        bool clash = false;
        for (const auto& other : accepted)
          if (touches(pix, other)) { clash = true; break; }
        if (!clash) break;
      }
      if (c.isolate) accepted.push_back(pix);
      int32_t pid = (int32_t)g.p_event.size();
      g.p_event.push_back(local_event);
      g.p_pv.push_back(ipv);
      g.p_displaced.push_back(displaced ? 1 : 0);
      g.p_ox.push_back(ox); g.p_oy.push_back(oy); g.p_oz.push_back(oz);
      g.p_tx.push_back(tx); g.p_ty.push_back(ty);
      g.p_n_crossings.push_back(n_cross);
      g.p_n_hits.push_back(n_hit);
      for (const Pix& p : pix) {
        g.x_event.push_back(local_event);
        g.x_sensor.push_back(p.sensor); g.x_col.push_back(p.col); g.x_row.push_back(p.row);
        g.x_particle.push_back(pid);
        g.x_main.push_back(p.main);
        fired.push_back({p.sensor, p.col, p.row});
      }
    }
  }
  // Noise: every pixel fires independently with probability noise_occ (count ~ Binomial(n_pixels, occ)),
  // drawn by geometric skipping over the pixel index.
  if (c.noise_occ > 0.0) {
    const double n_pix = (double)c.n_cols * c.n_rows;
    const double lg = std::log1p(-c.noise_occ);
    for (uint32_t s = 0; s < c.n_sensors; ++s) {
      double pos = -1.0;
      for (;;) {
        pos += 1.0 + std::floor(std::log(rng.uniform_open()) / lg);
        if (pos >= n_pix) break;
        uint32_t idx = (uint32_t)pos;
        uint16_t row = (uint16_t)(idx / c.n_cols), col = (uint16_t)(idx % c.n_cols);
        g.x_event.push_back(local_event);
        g.x_sensor.push_back((uint16_t)s); g.x_col.push_back(col); g.x_row.push_back(row);
        g.x_particle.push_back(-1);
        g.x_main.push_back(0);
        fired.push_back({(uint16_t)s, col, row});
      }
    }
  }
  // Pack: per sensor, OR pixels into 2(col) x 4(row) super-pixel words.
  std::vector<uint64_t> keys;  // (sensor, sp_col, sp_row, bit)
  keys.reserve(fired.size());
  for (const EvPix& p : fired) {
    uint32_t spc = p.col >> 1, spr = p.row >> 2, bit = 4 * (p.col & 1) + (p.row & 3);
    keys.push_back(((uint64_t)p.sensor << 32) | ((uint64_t)spc << 14) | ((uint64_t)spr << 8) | bit);
  }
  std::sort(keys.begin(), keys.end());
  std::vector<std::vector<uint32_t>> banks(c.n_sensors);
  for (size_t i = 0; i < keys.size();) {
    uint64_t addr = keys[i] >> 8;
    uint32_t hitmap = 0;
    while (i < keys.size() && (keys[i] >> 8) == addr) { hitmap |= 1u << (keys[i] & 0xFF); ++i; }
    uint32_t sensor = (uint32_t)(addr >> 24);
    uint32_t word = ((uint32_t)(addr & 0xFFFFFF) << 8) | hitmap;  // bits 22:14 sp_col, 13:8 sp_row, 7:0 hitmap
    banks[sensor].push_back(word);
  }
  if (c.shuffle_sp) {
    for (auto& b : banks)
      for (size_t i = b.size(); i > 1; --i) std::swap(b[i - 1], b[rng.below((uint32_t)i)]);
  }
  uint32_t n_sp = 0;
  for (auto& b : banks) n_sp += (uint32_t)b.size();
  std::vector<uint32_t> words;
  words.push_back(0x56454C4Fu);
  words.push_back(c.n_sensors);
  words.push_back(n_sp);
  words.push_back(0);
  uint32_t off = 0;
  for (uint32_t s = 0; s < c.n_sensors; ++s) { words.push_back(off); off += (uint32_t)banks[s].size(); }
  words.push_back(off);
  while (words.size() % 4) words.push_back(0);
  for (auto& b : banks) words.insert(words.end(), b.begin(), b.end());
  while (words.size() % 4) words.push_back(0);
  size_t pos = g.raw.size();
  g.raw.resize(pos + words.size() * 4);
  std::memcpy(g.raw.data() + pos, words.data(), words.size() * 4);
  g.event_offsets.push_back((uint32_t)g.raw.size());
}

}  // namespace

extern "C" {

// geometry arrays: sensors[n_sensors][7] = ox, oy, ecx, ecy, erx, ery, z (doubles); sensor_module[n_sensors].
void* velo_gen_run(const Config* cfg, const double* sensors, const uint16_t* sensor_module) {
  Gen* g = new Gen();
  g->cfg = *cfg;
  const Config& c = g->cfg;
  g->sensors.resize(c.n_sensors);
  g->sensor_module.assign(sensor_module, sensor_module + c.n_sensors);
  g->module_z.assign(c.n_modules, 0.0);
  g->module_sensors.resize(c.n_modules);
  for (uint32_t s = 0; s < c.n_sensors; ++s) {
    const double* p = sensors + 7 * s;
    g->sensors[s] = {p[0], p[1], p[2], p[3], p[4], p[5], p[6]};
    g->module_z[sensor_module[s]] = p[6];
    g->module_sensors[sensor_module[s]].push_back(s);
  }
  g->module_order.resize(c.n_modules);
  for (uint32_t m = 0; m < c.n_modules; ++m) g->module_order[m] = m;
  std::stable_sort(g->module_order.begin(), g->module_order.end(),
                   [&](uint32_t a, uint32_t b) { return g->module_z[a] < g->module_z[b]; });
  g->event_offsets.push_back(0);
  for (uint32_t e = 0; e < c.n_events; ++e) generate_event(*g, c.first_event + e, e);
  return g;
}

void velo_gen_free(void* h) { delete (Gen*)h; }

uint64_t velo_gen_size(void* h, int what) {
  Gen* g = (Gen*)h;
  switch (what) {
    case 0: return g->raw.size();
    case 1: return g->event_offsets.size();
    case 2: return g->p_event.size();
    case 3: return g->x_event.size();
    case 4: return g->v_event.size();
  }
  return 0;
}

const void* velo_gen_ptr(void* h, int what) {
  Gen* g = (Gen*)h;
  switch (what) {
    case 0: return g->raw.data();
    case 1: return g->event_offsets.data();
    case 10: return g->p_event.data();
    case 11: return g->p_pv.data();
    case 12: return g->p_displaced.data();
    case 13: return g->p_ox.data();
    case 14: return g->p_oy.data();
    case 15: return g->p_oz.data();
    case 16: return g->p_tx.data();
    case 17: return g->p_ty.data();
    case 18: return g->p_n_crossings.data();
    case 19: return g->p_n_hits.data();
    case 20: return g->x_event.data();
    case 21: return g->x_sensor.data();
    case 22: return g->x_col.data();
    case 23: return g->x_row.data();
    case 24: return g->x_particle.data();
    case 25: return g->x_main.data();
    case 30: return g->v_event.data();
    case 31: return g->v_x.data();
    case 32: return g->v_y.data();
    case 33: return g->v_z.data();
  }
  return nullptr;
}

}  // extern "C"
