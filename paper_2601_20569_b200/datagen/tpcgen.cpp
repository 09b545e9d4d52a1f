// tpcgen.cpp — seeded synthetic TPC time-frame generator (C ABI, host only).
//
// This module is INPUT GENERATION ONLY.  It is the one piece of code that both the CUDA
// path and the CPU oracle are fed from; it contains none of the tracking method's
// arithmetic (no grid, no links, no Kalman filter, no selection).  It simulates what the
// detector would record: helix trajectories of charged particles in a uniform solenoid
// field crossing the pad-row planes of the 36 TPC sectors, smeared, with a
// hit efficiency, noise clusters, overlapping collisions at random times shifting z by the
// drift velocity (continuous readout) and, for the 2.8 ms frame, a smooth
// space-charge-like distortion.  The five workloads of BASELINE.json are
// presets over the knobs of tpcgen_config (see datagen/__init__.py and DESIGN.md "Input
// recipe").  Real ALICE data is not available; these frames stand in for it.
//
// Random numbers: counter-based (splitmix64 finaliser keyed by seed, event, track, stream,
// counter), so the output does not depend on the number of worker threads.
//
// Output order: clusters grouped by (sector,row) ascending — the order the ALICE
// clusteriser delivers native clusters in — and, inside a row, in generation order
// (event, track, crossing; noise last).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

struct Cluster {  // identical layout to the 16-byte input struct of the C ABI
  float y, z, q;
  uint8_t sector, row;
  uint16_t flags;
};
static_assert(sizeof(Cluster) == 16, "cluster must be 16 bytes");

struct Truth {  // one per generated particle
  int32_t event;
  int32_t charge;
  float pt, phi0, tanl, t_coll_us;
  int32_t n_clusters;  // signal clusters kept, all legs
  int32_t pad;
};
static_assert(sizeof(Truth) == 32, "truth must be 32 bytes");

}  // namespace

extern "C" {

struct tpcgen_config {
  uint64_t seed;
  int32_t n_events;
  int32_t tracks_per_event;
  int32_t n_rows;        // 152
  int32_t row_lo, row_hi;  // clusters only on rows row_lo..row_hi-1
  int32_t single_sector;   // -1: all 36 sectors; else only this sector and azimuth inside it
  float r_min, r_max;      // 85, 245
  float half_angle_deg;    // 10
  float z_max;             // 250
  float bz_tesla;          // 0.5
  float pt_mean, pt_lo, pt_hi;  // exponential law, clipped by rejection
  int32_t pt_uniform;      // 1: pT uniform in [pt_lo, pt_hi] instead
  float eta_max;           // 0.9
  float looper_frac;       // fraction of tracks redrawn with pT uniform in [looper_lo, looper_hi]
  float looper_lo, looper_hi;
  float smear_y, smear_z;  // gaussian sigma, cm
  float p_hit;             // probability that a crossing leaves a cluster
  float noise_frac;        // noise clusters as a fraction of the signal clusters
  int32_t noise_inner_peaked;  // 1: noise row weight ~ (r_min/x_r)^2
  float t_window_us;       // collision times uniform in [0, t_window_us]
  float v_drift;           // cm/us
  int32_t distortion;      // 1: radial shift dist_r*(r_min/x_r)^2, azimuthal dist_y*(r_min/x_r)^2
  float dist_r, dist_y;    // 8, 1 cm
  int32_t n_threads;       // 0 = hardware concurrency
  int32_t max_turns;       // 3
};

struct tpcgen_result {
  std::vector<Cluster> clusters;
  std::vector<int32_t> labels;  // particle*8 + leg, -1 = noise
  std::vector<Truth> truth;
};

}  // extern "C"

namespace {

inline uint64_t mix64(uint64_t x) {
  x += 0x9E3779B97F4A7C15ull;
  x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
  x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
  return x ^ (x >> 31);
}

struct Rng {  // counter-based stream
  uint64_t key;
  uint64_t ctr;
  Rng(uint64_t seed, uint64_t a, uint64_t b, uint64_t c) {
    key = mix64(seed ^ mix64(a + 0x1234567ull) ^ mix64(mix64(b) + 0x89ABCDEFull) ^ mix64(mix64(mix64(c)) + 77ull));
    ctr = 0;
  }
  uint64_t next() { return mix64(key + 0x632BE59BD9B4E019ull * (++ctr)); }
  double uniform() { return ((next() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }  // (0,1)
  double gauss() {
    double u1 = uniform(), u2 = uniform();
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586 * u2);
  }
};

struct Raw {
  Cluster c;
  int32_t label;
};

struct Geo {
  int n_rows;
  std::vector<double> x, ymax;
  double alpha[18];
  double cosA[18], sinA[18];
  double tanHalf;
  double r_exit;  // radius beyond which a particle has left the TPC
};

Geo make_geo(const tpcgen_config& cfg) {
  Geo g;
  g.n_rows = cfg.n_rows;
  g.x.resize(cfg.n_rows);
  g.ymax.resize(cfg.n_rows);
  const double deg = 3.14159265358979323846 / 180.0;
  g.tanHalf = std::tan(cfg.half_angle_deg * deg);
  for (int r = 0; r < cfg.n_rows; ++r) {
    g.x[r] = cfg.r_min + r * (double(cfg.r_max) - cfg.r_min) / (cfg.n_rows - 1);
    g.ymax[r] = g.x[r] * g.tanHalf;
  }
  for (int s = 0; s < 18; ++s) {
    g.alpha[s] = (s + 0.5) * 2.0 * cfg.half_angle_deg * deg;
    g.cosA[s] = std::cos(g.alpha[s]);
    g.sinA[s] = std::sin(g.alpha[s]);
  }
  g.r_exit = cfg.r_max / std::cos(cfg.half_angle_deg * deg) + 1.0;
  return g;
}

// Generate all clusters of one particle.  Helix from the origin:
//   direction angle phi(psi) = phi0 - q*psi, psi >= 0 the turning angle, R = pT/(0.3*B)
//   X = q R (sin phi0 - sin(phi0 - q psi)),  Y = q R (cos(phi0 - q psi) - cos phi0),
//   Z = tanl * R * psi.
// (positive charge bends towards -y when moving along +x with B along +z.)
void gen_particle(const tpcgen_config& cfg, const Geo& g, int ev, int tr, int pid, double t_coll,
                  std::vector<Raw>& out, Truth& truth) {
  Rng rng(cfg.seed, 1, (uint64_t)ev, (uint64_t)tr);
  const double PI = 3.14159265358979323846;
  const double deg = PI / 180.0;
  double phi0;
  if (cfg.single_sector >= 0) {
    double a0 = g.alpha[cfg.single_sector % 18];
    phi0 = a0 + (2.0 * rng.uniform() - 1.0) * cfg.half_angle_deg * deg;
  } else {
    phi0 = 2.0 * PI * rng.uniform();
  }
  double eta = (2.0 * rng.uniform() - 1.0) * cfg.eta_max;
  double tanl = std::sinh(eta);
  if (cfg.single_sector >= 0) tanl = std::fabs(tanl);  // keep the whole sample on one drift side
  int q = rng.uniform() < 0.5 ? 1 : -1;
  double pt;
  bool looper = rng.uniform() < cfg.looper_frac;
  if (looper) {
    pt = cfg.looper_lo + rng.uniform() * (cfg.looper_hi - cfg.looper_lo);
  } else if (cfg.pt_uniform) {
    pt = cfg.pt_lo + rng.uniform() * (cfg.pt_hi - cfg.pt_lo);
  } else {
    do {
      pt = -cfg.pt_mean * std::log(rng.uniform());
    } while (pt < cfg.pt_lo || pt > cfg.pt_hi);
  }
  truth.event = ev;
  truth.charge = q;
  truth.pt = (float)pt;
  truth.phi0 = (float)phi0;
  truth.tanl = (float)tanl;
  truth.t_coll_us = (float)t_coll;
  truth.n_clusters = 0;
  truth.pad = 0;

  const double R = pt / (0.00299792458 * cfg.bz_tesla);
  const double Xc = q * R * std::sin(phi0), Yc = -q * R * std::cos(phi0);
  // side: A (sectors 0..17) for z>0, C (18..35) for z<0; tanl==0 -> A
  const int side = tanl >= 0 ? 0 : 1;
  const double zsign = side == 0 ? 1.0 : -1.0;
  const double zshift = -zsign * cfg.v_drift * t_coll;  // z_in = z_true - side*v*t
  // maximal turning angle: leaves the drift volume in z, exits radially, or max_turns
  double psi_max = 2.0 * PI * cfg.max_turns;
  if (std::fabs(tanl) > 1e-12) psi_max = std::min(psi_max, cfg.z_max / (std::fabs(tanl) * R));
  if (2.0 * R > g.r_exit) psi_max = std::min(psi_max, 2.0 * std::asin(g.r_exit / (2.0 * R)));

  // angular position on the circle at psi=0 (the origin seen from the centre)
  // and sector pruning by the azimuth interval the trajectory sweeps.
  for (int s = 0; s < 18; ++s) {
    if (cfg.single_sector >= 0 && s != cfg.single_sector % 18) continue;
    // circle centre in the sector frame
    const double cx = Xc * g.cosA[s] + Yc * g.sinA[s];
    const double cy = -Xc * g.sinA[s] + Yc * g.cosA[s];
    // bounding-box rejection
    if (cx + R < g.x[0] || cx - R > g.x[g.n_rows - 1] + cfg.dist_r + 1) continue;
    if (cy - R > g.ymax[g.n_rows - 1] + 2 || cy + R < -g.ymax[g.n_rows - 1] - 2) continue;
    const double theta0 = std::atan2(-cy, -cx);  // origin = centre + R(cos theta0, sin theta0)
    const int sector = cfg.single_sector >= 0 ? cfg.single_sector : side * 18 + s;
    for (int r = cfg.row_lo; r < cfg.row_hi; ++r) {
      double xs = g.x[r];
      double scale = (cfg.r_min / g.x[r]) * (cfg.r_min / g.x[r]);
      if (cfg.distortion) xs += cfg.dist_r * scale;  // sample the helix further out
      double u = (xs - cx) / R;
      if (u < -1.0 || u > 1.0) continue;
      double th = std::acos(u);
      for (int sol = 0; sol < 2; ++sol) {
        double theta = sol == 0 ? th : -th;
        double yl = cy + R * std::sin(theta);
        if (std::fabs(yl) > g.ymax[r]) continue;
        // psi = q*(theta0 - theta) mod 2pi
        double psi = q * (theta0 - theta);
        psi -= 2.0 * PI * std::floor(psi / (2.0 * PI));
        for (int turn = 0; turn < cfg.max_turns; ++turn) {
          double ps = psi + 2.0 * PI * turn;
          if (ps > psi_max) break;
          int leg = (int)std::floor(ps / PI);
          // stable per-crossing random stream
          Rng cr(cfg.seed, 2 + (uint64_t)sol + 2 * (uint64_t)turn, ((uint64_t)ev << 32) | (uint32_t)tr,
                 ((uint64_t)sector << 16) | (uint64_t)r);
          if (cr.uniform() >= cfg.p_hit) continue;
          double yy = yl, zz = tanl * R * ps + zshift;
          if (cfg.distortion) yy += cfg.dist_y * scale;
          yy += cfg.smear_y * cr.gauss();
          zz += cfg.smear_z * cr.gauss();
          Raw raw;
          raw.c.y = (float)yy;
          raw.c.z = (float)zz;
          raw.c.q = (float)(-std::log(cr.uniform()));
          raw.c.sector = (uint8_t)sector;
          raw.c.row = (uint8_t)r;
          raw.c.flags = 0;
          raw.label = pid * 8 + std::min(leg, 7);
          out.push_back(raw);
          truth.n_clusters++;
        }
      }
    }
  }
}

}  // namespace

extern "C" {

tpcgen_result* tpcgen_run(const tpcgen_config* cfgp) {
  const tpcgen_config cfg = *cfgp;
  Geo g = make_geo(cfg);
  int nthr = cfg.n_threads > 0 ? cfg.n_threads : (int)std::thread::hardware_concurrency();
  if (nthr < 1) nthr = 1;
  const int64_t n_part = (int64_t)cfg.n_events * cfg.tracks_per_event;
  auto* res = new tpcgen_result();
  res->truth.resize(n_part);

  // collision times
  std::vector<double> t_coll(cfg.n_events);
  for (int ev = 0; ev < cfg.n_events; ++ev) {
    Rng r(cfg.seed, 0, (uint64_t)ev, 0);
    t_coll[ev] = cfg.t_window_us > 0 ? r.uniform() * cfg.t_window_us : 0.0;
  }

  // particles in fixed-size chunks so the result is independent of the thread count
  const int64_t chunk = 256;
  const int64_t n_chunks = (n_part + chunk - 1) / chunk;
  std::vector<std::vector<Raw>> parts(n_chunks);
  {
    std::vector<std::thread> thr;
    for (int t = 0; t < nthr; ++t) {
      thr.emplace_back([&, t]() {
        for (int64_t c = t; c < n_chunks; c += nthr) {
          auto& v = parts[c];
          int64_t lo = c * chunk, hi = std::min(n_part, lo + chunk);
          for (int64_t p = lo; p < hi; ++p) {
            int ev = (int)(p / cfg.tracks_per_event), tr = (int)(p % cfg.tracks_per_event);
            gen_particle(cfg, g, ev, tr, (int)p, t_coll[ev], v, res->truth[p]);
          }
        }
      });
    }
    for (auto& th : thr) th.join();
  }
  int64_t n_sig = 0;
  for (auto& v : parts) n_sig += (int64_t)v.size();

  // noise
  const int n_sec = 36;
  const int64_t n_noise = (int64_t)std::llround(cfg.noise_frac * (double)n_sig);
  std::vector<Raw> noise(n_noise);
  {
    // cumulative row weights
    std::vector<double> cum(cfg.row_hi - cfg.row_lo);
    double acc = 0;
    for (int r = cfg.row_lo; r < cfg.row_hi; ++r) {
      double w = cfg.noise_inner_peaked ? (cfg.r_min / g.x[r]) * (cfg.r_min / g.x[r]) : 1.0;
      acc += w;
      cum[r - cfg.row_lo] = acc;
    }
    const double zext = cfg.v_drift * cfg.t_window_us;  // extra z extent from event times
    std::vector<std::thread> thr;
    for (int t = 0; t < nthr; ++t) {
      thr.emplace_back([&, t]() {
        for (int64_t i = t; i < n_noise; i += nthr) {
          Rng r(cfg.seed, 3, (uint64_t)i, 0);
          int sector = cfg.single_sector >= 0 ? cfg.single_sector : (int)(r.uniform() * n_sec);
          if (sector >= n_sec) sector = n_sec - 1;
          double u = r.uniform() * acc;
          int row = (int)(std::lower_bound(cum.begin(), cum.end(), u) - cum.begin()) + cfg.row_lo;
          if (row >= cfg.row_hi) row = cfg.row_hi - 1;
          double y = (2.0 * r.uniform() - 1.0) * g.ymax[row];
          // A side: z_in in [-zext, z_max]; C side mirrored
          double zz = -zext + r.uniform() * (cfg.z_max + zext);
          if (sector >= 18) zz = -zz;
          Raw raw;
          raw.c.y = (float)y;
          raw.c.z = (float)zz;
          raw.c.q = (float)(-std::log(r.uniform()));
          raw.c.sector = (uint8_t)sector;
          raw.c.row = (uint8_t)row;
          raw.c.flags = 0;
          raw.label = -1;
          noise[i] = raw;
        }
      });
    }
    for (auto& th : thr) th.join();
  }

  // stable counting sort by (sector,row)
  const int n_sr = n_sec * cfg.n_rows;
  std::vector<int64_t> cnt(n_sr + 1, 0);
  for (auto& v : parts)
    for (auto& r : v) cnt[(int)r.c.sector * cfg.n_rows + r.c.row + 1]++;
  for (auto& r : noise) cnt[(int)r.c.sector * cfg.n_rows + r.c.row + 1]++;
  for (int i = 0; i < n_sr; ++i) cnt[i + 1] += cnt[i];
  const int64_t n_tot = cnt[n_sr];
  res->clusters.resize(n_tot);
  res->labels.resize(n_tot);
  std::vector<int64_t> cur(cnt.begin(), cnt.end() - 1);
  for (auto& v : parts) {
    for (auto& r : v) {
      int64_t pos = cur[(int)r.c.sector * cfg.n_rows + r.c.row]++;
      res->clusters[pos] = r.c;
      res->labels[pos] = r.label;
    }
    std::vector<Raw>().swap(v);
  }
  for (auto& r : noise) {
    int64_t pos = cur[(int)r.c.sector * cfg.n_rows + r.c.row]++;
    res->clusters[pos] = r.c;
    res->labels[pos] = r.label;
  }
  return res;
}

int64_t tpcgen_n_clusters(const tpcgen_result* r) { return (int64_t)r->clusters.size(); }
int64_t tpcgen_n_particles(const tpcgen_result* r) { return (int64_t)r->truth.size(); }

// Copy the result into caller buffers (any may be NULL).
void tpcgen_fetch(const tpcgen_result* r, void* clusters, int32_t* labels, void* truth) {
  if (clusters) std::memcpy(clusters, r->clusters.data(), r->clusters.size() * sizeof(Cluster));
  if (labels) std::memcpy(labels, r->labels.data(), r->labels.size() * sizeof(int32_t));
  if (truth) std::memcpy(truth, r->truth.data(), r->truth.size() * sizeof(Truth));
}

void tpcgen_free(tpcgen_result* r) { delete r; }

}  // extern "C"
