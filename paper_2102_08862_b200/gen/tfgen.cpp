// Synthetic TPC time-frame generator (seeded, counter-based RNG, double precision inside,
// fp32 SoA out).  It stands in for the paper's Monte-Carlo time frames (§2:
// "simulated Monte-Carlo time frames converted to raw data"), which are not available.
// Recipe: BASELINE.json configs[0..4] (L7-L11) and SURVEY.md §8(d).
//
// This module serves BOTH the oracle tests and the CUDA path as an input source.  It holds
// none of the tracker's arithmetic: it only draws particles, intersects ideal helices with
// pad rows, smears, drops, adds noise and shuffles.
//
// Build: g++ -O2 -shared -fPIC -pthread -o libtfgen.so tfgen.cpp
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>
#include <atomic>

extern "C" {

struct tfgen_config {
  int32_t n_sectors;       // 1 (configs[0]: both drift sides folded into sector 0) or 36
  int32_t n_rows;          // 152
  double x0_cm;            // 85.0
  double row_pitch_cm;     // 1.07
  double pad_pitch_cm;     // 0.5
  double half_sector_deg;  // 10
  double time_bin_cm;      // 0.516
  double drift_len_cm;     // 250
  double v_drift_cm_us;    // 2.58
  double frame_us;         // 0 -> exactly one collision at t0 = 0
  double rate_khz;         // 50
  int32_t fixed_tracks;    // >0: exactly this many tracks per collision; 0: floor(max_tracks*(1-sqrt(u)))
  int32_t max_tracks;      // 4000
  double sigma_y_cm, sigma_z_cm;
  double dropout;          // probability that a cluster is dropped
  double noise_frac;       // extra uniform clusters = round(noise_frac * n_real)
  double pt_min, pt_mean, pt_cap;  // pT = min(pt_min + Exp(pt_mean), pt_cap)
  double eta_max;          // 0.9
  double zv_sigma_cm;      // 5
  double radius_per_pt;    // 666.7 cm / GeV  (Bz = 0.5 T)
  int32_t max_turns;       // looper cut-off in turns (5)
  int32_t shuffle;         // 1: seeded permutation of the output order
  uint64_t seed;
  int32_t n_threads;       // 0 = hardware concurrency
  int32_t reserved;
};

struct tfgen_track {       // truth table, one row per generated particle
  int32_t collision;
  int32_t charge_sense;    // h = +-1 : sign of d(sin phi_local)/dx
  double t0_us, z_v, phi0, eta, pt;
};

struct tfgen_frame;

}  // extern "C"

namespace {

constexpr double kPi = 3.14159265358979323846;

inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// Counter-based stream: value i of stream (seed, a, b, purpose) is a pure function of those.
struct Stream {
  uint64_t key, ctr;
  Stream(uint64_t seed, uint64_t a, uint64_t b, uint64_t purpose) : ctr(0) {
    uint64_t k = mix64(seed ^ 0xA5A5A5A55A5A5A5Aull);
    k = mix64(k + a * 0xD1B54A32D192ED03ull);
    k = mix64(k + b * 0x8CB92BA72F3D8DD7ull);
    key = mix64(k + purpose * 0xDB4F0B9175AE2165ull);
  }
  uint64_t u64() { return mix64(key + (ctr++) * 0x9E3779B97F4A7C15ull); }
  double uniform() { return (double)(u64() >> 11) * (1.0 / 9007199254740992.0); }  // [0,1)
  double uniform_open() { return ((double)(u64() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }  // (0,1)
  double gauss() {  // Box-Muller, one value per two draws
    double u1 = uniform_open(), u2 = uniform();
    return std::sqrt(-2.0 * std::log(u1)) * std::cos(2.0 * kPi * u2);
  }
  double expo(double mean) { return -mean * std::log(uniform_open()); }
};

struct Cluster {
  float row, pad, time, charge;
  int32_t truth_track;   // global particle index, -1 = noise
  int16_t truth_arc;     // 2*turn + (returning ? 1 : 0)
};

struct Collision {
  double t0_us, z_v;
  int32_t n_tracks;
  int64_t first_track;
};

// Seeded bijection of [0, n): 4-round Feistel network on 2*half bits with cycle walking.
struct Permutation {
  uint64_t n; int half; uint64_t mask; uint64_t keys[4];
  Permutation(uint64_t n_, uint64_t seed) : n(n_) {
    int bits = 1; while ((1ull << bits) < n) ++bits;
    half = (bits + 1) / 2; if (half < 1) half = 1;
    mask = (1ull << half) - 1;
    for (int i = 0; i < 4; ++i) keys[i] = mix64(seed + 0x1234567ull * (i + 1));
  }
  uint64_t once(uint64_t v) const {
    uint64_t l = v >> half, r = v & mask;
    for (int i = 0; i < 4; ++i) { uint64_t f = mix64(r ^ keys[i]) & mask; uint64_t nl = r; r = l ^ f; l = nl; }
    return (l << half) | r;
  }
  uint64_t operator()(uint64_t i) const { uint64_t v = once(i); while (v >= n) v = once(v); return v; }
};

}  // namespace

struct tfgen_frame {
  std::vector<float> row, pad, time, charge;
  std::vector<int32_t> truth_track;
  std::vector<int16_t> truth_arc;
  std::vector<tfgen_track> tracks;
  int64_t n_real = 0, n_noise = 0;
  int32_t n_collisions = 0;
  double max_time_bin = 0;
};

namespace {

void gen_collision(const tfgen_config& c, const Collision& col, int32_t icol,
                   const std::vector<double>& xr, const std::vector<int>& npads,
                   std::vector<Cluster>& out, tfgen_track* tracks, double t_max) {
  const int n_phi_sectors = (c.n_sectors == 1) ? 1 : 18;
  const double two_pi = 2.0 * kPi;
  const double half = c.half_sector_deg * kPi / 180.0;
  for (int32_t it = 0; it < col.n_tracks; ++it) {
    Stream s(c.seed, (uint64_t)icol, (uint64_t)it, 2);
    double phi0 = (c.n_sectors == 1) ? (-half + 2.0 * half * s.uniform()) : two_pi * s.uniform();
    double eta = -c.eta_max + 2.0 * c.eta_max * s.uniform();
    int h = (s.uniform() < 0.5) ? -1 : 1;
    double pt = std::min(c.pt_min + s.expo(c.pt_mean), c.pt_cap);
    const int64_t gtrack = col.first_track + it;
    tracks[gtrack] = tfgen_track{icol, h, col.t0_us, col.z_v, phi0, eta, pt};
    const double R = c.radius_per_pt * pt;
    const double sh = std::sinh(eta);
    const double theta_max = two_pi * c.max_turns;
    for (int sec = 0; sec < n_phi_sectors; ++sec) {
      const double alpha = (c.n_sectors == 1) ? 0.0 : (2.0 * half * sec + half);
      const double psi0 = phi0 - alpha;
      const double sp0 = std::sin(psi0), cp0 = std::cos(psi0);
      // v(x) = sp0 + h x / R is linear in x: skip the sector if no row can have |v| <= 1
      const double v_first = sp0 + h * xr.front() / R, v_last = sp0 + h * xr.back() / R;
      if ((v_first > 1.0 && v_last > 1.0) || (v_first < -1.0 && v_last < -1.0)) continue;
      for (int r = 0; r < c.n_rows; ++r) {
        const double v = sp0 + h * xr[r] / R;
        if (!(std::fabs(v) <= 1.0)) continue;
        const double cabs = std::sqrt(1.0 - v * v);
        const double half_width = 0.5 * c.pad_pitch_cm * npads[r];
        for (int ret = 0; ret < 2; ++ret) {
          const double cpsi = ret ? -cabs : cabs;
          const double y = (R / h) * (cp0 - cpsi);
          if (!(std::fabs(y) <= half_width + 1.0)) continue;   // pre-filter before any RNG draw
          const double psi = std::atan2(v, cpsi);
          double theta = std::fmod(h * (psi - psi0), two_pi);
          if (theta < 0) theta += two_pi;
          for (int turn = 0; turn < c.max_turns; ++turn) {
            const double th = theta + two_pi * turn;
            if (th >= theta_max) break;
            const double z = col.z_v + R * th * sh;
            if (!(std::fabs(z) < c.drift_len_cm)) break;       // particle left the drift volume
            // one fixed block of draws per candidate crossing -> reproducible streams
            const double gy = s.gauss(), gz = s.gauss(), ud = s.uniform(), uq = s.uniform();
            if (ud < c.dropout) continue;
            const double ys = y + c.sigma_y_cm * gy;
            const double padf = ys / c.pad_pitch_cm + 0.5 * (npads[r] - 1);
            if (!(padf >= -0.5 && padf < npads[r] - 0.5)) continue;
            // the tracker tests the fp32 values: a pad that rounds up onto the row's edge is outside the row
            if (!((float)padf >= -0.5f && (float)padf < (float)npads[r] - 0.5f)) continue;
            const double drift = c.drift_len_cm - std::fabs(z) + c.sigma_z_cm * gz;
            const double tb = (col.t0_us * c.v_drift_cm_us + drift) / c.time_bin_cm;
            if (!(tb >= 0.0 && (float)tb <= (float)t_max)) continue;      // beyond the frame's last time bin (> 4 sigma): not read out
            const int sector = (c.n_sectors == 1) ? 0 : (z >= 0 ? sec : 18 + sec);
            Cluster cl;
            cl.row = (float)(sector * c.n_rows + r);
            cl.pad = (float)padf;
            cl.time = (float)tb;
            cl.charge = (float)(20.0 + 180.0 * uq);
            cl.truth_track = (int32_t)gtrack;
            cl.truth_arc = (int16_t)(2 * turn + ret);
            out.push_back(cl);
          }
        }
      }
    }
  }
}

}  // namespace

extern "C" {

int tfgen_generate(const tfgen_config* cfg, tfgen_frame** out_frame) {
  if (!cfg || !out_frame) return -1;
  const tfgen_config c = *cfg;
  if (c.n_rows <= 0 || (c.n_sectors != 1 && c.n_sectors != 36) || c.max_turns < 1) return -1;
  tfgen_frame* f = new tfgen_frame();

  std::vector<double> xr(c.n_rows);
  std::vector<int> npads(c.n_rows);
  const double tan_half = std::tan(c.half_sector_deg * kPi / 180.0);
  for (int r = 0; r < c.n_rows; ++r) {
    xr[r] = c.x0_cm + c.row_pitch_cm * r;
    npads[r] = (int)std::floor(2.0 * xr[r] * tan_half / c.pad_pitch_cm);
  }

  // collisions: Poisson process = exponential gaps with mean 1/rate
  std::vector<Collision> cols;
  {
    Stream sc(c.seed, 0, 0, 0);
    if (c.frame_us <= 0) {
      cols.push_back(Collision{0.0, 0.0, 0, 0});
    } else {
      const double mean_gap_us = 1000.0 / c.rate_khz;
      double t = sc.expo(mean_gap_us);
      while (t < c.frame_us) { cols.push_back(Collision{t, 0.0, 0, 0}); t += sc.expo(mean_gap_us); }
    }
    int64_t first = 0;
    for (size_t i = 0; i < cols.size(); ++i) {
      Stream s1(c.seed, (uint64_t)i, 0, 1);
      cols[i].z_v = c.zv_sigma_cm * s1.gauss();
      const double u = s1.uniform();
      cols[i].n_tracks = c.fixed_tracks > 0 ? c.fixed_tracks
                                            : (int32_t)std::floor(c.max_tracks * (1.0 - std::sqrt(u)));
      cols[i].first_track = first;
      first += cols[i].n_tracks;
    }
    f->tracks.resize((size_t)first);
  }
  f->n_collisions = (int32_t)cols.size();
  const double t_last = c.frame_us > 0 ? c.frame_us : 0.0;
  f->max_time_bin = (t_last * c.v_drift_cm_us + c.drift_len_cm) / c.time_bin_cm + 4.0 * c.sigma_z_cm / c.time_bin_cm + 1.0;

  // real clusters, collisions in parallel
  int nt = c.n_threads > 0 ? c.n_threads : (int)std::thread::hardware_concurrency();
  if (nt < 1) nt = 1;
  nt = std::min<int>(nt, std::max<size_t>(1, cols.size()));
  std::vector<std::vector<Cluster>> per_col(cols.size());
  {
    std::atomic<size_t> next{0};
    auto work = [&]() {
      for (;;) {
        size_t i = next.fetch_add(1);
        if (i >= cols.size()) break;
        gen_collision(c, cols[i], (int32_t)i, xr, npads, per_col[i], f->tracks.data(), f->max_time_bin);
      }
    };
    std::vector<std::thread> th;
    for (int t = 1; t < nt; ++t) th.emplace_back(work);
    work();
    for (auto& t : th) t.join();
  }
  std::vector<int64_t> col_off(cols.size() + 1, 0);
  for (size_t i = 0; i < cols.size(); ++i) col_off[i + 1] = col_off[i] + (int64_t)per_col[i].size();
  const int64_t n_real = col_off.back();
  const int64_t n_noise = (int64_t)std::llround(c.noise_frac * (double)n_real);
  const int64_t n = n_real + n_noise;
  f->n_real = n_real; f->n_noise = n_noise;

  f->row.resize(n); f->pad.resize(n); f->time.resize(n); f->charge.resize(n);
  f->truth_track.resize(n); f->truth_arc.resize(n);
  Permutation perm((uint64_t)std::max<int64_t>(n, 1), mix64(c.seed ^ 0x5EEDull));
  auto place = [&](int64_t i, const Cluster& cl) {
    const int64_t p = c.shuffle ? (int64_t)perm((uint64_t)i) : i;
    f->row[p] = cl.row; f->pad[p] = cl.pad; f->time[p] = cl.time; f->charge[p] = cl.charge;
    f->truth_track[p] = cl.truth_track; f->truth_arc[p] = cl.truth_arc;
  };
  {
    // scatter real clusters (parallel over collisions) and noise (parallel over blocks of 1<<16)
    const int64_t noise_block = 1 << 16;
    const int64_t n_noise_blocks = (n_noise + noise_block - 1) / noise_block;
    const double t_hi = (t_last * c.v_drift_cm_us + c.drift_len_cm) / c.time_bin_cm;
    std::atomic<int64_t> next{0};
    const int64_t n_items = (int64_t)cols.size() + n_noise_blocks;
    auto work = [&]() {
      for (;;) {
        int64_t it = next.fetch_add(1);
        if (it >= n_items) break;
        if (it < (int64_t)cols.size()) {
          const auto& v = per_col[it];
          for (size_t k = 0; k < v.size(); ++k) place(col_off[it] + (int64_t)k, v[k]);
          std::vector<Cluster>().swap(per_col[it]);
        } else {
          const int64_t b = it - (int64_t)cols.size();
          const int64_t lo = b * noise_block, hi = std::min(n_noise, lo + noise_block);
          for (int64_t k = lo; k < hi; ++k) {
            Stream s(c.seed, (uint64_t)k, 0, 3);
            const int sr = (int)(s.uniform() * (c.n_sectors * c.n_rows));
            const int r = sr % c.n_rows;
            Cluster cl;
            cl.row = (float)sr;
            cl.pad = (float)(-0.5 + npads[r] * s.uniform());
            if (!(cl.pad < npads[r] - 0.5f)) cl.pad = (float)(npads[r] - 1);
            cl.time = (float)(t_hi * s.uniform());
            cl.charge = (float)(20.0 + 180.0 * s.uniform());
            cl.truth_track = -1; cl.truth_arc = 0;
            place(n_real + k, cl);
          }
        }
      }
    };
    int nt2 = c.n_threads > 0 ? c.n_threads : (int)std::thread::hardware_concurrency();
    if (nt2 < 1) nt2 = 1;
    std::vector<std::thread> th;
    for (int t = 1; t < nt2; ++t) th.emplace_back(work);
    work();
    for (auto& t : th) t.join();
  }
  *out_frame = f;
  return 0;
}

int64_t tfgen_n_clusters(const tfgen_frame* f) { return f ? (int64_t)f->row.size() : -1; }
int64_t tfgen_n_real(const tfgen_frame* f) { return f ? f->n_real : -1; }
int64_t tfgen_n_tracks(const tfgen_frame* f) { return f ? (int64_t)f->tracks.size() : -1; }
int32_t tfgen_n_collisions(const tfgen_frame* f) { return f ? f->n_collisions : -1; }
double tfgen_max_time_bin(const tfgen_frame* f) { return f ? f->max_time_bin : -1; }

// Copies into caller-owned host arrays (any pointer may be NULL to skip it).
int tfgen_copy(const tfgen_frame* f, float* row, float* pad, float* time, float* charge,
               int32_t* truth_track, int16_t* truth_arc, tfgen_track* tracks) {
  if (!f) return -1;
  const size_t n = f->row.size();
  if (row) std::memcpy(row, f->row.data(), n * sizeof(float));
  if (pad) std::memcpy(pad, f->pad.data(), n * sizeof(float));
  if (time) std::memcpy(time, f->time.data(), n * sizeof(float));
  if (charge) std::memcpy(charge, f->charge.data(), n * sizeof(float));
  if (truth_track) std::memcpy(truth_track, f->truth_track.data(), n * sizeof(int32_t));
  if (truth_arc) std::memcpy(truth_arc, f->truth_arc.data(), n * sizeof(int16_t));
  if (tracks) std::memcpy(tracks, f->tracks.data(), f->tracks.size() * sizeof(tfgen_track));
  return 0;
}

void tfgen_free(tfgen_frame* f) { delete f; }


// ---- digitisation: clusters -> zero-suppressed ADC samples (input of the cluster finder) ----
// Stands in for "simulated Monte-Carlo time frames converted to raw data" one step earlier in the chain.
// Every cluster (sector_row, pad, time, charge) deposits its charge on the 3 x 3 cells around (round(pad), round(time))
// of its sector-row with separable weights = the integral of a Gaussian (sigma_pad, sigma_time, in cells) over each cell;
// deposits that fall on the same cell add up; ADC = floor(sum); cells below `threshold` are suppressed (zero suppression in
// the readout).  Output: samples sorted by (sector_row, time bin, pad), no duplicates -- the readout order the
// cluster finder's input contract names.  Holds none of the cluster finder's arithmetic.
struct tfgen_digits {
  std::vector<int32_t> row, pad, time;
  std::vector<float> adc;
};

int tfgen_digitize(int64_t n, const float* row, const float* pad, const float* time, const float* charge, int32_t n_sector_rows,
                   int32_t n_rows, const int32_t* n_pads_of_row, int32_t max_time_bin, double sigma_pad, double sigma_time,
                   int32_t threshold, int32_t n_threads, tfgen_digits** out) {
  if (!out || n < 0 || n_sector_rows < 1 || n_rows < 1 || !n_pads_of_row || !(sigma_pad > 0) || !(sigma_time > 0)) return -1;
  std::vector<int64_t> start((size_t)n_sector_rows + 1, 0);
  for (int64_t i = 0; i < n; ++i) { const int sr = (int)row[i]; if (sr >= 0 && sr < n_sector_rows) ++start[(size_t)sr + 1]; }
  for (int s = 0; s < n_sector_rows; ++s) start[(size_t)s + 1] += start[(size_t)s];
  std::vector<int64_t> idx((size_t)start[(size_t)n_sector_rows]);
  {
    std::vector<int64_t> fill(start.begin(), start.end() - 1);
    for (int64_t i = 0; i < n; ++i) { const int sr = (int)row[i]; if (sr >= 0 && sr < n_sector_rows) idx[(size_t)fill[(size_t)sr]++] = i; }
  }
  struct Part { std::vector<int32_t> pad, time; std::vector<float> adc; };
  std::vector<Part> parts((size_t)n_sector_rows);
  auto cdf = [](double x) { return 0.5 * std::erfc(-x / std::sqrt(2.0)); };
  std::atomic<int> next(0);
  auto work = [&]() {
    std::vector<std::pair<uint64_t, double>> dep;
    for (;;) {
      const int sr = next.fetch_add(1);
      if (sr >= n_sector_rows) break;
      const int np = n_pads_of_row[sr % n_rows];
      dep.clear();
      for (int64_t q = start[(size_t)sr]; q < start[(size_t)sr + 1]; ++q) {
        const int64_t i = idx[(size_t)q];
        const int p0 = (int)std::floor((double)pad[i] + 0.5), t0 = (int)std::floor((double)time[i] + 0.5);
        const double dp = (double)pad[i] - p0, dt = (double)time[i] - t0;
        double wp[3], wt[3];
        for (int k = -1; k <= 1; ++k) {
          wp[k + 1] = cdf((k + 0.5 - dp) / sigma_pad) - cdf((k - 0.5 - dp) / sigma_pad);
          wt[k + 1] = cdf((k + 0.5 - dt) / sigma_time) - cdf((k - 0.5 - dt) / sigma_time);
        }
        for (int a = -1; a <= 1; ++a)
          for (int b = -1; b <= 1; ++b) {
            const int pp = p0 + b, tt = t0 + a;
            if (pp < 0 || pp >= np || tt < 0 || tt > max_time_bin) continue;
            dep.emplace_back(((uint64_t)(uint32_t)tt << 16) | (uint64_t)(uint32_t)pp, (double)charge[i] * wt[a + 1] * wp[b + 1]);
          }
      }
      std::sort(dep.begin(), dep.end(), [](const std::pair<uint64_t, double>& x, const std::pair<uint64_t, double>& y) { return x.first < y.first; });
      Part& P = parts[(size_t)sr];
      for (size_t a = 0; a < dep.size();) {
        size_t b = a;
        double sum = 0.0;
        while (b < dep.size() && dep[b].first == dep[a].first) sum += dep[b++].second;
        const double adc = std::floor(sum);
        if (adc >= (double)threshold) { P.time.push_back((int32_t)(dep[a].first >> 16)); P.pad.push_back((int32_t)(dep[a].first & 0xFFFF)); P.adc.push_back((float)adc); }
        a = b;
      }
    }
  };
  const int nt = std::max(1, n_threads > 0 ? n_threads : (int)std::thread::hardware_concurrency());
  std::vector<std::thread> th;
  for (int t = 0; t < nt; ++t) th.emplace_back(work);
  for (auto& t : th) t.join();
  tfgen_digits* D = new tfgen_digits();
  size_t total = 0;
  for (const Part& P : parts) total += P.adc.size();
  D->row.reserve(total); D->pad.reserve(total); D->time.reserve(total); D->adc.reserve(total);
  for (int sr = 0; sr < n_sector_rows; ++sr) {
    const Part& P = parts[(size_t)sr];
    D->row.insert(D->row.end(), P.adc.size(), sr);
    D->pad.insert(D->pad.end(), P.pad.begin(), P.pad.end());
    D->time.insert(D->time.end(), P.time.begin(), P.time.end());
    D->adc.insert(D->adc.end(), P.adc.begin(), P.adc.end());
  }
  *out = D;
  return 0;
}
int64_t tfgen_digits_n(const tfgen_digits* d) { return d ? (int64_t)d->adc.size() : -1; }
void tfgen_digits_copy(const tfgen_digits* d, int32_t* row, int32_t* pad, int32_t* time, float* adc) {
  const size_t n = d->adc.size();
  std::memcpy(row, d->row.data(), n * 4); std::memcpy(pad, d->pad.data(), n * 4); std::memcpy(time, d->time.data(), n * 4); std::memcpy(adc, d->adc.data(), n * 4);
}
void tfgen_digits_free(tfgen_digits* d) { delete d; }

}  // extern "C"
