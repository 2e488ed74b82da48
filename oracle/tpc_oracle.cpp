// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded C++ fp32 CPU implementation of
// TPC sector tracking of a continuous-readout time frame: cellular-automaton seeding in native
// (pad row, pad, time) coordinates followed by Kalman-filter track following.
//
// What it follows:
//   * PAPER.md L23 (§1): "the track seeding operates using the time as coordinate instead of the
//     spatial z coordinate"  -> z is only ever a difference of raw time values times the bin size.
//   * PAPER.md L25 (§1): tracker derived from the Run 2 HLT TPC tracker, time frame processed as a whole.
//   * BASELINE.json L5 (north_star): the five steps (ingest, neighbours finder, neighbours cleaner +
//     start-hit finder, tracklet constructor, tracklet selector), fp32, lowest-index tie-breaking.
//   * BASELINE.json L7: the cuts (windows 0.05*dx+0.5 cm, chi2 cut 9, miss limit 10, >= 30 unshared hits).
//   * SURVEY.md §8(c) C1..C6 / DESIGN.md "Readings": every point on which those sources are silent.
// The paper gives no algorithm listing, so this is a HEURISTIC followed step by step; there is no
// closed-form result.  Every fp32 statement below is one rounded operation sequence evaluated left to
// right as written; build with -O2 -ffp-contract=off (no FMA contraction, no fast-math).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// this.  It shares no code, header, table or constant generator with the CUDA path.
//
// Pins (tests/test_oracle_*.py): G1 geometry closed forms; N1 brute force == time-window search;
// N2 noise-free straight track links; N3 reciprocity; K1 transport round trip / composition / exact
// circle; K2 arc-length series vs asin; K3 KF == weighted least-squares line; K4 noise-free helix
// end to end; S1 selector == sort-by-key first-come-first-served; E1 efficiency >= 95 % (pT > 0.2).
// Also holds C8 (orc_refit_chains, further down: refit of the chains linked by the C7 oracle tpc_merge_oracle.cpp), pinned by
// tests/test_refit_oracle_pins.py: F-J rotation Jacobian vs numerical derivative, F-H noise-free helices, F-N resolution and
// pull width against generator truth, F-I bookkeeping.
// Also holds C11 (orc_compress_tracks, pins Q-* in tests/test_compress_oracle_pins.py) and C12 (orc_refit_full: full 5x5
// covariance, multiple scattering, energy loss; pins FF-* in tests/test_fullfit_oracle_pins.py).
// Parity unpinned (no external truth exists): absolute fitted values on noisy data.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

extern "C" {

struct orc_geometry {
  int32_t n_sectors, n_rows;
  float x0_cm, row_pitch_cm, pad_pitch_cm, tan_half_sector, time_bin_cm, drift_len_cm, max_time_bin;
};

struct orc_params {
  float win_slope, win_const, chi2_cut;
  int32_t miss_limit, min_hits;
  float sigma_y_cm, sigma_z_cm, slope_y_max, slope_z_max;
  int32_t seed_min_hits;
  float sin_phi_max, inv_R_per_qpt;
  float c0_y2, c0_s2, c0_k2, c0_z2, c0_t2;
  int32_t brute_force;   // 1: neighbour / window searches scan whole rows (pin N1)
};

}  // extern "C"

namespace {

struct Derived {   // constants derived in double from the fp32 parameter values, rounded once
  float W1, Ay, Az, wy, wz, ry, rz, Z, P, cB;
  std::vector<float> xr, cr;      // row x, pad centre c_r = 0.5*(n_pads_r - 1)
  std::vector<int32_t> npads;
};

Derived derive(const orc_geometry& g, const orc_params& p) {
  Derived d;
  const double pitch = (double)g.row_pitch_cm;
  const double w1 = (double)p.win_slope * pitch + (double)p.win_const;
  d.W1 = (float)w1;
  d.Ay = (float)((double)p.slope_y_max * pitch + w1);
  d.Az = (float)((double)p.slope_z_max * pitch + w1);
  const double sy2 = (double)p.sigma_y_cm * (double)p.sigma_y_cm;
  const double sz2 = (double)p.sigma_z_cm * (double)p.sigma_z_cm;
  d.wy = (float)(1.0 / (6.0 * sy2));
  d.wz = (float)(1.0 / (6.0 * sz2));
  d.ry = (float)sy2;
  d.rz = (float)sz2;
  d.Z = g.time_bin_cm;
  d.P = g.pad_pitch_cm;
  d.cB = p.inv_R_per_qpt;
  d.xr.resize(g.n_rows); d.cr.resize(g.n_rows); d.npads.resize(g.n_rows);
  for (int r = 0; r < g.n_rows; ++r) {
    const double x = (double)g.x0_cm + pitch * (double)r;
    d.xr[r] = (float)x;
    d.npads[r] = (int32_t)std::floor(2.0 * x * (double)g.tan_half_sector / (double)g.pad_pitch_cm);
    d.cr[r] = (float)(0.5 * (double)(d.npads[r] - 1));
  }
  return d;
}

struct State {       // C5: (x; y, z, s = sin phi, t = dz/ds, k = q/pT), block covariance
  float x, y, z, s, t, k;
  float c0, c1, c2, c3, c4, c5;   // (yy, ys, ss, yk, sk, kk)
  float d0, d1, d2;               // (zz, zt, tt)
};

// C5 transport: exact circle in the local x-y plane.  Returns false (state unchanged) on FAIL.
bool transport(State& S, float xn, float cB, float sin_phi_max) {
  const float dx = xn - S.x;
  const float kc = cB * S.k;
  const float sn = S.s + kc * dx;
  if (!(std::fabs(S.s) < sin_phi_max && std::fabs(sn) < sin_phi_max)) return false;   // A12: at BOTH ends (an update may have pushed s past the limit)
  const float c = std::sqrt(1.0f - S.s * S.s);
  const float cn = std::sqrt(1.0f - sn * sn);
  const float ss = S.s + sn;
  const float cc = c + cn;
  const float icc = 1.0f / cc;
  const float T = ss * icc;
  const float q = 1.0f + T * T;
  const float rq = std::sqrt(q);
  const float u = kc * dx;
  const float a = (u * u) * q;
  const float dS = (dx * rq) * (1.0f + a * (0.041666668f + a * (0.0046875f + a * 0.00069754466f)));
  const float g0 = (1.0f + T * (S.s / c)) * icc;
  const float g1 = (1.0f + T * (sn / cn)) * icc;
  const float fa = dx * (g0 + g1);
  const float e = cB * dx;
  const float fb = (dx * g1) * e;
  S.y = S.y + dx * T;
  S.z = S.z + S.t * dS;
  S.s = sn;
  S.x = xn;
  const float h3 = S.c3 + fa * S.c4 + fb * S.c5;
  const float h4 = S.c4 + e * S.c5;
  const float h1 = S.c1 + fa * S.c2 + fb * S.c4;
  S.c0 = S.c0 + fa * S.c1 + fb * S.c3 + fa * h1 + fb * h3;
  S.c1 = h1 + e * h3;
  S.c2 = S.c2 + e * S.c4 + e * h4;
  S.c3 = h3;
  S.c4 = h4;
  const float n1 = S.d1 + dS * S.d2;
  S.d0 = S.d0 + dS * S.d1 + dS * n1;
  S.d1 = n1;
  return true;
}

// C5 update with a measurement (ym, zm) of variances (ry, rz).
void update(State& S, float ym, float zm, float ry, float rz) {
  const float wy = 1.0f / (S.c0 + ry);
  const float resy = ym - S.y;
  const float k0 = S.c0 * wy, k1 = S.c1 * wy, k3 = S.c3 * wy;
  S.y += k0 * resy;
  S.s += k1 * resy;
  S.k += k3 * resy;
  S.c5 -= k3 * S.c3;
  S.c4 -= k1 * S.c3;
  S.c2 -= k1 * S.c1;
  S.c3 -= k0 * S.c3;
  S.c1 -= k0 * S.c1;
  S.c0 -= k0 * S.c0;
  const float wz = 1.0f / (S.d0 + rz);
  const float resz = zm - S.z;
  const float j0 = S.d0 * wz, j1 = S.d1 * wz;
  S.z += j0 * resz;
  S.t += j1 * resz;
  S.d2 -= j1 * S.d1;
  S.d1 -= j0 * S.d1;
  S.d0 -= j0 * S.d0;
}

struct Tracklet {
  int32_t seed;                 // original index of the start hit == tracklet id
  int32_t n_hits, first_row, last_row;
  std::vector<int32_t> row_hit; // [n_rows], original indices, -1 = none
  State snap;                   // state after the last update (innermost hit)
  float time_ref;
};

struct Track {
  int32_t seed, sector, first_row, last_row, n_hits;
  int64_t hit_offset;
  State snap;
  float time_ref;
};

}  // namespace

struct orc_result {
  int64_t n = 0;
  int32_t n_rows = 0;
  std::vector<int32_t> up_raw, down_raw, up, down;
  std::vector<uint8_t> is_start;
  std::vector<Tracklet> tracklets;
  std::vector<Track> tracks;
  std::vector<int32_t> track_hits;
  double stats[16] = {0};
  // [0..4] seconds: ingest, finder, cleaner+start, constructor, selector
  // [5] candidates scanned in finder  [6] pairs tested  [7] transports  [8] searches
  // [9] candidates scanned in searches [10] updates [11] invalid clusters [12] start hits
};

namespace {

struct RowIndex {   // C1: hits grouped by (sector,row); sorted by (time, orig) as an acceleration only
  std::vector<int64_t> start;     // [n_sr + 1]
  std::vector<int32_t> idx;       // original indices
  std::vector<float> t;           // time of idx[i], same order
};

inline double now() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

}  // namespace

extern "C" {

int orc_track(const orc_geometry* gp, const orc_params* pp, const float* row, const float* pad,
              const float* time, int64_t n, orc_result** out) {
  if (!gp || !pp || !out || n < 0 || n >= (int64_t)1 << 31 || (n > 0 && (!row || !pad || !time))) return -1;
  const orc_geometry g = *gp;
  const orc_params p = *pp;
  if (g.n_rows < 3 || g.n_sectors < 1) return -1;
  const Derived D = derive(g, p);
  const int n_rows = g.n_rows;
  const int64_t n_sr = (int64_t)g.n_sectors * n_rows;
  orc_result* R = new orc_result();
  R->n = n; R->n_rows = n_rows;

  // ---------------- C1 ingest ----------------
  double t0 = now();
  std::vector<int32_t> sr(n, -1);     // sector*n_rows + row, -1 = outside the geometry (ignored)
  std::vector<float> y(n, 0.0f);
  RowIndex ri;
  ri.start.assign(n_sr + 1, 0);
  int64_t n_invalid = 0;
  for (int64_t i = 0; i < n; ++i) {
    const float rf = row[i];
    bool ok = rf >= 0.0f && rf < (float)n_sr && rf == std::floor(rf);
    int32_t isr = -1;
    if (ok) {
      isr = (int32_t)rf;
      const int r = isr % n_rows;
      ok = pad[i] >= -0.5f && pad[i] < (float)D.npads[r] - 0.5f && time[i] >= 0.0f && time[i] <= g.max_time_bin;
      if (ok) y[i] = (pad[i] - D.cr[r]) * D.P;
    }
    if (!ok) { ++n_invalid; continue; }
    sr[i] = isr;
    ++ri.start[isr + 1];
  }
  for (int64_t b = 0; b < n_sr; ++b) ri.start[b + 1] += ri.start[b];
  ri.idx.resize(ri.start[n_sr]);
  {
    std::vector<int64_t> fill(ri.start.begin(), ri.start.end() - 1);
    for (int64_t i = 0; i < n; ++i) if (sr[i] >= 0) ri.idx[fill[sr[i]]++] = (int32_t)i;
    for (int64_t b = 0; b < n_sr; ++b)
      std::sort(ri.idx.begin() + ri.start[b], ri.idx.begin() + ri.start[b + 1],
                [&](int32_t a, int32_t c) { return time[a] < time[c] || (time[a] == time[c] && a < c); });
    ri.t.resize(ri.idx.size());
    for (size_t k = 0; k < ri.idx.size(); ++k) ri.t[k] = time[ri.idx[k]];
  }
  R->stats[11] = (double)n_invalid;
  // candidate range of bin b whose time lies in [tc - hw, tc + hw] (a superset is all that is needed)
  auto range = [&](int64_t b, double tc, double hw, int64_t& lo, int64_t& hi) {
    lo = ri.start[b]; hi = ri.start[b + 1];
    if (p.brute_force) return;
    const float* tb = ri.t.data();
    lo = std::lower_bound(tb + lo, tb + hi, (float)(tc - hw - 0.05)) - tb;
    hi = std::upper_bound(tb + lo, tb + hi, (float)(tc + hw + 0.05)) - tb;
  };
  double t1 = now();
  R->stats[0] = t1 - t0;

  // ---------------- C2 neighbours finder ----------------
  R->up_raw.assign(n, -1); R->down_raw.assign(n, -1);
  {
    std::vector<int32_t> U, Dn;
    double n_cand = 0, n_pairs = 0;
    const double tw = (double)D.Az / (double)D.Z;
    for (int64_t h = 0; h < n; ++h) {
      if (sr[h] < 0) continue;
      const int r = sr[h] % n_rows;
      if (r < 1 || r > n_rows - 2) continue;
      const float yh = y[h], th = time[h];
      U.clear(); Dn.clear();
      for (int side = 0; side < 2; ++side) {
        const int64_t b = sr[h] + (side == 0 ? 1 : -1);
        int64_t lo, hi;
        range(b, (double)th, tw, lo, hi);
        n_cand += (double)(hi - lo);
        for (int64_t q = lo; q < hi; ++q) {
          const int32_t c = ri.idx[q];
          const float dy = y[c] - yh;
          const float dz = (time[c] - th) * D.Z;
          if (std::fabs(dy) < D.Ay && std::fabs(dz) < D.Az) (side == 0 ? U : Dn).push_back(c);
        }
      }
      float best = 0.0f; int32_t bu = -1, bd = -1;
      for (int32_t u : U) {
        for (int32_t d : Dn) {
          n_pairs += 1;
          const float ay = y[u] - yh;
          const float by = yh - y[d];
          const float ey = ay - by;
          const float az = (time[u] - th) * D.Z;
          const float bz = (th - time[d]) * D.Z;
          const float ez = az - bz;
          if (!(std::fabs(ey) < D.W1 && std::fabs(ez) < D.W1)) continue;
          const float chi2 = (ey * ey) * D.wy + (ez * ez) * D.wz;
          if (!(chi2 < p.chi2_cut)) continue;
          if (bu < 0 || chi2 < best || (chi2 == best && (u < bu || (u == bu && d < bd)))) {
            best = chi2; bu = u; bd = d;
          }
        }
      }
      R->up_raw[h] = bu; R->down_raw[h] = bd;
    }
    R->stats[5] = n_cand; R->stats[6] = n_pairs;
  }
  double t2 = now();
  R->stats[1] = t2 - t1;

  // ---------------- C3 cleaner, C4 start hits ----------------
  R->up.assign(n, -1); R->down.assign(n, -1); R->is_start.assign(n, 0);
  for (int64_t h = 0; h < n; ++h) {
    const int32_t u = R->up_raw[h], d = R->down_raw[h];
    R->up[h] = (u >= 0 && R->down_raw[u] == (int32_t)h) ? u : -1;
    R->down[h] = (d >= 0 && R->up_raw[d] == (int32_t)h) ? d : -1;
  }
  std::vector<int32_t> start_hits;
  for (int64_t h = 0; h < n; ++h) {
    if (sr[h] < 0 || R->down[h] >= 0) continue;
    int len = 1; int32_t c = (int32_t)h;
    while (len < p.seed_min_hits && R->up[c] >= 0) { c = R->up[c]; ++len; }
    if (len >= p.seed_min_hits) { R->is_start[h] = 1; start_hits.push_back((int32_t)h); }
  }
  R->stats[12] = (double)start_hits.size();
  double t3 = now();
  R->stats[2] = t3 - t2;

  // ---------------- C5 tracklet constructor ----------------
  {
    double n_tr = 0, n_se = 0, n_sc = 0, n_up = 0;
    R->tracklets.reserve(start_hits.size());
    for (int32_t h0 : start_hits) {
      Tracklet T;
      T.seed = h0; T.row_hit.assign(n_rows, -1); T.time_ref = time[h0];
      const int64_t sec_base = (int64_t)(sr[h0] / n_rows) * n_rows;
      const int r0 = sr[h0] % n_rows;
      const float tstart = time[h0];
      const int32_t h1 = R->up[h0];
      const int r1 = sr[h1] % n_rows;
      State S;
      // 1. init from the first two chain hits
      S.x = D.xr[r0]; S.y = y[h0]; S.z = 0.0f;
      {
        const float dxl = D.xr[r1] - D.xr[r0];
        const float dy = y[h1] - y[h0];
        const float dzl = (time[h1] - tstart) * D.Z;
        const float L = std::sqrt(dxl * dxl + dy * dy);
        S.s = dy / L; S.t = dzl / L; S.k = 0.0f;
      }
      S.c0 = D.ry; S.c1 = 0; S.c2 = p.c0_s2; S.c3 = 0; S.c4 = 0; S.c5 = p.c0_k2;
      S.d0 = D.rz; S.d1 = 0; S.d2 = p.c0_t2;
      T.row_hit[r0] = h0;
      float x_last = S.x;
      T.snap = S;
      auto attach = [&](int32_t m, int r) {
        update(S, y[m], (time[m] - tstart) * D.Z, D.ry, D.rz);
        n_up += 1;
        T.row_hit[r] = m; x_last = S.x; T.snap = S;
      };
      auto search = [&](int r) -> int32_t {
        n_se += 1;
        const float w = p.win_slope * std::fabs(D.xr[r] - x_last) + p.win_const;
        int64_t lo, hi;
        range(sec_base + r, (double)tstart + (double)S.z / (double)D.Z, (double)w / (double)D.Z, lo, hi);
        n_sc += (double)(hi - lo);
        int32_t bm = -1; float bdd = 0.0f;
        for (int64_t q = lo; q < hi; ++q) {
          const int32_t m = ri.idx[q];
          const float ey = y[m] - S.y;
          const float ez = (time[m] - tstart) * D.Z - S.z;
          if (!(std::fabs(ey) < w && std::fabs(ez) < w)) continue;
          const float dd = ey * ey + ez * ez;
          if (bm < 0 || dd < bdd || (dd == bdd && m < bm)) { bm = m; bdd = dd; }
        }
        return bm;
      };
      // 2. chain phase (up), no gating
      bool ok = true;
      int r_last = r0;
      for (int32_t c = h1; c >= 0; c = R->up[c]) {
        const int r = sr[c] % n_rows;
        n_tr += 1;
        if (!transport(S, D.xr[r], D.cB, p.sin_phi_max)) { ok = false; break; }
        attach(c, r);
        r_last = r;
      }
      // 3. following (up)
      if (ok) {
        int misses = 0;
        for (int r = r_last + 1; r < n_rows; ++r) {
          n_tr += 1;
          if (!transport(S, D.xr[r], D.cB, p.sin_phi_max)) break;
          const int32_t m = search(r);
          if (m >= 0) { attach(m, r); misses = 0; }
          else if (++misses == p.miss_limit) break;
        }
      }
      // 4. turn round: keep the state, reset the covariance
      S.c0 = p.c0_y2; S.c1 = 0; S.c2 = p.c0_s2; S.c3 = 0; S.c4 = 0; S.c5 = p.c0_k2;
      S.d0 = p.c0_z2; S.d1 = 0; S.d2 = p.c0_t2;
      // 5. down pass
      {
        int r_top = n_rows - 1;
        while (T.row_hit[r_top] < 0) --r_top;
        int misses = 0;
        for (int r = r_top; r >= 0; --r) {
          n_tr += 1;
          if (!transport(S, D.xr[r], D.cB, p.sin_phi_max)) break;
          if (T.row_hit[r] >= 0) attach(T.row_hit[r], r);
          else if (r < r0) {
            const int32_t m = search(r);
            if (m >= 0) { attach(m, r); misses = 0; }
            else if (++misses == p.miss_limit) break;
          }
        }
      }
      // 6. result
      T.n_hits = 0; T.first_row = -1; T.last_row = -1;
      for (int r = 0; r < n_rows; ++r) if (T.row_hit[r] >= 0) { ++T.n_hits; if (T.first_row < 0) T.first_row = r; T.last_row = r; }
      R->tracklets.push_back(std::move(T));
    }
    R->stats[7] = n_tr; R->stats[8] = n_se; R->stats[9] = n_sc; R->stats[10] = n_up;
  }
  double t4 = now();
  R->stats[3] = t4 - t3;

  // ---------------- C6 tracklet selector ----------------
  {
    std::vector<uint64_t> claim(n, 0);
    auto key = [&](const Tracklet& T) { return ((uint64_t)(uint32_t)T.n_hits << 32) | (uint64_t)(0xFFFFFFFFu - (uint32_t)T.seed); };
    for (const Tracklet& T : R->tracklets) {
      if (T.n_hits < p.min_hits) continue;
      const uint64_t k = key(T);
      for (int r = 0; r < n_rows; ++r) if (T.row_hit[r] >= 0) claim[T.row_hit[r]] = std::max(claim[T.row_hit[r]], k);
    }
    for (const Tracklet& T : R->tracklets) {
      if (T.n_hits < p.min_hits) continue;
      const uint64_t k = key(T);
      int owned = 0, first = -1, last = -1;
      for (int r = 0; r < n_rows; ++r) if (T.row_hit[r] >= 0 && claim[T.row_hit[r]] == k) { ++owned; if (first < 0) first = r; last = r; }
      if (owned < p.min_hits) continue;
      Track K;
      K.seed = T.seed; K.sector = sr[T.seed] / n_rows; K.first_row = first; K.last_row = last; K.n_hits = owned;
      K.hit_offset = (int64_t)R->track_hits.size(); K.snap = T.snap; K.time_ref = T.time_ref;
      for (int r = 0; r < n_rows; ++r) if (T.row_hit[r] >= 0 && claim[T.row_hit[r]] == k) R->track_hits.push_back(T.row_hit[r]);
      R->tracks.push_back(K);
    }
  }
  double t5 = now();
  R->stats[4] = t5 - t4;
  *out = R;
  return 0;
}

int64_t orc_n_tracklets(const orc_result* r) { return (int64_t)r->tracklets.size(); }
int64_t orc_n_tracks(const orc_result* r) { return (int64_t)r->tracks.size(); }
int64_t orc_n_track_hits(const orc_result* r) { return (int64_t)r->track_hits.size(); }

void orc_copy_links(const orc_result* r, int32_t* up_raw, int32_t* down_raw, int32_t* up, int32_t* down, uint8_t* is_start) {
  const size_t n = (size_t)r->n;
  if (up_raw) std::memcpy(up_raw, r->up_raw.data(), n * 4);
  if (down_raw) std::memcpy(down_raw, r->down_raw.data(), n * 4);
  if (up) std::memcpy(up, r->up.data(), n * 4);
  if (down) std::memcpy(down, r->down.data(), n * 4);
  if (is_start) std::memcpy(is_start, r->is_start.data(), n);
}

static void put_state(const State& S, float time_ref, float* par, float* cov) {
  if (par) { par[0] = S.x; par[1] = S.y; par[2] = S.z; par[3] = S.s; par[4] = S.t; par[5] = S.k; par[6] = time_ref; }
  if (cov) { cov[0] = S.c0; cov[1] = S.c1; cov[2] = S.c2; cov[3] = S.c3; cov[4] = S.c4; cov[5] = S.c5; cov[6] = S.d0; cov[7] = S.d1; cov[8] = S.d2; }
}

// par: [nt*7] = (x, y, z_rel, sin_phi, dzds, q_pt, time_ref); cov: [nt*9] = (c0..c5, d0..d2); row_hit: [nt*n_rows]
void orc_copy_tracklets(const orc_result* r, int32_t* seed, int32_t* n_hits, int32_t* first_row, int32_t* last_row,
                        int32_t* row_hit, float* par, float* cov) {
  for (size_t i = 0; i < r->tracklets.size(); ++i) {
    const Tracklet& T = r->tracklets[i];
    if (seed) seed[i] = T.seed;
    if (n_hits) n_hits[i] = T.n_hits;
    if (first_row) first_row[i] = T.first_row;
    if (last_row) last_row[i] = T.last_row;
    if (row_hit) std::memcpy(row_hit + i * r->n_rows, T.row_hit.data(), (size_t)r->n_rows * 4);
    put_state(T.snap, T.time_ref, par ? par + i * 7 : nullptr, cov ? cov + i * 9 : nullptr);
  }
}

void orc_copy_tracks(const orc_result* r, int32_t* seed, int32_t* sector, int32_t* first_row, int32_t* last_row,
                     int32_t* n_hits, int64_t* hit_offset, float* par, float* cov, int32_t* hit_index) {
  for (size_t i = 0; i < r->tracks.size(); ++i) {
    const Track& K = r->tracks[i];
    if (seed) seed[i] = K.seed;
    if (sector) sector[i] = K.sector;
    if (first_row) first_row[i] = K.first_row;
    if (last_row) last_row[i] = K.last_row;
    if (n_hits) n_hits[i] = K.n_hits;
    if (hit_offset) hit_offset[i] = K.hit_offset;
    put_state(K.snap, K.time_ref, par ? par + i * 7 : nullptr, cov ? cov + i * 9 : nullptr);
  }
  if (hit_index) std::memcpy(hit_index, r->track_hits.data(), r->track_hits.size() * 4);
}

void orc_copy_stats(const orc_result* r, double* out16) { std::memcpy(out16, r->stats, sizeof(r->stats)); }
void orc_free(orc_result* r) { delete r; }

// C8 rotation of a state and its covariance by q * (sector angle), q = +-1 (statement list in the C8 header below).
static bool rotate_with_cov(State& S, float qd, float Cd, float Sd, float sin_phi_max) {
  const float cs = std::sqrt(1.0f - S.s * S.s);
  const float J = Cd + qd * ((S.s / cs) * Sd);
  const float x1 = S.x * Cd + qd * (S.y * Sd);
  const float y1 = S.y * Cd - qd * (S.x * Sd);
  const float s1 = S.s * Cd - qd * (cs * Sd);
  if (!(std::fabs(s1) < sin_phi_max)) return false;
  S.x = x1; S.y = y1; S.s = s1;
  S.c1 = S.c1 * J; S.c2 = (S.c2 * J) * J; S.c4 = S.c4 * J;
  return true;
}

// ---- C8: refit of the chains linked by C7 (second half; DESIGN.md §3 "C8", readings F1..F6).
// PAPER.md L23 / L25 name "full TPC tracking"; the paper gives no listing.  One Kalman pass per chain of >= 2 pieces
// P0 -> P1 -> ... -> Pm (inner to outer), from the outermost hit of Pm inward to the innermost hit of P0, over the hits
// each piece OWNS (C6), each piece in its own sector frame; at a piece boundary the state and its covariance are rotated
// into the frame of the next inner piece and z is re-referenced to that piece's time_ref:
//   S = state of Pm (its C6 parameters);  transport(S, x of Pm's outermost hit);  cov = diag(c0_y2, c0_s2, c0_k2 | c0_z2, c0_t2)
//   for p = m .. 0:
//       for the hits of Pp, outermost first:  transport(S, x_row(hit));  update(S, y(hit), (time(hit) - time_ref_p) * Z)
//       if p > 0 (q = -sg, sg = side of the link P(p-1) -> Pp; Cd, Sd = cos, sin of the sector angle as in C7):
//           cs = sqrtf(1 - s*s);  J = Cd + q*((s/cs)*Sd)                       # d s' / d s
//           x' = x*Cd + q*(y*Sd);  y' = y*Cd - q*(x*Sd);  s' = s*Cd - q*(cs*Sd);  FAIL unless |s'| < sin_phi_max
//           c1 = c1*J;  c2 = (c2*J)*J;  c4 = c4*J;   z = z + (time_ref_p - time_ref_(p-1)) * Z
//   any transport FAIL -> the chain is flagged (ok = -1) and keeps the parameters of P0.
// Output per root: state + covariance at P0's innermost hit (z relative to P0's time_ref), hits and pieces of the chain.
void orc_refit_chains(const orc_geometry* gp, const orc_params* pp, const float* row, const float* pad, const float* time,
                      int64_t n_tracks, const int32_t* sector, const int32_t* n_hits, const int64_t* hit_offset,
                      const int32_t* hit_index, const float* par, const int32_t* next, const int32_t* prev,
                      int32_t* ok, int32_t* chain_hits, int32_t* chain_pieces, float* rpar, float* rcov) {
  const Derived D = derive(*gp, *pp);
  const double T = (double)gp->tan_half_sector;
  const float Cd = (float)((1.0 - T * T) / (1.0 + T * T)), Sd = (float)(2.0 * T / (1.0 + T * T));
  const int nr = gp->n_rows;
  for (int64_t i = 0; i < n_tracks; ++i) {
    ok[i] = 0; chain_hits[i] = n_hits[i]; chain_pieces[i] = 1;
    for (int k = 0; k < 7; ++k) rpar[7 * i + k] = par[7 * i + k];
    for (int k = 0; k < 9; ++k) rcov[9 * i + k] = 0.0f;
    if (prev[i] >= 0 || next[i] < 0) continue;
    std::vector<int64_t> pieces;
    for (int64_t p = i; p >= 0; p = next[p]) pieces.push_back(p);
    int32_t total = 0;
    for (int64_t p : pieces) total += n_hits[p];
    chain_hits[i] = total; chain_pieces[i] = (int32_t)pieces.size();
    const int64_t pm = pieces.back();
    const float* q = par + 7 * pm;
    State S{q[0], q[1], q[2], q[3], q[4], q[5], 0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool good = true;
    {
      const int32_t h = hit_index[hit_offset[pm] + n_hits[pm] - 1];
      good = transport(S, D.xr[(int)row[h] % nr], D.cB, pp->sin_phi_max);
    }
    S.c0 = pp->c0_y2; S.c1 = 0; S.c2 = pp->c0_s2; S.c3 = 0; S.c4 = 0; S.c5 = pp->c0_k2; S.d0 = pp->c0_z2; S.d1 = 0; S.d2 = pp->c0_t2;
    for (int ip = (int)pieces.size() - 1; ip >= 0 && good; --ip) {
      const int64_t p = pieces[ip];
      const float tref = par[7 * p + 6];
      for (int64_t j = hit_offset[p] + n_hits[p] - 1; j >= hit_offset[p] && good; --j) {
        const int32_t h = hit_index[j];
        const int r = (int)row[h] % nr;
        good = transport(S, D.xr[r], D.cB, pp->sin_phi_max);
        if (!good) break;
        const float ym = (pad[h] - D.cr[r]) * D.P;
        const float zm = (time[h] - tref) * D.Z;
        update(S, ym, zm, D.ry, D.rz);
      }
      if (good && ip > 0) {
        const int64_t pin = pieces[ip - 1];
        const float sg = ((sector[p] % 18) == ((sector[pin] % 18) + 1) % 18) ? 1.0f : -1.0f;
        if (!rotate_with_cov(S, -sg, Cd, Sd, pp->sin_phi_max)) { good = false; break; }
        S.z = S.z + (tref - par[7 * pin + 6]) * D.Z;
      }
    }
    if (good) {
      ok[i] = 1;
      put_state(S, par[7 * i + 6], rpar + 7 * i, rcov + 9 * i);
    } else {
      ok[i] = -1;
    }
  }
}

// ---- C11: track-based hit rejection and track-model residual coding ("the step after the path";
// PAPER.md L23 (§1): the TPC data are compressed online by "removal of TPC hits of tracks not used for physics" and "reduction
// of the hit property entropy" -- the reason the tracking runs synchronously at all).  The paper gives neither rule nor
// format, so the definitions are readings of this build (R11-1..R11-6, DESIGN.md §3 "C11"); the entropy coder behind it (ANS)
// is out of scope.
//   Rejection: every hit a track OWNS (C6) is rejected iff |q/pT| of the track > reject_qpt (a low-momentum looper, "not used
//   for physics"); hits no track owns are kept (R11-1).
//   Residual coding of the hits of every KEPT track, a closed-loop predictive coder (R11-2..5): the state starts as the
//   track's C6 parameters and covariance (they travel in the stream as the track header); for the owned hits in ascending row:
//       transport(S, x_row)                          FAIL -> the track is flagged ok = 0 and its remaining symbols are 0
//       ry = y(hit) - S.y;  rz = (time(hit) - time_ref) * Z - S.z
//       qy = (int)rintf(ry / step_y), qz = (int)rintf(rz / step_z), each clamped to [-32767, 32767]
//       yq = S.y + (float)qy * step_y;  zq = S.z + (float)qz * step_z        # what a decoder reconstructs
//       update(S, yq, zq)                            # with the RECONSTRUCTED hit: the decoder's state is the same
//   Output: (qy, qz) per track hit in hit_index order, ok per track, reject per cluster.
// orc_decompress_tracks is the decoder (headers + symbols -> hit coordinates), used by the pins only.
void orc_compress_tracks(const orc_geometry* gp, const orc_params* pp, float reject_qpt, float step_y, float step_z,
                         const float* row, const float* pad, const float* time, int64_t n_clusters,
                         int64_t n_tracks, const int32_t* n_hits, const int64_t* hit_offset, const int32_t* hit_index,
                         const float* par, const float* cov, uint8_t* reject, int32_t* ok, int16_t* qy, int16_t* qz) {
  const Derived D = derive(*gp, *pp);
  const int nr = gp->n_rows;
  for (int64_t i = 0; i < n_clusters; ++i) reject[i] = 0;
  for (int64_t k = 0; k < n_tracks; ++k) {
    const float* q = par + 7 * k;
    const float* cv = cov + 9 * k;
    const bool rej = std::fabs(q[5]) > reject_qpt;
    ok[k] = rej ? -1 : 1;
    State S{q[0], q[1], q[2], q[3], q[4], q[5], cv[0], cv[1], cv[2], cv[3], cv[4], cv[5], cv[6], cv[7], cv[8]};
    bool good = !rej;
    for (int64_t j = hit_offset[k]; j < hit_offset[k] + n_hits[k]; ++j) {
      const int32_t h = hit_index[j];
      if (rej) { reject[h] = 1; qy[j] = 0; qz[j] = 0; continue; }
      if (good) good = transport(S, D.xr[(int)row[h] % nr], D.cB, pp->sin_phi_max);
      if (!good) { ok[k] = 0; qy[j] = 0; qz[j] = 0; continue; }
      const int r = (int)row[h] % nr;
      const float ym = (pad[h] - D.cr[r]) * D.P;
      const float zm = (time[h] - q[6]) * D.Z;
      const float ry = ym - S.y, rz = zm - S.z;
      int iy = (int)std::rint(ry / step_y), iz = (int)std::rint(rz / step_z);
      iy = std::min(std::max(iy, -32767), 32767); iz = std::min(std::max(iz, -32767), 32767);
      qy[j] = (int16_t)iy; qz[j] = (int16_t)iz;
      const float yq = S.y + (float)iy * step_y, zq = S.z + (float)iz * step_z;
      update(S, yq, zq, D.ry, D.rz);
    }
  }
}

// The decoder: from the track headers (par, cov, n_hits, rows of the hits) and the symbols back to (y, z relative to
// time_ref) of every hit of the tracks with ok == 1.  Mirrors the encoder's state exactly.
void orc_decompress_tracks(const orc_geometry* gp, const orc_params* pp, float step_y, float step_z, int64_t n_tracks,
                           const int32_t* n_hits, const int64_t* hit_offset, const uint8_t* hit_row, const float* par, const float* cov,
                           const int32_t* ok, const int16_t* qy, const int16_t* qz, float* y_out, float* z_out) {
  const Derived D = derive(*gp, *pp);
  for (int64_t k = 0; k < n_tracks; ++k) {
    if (ok[k] != 1) continue;
    const float* q = par + 7 * k;
    const float* cv = cov + 9 * k;
    State S{q[0], q[1], q[2], q[3], q[4], q[5], cv[0], cv[1], cv[2], cv[3], cv[4], cv[5], cv[6], cv[7], cv[8]};
    for (int64_t j = hit_offset[k]; j < hit_offset[k] + n_hits[k]; ++j) {
      transport(S, D.xr[hit_row[j]], D.cB, pp->sin_phi_max);
      const float yq = S.y + (float)qy[j] * step_y, zq = S.z + (float)qz[j] * step_z;
      y_out[j] = yq; z_out[j] = zq;
      update(S, yq, zq, D.ry, D.rz);
    }
  }
}

// ---- C12: refit with the full 5x5 covariance, multiple scattering and energy loss ("Full 5x5
// covariance with multiple scattering / energy loss"; PAPER.md L37 (§2): "future improvement of the tracking efficiency, which
// will require the fit of more tracks and more attached hits").  The paper gives no listing: the definitions are readings of
// this build (FF1..FF7, DESIGN.md §3 "C12").  One inward Kalman pass over every ROOT of C7's chains -- single tracks too --
// in C8's hit order and with C8's start (FF1); state (y, z, s, t, k) at x, covariance the full symmetric 5x5 matrix, stored as
// its lower triangle in the order (yy | zy zz | sy sz ss | ty tz ts tt | ky kz ks kt kk).
//   step(S, x_row):                                              # transport + material, FAIL as in C5
//     state part and dx, T, rq, dS, fa, e, fb exactly as the C5 transport
//     gm = t * (T / rq);  zs = gm * fa;  zk = gm * fb             # dz/ds, dz/dk to first order in the chord (FF2)
//     F = rows  y: (1, 0, fa, 0, fb)   z: (0, 1, zs, dS, zk)   s: (0, 0, 1, 0, e)   t, k: unit
//     A = F P:     A[y][j] = P[y][j] + fa*P[s][j] + fb*P[k][j];  A[z][j] = P[z][j] + zs*P[s][j] + dS*P[t][j] + zk*P[k][j];
//                  A[s][j] = P[s][j] + e*P[k][j];  rows t, k unchanged
//     P = A F^T:   P[i][y] = A[i][y] + fa*A[i][s] + fb*A[i][k];  P[i][z] = A[i][z] + zs*A[i][s] + dS*A[i][t] + zk*A[i][k];
//                  P[i][s] = A[i][s] + e*A[i][k];  columns t, k = A's                      (lower triangle only)
//     material of the step (FF3..FF6), with s the NEW sin phi and t, k unchanged by the transport:
//       tt1 = 1 + t*t;  Lp = fabsf(dS) * sqrtf(tt1);  ip2 = (k*k) / tt1;  ib2 = 1 + m2*ip2;  ibp2 = ip2 * ib2
//       th2 = (ms2 * ibp2) * (Lp * inv_x0)                         # Highland theta0^2 without the log term, ms2 = 0.0136^2
//       P[ss] += th2 * ((1 - s*s) * tt1);  P[tt] += th2 * (tt1*tt1);  tk = t*k;  P[kt] += th2 * (tk * tt1);  P[kk] += th2 * (tk*tk)
//       dl = ((dedx * ib2) * Lp) * sqrtf(ibp2)                     # dE / (beta p), dE/dx = dedx_mip / beta^2
//       k = k * (1 - dl)                                           # inward = against the flight: the momentum comes back
//       ek = (k * dl) * eloss_sigma;  P[kk] += ek * ek             # straggling (k already corrected)
//   update1(S, i, meas, r):  scalar measurement of component i (0 = y, 1 = z)
//       col[j] = P[j][i] (j = 0..4);  w = 1 / (col[i] + r);  res = meas - S[i];  K[j] = col[j] * w
//       S[j] = S[j] + K[j]*res;  P[j][l] = P[j][l] - K[j]*col[l]   (l <= j)
//   per hit:  step(S, x_row);  update1(S, 0, y(hit), r_y);  update1(S, 1, (time - time_ref_p)*Z, r_z)
//   boundary: C8's rotation of (x, y, s); the row and column s of P are multiplied by J (ss by J twice) (FF7); z re-referenced.
// Output per root: ok (1 fitted, -1 FAIL, 0 not a root), chain_hits, chain_pieces, par7, and the 15 covariance values.
namespace {
struct FullParams { float inv_x0, dedx_mip, mass, eloss_sigma; };
struct FullState { float x, v[5]; float P[5][5]; };     // v = (y, z, s, t, k); P kept as a full symmetric matrix
inline int tri(int i, int j) { return i >= j ? i * (i + 1) / 2 + j : j * (j + 1) / 2 + i; }

// mass^2 and the squared Highland constant (13.6 MeV)^2 in GeV^2, derived in double and rounded once
void full_consts(const FullParams& fp, float& m2, float& ms2) {
  m2 = (float)((double)fp.mass * (double)fp.mass);
  ms2 = (float)(0.0136 * 0.0136);
}

bool full_step(FullState& S, float xn, float cB, float sin_phi_max, const FullParams& fp, float m2, float ms2) {
  const float s0 = S.v[2], t = S.v[3], k0 = S.v[4];
  const float dx = xn - S.x;
  const float kc = cB * k0;
  const float sn = s0 + kc * dx;
  if (!(std::fabs(s0) < sin_phi_max && std::fabs(sn) < sin_phi_max)) return false;
  const float c = std::sqrt(1.0f - s0 * s0);
  const float cn = std::sqrt(1.0f - sn * sn);
  const float ss = s0 + sn;
  const float cc = c + cn;
  const float icc = 1.0f / cc;
  const float T = ss * icc;
  const float q = 1.0f + T * T;
  const float rq = std::sqrt(q);
  const float u = kc * dx;
  const float a = (u * u) * q;
  const float dS = (dx * rq) * (1.0f + a * (0.041666668f + a * (0.0046875f + a * 0.00069754466f)));
  const float g0 = (1.0f + T * (s0 / c)) * icc;
  const float g1 = (1.0f + T * (sn / cn)) * icc;
  const float fa = dx * (g0 + g1);
  const float e = cB * dx;
  const float fb = (dx * g1) * e;
  const float gm = t * (T / rq);
  const float zs = gm * fa;
  const float zk = gm * fb;
  S.v[0] = S.v[0] + dx * T;
  S.v[1] = S.v[1] + t * dS;
  S.v[2] = sn;
  S.x = xn;
  float A[5][5];
  for (int j = 0; j < 5; ++j) {
    A[0][j] = S.P[0][j] + fa * S.P[2][j] + fb * S.P[4][j];
    A[1][j] = S.P[1][j] + zs * S.P[2][j] + dS * S.P[3][j] + zk * S.P[4][j];
    A[2][j] = S.P[2][j] + e * S.P[4][j];
    A[3][j] = S.P[3][j];
    A[4][j] = S.P[4][j];
  }
  float B[5][5];
  for (int i = 0; i < 5; ++i) {
    B[i][0] = A[i][0] + fa * A[i][2] + fb * A[i][4];
    B[i][1] = A[i][1] + zs * A[i][2] + dS * A[i][3] + zk * A[i][4];
    B[i][2] = A[i][2] + e * A[i][4];
    B[i][3] = A[i][3];
    B[i][4] = A[i][4];
  }
  for (int i = 0; i < 5; ++i) for (int j = 0; j <= i; ++j) { S.P[i][j] = B[i][j]; S.P[j][i] = B[i][j]; }   // the lower triangle is the result
  // material
  const float tt1 = 1.0f + t * t;
  const float Lp = std::fabs(dS) * std::sqrt(tt1);
  const float ip2 = (k0 * k0) / tt1;
  const float ib2 = 1.0f + m2 * ip2;
  const float ibp2 = ip2 * ib2;
  const float th2 = (ms2 * ibp2) * (Lp * fp.inv_x0);
  S.P[2][2] = S.P[2][2] + th2 * ((1.0f - sn * sn) * tt1);
  S.P[3][3] = S.P[3][3] + th2 * (tt1 * tt1);
  const float tk = t * k0;
  S.P[4][3] = S.P[4][3] + th2 * (tk * tt1); S.P[3][4] = S.P[4][3];
  S.P[4][4] = S.P[4][4] + th2 * (tk * tk);
  const float dl = ((fp.dedx_mip * ib2) * Lp) * std::sqrt(ibp2);
  S.v[4] = k0 * (1.0f - dl);
  const float ek = (S.v[4] * dl) * fp.eloss_sigma;
  S.P[4][4] = S.P[4][4] + ek * ek;
  return true;
}

void full_update1(FullState& S, int i, float meas, float r) {
  float col[5], K[5];
  for (int j = 0; j < 5; ++j) col[j] = S.P[j][i];
  const float w = 1.0f / (col[i] + r);
  const float res = meas - S.v[i];
  for (int j = 0; j < 5; ++j) K[j] = col[j] * w;
  for (int j = 0; j < 5; ++j) S.v[j] = S.v[j] + K[j] * res;
  for (int j = 0; j < 5; ++j) for (int l = 0; l <= j; ++l) { S.P[j][l] = S.P[j][l] - K[j] * col[l]; S.P[l][j] = S.P[j][l]; }
}

void full_reset(FullState& S, const orc_params& p) {
  for (int i = 0; i < 5; ++i) for (int j = 0; j < 5; ++j) S.P[i][j] = 0.0f;
  S.P[0][0] = p.c0_y2; S.P[1][1] = p.c0_z2; S.P[2][2] = p.c0_s2; S.P[3][3] = p.c0_t2; S.P[4][4] = p.c0_k2;
}

// C12 at the central electrode (FF8): the time coordinate reflected about the crossing time tc; z was relative to tref_b (the
// piece behind the electrode) and becomes relative to tref_e (the piece in front of it).
void full_reflect(FullState& S, float tc, float tref_b, float tref_e, float Z) {
  S.v[1] = (((tc + tc) - tref_b) - tref_e) * Z - S.v[1];
  S.v[3] = -S.v[3];
  for (int a = 0; a < 5; ++a) for (int b = 0; b < 5; ++b)
    if (((a == 1 || a == 3) ? 1 : 0) != ((b == 1 || b == 3) ? 1 : 0)) S.P[a][b] = -S.P[a][b];
}

bool full_rotate(FullState& S, float qd, float Cd, float Sd, float sin_phi_max) {
  const float s0 = S.v[2];
  const float cs = std::sqrt(1.0f - s0 * s0);
  const float J = Cd + qd * ((s0 / cs) * Sd);
  const float x1 = S.x * Cd + qd * (S.v[0] * Sd);
  const float y1 = S.v[0] * Cd - qd * (S.x * Sd);
  const float s1 = s0 * Cd - qd * (cs * Sd);
  if (!(std::fabs(s1) < sin_phi_max)) return false;
  S.x = x1; S.v[0] = y1; S.v[2] = s1;
  for (int j = 0; j < 5; ++j) if (j != 2) { S.P[2][j] = S.P[2][j] * J; S.P[j][2] = S.P[2][j]; }
  S.P[2][2] = (S.P[2][2] * J) * J;
  return true;
}
}  // namespace

// C12 with the links of C10 (reading FF8): a chain may continue behind the central electrode.  Pieces of a root: follow C7's
// `next`; where that ends at piece e, a C10 link ce_next[e] = b is taken iff prev[b] < 0 (b starts a C7 chain on the other
// side) and the chain has not crossed yet; then b's `next` links.  A track is a root iff prev < 0 and it is not such a b.
// The pass runs inward as before.  At the electrode, between b (just fitted down to its innermost hit) and e:
//     z = (((t_ce[e] + t_ce[e]) - time_ref_b) - time_ref_e) * Z - z          # the time coordinate reflected about t_ce, now relative to e
//     t = -t;   P[i][j] = -P[i][j] for exactly one of i, j in {z, t}              # D P D with D = diag(1, -1, 1, -1, 1)
// x, y, sin phi, q/pT are continuous: the mirror sector shares the local frame (no rotation).  ce_next == nullptr: plain C12.
void orc_refit_full_ce(const orc_geometry* gp, const orc_params* pp, const float* full4, const float* row, const float* pad,
                       const float* time, int64_t n_tracks, const int32_t* sector, const int32_t* n_hits, const int64_t* hit_offset,
                       const int32_t* hit_index, const float* par, const int32_t* next, const int32_t* prev,
                       const int32_t* ce_next, const int32_t* ce_prev, const float* t_ce,
                       int32_t* ok, int32_t* chain_hits, int32_t* chain_pieces, float* rpar, float* rcov15) {
  const Derived D = derive(*gp, *pp);
  const FullParams fp{full4[0], full4[1], full4[2], full4[3]};
  float m2, ms2;
  full_consts(fp, m2, ms2);
  const double T = (double)gp->tan_half_sector;
  const float Cd = (float)((1.0 - T * T) / (1.0 + T * T)), Sd = (float)(2.0 * T / (1.0 + T * T));
  const int nr = gp->n_rows;
  auto crosses_into = [&](int64_t e) -> int64_t {      // the piece behind the electrode that continues e, or -1
    if (!ce_next || next[e] >= 0) return -1;
    const int64_t b = ce_next[e];
    return (b >= 0 && prev[b] < 0) ? b : -1;
  };
  for (int64_t i = 0; i < n_tracks; ++i) {
    ok[i] = 0; chain_hits[i] = n_hits[i]; chain_pieces[i] = 1;
    for (int k = 0; k < 7; ++k) rpar[7 * i + k] = par[7 * i + k];
    for (int k = 0; k < 15; ++k) rcov15[15 * i + k] = 0.0f;
    if (prev[i] >= 0) continue;
    if (ce_next && ce_prev[i] >= 0 && crosses_into(ce_prev[i]) == i) continue;      // continuation of a chain from the other side
    std::vector<int64_t> pieces;
    int64_t ce_at = -1;                                // index in `pieces` of the first piece behind the electrode
    for (int64_t p = i; p >= 0;) {
      pieces.push_back(p);
      if ((int64_t)pieces.size() > 4 * (int64_t)nr) break;          // cannot happen (M7): never walk a corrupted link list for ever
      if (next[p] >= 0) { p = next[p]; continue; }
      const int64_t b = ce_at < 0 ? crosses_into(p) : -1;
      if (b >= 0) ce_at = (int64_t)pieces.size();
      p = b;
    }
    int32_t total = 0;
    for (int64_t p : pieces) total += n_hits[p];
    chain_hits[i] = total; chain_pieces[i] = (int32_t)pieces.size();
    const int64_t pm = pieces.back();
    const float* q = par + 7 * pm;
    FullState S;
    S.x = q[0]; S.v[0] = q[1]; S.v[1] = q[2]; S.v[2] = q[3]; S.v[3] = q[4]; S.v[4] = q[5];
    bool good = n_hits[pm] > 0;
    if (good) {     // FF1: to the outermost hit with the plain C5 transport (no material), then the reset covariance
      State S0{q[0], q[1], q[2], q[3], q[4], q[5], 0, 0, 0, 0, 0, 0, 0, 0, 0};
      const int32_t h = hit_index[hit_offset[pm] + n_hits[pm] - 1];
      good = transport(S0, D.xr[(int)row[h] % nr], D.cB, pp->sin_phi_max);
      S.x = S0.x; S.v[0] = S0.y; S.v[1] = S0.z; S.v[2] = S0.s;
    }
    full_reset(S, *pp);
    for (int ip = (int)pieces.size() - 1; ip >= 0 && good; --ip) {
      const int64_t p = pieces[ip];
      const float tref = par[7 * p + 6];
      for (int64_t j = hit_offset[p] + n_hits[p] - 1; j >= hit_offset[p] && good; --j) {
        const int32_t h = hit_index[j];
        const int r = (int)row[h] % nr;
        good = full_step(S, D.xr[r], D.cB, pp->sin_phi_max, fp, m2, ms2);
        if (!good) break;
        full_update1(S, 0, (pad[h] - D.cr[r]) * D.P, D.ry);
        full_update1(S, 1, (time[h] - tref) * D.Z, D.rz);
      }
      if (good && ip > 0) {
        const int64_t pin = pieces[ip - 1];
        if (ip == ce_at) {                             // the central electrode: reflect the time coordinate
          full_reflect(S, t_ce[pin], tref, par[7 * pin + 6], D.Z);
        } else {
          const float sg = ((sector[p] % 18) == ((sector[pin] % 18) + 1) % 18) ? 1.0f : -1.0f;
          if (!full_rotate(S, -sg, Cd, Sd, pp->sin_phi_max)) { good = false; break; }
          S.v[1] = S.v[1] + (tref - par[7 * pin + 6]) * D.Z;
        }
      }
    }
    if (good) {
      ok[i] = 1;
      float* o = rpar + 7 * i;
      o[0] = S.x; o[1] = S.v[0]; o[2] = S.v[1]; o[3] = S.v[2]; o[4] = S.v[3]; o[5] = S.v[4];
      for (int a = 0; a < 5; ++a) for (int b = 0; b <= a; ++b) rcov15[15 * i + tri(a, b)] = S.P[a][b];
    } else {
      ok[i] = -1;
    }
  }
}

void orc_refit_full(const orc_geometry* gp, const orc_params* pp, const float* full4, const float* row, const float* pad,
                    const float* time, int64_t n_tracks, const int32_t* sector, const int32_t* n_hits, const int64_t* hit_offset,
                    const int32_t* hit_index, const float* par, const int32_t* next, const int32_t* prev,
                    int32_t* ok, int32_t* chain_hits, int32_t* chain_pieces, float* rpar, float* rcov15) {
  orc_refit_full_ce(gp, pp, full4, row, pad, time, n_tracks, sector, n_hits, hit_offset, hit_index, par, next, prev, nullptr, nullptr, nullptr,
                    ok, chain_hits, chain_pieces, rpar, rcov15);
}

// One step / one update of C12 on their own (pins FF-*): st6 = (x, y, z, s, t, k), cov15 = lower triangle.
int orc_full_step(const orc_params* p, const float* full4, float* st, float* cov15, float xn) {
  const FullParams fp{full4[0], full4[1], full4[2], full4[3]};
  float m2, ms2;
  full_consts(fp, m2, ms2);
  FullState S;
  S.x = st[0]; for (int j = 0; j < 5; ++j) S.v[j] = st[1 + j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b < 5; ++b) S.P[a][b] = cov15[tri(a, b)];
  const bool ok = full_step(S, xn, p->inv_R_per_qpt, p->sin_phi_max, fp, m2, ms2);
  st[0] = S.x; for (int j = 0; j < 5; ++j) st[1 + j] = S.v[j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b <= a; ++b) cov15[tri(a, b)] = S.P[a][b];
  return ok ? 0 : 1;
}
// C12 rotation on its own (pin FF-R): q = +1 / -1.  Returns 0, or 1 when |s'| >= sin_phi_max (state unchanged).
int orc_full_rotate(const orc_geometry* g, const orc_params* p, float* st, float* cov15, int32_t q) {
  const double T = (double)g->tan_half_sector;
  const float Cd = (float)((1.0 - T * T) / (1.0 + T * T)), Sd = (float)(2.0 * T / (1.0 + T * T));
  FullState S;
  S.x = st[0]; for (int j = 0; j < 5; ++j) S.v[j] = st[1 + j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b < 5; ++b) S.P[a][b] = cov15[tri(a, b)];
  const bool ok = full_rotate(S, q >= 0 ? 1.0f : -1.0f, Cd, Sd, p->sin_phi_max);
  st[0] = S.x; for (int j = 0; j < 5; ++j) st[1 + j] = S.v[j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b <= a; ++b) cov15[tri(a, b)] = S.P[a][b];
  return ok ? 0 : 1;
}
void orc_full_reflect(float* st, float* cov15, float tc, float tref_b, float tref_e, float Z) {
  FullState S;
  S.x = st[0]; for (int j = 0; j < 5; ++j) S.v[j] = st[1 + j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b < 5; ++b) S.P[a][b] = cov15[tri(a, b)];
  full_reflect(S, tc, tref_b, tref_e, Z);
  for (int j = 0; j < 5; ++j) st[1 + j] = S.v[j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b <= a; ++b) cov15[tri(a, b)] = S.P[a][b];
}
void orc_full_update(float* st, float* cov15, float ym, float zm, float ry, float rz) {
  FullState S;
  S.x = st[0]; for (int j = 0; j < 5; ++j) S.v[j] = st[1 + j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b < 5; ++b) S.P[a][b] = cov15[tri(a, b)];
  full_update1(S, 0, ym, ry);
  full_update1(S, 1, zm, rz);
  for (int j = 0; j < 5; ++j) st[1 + j] = S.v[j];
  for (int a = 0; a < 5; ++a) for (int b = 0; b <= a; ++b) cov15[tri(a, b)] = S.P[a][b];
}

// ---- hooks for the pins (K1..K3, G1): the same functions the tracker uses, callable one at a time ----
// state6 = (x, y, z, s, t, k); cov9 = (c0..c5, d0..d2).  Returns 0, or 1 on transport FAIL.
int orc_transport(const orc_params* p, float* st, float* cv, float xn) {
  State S{st[0], st[1], st[2], st[3], st[4], st[5], cv[0], cv[1], cv[2], cv[3], cv[4], cv[5], cv[6], cv[7], cv[8]};
  const bool ok = transport(S, xn, p->inv_R_per_qpt, p->sin_phi_max);
  put_state(S, 0.0f, nullptr, cv);
  st[0] = S.x; st[1] = S.y; st[2] = S.z; st[3] = S.s; st[4] = S.t; st[5] = S.k;
  return ok ? 0 : 1;
}

void orc_update(float* st, float* cv, float ym, float zm, float ry, float rz) {
  State S{st[0], st[1], st[2], st[3], st[4], st[5], cv[0], cv[1], cv[2], cv[3], cv[4], cv[5], cv[6], cv[7], cv[8]};
  update(S, ym, zm, ry, rz);
  put_state(S, 0.0f, nullptr, cv);
  st[0] = S.x; st[1] = S.y; st[2] = S.z; st[3] = S.s; st[4] = S.t; st[5] = S.k;
}

// C8 rotation on its own (pin F-J): q = +1 / -1.  Returns 0, or 1 when |s'| >= sin_phi_max (state unchanged).
int orc_rotate_with_cov(const orc_geometry* g, const orc_params* p, float* st, float* cv, int32_t q) {
  const double T = (double)g->tan_half_sector;
  const float Cd = (float)((1.0 - T * T) / (1.0 + T * T)), Sd = (float)(2.0 * T / (1.0 + T * T));
  State S{st[0], st[1], st[2], st[3], st[4], st[5], cv[0], cv[1], cv[2], cv[3], cv[4], cv[5], cv[6], cv[7], cv[8]};
  const bool ok = rotate_with_cov(S, q >= 0 ? 1.0f : -1.0f, Cd, Sd, p->sin_phi_max);
  put_state(S, 0.0f, nullptr, cv);
  st[0] = S.x; st[1] = S.y; st[2] = S.z; st[3] = S.s; st[4] = S.t; st[5] = S.k;
  return ok ? 0 : 1;
}

// x_r [n_rows], n_pads [n_rows], c_r [n_rows]; consts8 = (W1, Ay, Az, wy, wz, ry, rz, 0)
void orc_tables(const orc_geometry* g, const orc_params* p, float* x_r, int32_t* n_pads, float* c_r, float* consts8) {
  const Derived D = derive(*g, *p);
  for (int r = 0; r < g->n_rows; ++r) {
    if (x_r) x_r[r] = D.xr[r];
    if (n_pads) n_pads[r] = D.npads[r];
    if (c_r) c_r[r] = D.cr[r];
  }
  if (consts8) { consts8[0] = D.W1; consts8[1] = D.Ay; consts8[2] = D.Az; consts8[3] = D.wy; consts8[4] = D.wz; consts8[5] = D.ry; consts8[6] = D.rz; consts8[7] = 0; }
}

}  // extern "C"
