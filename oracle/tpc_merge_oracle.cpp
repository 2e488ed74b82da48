// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain single-threaded C++ fp32 CPU implementation of step C7:
// merging of the per-sector TPC tracks of C6 across SECTOR BOUNDARIES (first half:
// the linking of track pieces; the global refit of a merged chain is not part of this step).
//
// What it follows:
//   * PAPER.md L23 / L25: "full TPC tracking"; the per-sector tracker (Run 2 HLT design) is followed by a
//     merger of the sector tracks.  The paper gives no listing and no cuts, so every definition below is a
//     reading of this build, listed as M1..M8 in DESIGN.md §3 ("C7").
//   * BASELINE.json L8: 36 sectors, A side 0-17, C side 18-35, 20 degree slices, each in its rotated local frame.
// It is a HEURISTIC (greedy reciprocal best match), followed step by step; all decisions in fp32, one rounded
// operation per statement, evaluated left to right, built with -O2 -ffp-contract=off.
//
// Definition (notation of DESIGN.md §3; a track is (sector S, first_row f, last_row l, seed id, state
// (x; y, z, s, t, k) at its innermost point, time_ref)):
//   Cd = (1 - T^2) / (1 + T^2), Sd = 2 T / (1 + T^2) with T = tan_half_sector: cos / sin of the sector angle,
//   derived in double from the fp32 geometry value and rounded once (no libm).
//   For a track A and a side sg in {+1, -1}, the neighbour sector is S' = side(S)*18 + ((S mod 18) + sg) mod 18;
//   A's state in the frame of S' (rotation by sg * 20 degrees about the beam axis):
//       c  = sqrtf(1 - s*s)
//       x1 = x*Cd + sg*(y*Sd);   y1 = y*Cd - sg*(x*Sd);   s1 = s*Cd - sg*(c*Sd)       (z, t, k unchanged)
//       skip the side unless |s1| < sin_phi_max
//   r_X = (int)floorf((x_X - x0) / pitch + 0.5f) is the pad row the state of track X sits on: the row of the tracklet's last
//   Kalman update -- normally its innermost hit (r_X <= f_X), but a down refit that FAILs early leaves the state higher up.
//   A candidate continuation is a track B in S' whose state really is at its inner end,  r_B <= f_B,  with
//   r_B > max(f_A, r_A)  and  l_A + 1 - overlap <= r_B <= l_A + 1 + gap   (reading M7: state rows strictly increase along
//   a chain, so chains are acyclic and hold at most n_rows pieces).
//   The rotated state is transported to x_B with the state part of the C5 transport (exact circle, 3-term arc
//   length series; FAIL -> no candidate), giving (y2, z2, s2); then
//       dy = y2 - y_B;  dz = (z2 - z_B) + (time_ref_A - time_ref_B)*Z;  ds = s2 - s_B;  dk = k_A - k_B
//       require |dy| < cut_y, |dz| < cut_z, |ds| < cut_s, |dk| < cut_k
//       d2 = (dy*dy)*wy + (dz*dz)*wz + (ds*ds)*ws + (dk*dk)*wk            w = (float)(1 / cut^2), from double
//   out[A] = the candidate with the smallest d2 over both sides (ties -> smallest seed id of B);
//   in[B]  = the A with the smallest d2(A, B) among all A that have B as a candidate (ties -> smallest seed id of A).
//   A and B are LINKED (next[A] = B, prev[B] = A) iff out[A] == B and in[B] == A.
//   root[i] = the first piece of i's chain (follow prev).  A geometry with fewer than 18 sectors has no neighbours.
//
// Pins (tests/test_merge_oracle_pins.py): M-R rotation against the double-precision helix in global coordinates
// and there-and-back identity; M-H noise-free helices crossing one or two boundaries are linked into one chain
// and nothing else is linked; M-I invariants (reciprocity, adjacency, row order, acyclic); M-E link efficiency and
// purity against generator truth on configs[1].  Parity unpinned: the values of the cuts themselves.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.  It
// shares no code, header, table or constant generator with the CUDA path.
#include <cmath>
#include <cstdint>
#include <vector>

extern "C" {

struct orc_merge_params {
  int32_t n_sectors;
  float x0_cm, row_pitch_cm;
  float tan_half_sector, time_bin_cm;
  float sin_phi_max, inv_R_per_qpt;
  float cut_y_cm, cut_z_cm, cut_sin_phi, cut_q_pt;
  int32_t max_row_gap, max_row_overlap;
};

}  // extern "C"

namespace {

struct St { float x, y, z, s, t, k; };

// State part of the C5 transport: same statements, same order; false = FAIL (state unchanged).
bool transport_state(St& S, float xn, float cB, float sin_phi_max) {
  const float dx = xn - S.x;
  const float kc = cB * S.k;
  const float sn = S.s + kc * dx;
  if (!(std::fabs(S.s) < sin_phi_max && std::fabs(sn) < sin_phi_max)) return false;
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
  S.y = S.y + dx * T;
  S.z = S.z + S.t * dS;
  S.s = sn;
  S.x = xn;
  return true;
}

struct Consts { float Cd, Sd, wy, wz, ws, wk; };

Consts derive(const orc_merge_params& p) {
  const double T = (double)p.tan_half_sector;
  Consts c;
  c.Cd = (float)((1.0 - T * T) / (1.0 + T * T));
  c.Sd = (float)(2.0 * T / (1.0 + T * T));
  c.wy = (float)(1.0 / ((double)p.cut_y_cm * (double)p.cut_y_cm));
  c.wz = (float)(1.0 / ((double)p.cut_z_cm * (double)p.cut_z_cm));
  c.ws = (float)(1.0 / ((double)p.cut_sin_phi * (double)p.cut_sin_phi));
  c.wk = (float)(1.0 / ((double)p.cut_q_pt * (double)p.cut_q_pt));
  return c;
}

// Rotation of a state into the neighbour frame on side sg (+1 / -1).
St rotate(const St& A, float sg, const Consts& c) {
  St R = A;
  const float cs = std::sqrt(1.0f - A.s * A.s);
  R.x = A.x * c.Cd + sg * (A.y * c.Sd);
  R.y = A.y * c.Cd - sg * (A.x * c.Sd);
  R.s = A.s * c.Cd - sg * (cs * c.Sd);
  return R;
}

}  // namespace

extern "C" {

// par: [n*7] = (x, y, z_rel, sin_phi, dzds, q_pt, time_ref) as written by the tracker / orc_copy_tracks.
// next, prev, root: [n] track indices (-1 = none; root[i] = i for an unmerged track).  Returns the number of links.
int64_t orc_merge(const orc_merge_params* pp, int64_t n, const int32_t* seed, const int32_t* sector,
                  const int32_t* first_row, const int32_t* last_row, const float* par,
                  int32_t* next, int32_t* prev, int32_t* root, float* best_d2_out) {
  const orc_merge_params& p = *pp;
  const Consts c = derive(p);
  std::vector<int32_t> out(n, -1), in(n, -1);
  std::vector<float> d_out(n, 0.0f), d_in(n, 0.0f);
  if (p.n_sectors >= 18) {
    for (int64_t a = 0; a < n; ++a) {
      const float* pa = par + 7 * a;
      const St A{pa[0], pa[1], pa[2], pa[3], pa[4], pa[5]};
      const int32_t side = sector[a] / 18, phi = sector[a] % 18;
      for (int isg = 0; isg < 2; ++isg) {
        const float sg = isg == 0 ? 1.0f : -1.0f;
        const int32_t nb = side * 18 + (phi + (isg == 0 ? 1 : 17)) % 18;
        if (nb >= p.n_sectors) continue;
        const St R = rotate(A, sg, c);
        if (!(std::fabs(R.s) < p.sin_phi_max)) continue;
        for (int64_t b = 0; b < n; ++b) {            // brute force over all tracks: the definition, nothing else
          if (sector[b] != nb) continue;
          const float* pb = par + 7 * b;
          const int32_t rb = (int32_t)std::floor((pb[0] - p.x0_cm) / p.row_pitch_cm + 0.5f);
          const int32_t ra = (int32_t)std::floor((pa[0] - p.x0_cm) / p.row_pitch_cm + 0.5f);
          if (!(rb > first_row[a] && rb > ra)) continue;
          if (!(rb <= first_row[b])) continue;       // B's state must sit at its inner end (M7)
          if (rb < last_row[a] + 1 - p.max_row_overlap || rb > last_row[a] + 1 + p.max_row_gap) continue;
          St S = R;
          if (!transport_state(S, pb[0], p.inv_R_per_qpt, p.sin_phi_max)) continue;
          const float dy = S.y - pb[1];
          const float dz = (S.z - pb[2]) + (pa[6] - pb[6]) * p.time_bin_cm;
          const float ds = S.s - pb[3];
          const float dk = A.k - pb[5];
          if (!(std::fabs(dy) < p.cut_y_cm && std::fabs(dz) < p.cut_z_cm && std::fabs(ds) < p.cut_sin_phi &&
                std::fabs(dk) < p.cut_q_pt)) continue;
          const float d2 = (dy * dy) * c.wy + (dz * dz) * c.wz + (ds * ds) * c.ws + (dk * dk) * c.wk;
          if (out[a] < 0 || d2 < d_out[a] || (d2 == d_out[a] && (uint32_t)seed[b] < (uint32_t)seed[out[a]])) { out[a] = (int32_t)b; d_out[a] = d2; }
          if (in[b] < 0 || d2 < d_in[b] || (d2 == d_in[b] && (uint32_t)seed[a] < (uint32_t)seed[in[b]])) { in[b] = (int32_t)a; d_in[b] = d2; }
        }
      }
    }
  }
  int64_t n_links = 0;
  for (int64_t i = 0; i < n; ++i) { next[i] = -1; prev[i] = -1; }
  for (int64_t a = 0; a < n; ++a) {
    const int32_t b = out[a];
    if (b >= 0 && in[b] == (int32_t)a) { next[a] = b; prev[b] = (int32_t)a; ++n_links; }
    if (best_d2_out) best_d2_out[a] = out[a] >= 0 ? d_out[a] : -1.0f;
  }
  for (int64_t i = 0; i < n; ++i) {
    int32_t r = (int32_t)i;
    for (int steps = 0; prev[r] >= 0 && steps < 1024; ++steps) r = prev[r];   // r_B > r_A: state rows strictly increase along a chain, no cycles (the bound is never reached)
    root[i] = r;
  }
  return n_links;
}

// Pin helpers: the rotation and the state-only transport on their own.  st = (x, y, z, s, t, k).
void orc_merge_rotate(const orc_merge_params* p, float* st, int32_t side_sign) {
  const Consts c = derive(*p);
  const St A{st[0], st[1], st[2], st[3], st[4], st[5]};
  const St R = rotate(A, side_sign >= 0 ? 1.0f : -1.0f, c);
  st[0] = R.x; st[1] = R.y; st[2] = R.z; st[3] = R.s; st[4] = R.t; st[5] = R.k;
}

int orc_merge_transport(const orc_merge_params* p, float* st, float xn) {
  St S{st[0], st[1], st[2], st[3], st[4], st[5]};
  const bool ok = transport_state(S, xn, p->inv_R_per_qpt, p->sin_phi_max);
  st[0] = S.x; st[1] = S.y; st[2] = S.z; st[3] = S.s; st[4] = S.t; st[5] = S.k;
  return ok ? 1 : 0;
}

// ---- C9: time and offset at which a track passes the beam line ("t0 / vertex-z estimation from the
// time coordinate"; the z position is only known once the collision time is).  The beam axis is x = y = 0 in
// every sector frame, so the state (x; y, z, s, t, k | time_ref) is transported to x = 0 with the state part of the C5
// transport:  ok = transport(S, 0);  vertex_time = time_ref + S.z / Z  [time bins];  vertex_y = S.y  [cm].
// With time = (t0 * v_drift + drift_len - |z|) / Z this is (t0 * v_drift + drift_len - side * z_vertex) / Z for a primary
// track (side = +1 on the A side, -1 on the C side): the collision time up to the (few cm) vertex spread.  FAIL (|sin phi| would reach sin_phi_max): ok = 0, outputs 0.
// par: [n*7] as in orc_merge.  Pin (tests/test_merge_oracle_pins.py::test_MV_*): generator truth of t0 and z_vertex.
void orc_vertex_time(const orc_merge_params* p, int64_t n, const float* par, int32_t* ok, float* vertex_time, float* vertex_y) {
  for (int64_t i = 0; i < n; ++i) {
    const float* q = par + 7 * i;
    St S{q[0], q[1], q[2], q[3], q[4], q[5]};
    const bool good = transport_state(S, 0.0f, p->inv_R_per_qpt, p->sin_phi_max);
    ok[i] = good ? 1 : 0;
    vertex_time[i] = good ? q[6] + S.z / p->time_bin_cm : 0.0f;
    vertex_y[i] = good ? S.y : 0.0f;
  }
}


// ---- C10: merging across the CENTRAL ELECTRODE ("sector-boundary and central-electrode track
// merging"; the z position of a hit is only known through its time, so a track that crosses z = 0 continues in
// the mirror sector of the other TPC side with the time coordinate REFLECTED).  Readings CE1..CE6, DESIGN.md §3 "C10":
//   BASELINE.json L8/L9: sector S (A side, z > 0) and S + 18 (C side) share one local frame; time = (t0 v + L - |z|) / Z.
//   Moving outward towards the electrode |z| falls, so the time coordinate RISES (dz/ds = t > 0); behind the electrode it
//   falls again with the mirrored slope.  x, y, sin phi and q/pT are continuous.
//   For a track A (sector S, rows [f, l], state on row r_A, t_A > 0) the candidates are the tracks B of the mirror sector
//   (S + 18) mod 36 with the row window of C7:  r_B <= f_B,  r_B > max(f_A, r_A),  l_A + 1 - overlap <= r_B <= l_A + 1 + gap.
//       L = transport(A, x of row l_A)            (FAIL -> A has no candidate)
//       E = transport(L, x_B)                     (FAIL -> no candidate)
//       dy = E.y - y_B;  ds = E.s - s_B;  dk = k_A - k_B;  dt = t_A + t_B                       (mirrored slope)
//       dzm = (E.z - z_B) + (time_ref_A - time_ref_B) * Z      # A extrapolated THROUGH the electrode minus B, time-derived cm
//       zg  = E.z - L.z;   hi = zg + zg  (0 unless zg > 0)     # twice what A's z advances between its last row and x_B
//       ez  = dzm            if dzm < 0                        # the crossing must lie between A's last row and x_B:
//           = dzm - hi       if dzm > hi                       #   0 <= dzm <= hi;  ez = distance from that interval
//           = 0              otherwise
//       require |dy| < cut_y, |ez| < cut_z, |ds| < cut_s, |dk| < cut_k, |dt| < cut_t
//       d2 = (dy*dy)*wy + (ez*ez)*wz + (ds*ds)*ws + (dk*dk)*wk + (dt*dt)*wt          w = (float)(1 / cut^2), from double
//   Reciprocal best match exactly as in C7 (ties -> lowest seed id).  For a linked A:
//       cl = min(max(dzm, 0), hi);   t_ce[A] = time_ref_B + (z_B + 0.5f*cl) / Z       # time coordinate of the crossing
//   = (t0 v + L) / Z: the collision time itself, with no vertex assumption.  Unlinked tracks: t_ce = 0.
// Pins (tests/test_merge_oracle_pins.py): CE-L closed form on hand-made mirrored lines (link, t_ce), CE-S the sign and
// mirror conditions, CE-H noise-free helices through the electrode against generator truth, CE-T t_ce against the
// generator's t0, CE-I invariants, CE-P order independence.  Parity unpinned: the values of the cuts.
struct orc_ce_params {
  int32_t n_sectors, n_rows;
  float x0_cm, row_pitch_cm, time_bin_cm, sin_phi_max, inv_R_per_qpt;
  float cut_y_cm, cut_z_cm, cut_sin_phi, cut_q_pt, cut_dzds;
  int32_t max_row_gap, max_row_overlap;
};

int64_t orc_merge_ce(const orc_ce_params* pp, int64_t n, const int32_t* seed, const int32_t* sector, const int32_t* first_row,
                     const int32_t* last_row, const float* par, int32_t* next, int32_t* prev, float* t_ce) {
  const orc_ce_params& p = *pp;
  const float wy = (float)(1.0 / ((double)p.cut_y_cm * (double)p.cut_y_cm)), wz = (float)(1.0 / ((double)p.cut_z_cm * (double)p.cut_z_cm));
  const float ws = (float)(1.0 / ((double)p.cut_sin_phi * (double)p.cut_sin_phi)), wk = (float)(1.0 / ((double)p.cut_q_pt * (double)p.cut_q_pt));
  const float wt = (float)(1.0 / ((double)p.cut_dzds * (double)p.cut_dzds));
  std::vector<int32_t> out(n, -1), in(n, -1);
  std::vector<float> d_out(n, 0.0f), d_in(n, 0.0f), t_out(n, 0.0f);
  if (p.n_sectors == 36) {
    for (int64_t a = 0; a < n; ++a) {
      const float* pa = par + 7 * a;
      if (!(pa[4] > 0.0f)) continue;                                    // CE2: only a track approaching the electrode can cross it
      St L{pa[0], pa[1], pa[2], pa[3], pa[4], pa[5]};
      const float x_l = (float)((double)p.x0_cm + (double)p.row_pitch_cm * (double)last_row[a]);
      if (!transport_state(L, x_l, p.inv_R_per_qpt, p.sin_phi_max)) continue;
      const int32_t ra = (int32_t)std::floor((pa[0] - p.x0_cm) / p.row_pitch_cm + 0.5f);
      const int32_t nb = (sector[a] + 18) % 36;
      for (int64_t b = 0; b < n; ++b) {
        if (sector[b] != nb) continue;
        const float* pb = par + 7 * b;
        const int32_t rb = (int32_t)std::floor((pb[0] - p.x0_cm) / p.row_pitch_cm + 0.5f);
        if (!(rb > first_row[a] && rb > ra)) continue;
        if (!(rb <= first_row[b])) continue;
        if (rb < last_row[a] + 1 - p.max_row_overlap || rb > last_row[a] + 1 + p.max_row_gap) continue;
        St E = L;
        if (!transport_state(E, pb[0], p.inv_R_per_qpt, p.sin_phi_max)) continue;
        const float dy = E.y - pb[1];
        const float ds = E.s - pb[3];
        const float dk = pa[5] - pb[5];
        const float dt = pa[4] + pb[4];
        const float dzm = (E.z - pb[2]) + (pa[6] - pb[6]) * p.time_bin_cm;
        const float zg = E.z - L.z;
        const float hi = zg > 0.0f ? zg + zg : 0.0f;
        const float ez = dzm < 0.0f ? dzm : (dzm > hi ? dzm - hi : 0.0f);
        if (!(std::fabs(dy) < p.cut_y_cm && std::fabs(ez) < p.cut_z_cm && std::fabs(ds) < p.cut_sin_phi && std::fabs(dk) < p.cut_q_pt &&
              std::fabs(dt) < p.cut_dzds)) continue;
        const float d2 = (dy * dy) * wy + (ez * ez) * wz + (ds * ds) * ws + (dk * dk) * wk + (dt * dt) * wt;
        const float cl = std::fmin(std::fmax(dzm, 0.0f), hi);
        const float tce = pb[6] + (pb[2] + 0.5f * cl) / p.time_bin_cm;
        if (out[a] < 0 || d2 < d_out[a] || (d2 == d_out[a] && (uint32_t)seed[b] < (uint32_t)seed[out[a]])) { out[a] = (int32_t)b; d_out[a] = d2; t_out[a] = tce; }
        if (in[b] < 0 || d2 < d_in[b] || (d2 == d_in[b] && (uint32_t)seed[a] < (uint32_t)seed[in[b]])) { in[b] = (int32_t)a; d_in[b] = d2; }
      }
    }
  }
  int64_t n_links = 0;
  for (int64_t i = 0; i < n; ++i) { next[i] = -1; prev[i] = -1; t_ce[i] = 0.0f; }
  for (int64_t a = 0; a < n; ++a) {
    const int32_t b = out[a];
    if (b >= 0 && in[b] == (int32_t)a) { next[a] = b; prev[b] = (int32_t)a; t_ce[a] = t_out[a]; ++n_links; }
  }
  return n_links;
}

}  // extern "C"
