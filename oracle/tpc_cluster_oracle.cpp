// ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain single-threaded C++ fp32 CPU implementation of step C0: the TPC CLUSTER FINDER
// that turns zero-suppressed ADC samples into the clusters the tracker reads ("the step before the
// path"; PAPER.md L43 (§3): TPC clusterization is part of the synchronous GPU load; zero suppression happens in
// the readout, so only samples above threshold arrive).
//
// The paper names the step and gives no algorithm, so every definition is a reading of this build, listed as D1..D6 in
// DESIGN.md §3 ("C0").  It is a local-maximum finder followed by a 3 x 3 centre of gravity, followed step by step:
//   A sample d = (sector_row, pad, time bin, adc).  Input: samples sorted by (sector_row, time bin, pad), no duplicates (D1).
//   N(d) = the samples of the same sector_row with |pad - pad_d| <= 1 and |time - time_d| <= 1, d excluded (D2).
//   d BEATS e  iff  adc_d > adc_e  or  (adc_d == adc_e and d comes before e in the input order) (D3).
//   d is a PEAK iff adc_d >= peak_threshold and d beats every e in N(d) (D4).
//   Cluster of a peak d, all fp32, one rounded operation per statement, in this order (D5):
//       q = 0; sp = 0; st = 0
//       for dt in (-1, 0, +1): for dp in (-1, 0, +1): if the sample (pad_d + dp, time_d + dt) exists with adc a:
//           q = q + a;  sp = sp + (float)dp * a;  st = st + (float)dt * a
//       pad = (float)pad_d + sp / q;   time = (float)time_d + st / q;   charge = q;   row = (float)sector_row
//   Clusters are emitted in the input order of their peaks (D6).  Neighbouring clusters share samples (no splitting).
// Pins (tests/test_cluster_oracle_pins.py): D-C closed form of the centroid of one isolated deposit, D-B a dense-array
// restatement on tiny frames, D-T the tie rule on plateaus, D-I invariants (no two peaks are neighbours, charge bookkeeping),
// D-E generated clusters -> samples -> clusters recovers the isolated ones (position resolution, efficiency).
// Parity unpinned: the threshold values.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this.  It shares no code,
// header, table or constant generator with the CUDA path.
#include <cstdint>
#include <unordered_map>
#include <vector>

extern "C" {

struct orc_cf_result {
  std::vector<float> row, pad, time, charge;
  std::vector<int64_t> peak;      // input index of the peak sample of each cluster
};

int orc_find_clusters(int64_t n, const int32_t* row, const int32_t* pad, const int32_t* time, const float* adc, float peak_threshold,
                      orc_cf_result** out) {
  if (!out || n < 0 || (n > 0 && (!row || !pad || !time || !adc))) return -1;
  std::unordered_map<uint64_t, int64_t> at;
  at.reserve((size_t)n * 2);
  auto key = [](int32_t r, int32_t p, int32_t t) { return ((uint64_t)(uint32_t)r << 44) | ((uint64_t)(uint32_t)(t + 1) << 12) | (uint64_t)(uint32_t)(p + 1); };
  for (int64_t i = 0; i < n; ++i) {
    if (i > 0) {                                     // D1: the input contract
      const bool ordered = row[i - 1] < row[i] || (row[i - 1] == row[i] && (time[i - 1] < time[i] || (time[i - 1] == time[i] && pad[i - 1] < pad[i])));
      if (!ordered) return -2;
    }
    if (pad[i] < 0 || pad[i] > 4000 || time[i] < 0 || row[i] < 0) return -2;
    at[key(row[i], pad[i], time[i])] = i;
  }
  orc_cf_result* R = new orc_cf_result();
  for (int64_t d = 0; d < n; ++d) {
    if (!(adc[d] >= peak_threshold)) continue;
    bool peak = true;
    float q = 0.0f, sp = 0.0f, st = 0.0f;
    for (int dt = -1; dt <= 1 && peak; ++dt)
      for (int dp = -1; dp <= 1; ++dp) {
        const auto it = at.find(key(row[d], pad[d] + dp, time[d] + dt));
        if (it == at.end()) continue;
        const int64_t e = it->second;
        const float a = adc[e];
        if (e != d && !(adc[d] > a || (adc[d] == a && d < e))) { peak = false; break; }
        q = q + a;
        sp = sp + (float)dp * a;
        st = st + (float)dt * a;
      }
    if (!peak) continue;
    R->row.push_back((float)row[d]);
    R->pad.push_back((float)pad[d] + sp / q);
    R->time.push_back((float)time[d] + st / q);
    R->charge.push_back(q);
    R->peak.push_back(d);
  }
  *out = R;
  return 0;
}
int64_t orc_cf_n(const orc_cf_result* r) { return (int64_t)r->peak.size(); }
void orc_cf_copy(const orc_cf_result* r, float* row, float* pad, float* time, float* charge, int64_t* peak) {
  for (size_t i = 0; i < r->peak.size(); ++i) { row[i] = r->row[i]; pad[i] = r->pad[i]; time[i] = r->time[i]; charge[i] = r->charge[i]; peak[i] = r->peak[i]; }
}
void orc_cf_free(orc_cf_result* r) { delete r; }

}  // extern "C"
