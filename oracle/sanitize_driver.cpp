// sanitize_driver.cpp — runs the CPU oracle (R0..R6, R8, R9, R10) once on a frame read from a file,
// for a build under -fsanitize=address,undefined (the oracle is checked for
// memory errors and undefined behaviour).  TEST INFRASTRUCTURE: built and run by
// tests/test_oracle_sanitizers.py only.  Input file: n (uint64) followed by n 16-byte cluster records.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "tpc_oracle.h"

int main(int argc, char** argv) {
  if (argc < 2) return 2;
  FILE* f = std::fopen(argv[1], "rb");
  if (!f) return 2;
  uint64_t n = 0;
  if (std::fread(&n, 8, 1, f) != 1) return 2;
  std::vector<orc_cluster> cl(n);
  if (n && std::fread(cl.data(), sizeof(orc_cluster), n, f) != n) return 2;
  std::fclose(f);
  orc_geom g = {36, 152, 63, 85.0f, 245.0f, 0.4f, 0.6f, 250.0f, 0.5f, 10.0f};
  orc_params P;
  orc_default_params(&P);
  orc_result* r = orc_run(cl.data(), n, &g, &P, 0, 36, 2);
  if (!r) return 3;
  uint64_t sz[10];
  orc_sizes(r, sz);
  std::vector<orc_track> tracks(sz[4]);
  std::vector<uint32_t> ids(sz[5]);
  std::vector<uint8_t> sh(sz[5]);
  orc_fetch_tracks(r, tracks.data(), ids.data(), sh.data());
  std::vector<int32_t> up(n), dn(n), up2(n), dn2(n);
  orc_fetch_links(r, up.data(), dn.data(), up2.data(), dn2.data());
  std::vector<orc_tracklet> tl(sz[3]);
  std::vector<int32_t> rh(sz[3] * 152);
  orc_fetch_tracklets(r, tl.data(), rh.data());
  // R8 refit -> R9 merging input
  std::vector<orc_merge_track> mt(tracks.size());
  for (size_t k = 0; k < tracks.size(); ++k) {
    const orc_track& t = tracks[k];
    std::vector<int32_t> rows(t.n_clusters);
    std::vector<float> y(t.n_clusters), z(t.n_clusters);
    for (int i = 0; i < t.n_clusters; ++i) {
      const orc_cluster& c = cl[ids[t.cluster_ofs + i]];
      rows[i] = c.row; y[i] = c.y; z[i] = c.z;
    }
    float st[48];
    const float chi2 = orc_refit_hits(&g, &P, rows.data(), y.data(), z.data(), t.n_clusters, st);
    orc_merge_track& m = mt[k];
    std::memset(&m, 0, sizeof(m));
    m.sector = t.sector; m.row_first = t.row_first; m.row_last = t.row_last; m.valid = chi2 >= 0;
    m.seed_id = t.seed_id; m.segment = t.segment; m.iter = 0;
    if (m.valid) {
      std::memcpy(m.p_in, st + 1, 20); std::memcpy(m.c_in, st + 6, 60);
      std::memcpy(m.p_out, st + 23, 20); std::memcpy(m.c_out, st + 28, 60);
    }
  }
  std::vector<int32_t> next(mt.size()), prev(mt.size());
  std::vector<float> lchi(mt.size());
  const int n_links = orc_merge_links(&g, &P, nullptr, mt.data(), (int32_t)mt.size(), next.data(), prev.data(), lchi.data());
  // R10 on every chain
  int n_fit = 0, n_rej = 0;
  for (size_t h = 0; h < mt.size(); ++h) {
    if (prev[h] >= 0) continue;
    std::vector<int32_t> sec, rows;
    std::vector<float> y, z;
    int32_t tail = (int32_t)h;
    for (int32_t k = (int32_t)h; k >= 0; k = next[k]) {
      const orc_track& t = tracks[k];
      for (int i = 0; i < t.n_clusters; ++i) {
        const orc_cluster& c = cl[ids[t.cluster_ofs + i]];
        sec.push_back(c.sector); rows.push_back(c.row); y.push_back(c.y); z.push_back(c.z);
      }
      tail = k;
    }
    if (!mt[tail].valid) continue;
    std::vector<float> chi(rows.size());
    std::vector<uint8_t> rej(rows.size());
    float out[24];
    int32_t n_used = 0;
    const float c2 = orc_fit_track(&g, &P, nullptr, sec.data(), rows.data(), y.data(), z.data(), (int)rows.size(),
                                   mt[tail].p_out + 2, out, chi.data(), rej.data(), &n_used);
    n_fit += c2 >= 0;
    for (uint8_t v : rej) n_rej += v;
  }
  std::printf("clusters %llu seeds %llu tracks %llu links %d fits %d rejected %d\n", (unsigned long long)n,
              (unsigned long long)sz[3], (unsigned long long)sz[4], n_links, n_fit, n_rej);
  orc_free(r);
  return 0;
}
