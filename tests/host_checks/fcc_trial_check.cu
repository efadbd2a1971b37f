// Host-side check of the trial arithmetic of the packed FCC kernel (sweep_fcc.cuh: fcc_trial is __host__ __device__).
// Every trial is compared with a brute-force energy difference computed from the species at their positions in a
// random 8x8x8-cell tile (shells generated here from the definition S0: FCC translations by squared length, ascending
// (dz, dy, dx)), the integer form of Eq. 3 and an explicit swap.  Shares nothing with oracle/.
// Built and run by tests/test_thread_kernel_host.py with nvcc as a host program (no GPU needed).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <random>
#include <vector>
#include "../../paper_2509_20949_b200/csrc/sweep_fcc.cuh"
using namespace smcxk;
#ifndef __CUDA_ARCH__

struct Off { int x, y, z; };
static std::vector<std::vector<Off>> g_shell;   // [s] offsets
static int V[3][8][8];
static const int kBeta[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};

static void make_shells() {
  const int d2s[3] = {2, 4, 6};
  for (int s = 0; s < 3; ++s) {
    std::vector<Off> v;
    for (int z = -3; z <= 3; ++z) for (int y = -3; y <= 3; ++y) for (int x = -3; x <= 3; ++x)
      if (((x + y + z) & 1) == 0 && x * x + y * y + z * z == d2s[s]) v.push_back({x, y, z});
    g_shell.push_back(v);
  }
}
// tile word (sub * 64 + y + 8 z), nibble X
static int spec_pos(const uint32_t* tile, int px, int py, int pz) {
  const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
  const int b = par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : par == 3 ? 3 : -1;
  if (b < 0) { printf("not a lattice site\n"); exit(1); }
  const int X = px >> 1, y = py >> 1, z = pz >> 1;
  if (X < 0 || X > 7 || y < 0 || y > 7 || z < 0 || z > 7) { printf("outside the tile\n"); exit(1); }
  return (tile[b * 64 + y + 8 * z] >> (4 * X)) & 15;
}
static void set_pos(uint32_t* tile, int px, int py, int pz, int s) {
  const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
  const int b = par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3;
  uint32_t& w = tile[b * 64 + (py >> 1) + 8 * (pz >> 1)];
  w = (w & ~(15u << (4 * (px >> 1)))) | ((uint32_t)s << (4 * (px >> 1)));
}
static long long local_energy(const uint32_t* tile, int n_shells, const int p[3], const int q[3]) {
  long long e = 0;
  const int sp = spec_pos(tile, p[0], p[1], p[2]), sq = spec_pos(tile, q[0], q[1], q[2]);
  for (int s = 0; s < n_shells; ++s)
    for (const Off& o : g_shell[s]) {
      e += V[s][sp][spec_pos(tile, p[0] + o.x, p[1] + o.y, p[2] + o.z)];
      const int x = q[0] + o.x, y = q[1] + o.y, z = q[2] + o.z;
      if (x == p[0] && y == p[1] && z == p[2]) continue;     // the p-q bond once
      e += V[s][sq][spec_pos(tile, x, y, z)];
    }
  return e;
}

template <int F>
static void run_trial(int b, uint32_t* p_own, uint32_t X4, const FccDirEntry& E, uint32_t u, const FccEnv& env, int& es, unsigned& na) {
  switch (b) {
    case 0: fcc_trial<0, 1, F>(p_own, X4, E, u, env, es, na); break;
    case 1: fcc_trial<1, 1, F>(p_own, X4, E, u, env, es, na); break;
    case 2: fcc_trial<2, 1, F>(p_own, X4, E, u, env, es, na); break;
    default: fcc_trial<3, 1, F>(p_own, X4, E, u, env, es, na); break;
  }
}

int main() {
  make_shells();
  if (g_shell[0].size() != 12 || g_shell[1].size() != 6 || g_shell[2].size() != 24) { printf("bad shells\n"); return 1; }
  std::mt19937 rng(4242);
  const int kT = 690;
  const int len = (int)std::floor(32.0 * std::log(2.0) * kT) + 2;
  std::vector<uint32_t> T(len);
  for (int d = 0; d < len; ++d) { double x = std::exp(-(double)d / kT) * 4294967296.0; T[d] = x >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)std::floor(x); }
  alignas(16) static uint32_t filt[kFilterWords];
  int nq; const int Ef = build_accept_filter(T.data(), len, filt, &nq);
  printf("len %d filter E %d nq %d\n", len, Ef, nq);
  Geom G; memset(&G, 0, sizeof(G));
  G.Z0 = 12;
  for (int d = 0; d < 12; ++d) { G.off[d][0] = (signed char)g_shell[0][d].x; G.off[d][1] = (signed char)g_shell[0][d].y; G.off[d][2] = (signed char)g_shell[0][d].z; }
  FccTables FT;
  if (!fcc_build_tables<1>(G, FT)) { printf("table build failed\n"); return 1; }
  long long n_checked = 0, n_acc = 0, n_rare = 0, bad = 0;
  for (int rep = 0; rep < 300; ++rep) {
    const int nsp = 2 + rep % 7, n_shells = 2 + (rep % 5 != 0);
    const int amp = rep % 9 == 0 ? 15000 : 400;
    for (int s = 0; s < 3; ++s) for (int a = 0; a < 8; ++a) for (int b = a; b < 8; ++b)
      V[s][a][b] = V[s][b][a] = (int)(rng() % (2 * amp + 1)) - amp;
    std::vector<int32_t> epi((size_t)n_shells * nsp * nsp);
    for (int s = 0; s < n_shells; ++s) for (int a = 0; a < nsp; ++a) for (int b = 0; b < nsp; ++b) epi[(s * nsp + a) * nsp + b] = V[s][a][b];
    std::vector<uint32_t> lut; std::vector<int32_t> corr;
    const int lrep = 1 + rep % 2;
    if (!fcc_build_lut(epi.data(), nsp, n_shells, lrep, lut, corr)) { printf("lut build failed\n"); return 1; }
    std::vector<uint32_t> lut_al(lut.size() + 4);
    uint32_t* lut_p = lut_al.data(); while (((uintptr_t)lut_p) & 15) ++lut_p;
    memcpy(lut_p, lut.data(), lut.size() * 4);
    FccEnv env;
    env.lut = smem_ptr(lut_p) + (rep % lrep) * 16; env.corr = smem_ptr(corr.data()); env.filt = smem_ptr(filt);
    env.lut_pair_bytes = 3u * lrep * 16u; env.lut_shell_bytes = lrep * 16u;
    env.accept = T.data(); env.accept_len = len; env.filter_E = Ef; env.direct_len = 0;
    // MODE 2: the first K entries of T and the bound T[K] in "shared memory" (K = len: the whole table and a zero)
    const int K = rep % 3 == 0 ? len : 1 + (int)(rng() % (uint32_t)len);
    std::vector<uint32_t> direct((size_t)K + 1);
    for (int d = 0; d <= K; ++d) direct[d] = d < len ? T[d] : 0u;
    FccEnv env2 = env;
    env2.filt = smem_ptr(direct.data()); env2.direct_len = K;
    uint32_t tile[256];
    for (auto& w : tile) { w = 0; for (int f = 0; f < 8; ++f) w |= (uint32_t)(rng() % nsp) << (4 * f); }
    for (int it = 0; it < 3000; ++it) {
      const int b = rng() & 3, X = 2 + (rng() & 3), y = 2 + (rng() & 3), z = 2 + (rng() & 3);
      const uint32_t w_dir = rng();
      const int dir = (int)(((uint64_t)w_dir * 12u) >> 32);
      const int p[3] = {2 * X + kBeta[b][0], 2 * y + kBeta[b][1], 2 * z + kBeta[b][2]};
      const Off& o = g_shell[0][dir];
      const int q[3] = {p[0] + o.x, p[1] + o.y, p[2] + o.z};
      uint32_t ref[256]; memcpy(ref, tile, sizeof(tile));
      const int sa = spec_pos(ref, p[0], p[1], p[2]), sb = spec_pos(ref, q[0], q[1], q[2]);
      long long dEref = 0; bool okref = false;
      uint32_t u = rng();
      if (sa != sb) {
        const long long e0 = local_energy(ref, n_shells, p, q);
        set_pos(ref, p[0], p[1], p[2], sb); set_pos(ref, q[0], q[1], q[2], sa);
        const long long e1 = local_energy(ref, n_shells, p, q);
        dEref = e1 - e0;
        if (it % 5 == 0 && dEref > 0 && dEref < len) { u = T[dEref] + (uint32_t)((int)(rng() % 7) - 3); ++n_rare; }
        if (it % 11 == 0 && dEref <= 0) u = 0xFFFFFFFFu - (rng() % 3);
        okref = dEref <= 0 || (dEref < len && u < T[dEref]);
        if (!okref) memcpy(ref, tile, sizeof(tile));
      } else if (it % 3 == 0) u = rng() % 4;
      for (int variant = 0; variant < 3; ++variant) {
        uint32_t got[256]; memcpy(got, tile, sizeof(tile));
        int es = 0; unsigned na = 0;
        uint32_t* p_own = got + b * 64 + y + 8 * z;
        if (variant == 0) run_trial<1>(b, p_own, 4u * X, FT.dir[b][dir], u, env, es, na);
        else if (variant == 1) run_trial<0>(b, p_own, 4u * X, FT.dir[b][dir], u, env, es, na);
        else run_trial<2>(b, p_own, 4u * X, FT.dir[b][dir], u, env2, es, na);
        const bool same = memcmp(got, ref, sizeof(ref)) == 0;
        if (!same || na != (okref ? 1u : 0u) || es != (okref ? (int)dEref : 0)) {
          if (bad < 10) printf("MISMATCH variant %d b %d X %d y %d z %d dir %d a %d b %d dEref %lld okref %d got es %d na %u same %d u %u nsp %d shells %d\n",
                               variant, b, X, y, z, dir, sa, sb, dEref, (int)okref, es, na, (int)same, u, nsp, n_shells);
          ++bad;
        }
      }
      memcpy(tile, ref, sizeof(tile));
      ++n_checked; n_acc += okref;
    }
  }
  printf("checked %lld trials, accepted %lld, forced-near-threshold %lld, mismatches %lld\n", n_checked, n_acc, n_rare, bad);
  return bad != 0;
}
#endif
