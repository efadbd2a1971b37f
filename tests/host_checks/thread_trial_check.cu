// Host-side check of the trial arithmetic of the thread-per-cell kernel (sweep_thread.cuh:
// trial_thread is __host__ __device__).  Every trial is compared with a brute-force energy
// difference computed from the unpacked species of a random 8x8x8 tile, the integer form of Eq. 3
// and an explicit swap.  Shares nothing with oracle/.  Built and run by
// tests/test_thread_kernel_host.py with nvcc as a host program (no GPU needed).
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <vector>
#include <random>
#include "../../paper_2509_20949_b200/csrc/sweep_thread.cuh"
using namespace smcxk;
#ifndef __CUDA_ARCH__

static int V[2][4][4];
static int spec(const uint32_t* tile, int x, int y, int z, int b) { return (tile[z * 8 + y] >> (4 * x + 2 * b)) & 3; }
static void setspec(uint32_t* tile, int x, int y, int z, int b, int s) {
  uint32_t& w = tile[z * 8 + y]; w = (w & ~(3u << (4 * x + 2 * b))) | ((uint32_t)s << (4 * x + 2 * b));
}
// half-unit position -> (cell, b)
static int spec_pos(const uint32_t* tile, int px, int py, int pz) {
  int b = px & 1; return spec(tile, (px - b) / 2, (py - b) / 2, (pz - b) / 2, b);
}
static long long local_energy(const uint32_t* tile, int px, int py, int pz, int qx, int qy, int qz) {
  // sum of all bonds touching p or q (bond p-q once)
  long long e = 0;
  static const int o1[8][3] = {{-1,-1,-1},{1,-1,-1},{-1,1,-1},{1,1,-1},{-1,-1,1},{1,-1,1},{-1,1,1},{1,1,1}};
  static const int o2[6][3] = {{0,0,-2},{0,-2,0},{-2,0,0},{2,0,0},{0,2,0},{0,0,2}};
  int sp = spec_pos(tile, px, py, pz), sq = spec_pos(tile, qx, qy, qz);
  for (auto& o : o1) { e += V[0][sp][spec_pos(tile, px + o[0], py + o[1], pz + o[2])]; }
  for (auto& o : o2) { e += V[1][sp][spec_pos(tile, px + o[0], py + o[1], pz + o[2])]; }
  for (auto& o : o1) { int x = qx + o[0], y = qy + o[1], z = qz + o[2]; if (x == px && y == py && z == pz) continue; e += V[0][sq][spec_pos(tile, x, y, z)]; }
  for (auto& o : o2) { int x = qx + o[0], y = qy + o[1], z = qz + o[2]; if (x == px && y == py && z == pz) continue; e += V[1][sq][spec_pos(tile, x, y, z)]; }
  return e;
}

// F: kAcceptGlobal / kAcceptFilter (filt = two-level tables) / kAcceptDirect (filt = T followed by one zero entry)
template <int F, bool PK = false>
static void run_trial(int bi, int X, uint32_t* p, const char* cb, const uint32_t* filt, const uint32_t* T, int len, int E,
                      uint32_t w, uint32_t u, int& es, unsigned& na) {
  TrialEnv env; env.coef = smem_ptr(cb); env.filt = smem_ptr(filt); env.accept = T; env.accept_len = len; env.filter_E = E;
  env.tmax4 = 4u * (uint32_t)len;
  static Geom G; static bool init = false; if (!init) { G.key0 = 1; G.key1 = 2; set_thread_masks(G); init = true; }
  uint32_t ra = bi ? p[1] : p[-1], rb = bi ? p[8] : p[-8];
  const uint32_t era = bi ? p[-1] : p[1], erb = bi ? p[-8] : p[8];
#define C(B, XX) if (bi == B && X == XX) { trial_thread<B, XX, F, 1, PK>(G, p, env, w, u, ra, rb, es, na); if (ra != era || rb != erb) { printf("row carry mismatch\n"); exit(1);} es /= 4; return; }
  C(0,2) C(0,3) C(0,4) C(0,5) C(1,2) C(1,3) C(1,4) C(1,5)
#undef C
}

int main() {
  std::mt19937 rng(12345);
  const int kT = 600;
  const int len = (int)std::floor(32.0 * std::log(2.0) * kT) + 2;
  std::vector<uint32_t> T(len);
  for (int d = 0; d < len; ++d) { double x = std::exp(-(double)d / kT) * 4294967296.0; T[d] = x >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)std::floor(x); }
  std::vector<uint32_t> Tz(T); Tz.push_back(0u);   // the table as the persistent kernel keeps it in shared memory
  std::vector<uint32_t> filt(kFilterWords);
  int nq; const int E = build_accept_filter(T.data(), len, filt.data(), &nq);
  printf("len %d filter E %d nq %d\n", len, E, nq);
  long long n_packed = 0, n_over = 0, n_checked = 0, n_acc = 0, n_rare = 0, bad = 0;
  for (int rep = 0; rep < 400; ++rep) {
    const int nsp = 2 + rep % 3;
    for (int s = 0; s < 2; ++s) for (int a = 0; a < 4; ++a) for (int b = a; b < 4; ++b) {
      int v = (int)(rng() % 601) - 300; if (rep % 7 == 0) v = (int)(rng() % 20001) - 10000;
      V[s][a][b] = V[s][b][a] = v;
    }
    int epi[2 * 4 * 4];
    for (int s = 0; s < 2; ++s) for (int a = 0; a < nsp; ++a) for (int b = 0; b < nsp; ++b) epi[(s * nsp + a) * nsp + b] = V[s][a][b];
    alignas(16) int32_t coef[16 * kCoefInts];
    const int cls = build_thread_coefficients(epi, nsp, coef); if (cls == 0) { printf("overflow\n"); return 1; } if (cls == 1) ++n_over;
    // layout expected by the kernel: [ent][8 slots] int4 x 2 halves: coef_base + a4*32 + b4*8 -> (a*4+b)*128 bytes; second half at +2048
    alignas(16) static int32_t tab[2 * 16 * 8 * 4];
    for (int ent = 0; ent < 16; ++ent) for (int slot = 0; slot < 8; ++slot) for (int k = 0; k < 4; ++k) {
      tab[(ent * 8 + slot) * 4 + k] = coef[ent * 8 + k];
      tab[512 + (ent * 8 + slot) * 4 + k] = coef[ent * 8 + 4 + k];
    }
    // packed 16-bit rows of the persistent kernel: [ent][8 slots] int4
    int32_t pk[16 * 4];
    const bool packable = pack_thread_coefficients(coef, pk);
    alignas(16) static int32_t tabpk[16 * 8 * 4];
    for (int ent = 0; ent < 16; ++ent) for (int slot = 0; slot < 8; ++slot) for (int k = 0; k < 4; ++k)
      tabpk[(ent * 8 + slot) * 4 + k] = pk[ent * 4 + k];
    if (packable) ++n_packed;
    uint32_t tile[64];
    for (auto& w : tile) { w = 0; for (int f = 0; f < 16; ++f) w |= (uint32_t)(rng() % nsp) << (2 * f); }
    for (int it = 0; it < 3000; ++it) {
      const int bi = rng() & 1, X = 2 + (rng() & 3), y = 2 + (rng() & 3), z = 2 + (rng() & 3);
      const uint32_t w = rng();
      const int dir = w >> 29, dx = dir & 1, dy = (dir >> 1) & 1, dz = dir >> 2;
      const int px = 2 * X + bi, py = 2 * y + bi, pz = 2 * z + bi;
      const int qx = px + 2 * dx - 1, qy = py + 2 * dy - 1, qz = pz + 2 * dz - 1;
      uint32_t ref[64]; memcpy(ref, tile, sizeof(tile));
      const int a = spec_pos(ref, px, py, pz), b = spec_pos(ref, qx, qy, qz);
      long long dEref = 0; bool okref = false;
      uint32_t u = rng();
      if (a != b) {
        const long long e0 = local_energy(ref, px, py, pz, qx, qy, qz);
        const int bb = px & 1;
        setspec(ref, (px - bb) / 2, (py - bb) / 2, (pz - bb) / 2, bb, b);
        const int qb = qx & 1;
        setspec(ref, (qx - qb) / 2, (qy - qb) / 2, (qz - qb) / 2, qb, a);
        const long long e1 = local_energy(ref, px, py, pz, qx, qy, qz);
        dEref = e1 - e0;
        if (it % 5 == 0 && dEref > 0 && dEref < len) { u = T[dEref] + (uint32_t)((int)(rng() % 7) - 3); ++n_rare; }
        if (it % 11 == 0 && dEref <= 0) u = 0xFFFFFFFFu - (rng() % 3);
        okref = dEref <= 0 || (dEref < len && u < T[dEref]);
        if (!okref) memcpy(ref, tile, sizeof(tile));
      } else if (it % 3 == 0) u = rng() % 4;
      for (int variant = (cls == 2 ? 0 : 1); variant < (packable ? 4 : 3); ++variant) {
        uint32_t got[64]; memcpy(got, tile, sizeof(tile));
        int es = 0; unsigned na = 0;
        uint32_t* p = got + z * 8 + y;
        const char* cb = reinterpret_cast<const char*>(tab) + (it & 7) * 16;
        if (variant == 0) run_trial<kAcceptFilter>(bi, X, p, cb, filt.data(), T.data(), len, E, w, u, es, na);
        else if (variant == 1) run_trial<kAcceptGlobal>(bi, X, p, cb, filt.data(), T.data(), len, E, w, u, es, na);
        else if (variant == 2) run_trial<kAcceptDirect>(bi, X, p, cb, Tz.data(), T.data(), len, E, w, u, es, na);
        else run_trial<kAcceptDirect, true>(bi, X, p, reinterpret_cast<const char*>(tabpk) + (it & 7) * 16, Tz.data(), T.data(), len, E, w, u, es, na);
        const bool same = memcmp(got, ref, sizeof(ref)) == 0;
        if (!same || na != (okref ? 1u : 0u) || es != (okref ? (int)dEref : 0)) {
          if (bad < 10) printf("MISMATCH variant %d bi %d X %d y %d z %d dir %d a %d b %d dEref %lld okref %d got es %d na %u same %d u %u\n",
                               variant, bi, X, y, z, dir, a, b, dEref, (int)okref, es, na, (int)same, u);
          ++bad;
        }
      }
      memcpy(tile, ref, sizeof(tile));
      ++n_checked; n_acc += okref;
    }
  }
  printf("packed-coefficient reps %lld, coef-overflow reps %lld; checked %lld trials, accepted %lld, forced-near-threshold %lld, mismatches %lld\n", n_packed, n_over, n_checked, n_acc, n_rare, bad);
  return bad != 0;
}
#endif
