// Sub-warp colour-pass kernel: L lanes (4, 8, 16 or 32) per link cell, uint8 species, any lattice /
// shell list / link-cell size ("sub-warp variants of the same path").
//
// Same steps a1-a8 and the same schedule as sweep_warp_per_cell, arranged for a short chain of
// instructions per trial (a lattice with few cells per colour, such as BASELINE.json's FCC 128^3, is bound
// by the latency of one cell's chain of 256 dependent trials):
//  * the serial part of a trial (slot -> site, direction, species of i and j, acceptance) is replicated
//    over L lanes instead of 32, and 32 / L cells share a warp;
//  * the tile index of a site is LINEAR in its position, (px + A py + B pz) >> shift in units of a/2 (see
//    below), so the tile-index step to neighbour m is the same for every site whatever its basis: lane g
//    keeps the steps and the table rows of its neighbours (slots g, g + L, ... of G.gslot) in registers,
//    and a neighbour visit is one add, the species load, one add and the load of
//    D[(a,b)][s][x] = V_s(b,x) - V_s(a,x) from a table the host builds once (group_build_table) and every
//    block copies into shared memory.
//    The sums over the neighbours of i and of j both include the i-j bond;
//    corr(a,b) = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) takes it out again (exact integer identity);
//  * the partial dE of the lanes are summed by one whole-warp REDUX per cell of the warp with 16 or 32 lanes
//    (the other cells' lanes contribute 0), by an xor-shuffle tree with fewer;
//  * Philox: lane g of a group computes the call of slot pair q0 + g, so a group draws 2 L slots at a
//    time, looks the tile step of the drawn direction up right away (off the chain of dependent trials)
//    and hands step and acceptance draw round with group-wide shuffles;
//  * control flow is uniform over the warp (a trial between equal species is computed and masked; a lane
//    with fewer neighbours than the others visits the two sites themselves with the row of shell 0: a term that
//    depends on the pair (a,b) only and is taken out of corr(a,b) when the table is built), so the 32 / L cells of a warp never
//    serialise, and the acceptance test reads the two-level filter tables in shared memory (see
//    sweep_thread.cuh; the exact table in global memory only when u falls within E of the bound).
// Results are bit-identical to the other kernels (tests/test_gpu_parity.py).
#pragma once
#include <mutex>
#include <vector>
#include "smcx_common.cuh"
#include "sweep_thread.cuh"   // two-level acceptance filter (kFilterTr, kFilterWords, build_accept_filter)
#include "sweep_warp.cuh"

namespace smcxk {

#ifndef SMCX_GROUP_REDUX_MIN_LANES
#define SMCX_GROUP_REDUX_MIN_LANES 16   // measured: 16 lanes 0.866 -> 0.772 ms per sweep of FCC 128^3, 8 lanes 0.949 -> 1.003
#endif
constexpr int kGroupWarpsPerBlock = 8;    // at most; group_warps_per_block() picks fewer when that lets more blocks share an SM
// Tile layout in shared memory: the species of the site at position (px, py, pz) (units of a/2, tile-relative)
// is the byte at index (px + A py + B pz) >> shift.  The index is LINEAR in the position, so the step to
// neighbour m is the same number for every site whatever its basis, and lane g keeps its steps in registers.
// shift = 1 with suitable odd / even A, B enumerates the lattice sites only (every lattice vector has an even
// px + A py + B pz), about 2.2 KB per FCC cell at w = 4 and 1.1 KB per BCC cell, where a plain pitched grid
// over all positions (shift = 0) takes 4.3 KB.  The tiles of the cells of a warp are G.gskew bytes further
// apart than a multiple of 128 bytes.  A, B, skew and the assignment of neighbours to (lane, visit) slots
// (G.gslot) are chosen on the host by group_tune_layout() from a model of the 32 banks: ncu on FCC 128^3
// showed 71 % of the shared-memory wavefronts to be bank conflicts with an unpadded grid and 2.5-3.0
// wavefronts per neighbour load with a fixed pad and neighbours dealt to the lanes in shell order.
__host__ __device__ inline int group_index(int px, int py, int pz, int A, int B, int sh) { return (px + A * py + B * pz) >> sh; }

inline void group_basis_pos_host(int Bsites, int b, int p[3]) {
  if (Bsites == 2) { p[0] = p[1] = p[2] = b; return; }
  p[0] = (b >> 1) & 1; p[1] = b & 1; p[2] = (b == 1 || b == 2) ? 1 : 0;
}

// Bytes of a tile (largest site index + 1, rounded up to 128) if every site of the TW^3 conventional cells
// gets an integral index of its own, else 0.
inline int group_layout_extent(const Geom& G, int A, int B, int sh) {
  const int P = 2 * G.TW;
  const long long top = ((long long)(P - 1) * (1 + A + B)) >> sh;
  if (A <= 0 || B <= 0 || top > 60000) return 0;
  std::vector<unsigned char> seen((size_t)top + 1, 0);
  for (int tz = 0; tz < G.TW; ++tz)
    for (int ty = 0; ty < G.TW; ++ty)
      for (int tx = 0; tx < G.TW; ++tx)
        for (int b = 0; b < G.B; ++b) {
          int bp[3];
          group_basis_pos_host(G.B, b, bp);
          const int num = (2 * tx + bp[0]) + A * (2 * ty + bp[1]) + B * (2 * tz + bp[2]);
          if (num & ((1 << sh) - 1)) return 0;
          const int idx = num >> sh;
          if (seen[(size_t)idx]) return 0;
          seen[(size_t)idx] = 1;
        }
  return ((int)top + 1 + 127) & ~127;
}

inline void group_default_layout(Geom& G) {   // plain pitched grid over all positions
  G.gshift = 0;
  G.gA = (2 * G.TW + 3) & ~3;
  G.gB = 2 * G.TW * G.gA + 8;
  G.gskew = 64;
  G.gtile = ((2 * G.TW * G.gB + 127) & ~127);
  for (int s = 0; s < kMaxGroupSlots; ++s) G.gslot[s] = s < G.ZT ? (unsigned char)s : (unsigned char)255;
}

// Register-resident neighbour lists exist for 2, 3 and 6 visits per lane (FCC with three shells: 42
// neighbours over 32 / 16 / 8 lanes; BCC with two shells: 14 over 8 / 16 / 32); anything else takes the
// variant that reads the steps from shared memory (11 visits in registers, FCC with 4 lanes, was measured: 23 ms
// per sweep of FCC 400^3 against 15 ms with 8 lanes).
inline int group_nit(const Geom& G, int lanes) {
  const int need = (G.ZT + lanes - 1) / lanes;
  return need <= 2 ? 2 : need <= 3 ? 3 : need <= 6 ? 6 : 0;
}
inline int group_visits(const Geom& G, int lanes) {
  const int nit = group_nit(G, lanes);
  return nit > 0 ? nit : (G.ZT + lanes - 1) / lanes;
}

// Bank model: one neighbour load of a warp = for every cell of the warp (bank shift c * tile words) the
// lanes' steps from a common site address A; wavefronts = the largest number of distinct words that fall
// into one bank.  Summed over the visits and averaged over A mod 4 (all that matters of A).
inline double group_bank_cost(const int* step, const unsigned char* slot, int lanes, int visits, int tile_words) {
  const int cells = 32 / lanes;
  int total = 0;
  for (int a = 0; a < 4; ++a)
    for (int v = 0; v < visits; ++v) {
      int words[32], banks[32], nw = 0, worst = 0;
      for (int c = 0; c < cells; ++c)
        for (int l = 0; l < lanes; ++l) {
          const int m = slot[v * lanes + l];
          const int st = m == 255 ? 0 : step[m];
          const int w = ((a + st + (1 << 20)) >> 2) + c * tile_words + c * (1 << 22);   // distinct words per cell
          bool seen = false;
          for (int k = 0; k < nw; ++k) seen = seen || words[k] == w;
          if (!seen) { words[nw] = w; banks[nw] = (w - c * (1 << 22)) & 31; ++nw; }
        }
      for (int k = 0; k < nw; ++k) {
        int cnt = 0;
        for (int j = 0; j < nw; ++j) cnt += banks[j] == banks[k];
        worst = cnt > worst ? cnt : worst;
      }
      total += worst;
    }
  return total / 4.0;
}

// Chooses the layout (G.gA, G.gB, G.gshift, G.gtile, G.gskew) and G.gslot for this lane count: candidate
// index maps (the pitched grid with a few paddings; compact maps with shift 1, the smallest B for every A in
// a range) no more than 8 % above the smallest tile, every skew, neighbours in shell order first; then a
// deterministic local search (swaps of two slots) on the best few.
inline void group_tune_layout_search(Geom& G, int lanes) {
  const int visits = group_visits(G, lanes), slots = visits * lanes, ZT = G.ZT, P = 2 * G.TW;
  group_default_layout(G);
  if (slots > kMaxGroupSlots || lanes > 32) return;
  struct Map { int A, B, sh, bytes; };
  std::vector<Map> maps;
  for (int pad = 0; pad < 32; pad += 4) {
    const int A = (P + 3) & ~3, B = P * A + pad;
    maps.push_back({A, B, 0, (P * B + 127) & ~127});
  }
  for (int A = P / 2; A <= 2 * P + 8; ++A) {
    int found = 0;
    for (int B = A * (P / 2); B <= A * (P + 2) + P + 2 && found < 2; ++B) {
      const int bytes = group_layout_extent(G, A, B, 1);
      if (bytes > 0) { maps.push_back({A, B, 1, bytes}); ++found; }
    }
  }
  int min_bytes = 1 << 30;
  for (const Map& m : maps) min_bytes = std::min(min_bytes, m.bytes);
  struct Cand { double cost; Map m; int skew; };
  Cand best[4];
  for (int k = 0; k < 4; ++k) best[k] = {1e30, maps[0], 64};
  int step[kMaxNeighbours];
  for (const Map& m : maps) {
    if (m.bytes > min_bytes + min_bytes / 12) continue;
    for (int q = 0; q < ZT; ++q) step[q] = (G.off[q][0] + m.A * G.off[q][1] + m.B * G.off[q][2]) >> m.sh;
    unsigned char ident[kMaxGroupSlots];
    for (int s = 0; s < kMaxGroupSlots; ++s) ident[s] = s < ZT ? (unsigned char)s : (unsigned char)255;
    for (int skew = 4; skew < 128; skew += 4) {
      const double c = group_bank_cost(step, ident, lanes, visits, (m.bytes + skew) / 4);
      for (int k = 0; k < 4; ++k)
        if (c < best[k].cost) { for (int j = 3; j > k; --j) best[j] = best[j - 1]; best[k] = {c, m, skew}; break; }
      if (lanes == 32) break;   // one cell per warp: the skew does not matter
    }
  }
  double best_cost = 1e30;
  for (int k = 0; k < 4; ++k) {
    if (best[k].cost >= 1e30) continue;
    const Map m = best[k].m;
    const int skew = best[k].skew, tw = (m.bytes + skew) / 4;
    for (int q = 0; q < ZT; ++q) step[q] = (G.off[q][0] + m.A * G.off[q][1] + m.B * G.off[q][2]) >> m.sh;
    unsigned char slot[kMaxGroupSlots];
    for (int s = 0; s < kMaxGroupSlots; ++s) slot[s] = s < ZT ? (unsigned char)s : (unsigned char)255;
    double c = group_bank_cost(step, slot, lanes, visits, tw);
    uint32_t rng = 12345u + (uint32_t)k;
    for (int iter = 0; iter < 2500 && c > visits; ++iter) {
      rng = rng * 1664525u + 1013904223u; const int s1 = (int)((rng >> 8) % (uint32_t)slots);
      rng = rng * 1664525u + 1013904223u; const int s2 = (int)((rng >> 8) % (uint32_t)slots);
      if (s1 / lanes == s2 / lanes || slot[s1] == slot[s2]) continue;
      const unsigned char t1 = slot[s1]; slot[s1] = slot[s2]; slot[s2] = t1;
      const double c2 = group_bank_cost(step, slot, lanes, visits, tw);
      if (c2 <= c) c = c2; else { slot[s2] = slot[s1]; slot[s1] = t1; }
    }
    if (c < best_cost) {
      best_cost = c;
      G.gA = m.A; G.gB = m.B; G.gshift = (short)m.sh; G.gtile = m.bytes; G.gskew = (short)skew;
      for (int s = 0; s < kMaxGroupSlots; ++s) G.gslot[s] = slot[s];
    }
  }
}

struct GroupTuneEntry { int lattice, n_shells, TW, lanes, A, B, tile; short shift, skew; unsigned char slot[kMaxGroupSlots]; };
inline void group_tune_layout(Geom& G, int lanes) {
  // the result depends on (lattice, shells, tile edge, lanes) only: computed once per process
  static std::mutex mu;
  static std::vector<GroupTuneEntry> cache;
  {
    std::lock_guard<std::mutex> lock(mu);
    for (const GroupTuneEntry& e : cache)
      if (e.lattice == G.lattice && e.n_shells == G.n_shells && e.TW == G.TW && e.lanes == lanes) {
        G.gA = e.A; G.gB = e.B; G.gtile = e.tile; G.gshift = e.shift; G.gskew = e.skew;
        for (int s = 0; s < kMaxGroupSlots; ++s) G.gslot[s] = e.slot[s];
        return;
      }
  }
  group_tune_layout_search(G, lanes);
  GroupTuneEntry e{G.lattice, G.n_shells, G.TW, lanes, G.gA, G.gB, G.gtile, G.gshift, G.gskew, {}};
  for (int s = 0; s < kMaxGroupSlots; ++s) e.slot[s] = G.gslot[s];
  std::lock_guard<std::mutex> lock(mu);
  cache.push_back(e);
}

struct GroupSmem {
  int d_stride;        // ints per ordered pair in the difference table
  int d_copies;        // 2: every 32-word stripe holds the pair's row twice, cells with odd index in their warp read the upper
                       // half; 4: 16-bit rows, four per stripe (one per cell of a warp), corr in a table of its own
  int d_bytes, nb_bytes, filt_bytes, tile_bytes, total;
};

// Difference table row of the ordered pair (a,b): [s * n + x] for the shells, then corr(a,b).  When a row fits
// 16 words and a warp holds several cells, rows are 32 words apart and stored twice (words 0..15 and 16..31):
// the rows two cells of a warp read at the same time then lie in different halves of the banks whatever the pairs
// (ncu, FCC 256^3, 16 lanes: 1.3-1.5 wavefronts per table load with one copy and a row stride of 21).
inline GroupSmem group_smem_layout(const Geom& G, int lanes, int warps = kGroupWarpsPerBlock) {
  GroupSmem L;
  const int n = G.n_species;
  const int row = G.n_shells * n + 1;
  if (lanes == 8 && G.gd16 && row - 1 <= 16) {
    // four cells per warp and differences that fit 16 bits: rows of 16 halfwords (8 words), one 8-bank window
    // of every 32-word stripe per cell of the warp, so that the four rows a warp reads at the same time never
    // share a bank (ncu, FCC 256^3, 8 lanes, doubled 32-bit rows: 1.87 wavefronts per table load); corr(a,b)
    // stays 32-bit in a table of its own behind the stripes
    L.d_stride = 32; L.d_copies = 4;
    L.d_bytes = ((n * n * 32 + n * n) * 4 + 15) & ~15;
  } else {
    if (lanes < 32 && row <= 16) { L.d_stride = 32; L.d_copies = 2; }
    else { L.d_stride = row | 1; L.d_copies = 1; }
    L.d_bytes = (n * n * L.d_stride * 4 + 15) & ~15;
  }
  L.nb_bytes = (G.ZT * 4 + 15) & ~15;     // per neighbour: (step & 0xffff) | row << 16
  L.tile_bytes = G.gtile + G.gskew;
  const int cells_per_block = warps * (32 / lanes);
  L.filt_bytes = kFilterWords * 4;
  L.total = (L.d_bytes + L.nb_bytes + L.filt_bytes + cells_per_block * L.tile_bytes + 15) & ~15;
  return L;
}

// The difference table of a handle in the layout group_smem_layout() describes, built once on the host:
// D[(a,b)][s][x] = V_s(b,x) - V_s(a,x) and corr(a,b) = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) less what the empty
// neighbour slots add (each reads D_0(a) - D_0(b), see the kernel).
inline void group_build_table(const Geom& G, int lanes, const int32_t* epi, std::vector<int32_t>& tab) {
  const GroupSmem S = group_smem_layout(G, lanes);
  const int n = G.n_species, corr_at = G.n_shells * n;
  const int n_empty = group_visits(G, lanes) * lanes - G.ZT;
  tab.assign((size_t)S.d_bytes / 4, 0);
  auto D = [&](int s, int a, int b, int x) { return epi[(s * n + b) * n + x] - epi[(s * n + a) * n + x]; };
  auto corr = [&](int a, int b) {
    return 2 * epi[a * n + b] - epi[a * n + a] - epi[b * n + b] - n_empty * (D(0, a, b, a) - D(0, a, b, b));
  };
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b) {
      const int pair = a * n + b;
      if (S.d_copies == 4) {                       // halfword rows, four windows of 16 per stripe; corr behind the stripes
        int16_t* h = reinterpret_cast<int16_t*>(tab.data()) + (size_t)pair * 64;
        for (int c = 0; c < 4; ++c)
          for (int e = 0; e < corr_at; ++e) h[c * 16 + e] = (int16_t)D(e / n, a, b, e % n);
        tab[(size_t)n * n * 32 + pair] = corr(a, b);
      } else {
        int32_t* r = tab.data() + (size_t)pair * S.d_stride;
        for (int c = 0; c < (S.d_copies == 2 ? 2 : 1); ++c) {
          for (int e = 0; e < corr_at; ++e) r[c * 16 + e] = D(e / n, a, b, e % n);
          r[c * 16 + corr_at] = corr(a, b);
        }
      }
    }
}

// basis position (units of a/2) of basis index b along axis a (0 = x, 1 = y, 2 = z); S0
template <int B>
__device__ __forceinline__ int group_basis_pos(int b, int a) {
  if (B == 2) return b;
  return a == 0 ? ((b >> 1) & 1) : a == 1 ? (b & 1) : ((b == 1 || b == 2) ? 1 : 0);
}

// idx = (tz * TW + ty) * TW + tx -> (tx, ty, tz) without integer division: (idx + 0.5) / TW is at least
// 0.5 / TW away from an integer, far more than the rounding error of the float product for idx < 2^20.
__device__ __forceinline__ void group_split_index(int idx, int TW, float inv_TW, int& tx, int& ty, int& tz) {
  const int row = (int)(((float)idx + 0.5f) * inv_TW);
  tx = idx - row * TW;
  tz = (int)(((float)row + 0.5f) * inv_TW);
  ty = row - tz * TW;
}

// NIT > 0: every lane visits exactly NIT neighbours per site, their steps and rows in registers (NIT >=
// ceil(ZT / L); surplus visits are compensated in corr, see above).  NIT == 0: any ZT, steps from shared memory.
template <int B, int L, int NIT>
__global__ void __launch_bounds__(kGroupWarpsPerBlock * 32)
sweep_group_per_cell(const Geom G, uint8_t* __restrict__ species, const int32_t* __restrict__ table,
                     const uint32_t* __restrict__ accept, const uint32_t* __restrict__ filt, DevState* __restrict__ st,
                     int colour, int d_stride, int d_copies, int d_bytes, int nb_bytes, int tile_bytes) {
  constexpr int CPW = 32 / L;                                   // cells per warp
  extern __shared__ __align__(16) unsigned char smem[];
  int32_t* s_D = reinterpret_cast<int32_t*>(smem);              // [a * n + b][d_stride]
  uint32_t* s_nb = reinterpret_cast<uint32_t*>(smem + d_bytes); // [ZT]
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int grp = lane / L, g = lane % L;
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(smem + d_bytes + nb_bytes);   // Tr[64] then Tq[1024]
  unsigned char* tile = smem + d_bytes + nb_bytes + kFilterWords * 4 + (warp * CPW + grp) * tile_bytes;
  __shared__ long long s_dE[kGroupWarpsPerBlock];
  __shared__ unsigned s_acc[kGroupWarpsPerBlock];

  const int n = G.n_species, ZT = G.ZT;
  const int corr_at = G.n_shells * n;
  const bool d_twice = d_copies == 2, d_half = L == 8 && d_copies == 4;   // see group_smem_layout (d_half: 8 lanes only, compile-time false elsewhere)
  // the difference table comes ready-made from the host (group_build_table): a plain copy
#pragma unroll 4
  for (int k = threadIdx.x; k < d_bytes / 4; k += blockDim.x) s_D[k] = table[k];
  const int32_t* s_Dg = s_D + (d_twice ? (grp & 1) * 16 : 0);   // this cell's half of the stripes
  const short* s_Dh = reinterpret_cast<const short*>(s_D) + grp * 16;   // d_half: this cell's window
  if (G.filter_E >= 0) {
#pragma unroll 5
    for (int k = threadIdx.x; k < kFilterWords; k += blockDim.x) s_filt[k] = filt[k];
  }
  const int cA = G.gA, cB = G.gB, csh = G.gshift;
  for (int k = threadIdx.x; k < ZT; k += blockDim.x) {
    const int step = group_index(G.off[k][0], G.off[k][1], G.off[k][2], cA, cB, csh);
    s_nb[k] = ((uint32_t)(uint16_t)(short)step) | ((uint32_t)(G.shell_of[k] * n) << 16);
  }
  // this lane's neighbours
  int nstep[NIT > 0 ? NIT : 1], nrow[NIT > 0 ? NIT : 1];
#pragma unroll
  for (int it = 0; it < NIT; ++it) {
    const int mm = G.gslot[g + it * L];
    const bool valid = mm != 255;
    nstep[it] = valid ? group_index(G.off[mm][0], G.off[mm][1], G.off[mm][2], cA, cB, csh) : 0;
    nrow[it] = valid ? G.shell_of[mm] * n : 0;
  }

  const uint32_t t = (uint32_t)st->sweep;
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  const int n_warps = blockDim.x >> 5;
  const uint32_t m = (blockIdx.x * n_warps + warp) * CPW + grp;
  const bool active = m < G.cells_per_colour;
  long long sum_dE = 0;
  unsigned n_acc = 0;
  int cx = 0, cy = 0, cz = 0, t0x = 0, t0y = 0, t0z = 0;
  const int TW = G.TW, H = G.H, w = G.w;
  const int n_conv = TW * TW * TW;
  const float inv_TW = 1.0f / (float)TW;
  if (active) {
    colour_cell(G, m, colour, cx, cy, cz);
    t0x = (ox + cx * w - H + G.Lx) % G.Lx;
    t0y = (oy + cy * w - H + G.Ly) % G.Ly;
    t0z = tile_z0(G, oz, cz);
  }
  // a3: stage the tile, eight conventional cells per lane in flight (a group without a cell stages species
  // 0 everywhere: all its trials are no-ops)
  for (int idx0 = g; idx0 < n_conv; idx0 += 8 * L) {
    uint32_t v[8];
    int at[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const int idx = idx0 + q * L;
      int tx, ty, tz;
      group_split_index(idx, TW, inv_TW, tx, ty, tz);
      v[q] = 0;
      at[q] = idx < n_conv ? group_index(2 * tx, 2 * ty, 2 * tz, cA, cB, csh) : -1;
      if (active && idx < n_conv) {
        int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
        int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
        int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
        const long long gi = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
        v[q] = B == 2 ? (uint32_t)*reinterpret_cast<const uint16_t*>(species + gi) : *reinterpret_cast<const uint32_t*>(species + gi);
      }
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      if (at[q] < 0) continue;
      unsigned char* dst = tile + at[q];
#pragma unroll
      for (int b = 0; b < B; ++b)
        dst[group_index(group_basis_pos<B>(b, 0), group_basis_pos<B>(b, 1), group_basis_pos<B>(b, 2), cA, cB, csh)] =
            (unsigned char)(v[q] >> (8 * b));
    }
  }
  __syncthreads();  // tables + tiles visible

  {
    const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    const int nit = NIT > 0 ? NIT : (ZT + L - 1) / L;
    const int filter_E = G.filter_E;
    uint32_t r_u_even = 0, r_u_odd = 0;
    int r_step_even = 0, r_step_odd = 0;
    int kc = 0;   // conventional cells of the link cell done so far: slot k = kc * B + b, so k & 1 = b & 1 at compile time
    for (int lz = 0; lz < w; ++lz)
      for (int ly = 0; ly < w; ++ly)
        for (int lx = 0; lx < w; ++lx) {
          const int conv = group_index(2 * (lx + H), 2 * (ly + H), 2 * (lz + H), cA, cB, csh);   // position (0,0,0) of the conventional cell
#pragma unroll
          for (int b = 0; b < B; ++b) {
            const int k = kc * B + b;
            // a4: the L Philox calls of a group cover the next 2 L slots (2 L is a multiple of B: only b == 0 can start a batch)
            if ((2 * L) % B == 0 ? (b == 0 && (kc & (2 * L / B - 1)) == 0) : ((k & (2 * L - 1)) == 0)) {
              const Philox4 r = philox4x32_10(cell_id, (uint32_t)(k >> 1) + g, t, ctr3, G.key0, G.key1);
              // direction -> tile step of the partner, looked up here, off the chain of dependent trials
              r_step_even = (int)(short)(s_nb[mulhi_u32(r.x, (uint32_t)G.Z0)] & 0xffffu);
              r_step_odd = (int)(short)(s_nb[mulhi_u32(r.z, (uint32_t)G.Z0)] & 0xffffu);
              r_u_even = r.y; r_u_odd = r.w;
            }
            const int src = (k >> 1) & (L - 1);
            const int step_j = __shfl_sync(0xffffffffu, (b & 1) ? r_step_odd : r_step_even, src, L);
            const uint32_t u = __shfl_sync(0xffffffffu, (b & 1) ? r_u_odd : r_u_even, src, L);
            const unsigned char* p_i = tile + conv + group_index(group_basis_pos<B>(b, 0), group_basis_pos<B>(b, 1),
                                                                 group_basis_pos<B>(b, 2), cA, cB, csh);
            const unsigned char* p_j = p_i + step_j;
            const int sa = *p_i, sb = *p_j;
            // a5: partial sums over this lane's neighbours of i (a -> b) and of j (b -> a); a trial between
            // equal species runs through the same code (its row of D is all zeros) and is masked below
            const int pair = sa * n + sb;
            const int32_t* Drow = s_Dg + pair * d_stride;
            const short* Dh = s_Dh + pair * 64;
            int part = 0;
            if (NIT > 0) {
#pragma unroll
              for (int it = 0; it < NIT; ++it)
                part += d_half ? (int)Dh[nrow[it] + p_i[nstep[it]]] - (int)Dh[nrow[it] + p_j[nstep[it]]]
                               : Drow[nrow[it] + p_i[nstep[it]]] - Drow[nrow[it] + p_j[nstep[it]]];
            } else {
#pragma unroll 2
              for (int it = 0; it < nit; ++it) {
                const int mm = G.gslot[g + it * L];
                const bool valid = mm != 255;
                const uint32_t e = s_nb[valid ? mm : 0];
                const int step = valid ? (int)(short)(e & 0xffffu) : 0, row = valid ? (int)(e >> 16) : 0;
                part += d_half ? (int)Dh[row + p_i[step]] - (int)Dh[row + p_j[step]] : Drow[row + p_i[step]] - Drow[row + p_j[step]];
              }
            }
            // sum over the lanes of the group: one REDUX for a whole warp; a shuffle tree for smaller groups
            // (a REDUX per member mask was measured slower: FCC 128^3, 8 lanes, 1.49 against 1.26 ms per sweep)
            if (L == 32) {
              part = __reduce_add_sync(0xffffffffu, part);
            } else if (L >= SMCX_GROUP_REDUX_MIN_LANES) {
              // one whole-warp REDUX per cell of the warp, the other cells' lanes contributing 0: CPW independent
              // instructions instead of a chain of log2(L) shuffles and adds
              int sum = 0;
#pragma unroll
              for (int c = 0; c < CPW; ++c) {
                const int r = __reduce_add_sync(0xffffffffu, grp == c ? part : 0);
                sum = grp == c ? r : sum;
              }
              part = sum;
            } else {
#pragma unroll
              for (int o = L >> 1; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o, L);
            }
            const int dE = part + (d_half ? s_D[n * n * 32 + pair] : Drow[corr_at]);
            // a6: Eq. 3 in integer form.  ta <= T[dE] <= ta + E (host-verified); dE <= 0 maps to entry 0.
            bool ok;
            if (filter_E >= 0) {
              const uint32_t dc = (uint32_t)min(max(dE, 0), kFilterDmax);
              const uint32_t ta = mulhi_u32(s_filt[kFilterTr + (dc >> 6)], s_filt[dc & 63u]);
              ok = u < ta;
              if (u - ta <= (uint32_t)filter_E) ok = dE <= 0 || (dE < G.accept_len && u < __ldg(accept + dE));
            } else {
              ok = dE <= 0 || (dE < G.accept_len && u < __ldg(accept + dE));
            }
            ok = ok && sa != sb;
            __syncwarp();
            if (ok) {
              if (g == 0) {
                const_cast<unsigned char*>(p_i)[0] = (unsigned char)sb;
                const_cast<unsigned char*>(p_j)[0] = (unsigned char)sa;
              }
              sum_dE += dE;
              ++n_acc;
            }
            __syncwarp();
          }
          ++kc;
        }
  }
  if (active) {
    // a7: write back the sites a swap can have touched: positions within r0 of the cell.  Only the conventional
    // cells that hold such a position are visited (6^3 of the 8^3 of the tile at w = 4), two per lane in flight.
    const int lo = 2 * H - G.r0, hi = 2 * (H + w) - 1 + G.r0;  // tile positions, inclusive
    const int c0 = lo >> 1, WB = (hi >> 1) - c0 + 1, n_wb = WB * WB * WB;
    const float inv_WB = 1.0f / (float)WB;
    for (int idx0 = g; idx0 < n_wb; idx0 += 2 * L) {
      uint32_t val[2];
      uint32_t keep[2];          // bit b: site b of the conventional cell lies in the written range
      long long gi[2];
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int idx = idx0 + q * L;
        int tx, ty, tz;
        group_split_index(idx < n_wb ? idx : 0, WB, inv_WB, tx, ty, tz);
        tx += c0; ty += c0; tz += c0;
        int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
        int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
        int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
        gi[q] = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
        val[q] = 0; keep[q] = 0;
#pragma unroll
        for (int b = 0; b < B; ++b) {
          const int px = 2 * tx + group_basis_pos<B>(b, 0), py = 2 * ty + group_basis_pos<B>(b, 1),
                    pz = 2 * tz + group_basis_pos<B>(b, 2);
          const bool in = idx < n_wb && px >= lo && px <= hi && py >= lo && py <= hi && pz >= lo && pz <= hi;
          val[q] |= (uint32_t)tile[group_index(px, py, pz, cA, cB, csh)] << (8 * b);
          keep[q] |= in ? 1u << b : 0u;
        }
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        if (keep[q] == (1u << B) - 1u) {          // whole conventional cell: one store
          if (B == 2) *reinterpret_cast<uint16_t*>(species + gi[q]) = (uint16_t)val[q];
          else        *reinterpret_cast<uint32_t*>(species + gi[q]) = val[q];
        } else {
#pragma unroll
          for (int b = 0; b < B; ++b)
            if (keep[q] >> b & 1u) species[gi[q] + b] = (unsigned char)(val[q] >> (8 * b));
        }
      }
    }
  }
  // a8: one atomic pair per block (every lane of a group holds the group's sums: count lane g == 0 only)
  if (g != 0) { sum_dE = 0; n_acc = 0; }
  for (int o = 16; o > 0; o >>= 1) {
    sum_dE += __shfl_down_sync(0xffffffffu, sum_dE, o);
    n_acc += __shfl_down_sync(0xffffffffu, n_acc, o);
  }
  if (lane == 0) { s_dE[warp] = sum_dE; s_acc[warp] = n_acc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < n_warps; ++i) { e += s_dE[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

// f<B, L, NIT>() for the runtime (B, lanes, nit)
#define SMCX_GROUP_DISPATCH_NIT(BB, LL, nit, ...)             \
  switch (nit) {                                               \
    case 2: { constexpr int B_ = BB, L_ = LL, N_ = 2; __VA_ARGS__; } break; \
    case 3: { constexpr int B_ = BB, L_ = LL, N_ = 3; __VA_ARGS__; } break; \
    case 6: { constexpr int B_ = BB, L_ = LL, N_ = 6; __VA_ARGS__; } break; \
    default: { constexpr int B_ = BB, L_ = LL, N_ = 0; __VA_ARGS__; } break; \
  }
#define SMCX_GROUP_DISPATCH_L(BB, lanes, nit, ...)            \
  switch (lanes) {                                             \
    case 4: SMCX_GROUP_DISPATCH_NIT(BB, 4, nit, __VA_ARGS__) break;   \
    case 8: SMCX_GROUP_DISPATCH_NIT(BB, 8, nit, __VA_ARGS__) break;   \
    case 16: SMCX_GROUP_DISPATCH_NIT(BB, 16, nit, __VA_ARGS__) break; \
    default: SMCX_GROUP_DISPATCH_NIT(BB, 32, nit, __VA_ARGS__) break; \
  }
#define SMCX_GROUP_DISPATCH(Bv, lanes, nit, ...)              \
  if ((Bv) == 2) { SMCX_GROUP_DISPATCH_L(2, lanes, nit, __VA_ARGS__) } else { SMCX_GROUP_DISPATCH_L(4, lanes, nit, __VA_ARGS__) }

// Warps per block: 8, or 4 / 2 when a block of 8 warps of tiles would leave an SM with fewer than four
// blocks (measured, FCC 400^3, 8 lanes: 16.8 / 14.9 / 16.5 ms per sweep with 8 / 4 / 2 warps per block);
// `requested` (smcx_params_t::group_warps, 0 = auto) overrides it when that many warps of tiles fit.
inline int group_warps_per_block(const Geom& G, int lanes, int requested) {
  int warps = kGroupWarpsPerBlock;
  while (warps > 2 && 4 * group_smem_layout(G, lanes, warps).total > 227 * 1024) warps >>= 1;
  if (requested >= 1 && requested <= kGroupWarpsPerBlock && group_smem_layout(G, lanes, requested).total <= 227 * 1024)
    warps = requested;
  return warps;
}

inline cudaError_t configure_group_per_cell(const Geom& G, int lanes, int warps) {
  const int sm = group_smem_layout(G, lanes, warps).total;
  const int nit = group_nit(G, lanes);
  cudaError_t e = cudaSuccess;
  SMCX_GROUP_DISPATCH(G.B, lanes, nit, {
    e = cudaFuncSetAttribute(sweep_group_per_cell<B_, L_, N_>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute(sweep_group_per_cell<B_, L_, N_>, cudaFuncAttributePreferredSharedMemoryCarveout,
                               cudaSharedmemCarveoutMaxShared);
  })
  return e;
}

inline void launch_group_per_cell(const Geom& G, int lanes, int warps, uint8_t* species, const int32_t* table, const uint32_t* accept,
                                  const uint32_t* filt, DevState* st, int colour, cudaStream_t stream) {
  const GroupSmem S = group_smem_layout(G, lanes, warps);
  const unsigned cpb = warps * (32 / lanes);
  const unsigned grid = (G.cells_per_colour + cpb - 1) / cpb;
  const int nt = warps * 32;
  const int nit = group_nit(G, lanes);
  SMCX_GROUP_DISPATCH(G.B, lanes, nit, {
    sweep_group_per_cell<B_, L_, N_><<<grid, nt, S.total, stream>>>(G, species, table, accept, filt, st, colour, S.d_stride, S.d_copies,
                                                                     S.d_bytes, S.nb_bytes, S.tile_bytes);
  })
}

}  // namespace smcxk
