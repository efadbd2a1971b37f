// Colour-pass kernel and energy reduction for the nonlinear local-energy model (reading S12 of
// DESIGN.md; "a general nonlinear short-range model, where the local energies of all lattice sites within
// LIZ are calculated to determine the energy change due to a MC move").
//
//   H = sum_i eps(sigma_i, n_i),   n_i[s][x] = neighbours of species x in shell s of site i,
//   eps(a, n) = sum_s ( sum_x W1[s][a][x] n[s][x] + sum_{x <= y} W2[s][a][x][y] n[s][x] n[s][y] ).
//
// One warp per link cell, uint8 species, the tile of the cell plus a halo of H = ceil((r0 + 2 R) / 2) conventional
// cells in shared memory (a trial reads the neighbours of the neighbours of i and j).  A swap of i and j changes the
// local energy of the sites U = {i, j} + N(i) + N(j); which tile positions those are, relative to i, depends on the
// basis index of i and on the drawn direction only, so the host lists them once (LocalUEntry) together with the
// shells in which such a site sees i and j.  eps is a sum over shells, and the swap changes the term of shell s of a
// site only if the site sees i or j in THAT shell (or is i or j itself): the host therefore lists the affected
// (site, shell) pairs shell by shell (2 Z_s + 2 entries per shell instead of 2 ZT + 2 sites with all their shells).
// The lanes of the warp share the entries of one shell at a time -- so all lanes count the same shell: no divergence --
// : a lane counts the species of that shell around its site (eight 8-bit fields of a 64-bit word), evaluates the
// shell's term before the swap, corrects the counts and the centre species for the swap -- the algebraic shortcut the
// oracle does not take: it swaps and recounts whole sites -- evaluates it after, and one warp reduction gives dE.
// Integer arithmetic throughout: the sum of the changed terms is exactly the oracle's difference of whole energies.
#pragma once
#include "smcx_common.cuh"
#include "sweep_warp.cuh"

namespace smcxk {

constexpr int kLocalWarps = 8;
constexpr int kLocalMaxSpecies = 8;      // eight 8-bit counters per shell word
constexpr int kLocalMaxU = 2 + 2 * kMaxNeighbours;

// One unit of work of a trial (b, dir): a site u other than i and j that sees exactly one of them in shell s, and a chunk
// of at most kLocalChunk of u's shell-s neighbours to count (the change of u's shell term is linear in its counts, see
// local_delta_shell, so the chunks of a site simply add up; the first chunk adds the constant).  delta: tile-linear step
// from i to u; bits: 0 = u sees j (else i), 1 = first chunk of the site, 2-3 = basis index of u, 4-6 = shell,
// 7-13 = first neighbour (index into the shell list) of the chunk, 14-15 = chunk length code.
constexpr int kLocalChunk = 12;
__host__ __device__ inline int local_chunk_code(int len) { return len == 12 ? 3 : len == 8 ? 2 : len == 6 ? 1 : len == 4 ? 0 : -1; }
struct LocalUEntry {
  short delta;
  unsigned short bits;
};
static_assert(sizeof(LocalUEntry) == 4, "LocalUEntry is loaded as one word");

struct LocalTables {
  const int32_t* w1;          // [n_shells][n][n]
  const int32_t* w2;          // [n_shells][n][n][n], x <= y used
  const LocalUEntry* utab;    // [B][Z0][umax]: the units of (basis of i, direction), longest chunks first
  const int* ucount;          // [B][Z0]
  int umax;
};

// The term of shell s of eps(c, .): v holds the counts of that shell, species x in bits 8x .. 8x + 7.  The loops run over
// all kLocalMaxSpecies fields with compile-time bounds (fields of species >= n are zero, their weights are not read),
// so that the weight loads are independent of one another and can all be in flight.  Not inlined, and the loop over the
// basis index in the kernel is not unrolled: with both inlined / unrolled the trial loop was several times the
// instruction cache and ncu showed the warps waiting for instructions most of the time (stall no_instruction 14.8 per
// issue).
__device__ __noinline__ int local_eps_shell(const int32_t* __restrict__ s_w1, const int32_t* __restrict__ s_w2, int n, int s, int c,
                                            unsigned long long v) {
  const int32_t* l = s_w1 + (s * n + c) * n;
  const int32_t* q = s_w2 + (s * n + c) * n * n;
  int nx[kLocalMaxSpecies];
#pragma unroll
  for (int x = 0; x < kLocalMaxSpecies; ++x) nx[x] = (int)((v >> (8 * x)) & 255ull);
  int e = 0;
#pragma unroll
  for (int x = 0; x < kLocalMaxSpecies; ++x) {
    if (x < n) {
      int row = l[x];
#pragma unroll
      for (int y = x; y < kLocalMaxSpecies; ++y)
        if (y < n) row += q[x * n + y] * nx[y];
      e += row * nx[x];
    }
  }
  return e;
}

// eps_s(c, n + e_to - e_from) - eps_s(c, n) for a site that keeps its own species c and sees ONE of the swapped sites in
// shell s (that neighbour turns from species `from` into `to`): with g_t(y) = 2 q_tt for y = t, q_{min(t,y) max(t,y)}
// otherwise (s_g, built by the block from W2),
//   l_to - l_from + q_toto + q_fromfrom - q_fromto + sum_y (g_to(y) - g_from(y)) n_y
// -- n multiply-adds instead of two evaluations of the quadratic form.  Exact integer algebra: the same value (mod 2^32)
// as the difference of the two evaluations.
template <class CountWord, int FIELD>
__device__ __forceinline__ int local_delta_shell(const int32_t* __restrict__ s_w1, const int32_t* __restrict__ s_g, int n, int s,
                                                 int c, int from, int to, bool with_const, CountWord v) {
  const int32_t* l = s_w1 + (s * n + c) * n;
  const int32_t* gt = s_g + ((s * n + c) * n + to) * n;
  const int32_t* gf = s_g + ((s * n + c) * n + from) * n;
  int e = with_const ? l[to] - l[from] + ((gt[to] + gf[from]) >> 1) - gf[to] : 0;
  constexpr int kFields = (int)(8 * sizeof(CountWord)) / FIELD;
#pragma unroll
  for (int y = 0; y < kFields; ++y)
    if (y < n) e += (gt[y] - gf[y]) * (int)((v >> (FIELD * y)) & (CountWord)((1 << FIELD) - 1));
  return e;
}
// The counts of the sites that keep their species: eight 8-bit fields of a 64-bit word, or -- n_species <= 6 -- six 5-bit
// fields of a 32-bit word (a shell has at most 24 neighbours), which halves the arithmetic of the counting loop.
constexpr int kLocalNarrowSpecies = 6;
constexpr int kLocalNarrowMaxZ = 31;

inline size_t local_smem_bytes(const Geom& G, int umax) {
  const int n = G.n_species;
  size_t b = (size_t)G.n_shells * n * n * 4 + 2 * (size_t)G.n_shells * n * n * n * 4;     // W1, W2, g
  b += (size_t)G.B * G.Z0 * umax * sizeof(LocalUEntry) + (size_t)G.B * G.Z0 * 4;
  b += (size_t)G.B * G.ZT * 2 + 16;
  b = (b + 15) & ~(size_t)15;
  return b + (size_t)kLocalWarps * (((size_t)G.TW * G.TW * G.TW * G.B + 15) & ~(size_t)15);
}

template <int B, bool NARROW>
__global__ void __launch_bounds__(kLocalWarps * 32, 3)
sweep_local_warp(const Geom G, uint8_t* __restrict__ species, const LocalTables T, const uint32_t* __restrict__ accept,
                 DevState* __restrict__ st, int colour) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n = G.n_species, n_shells = G.n_shells, ZT = G.ZT, Z0 = G.Z0;
  int32_t* s_w1 = reinterpret_cast<int32_t*>(smem);
  int32_t* s_w2 = s_w1 + n_shells * n * n;
  int32_t* s_g = s_w2 + n_shells * n * n * n;
  LocalUEntry* s_u = reinterpret_cast<LocalUEntry*>(s_g + n_shells * n * n * n);
  int* s_ucount = reinterpret_cast<int*>(s_u + B * Z0 * T.umax);
  short* s_delta = reinterpret_cast<short*>(s_ucount + B * Z0);
  const int tile_sites = G.TW * G.TW * G.TW * B;
  size_t tables = (size_t)(reinterpret_cast<unsigned char*>(s_delta + B * ZT) - smem) + 16;
  tables = (tables + 15) & ~(size_t)15;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned char* tile = smem + tables + (size_t)warp * ((tile_sites + 15) & ~15);
  __shared__ long long s_dE[kLocalWarps];
  __shared__ unsigned s_acc[kLocalWarps];
  __shared__ int s_start[kMaxShells + 1];

  for (int k = threadIdx.x; k < n_shells * n * n; k += blockDim.x) s_w1[k] = T.w1[k];
  for (int k = threadIdx.x; k < n_shells * n * n * n; k += blockDim.x) {
    s_w2[k] = T.w2[k];
    const int y = k % n, tt = (k / n) % n, sc = k / (n * n);          // g_t(y) of (shell, centre) sc
    s_g[k] = y == tt ? 2 * T.w2[(sc * n + tt) * n + tt] : T.w2[(sc * n + min(tt, y)) * n + max(tt, y)];
  }
  for (int k = threadIdx.x; k < B * Z0 * T.umax; k += blockDim.x) s_u[k] = T.utab[k];
  for (int k = threadIdx.x; k < B * Z0; k += blockDim.x) s_ucount[k] = T.ucount[k];
  for (int k = threadIdx.x; k < B * ZT; k += blockDim.x) s_delta[k] = G.delta[k / ZT][k % ZT];
  if (threadIdx.x <= kMaxShells) {      // shells are listed one after the other: first neighbour of every shell
    int first = ZT;
    for (int m = ZT - 1; m >= 0; --m)
      if ((int)G.shell_of[m] >= (int)threadIdx.x) first = m;
    s_start[threadIdx.x] = (int)threadIdx.x >= n_shells ? ZT : first;
  }

  const uint32_t t = (uint32_t)st->sweep;
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  const uint32_t m = blockIdx.x * kLocalWarps + warp;
  const bool active = m < G.cells_per_colour;
  long long sum_dE = 0;
  unsigned n_acc = 0;
  int cx = 0, cy = 0, cz = 0, t0x = 0, t0y = 0, t0z = 0;
  const int TW = G.TW, H = G.H, w = G.w;
  if (active) {
    colour_cell(G, m, colour, cx, cy, cz);
    t0x = (ox + cx * w - H + G.Lx) % G.Lx;
    t0y = (oy + cy * w - H + G.Ly) % G.Ly;
    t0z = tile_z0(G, oz, cz);
    for (int idx = lane; idx < TW * TW * TW; idx += 32) {
      const int tx = idx % TW, ty = (idx / TW) % TW, tz = idx / (TW * TW);
      int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
      int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
      int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
      const long long g = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
      if (B == 2) *reinterpret_cast<uint16_t*>(tile + idx * 2) = *reinterpret_cast<const uint16_t*>(species + g);
      else        *reinterpret_cast<uint32_t*>(tile + idx * 4) = *reinterpret_cast<const uint32_t*>(species + g);
    }
  }
  __syncthreads();

  if (active) {
    const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    uint32_t r_dir_even = 0, r_u_even = 0, r_dir_odd = 0, r_u_odd = 0;
    int k = 0;
    for (int lz = 0; lz < w; ++lz)
      for (int ly = 0; ly < w; ++ly)
        for (int lx = 0; lx < w; ++lx) {
          const int conv = ((lz + H) * TW + (ly + H)) * TW + (lx + H);
#pragma unroll 1
          for (int b = 0; b < B; ++b, ++k) {
            if ((k & 63) == 0) {   // a4: 32 Philox calls cover the next 64 slots
              const Philox4 r = philox4x32_10(cell_id, (uint32_t)(k >> 1) + lane, t, ctr3, G.key0, G.key1);
              r_dir_even = r.x; r_u_even = r.y; r_dir_odd = r.z; r_u_odd = r.w;
            }
            const int src = (k >> 1) & 31;
            const uint32_t w_dir = __shfl_sync(0xffffffffu, (k & 1) ? r_dir_odd : r_dir_even, src);
            const uint32_t u = __shfl_sync(0xffffffffu, (k & 1) ? r_u_odd : r_u_even, src);
            const int si = conv * B + b;
            const int dir = (int)mulhi_u32(w_dir, (uint32_t)Z0);
            const int sj = si + s_delta[b * ZT + dir];
            const int sa = tile[si], sb = tile[sj];
            if (sa == sb) continue;   // same species: counts as a trial only
            // a5: the changed terms of the local energies, before and after, shell by shell
            const unsigned long long da = 1ull << (8 * sa), db = 1ull << (8 * sb);
            int part = 0;
            // sites other than i and j keep their species, and the shell-s term of such a site changes only if it sees
            // exactly one of i, j in shell s (one neighbour changes species; seeing both, its counts stay): the host lists
            // those sites, their neighbours cut into chunks of at most kLocalChunk (LocalUEntry), one unit per lane
            {
              const LocalUEntry* ue = s_u + (b * Z0 + dir) * T.umax;
              const int nu = s_ucount[b * Z0 + dir];
              for (int q = lane; q < nu; q += 32) {
                const LocalUEntry e = ue[q];
                const unsigned bits = e.bits;
                const int su = si + e.delta;
                const short* dl = s_delta + (int)((bits >> 2) & 3u) * ZT + (int)((bits >> 7) & 127u);
                const unsigned code = bits >> 14;                        // chunk length 4, 6, 8, 12
                const int s = (int)((bits >> 4) & 7u);
                // sees i: that neighbour turns from a into b; sees j: from b into a
                const int from = (bits & 1u) ? sb : sa, to = (bits & 1u) ? sa : sb;
                if (NARROW) {
                  uint32_t cnt = 0u;
#pragma unroll
                  for (int mm = 0; mm < 4; ++mm) cnt += 1u << (5 * (int)tile[su + dl[mm]]);
                  if (code >= 1u) {
#pragma unroll
                    for (int mm = 4; mm < 6; ++mm) cnt += 1u << (5 * (int)tile[su + dl[mm]]);
                  }
                  if (code >= 2u) {
#pragma unroll
                    for (int mm = 6; mm < 8; ++mm) cnt += 1u << (5 * (int)tile[su + dl[mm]]);
                  }
                  if (code >= 3u) {
#pragma unroll
                    for (int mm = 8; mm < 12; ++mm) cnt += 1u << (5 * (int)tile[su + dl[mm]]);
                  }
                  part += local_delta_shell<uint32_t, 5>(s_w1, s_g, n, s, tile[su], from, to, (bits & 2u) != 0u, cnt);
                } else {
                  unsigned long long cnt = 0ull;
                  const int len = code == 3u ? 12 : 4 + 2 * (int)code;
#pragma unroll 6
                  for (int mm = 0; mm < len; ++mm) cnt += 1ull << (8 * (int)tile[su + dl[mm]]);
                  part += local_delta_shell<unsigned long long, 8>(s_w1, s_g, n, s, tile[su], from, to, (bits & 2u) != 0u, cnt);
                }
              }
            }
            // i and j themselves change species (and see each other in shell 0, where j is a nearest neighbour of i):
            // the shell terms before and after, one (site, shell, before / after) per lane
            if (lane < 4 * n_shells) {
              const int s = lane >> 2, who = (lane >> 1) & 1, after = lane & 1;
              const int su = who ? sj : si;
              const short* dl = s_delta + (su & (B - 1)) * ZT;           // tile index = cell * B + basis
              unsigned long long cnt = 0ull;
#pragma unroll 6
              for (int mm = s_start[s]; mm < s_start[s + 1]; ++mm) cnt += 1ull << (8 * (int)tile[su + dl[mm]]);
              if (after && s == 0) cnt += who ? db - da : da - db;       // j sees i turn from a into b; i sees j turn from b into a
              const int v = local_eps_shell(s_w1, s_w2, n, s, (who != 0) == (after != 0) ? sa : sb, cnt);
              part += after ? v : -v;
            }
            const int dE = __reduce_add_sync(0xffffffffu, part);
            // a6: Eq. 3 in integer form
            bool ok = dE <= 0;
            if (!ok && dE < G.accept_len) ok = u < __ldg(accept + dE);
            if (ok) {
              __syncwarp();
              if (lane == 0) { tile[si] = (unsigned char)sb; tile[sj] = (unsigned char)sa; }
              __syncwarp();
              sum_dE += dE;
              ++n_acc;
            }
          }
        }
    // a7: write back the sites a swap can have touched: positions within r0 of the cell
    const int lo = 2 * H - G.r0, hi = 2 * (H + w) - 1 + G.r0;
    for (int idx = lane; idx < TW * TW * TW; idx += 32) {
      const int tx = idx % TW, ty = (idx / TW) % TW, tz = idx / (TW * TW);
      int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
      int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
      int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
      const long long g = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
#pragma unroll
      for (int b = 0; b < B; ++b) {
        int px, py, pz;
        if (B == 2) { px = 2 * tx + b; py = 2 * ty + b; pz = 2 * tz + b; }
        else { px = 2 * tx + ((b >> 1) & 1); py = 2 * ty + ((b == 1 || b == 3) ? 1 : 0); pz = 2 * tz + ((b == 1 || b == 2) ? 1 : 0); }
        if (px >= lo && px <= hi && py >= lo && py <= hi && pz >= lo && pz <= hi) species[g + b] = tile[idx * B + b];
      }
    }
  }
  if (lane == 0) { s_dE[warp] = sum_dE; s_acc[warp] = n_acc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < kLocalWarps; ++i) { e += s_dE[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

// a9 for the local model: H = sum_i eps_i, one thread per site, neighbours through the periodic lattice.
template <int B>
__global__ void __launch_bounds__(256)
local_energy_kernel(const Geom G, const uint8_t* __restrict__ species, const int32_t* __restrict__ w1, const int32_t* __restrict__ w2,
                    unsigned long long* __restrict__ out) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n = G.n_species, n_shells = G.n_shells;
  int32_t* s_w1 = reinterpret_cast<int32_t*>(smem);
  int32_t* s_w2 = s_w1 + n_shells * n * n;
  __shared__ long long s_sum[8];
  for (int k = threadIdx.x; k < n_shells * n * n; k += blockDim.x) s_w1[k] = w1[k];
  for (int k = threadIdx.x; k < n_shells * n * n * n; k += blockDim.x) s_w2[k] = w2[k];
  __syncthreads();
  // sites of the layers [pc_z0, pc_z1): the whole lattice, or the layers a slab owns (their neighbours lie inside
  // its window, so the periodic wrap below never acts along z there)
  const long long i_first = (long long)G.Lx * G.Ly * G.pc_z0 * B;
  const long long n_sites = (long long)G.Lx * G.Ly * G.pc_z1 * B;
  const int Px = 2 * G.Lx, Py = 2 * G.Ly, Pz = 2 * G.Lz;
  long long sum = 0;
  for (long long i = i_first + blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n_sites; i += (long long)gridDim.x * blockDim.x) {
    const int b = (int)(i % B);
    const long long c = i / B;
    const int x = (int)(c % G.Lx);
    const long long r = c / G.Lx;
    const int y = (int)(r % G.Ly), z = (int)(r / G.Ly);
    int bx, by, bz;
    if (B == 2) { bx = by = bz = b; }
    else { bx = (b >> 1) & 1; by = (b == 1 || b == 3) ? 1 : 0; bz = (b == 1 || b == 2) ? 1 : 0; }
    unsigned long long cnt[kMaxShells];
#pragma unroll
    for (int s = 0; s < kMaxShells; ++s) cnt[s] = 0ull;
    for (int m = 0; m < G.ZT; ++m) {
      int px = 2 * x + bx + G.off[m][0], py = 2 * y + by + G.off[m][1], pz = 2 * z + bz + G.off[m][2];
      if (px < 0) px += Px; else if (px >= Px) px -= Px;
      if (py < 0) py += Py; else if (py >= Py) py -= Py;
      if (pz < 0) pz += Pz; else if (pz >= Pz) pz -= Pz;
      int nb;
      if (B == 2) nb = px & 1;
      else {
        const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
        nb = par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3;
      }
      const long long ns = (((long long)(pz >> 1) * G.Ly + (py >> 1)) * G.Lx + (px >> 1)) * B + nb;
      const unsigned long long one = 1ull << (8 * (int)species[ns]);
      const int sh = G.shell_of[m];
#pragma unroll
      for (int s = 0; s < kMaxShells; ++s)
        if (sh == s) cnt[s] += one;
    }
#pragma unroll
    for (int s = 0; s < kMaxShells; ++s)
      if (s < n_shells) sum += local_eps_shell(s_w1, s_w2, n, s, (int)species[i], cnt[s]);
  }
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
  if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = sum;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long tot = 0;
    for (int k = 0; k < (int)(blockDim.x >> 5); ++k) tot += s_sum[k];
    atomicAdd(out, (unsigned long long)tot);
  }
}

}  // namespace smcxk
