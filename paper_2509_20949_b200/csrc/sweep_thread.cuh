// Thread-per-cell colour-pass kernel: BCC, first two shells, link cell w = 4, <= 4 species,
// 2-bit packed storage (16 sites per 32-bit word in site-id order).
//
// Layout facts this kernel rests on:
//  * a row of 8 conventional cells (both sublattices) is exactly one 32-bit word: conventional
//    cell X sits in bits [4X, 4X+4), its corner site in the low two, its body site in the high two;
//  * with w = 4 the LIZ+ tile is 8^3 conventional cells = 64 such words, and the tiles of the
//    cells of one colour tile the whole lattice exactly once, so a pass streams the lattice
//    through shared memory once and no two threads ever touch the same tile;
//  * the tile of thread t is kept at smem[row * NT + t]: every access of a warp hits 32 distinct
//    banks whatever row each lane addresses (lanes differ in the direction they drew);
//  * the 8 + 6 neighbour species of a site are gathered into two 16-bit words of 2-bit fields and
//    reduced with population counts: with species x = lo + 2 hi,
//      D_s(x) = V_s(b,x) - V_s(a,x) = D_s(0) + lo cl_s + hi ch_s + lo hi cb_s,
//    so dE = sum_s [cl_s dlo_s + ch_s dhi_s + cb_s dboth_s] + corr(a,b) with d* the differences of
//    the bit counts around i and around j and corr = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) undoing
//    the i-j bond that both sums include.  Integer arithmetic throughout: results are bit-identical
//    to the plain before/after energy difference.
#pragma once
#include "smcx_common.cuh"
#include "sweep_warp.cuh"

namespace smcxk {

constexpr int kThreadNT = 128;          // threads (= cells) per block
constexpr int kThreadTileWords = 64;    // 8 x 8 rows of one word
constexpr int kCoefInts = 8;            // per (a,b): cl0 ch0 cb0 cl1 ch1 cb1 corr' pad

inline bool thread_kernel_supported(const Geom& G) {
  return G.lattice == 0 && G.n_shells == 2 && G.w == 4 && G.n_species <= 4 && G.H == 2 && G.TW == 8;
}

// Host: coefficient table from the EPI tables, [a*4+b][8] int32.
inline void build_thread_coefficients(const int32_t* epi, int n_species, int32_t* coef /*16*8*/) {
  auto V = [&](int s, int a, int b) -> int32_t {
    return (a < n_species && b < n_species) ? epi[(s * n_species + a) * n_species + b] : 0;
  };
  const int Z[2] = {8, 6};
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b) {
      int32_t* c = coef + (a * 4 + b) * kCoefInts;
      int32_t corr = 2 * V(0, a, b) - V(0, a, a) - V(0, b, b);
      for (int s = 0; s < 2; ++s) {
        int32_t D[4];
        for (int x = 0; x < 4; ++x) D[x] = V(s, b, x) - V(s, a, x);
        const int32_t cl = D[1] - D[0], ch = D[2] - D[0], cb = D[3] - D[1] - D[2] + D[0];
        c[3 * s + 0] = cl; c[3 * s + 1] = ch; c[3 * s + 2] = cb;
        // the merged population counts carry an offset of Z_s per term (see count3)
        corr -= Z[s] * (cl + ch + cb);
      }
      c[6] = corr;
      c[7] = 0;
    }
}

__device__ __forceinline__ uint32_t rotr32(uint32_t v, int n) { return __funnelshift_r(v, v, n); }

// Gather the shell-0 (8 fields, bits 0..15) and shell-1 (6 fields at bits 0,2,4,6,8,12) neighbour
// species of site (X,Y,Z,b) of this thread's tile; also returns the site's own row word.
template <int b>
__device__ __forceinline__ void gather_site(const uint32_t* tile, int X, int row, uint32_t& V1, uint32_t& V2,
                                            uint32_t& own) {
  constexpr int NT = kThreadNT;
  const uint32_t* p = tile + row * NT;
  own = p[0];
  const uint32_t yM = p[-NT], yP = p[NT], zM = p[-8 * NT], zP = p[8 * NT];
  const uint32_t dg = b ? p[9 * NT] : p[-9 * NT];
  // shell 0: the 2x2x2 block of the other sublattice; fields at bit s1 and s1+4 of four rows
  const int s1 = 4 * X + 2 * b - 2;
  const uint32_t A = b ? own : dg, Bq = b ? yP : zM, Cq = b ? zP : yM, Dq = b ? dg : own;
  const uint32_t b01 = ((A >> s1) & 0x33u) | ((Bq >> (s1 - 2)) & 0xCCu);
  const uint32_t b23 = ((Cq >> s1) & 0x33u) | ((Dq >> (s1 - 2)) & 0xCCu);
  V1 = b01 | (b23 << 8);
  // shell 1: same sublattice at X-1, X+1 of the own row and at X of the four adjacent rows
  const int s0 = 4 * X + 2 * b;
  uint32_t acc = (own >> (s0 - 4)) & 0x303u;
  acc |= rotr32(yM, (s0 - 2) & 31) & 0xCu;
  acc |= rotr32(yP, (s0 - 4) & 31) & 0x30u;
  acc |= rotr32(zM, (s0 - 6) & 31) & 0xC0u;
  acc |= rotr32(zP, (s0 - 12) & 31) & 0x3000u;
  V2 = acc;
}

// U holds the fields around i in its low half and around j in its high half.  Returns the three
// merged counts; each equals (count around i) - (count around j) + (number of fields).
__device__ __forceinline__ void count3(uint32_t U, uint32_t M, uint32_t F, int& plo, int& phi, int& pbt) {
  const uint32_t Us = U >> 1;
  plo = __popc((U & M) ^ F);
  phi = __popc((Us & M) ^ F);
  pbt = __popc((U & Us & M) ^ F);
}

template <int bi>
__device__ __forceinline__ void trial_thread(uint32_t* tile, const int4* s_coef, const uint32_t* __restrict__ accept,
                                             int accept_len, int X, int Y, int Z, uint32_t w_dir, uint32_t u,
                                             int& esum, unsigned& nacc) {
  constexpr int NT = kThreadNT;
  constexpr int bj = 1 - bi;
  const int dir = (int)(w_dir >> 29);                 // mulhi(w_dir, 8)
  const int Xj = X - 1 + bi + (dir & 1);
  const int Yj = Y - 1 + bi + ((dir >> 1) & 1);
  const int Zj = Z - 1 + bi + (dir >> 2);
  const int row_i = Z * 8 + Y, row_j = Zj * 8 + Yj;
  uint32_t V1i, V2i, own_i, V1j, V2j, own_j;
  gather_site<bi>(tile, X, row_i, V1i, V2i, own_i);
  gather_site<bj>(tile, Xj, row_j, V1j, V2j, own_j);
  const int sh_i = 4 * X + 2 * bi, sh_j = 4 * Xj + 2 * bj;
  const uint32_t a = (own_i >> sh_i) & 3u, b = (own_j >> sh_j) & 3u;
  const int4 c0 = s_coef[(a * 4 + b) * 2], c1 = s_coef[(a * 4 + b) * 2 + 1];
  int p1l, p1h, p1b, p2l, p2h, p2b;
  count3(__byte_perm(V1i, V1j, 0x5410), 0x55555555u, 0x55550000u, p1l, p1h, p1b);
  count3(__byte_perm(V2i, V2j, 0x5410), 0x11551155u, 0x11550000u, p2l, p2h, p2b);
  const int dE = c1.z + c0.x * p1l + c0.y * p1h + c0.z * p1b + c0.w * p2l + c1.x * p2h + c1.y * p2b;
  bool ok = dE <= 0;
  if (!ok && dE < accept_len) ok = u < __ldg(accept + dE);
  ok = ok && (a != b);
  if (ok) {
    const uint32_t x = a ^ b;
    const uint32_t new_i = own_i ^ (x << sh_i);
    const uint32_t new_j = (row_j == row_i ? new_i : own_j) ^ (x << sh_j);
    tile[row_i * NT] = new_i;
    tile[row_j * NT] = new_j;
    esum += dE;
    ++nacc;
  }
}

__global__ void __launch_bounds__(kThreadNT, 6)
sweep_thread_per_cell(const Geom G, uint32_t* __restrict__ lattice, const int4* __restrict__ coef,
                      const uint32_t* __restrict__ accept, DevState* __restrict__ st, int colour) {
  constexpr int NT = kThreadNT;
  extern __shared__ __align__(16) uint32_t smem_w[];
  uint32_t* tile = smem_w + threadIdx.x;                        // row r at tile[r * NT]
  int4* s_coef = reinterpret_cast<int4*>(smem_w + kThreadTileWords * NT);
  __shared__ int s_dE[NT / 32];
  __shared__ unsigned s_acc[NT / 32];
  if (threadIdx.x < 32) s_coef[threadIdx.x] = coef[threadIdx.x];

  const uint32_t t = (uint32_t)st->sweep;
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  const uint32_t m = blockIdx.x * NT + threadIdx.x;
  const bool active = m < G.cells_per_colour;
  int esum = 0;
  unsigned nacc = 0;
  __syncthreads();
  if (active) {
    int cx, cy, cz;
    colour_cell(G, m, colour, cx, cy, cz);
    const int x0 = (ox + cx * 4 - 2 + G.Lx) % G.Lx;
    const int t0y = (oy + cy * 4 - 2 + G.Ly) % G.Ly;
    const int t0z = (oz + cz * 4 - 2 + G.Lz) % G.Lz;
    const int rw = G.Lx >> 3;                                   // words per lattice row
    const int wlo = x0 >> 3, sh = 4 * (x0 & 7);
    const int whi = wlo + 1 == rw ? 0 : wlo + 1;
    // a3: stage the tile (funnel-shift two aligned words per row into one tile word)
#pragma unroll 2
    for (int rz = 0; rz < 8; ++rz) {
      int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
      uint32_t lo[8], hi[8];
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        const uint32_t* rowp = lattice + ((long long)gz * G.Ly + gy) * rw;
        lo[ry] = rowp[wlo];
        hi[ry] = sh ? rowp[whi] : 0u;
      }
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) tile[(rz * 8 + ry) * NT] = __funnelshift_r(lo[ry], hi[ry], sh);
    }
    // a4-a6: the 128 trials of this cell, raster order, one Philox call per two slots
    const uint32_t cell_id = (uint32_t)((cz * G.ncy + cy) * G.ncx + cx);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    const int accept_len = G.accept_len;
    for (int lz = 0; lz < 4; ++lz)
      for (int ly = 0; ly < 4; ++ly)
#pragma unroll 1
        for (int lx = 0; lx < 4; ++lx) {
          const Philox4 r = philox4x32_10(cell_id, (uint32_t)((lz * 4 + ly) * 4 + lx), t, ctr3, G.key0, G.key1);
          trial_thread<0>(tile, s_coef, accept, accept_len, lx + 2, ly + 2, lz + 2, r.x, r.y, esum, nacc);
          trial_thread<1>(tile, s_coef, accept, accept_len, lx + 2, ly + 2, lz + 2, r.z, r.w, esum, nacc);
        }
    // a7: write back tile rows 1..6 x 1..6; only the bytes that lie wholly inside this tile and
    // can hold a modified site (conventional cells 1..6 of the row)
    const int rb = G.Lx >> 1;                                   // bytes per lattice row
    const bool odd = x0 & 1;
    const int nbytes = odd ? 3 : 4;
    const int byte0 = (x0 + (odd ? 1 : 0)) >> 1;
    for (int rz = 1; rz < 7; ++rz) {
      int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
      for (int ry = 1; ry < 7; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        unsigned char* rowb = reinterpret_cast<unsigned char*>(lattice) + ((long long)gz * G.Ly + gy) * rb;
        const uint32_t wv = tile[(rz * 8 + ry) * NT] >> (odd ? 4 : 0);
        for (int k = 0; k < nbytes; ++k) {
          int bx = byte0 + k; if (bx >= rb) bx -= rb;
          rowb[bx] = (unsigned char)((wv >> (8 * k)) & 0xffu);
        }
      }
    }
  }
  // a8: block reduction, one atomic pair per block
  for (int o = 16; o > 0; o >>= 1) {
    esum += __shfl_down_sync(0xffffffffu, esum, o);
    nacc += __shfl_down_sync(0xffffffffu, nacc, o);
  }
  if ((threadIdx.x & 31) == 0) { s_dE[threadIdx.x >> 5] = esum; s_acc[threadIdx.x >> 5] = nacc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < NT / 32; ++i) { e += s_dE[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

inline size_t thread_kernel_smem() { return (size_t)kThreadTileWords * kThreadNT * 4 + 16 * kCoefInts * 4; }

inline int configure_thread_per_cell() {
  return cudaFuncSetAttribute(sweep_thread_per_cell, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)thread_kernel_smem()) == cudaSuccess ? 0 : -1;
}

inline int launch_thread_per_cell(const Geom& G, uint32_t* lattice, const int32_t* d_coef, const uint32_t* accept,
                                  DevState* st, int colour, cudaStream_t stream) {
  const unsigned grid = (G.cells_per_colour + kThreadNT - 1) / kThreadNT;
  sweep_thread_per_cell<<<grid, kThreadNT, thread_kernel_smem(), stream>>>(
      G, lattice, reinterpret_cast<const int4*>(d_coef), accept, st, colour);
  return 0;
}

}  // namespace smcxk
