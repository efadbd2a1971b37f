// Packed thread-per-cell colour-pass kernel for BCC lattices with up to 8 species (packed-species
// variants; the 2-bit kernels of sweep_thread.cuh stop at 4 species): BCC, the first two neighbour shells (8 + 6
// neighbours), link cell w = 4, n_species <= 8, SMCX_STORAGE_4BIT.  The BCC counterpart of sweep_fcc.cuh, whose look-up
// machinery (PRMT look-ups of four neighbours at a time, IDP.4A byte sums) it shares.
//
// Layout: BCC is two interpenetrating simple-cubic sublattices (basis 0 at (0,0,0), 1 at (1,1,1), units of a/2).  With 4
// bits per site a row of 8 conventional cells of ONE sublattice is one 32-bit word, in device memory (Store4<2>) and in
// the shared-memory tile alike: 2 sublattices x 64 rows (y + 8 z of the 8^3-cell LIZ+ tile) = 512 B per link cell, word
// (s * 64 + row) of lane l at tile[(s * 64 + row) * 32 + l] (no bank conflicts whatever rows the lanes address).
// Seen from a site of sublattice bs at nibble X of row r (o = bs - 1: the block starts one cell lower when the site is a
// corner site):
//   shell 0 (8 neighbours, other sublattice): nibbles X + o, X + o + 1 of rows (y + o .. y + o + 1, z + o .. z + o + 1);
//   shell 1 (6 neighbours, same sublattice): nibbles X -+ 1 of the own row, nibble X of rows y -+ 1 and z -+ 1.
// Nine row loads per site, each rotated so that its wanted nibbles land on free nibbles of an accumulator; four
// accumulators per site (two per shell), each looked up with two PRMT and summed with two IDP.4A, exactly as in the FCC
// kernel: dE = sum over N(i) of D_s(x) - the same over N(j) + corr(a, b), D_s(x) = V_s(b, x) - V_s(a, x); offsets and
// empty nibbles occur equally often for i and j and cancel.  Pure integer arithmetic: dE is the oracle's before/after
// difference.  One block of kBcc4Warps warps per SM for a whole colour pass, batches of 32 cells from a counter in
// DevState.
#pragma once
#include <type_traits>
#include "smcx_common.cuh"
#include "sweep_fcc.cuh"      // rotr32, add_bytes, FccLut, fcc_lookup, fcc_load_lut, fcc_build_lut, FccEnv, kFccMaxSpecies
#include "sweep_thread.cuh"   // prmt, lop3, smem helpers, acceptance filter, store_tile_bytes, factored Philox
#include "sweep_warp.cuh"

namespace smcxk {

constexpr int kBcc4Warps = 12;                // 12 x 16 KB of tiles + tables in 227 KB
constexpr int kBcc4Rows = 64;                 // rows (y + 8 z) per sublattice of a tile

template <int NT> struct Bcc4Tile {
  static constexpr int kRow = 4 * NT;                 // bytes from one row to the next (NT lanes interleaved)
  static constexpr int kSub = kBcc4Rows * kRow;       // bytes from one sublattice to the other
};

// Direction table, [b][dir] (dir = dx | dy << 1 | dz << 2, S0's order of the eight nearest neighbours): byte offsets from
// i's own row pointer to j's own row (d0) and to the base row of j's other sublattice (d1); a3_j = a3_i + e3,
// a2_j = 4 X + e2 (rotation amounts, see Bcc4Site).
struct Bcc4DirEntry { int32_t d0, d1, e3, e2; };
struct Bcc4Tables { Bcc4DirEntry dir[2][8]; };

template <int NT>
inline bool bcc4_build_tables(const Geom& G, Bcc4Tables& T) {
  if (G.Z0 != 8) return false;
  for (int b = 0; b < 2; ++b)
    for (int d = 0; d < 8; ++d) {
      // j = i + off[d]: the other sublattice; its cell relative to i's
      int cell[3];
      for (int a = 0; a < 3; ++a) {
        const int p = b + G.off[d][a];                // -1 .. 2 (b is the position of basis b along every axis)
        if (G.off[d][a] != 1 && G.off[d][a] != -1) return false;
        cell[a] = p < 0 ? -1 : p >> 1;
      }
      const int bj = 1 - b, oj = bj - 1;
      const int dr = cell[1] + 8 * cell[2];
      Bcc4DirEntry& e = T.dir[b][d];
      e.d0 = (bj - b) * Bcc4Tile<NT>::kSub + dr * Bcc4Tile<NT>::kRow;
      e.d1 = (dr + oj + 8 * oj) * Bcc4Tile<NT>::kRow;  // back on i's sublattice: (b - b) * kSub = 0
      e.e3 = 4 * cell[0];
      e.e2 = 4 * (cell[0] + oj);
    }
  return true;
}

inline bool bcc4_kernel_supported(const Geom& G) {
  return G.lattice == 0 && G.n_shells == 2 && G.w == 4 && G.n_species <= kFccMaxSpecies && G.H == 2 &&
         G.TW == 8 && (G.Lx & 7) == 0 && (long long)G.Lx * G.Ly * G.Lz / 4 < (1ll << 32);
}

// A site as the gather sees it: its own row and the base row of the other sublattice (into this lane's tile), and the
// rotations that bring the window X - 1 .. X + 1 (a3) / X + o, X + o + 1 (a2) to nibble 0.
struct Bcc4Site { const uint32_t *p0, *p1; uint32_t a3, a2; };

// Sum over the 14 neighbours of the site (plus two empty nibbles) of the low / high bytes of D_s(x) + bias.
// own_rot = the site's own row rotated by a3 (its species sits in nibble 1), loaded by the caller.
template <int NT>
__host__ __device__ __forceinline__ void bcc4_site_sum(const Bcc4Site& S, uint32_t own_rot, const FccLut& L0, const FccLut& L1,
                                                       uint32_t& lo, uint32_t& hi) {
  const uint32_t a3 = S.a3, a3m8 = a3 - 8u, a3p4 = a3 + 4u, a2 = S.a2, a2m8 = a2 - 8u;
  // shell 1: same sublattice
  {
    uint32_t A = lop3<kLutSel>(rotr32(fcc_ld<NT, -1>(S.p0), a3), own_rot, 0x00F0u);        // (y - 1): nibble X -> 1; own row: X - 1, X + 1 at 0, 2
    A = lop3<kLutSel>(rotr32(fcc_ld<NT, 1>(S.p0), a3m8), A, 0xF000u);                      // (y + 1): nibble X -> 3
    const uint32_t B0 = rotr32(fcc_ld<NT, -8>(S.p0), a3p4) & 0x000Fu;                      // (z - 1): nibble X -> 0
    const uint32_t B = lop3<kLutAndOr2>(rotr32(fcc_ld<NT, 8>(S.p0), a3), 0x00F0u, B0);     // (z + 1): nibble X -> 1; nibbles 2, 3 empty
    fcc_lookup(L1, A, lo, hi);
    fcc_lookup(L1, B, lo, hi);
  }
  // shell 0: other sublattice, rows (0, 1, 8, 9) of its base row, two nibbles each
  {
    const uint32_t r0 = rotr32(fcc_ld<NT, 0>(S.p1), a2), r1 = rotr32(fcc_ld<NT, 1>(S.p1), a2m8);
    const uint32_t r8 = rotr32(fcc_ld<NT, 8>(S.p1), a2), r9 = rotr32(fcc_ld<NT, 9>(S.p1), a2m8);
    fcc_lookup(L0, lop3<kLutSel>(r1, r0, 0xFF00u), lo, hi);
    fcc_lookup(L0, lop3<kLutSel>(r9, r8, 0xFF00u), lo, hi);
  }
}

// One trial (a4-a6).  p_own: row r of sublattice b in this lane's tile; X4 = 4 X, X the nibble of site i; E = the
// direction-table entry of (b, drawn direction); u = acceptance draw.  MODE as in fcc_trial (0 global, 1 filter).
template <int b, int NT, int MODE>
__host__ __device__ __forceinline__ void bcc4_trial(uint32_t* p_own, uint32_t X4, const Bcc4DirEntry& E, uint32_t u,
                                                    const FccEnv& env, int& esum, unsigned& nacc) {
  using T = Bcc4Tile<NT>;
  constexpr int o = b - 1;
  Bcc4Site si, sj;
  si.p0 = p_own;
  si.p1 = fcc_at<NT>(p_own, ((1 - b) - b) * T::kSub + (o + 8 * o) * T::kRow);
  si.a3 = X4 - 4u;
  si.a2 = X4 + (uint32_t)(4 * o);
  sj.p0 = fcc_at<NT>(p_own, E.d0);
  sj.p1 = fcc_at<NT>(p_own, E.d1);
  sj.a3 = si.a3 + (uint32_t)E.e3;
  sj.a2 = X4 + (uint32_t)E.e2;
  const uint32_t own_i = rotr32(fcc_ld<NT, 0>(si.p0), si.a3), own_j = rotr32(fcc_ld<NT, 0>(sj.p0), sj.a3);
  const uint32_t a = (own_i >> 4) & 7u, sb = (own_j >> 4) & 7u;
  const uint32_t pair = a * 8u + sb;
  const smem_ptr_t lp = smem_index(env.lut, pair, env.lut_pair_bytes);
  const FccLut L0 = fcc_load_lut(lp), L1 = fcc_load_lut(lp + env.lut_shell_bytes);
  const int corr = (int)lds_u32(env.corr, pair * 4u);
  uint32_t lo_i = 0u, hi_i = 0u, lo_j = 0u, hi_j = 0u;
  bcc4_site_sum<NT>(si, own_i, L0, L1, lo_i, hi_i);
  bcc4_site_sum<NT>(sj, own_j, L0, L1, lo_j, hi_j);
  const int dE = (int)(lo_i - lo_j) + 256 * (int)(hi_i - hi_j) + corr;
  bool ok;
  if (MODE == 1) {
    const uint32_t dc = (uint32_t)min(max(dE, 0), kFilterDmax);
    const uint32_t ta = mulhi_u32(lds_u32(env.filt, 4u * (kFilterTr + (dc >> 6))), lds_u32(env.filt, 4u * (dc & 63u)));
    ok = u < ta;
    if (u - ta <= (uint32_t)env.filter_E) ok = dE <= 0 || (dE < env.accept_len && u < ldg_u32(env.accept + dE));
  } else {
    ok = dE <= 0 || (dE < env.accept_len && u < ldg_u32(env.accept + dE));
  }
  ok = ok && a != sb;
  const uint32_t x = ok ? (a ^ sb) : 0u;                       // both nibbles change by a ^ b; a rejected trial XORs zeros
#ifdef __CUDA_ARCH__
  atomicXor(const_cast<uint32_t*>(si.p0), x << X4);
  atomicXor(const_cast<uint32_t*>(sj.p0), x << (sj.a3 + 4u));
#else
  *const_cast<uint32_t*>(si.p0) ^= x << X4;
  *const_cast<uint32_t*>(sj.p0) ^= x << (sj.a3 + 4u);
#endif
  esum += ok ? dE : 0;
  nacc += ok ? 1u : 0u;
}


#ifdef __CUDACC__
inline size_t bcc4_smem_bytes(int rep) {
  return (size_t)kBcc4Warps * Bcc4Tile<32>::kSub * 2 + (size_t)64 * 3 * rep * 16 + 64 * 4 + sizeof(Bcc4Tables) + kFilterWords * 4;
}
inline int bcc4_lut_rep() {
  for (int rep = 8; rep >= 1; rep >>= 1)
    if (bcc4_smem_bytes(rep) + 2560 <= 227 * 1024) return rep;
  return 1;
}

template <int MODE>
__global__ void __launch_bounds__(kBcc4Warps * 32, 1)
sweep_bcc4_thread(const Geom G, const Bcc4Tables BT, uint32_t* __restrict__ lattice, const uint4* __restrict__ lut,
                  const int32_t* __restrict__ corr, int rep, const uint32_t* __restrict__ accept,
                  const uint32_t* __restrict__ filt, DevState* __restrict__ st, int colour) {
  constexpr int NT = 32;
  constexpr int R = kBcc4Rows;
  extern __shared__ __align__(16) uint32_t smem_w[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint32_t* tile = smem_w + warp * (2 * R * NT) + lane;                        // word (s * 64 + row) at tile[(s * 64 + row) * NT]
  uint4* s_lut = reinterpret_cast<uint4*>(smem_w + kBcc4Warps * (2 * R * NT));
  int32_t* s_corr = reinterpret_cast<int32_t*>(s_lut + 64 * 3 * rep);
  Bcc4DirEntry* s_dir = reinterpret_cast<Bcc4DirEntry*>(s_corr + 64);
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(s_dir + 16);
  __shared__ uint2 s_slot[64];                                                 // Philox products that depend on the slot pair only
  __shared__ long long s_e64[kBcc4Warps];
  __shared__ unsigned s_acc[kBcc4Warps];

  for (int k = threadIdx.x; k < 64 * 3 * rep; k += blockDim.x) s_lut[k] = lut[k];
  for (int k = threadIdx.x; k < 64; k += blockDim.x) s_corr[k] = corr[k];
  if (MODE == 1)
    for (int k = threadIdx.x; k < kFilterWords; k += blockDim.x) s_filt[k] = filt[k];
  for (int k = threadIdx.x; k < 16; k += blockDim.x) s_dir[k] = BT.dir[k >> 3][k & 7];
  const uint32_t t = (uint32_t)st->sweep;
  if (threadIdx.x < 64) s_slot[threadIdx.x] = philox_slot_entry(threadIdx.x, t, G.rk0, G.rk1);
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
  FccEnv env;
  env.lut = smem_ptr(s_lut) + (uint32_t)((lane % rep) * 16);
  env.corr = smem_ptr(s_corr);
  env.filt = smem_ptr(s_filt);
  env.lut_pair_bytes = 3u * (uint32_t)rep * 16u;
  env.lut_shell_bytes = (uint32_t)rep * 16u;
  env.accept = accept;
  env.accept_len = G.accept_len;
  env.filter_E = G.filter_E;
  const smem_ptr_t dir_p = smem_ptr(s_dir);
  const int rw = G.Lx >> 3;                                     // groups of 8 cells per lattice row
  const uint32_t zstride = (uint32_t)G.Ly * (uint32_t)rw;
  const uint32_t n_batches = (G.cells_per_colour + 31u) >> 5;
  long long esum_total = 0;
  unsigned nacc = 0;
  __syncthreads();
  for (;;) {
    // a2: the next batch of 32 consecutive cells of the colour
    uint32_t batch = 0;
    if (lane == 0) batch = atomicAdd(&st->work[G.work_base + colour], 1u);
    batch = __shfl_sync(0xffffffffu, batch, 0);
    if (batch >= n_batches) break;
    const uint32_t m = batch * 32u + (uint32_t)lane;
    if (m < G.cells_per_colour) {
      int cx, cy, cz;
      colour_cell(G, m, colour, cx, cy, cz);
      const int x0 = (ox + cx * 4 - 2 + G.Lx) % G.Lx;
      const int t0y = (oy + cy * 4 - 2 + G.Ly) % G.Ly;
      const int t0z = tile_z0(G, oz, cz);
      const int wlo = x0 >> 3, sh = 4 * (x0 & 7);
      const int whi = wlo + 1 == rw ? 0 : wlo + 1;
      uint32_t offy[8];
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        offy[ry] = (uint32_t)gy * (uint32_t)rw;
      }
      // a3: stage the tile: per row two 8-byte groups (the two sublattice words each), funnel-shifted into two tile words
#pragma unroll 1
      for (int rz = 0; rz < 8; ++rz) {
        int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
        const uint32_t zoff = (uint32_t)gz * zstride;
        uint2 lo[8], hi[8];
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          const uint2* row = reinterpret_cast<const uint2*>(lattice) + (zoff + offy[ry]);
          lo[ry] = row[wlo];
          hi[ry] = row[whi];
        }
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          uint32_t* d = tile + (rz * 8 + ry) * NT;
          d[0] = __funnelshift_r(lo[ry].x, hi[ry].x, sh);
          d[R * NT] = __funnelshift_r(lo[ry].y, hi[ry].y, sh);
        }
      }
      // a4-a6: the 128 trials of the cell, raster order: conventional cell c = (lz * 4 + ly) * 4 + lx, then b; one Philox
      // call per conventional cell (slots 2 c and 2 c + 1)
      const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
      const PhiloxCell pc = philox_cell_setup(cell_id, t, ctr3, G.rk0, G.rk1);
      int esum = 0;
#pragma unroll 1
      for (int c = 0; c < 64; ++c) {
        const uint32_t X4 = 4u * (uint32_t)((c & 3) + 2);
        const int row = ((c >> 2) & 3) + 2 + 8 * ((c >> 4) + 2);
        uint32_t* p_row = tile + row * NT;
        const Philox4 r = philox_factored(pc, s_slot[c], G.rk0, G.rk1);
#define SMCX_BCC4_TRIAL(B, WDIR, U)                                                                        \
        {                                                                                                    \
          const int4 e = lds_int4(dir_p, (int)((B * 8u + ((WDIR) >> 29)) * 16u));                          \
          const Bcc4DirEntry E{e.x, e.y, e.z, e.w};                                                         \
          bcc4_trial<B, NT, MODE>(p_row + B * (R * NT), X4, E, U, env, esum, nacc);                         \
        }
        SMCX_BCC4_TRIAL(0, r.x, r.y) SMCX_BCC4_TRIAL(1, r.z, r.w)
#undef SMCX_BCC4_TRIAL
      }
      esum_total += esum;     // |dE| < 2^23 (host check), 128 trials: exact in int32 per cell
      // a7: write back rows 1..6 x 1..6 of both sublattices: the bytes that lie wholly inside this tile
      {
        const uint32_t dwh = (uint32_t)(whi - wlo) * 2u;            // word step from the low to the high group of a row
        uint32_t* const peer = reinterpret_cast<uint32_t*>(G.peer_lat);
        auto wb = [&](auto cc) {
          constexpr int C = decltype(cc)::value;
#pragma unroll 1
          for (int rz = 1; rz < 7; ++rz) {
            int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
            const bool mirror = peer != nullptr && gz >= G.peer_z0 && gz < G.peer_z1;   // fused ghost-layer message
#pragma unroll
            for (int ry = 1; ry < 7; ++ry) {
              const uint32_t base = (((uint32_t)gz * zstride) + offy[ry] + (uint32_t)wlo) * 2u;
#pragma unroll
              for (int s = 0; s < 2; ++s) {
                const uint32_t v = tile[(s * R + rz * 8 + ry) * NT];
                store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(lattice + base + s),
                                                     reinterpret_cast<unsigned char*>(lattice + (uint32_t)(base + s + dwh)), v);
                if (mirror)
                  store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(peer + base + s),
                                                       reinterpret_cast<unsigned char*>(peer + (uint32_t)(base + s + dwh)), v);
              }
            }
          }
        };
        switch (x0 & 7) {
          case 0: wb(std::integral_constant<int, 0>{}); break;
          case 1: wb(std::integral_constant<int, 1>{}); break;
          case 2: wb(std::integral_constant<int, 2>{}); break;
          case 3: wb(std::integral_constant<int, 3>{}); break;
          case 4: wb(std::integral_constant<int, 4>{}); break;
          case 5: wb(std::integral_constant<int, 5>{}); break;
          case 6: wb(std::integral_constant<int, 6>{}); break;
          default: wb(std::integral_constant<int, 7>{}); break;
        }
      }
    }
  }
  // a8: one atomic pair per block
  for (int o = 16; o > 0; o >>= 1) {
    esum_total += __shfl_down_sync(0xffffffffu, esum_total, o);
    nacc += __shfl_down_sync(0xffffffffu, nacc, o);
  }
  if (lane == 0) { s_e64[warp] = esum_total; s_acc[warp] = nacc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < kBcc4Warps; ++i) { e += s_e64[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

inline int configure_bcc4_thread(int rep) {
  const int sm = (int)bcc4_smem_bytes(rep);
  if (cudaFuncSetAttribute(sweep_bcc4_thread<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_bcc4_thread<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
  cudaFuncSetAttribute(sweep_bcc4_thread<0>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_bcc4_thread<1>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  return 0;
}

inline int launch_bcc4_thread(const Geom& G, const Bcc4Tables& BT, uint32_t* lattice, const uint32_t* d_lut, const int32_t* d_corr,
                              int rep, const uint32_t* accept, const uint32_t* d_filter, DevState* st, int colour, int sm_count,
                              cudaStream_t stream) {
  const unsigned n_batches = (G.cells_per_colour + 31u) / 32u;
  const unsigned want = (n_batches + kBcc4Warps - 1) / kBcc4Warps;
  const unsigned grid = want < (unsigned)sm_count ? want : (unsigned)sm_count;
  const size_t sm = bcc4_smem_bytes(rep);
  const uint4* lut4 = reinterpret_cast<const uint4*>(d_lut);
  if (G.filter_E >= 0)
    sweep_bcc4_thread<1><<<grid, kBcc4Warps * 32, sm, stream>>>(G, BT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour);
  else
    sweep_bcc4_thread<0><<<grid, kBcc4Warps * 32, sm, stream>>>(G, BT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}
#endif  // __CUDACC__

}  // namespace smcxk
