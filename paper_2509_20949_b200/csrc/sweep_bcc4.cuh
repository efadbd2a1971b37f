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

constexpr int kBcc4Warps = 20;                // 20 x 8 KB of tile windows + tables + the head of T in 227 KB
constexpr int kBcc4Rows = 64;                 // rows (y + 8 z) per sublattice of a whole tile (8 layers)
constexpr int kBcc4WinRows = 32;              // the kernel keeps four layers per sublattice resident

// ROWS = 64: the whole tile.  ROWS < 64 (the kernel's window): the trials of layer lz of the cell (tile layer lz + 2)
// reach three half-units up and down, i.e. tile layers lz + 1 .. lz + 4 of the corner sublattice and lz .. lz + 3 of
// the centre sublattice; sublattice s keeps tile layer rz in slot rz - lz - (1 - s), which the row pointers of the
// gather see as a constant offset per sublattice (sub()), exactly as in sweep_fcc.cuh.
template <int NT, int ROWS = kBcc4Rows> struct Bcc4Tile {
  static constexpr int kRow = 4 * NT;                 // bytes from one row to the next (NT lanes interleaved)
  static constexpr int kSub = ROWS * kRow;            // bytes from one sublattice to the other
  __host__ __device__ static constexpr int sub(int s) { return s * kSub - (ROWS < kBcc4Rows ? (1 - s) * 8 * kRow : 0); }
};

// Direction table, [b][dir] (dir = dx | dy << 1 | dz << 2, S0's order of the eight nearest neighbours): byte offsets from
// i's own row pointer to j's own row (d0) and to the base row of j's other sublattice (d1); a3_j = a3_i + e3,
// a2_j = 4 X + e2 (rotation amounts, see Bcc4Site).
struct Bcc4DirEntry { int32_t d0, d1, e3, e2; };
struct Bcc4Tables { Bcc4DirEntry dir[2][8]; };

template <int NT, int ROWS = kBcc4Rows>
inline bool bcc4_build_tables(const Geom& G, Bcc4Tables& T) {
  using TL = Bcc4Tile<NT, ROWS>;
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
      e.d0 = TL::sub(bj) - TL::sub(b) + dr * TL::kRow;
      e.d1 = (dr + oj + 8 * oj) * TL::kRow;            // back on i's sublattice
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
// direction-table entry of (b, drawn direction); u = acceptance draw.  MODE as in fcc_trial (0 global, 1 filter, 2 head
// of the table in shared memory).
template <int b, int NT, int MODE, int ROWS = kBcc4Rows>
__host__ __device__ __forceinline__ void bcc4_trial(uint32_t* p_own, uint32_t X4, const Bcc4DirEntry& E, uint32_t u,
                                                    const FccEnv& env, int& esum, unsigned& nacc) {
  using T = Bcc4Tile<NT, ROWS>;
  constexpr int o = b - 1;
  Bcc4Site si, sj;
  si.p0 = p_own;
  si.p1 = fcc_at<NT>(p_own, T::sub(1 - b) - T::sub(b) + (o + 8 * o) * T::kRow);
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
  if (MODE == 2) {
    // as sweep_fcc_thread<2>: the head of T in shared memory followed by the bound T[direct_len]; behind it T[dE] itself
    // by a predicated load (the library keeps a zero entry behind T in device memory, which serves dE >= len)
    uint32_t thr = lds_u32(env.filt, 4u * min((uint32_t)dE, (uint32_t)env.direct_len));
    const bool far = dE >= env.direct_len && u < thr;
    const uint32_t* tp = env.accept + min(dE, env.accept_len);
#ifdef __CUDA_ARCH__
    asm("{ .reg .pred p; setp.ne.u32 p, %2, 0; @p ld.global.nc.u32 %0, [%1]; }" : "+r"(thr) : "l"(tp), "r"((uint32_t)far));
#else
    if (far) thr = *tp;
#endif
    ok = dE <= 0 || u < thr;
  } else if (MODE == 1) {
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
constexpr int kBcc4SmemMax = 232448 - 1024;                    // 227 KB less the static part
// dynamic shared memory: tile windows, look-up rows, corr, direction table, then the filter tables (accept_words =
// kFilterWords) or the head of the threshold table plus its bound entry
inline size_t bcc4_smem_bytes(int rep, size_t accept_words = kFilterWords) {
  return (size_t)kBcc4Warps * Bcc4Tile<32, kBcc4WinRows>::kSub * 2 + (size_t)64 * 3 * rep * 16 + 64 * 4 + sizeof(Bcc4Tables) + accept_words * 4;
}
inline int bcc4_lut_rep() {
  for (int rep = 8; rep >= 1; rep >>= 1)
    if (bcc4_smem_bytes(rep) <= (size_t)kBcc4SmemMax) return rep;
  return 1;
}
// entries of T to hold in shared memory (sweep_bcc4_thread<2>), or 0: too few fit
constexpr int kBcc4DirectMin = 4096;
inline int bcc4_direct_entries(int rep, int accept_len) {
  const size_t fixed = bcc4_smem_bytes(rep, 1);
  if (fixed > (size_t)kBcc4SmemMax) return 0;
  const size_t room = ((size_t)kBcc4SmemMax - fixed) / 4;
  if (room >= (size_t)accept_len) return accept_len;
  return room >= (size_t)kBcc4DirectMin ? (int)room : 0;
}

template <int MODE>
__global__ void __launch_bounds__(kBcc4Warps * 32, 1)
sweep_bcc4_thread(const Geom G, const Bcc4Tables BT, uint32_t* __restrict__ lattice, const uint4* __restrict__ lut,
                  const int32_t* __restrict__ corr, int rep, const uint32_t* __restrict__ accept,
                  const uint32_t* __restrict__ filt, DevState* __restrict__ st, int colour, int direct_len) {
  constexpr int NT = 32;
  constexpr int WR = kBcc4WinRows;
  extern __shared__ __align__(16) uint32_t smem_w[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint32_t* tile = smem_w + warp * (2 * WR * NT) + lane;                       // word (s * WR + row) at tile[(s * WR + row) * NT]
  uint4* s_lut = reinterpret_cast<uint4*>(smem_w + kBcc4Warps * (2 * WR * NT));
  int32_t* s_corr = reinterpret_cast<int32_t*>(s_lut + 64 * 3 * rep);
  Bcc4DirEntry* s_dir = reinterpret_cast<Bcc4DirEntry*>(s_corr + 64);
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(s_dir + 16);                  // filter tables, or the head of T + its bound
  __shared__ uint2 s_slot[64];                                                 // Philox products that depend on the slot pair only
  __shared__ long long s_e64[kBcc4Warps];
  __shared__ unsigned s_acc[kBcc4Warps];

  for (int k = threadIdx.x; k < 64 * 3 * rep; k += blockDim.x) s_lut[k] = lut[k];
  for (int k = threadIdx.x; k < 64; k += blockDim.x) s_corr[k] = corr[k];
  if (MODE == 1)
    for (int k = threadIdx.x; k < kFilterWords; k += blockDim.x) s_filt[k] = filt[k];
  if (MODE == 2)
    for (int k = threadIdx.x; k <= direct_len; k += blockDim.x) s_filt[k] = k < G.accept_len ? accept[k] : 0u;
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
  env.direct_len = direct_len;
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
      const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
      const PhiloxCell pc = philox_cell_setup(cell_id, t, ctr3, G.rk0, G.rk1);
      const uint32_t dwh = (uint32_t)(whi - wlo) * 2u;            // word step from the low to the high group of a row
      uint32_t* const peer = reinterpret_cast<uint32_t*>(G.peer_lat);
      int esum = 0;
      // The cell runs in four steps of 32 trials (layer lz of the cell); between two steps the lowest layer of either
      // window is written back (final: later trials only reach higher layers), the other three move down a slot and one
      // new layer is staged.  Sublattice 0 holds tile layers lz + 1 .. lz + 4, sublattice 1 lz .. lz + 3.
      // a3: stage tile layer rz of sublattice S into a slot: per row two 8-byte groups (the two sublattice words, one of
      // them used), funnel-shifted into the tile word
      auto stage = [&](auto sub_c, int slot, int rz) {
        constexpr int S = decltype(sub_c)::value;
        int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
        const uint32_t zoff = (uint32_t)gz * zstride;
        uint32_t lo[8], hi[8];
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          const uint32_t* row = lattice + 2u * (zoff + offy[ry]) + S;
          lo[ry] = row[2 * wlo];
          hi[ry] = row[2 * whi];
        }
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) tile[(S * WR + slot * 8 + ry) * NT] = __funnelshift_r(lo[ry], hi[ry], sh);
      };
      // a7: write back rows 1..6 of the layers that leave the windows after step lz - 1 (lz = 4: of everything still
      // resident), tile layers 1..6 only: the bytes that lie wholly inside this tile
      auto wb = [&](auto cc, int lz) {
        constexpr int C = decltype(cc)::value;
#pragma unroll 1
        for (int sq = 0; sq < 2; ++sq) {
          const int first = lz - sq, n_slots = lz == 4 ? 4 : 1;   // window of sublattice sq in step lz - 1: from lz - 1 + (1 - sq)
#pragma unroll 1
          for (int slot = 0; slot < n_slots; ++slot) {
            const int rz = first + slot;
            if (rz < 1 || rz > 6) continue;
            int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
            const bool mirror = peer != nullptr && gz >= G.peer_z0 && gz < G.peer_z1;   // fused ghost-layer message
#pragma unroll
            for (int ry = 1; ry < 7; ++ry) {
              const uint32_t base = (((uint32_t)gz * zstride) + offy[ry] + (uint32_t)wlo) * 2u + (uint32_t)sq;
              const uint32_t v = tile[(sq * WR + slot * 8 + ry) * NT];
              store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(lattice + base),
                                                   reinterpret_cast<unsigned char*>(lattice + (uint32_t)(base + dwh)), v);
              if (mirror)
                store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(peer + base),
                                                     reinterpret_cast<unsigned char*>(peer + (uint32_t)(base + dwh)), v);
            }
          }
        }
      };
      auto write_back = [&](int lz) {
        switch (x0 & 7) {
          case 0: wb(std::integral_constant<int, 0>{}, lz); break;
          case 1: wb(std::integral_constant<int, 1>{}, lz); break;
          case 2: wb(std::integral_constant<int, 2>{}, lz); break;
          case 3: wb(std::integral_constant<int, 3>{}, lz); break;
          case 4: wb(std::integral_constant<int, 4>{}, lz); break;
          case 5: wb(std::integral_constant<int, 5>{}, lz); break;
          case 6: wb(std::integral_constant<int, 6>{}, lz); break;
          default: wb(std::integral_constant<int, 7>{}, lz); break;
        }
      };
      using TW = Bcc4Tile<NT, WR>;
#pragma unroll 1
      for (int lz = 0; lz < 4; ++lz) {
        if (lz > 0) {
          write_back(lz);
#pragma unroll 1
          for (int s = 0; s < 2; ++s) {                           // slots 1..3 move down one slot
            uint32_t* d = tile + s * WR * NT;
#pragma unroll 8
            for (int r = 0; r < 24; ++r) d[r * NT] = d[(r + 8) * NT];
          }
        }
#pragma unroll 1
        for (int slot = lz ? 3 : 0; slot < 4; ++slot) {
          stage(std::integral_constant<int, 0>{}, slot, lz + 1 + slot);
          stage(std::integral_constant<int, 1>{}, slot, lz + slot);
        }
        // a4-a6: the 32 trials of layer lz of the cell, raster order: conventional cell c = (lz * 4 + ly) * 4 + lx, then
        // b; one Philox call per conventional cell (slots 2 c and 2 c + 1); site i sits in (virtual) slot 2 of its window
#pragma unroll 1
        for (int c = 16 * lz; c < 16 * lz + 16; ++c) {
          const uint32_t X4 = 4u * (uint32_t)((c & 3) + 2);
          uint32_t* p_row = tile + (((c >> 2) & 3) + 2 + 16) * NT;
          const Philox4 r = philox_factored(pc, s_slot[c], G.rk0, G.rk1);
#define SMCX_BCC4_TRIAL(B, WDIR, U)                                                                        \
          {                                                                                                  \
            const int4 e = lds_int4(dir_p, (int)((B * 8u + ((WDIR) >> 29)) * 16u));                        \
            const Bcc4DirEntry E{e.x, e.y, e.z, e.w};                                                       \
            bcc4_trial<B, NT, MODE, WR>(const_cast<uint32_t*>(fcc_at<NT>(p_row, TW::sub(B))), X4, E, U, env, esum, nacc); \
          }
          SMCX_BCC4_TRIAL(0, r.x, r.y) SMCX_BCC4_TRIAL(1, r.z, r.w)
#undef SMCX_BCC4_TRIAL
        }
      }
      write_back(4);
      esum_total += esum;     // |dE| < 2^23 (host check), 128 trials: exact in int32 per cell
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
  (void)rep;
  if (cudaFuncSetAttribute(sweep_bcc4_thread<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBcc4SmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_bcc4_thread<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBcc4SmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_bcc4_thread<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBcc4SmemMax) != cudaSuccess) return -1;
  cudaFuncSetAttribute(sweep_bcc4_thread<0>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_bcc4_thread<1>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_bcc4_thread<2>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  return 0;
}

inline int launch_bcc4_thread(const Geom& G, const Bcc4Tables& BT, uint32_t* lattice, const uint32_t* d_lut, const int32_t* d_corr,
                              int rep, const uint32_t* accept, const uint32_t* d_filter, DevState* st, int colour, int sm_count,
                              int tail_from, cudaStream_t stream) {
  const unsigned n_batches = (G.cells_per_colour + 31u) / 32u;
  const unsigned want = (n_batches + kBcc4Warps - 1) / kBcc4Warps;
  const unsigned grid = want < (unsigned)sm_count ? want : (unsigned)sm_count;
  const uint4* lut4 = reinterpret_cast<const uint4*>(d_lut);
  // the head of T in shared memory: sound if T[direct] bounds every later entry (tail_from: checked by the host at upload)
  int direct = bcc4_direct_entries(rep, G.accept_len);
  if (direct < G.accept_len && direct < tail_from) direct = 0;
  if (direct > 0)
    sweep_bcc4_thread<2><<<grid, kBcc4Warps * 32, bcc4_smem_bytes(rep, (size_t)direct + 1), stream>>>(
        G, BT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, direct);
  else if (G.filter_E >= 0)
    sweep_bcc4_thread<1><<<grid, kBcc4Warps * 32, bcc4_smem_bytes(rep), stream>>>(G, BT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, 0);
  else
    sweep_bcc4_thread<0><<<grid, kBcc4Warps * 32, bcc4_smem_bytes(rep), stream>>>(G, BT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, 0);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}
#endif  // __CUDACC__

}  // namespace smcxk
