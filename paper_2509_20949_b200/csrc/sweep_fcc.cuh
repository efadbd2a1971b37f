// Packed thread-per-cell colour-pass kernel for FCC lattices (the paper's own lattice:
// PAPER.md:118, 141, 165): FCC, the first 2..3 neighbour shells (12 + 6 + 24 neighbours; the tile is 8^3 cells), link cell w = 4,
// n_species <= 8, SMCX_STORAGE_4BIT.
//
// Layout facts the kernel rests on:
//  * FCC is four interpenetrating simple-cubic sublattices (basis index b, beta_b = (0,0,0), (0,1,1), (1,0,1),
//    (1,1,0) in units of a/2; beta as bit vectors form a group under XOR: beta_{b ^ k} = beta_b ^ beta_k).
//    With 4 bits per site a row of 8 conventional cells of ONE sublattice is one 32-bit word (cell X = nibble X),
//    in device memory (Store4, lattice_kernels.cuh) and in the shared-memory tile alike: 4 sublattices x 64 rows
//    (y + 8 z of the 8^3-cell LIZ+ tile) = 256 words = 1 KB per link cell, word (s * 64 + row) of lane l at
//    tile[(s * 64 + row) * 32 + l], so the 32 cells of a warp never share a bank.
//  * Seen from a site of sublattice bs at nibble X of row r, the 42 neighbours sort by partner sublattice bs ^ k:
//      k = 0 (same sublattice): shell 1 -- nibbles X -+ 1 of row r, nibble X of rows r -+ 1, r -+ 8;
//      k = 1 (long axis x): a 3 x 2 x 2 block, nibbles X - 1 .. X + 1 of rows (oy .. oy + 1, oz .. oz + 1): the middle
//            nibbles are shell 0, the outer ones shell 2;
//      k = 2 (long axis y): nibbles X + ox, X + ox + 1 of rows y - 1 .. y + 1 (dy = 0: shell 0, else shell 2) x (oz, oz + 1);
//      k = 3 (long axis z): the same with y and z exchanged;
//    with o_a = beta_a(bs) - 1, i.e. the block starts one cell lower along axis a when the site's beta_a is 0.  Which
//    rows and which nibbles depends on k only; bs and X merely move four row pointers and two rotation amounts.
//    Hence ONE gather routine serves the site i (compile-time b) and its partner j (whose sublattice, row and
//    column come from a 12-entry table per b indexed by the drawn direction): 21 row loads per site.
//  * A row is rotated (one funnel shift) so that its wanted nibbles land on the free nibbles of an accumulator
//    and merged with one bit-select; every accumulator holds four nibbles of ONE shell in its low 16 bits.
//  * dE needs sum_n D_s(sigma_n), D_s(x) = V_s(b,x) - V_s(a,x), over the neighbours of i minus the same over the
//    neighbours of j, plus corr(a,b) = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) for the i-j bond both sums include.  The
//    four nibbles of an accumulator are the selectors of a byte permute (PRMT) whose two source registers hold the
//    eight values (D_s(x) + 32768) & 255, x = 0..7 -- a look-up of four neighbours in one instruction; a second PRMT
//    looks up (D_s(x) + 32768) >> 8, and two byte dot products with 0x01010101 (IDP.4A) add the bytes up.  The
//    offsets and the empty nibbles (species code 0) occur equally often for i and for j and cancel.  Pure integer
//    arithmetic: dE is exactly the oracle's before/after difference.
// Acceptance: the two-level filter of sweep_thread.cuh (exact look-up in global memory when u falls within E of
// the bound).  One block of kFccWarps warps per SM for a whole colour pass; warps fetch batches of 32 cells from a
// counter in DevState (the four sub-partitions hold different numbers of warps, so a static split would wait for
// the fullest one).
#pragma once
#include <algorithm>
#include <type_traits>
#include <vector>
#include "smcx_common.cuh"
#include "sweep_thread.cuh"   // prmt, lop3, smem helpers, acceptance filter, store_tile_bytes, factored Philox
#include "sweep_warp.cuh"

namespace smcxk {

constexpr int kFccWarps = 12;                // 12 x 16 KB of tile windows + tables in 227 KB
constexpr int kFccRows = 64;                 // rows (y + 8 z) per sublattice of a whole tile (8 layers)
constexpr int kFccWinLayers = 4;             // z layers per sublattice the kernel keeps in shared memory at a time
constexpr int kFccWinRows = 8 * kFccWinLayers;
constexpr int kFccMaxSpecies = 8;            // PRMT selectors are 3 bits
constexpr int kFccBias = 32768;              // D + bias is looked up as two unsigned bytes

__host__ __device__ constexpr int fcc_beta(int b, int axis) {   // S0: basis positions, units of a/2
  return axis == 0 ? ((b >> 1) & 1) : axis == 1 ? (b & 1) : (((b >> 1) ^ b) & 1);
}

// ROWS = 64: the whole tile, row y + 8 z of sublattice s at word s * 64 + row.
// ROWS < 64 (the kernel's window of kFccWinLayers layers): the trials of layer lz of the cell (tile layer lz + 2) reach
// three half-units up and down, i.e. tile layers lz + 1 .. lz + 4 of the sublattices with beta_z = 0 and lz .. lz + 3 of
// those with beta_z = 1 -- four layers each.  Sublattice s keeps tile layer rz in slot rz - lz - (1 - beta_z(s)); seen
// from the row pointers of the gather this is a constant offset per sublattice (sub()), so the trial code is the same.
template <int NT, int ROWS = kFccRows> struct FccTile {
  static constexpr int kRow = 4 * NT;                 // bytes from one row to the next (NT lanes interleaved)
  static constexpr int kSub = ROWS * kRow;            // bytes from one sublattice to the next (ROWS rows each)
  __host__ __device__ static constexpr int sub(int s) {   // byte offset of row 0 of (virtual) slot 0 of sublattice s
    return s * kSub - (ROWS < kFccRows ? (1 - fcc_beta(s, 2)) * 8 * kRow : 0);
  }
};

// Direction table, [b][dir]: what the partner j = i + O_0[dir] of a site of sublattice b needs.
//   d[k]: byte offset from i's own row pointer to the base row of j's partner sublattice k (k = 0: j's own row);
//   e3, e2: a3_j = a3_i + e3, a2_j = 4 X + e2 (rotation amounts, see fcc_site).
// Full-width fields: two 16-byte loads per trial and no unpacking (the 16-bit packed form cost eight integer-pipe
// instructions per trial, and that pipe is what binds the kernel: profiles/r2_fcc_kernel_ncu.md).
struct FccDirEntry { int32_t d[4]; int32_t e3, e2, pad0, pad1; };
struct FccTables { FccDirEntry dir[4][12]; };

// offset (rows) of the base row of partner sublattice bs ^ k relative to the site's own row
__host__ __device__ constexpr int fcc_base_adj(int bs, int k) {
  const int oy = fcc_beta(bs, 1) - 1, oz = fcc_beta(bs, 2) - 1;
  return k == 1 ? oy + 8 * oz : k == 2 ? 8 * oz : k == 3 ? oy : 0;
}

// Host: the table for row stride NT, from the shell-0 offsets of G (ascending (dz, dy, dx), S0).
template <int NT, int ROWS = kFccRows>
inline bool fcc_build_tables(const Geom& G, FccTables& T) {
  if (G.Z0 != 12) return false;
  for (int b = 0; b < 4; ++b)
    for (int d = 0; d < 12; ++d) {
      int cell[3], bits = 0;
      for (int a = 0; a < 3; ++a) {
        const int p = fcc_beta(b, a) + G.off[d][a];          // -1 .. 2
        cell[a] = p < 0 ? -1 : p >> 1;
        bits |= (p & 1) << a;
      }
      // parity (x, y, z) -> basis index: 000 -> 0, 110 (y, z) -> 1, 101 (x, z) -> 2, 011 (x, y) -> 3
      const int bj = bits == 0 ? 0 : bits == 6 ? 1 : bits == 5 ? 2 : bits == 3 ? 3 : -1;
      if (bj < 0) return false;
      const int dr = cell[1] + 8 * cell[2];
      FccDirEntry& e = T.dir[b][d];
      for (int k = 0; k < 4; ++k)
        e.d[k] = FccTile<NT, ROWS>::sub(bj ^ k) - FccTile<NT, ROWS>::sub(b) + (dr + fcc_base_adj(bj, k)) * FccTile<NT, ROWS>::kRow;
      e.e3 = 4 * cell[0];
      e.e2 = 4 * (cell[0] + fcc_beta(bj, 0) - 1);
      e.pad0 = e.pad1 = 0;
    }
  return true;
}

inline bool fcc_kernel_supported(const Geom& G) {
  return G.lattice == 1 && G.n_shells >= 1 && G.n_shells <= 3 && G.w == 4 && G.n_species <= kFccMaxSpecies && G.H == 2 &&
         G.TW == 8 && (G.Lx & 7) == 0 && (long long)G.Lx * G.Ly * G.Lz / 2 < (1ll << 32);
}

// Host: look-up rows.  lut[((a * 8 + b) * 3 + s) * rep + slot] = { lo(x = 0..3), lo(x = 4..7), hi(0..3), hi(4..7) } with
// lo / hi the low / high byte of D_s(x) + kFccBias, D_s(x) = V_s(b,x) - V_s(a,x) (0 for x >= n_species or s >= n_shells),
// replicated `rep` times so that the lanes of a quarter warp read different banks; corr[a * 8 + b].
// Returns false if a difference does not fit (|D| < kFccBias) or dE could overflow int32.
inline bool fcc_build_lut(const int32_t* epi, int n, int n_shells, int rep, std::vector<uint32_t>& lut, std::vector<int32_t>& corr) {
  auto V = [&](int s, int a, int b) -> long long {
    return (s < n_shells && a < n && b < n) ? (long long)epi[(s * n + a) * n + b] : 0ll;
  };
  lut.assign((size_t)64 * 3 * rep * 4, 0u);
  corr.assign(64, 0);
  for (int a = 0; a < 8; ++a)
    for (int b = 0; b < 8; ++b) {
      for (int s = 0; s < 3; ++s) {
        uint32_t w[4] = {0u, 0u, 0u, 0u};
        for (int x = 0; x < 8; ++x) {
          const long long D = (a < n && b < n) ? V(s, b, x) - V(s, a, x) : 0ll;
          if (D <= -kFccBias || D >= kFccBias) return false;
          const uint32_t e = (uint32_t)(D + kFccBias);
          w[x >> 2] |= (e & 0xFFu) << (8 * (x & 3));
          w[2 + (x >> 2)] |= (e >> 8) << (8 * (x & 3));
        }
        for (int slot = 0; slot < rep; ++slot)
          for (int k = 0; k < 4; ++k) lut[(((size_t)(a * 8 + b) * 3 + s) * rep + slot) * 4 + k] = w[k];
      }
      corr[a * 8 + b] = (int32_t)(2 * V(0, a, b) - V(0, a, a) - V(0, b, b));
    }
  return true;
}

// ---- portable helpers (device instructions with host equivalents, so that the trial arithmetic can be unit-tested) ----
__host__ __device__ __forceinline__ uint32_t rotr32(uint32_t w, uint32_t amt) {
#ifdef __CUDA_ARCH__
  return __funnelshift_r(w, w, amt);            // one SHF, amount taken modulo 32
#else
  amt &= 31u;
  return amt ? (w >> amt) | (w << (32u - amt)) : w;
#endif
}
// c + sum of the four bytes of a (all unsigned): IDP.4A with the multiplier 0x01010101
__host__ __device__ __forceinline__ uint32_t add_bytes(uint32_t a, uint32_t c) {
#ifdef __CUDA_ARCH__
  uint32_t d;
  asm("dp4a.u32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(0x01010101u), "r"(c));
  return d;
#else
  return c + (a & 0xFFu) + ((a >> 8) & 0xFFu) + ((a >> 16) & 0xFFu) + (a >> 24);
#endif
}
// A site as the gather sees it: row pointers (into this lane's tile) of the four partner sublattices (own row; base
// rows of k = 1, 2, 3) and the rotation amounts that bring the window X - 1 .. X + 1 (a3) / X + ox, X + ox + 1 (a2)
// to nibble 0.  Tile rows are read and written through ordinary pointers (the swaps of one trial must be seen by
// the loads of the next); the read-only tables go through the lds_* helpers of sweep_thread.cuh.
struct FccSite { const uint32_t *p0, *p1, *p2, *p3; uint32_t a3, a2; };

template <int NT>
__host__ __device__ __forceinline__ const uint32_t* fcc_at(const uint32_t* p, int bytes) {
  return reinterpret_cast<const uint32_t*>(reinterpret_cast<const char*>(p) + bytes);
}
template <int NT, int ROWS>
__host__ __device__ __forceinline__ uint32_t fcc_ld(const uint32_t* p) { return p[ROWS * NT]; }

struct FccLut { uint32_t lo03, lo47, hi03, hi47; };

// look up the four nibbles in the low 16 bits of sel and add the bytes to (lo, hi)
__host__ __device__ __forceinline__ void fcc_lookup(const FccLut& L, uint32_t sel, uint32_t& lo, uint32_t& hi) {
  lo = add_bytes(prmt(L.lo03, L.lo47, sel), lo);
  hi = add_bytes(prmt(L.hi03, L.hi47, sel), hi);
}

// Sum over the 42 neighbours of the site (plus six empty nibbles) of the low / high bytes of D_s(x) + bias.
// own_rot = the site's own row rotated by a3 (its species sits in nibble 1), loaded by the caller.
template <int NT>
__host__ __device__ __forceinline__ void fcc_site_sum(const FccSite& S, uint32_t own_rot, const FccLut& L0, const FccLut& L1,
                                                      const FccLut& L2, uint32_t& lo, uint32_t& hi) {
  const uint32_t a3 = S.a3, a3m4 = a3 - 4u, a3m8 = a3 - 8u, a3p4 = a3 + 4u, a2 = S.a2, a2m8 = a2 - 8u;
  // A look-up (PRMT) reads the low four nibbles of its selector word only, so an accumulator whose four nibbles all
  // hold neighbours is ONE bit-select of two rotated rows (whatever lands in its upper half is ignored); nibbles
  // that hold no neighbour must be zero (species code 0, cancelling between i and j), which costs a second operation.
  // k = 0: shell 1
  {
    uint32_t A = lop3<kLutSel>(rotr32(fcc_ld<NT, -1>(S.p0), a3), own_rot, 0x00F0u);        // (y - 1): nibble X -> 1; own row: X - 1, X + 1 at 0, 2
    A = lop3<kLutSel>(rotr32(fcc_ld<NT, 1>(S.p0), a3m8), A, 0xF000u);                      // (y + 1): nibble X -> 3
    const uint32_t B0 = rotr32(fcc_ld<NT, -8>(S.p0), a3p4) & 0x000Fu;                      // (z - 1): nibble X -> 0
    const uint32_t B = lop3<kLutAndOr2>(rotr32(fcc_ld<NT, 8>(S.p0), a3), 0x00F0u, B0);     // (z + 1): nibble X -> 1; nibbles 2, 3 empty
    fcc_lookup(L1, A, lo, hi);
    fcc_lookup(L1, B, lo, hi);
  }
  // k = 1: rows (0, 1, 8, 9) of its base row, window X - 1 .. X + 1: middle nibble shell 0, outer nibbles shell 2
  {
    const uint32_t w0 = rotr32(fcc_ld<NT, 0>(S.p1), a3), w1 = rotr32(fcc_ld<NT, 1>(S.p1), a3m4);
    const uint32_t w8 = rotr32(fcc_ld<NT, 8>(S.p1), a3), w9 = rotr32(fcc_ld<NT, 9>(S.p1), a3m4);
    fcc_lookup(L2, lop3<kLutSel>(w1, w0, 0xF0F0u), lo, hi);
    fcc_lookup(L2, lop3<kLutSel>(w9, w8, 0xF0F0u), lo, hi);
    fcc_lookup(L0, lop3<kLutAndOr2>(w1, 0x0F00u, w0 & 0x00F0u), lo, hi);                   // two nibbles empty
    fcc_lookup(L0, lop3<kLutAndOr2>(w9, 0x0F00u, w8 & 0x00F0u), lo, hi);
  }
  // k = 2: rows y - 1 .. y + 1 of two z layers, window of two nibbles: dy = 0 shell 0, else shell 2
  {
    const uint32_t m = rotr32(fcc_ld<NT, -1>(S.p2), a2), c = rotr32(fcc_ld<NT, 0>(S.p2), a2), p = rotr32(fcc_ld<NT, 1>(S.p2), a2m8);
    const uint32_t m8 = rotr32(fcc_ld<NT, 7>(S.p2), a2), c8 = rotr32(fcc_ld<NT, 8>(S.p2), a2m8), p8 = rotr32(fcc_ld<NT, 9>(S.p2), a2m8);
    fcc_lookup(L0, lop3<kLutSel>(c8, c, 0xFF00u), lo, hi);
    fcc_lookup(L2, lop3<kLutSel>(p, m, 0xFF00u), lo, hi);
    fcc_lookup(L2, lop3<kLutSel>(p8, m8, 0xFF00u), lo, hi);
  }
  // k = 3: rows z - 1 .. z + 1 of two y rows: dz = 0 shell 0, else shell 2
  {
    const uint32_t m = rotr32(fcc_ld<NT, -8>(S.p3), a2), m1 = rotr32(fcc_ld<NT, -7>(S.p3), a2m8);
    const uint32_t c = rotr32(fcc_ld<NT, 0>(S.p3), a2), c1 = rotr32(fcc_ld<NT, 1>(S.p3), a2m8);
    const uint32_t p = rotr32(fcc_ld<NT, 8>(S.p3), a2), p1 = rotr32(fcc_ld<NT, 9>(S.p3), a2m8);
    fcc_lookup(L0, lop3<kLutSel>(c1, c, 0xFF00u), lo, hi);
    fcc_lookup(L2, lop3<kLutSel>(m1, m, 0xFF00u), lo, hi);
    fcc_lookup(L2, lop3<kLutSel>(p1, p, 0xFF00u), lo, hi);
  }
}

// Loop-invariant operands of a trial.
struct FccEnv {
  smem_ptr_t lut;            // look-up rows, this lane's replica slot
  smem_ptr_t corr;           // corr[a * 8 + b]
  smem_ptr_t filt;           // Tr[64] then Tq[1024]
  uint32_t lut_pair_bytes;   // bytes from one ordered pair to the next = 3 * rep * 16
  uint32_t lut_shell_bytes;  // bytes from one shell to the next = rep * 16
  const uint32_t* accept;
  int accept_len, filter_E;
  int direct_len;            // MODE 2: entries of T held in shared memory at filt (followed by one bound entry)
};

__host__ __device__ __forceinline__ FccLut fcc_load_lut(smem_ptr_t p) {
  const int4 v = lds_int4(p, 0);
  return FccLut{(uint32_t)v.x, (uint32_t)v.y, (uint32_t)v.z, (uint32_t)v.w};
}

// One trial (a4-a6).  p_own: row r of sublattice b in this lane's tile; X4 = 4 X, X the nibble of site i; E = the
// direction-table entry of (b, drawn direction); u = acceptance draw.
// MODE (acceptance): 0 = T[dE] from global memory, 1 = two-level filter in shared memory (exact look-up in global memory
// when u falls within E of the bound), 2 = the first direct_len entries of T in shared memory at env.filt, followed by
// the bound T[direct_len] (0 when that is the whole table): T does not increase, so for dE >= direct_len a draw
// u >= T[direct_len] is a rejection and only a smaller one (rare: T[direct_len] is small) needs T[dE] from global memory.
template <int b, int NT, int MODE, int ROWS = kFccRows>
__host__ __device__ __forceinline__ void fcc_trial(uint32_t* p_own, uint32_t X4, const FccDirEntry& E, uint32_t u,
                                                   const FccEnv& env, int& esum, unsigned& nacc) {
  using T = FccTile<NT, ROWS>;
  FccSite si, sj;
  si.p0 = p_own;
  si.p1 = fcc_at<NT>(p_own, T::sub(b ^ 1) - T::sub(b) + fcc_base_adj(b, 1) * T::kRow);
  si.p2 = fcc_at<NT>(p_own, T::sub(b ^ 2) - T::sub(b) + fcc_base_adj(b, 2) * T::kRow);
  si.p3 = fcc_at<NT>(p_own, T::sub(b ^ 3) - T::sub(b) + fcc_base_adj(b, 3) * T::kRow);
  si.a3 = X4 - 4u;
  si.a2 = X4 + (uint32_t)(4 * (fcc_beta(b, 0) - 1));
  sj.p0 = fcc_at<NT>(p_own, E.d[0]);
  sj.p1 = fcc_at<NT>(p_own, E.d[1]);
  sj.p2 = fcc_at<NT>(p_own, E.d[2]);
  sj.p3 = fcc_at<NT>(p_own, E.d[3]);
  sj.a3 = si.a3 + (uint32_t)E.e3;
  sj.a2 = X4 + (uint32_t)E.e2;
  const uint32_t own_i = rotr32(fcc_ld<NT, 0>(si.p0), si.a3), own_j = rotr32(fcc_ld<NT, 0>(sj.p0), sj.a3);
  const uint32_t a = (own_i >> 4) & 7u, sb = (own_j >> 4) & 7u;
  const uint32_t pair = a * 8u + sb;
  const smem_ptr_t lp = smem_index(env.lut, pair, env.lut_pair_bytes);
  const FccLut L0 = fcc_load_lut(lp), L1 = fcc_load_lut(lp + env.lut_shell_bytes), L2 = fcc_load_lut(lp + 2u * env.lut_shell_bytes);
  const int corr = (int)lds_u32(env.corr, pair * 4u);
  uint32_t lo_i = 0u, hi_i = 0u, lo_j = 0u, hi_j = 0u;
  fcc_site_sum<NT>(si, own_i, L0, L1, L2, lo_i, hi_i);
  fcc_site_sum<NT>(sj, own_j, L0, L1, L2, lo_j, hi_j);
  const int dE = (int)(lo_i - lo_j) + 256 * (int)(hi_i - hi_j) + corr;
  // Eq. 3 in integer form
  bool ok;
  if (MODE == 2) {
    // dE <= 0 (huge as unsigned) and dE >= direct_len clamp to the bound entry behind the table
    uint32_t thr = lds_u32(env.filt, 4u * min((uint32_t)dE, (uint32_t)env.direct_len));
    // beyond the resident part: T[dE] itself, by a predicated load (no branch: the trial stays one basic block); the
    // library keeps a zero entry behind T in device memory, which serves dE >= len
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
  atomicXor(const_cast<uint32_t*>(si.p0), x << X4);             // shared-memory ATOMS: no read-modify-write chain in registers
  atomicXor(const_cast<uint32_t*>(sj.p0), x << (sj.a3 + 4u));
#else
  *const_cast<uint32_t*>(si.p0) ^= x << X4;
  *const_cast<uint32_t*>(sj.p0) ^= x << (sj.a3 + 4u);
#endif
  esum += ok ? dE : 0;
  nacc += ok ? 1u : 0u;
}

#ifdef __CUDACC__
__device__ __forceinline__ int2 lds_int2(smem_ptr_t addr) {
  int2 v;
  asm("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
  return v;
}
constexpr int kFccSmemMax = 232448 - 1536;                     // 227 KB less the static part / reserve
// dynamic shared memory: tile windows of `warps` warps, look-up rows, corr, direction table, then the filter tables
// (accept_words = kFilterWords) or the whole threshold table plus its zero entry (accept_words = len + 1)
inline size_t fcc_smem_bytes(int rep, int warps = kFccWarps, size_t accept_words = kFilterWords) {
  return (size_t)warps * FccTile<32, kFccWinRows>::kSub * 4 + (size_t)64 * 3 * rep * 16 + 64 * 4 + sizeof(FccTables) + accept_words * 4;
}
// replicas of the look-up rows: as many (8, 4, 2, 1) as fit next to the tiles
inline int fcc_lut_rep(int n_species) {
  (void)n_species;
  for (int rep = 8; rep >= 1; rep >>= 1)
    if (fcc_smem_bytes(rep) <= (size_t)kFccSmemMax) return rep;
  return 1;
}
// Acceptance from the table itself (MODE 2) when at least kFccDirectMin of its entries fit shared memory next to
// kFccDirectWarps warps of tiles (beyond them T is small and the exact look-up in global memory rare); measured on
// FCC 640^3: the table next to 10 / 9 / 8 / 7 warps 7.87 / 7.65 / 7.42 / 7.04e10 against 7.50e10 with the two-level
// filter and twelve warps.  Returns the number of entries to hold (<= accept_len), or 0: then the filter serves.
constexpr int kFccDirectWarps = 11;
constexpr int kFccDirectMin = 4096;
inline int fcc_direct_entries(int rep, int accept_len, int* warps) {
  if (fcc_smem_bytes(rep, kFccWarps, (size_t)accept_len + 1) <= (size_t)kFccSmemMax) { *warps = kFccWarps; return accept_len; }
  *warps = kFccDirectWarps;
  const size_t fixed = fcc_smem_bytes(rep, kFccDirectWarps, 1);
  if (fixed > (size_t)kFccSmemMax) return 0;
  const size_t room = ((size_t)kFccSmemMax - fixed) / 4;
  if (room >= (size_t)accept_len) return accept_len;
  return room >= (size_t)kFccDirectMin ? (int)room : 0;
}

template <int MODE>
__global__ void __launch_bounds__(kFccWarps * 32, 1)
sweep_fcc_thread(const Geom G, const FccTables FT, uint32_t* __restrict__ lattice, const uint4* __restrict__ lut,
                 const int32_t* __restrict__ corr, int rep, const uint32_t* __restrict__ accept,
                 const uint32_t* __restrict__ filt, DevState* __restrict__ st, int colour, int direct_len) {
  constexpr int NT = 32;
  extern __shared__ __align__(16) uint32_t smem_w[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  constexpr int WR = kFccWinRows;                                              // rows per sublattice of the resident window
  uint32_t* tile = smem_w + warp * (4 * WR * NT) + lane;                       // word (s * WR + row) at tile[(s * WR + row) * NT]
  uint4* s_lut = reinterpret_cast<uint4*>(smem_w + n_warps * (4 * WR * NT));
  int32_t* s_corr = reinterpret_cast<int32_t*>(s_lut + 64 * 3 * rep);
  // direction table as three arrays of 8-byte entries (row offsets d0, d1; d2, d3; rotation amounts): the twelve entries
  // of a sublattice lie in 24 different banks, so the lanes of a warp, each with its own direction, never collide (with
  // 32-byte entries side by side a 16-byte load took 2.3 wavefronts per quarter warp)
  int2* s_dir = reinterpret_cast<int2*>(s_corr + 64);
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(s_dir + 3 * 48);              // filter tables, or the whole table T + a zero entry
  __shared__ uint2 s_slot[128];                                                // Philox products that depend on the slot pair only
  __shared__ long long s_e64[kFccWarps];
  __shared__ unsigned s_acc[kFccWarps];

  for (int k = threadIdx.x; k < 64 * 3 * rep; k += blockDim.x) s_lut[k] = lut[k];
  for (int k = threadIdx.x; k < 64; k += blockDim.x) s_corr[k] = corr[k];
  if (MODE == 1)
    for (int k = threadIdx.x; k < kFilterWords; k += blockDim.x) s_filt[k] = filt[k];
  if (MODE == 2)
    for (int k = threadIdx.x; k <= direct_len; k += blockDim.x) s_filt[k] = k < G.accept_len ? accept[k] : 0u;
  for (int k = threadIdx.x; k < 48; k += blockDim.x) {
    const FccDirEntry& e = FT.dir[k / 12][k % 12];
    s_dir[k] = make_int2(e.d[0], e.d[1]);
    s_dir[48 + k] = make_int2(e.d[2], e.d[3]);
    s_dir[96 + k] = make_int2(e.e3, e.e2);
  }
  const uint32_t t = (uint32_t)st->sweep;
  if (threadIdx.x < 128) s_slot[threadIdx.x] = philox_slot_entry(threadIdx.x, t, G.rk0, G.rk1);
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
      // The tile of a cell is 8 layers of conventional cells, but the trials of layer lz of the cell only touch four
      // layers of every sublattice (FccTile): the kernel keeps those resident (16 KB per warp: twelve warps per SM) and
      // runs the cell in four steps.  Between two steps the lowest layer of every window is written back (it is final:
      // later trials only reach higher layers), the other three move down a slot and one new layer is staged.
      // Class 1 = sublattices 0, 3 (beta_z = 0, window tile layers lz + 1 .. lz + 4), class 0 = sublattices 1, 2 (lz .. lz + 3).
      uint32_t offy[8];
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        offy[ry] = (uint32_t)gy * (uint32_t)rw;
      }
      const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
      const PhiloxCell pc = philox_cell_setup(cell_id, t, ctr3, G.rk0, G.rk1);
      const uint32_t dwh = (uint32_t)(whi - wlo) * 4u;            // word step from the low to the high group of a row
      uint32_t* const peer = reinterpret_cast<uint32_t*>(G.peer_lat);
      int esum = 0;
      // a3: stage tile layer rz of the two sublattices of a class into a slot: per row two 16-byte groups (four
      // sublattice words each, two of them used), funnel-shifted into the tile words
      auto stage = [&](auto cls_c, int slot, int rz) {
        constexpr int CLS = decltype(cls_c)::value;
        int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
        const uint32_t zoff = (uint32_t)gz * zstride;
        uint4 lo[8], hi[8];
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          const uint4* row = reinterpret_cast<const uint4*>(lattice) + (zoff + offy[ry]);
          lo[ry] = row[wlo];
          hi[ry] = row[whi];
        }
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          uint32_t* d = tile + (slot * 8 + ry) * NT;
          if (CLS) {
            d[0 * WR * NT] = __funnelshift_r(lo[ry].x, hi[ry].x, sh);
            d[3 * WR * NT] = __funnelshift_r(lo[ry].w, hi[ry].w, sh);
          } else {
            d[1 * WR * NT] = __funnelshift_r(lo[ry].y, hi[ry].y, sh);
            d[2 * WR * NT] = __funnelshift_r(lo[ry].z, hi[ry].z, sh);
          }
        }
      };
      // a7: write back rows 1..6 of the layers that leave the windows after step lz - 1 (lz = 4: of everything still
      // resident), tile layers 1..6 only: the bytes that lie wholly inside this tile
      auto wb = [&](auto cc, int lz) {
        constexpr int C = decltype(cc)::value;
#pragma unroll 1
        for (int cls = 0; cls < 2; ++cls) {
          const int first = lz - 1 + cls, n_slots = lz == 4 ? 4 : 1;
          const int sa = cls ? 0 : 1, sb = cls ? 3 : 2;
#pragma unroll 1
          for (int slot = 0; slot < n_slots; ++slot) {
            const int rz = first + slot;
            if (rz < 1 || rz > 6) continue;
            int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
            // fused ghost-layer message: layers the neighbour slab holds a copy of also go into its storage
            const bool mirror = peer != nullptr && gz >= G.peer_z0 && gz < G.peer_z1;
#pragma unroll
            for (int ry = 1; ry < 7; ++ry) {
              const uint32_t base = (((uint32_t)gz * zstride) + offy[ry] + (uint32_t)wlo) * 4u;
#pragma unroll
              for (int q = 0; q < 2; ++q) {
                const int sq = q ? sb : sa;
                const uint32_t v = tile[(sq * WR + slot * 8 + ry) * NT];
                store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(lattice + base + sq),
                                                     reinterpret_cast<unsigned char*>(lattice + (uint32_t)(base + sq + dwh)), v);
                if (mirror)
                  store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(peer + base + sq),
                                                       reinterpret_cast<unsigned char*>(peer + (uint32_t)(base + sq + dwh)), v);
              }
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
#pragma unroll 1
      for (int lz = 0; lz < 4; ++lz) {
        if (lz > 0) {
          write_back(lz);
          // slots 1..3 of every sublattice move down one slot
#pragma unroll 1
          for (int s = 0; s < 4; ++s) {
            uint32_t* d = tile + s * WR * NT;
#pragma unroll 8
            for (int r = 0; r < 24; ++r) d[r * NT] = d[(r + 8) * NT];
          }
        }
#pragma unroll 1
        for (int slot = lz ? 3 : 0; slot < 4; ++slot) {
          stage(std::integral_constant<int, 0>{}, slot, lz + slot);
          stage(std::integral_constant<int, 1>{}, slot, lz + 1 + slot);
        }
        // a4-a6: the 64 trials of layer lz of the cell, raster order: conventional cell c = (lz * 4 + ly) * 4 + lx, then b;
        // site i sits in (virtual) slot 2 of its sublattice's window
        using TW = FccTile<NT, WR>;
#pragma unroll 1
        for (int c = 16 * lz; c < 16 * lz + 16; ++c) {
          const uint32_t X4 = 4u * (uint32_t)((c & 3) + 2);
          uint32_t* p_row = tile + (((c >> 2) & 3) + 2 + 16) * NT;
          const Philox4 r0 = philox_factored(pc, s_slot[2 * c], G.rk0, G.rk1);
          const Philox4 r1 = philox_factored(pc, s_slot[2 * c + 1], G.rk0, G.rk1);
#define SMCX_FCC_TRIAL(B, WDIR, U)                                                                          \
          {                                                                                                   \
            const smem_ptr_t ep = dir_p + (B * 12u + mulhi_u32(WDIR, 12u)) * 8u;                             \
            const int2 e = lds_int2(ep), g = lds_int2(ep + 48u * 8u), f = lds_int2(ep + 96u * 8u);            \
            const FccDirEntry E{{e.x, e.y, g.x, g.y}, f.x, f.y, 0, 0};                                        \
            fcc_trial<B, NT, MODE, WR>(const_cast<uint32_t*>(fcc_at<NT>(p_row, TW::sub(B))), X4, E, U, env, esum, nacc); \
          }
          SMCX_FCC_TRIAL(0, r0.x, r0.y) SMCX_FCC_TRIAL(1, r0.z, r0.w) SMCX_FCC_TRIAL(2, r1.x, r1.y) SMCX_FCC_TRIAL(3, r1.z, r1.w)
#undef SMCX_FCC_TRIAL
        }
      }
      write_back(4);
      esum_total += esum;     // |dE| < 2^23 (host check), 256 trials: exact in int32 per cell
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
    for (int i = 0; i < n_warps; ++i) { e += s_e64[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

inline int configure_fcc_thread(int rep) {
  (void)rep;
  if (cudaFuncSetAttribute(sweep_fcc_thread<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFccSmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_fcc_thread<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFccSmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_fcc_thread<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kFccSmemMax) != cudaSuccess) return -1;
  cudaFuncSetAttribute(sweep_fcc_thread<0>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_fcc_thread<1>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_fcc_thread<2>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  return 0;
}

inline int launch_fcc_thread(const Geom& G, const FccTables& FT, uint32_t* lattice, const uint32_t* d_lut, const int32_t* d_corr,
                             int rep, const uint32_t* accept, const uint32_t* d_filter, DevState* st, int colour, int sm_count,
                             int tail_from, cudaStream_t stream) {
  const unsigned n_batches = (G.cells_per_colour + 31u) / 32u;
  int warps = kFccWarps;
  int direct = fcc_direct_entries(rep, G.accept_len, &warps);
  // the head of T only: sound if T[direct] bounds every later entry (tail_from: checked by the host at upload)
  if (direct < G.accept_len && direct < tail_from) direct = 0;
  if (direct == 0) warps = kFccWarps;
  const unsigned want = (n_batches + warps - 1) / warps;
  const unsigned grid = want < (unsigned)sm_count ? want : (unsigned)sm_count;
  const uint4* lut4 = reinterpret_cast<const uint4*>(d_lut);
  if (direct > 0)
    sweep_fcc_thread<2><<<grid, warps * 32, fcc_smem_bytes(rep, warps, (size_t)direct + 1), stream>>>(
        G, FT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, direct);
  else if (G.filter_E >= 0)
    sweep_fcc_thread<1><<<grid, warps * 32, fcc_smem_bytes(rep), stream>>>(G, FT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, 0);
  else
    sweep_fcc_thread<0><<<grid, warps * 32, fcc_smem_bytes(rep), stream>>>(G, FT, lattice, lut4, d_corr, rep, accept, d_filter, st, colour, 0);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}
#endif  // __CUDACC__

}  // namespace smcxk
