// Thread-per-cell colour-pass kernel: BCC, first two shells, link cell w = 4, <= 4 species,
// 2-bit packed storage (16 sites per 32-bit word in site-id order).
//
// Layout facts this kernel rests on:
//  * a row of 8 conventional cells (both sublattices) is exactly one 32-bit word: conventional
//    cell X is nibble X, its corner site the low two bits, its body site the high two;
//  * with w = 4 the LIZ+ tile is 8^3 conventional cells = 64 such words, and the tiles of the
//    cells of one colour tile the whole lattice exactly once, so a pass streams the lattice
//    through shared memory once and no two threads ever touch the same tile;
//  * the tile of thread t is kept at smem[row * NT + t]: every access of a warp hits 32 distinct
//    banks whatever row each lane addresses (lanes differ in the direction they drew);
//  * the neighbours of a site sit in at most two adjacent nibbles of four (shell 0) or five
//    (shell 1) rows.  They are gathered with byte permutes (PRMT) of 16-bit windows and one
//    bit-select per four rows; because the neighbours of i and of j lie on opposite sublattices,
//    the gathered words of i and (complemented) j interleave into one dense word per shell with a
//    single three-input logic operation.  Population counts then give, with species x = lo + 2 hi,
//      D_s(x) = V_s(b,x) - V_s(a,x) = D_s(0) + lo cl_s + hi ch_s + lo hi cb_s,
//    dE = sum_s [cl_s dlo_s + ch_s dhi_s + cb_s dboth_s] + corr(a,b), d* the differences of the
//    bit counts around i and around j, corr = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) undoing the i-j
//    bond that both sums include.  Integer arithmetic throughout: results are bit-identical to
//    the plain before/after energy difference;
//  * the site i of a trial is known at compile time (the 128 slots are unrolled per x-row), only
//    the direction is per lane: its y/z bits select rows (shared-memory addresses), its x bit
//    selects between two sets of masks (one multiply-add per mask on the FMA pipe).
//  * the integer pipe (LOP3/SHF/PRMT/ISETP) is the binding unit (ncu: profiles/), so everything
//    is arranged to keep its instruction count down.
#pragma once
#include <algorithm>
#include <cstdlib>
#include "smcx_common.cuh"
#include "sweep_warp.cuh"

namespace smcxk {

// Acceptance variants of trial_thread (template parameter MODE)
constexpr int kAcceptGlobal = 0;   // explicit a != b test, T[dE] from global memory
constexpr int kAcceptFilter = 1;   // two-level filter tables in shared memory, rare exact look-up
constexpr int kAcceptDirect = 2;   // the whole table T (plus one zero entry) in shared memory
constexpr int kThreadNT = 128;          // threads (= cells) per block of sweep_thread_per_cell
constexpr int kThreadBlocksPerSM = 5;   // 128 x 5 measured best (profiles/README.md, block shapes)
constexpr int kThreadTileWords = 64;    // 8 x 8 rows of one word
constexpr int kCoefInts = 8;            // per (a,b): cl0 ch0' cb0 cl1 | ch1' cb1 corr' pad
constexpr int kFilterTr = 64;           // Tr[r] = T[r], r < 64
constexpr int kFilterMaxTq = 1024;      // Tq[q] = T[64 q]
constexpr int kFilterWords = kFilterTr + kFilterMaxTq;
constexpr int kFilterDmax = 64 * kFilterMaxTq - 1;   // largest dE the filter tables cover (zero entries at the top)
constexpr int32_t kSameSpecies = kFilterDmax - 31;   // "dE" of a trial between equal species: never accepted
constexpr int kDEScale = 4;                          // the kernel computes 4 dE (= byte offset into Tr)

inline bool thread_kernel_supported(const Geom& G) {
  // the last condition keeps word indices of the packed lattice (16 sites per word) in 32 bits
  return G.lattice == 0 && G.n_shells == 2 && G.w == 4 && G.n_species <= 4 && G.H == 2 && G.TW == 8 &&
         (long long)G.Lx * G.Ly * G.Lz / 8 < (1ll << 32);
}

// Host: coefficient table from the EPI tables, [a*4+b][8] int32.  With PT / PH / PB the population
// counts of trial_thread (all fields, high bits, both bits; j's fields complemented, Z_s of them):
//   dE = corr' + sum_s cl_s PT_s + (ch_s - cl_s) PH_s + cb_s PB_s,
//   corr' = corr - sum_s Z_s (cl_s + ch_s + cb_s).
// The table holds kDEScale times these values.  Entries with a == b hold kSameSpecies in corr' and
// zeros elsewhere.  Returns, from the bound |dE| <= 2 sum_s Z_s max_x |D_s(x)| + |corr|:
//   0  the sum of kDEScale dE over the 128 trials of a cell could overflow the int32 a thread accumulates it in
//      (bound >= 2^22): the kernel cannot be used;
//   1  exact, but dE can reach kSameSpecies: only the variant without the filter tables applies;
//   2  every dE of a trial between different species is below kSameSpecies: the filter variant applies.
inline int build_thread_coefficients(const int32_t* epi, int n_species, int32_t* coef /*16*8*/) {
  auto V = [&](int s, int a, int b) -> long long {
    return (a < n_species && b < n_species) ? (long long)epi[(s * n_species + a) * n_species + b] : 0ll;
  };
  const int Z[2] = {8, 6};
  int cls = 2;
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b) {
      int32_t* c = coef + (a * 4 + b) * kCoefInts;
      for (int k = 0; k < kCoefInts; ++k) c[k] = 0;
      if (a == b) { c[6] = kDEScale * kSameSpecies; continue; }
      long long corr = 2 * V(0, a, b) - V(0, a, a) - V(0, b, b);
      long long bound = std::llabs(corr);
      for (int s = 0; s < 2; ++s) {
        long long D[4], maxD = 0;
        for (int x = 0; x < 4; ++x) { D[x] = V(s, b, x) - V(s, a, x); maxD = std::max(maxD, std::llabs(D[x])); }
        const long long cl = D[1] - D[0], ch = D[2] - D[0], cb = D[3] - D[1] - D[2] + D[0];
        c[3 * s + 0] = (int32_t)(kDEScale * cl); c[3 * s + 1] = (int32_t)(kDEScale * (ch - cl));
        c[3 * s + 2] = (int32_t)(kDEScale * cb);
        corr -= Z[s] * (cl + ch + cb);
        bound += 2 * Z[s] * maxD;
      }
      c[6] = (int32_t)(kDEScale * corr);
      if (bound >= kSameSpecies) cls = std::min(cls, 1);
      if (bound >= (1ll << 22)) cls = 0;
    }
  return cls;
}

// Host: the seven coefficients of every ordered pair as signed 16-bit halves, [a*4+b][4] int32:
//   { cl0 | ch0' << 16, cb0 | cl1 << 16, ch1' | cb1 << 16, corr' } (all times kDEScale, as in coef),
// the operand layout of dp2a (two 16-bit factors per word times two population counts packed in bytes).
// Returns false if a coefficient does not fit 16 bits (the persistent kernel then takes the 32-bit rows).
inline bool pack_thread_coefficients(const int32_t* coef /*16*8*/, int32_t* pk /*16*4*/) {
  bool fits = true;
  for (int e = 0; e < 16; ++e) {
    const int32_t* c = coef + e * kCoefInts;
    for (int k = 0; k < 6; ++k) fits = fits && c[k] >= -32768 && c[k] <= 32767;
    for (int k = 0; k < 3; ++k)
      pk[e * 4 + k] = (int32_t)(((uint32_t)c[2 * k] & 0xFFFFu) | ((uint32_t)c[2 * k + 1] << 16));
    pk[e * 4 + 3] = c[6];
  }
  return fits;
}

// Host: two-level filter tables for a threshold table T (T[d] = 0 understood for d >= len).
// Returns E >= 0 such that 0 <= T[d] - mulhi(Tq[d>>6], Tr[d&63]) <= E for all d <= kFilterDmax, or
// -1 if no such small bound holds (then the kernel reads T[d] directly).  For
// T[d] = floor(2^32 exp(-d/kT)) the product of the two floors never exceeds T[d] and falls short
// by a few units at most.  The last Tq slot is kept zero: clamped dE values land there.
inline int build_accept_filter(const uint32_t* T, int len, uint32_t* filt /*kFilterWords*/, int* nq_out) {
  const int nq = (len + 63) / 64;
  *nq_out = nq;
  if (nq > kFilterMaxTq - 1) return -1;
  for (int r = 0; r < kFilterTr; ++r) filt[r] = r < len ? T[r] : 0u;
  for (int q = 0; q < kFilterMaxTq; ++q) filt[kFilterTr + q] = q < nq ? T[64 * q] : 0u;
  uint32_t E = 0;
  for (int d = 0; d < 64 * nq; ++d) {
    const uint32_t ta = (uint32_t)(((uint64_t)filt[kFilterTr + (d >> 6)] * filt[d & 63]) >> 32);
    const uint32_t td = d < len ? T[d] : 0u;
    if (ta > td) return -1;
    E = td - ta > E ? td - ta : E;
  }
  return E <= 1024u ? (int)E : -1;
}

inline void set_thread_masks(Geom& G);   // below, after SlotConst

// ---- bit helpers (host versions exist so that the trial arithmetic can be unit-tested on the CPU) ----
__host__ __device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
#ifdef __CUDA_ARCH__
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));   // no selector masking (__byte_perm adds one)
  return d;
#else
  const uint64_t ab = ((uint64_t)b << 32) | a;
  uint32_t d = 0;
  for (int k = 0; k < 4; ++k) d |= (uint32_t)((ab >> (8 * ((sel >> (4 * k)) & 7u))) & 0xffu) << (8 * k);
  return d;
#endif
}
// d = f(a, b, c) with the truth table LUT (bit (4 a + 2 b + c) of LUT), one LOP3
template <int LUT>
__host__ __device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
#ifdef __CUDA_ARCH__
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
  return d;
#else
  uint32_t d = 0;
  for (int k = 0; k < 8; ++k)
    if ((LUT >> k) & 1) d |= ((k & 4) ? a : ~a) & ((k & 2) ? b : ~b) & ((k & 1) ? c : ~c);
  return d;
#endif
}
constexpr int kLutSel = 0xE4;      // c ? a : b
constexpr int kLutSelNotB = 0xB1;  // c ? a : ~b
constexpr int kLutMaj = 0xE8;      // majority
constexpr int kLutAndOr = 0xE0;    // a & (b | c)
constexpr int kLutAndOr2 = 0xEA;   // (a & b) | c
__host__ __device__ __forceinline__ int popc32(uint32_t v) {
#ifdef __CUDA_ARCH__
  return __popc(v);
#else
  return __builtin_popcount(v);
#endif
}
__host__ __device__ __forceinline__ uint32_t ldg_u32(const uint32_t* p) {
#ifdef __CUDA_ARCH__
  return __ldg(p);
#else
  return *p;
#endif
}

// a * b + c as one IMAD (FMA pipe); written in PTX so that it is not rewritten into shifts and masks
__host__ __device__ __forceinline__ uint32_t mad_u32(uint32_t a, uint32_t b, uint32_t c) {
#ifdef __CUDA_ARCH__
  uint32_t d;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
#else
  return a * b + c;
#endif
}
// c + lo16(a) * byte0(b) + hi16(a) * byte1(b), 16-bit halves signed, bytes unsigned: one IDP.2A (FMA pipe)
__host__ __device__ __forceinline__ int dp2a_lo(uint32_t a, uint32_t b, int c) {
#ifdef __CUDA_ARCH__
  int d;
  asm("dp2a.lo.s32.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
#else
  return c + (int)(int16_t)(a & 0xFFFFu) * (int)(b & 0xFFu) + (int)(int16_t)(a >> 16) * (int)((b >> 8) & 0xFFu);
#endif
}
// Shared-memory tables are addressed on the device by 32-bit shared addresses formed with mad_u32.
#ifdef __CUDA_ARCH__
typedef uint32_t smem_ptr_t;
__device__ __forceinline__ smem_ptr_t smem_ptr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lds_u32(smem_ptr_t base, uint32_t byte_off) {
  uint32_t v;
  asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(base + byte_off));
  return v;
}
__device__ __forceinline__ int4 lds_int4(smem_ptr_t addr, int imm) {
  int4 v;
  asm("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr + imm));
  return v;
}
#else
typedef const char* smem_ptr_t;
inline smem_ptr_t smem_ptr(const void* p) { return reinterpret_cast<const char*>(p); }
inline uint32_t lds_u32(smem_ptr_t base, uint32_t byte_off) { return *reinterpret_cast<const uint32_t*>(base + byte_off); }
inline int4 lds_int4(smem_ptr_t addr, int imm) { return *reinterpret_cast<const int4*>(addr + imm); }
#endif
__host__ __device__ __forceinline__ smem_ptr_t smem_index(smem_ptr_t base, uint32_t idx, uint32_t scale) {
#ifdef __CUDA_ARCH__
  return mad_u32(idx, scale, base);
#else
  return base + idx * scale;
#endif
}

// ---- compile-time description of a trial slot: site i = sublattice bi of tile nibble X ----------
__host__ __device__ constexpr uint32_t nib_mask(int n) { return 0xFu << (4 * n); }
__host__ __device__ constexpr uint32_t sel_win_a(int k) { return (uint32_t)(k | ((k + 1) << 4) | ((4 + k) << 8) | ((5 + k) << 12)); }
__host__ __device__ constexpr uint32_t sel_win_b(int k) { return (uint32_t)((5 + k) | (k << 4) | ((k + 1) << 8) | ((4 + k) << 12)); }
__host__ __device__ constexpr uint32_t sel_byte(int k) { return (uint32_t)(k | ((4 + k) << 4) | (k << 8) | ((4 + k) << 12)); }

template <int bi, int X>
struct SlotConst {
  static constexpr int bj = 1 - bi;
  static constexpr uint32_t Ci = bi ? 0xCCCCCCCCu : 0x33333333u;   // bits of the fields of sublattice bi
  static constexpr uint32_t Cj = ~Ci;
  static constexpr uint32_t kHi = 0xAAAAAAAAu;                     // high bit of every field
  // shell 0 of i: nibbles n0i, n0i + 1 of four rows (fields of sublattice bj)
  static constexpr int n0i = X - 1 + bi;
  static constexpr int ki = (n0i & 1) ? (n0i - 1) / 2 : n0i / 2;   // first byte of the 16-bit window
  static constexpr uint32_t mi = (n0i & 1) ? 0x0FF00FF0u : 0x00FF00FFu;
  // shell 0 of j: nibbles X - 1 + dx, X + dx (fields of sublattice bi); window holds X-1, X, X+1
  static constexpr int kj = (X & 1) ? (X - 1) / 2 : (X - 2) / 2;
  static constexpr uint32_t mj0 = (X & 1) ? 0x00FF00FFu : 0x0FF00FF0u;
  static constexpr uint32_t mj1 = mj0 << 4;
  // shell 1 of i: nibble X of the four adjacent rows, nibbles X - 1 and X + 1 of the own row
  static constexpr uint32_t s2i = sel_byte(X >> 1);
  static constexpr uint32_t moi = nib_mask(X - 1) | nib_mask(X + 1);
  static constexpr uint32_t Mi = ((0x0F0F0F0Fu << (4 * (X & 1))) | moi) & Ci;
  // shell 1 of j: the same around nibble Xj = X0 + dx
  static constexpr int X0 = X - 1 + bi;
  static constexpr uint32_t s2j_f(int dx) { return sel_byte((X0 + dx) >> 1); }
  static constexpr uint32_t moj_f(int dx) { return nib_mask(X0 + dx - 1) | nib_mask(X0 + dx + 1); }
  static constexpr uint32_t Mj_f(int dx) { return ((0x0F0F0F0Fu << (4 * ((X0 + dx) & 1))) | moj_f(dx)) & Cj; }
  static constexpr uint32_t s2j0 = s2j_f(0), s2j1 = s2j_f(1);
  static constexpr uint32_t moj0 = moj_f(0), moj1 = moj_f(1);
  static constexpr uint32_t Mj0 = Mj_f(0), Mj1 = Mj_f(1);
  static constexpr uint32_t swa_i = sel_win_a(ki), swb_i = sel_win_b(ki), swa_j = sel_win_a(kj), swb_j = sel_win_b(kj);
  // own fields, normalised to bits 4..5
  static constexpr int shi = 4 * X + 2 * bi - 4;
  static constexpr int shj0 = 4 * X0 + 2 * bj - 4;                 // + 4 dx
};

// c0 + dx * (c1 - c0): a per-lane choice between two compile-time constants as one IMAD
__host__ __device__ __forceinline__ uint32_t pick(uint32_t dx, uint32_t c0, uint32_t c1) {
  return c0 + dx * (c1 - c0);
}

// Loop-invariant operands of a trial, kept in registers.
struct TrialEnv {
  smem_ptr_t coef;           // coefficient rows of this lane's slot
  smem_ptr_t filt;           // Tr[64] then Tq[1024]
  const uint32_t* accept;    // global threshold table (rare exact look-up)
  int accept_len, filter_E;
  uint32_t tmax4;            // kAcceptDirect: byte offset of the zero entry that ends the table in shared memory
};

// Geom::kc: constants used as the constant-bank operand of an IMAD whose other constant is an
// immediate.  Slot = bi * 4 + X - 2.
constexpr int kKcOne = 0, kKc1111 = 1, kKcMjDelta = 2, kKcShj0 = 10;

template <int bi, int X>
inline void set_slot_constants(Geom& G) {
  using K = SlotConst<bi, X>;
  G.kc[kKcMjDelta + bi * 4 + X - 2] = K::Mj1 - K::Mj0;
  G.kc[kKcShj0 + bi * 4 + X - 2] = (uint32_t)K::shj0;
}

inline void set_thread_masks(Geom& G) {
  for (int r = 0; r < 10; ++r) {
    G.rk0[r] = G.key0 + (uint32_t)r * 0x9E3779B9u;
    G.rk1[r] = G.key1 + (uint32_t)r * 0xBB67AE85u;
  }
  G.kc[kKcOne] = 1u;
  G.kc[kKc1111] = 0x1111u;
  set_slot_constants<0, 2>(G); set_slot_constants<0, 3>(G); set_slot_constants<0, 4>(G); set_slot_constants<0, 5>(G);
  set_slot_constants<1, 2>(G); set_slot_constants<1, 3>(G); set_slot_constants<1, 4>(G); set_slot_constants<1, 5>(G);
}

// One trial (a4-a6).  p_i points at the tile row of site i (row stride STRIDE words).  ra / rb carry
// two rows from one trial of an x-row to the next: a trial with bi == 0 takes rows y-1 and z-1 and
// leaves y+1 and z+1 (which it cannot have modified), a trial with bi == 1 the other way round.
template <int bi, int X, int MODE, int STRIDE, bool PK = false>
__host__ __device__ __forceinline__ void trial_thread(const Geom& G, uint32_t* p_i, const TrialEnv& env, uint32_t w_dir,
                                                      uint32_t u, uint32_t& ra, uint32_t& rb, int& esum4,
                                                      unsigned& nacc) {
  using K = SlotConst<bi, X>;
  constexpr int NT = STRIDE;
  constexpr int slot = bi * 4 + X - 2;
  // direction: top three bits of the draw (= mulhi(w_dir, 8)); dx = bit 0, dy = bit 1, dz = bit 2.
  // row_j - row_i = (dy - 1 + bi) + 8 (dz - 1 + bi): byte (dy + 2 dz) of 0x09080100, less 9 if bi == 0
  const uint32_t t1 = w_dir >> 30;
  const uint32_t dx = mad_u32(t1, 0xFFFFFFFEu, w_dir >> 29);   // dir - 2 (dir >> 1), on the FMA pipe
  const uint32_t rdp = prmt(0x09080100u, 0u, t1);
  uint32_t* p_j = p_i - 9 * (1 - bi) * NT + rdp * NT;
  // rows around i and j
  const uint32_t own_i = p_i[0];
  const uint32_t yMi = bi ? p_i[-NT] : ra, zMi = bi ? p_i[-8 * NT] : rb;
  const uint32_t yPi = bi ? ra : p_i[NT], zPi = bi ? rb : p_i[8 * NT];
  const uint32_t dgi = bi ? p_i[9 * NT] : p_i[-9 * NT];
  const uint32_t own_j = p_j[0], yMj = p_j[-NT], yPj = p_j[NT], zMj = p_j[-8 * NT], zPj = p_j[8 * NT];
  const uint32_t dgj = bi ? p_j[-9 * NT] : p_j[9 * NT];
  ra = bi ? yMi : yPi;
  rb = bi ? zMi : zPi;
  const uint32_t mul = mad_u32(dx, 15u, G.kc[kKcOne]);     // 16^dx: masks that move by one nibble with dx
  // shell 0: i's rows are own, y-+1, z-+1, diagonal on the side of the other sublattice; j's mirror them
  const uint32_t Wi = lop3<kLutSel>(prmt(own_i, bi ? yPi : yMi, K::swa_i), prmt(bi ? zPi : zMi, dgi, K::swb_i), K::mi);
  const uint32_t Wj = lop3<kLutSel>(prmt(own_j, bi ? yMj : yPj, K::swa_j), prmt(bi ? zMj : zPj, dgj, K::swb_j),
                                    K::mj0 * mul);
  const uint32_t U1 = lop3<kLutSelNotB>(Wi, Wj, K::Cj);     // i's fields as they are, j's complemented
  // shell 1
  const uint32_t n3i = prmt(prmt(yMi, yPi, K::s2i), prmt(zMi, zPi, K::s2i), 0x7610u);
  const uint32_t W2i = lop3<kLutSel>(own_i, n3i, K::moi);
  const uint32_t s2j = (K::s2j0 == K::s2j1) ? K::s2j0 : mad_u32(dx, G.kc[kKc1111], K::s2j0);
  const uint32_t n3j = prmt(prmt(yMj, yPj, s2j), prmt(zMj, zPj, s2j), 0x7610u);
  const uint32_t W2j = lop3<kLutSel>(own_j, n3j, K::moj0 * mul);
  const uint32_t MjD = (K::Mj1 == (K::Mj0 << 4)) ? K::Mj0 * mul : mad_u32(dx, G.kc[kKcMjDelta + slot], K::Mj0);
  const uint32_t U2 = lop3<kLutAndOr>(lop3<kLutSelNotB>(W2i, W2j, K::Ci), MjD, K::Mi);
  // population counts: all field bits, high bits, "both bits" (AND for i, OR of complements for j)
  const uint32_t h1 = U1 & K::kHi, h2 = U2 & K::kHi;
  const uint32_t b1 = lop3<kLutMaj>(U1 << 1, h1, K::Ci & K::kHi);
  const uint32_t b2 = lop3<kLutMaj>(U2 << 1, h2, K::Cj & K::kHi);
  const int pt1 = popc32(U1), ph1 = popc32(h1), pb1 = popc32(b1);
  const int pt2 = popc32(U2), ph2 = popc32(h2), pb2 = popc32(b2);
  // species of i and j (times 16) and the coefficient row of the ordered pair: [(a*4+b)*8 + slot] int4
  const uint32_t a4 = (own_i >> K::shi) & 0x30u;
  const uint32_t b4 = (own_j >> mad_u32(dx, 4u, G.kc[kKcShj0 + slot])) & 0x30u;
  const smem_ptr_t crow = smem_index(smem_index(env.coef, a4, 32u), b4, 8u);
  int dE4;                                                   // 4 dE
  if (PK) {
    // 16-bit coefficient pairs: one LDS.128, three byte packs and three IDP.2A
    const int4 c = lds_int4(crow, 0);
    dE4 = dp2a_lo((uint32_t)c.x, mad_u32((uint32_t)ph1, 256u, (uint32_t)pt1), c.w);
    dE4 = dp2a_lo((uint32_t)c.y, mad_u32((uint32_t)pt2, 256u, (uint32_t)pb1), dE4);
    dE4 = dp2a_lo((uint32_t)c.z, mad_u32((uint32_t)pb2, 256u, (uint32_t)ph2), dE4);
  } else {
    const int4 c0 = lds_int4(crow, 0), c1 = lds_int4(crow, 2048);
    dE4 = c1.z + c0.x * pt1 + c0.y * ph1 + c0.z * pb1 + c0.w * pt2 + c1.x * ph2 + c1.y * pb2;
  }
  // Eq. 3 in integer form
  bool ok;
  if (MODE == kAcceptDirect) {
    // the whole table sits in shared memory, followed by one zero entry at byte offset tmax4: dE <= 0
    // (huge as unsigned), dE >= len and a trial between equal species (dE = kSameSpecies by
    // construction) all clamp to that entry and are decided by the sign test alone
    const uint32_t i4 = min((uint32_t)dE4, env.tmax4);
    const uint32_t thr = lds_u32(env.filt, i4);
#if defined(__CUDA_ARCH__)
    // decision without a branch or a 0/1 value: reject = dE > 0 and u >= T.  A rejected trial XORs
    // zeros (ptxas would wrap a predicated shared-memory atomic in a branch of its own).
    uint32_t xm;
    asm("{\n\t"
        ".reg .pred q, r;\n\t"
        "setp.gt.s32 q, %3, 0;\n\t"
        "setp.ge.and.u32 r, %4, %5, q;\n\t"
        "selp.b32 %2, 0, %6, r;\n\t"
        "@!r add.s32 %0, %0, %3;\n\t"
        "@!r add.u32 %1, %1, 1;\n\t"
        "}"
        : "+r"(esum4), "+r"(nacc), "=r"(xm)
        : "r"(dE4), "r"(u), "r"(thr), "r"(a4 ^ b4));
    atomicXor(p_i, xm << K::shi);
    atomicXor(p_j, xm * ((1u << K::shj0) * mul));
    return;
#else
    ok = (dE4 <= 0) | (u < thr);
#endif
  } else if (MODE == kAcceptFilter) {
    // two-level threshold: ta <= T[dE] <= ta + E; dE <= 0 maps to entry 0, a trial between equal
    // species (dE = kSameSpecies by construction) to the zero entries at the top of Tq
    const uint32_t dc4 = (uint32_t)max(dE4, 0);
    const uint32_t ta = mulhi_u32(lds_u32(env.filt, 4 * kFilterTr + ((dc4 >> 6) & 0xFFCu)), lds_u32(env.filt, dc4 & 0xFCu));
    ok = u < ta;
    if (u - ta <= (uint32_t)env.filter_E) {                // u in [ta, ta+E]: rare exact decision
      const int dE = dE4 >> 2;
      ok = dE <= 0 || (dE < env.accept_len && u < ldg_u32(env.accept + dE));
    }
  } else {
    const int dE = dE4 >> 2;
    ok = dE <= 0;
    if (dE > 0 && dE < env.accept_len) ok = u < ldg_u32(env.accept + dE);
    ok = ok && a4 != b4;
  }
  if (MODE == kAcceptDirect) {
    // host build of the XOR swap (the device build returned above): both fields change by a ^ b
    if (ok) {
      const uint32_t x4 = a4 ^ b4;
      p_i[0] ^= x4 << K::shi;
      p_j[0] ^= x4 * ((1u << K::shj0) * mul);
      esum4 += dE4;
      nacc += 1u;
    }
    return;
  }
  // swap by arithmetic: the field of i holds a and becomes b, that of j holds b and becomes a; a
  // rejected trial stores the rows back unchanged (no branch)
  const uint32_t oki = ok ? 1u : 0u;
  const uint32_t od = mad_u32(oki, b4 - a4, 0u);
#if defined(__CUDA_ARCH__)
  atomicAdd(p_i, od * (1u << K::shi));                       // shared-memory adds: i and j may share a row
  atomicAdd(p_j, od * ((0u - (1u << K::shj0)) * mul));
#else
  const uint32_t new_i = mad_u32(od, 1u << K::shi, own_i);
  const uint32_t new_j = mad_u32(od, (0u - (1u << K::shj0)) * mul, rdp == 9u * (1 - bi) ? new_i : own_j);
  p_i[0] = new_i;
  p_j[0] = new_j;
#endif
  esum4 = (int)mad_u32(oki, (uint32_t)dE4, (uint32_t)esum4);
  nacc += oki;
}

#ifdef __CUDACC__
// Write-back of one tile word whose first nibble sits at nibble C of the aligned word pair (hi:lo).
// Bytes [P0, P1) of the pair lie wholly inside the tile word; they are cut into naturally aligned
// 4 / 2 / 1-byte stores at compile time.
template <int C, int P>
__device__ __forceinline__ void store_tile_bytes(unsigned char* lo, unsigned char* hi, uint32_t wv) {
  constexpr int P1 = (4 * C + 32) / 8;
  if constexpr (P < P1) {
    constexpr int off = P & 3;
    constexpr int room = (P1 - P) < (4 - off) ? (P1 - P) : (4 - off);
    constexpr int size = (off == 0 && room >= 4) ? 4 : ((off % 2 == 0 && room >= 2) ? 2 : 1);
    unsigned char* dst = (P < 4 ? lo : hi) + off;
    const uint32_t val = wv >> (8 * P - 4 * C);
    if constexpr (size == 4) *reinterpret_cast<uint32_t*>(dst) = val;
    else if constexpr (size == 2) *reinterpret_cast<uint16_t*>(dst) = (uint16_t)val;
    else *dst = (unsigned char)val;
    store_tile_bytes<C, P + size>(lo, hi, wv);
  }
}

template <int C, int NT>
__device__ __forceinline__ void write_back_tile(const Geom& G, const uint32_t* tile, uint32_t* lattice, int wlo,
                                                uint32_t dwh, int t0y, int t0z, int rw, uint32_t zstride) {
  uint32_t offy[6];
#pragma unroll
  for (int ry = 1; ry < 7; ++ry) {
    int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
    offy[ry - 1] = (uint32_t)gy * (uint32_t)rw + (uint32_t)wlo;
  }
  uint32_t* const peer = reinterpret_cast<uint32_t*>(G.peer_lat);
#pragma unroll 1
  for (int rz = 1; rz < 7; ++rz) {
    int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
    const uint32_t zoff = (uint32_t)gz * zstride;
#pragma unroll
    for (int ry = 1; ry < 7; ++ry) {
      const uint32_t idx = zoff + offy[ry - 1];
      store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(lattice + idx),
                                           reinterpret_cast<unsigned char*>(lattice + (uint32_t)(idx + dwh)),
                                           tile[(rz * 8 + ry) * NT]);
    }
    // fused ghost-layer message: the layers the neighbour slab holds a copy of go straight into its storage
    if (peer != nullptr && gz >= G.peer_z0 && gz < G.peer_z1) {
#pragma unroll
      for (int ry = 1; ry < 7; ++ry) {
        const uint32_t idx = zoff + offy[ry - 1];
        store_tile_bytes<C, (4 * C + 7) / 8>(reinterpret_cast<unsigned char*>(peer + idx),
                                             reinterpret_cast<unsigned char*>(peer + (uint32_t)(idx + dwh)),
                                             tile[(rz * 8 + ry) * NT]);
      }
    }
  }
}
#endif

#ifdef __CUDACC__
template <int kFilter>
__global__ void __launch_bounds__(kThreadNT, kThreadBlocksPerSM)
sweep_thread_per_cell(const Geom G, uint32_t* __restrict__ lattice, const int4* __restrict__ coef,
                      const uint32_t* __restrict__ accept, const uint32_t* __restrict__ filt,
                      DevState* __restrict__ st, int colour) {
  constexpr int NT = kThreadNT;
  extern __shared__ __align__(16) uint32_t smem_w[];
  uint32_t* tile = smem_w + threadIdx.x;                        // row r at tile[r * NT]
  int4* s_coef0 = reinterpret_cast<int4*>(smem_w + kThreadTileWords * NT);   // [16][8 slots]
  int4* s_coef1 = s_coef0 + 16 * 8;
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(s_coef1 + 16 * 8);
  __shared__ long long s_dE[NT / 32];
  __shared__ unsigned s_acc[NT / 32];
  // coefficient rows replicated over the 8 lane slots of a quarter warp: conflict-free LDS.128
  for (int k = threadIdx.x; k < 128; k += NT) {
    const int ent = k >> 3;
    s_coef0[k] = coef[ent * 2];
    s_coef1[k] = coef[ent * 2 + 1];
  }
  if (kFilter)
    for (int k = threadIdx.x; k < kFilterWords; k += NT) s_filt[k] = filt[k];

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
    const int t0z = tile_z0(G, oz, cz);
    const int rw = G.Lx >> 3;                                   // words per lattice row
    const int wlo = x0 >> 3, sh = 4 * (x0 & 7);
    const int whi = wlo + 1 == rw ? 0 : wlo + 1;
    // a3: stage the tile (funnel-shift two aligned words per row into one tile word).  Row (gz, gy)
    // starts at word (gz Ly + gy) rw of the lattice (a 32-bit index: thread_kernel_supported).
    const uint32_t zstride = (uint32_t)G.Ly * (uint32_t)rw;
    const uint32_t dwh = (uint32_t)(whi - wlo);                 // index step from the low to the high word of a row
    {
      uint32_t offy[8];
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        offy[ry] = (uint32_t)gy * (uint32_t)rw + (uint32_t)wlo;
      }
#pragma unroll 2
      for (int rz = 0; rz < 8; ++rz) {
        int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
        const uint32_t zoff = (uint32_t)gz * zstride;
        uint32_t lo[8], hi[8];
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          const uint32_t idx = zoff + offy[ry];
          lo[ry] = lattice[idx];
          hi[ry] = lattice[idx + dwh];
        }
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) tile[(rz * 8 + ry) * NT] = __funnelshift_r(lo[ry], hi[ry], sh);
      }
    }
    // a4-a6: the 128 trials of this cell, raster order, one Philox call per two slots
    const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    TrialEnv env;
    env.coef = smem_ptr(s_coef0) + (threadIdx.x & 7) * 16;
    env.filt = smem_ptr(s_filt);
    env.accept = accept;
    env.accept_len = G.accept_len;
    env.filter_E = G.filter_E;
#pragma unroll 1
    for (int lzy = 0; lzy < 16; ++lzy) {
      uint32_t* p_row = tile + (((lzy >> 2) + 2) * 8 + (lzy & 3) + 2) * NT;
      const uint32_t q0 = (uint32_t)lzy * 4u;
      uint32_t ra = p_row[-NT], rb = p_row[-8 * NT];
#define SMCX_TRIAL_PAIR(LX)                                                                                          \
      {                                                                                                              \
        const Philox4 r = philox4x32_10_rk(cell_id, q0 + LX, t, ctr3, G.rk0, G.rk1);                                \
        trial_thread<0, LX + 2, kFilter, NT>(G, p_row, env, r.x, r.y, ra, rb, esum, nacc);                                                \
        trial_thread<1, LX + 2, kFilter, NT>(G, p_row, env, r.z, r.w, ra, rb, esum, nacc);                                                \
      }
      SMCX_TRIAL_PAIR(0) SMCX_TRIAL_PAIR(1) SMCX_TRIAL_PAIR(2) SMCX_TRIAL_PAIR(3)
#undef SMCX_TRIAL_PAIR
    }
    // a7: write back tile rows 1..6 x 1..6: the bytes that lie wholly inside this tile (no other
    // cell of the pass touches them) and can hold a modified site.  The byte pattern depends on
    // x0 mod 8 only, which is the same for every cell of a pass: one uniform switch.
    {
      switch (x0 & 7) {
        case 0: write_back_tile<0, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 1: write_back_tile<1, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 2: write_back_tile<2, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 3: write_back_tile<3, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 4: write_back_tile<4, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 5: write_back_tile<5, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 6: write_back_tile<6, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        default: write_back_tile<7, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
      }
    }
  }
  // a8: block reduction, one atomic pair per block (the trials accumulated kDEScale dE: exact in int32 per
  // cell by build_thread_coefficients' bound, summed over cells in 64 bits)
  long long esum64 = esum / kDEScale;
  for (int o = 16; o > 0; o >>= 1) {
    esum64 += __shfl_down_sync(0xffffffffu, esum64, o);
    nacc += __shfl_down_sync(0xffffffffu, nacc, o);
  }
  if ((threadIdx.x & 31) == 0) { s_dE[threadIdx.x >> 5] = esum64; s_acc[threadIdx.x >> 5] = nacc; }
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


// ---- Philox4x32-10 of a trial pair with the counter structure (cell_id, q, t, tag) factored -------------
// Rounds 1-3 contain six 32 x 32 -> 64 products; with ctr = (cell, q, sweep, tag) five of them do not depend
// on (cell, q) jointly: M1*t is uniform, M0*cell, B = M1*c2' and C = M0*c0'' depend on the cell only (once per
// cell), A_q = M0*(hi(M1*t) ^ q ^ k0) on q only (once per block, table in shared memory).  Per call that leaves
// one product and three XORs for rounds 1-3 instead of six and six.  Same function, same bits.
struct PhiloxCell { uint32_t l0, lB, hCk, lC; };   // per-cell constants (hCk = hi(C) ^ rk1[2])

__device__ __forceinline__ void mulwide(uint32_t a, uint32_t b, uint32_t& hi, uint32_t& lo) {
  const uint64_t p = (uint64_t)a * b;
  hi = (uint32_t)(p >> 32); lo = (uint32_t)p;
}
// Table entry q: (hi(A_q) ^ rk1[1], lo(A_q)); filled once per block for q < 64.
__device__ __forceinline__ uint2 philox_slot_entry(uint32_t q, uint32_t t, const uint32_t* rk0, const uint32_t* rk1) {
  uint32_t h1, l1, hA, lA;
  mulwide(0xCD9E8D57u, t, h1, l1);
  mulwide(0xD2511F53u, h1 ^ q ^ rk0[0], hA, lA);
  return make_uint2(hA ^ rk1[1], lA);
}
__device__ __forceinline__ PhiloxCell philox_cell_setup(uint32_t cell_id, uint32_t t, uint32_t ctr3, const uint32_t* rk0,
                                                        const uint32_t* rk1) {
  uint32_t h0, l0, h1, l1, hB, lB, hC, lC;
  mulwide(0xD2511F53u, cell_id, h0, l0);
  mulwide(0xCD9E8D57u, t, h1, l1);
  mulwide(0xCD9E8D57u, h0 ^ ctr3 ^ rk1[0], hB, lB);
  mulwide(0xD2511F53u, hB ^ l1 ^ rk0[1], hC, lC);
  return PhiloxCell{l0, lB, hC ^ rk1[2], lC};
}
__device__ __forceinline__ Philox4 philox_factored(const PhiloxCell& pc, uint2 slot, const uint32_t* rk0, const uint32_t* rk1) {
  uint32_t hD, lD;
  mulwide(0xCD9E8D57u, slot.x ^ pc.l0, hD, lD);                 // round 3: M1 * c2'' , c2'' = hi(A_q) ^ l0 ^ rk1[1]
  uint32_t c0 = hD ^ pc.lB ^ rk0[2], c1 = lD, c2 = pc.hCk ^ slot.y, c3 = pc.lC;
#pragma unroll
  for (int r = 3; r < 10; ++r) philox_round(c0, c1, c2, c3, rk0[r], rk1[r]);
  return Philox4{c0, c1, c2, c3};
}

// ---- persistent variant ---------------------------------------------------------------------------
// One block of kPersistWarps warps per SM for the whole colour pass.  Every warp owns an 8 KB tile
// area (32 cells, row r of lane l at word r * 32 + l) and walks over batches of 32 consecutive cells
// of the colour on its own: no block barrier after the table load, so the warps of an SM drift apart
// and the staging / write-back of one overlaps the trial arithmetic of the others.  The shared memory
// left over holds the whole threshold table T (kAcceptDirect), which turns the acceptance test into
// one clamp, one load and two compares.
constexpr int kPersistMaxWarps = 20;   // a multiple of the four sub-partitions: 18 or 21 warps load them unevenly (measured)
constexpr int kPersistMinWarps = 16;
constexpr int kPersistTileBytes = kThreadTileWords * 32 * 4;             // per warp
constexpr int kPersistSmemMax = 232448 - 1024;                          // 227 KB less the static part / reserve

// warps per block for a table of len entries, or 0 if the table does not fit next to 16 warps
inline int persist_warps_for(int accept_len) {
  for (int w = kPersistMaxWarps; w >= kPersistMinWarps; --w)
    if ((size_t)w * kPersistTileBytes + 2 * 16 * 8 * sizeof(int4) + ((size_t)accept_len + 1) * 4 <= (size_t)kPersistSmemMax)
      return w;
  return 0;
}
inline size_t persist_smem(int warps, int accept_len) {
  return (size_t)warps * kPersistTileBytes + 2 * 16 * 8 * sizeof(int4) + (((size_t)accept_len + 1) * 4 + 15) / 16 * 16;
}

template <bool PK>
__global__ void __launch_bounds__(kPersistMaxWarps * 32, 1)
sweep_thread_persistent(const Geom G, uint32_t* __restrict__ lattice, const int4* __restrict__ coef,
                        const uint32_t* __restrict__ accept, DevState* __restrict__ st, int colour) {
  constexpr int NT = 32;                                        // row stride of a warp's tile area (words)
  extern __shared__ __align__(16) uint32_t smem_w[];
  const int n_warps = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint32_t* tile = smem_w + warp * (kThreadTileWords * NT) + lane;
  int4* s_coef0 = reinterpret_cast<int4*>(smem_w + n_warps * (kThreadTileWords * NT));   // [16][8 slots]
  int4* s_coef1 = s_coef0 + 16 * 8;
  uint32_t* s_T = reinterpret_cast<uint32_t*>(s_coef1 + 16 * 8);
  __shared__ unsigned s_acc[kPersistMaxWarps];
  __shared__ uint2 s_slot[64];                                  // Philox round-2 products that depend on the slot pair only
  // PK: coef points at the packed rows [16] int4; else at the 32-bit rows [16][2] int4
  for (int k = threadIdx.x; k < 128; k += blockDim.x) {
    const int ent = k >> 3;
    if (PK) {
      s_coef0[k] = coef[ent];
    } else {
      s_coef0[k] = coef[ent * 2];
      s_coef1[k] = coef[ent * 2 + 1];
    }
  }
  for (int k = threadIdx.x; k <= G.accept_len; k += blockDim.x) s_T[k] = k < G.accept_len ? accept[k] : 0u;

  const uint32_t t = (uint32_t)st->sweep;
  if (threadIdx.x < 64) s_slot[threadIdx.x] = philox_slot_entry(threadIdx.x, t, G.rk0, G.rk1);
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  int esum = 0;                                                 // kDEScale * sum of accepted dE of this thread
  unsigned nacc = 0;
  long long esum_total = 0;
  const int rw = G.Lx >> 3;                                     // words per lattice row
  const uint32_t zstride = (uint32_t)G.Ly * (uint32_t)rw;
  const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
  TrialEnv env;
  env.coef = smem_ptr(s_coef0) + (lane & 7) * 16;
  env.filt = smem_ptr(s_T);
  env.accept = accept;
  env.accept_len = G.accept_len;
  env.filter_E = 0;
  env.tmax4 = 4u * (uint32_t)G.accept_len;
  const uint32_t n_batches = (G.cells_per_colour + 31u) >> 5;
  __syncthreads();
  // warp-major numbering: the batches left over after the last full round go to the low warps of
  // every block, not to all warps of the low blocks
  for (uint32_t batch = (uint32_t)warp * gridDim.x + blockIdx.x; batch < n_batches; batch += (uint32_t)n_warps * gridDim.x) {
    const uint32_t m = batch * 32u + (uint32_t)lane;
    if (m < G.cells_per_colour) {
      int cx, cy, cz;
      colour_cell(G, m, colour, cx, cy, cz);
      const int x0 = (ox + cx * 4 - 2 + G.Lx) % G.Lx;
      const int t0y = (oy + cy * 4 - 2 + G.Ly) % G.Ly;
      const int t0z = tile_z0(G, oz, cz);
      const int wlo = x0 >> 3, sh = 4 * (x0 & 7);
      const int whi = wlo + 1 == rw ? 0 : wlo + 1;
      const uint32_t dwh = (uint32_t)(whi - wlo);
      {
        uint32_t offy[8];
#pragma unroll
        for (int ry = 0; ry < 8; ++ry) {
          int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
          offy[ry] = (uint32_t)gy * (uint32_t)rw + (uint32_t)wlo;
        }
#pragma unroll 2
        for (int rz = 0; rz < 8; ++rz) {
          int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
          const uint32_t zoff = (uint32_t)gz * zstride;
          uint32_t lo[8], hi[8];
#pragma unroll
          for (int ry = 0; ry < 8; ++ry) {
            const uint32_t idx = zoff + offy[ry];
            lo[ry] = lattice[idx];
            hi[ry] = lattice[idx + dwh];
          }
#pragma unroll
          for (int ry = 0; ry < 8; ++ry) tile[(rz * 8 + ry) * NT] = __funnelshift_r(lo[ry], hi[ry], sh);
        }
      }
      const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
      const PhiloxCell pc = philox_cell_setup(cell_id, t, ctr3, G.rk0, G.rk1);
#define SMCX_PHILOX_PAIR(LX) philox_factored(pc, s_slot[q0 + LX], G.rk0, G.rk1)
#pragma unroll 1
      for (int lzy = 0; lzy < 16; ++lzy) {
        uint32_t* p_row = tile + (((lzy >> 2) + 2) * 8 + (lzy & 3) + 2) * NT;
        const uint32_t q0 = (uint32_t)lzy * 4u;
        uint32_t ra = p_row[-NT], rb = p_row[-8 * NT];
#define SMCX_TRIAL_PAIR(LX)                                                                                          \
        {                                                                                                            \
          const Philox4 r = SMCX_PHILOX_PAIR(LX);                                                                    \
          trial_thread<0, LX + 2, kAcceptDirect, NT, PK>(G, p_row, env, r.x, r.y, ra, rb, esum, nacc);               \
          trial_thread<1, LX + 2, kAcceptDirect, NT, PK>(G, p_row, env, r.z, r.w, ra, rb, esum, nacc);               \
        }
        SMCX_TRIAL_PAIR(0) SMCX_TRIAL_PAIR(1) SMCX_TRIAL_PAIR(2) SMCX_TRIAL_PAIR(3)
#undef SMCX_TRIAL_PAIR
#undef SMCX_PHILOX_PAIR
      }
      switch (x0 & 7) {
        case 0: write_back_tile<0, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 1: write_back_tile<1, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 2: write_back_tile<2, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 3: write_back_tile<3, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 4: write_back_tile<4, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 5: write_back_tile<5, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        case 6: write_back_tile<6, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
        default: write_back_tile<7, NT>(G, tile, lattice, wlo, dwh, t0y, t0z, rw, zstride); break;
      }
      esum_total += esum / kDEScale;                            // per cell: 128 trials cannot overflow int32
      esum = 0;
    }
  }
  // a8: one atomic pair per block
  for (int o = 16; o > 0; o >>= 1) {
    esum_total += __shfl_down_sync(0xffffffffu, esum_total, o);
    nacc += __shfl_down_sync(0xffffffffu, nacc, o);
  }
  __shared__ long long s_e64[kPersistMaxWarps];
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

inline size_t thread_kernel_smem() {
  return (size_t)kThreadTileWords * kThreadNT * 4 + 2 * 16 * 8 * sizeof(int4) + kFilterWords * 4;
}

// d_coef: the 32-bit rows [16][8] int32 followed by the packed rows [16][4] int32
inline int launch_thread_persistent(const Geom& G, uint32_t* lattice, const int32_t* d_coef, bool packed, const uint32_t* accept,
                                    DevState* st, int colour, int warps, int sm_count, cudaStream_t stream) {
  const unsigned n_batches = (G.cells_per_colour + 31u) / 32u;
  const unsigned want = (n_batches + warps - 1) / warps;
  const unsigned grid = want < (unsigned)sm_count ? want : (unsigned)sm_count;
  if (packed)
    sweep_thread_persistent<true><<<grid, warps * 32, persist_smem(warps, G.accept_len), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef + 16 * kCoefInts), accept, st, colour);
  else
    sweep_thread_persistent<false><<<grid, warps * 32, persist_smem(warps, G.accept_len), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef), accept, st, colour);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

inline int configure_thread_per_cell() {
  if (cudaFuncSetAttribute(sweep_thread_persistent<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           kPersistSmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_thread_persistent<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           kPersistSmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_thread_per_cell<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)thread_kernel_smem()) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_thread_per_cell<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)thread_kernel_smem()) != cudaSuccess) return -1;
  return 0;
}

inline int launch_thread_per_cell(const Geom& G, uint32_t* lattice, const int32_t* d_coef, const uint32_t* accept,
                                  const uint32_t* d_filter, DevState* st, int colour, cudaStream_t stream) {
  const unsigned grid = (G.cells_per_colour + kThreadNT - 1) / kThreadNT;
  if (G.filter_E >= 0)
    sweep_thread_per_cell<true><<<grid, kThreadNT, thread_kernel_smem(), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef), accept, d_filter, st, colour);
  else
    sweep_thread_per_cell<false><<<grid, kThreadNT, thread_kernel_smem(), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef), accept, d_filter, st, colour);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}
#endif  // __CUDACC__

}  // namespace smcxk
