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
//  * the integer pipe (LOP3/SHF) is the binding unit (ncu: profiles/), so the code is arranged to
//    keep its instruction count down: fused three-input logic with masks held in registers,
//    merges by multiply-add on the FMA pipe, coefficient tables replicated per lane slot so that
//    the 128-bit loads are conflict-free, and a two-level acceptance filter in shared memory.
#pragma once
#include "smcx_common.cuh"
#include "sweep_warp.cuh"

namespace smcxk {

#ifndef SMCX_NT
#define SMCX_NT 256
#endif
#ifndef SMCX_BLOCKS_PER_SM
#define SMCX_BLOCKS_PER_SM 3
#endif
#ifndef SMCX_OPT_RK
#define SMCX_OPT_RK 1   // Philox round keys from the constant bank
#endif
#ifndef SMCX_OPT_HI
#define SMCX_OPT_HI 0   // (measured slower: IMAD.HI issues at half the IMAD rate)  direction bits and U >> 1 via IMAD.HI (FMA pipe) instead of SHF (ALU pipe)
#endif
constexpr int kThreadNT = SMCX_NT;      // threads (= cells) per block
constexpr int kThreadTileWords = 64;    // 8 x 8 rows of one word
constexpr int kCoefInts = 8;            // per (a,b): cl0 ch0 cb0 cl1 | ch1 cb1 corr' pad
constexpr int kFilterTr = 64;           // Tr[r] = T[r], r < 64
constexpr int kFilterMaxTq = 1024;      // Tq[q] = T[64 q]; tables up to 65,536 entries (power of two: indices are masked)
constexpr int kFilterWords = kFilterTr + kFilterMaxTq;

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

// Host: two-level filter tables for a threshold table T.  Returns E >= 0 such that
// 0 <= T[d] - mulhi(Tq[d>>6], Tr[d&63]) <= E for all d < len, or -1 if no such small bound holds
// (then the kernel reads T[d] directly).  For T[d] = floor(2^32 exp(-d/kT)) the product of the
// two floors never exceeds T[d] and falls short by a few units at most.
inline int build_accept_filter(const uint32_t* T, int len, uint32_t* filt /*kFilterWords*/, int* nq_out) {
  const int nq = (len + 63) / 64;
  *nq_out = nq;
  if (nq > kFilterMaxTq) return -1;
  for (int r = 0; r < kFilterTr; ++r) filt[r] = r < len ? T[r] : 0u;
  for (int q = 0; q < kFilterMaxTq; ++q) filt[kFilterTr + q] = q < nq ? T[64 * q] : 0u;
  uint32_t E = 0;
  for (int d = 0; d < len; ++d) {
    const uint32_t ta = (uint32_t)(((uint64_t)filt[kFilterTr + (d >> 6)] * filt[d & 63]) >> 32);
    if (ta > T[d]) return -1;
    E = T[d] - ta > E ? T[d] - ta : E;
  }
  return E <= 1024u ? (int)E : -1;
}

inline void set_thread_masks(Geom& G) {
  // count words (see trial_thread): shell 0 = [n01_i n23_i | n01_j n23_j], one byte each;
  // shell 1 = [v_i | v_j | own-row fields of i at bits 16,24 and of j at bits 18,26]
  G.kH = 0xFFFF0000u; G.kM1 = 0x55555555u; G.kF1 = 0x55550000u;
  G.kH2 = 0x0C0CFF00u; G.kM2 = 0x05055555u; G.kF2 = 0x04045500u;
  for (int r = 0; r < 10; ++r) {
    G.rk0[r] = G.key0 + (uint32_t)r * 0x9E3779B9u;
    G.rk1[r] = G.key1 + (uint32_t)r * 0xBB67AE85u;
  }
  G.mul2 = 2u; G.mul4 = 4u; G.mul8 = 8u; G.mul_half = 0x80000000u;
}

__device__ __forceinline__ uint32_t lop3_maj(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

// Neighbour species of the site of sublattice b whose own 2-bit field sits at bit s0 of the row
// word at p (p1 = 1 << (s0 - 4)).  Fields are masked in place, merged by multiply-add (FMA pipe)
// and shifted down once:
//   n01, n23: shell 0, 4 fields each (the 2x2x2 block of the other sublattice, rows pairwise)
//   v:        shell 1, the fields at X of the four adjacent rows
//   t_own:    own row >> (s0 - 4): shell-1 fields of X-1 / X+1 at bits 0 / 8, own species at bit 4
template <int b>
__device__ __forceinline__ void gather_site(const uint32_t* p, int s0, uint32_t p1, uint32_t& n01, uint32_t& n23,
                                            uint32_t& v, uint32_t& own, uint32_t& t_own) {
  constexpr int NT = kThreadNT;
  own = p[0];
  const uint32_t yM = p[-NT], yP = p[NT], zM = p[-8 * NT], zP = p[8 * NT];
  const uint32_t dg = b ? p[9 * NT] : p[-9 * NT];
  const uint32_t A = b ? own : dg, Bq = b ? yP : zM, Cq = b ? zP : yM, Dq = b ? dg : own;
  const uint32_t mA = p1 * 204u;     // 0x33 << (s0 - 2)
  const uint32_t m0 = p1 * 48u;      // 0x3 << s0
  n01 = ((A & mA) + (Bq & mA) * 4u) >> (s0 - 2);
  n23 = ((Cq & mA) + (Dq & mA) * 4u) >> (s0 - 2);
  v = ((yM & m0) + (yP & m0) * 4u + (zM & m0) * 16u + (zP & m0) * 64u) >> s0;
  t_own = own >> (s0 - 4);
}

// U holds 2-bit fields; those selected by H belong to j, the others to i; M marks the low bit of
// every field, F = M & H.  Returns for lo bits, hi bits and lo&hi the merged population counts
// (count over i's fields) - (count over j's fields) + (number of j fields).
__device__ __forceinline__ void count3(uint32_t U, uint32_t half, uint32_t H, uint32_t M, uint32_t F, int& plo,
                                       int& phi, int& pbt) {
#if SMCX_OPT_HI
  const uint32_t Us = __umulhi(U, half);     // U >> 1 on the FMA pipe (half = 2^31)
#else
  const uint32_t Us = U >> 1; (void)half;
#endif
  const uint32_t tl = (U ^ H) & M;           // lo bits; complemented in j's fields
  const uint32_t th = (Us ^ H) & M;          // hi bits; complemented in j's fields
  const uint32_t tb = lop3_maj(tl, th, F);   // lo & hi for i, ~(lo & hi) for j
  plo = __popc(tl);
  phi = __popc(th);
  pbt = __popc(tb);
}

template <int bi, int X, bool kFilter>
__device__ __forceinline__ void trial_thread(const Geom& G, uint32_t* p_i, const char* coef_base,
                                             const uint32_t* s_filt, const uint32_t* __restrict__ accept,
                                             uint32_t w_dir, uint32_t u, int& esum, unsigned& nacc) {
  constexpr int NT = kThreadNT;
  constexpr int bj = 1 - bi;
  constexpr int s0_i = 4 * X + 2 * bi;
  // direction: top three bits of the draw (= mulhi(w_dir, 8)); dx = bit 0, dy = bit 1, dz = bit 2
#if SMCX_OPT_HI
  const int t1 = (int)__umulhi(w_dir, G.mul4);            // w_dir >> 30 = dy + 2 dz   (IMAD.HI: FMA pipe)
  const int dz = (int)__umulhi(w_dir, G.mul2);            // w_dir >> 31
  const int dir = (int)__umulhi(w_dir, G.mul8);           // w_dir >> 29
#else
  const int t1 = (int)(w_dir >> 30);                      // dy + 2 dz
  const int dz = (int)(w_dir >> 31);
  const int dir = (int)(w_dir >> 29);
#endif
  const int rd = t1 + 6 * dz - 9 * (1 - bi);              // row_j - row_i = (dy-1+bi) + 8 (dz-1+bi)
  const int s0_j = (4 * X + 4 * bi + 2 * bj - 4) + 4 * dir - 8 * t1;   // 4 (X-1+bi+dx) + 2 bj
  const uint32_t p1_j = 1u << (s0_j - 4);
  uint32_t* p_j = p_i + rd * NT;
  uint32_t n01i, n23i, vi, own_i, t_i, n01j, n23j, vj, own_j, t_j;
  gather_site<bi>(p_i, s0_i, 1u << (s0_i - 4), n01i, n23i, vi, own_i, t_i);
  gather_site<bj>(p_j, s0_j, p1_j, n01j, n23j, vj, own_j, t_j);
  const uint32_t a4 = t_i & 0x30u, b4 = t_j & 0x30u;      // species of i and j, times 16
  const int4 c0 = *reinterpret_cast<const int4*>(coef_base + a4 * 32u + b4 * 8u);            // [(a*4+b)*8 + slot]
  const int4 c1 = *reinterpret_cast<const int4*>(coef_base + 2048 + a4 * 32u + b4 * 8u);
  const uint32_t U1 = n01i + n23i * 256u + n01j * 65536u + n23j * 16777216u;
  const uint32_t U2 = vi + vj * 256u + (t_i & 0x303u) * 65536u + (t_j & 0x303u) * 262144u;
  int p1l, p1h, p1b, p2l, p2h, p2b;
  count3(U1, G.mul_half, G.kH, G.kM1, G.kF1, p1l, p1h, p1b);
  count3(U2, G.mul_half, G.kH2, G.kM2, G.kF2, p2l, p2h, p2b);
  const int dE = c1.z + c0.x * p1l + c0.y * p1h + c0.z * p1b + c0.w * p2l + c1.x * p2h + c1.y * p2b;
  // Eq. 3 in integer form.  in_tab: 0 < dE < len (one unsigned compare).
  const bool in_tab = (uint32_t)(dE - 1) < (uint32_t)(G.accept_len - 1);
  bool ok;
  if (kFilter) {
    // two-level threshold: ta <= T[dE] <= ta + E; tables are zero beyond the last entry and the
    // indices are masked, so every lane can evaluate it whatever its dE
    const uint32_t ta = __umulhi(s_filt[kFilterTr + (((uint32_t)dE >> 6) & (kFilterMaxTq - 1))], s_filt[dE & 63]);
    ok = dE <= 0 || (in_tab && u < ta);
    if (in_tab && u - ta <= (uint32_t)G.filter_E) ok = u < __ldg(accept + dE);   // u in [ta, ta+E]: rare exact look-up
  } else {
    ok = dE <= 0;
    if (in_tab) ok = u < __ldg(accept + dE);
  }
  // swap by arithmetic on the FMA pipe: the field of i holds a and becomes b, that of j holds b
  // and becomes a, so the row words change by +-(b - a) << position
  const int d4 = (int)b4 - (int)a4;
  if (ok && d4 != 0) {
    const uint32_t new_i = own_i + (uint32_t)d4 * (1u << (s0_i - 4));
    const uint32_t new_j = (rd == 0 ? new_i : own_j) - (uint32_t)d4 * p1_j;
    p_i[0] = new_i;
    p_j[0] = new_j;
    esum += dE;
    ++nacc;
  }
}

template <bool kFilter>
__global__ void __launch_bounds__(kThreadNT, SMCX_BLOCKS_PER_SM)
sweep_thread_per_cell(const Geom G, uint32_t* __restrict__ lattice, const int4* __restrict__ coef,
                      const uint32_t* __restrict__ accept, const uint32_t* __restrict__ filt,
                      DevState* __restrict__ st, int colour) {
  constexpr int NT = kThreadNT;
  extern __shared__ __align__(16) uint32_t smem_w[];
  uint32_t* tile = smem_w + threadIdx.x;                        // row r at tile[r * NT]
  int4* s_coef0 = reinterpret_cast<int4*>(smem_w + kThreadTileWords * NT);   // [16][8 slots]
  int4* s_coef1 = s_coef0 + 16 * 8;
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(s_coef1 + 16 * 8);
  __shared__ int s_dE[NT / 32];
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
    const int t0z = (oz + cz * 4 - 2 + G.Lz) % G.Lz;
    const int rw = G.Lx >> 3;                                   // words per lattice row
    const int wlo = x0 >> 3, sh = 4 * (x0 & 7);
    const int whi = wlo + 1 == rw ? 0 : wlo + 1;
    // a3: stage the tile (funnel-shift two aligned words per row into one tile word)
    const uint32_t* lat_lo = lattice + wlo;
    const uint32_t* lat_hi = lattice + whi;
#pragma unroll 2
    for (int rz = 0; rz < 8; ++rz) {
      int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
      uint32_t lo[8], hi[8];
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) {
        int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
        const size_t roff = (size_t)((uint32_t)(gz * G.Ly + gy)) * (uint32_t)rw;   // row index fits 32 bits
        lo[ry] = lat_lo[roff];
        hi[ry] = sh ? lat_hi[roff] : 0u;
      }
#pragma unroll
      for (int ry = 0; ry < 8; ++ry) tile[(rz * 8 + ry) * NT] = __funnelshift_r(lo[ry], hi[ry], sh);
    }
    // a4-a6: the 128 trials of this cell, raster order, one Philox call per two slots
    const uint32_t cell_id = (uint32_t)((cz * G.ncy + cy) * G.ncx + cx);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    const char* coef_base = reinterpret_cast<const char*>(s_coef0) + (threadIdx.x & 7) * 16;
#pragma unroll 1
    for (int lzy = 0; lzy < 16; ++lzy) {
      uint32_t* p_row = tile + (((lzy >> 2) + 2) * 8 + (lzy & 3) + 2) * NT;
      const uint32_t q0 = (uint32_t)lzy * 4u;
#define SMCX_TRIAL_PAIR(LX)                                                                                   \
      {                                                                                                       \
        const Philox4 r = SMCX_OPT_RK ? philox4x32_10_rk(cell_id, q0 + LX, t, ctr3, G.rk0, G.rk1)             \
                                      : philox4x32_10(cell_id, q0 + LX, t, ctr3, G.key0, G.key1);             \
        trial_thread<0, LX + 2, kFilter>(G, p_row, coef_base, s_filt, accept, r.x, r.y, esum, nacc);          \
        trial_thread<1, LX + 2, kFilter>(G, p_row, coef_base, s_filt, accept, r.z, r.w, esum, nacc);          \
      }
      SMCX_TRIAL_PAIR(0) SMCX_TRIAL_PAIR(1) SMCX_TRIAL_PAIR(2) SMCX_TRIAL_PAIR(3)
#undef SMCX_TRIAL_PAIR
    }
    // a7: write back tile rows 1..6 x 1..6; only the bytes that lie wholly inside this tile and can
    // hold a modified site (conventional cells 1..6 of the row: 4 bytes if x0 is even, else 3), cut
    // into at most three naturally aligned stores.  The cut depends on x0 mod 8 only, which is the
    // same for every cell of a pass, so the branches below are uniform.
    {
      const int rb = G.Lx >> 1;                                 // bytes per lattice row (multiple of 4)
      const bool odd = x0 & 1;
      int pos = (x0 + (odd ? 1 : 0)) >> 1;                      // first byte, before wrapping
      int rem = odd ? 3 : 4, done = 0, nseg = 0;
      int seg_sz[3] = {0, 0, 0}, seg_sh[3] = {0, 0, 0};
      unsigned char* seg_p[3] = {nullptr, nullptr, nullptr};
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        if (rem > 0) {
          const int sz = ((pos & 3) == 0 && rem >= 4) ? 4 : (((pos & 1) == 0 && rem >= 2) ? 2 : 1);
          seg_sz[k] = sz;
          seg_sh[k] = 8 * done + (odd ? 4 : 0);
          seg_p[k] = reinterpret_cast<unsigned char*>(lattice) + (pos >= rb ? pos - rb : pos);
          pos += sz; rem -= sz; done += sz; nseg = k + 1;
        }
      }
      for (int rz = 1; rz < 7; ++rz) {
        int gz = t0z + rz; if (gz >= G.Lz) gz -= G.Lz;
#pragma unroll
        for (int ry = 1; ry < 7; ++ry) {
          int gy = t0y + ry; if (gy >= G.Ly) gy -= G.Ly;
          const size_t roff = (size_t)((uint32_t)(gz * G.Ly + gy)) * (uint32_t)rb;
          const uint32_t wv = tile[(rz * 8 + ry) * NT];
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            if (k < nseg) {
              const uint32_t val = wv >> seg_sh[k];
              if (seg_sz[k] == 4) *reinterpret_cast<uint32_t*>(seg_p[k] + roff) = val;
              else if (seg_sz[k] == 2) *reinterpret_cast<uint16_t*>(seg_p[k] + roff) = (uint16_t)val;
              else seg_p[k][roff] = (unsigned char)val;
            }
          }
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

inline size_t thread_kernel_smem() {
  return (size_t)kThreadTileWords * kThreadNT * 4 + 2 * 16 * 8 * sizeof(int4) + kFilterWords * 4;
}

inline int configure_thread_per_cell() {
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
  return 0;
}

}  // namespace smcxk
