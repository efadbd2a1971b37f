// Lattice-wide kernels: seeded initial state (S6), pair-count reduction (a9: energy + Warren-
// Cowley counts), storage conversion and validation.
#pragma once
#include "smcx_common.cuh"

namespace smcxk {

// ---- species accessors for the device storage formats -------------------------------------
// load(): species of site i.  store16(): the 16 consecutive sites 16 g .. 16 g + 15 (vals[k] = species of site
// 16 g + k; sites >= n_sites are not written).
struct StoreU8 {
  static constexpr int kBits = 8;
  __device__ static __forceinline__ int load(const void* p, long long i) {
    return reinterpret_cast<const uint8_t*>(p)[i];
  }
  __device__ static __forceinline__ void store16(void* species, long long g, long long n_sites, const uint32_t* vals) {
    uint8_t* p = reinterpret_cast<uint8_t*>(species) + g * 16;
    if (g * 16 + 16 <= n_sites) {
      uint32_t w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
      for (int k = 0; k < 16; ++k) w[k >> 2] |= vals[k] << (8 * (k & 3));
      *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
    } else {
      for (int k = 0; k < 16 && g * 16 + k < n_sites; ++k) p[k] = (uint8_t)vals[k];
    }
  }
};
struct Store2 {
  static constexpr int kBits = 2;
  __device__ static __forceinline__ int load(const void* p, long long i) {
    return (int)((reinterpret_cast<const uint32_t*>(p)[i >> 4] >> (2 * (int)(i & 15))) & 3u);
  }
  __device__ static __forceinline__ void store16(void* species, long long g, long long, const uint32_t* vals) {
    uint32_t packed = 0;
#pragma unroll
    for (int k = 0; k < 16; ++k) packed |= vals[k] << (2 * k);
    reinterpret_cast<uint32_t*>(species)[g] = packed;
  }
};
// SMCX_STORAGE_4BIT: 4 bits per site, sublattice-planar in groups of 8 conventional cells along x (Lx is a multiple
// of 8): group G = c >> 3 of conventional cell c = (z Ly + y) Lx + x holds B words, word b = the sites of basis
// index b of its 8 cells, cell (c & 7) in nibble (c & 7).  A row of 8 cells of one sublattice is then one 32-bit
// word, which is what the packed FCC kernel (sweep_fcc.cuh) gathers neighbours from.
template <int B>
struct Store4 {
  static constexpr int kBits = 4;
  __device__ static __forceinline__ int load(const void* p, long long i) {
    const long long c = i / B;
    const int b = (int)(i - c * B);
    return (int)((reinterpret_cast<const uint32_t*>(p)[(c >> 3) * B + b] >> (4 * (int)(c & 7))) & 15u);
  }
  __device__ static __forceinline__ void store16(void* species, long long g, long long, const uint32_t* vals) {
    if (B == 2) {             // 16 sites = 8 conventional cells = one group of two words
      uint32_t w0 = 0, w1 = 0;
#pragma unroll
      for (int x = 0; x < 8; ++x) { w0 |= vals[2 * x] << (4 * x); w1 |= vals[2 * x + 1] << (4 * x); }
      reinterpret_cast<uint2*>(species)[g] = make_uint2(w0, w1);
    } else {                  // 16 sites = 4 conventional cells = half of each of the group's four words
      uint16_t* h = reinterpret_cast<uint16_t*>(species) + (g >> 1) * 8 + (g & 1);
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        uint32_t v = 0;
#pragma unroll
        for (int x = 0; x < 4; ++x) v |= vals[4 * x + b] << (4 * x);
        h[2 * b] = (uint16_t)v;
      }
    }
  }
};

// ---- S6: sigma_i = pi(i) mod n_species, pi = 4-round balanced Feistel over 2h bits ---------
__device__ __forceinline__ unsigned long long feistel_permute(unsigned long long v, int h,
                                                              unsigned long long n, uint32_t k0,
                                                              uint32_t k1) {
  const unsigned long long mask = (1ull << h) - 1ull;
  do {
    uint32_t left = (uint32_t)(v >> h), right = (uint32_t)(v & mask);
#pragma unroll
    for (uint32_t round = 0; round < 4; ++round) {
      const Philox4 r = philox4x32_10(right, round, 0u, TAG_INIT, k0, k1);
      const uint32_t nr = left ^ (r.x & (uint32_t)mask);
      left = right;
      right = nr;
    }
    v = ((unsigned long long)left << h) | right;
  } while (v >= n);
  return v;
}

// One thread per 16 consecutive sites (one packed word, or 16 bytes).
// A slab window holds the sites site_offset .. site_offset + n_sites - 1 (mod n_global) of the whole lattice, whose
// n_global sites the permutation acts on; a whole lattice has site_offset = 0, n_global = n_sites.
template <class Store>
__global__ void init_species_kernel(void* __restrict__ species, long long n_sites, int n_species, int h,
                                    uint32_t k0, uint32_t k1, long long site_offset, long long n_global) {
  const long long n_groups = (n_sites + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t vals[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const long long i = g * 16 + k;
      vals[k] = 0;
      if (i < n_sites) {
        long long ig = i + site_offset;
        if (ig >= n_global) ig -= n_global;
        vals[k] = (uint32_t)(feistel_permute((unsigned long long)ig, h, (unsigned long long)n_global, k0, k1) %
                             (unsigned long long)n_species);
      }
    }
    Store::store16(species, g, n_sites, vals);
  }
}

// S10: composition initial state.  cum[p] = n_0 + ... + n_p; site i holds the species whose range
// contains pi(i).  One thread per 16 consecutive sites, like init_species_kernel.
struct CompositionCum { long long cum[kMaxSpecies]; };

template <class Store>
__global__ void init_composition_kernel(void* __restrict__ species, long long n_sites, int n_species, int h,
                                        uint32_t k0, uint32_t k1, const CompositionCum C, long long site_offset,
                                        long long n_global) {
  const long long n_groups = (n_sites + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t vals[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const long long i = g * 16 + k;
      uint32_t s = 0;
      if (i < n_sites) {
        long long ig = i + site_offset;
        if (ig >= n_global) ig -= n_global;
        const long long r = (long long)feistel_permute((unsigned long long)ig, h, (unsigned long long)n_global, k0, k1);
        for (int p = 0; p < n_species - 1; ++p) s += r >= C.cum[p] ? 1u : 0u;
      }
      vals[k] = s;
    }
    Store::store16(species, g, n_sites, vals);
  }
}

// ---- storage conversion: uint8 site-id order <-> device storage ------------------------------
// One thread per 16 consecutive sites.  src / dst point at a chunk of n_sites_chunk sites that starts at site
// first_site (a multiple of 32) of the lattice; `lattice` is the whole array in device storage.  Validation is
// fused into the packing: any source value >= n_species raises st->bad_state (the caller reads it once, after the
// last chunk).
template <class Store>
__global__ void pack_kernel(const uint8_t* __restrict__ src, void* __restrict__ lattice, long long first_site,
                            long long n_sites_chunk, int n_species, DevState* __restrict__ st) {
  const long long n_groups = (n_sites_chunk + 15) >> 4;
  bool bad = false;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t vals[16];
    if (g * 16 + 16 <= n_sites_chunk) {
      const uint4 v = *reinterpret_cast<const uint4*>(src + g * 16);
      const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int k = 0; k < 16; ++k) vals[k] = (w[k >> 2] >> (8 * (k & 3))) & 0xffu;
    } else {
      for (int k = 0; k < 16; ++k) vals[k] = g * 16 + k < n_sites_chunk ? src[g * 16 + k] : 0u;
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      bad |= vals[k] >= (uint32_t)n_species;
      vals[k] &= (1u << Store::kBits) - 1u;
    }
    Store::store16(lattice, (first_site >> 4) + g, first_site + n_sites_chunk, vals);
  }
  if (bad) atomicOr(&st->bad_state, 1ull);
}

template <class Store>
__global__ void unpack_kernel(const void* __restrict__ lattice, uint8_t* __restrict__ dst, long long first_site,
                              long long n_sites_chunk) {
  const long long n_groups = (n_sites_chunk + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t vals[16];
    if (Store::kBits == 2) {
      const uint32_t packed = reinterpret_cast<const uint32_t*>(lattice)[(first_site >> 4) + g];
#pragma unroll
      for (int k = 0; k < 16; ++k) vals[k] = (packed >> (2 * k)) & 3u;
    } else {
#pragma unroll
      for (int k = 0; k < 16; ++k) vals[k] = (uint32_t)Store::load(lattice, first_site + g * 16 + k);
    }
    if (g * 16 + 16 <= n_sites_chunk) {
      uint32_t w[4] = {0u, 0u, 0u, 0u};
#pragma unroll
      for (int k = 0; k < 16; ++k) w[k >> 2] |= vals[k] << (8 * (k & 3));
      *reinterpret_cast<uint4*>(dst + g * 16) = make_uint4(w[0], w[1], w[2], w[3]);
    } else {
      for (int k = 0; k < 16; ++k)
        if (g * 16 + k < n_sites_chunk) dst[g * 16 + k] = (uint8_t)vals[k];
    }
  }
}

// Flags any field >= n_species in an array in device storage (smcx_set_species_packed).
template <class Store>
__global__ void validate_storage_kernel(const void* __restrict__ lattice, long long n_sites, int n_species, DevState* st) {
  bool bad = false;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n_sites; i += (long long)gridDim.x * blockDim.x)
    bad |= Store::load(lattice, i) >= n_species;
  if (bad) atomicOr(&st->bad_state, 1ull);
}

// Flags any byte >= n_species.
__global__ void validate_u8_kernel(const uint8_t* __restrict__ src, long long n, int n_species, DevState* st) {
  bool bad = false;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x)
    bad |= src[i] >= n_species;
  if (bad) atomicOr(&st->bad_state, 1ull);
}

// ---- a9: pair counts over the positive half of every shell ---------------------------------
// M[s][x][y] = #{(i, d): d in O_s^+, sigma_i = x, sigma_{i+d} = y}.  The ordered counts of Eq. 8
// follow on the host as N_s(p',p) = M_s(p',p) + M_s(p,p'), and H = sum_s sum_xy V_s(x,y) M_s(x,y).
// One thread per conventional cell; block-private histogram in shared memory, flushed with
// 64-bit atomics.
template <class Store, int B>
__global__ void __launch_bounds__(256)
pair_count_kernel(const Geom G, const void* __restrict__ species, unsigned long long* __restrict__ M) {
  extern __shared__ unsigned s_hist[];
  const int n2 = G.n_species * G.n_species;
  const int n_hist = G.n_shells * n2;
  for (int k = threadIdx.x; k < n_hist; k += blockDim.x) s_hist[k] = 0u;
  __syncthreads();
  // source sites: layers [pc_z0, pc_z1) (a slab counts the bonds of the layers it owns; their partners lie inside
  // its window, so the periodic wrap below never acts along z there)
  const long long c_first = (long long)G.Lx * G.Ly * G.pc_z0;
  const long long n_conv = (long long)G.Lx * G.Ly * G.pc_z1;
  const int Px = 2 * G.Lx, Py = 2 * G.Ly, Pz = 2 * G.Lz;
  for (long long c = c_first + blockIdx.x * (long long)blockDim.x + threadIdx.x; c < n_conv;
       c += (long long)gridDim.x * blockDim.x) {
    const int x = (int)(c % G.Lx);
    const long long r = c / G.Lx;
    const int y = (int)(r % G.Ly);
    const int z = (int)(r / G.Ly);
#pragma unroll
    for (int b = 0; b < B; ++b) {
      int bx, by, bz;
      if (B == 2) { bx = by = bz = b; }
      else { bx = (b >> 1) & 1; by = (b == 1 || b == 3) ? 1 : 0; bz = (b == 1 || b == 2) ? 1 : 0; }
      const int si = Store::load(species, c * B + b);
      for (int hh = 0; hh < G.ZH; ++hh) {
        const int m = G.half_idx[hh];
        int px = 2 * x + bx + G.off[m][0];
        int py = 2 * y + by + G.off[m][1];
        int pz = 2 * z + bz + G.off[m][2];
        if (px < 0) px += Px; else if (px >= Px) px -= Px;
        if (py < 0) py += Py; else if (py >= Py) py -= Py;
        if (pz < 0) pz += Pz; else if (pz >= Pz) pz -= Pz;
        int nb;
        if (B == 2) nb = px & 1;
        else {
          const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
          nb = par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3;
        }
        const long long nsite = (((long long)(pz >> 1) * G.Ly + (py >> 1)) * G.Lx + (px >> 1)) * B + nb;
        const int sn = Store::load(species, nsite);
        atomicAdd(&s_hist[(int)G.shell_of[m] * n2 + si * G.n_species + sn], 1u);
      }
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < n_hist; k += blockDim.x)
    if (s_hist[k]) atomicAdd(&M[k], (unsigned long long)s_hist[k]);
}

// ---- a9, bit-parallel: BCC, first two shells, packed 2-bit storage ----------------------------
// One thread per lattice word (a row of 8 conventional cells: nibble X = cell X, corner site in
// bits 0-1, body site in bits 2-3).  Every unordered bond is taken once, in an orientation chosen
// for the layout (the host only uses M + M^T and sum V M, V symmetric):
//   shell 0: corner site (X,y,z) with the body sites of cells (X-1..X, y-1..y, z-1..z);
//   shell 1: every site with the same-sublattice site of cells (X+1,y,z), (X,y+1,z), (X,y,z+1).
// Per species x an indicator word holds one bit per site of the word; the indicators of up to four
// neighbour alignments share a word (bits 0..3 of a nibble for shell 0, bits 0..1 of a field for
// shell 1), so one AND + POPC counts the pairs (x, y) of four (two) alignments at once:
// 64 POPC per 16 sites instead of 14 shared-memory atomics per cell.
__device__ __forceinline__ uint32_t lop3_ind(uint32_t lo, uint32_t hi, uint32_t mask, int x) {
  // bits where (lo, hi) spell species x, restricted to mask
  const uint32_t l = (x & 1) ? lo : ~lo, h = (x & 2) ? hi : ~hi;
  return l & h & mask;
}

__global__ void __launch_bounds__(256)
pair_count_bcc2_kernel(const Geom G, const uint32_t* __restrict__ lat, unsigned long long* __restrict__ M) {
  const int rw = G.Lx >> 3;                                    // words per lattice row
  const long long w_first = (long long)rw * G.Ly * G.pc_z0;    // layers [pc_z0, pc_z1), see pair_count_kernel
  const long long n_words = (long long)rw * G.Ly * G.pc_z1;
  uint32_t cnt0[16], cnt1[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) cnt0[k] = cnt1[k] = 0u;
  for (long long wi = w_first + blockIdx.x * (long long)blockDim.x + threadIdx.x; wi < n_words;
       wi += (long long)gridDim.x * blockDim.x) {
    const int xw = (int)(wi % rw);
    const long long r = wi / rw;
    const int y = (int)(r % G.Ly), z = (int)(r / G.Ly);
    const int xm = xw == 0 ? rw - 1 : xw - 1, xp = xw + 1 == rw ? 0 : xw + 1;
    const int ym = y == 0 ? G.Ly - 1 : y - 1, yp = y + 1 == G.Ly ? 0 : y + 1;
    const int zm = z == 0 ? G.Lz - 1 : z - 1, zp = z + 1 == G.Lz ? 0 : z + 1;
    auto row = [&](int zz, int yy) { return lat + ((long long)zz * G.Ly + yy) * rw; };
    const uint32_t* r00 = row(z, y);
    const uint32_t* rm0 = row(z, ym);
    const uint32_t* r0m = row(zm, y);
    const uint32_t* rmm = row(zm, ym);
    const uint32_t W = r00[xw];
    // ---- shell 0: corner fields of W against body fields of four rows, cells X and X - 1 ----
    {
      const uint32_t kN = 0x11111111u;
      uint32_t ia[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) ia[x] = lop3_ind(W, W >> 1, kN, x) * 0xFu;   // all four bits of the nibble
#pragma unroll
      for (int dx = 0; dx < 2; ++dx) {
        // body field of cell X (dx = 0: word >> 2) or X - 1 (dx = 1: (word << 2) | (previous word >> 30)) at bits 0-1
        uint32_t B[4];
        if (dx == 0) {
          B[0] = r00[xw] >> 2; B[1] = rm0[xw] >> 2; B[2] = r0m[xw] >> 2; B[3] = rmm[xw] >> 2;
        } else {
          B[0] = __funnelshift_l(r00[xm], r00[xw], 2); B[1] = __funnelshift_l(rm0[xm], rm0[xw], 2);
          B[2] = __funnelshift_l(r0m[xm], r0m[xw], 2); B[3] = __funnelshift_l(rmm[xm], rmm[xw], 2);
        }
        uint32_t ib[4] = {0u, 0u, 0u, 0u};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          // alignment k puts its indicator at bit k of the nibble: lo bit rotated to bit k, hi bit too
          const uint32_t lo = __funnelshift_l(B[k], B[k], k), hi = __funnelshift_l(B[k], B[k], (k + 31) & 31);
#pragma unroll
          for (int yv = 0; yv < 4; ++yv) ib[yv] |= lop3_ind(lo, hi, kN << k, yv);
        }
#pragma unroll
        for (int x = 0; x < 4; ++x)
#pragma unroll
          for (int yv = 0; yv < 4; ++yv) cnt0[x * 4 + yv] += (uint32_t)__popc(ia[x] & ib[yv]);
      }
    }
    // ---- shell 1: all 16 fields of W against the fields of cells X + 1, y + 1, z + 1 ----
    {
      const uint32_t kF = 0x55555555u;
      uint32_t ia[4];
#pragma unroll
      for (int x = 0; x < 4; ++x) ia[x] = lop3_ind(W, W >> 1, kF, x);
      const uint32_t Bx = __funnelshift_r(W, r00[xp], 4);       // cell X + 1 at nibble X
      const uint32_t By = row(z, yp)[xw], Bz = row(zp, y)[xw];
#pragma unroll
      for (int yv = 0; yv < 4; ++yv) {
        // alignments x + 1 and y + 1 share a word (bits 0 and 1 of a field), z + 1 has one of its own
        const uint32_t ib2 = lop3_ind(Bx, Bx >> 1, kF, yv) | (lop3_ind(By, By >> 1, kF, yv) << 1);
        const uint32_t ibz = lop3_ind(Bz, Bz >> 1, kF, yv);
#pragma unroll
        for (int x = 0; x < 4; ++x)
          cnt1[x * 4 + yv] += (uint32_t)__popc((ia[x] * 3u) & ib2) + (uint32_t)__popc(ia[x] & ibz);
      }
    }
  }
  // warp reduction, then one 64-bit atomic per (shell, x, y) and warp
  const int n = G.n_species, n2 = n * n;
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    uint32_t a = cnt0[k], b = cnt1[k];
    for (int o = 16; o > 0; o >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, o);
      b += __shfl_down_sync(0xffffffffu, b, o);
    }
    const int x = k >> 2, yv = k & 3;
    if ((threadIdx.x & 31) == 0 && x < n && yv < n) {
      if (a) atomicAdd(&M[x * n + yv], (unsigned long long)a);
      if (b) atomicAdd(&M[n2 + x * n + yv], (unsigned long long)b);
    }
  }
}

__global__ void zero_u64_kernel(unsigned long long* p, int n) {
  for (int k = threadIdx.x; k < n; k += blockDim.x) p[k] = 0ull;
}

}  // namespace smcxk
