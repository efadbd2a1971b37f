// Lattice-wide kernels: seeded initial state (S6), pair-count reduction (a9: energy + Warren-
// Cowley counts), storage conversion and validation.
#pragma once
#include "smcx_common.cuh"

namespace smcxk {

// ---- species accessors for the two device storage formats --------------------------------
struct StoreU8 {
  static constexpr int kBits = 8;
  __device__ static __forceinline__ int load(const void* p, long long i) {
    return reinterpret_cast<const uint8_t*>(p)[i];
  }
};
struct Store2 {
  static constexpr int kBits = 2;
  __device__ static __forceinline__ int load(const void* p, long long i) {
    return (int)((reinterpret_cast<const uint32_t*>(p)[i >> 4] >> (2 * (int)(i & 15))) & 3u);
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
template <class Store>
__global__ void init_species_kernel(void* __restrict__ species, long long n_sites, int n_species, int h,
                                    uint32_t k0, uint32_t k1) {
  const long long n_groups = (n_sites + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t packed = 0;
    uint32_t bytes[4] = {0, 0, 0, 0};
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const long long i = g * 16 + k;
      uint32_t s = 0;
      if (i < n_sites)
        s = (uint32_t)(feistel_permute((unsigned long long)i, h, (unsigned long long)n_sites, k0, k1) %
                       (unsigned long long)n_species);
      packed |= s << (2 * k);
      bytes[k >> 2] |= s << (8 * (k & 3));
    }
    if (Store::kBits == 2) {
      reinterpret_cast<uint32_t*>(species)[g] = packed;
    } else {
      uint8_t* p = reinterpret_cast<uint8_t*>(species) + g * 16;
      if (g * 16 + 16 <= n_sites) {
        *reinterpret_cast<uint4*>(p) = make_uint4(bytes[0], bytes[1], bytes[2], bytes[3]);
      } else {
        for (int k = 0; k < 16 && g * 16 + k < n_sites; ++k) p[k] = (uint8_t)((bytes[k >> 2] >> (8 * (k & 3))) & 0xff);
      }
    }
  }
}

// ---- storage conversion: uint8 site-id order <-> packed 2-bit ------------------------------
__global__ void pack2_kernel(const uint8_t* __restrict__ src, uint32_t* __restrict__ dst, long long first_site,
                             long long n_sites_chunk) {
  // first_site is a multiple of 16; src points at the chunk, dst at the whole packed array.
  const long long n_groups = (n_sites_chunk + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    uint32_t packed = 0;
    for (int k = 0; k < 16; ++k) {
      const long long i = g * 16 + k;
      const uint32_t s = i < n_sites_chunk ? src[i] : 0u;
      packed |= (s & 3u) << (2 * k);
    }
    dst[(first_site >> 4) + g] = packed;
  }
}

__global__ void unpack2_kernel(const uint32_t* __restrict__ src, uint8_t* __restrict__ dst, long long first_site,
                               long long n_sites_chunk) {
  const long long n_groups = (n_sites_chunk + 15) >> 4;
  for (long long g = blockIdx.x * (long long)blockDim.x + threadIdx.x; g < n_groups;
       g += (long long)gridDim.x * blockDim.x) {
    const uint32_t packed = src[(first_site >> 4) + g];
    for (int k = 0; k < 16; ++k) {
      const long long i = g * 16 + k;
      if (i < n_sites_chunk) dst[i] = (uint8_t)((packed >> (2 * k)) & 3u);
    }
  }
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
  const long long n_conv = (long long)G.Lx * G.Ly * G.Lz;
  const int Px = 2 * G.Lx, Py = 2 * G.Ly, Pz = 2 * G.Lz;
  for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < n_conv;
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

__global__ void zero_u64_kernel(unsigned long long* p, int n) {
  for (int k = threadIdx.x; k < n; k += blockDim.x) p[k] = 0ull;
}

}  // namespace smcxk
