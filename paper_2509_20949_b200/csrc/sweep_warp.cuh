// Generic colour-pass kernel: one warp per link cell, uint8 species, any lattice / shell list.
//
// Steps a1-a8 of DESIGN.md: derive the link-cell origin of this sweep, stage the
// cell + LIZ+ halo tile into shared memory, run the S trials of the cell back to back (Philox
// draws are produced 32 calls = 64 trials at a time, one call per lane; the 2*ZT bond terms of a
// trial are spread over the lanes and summed with one warp reduction), write the modified region
// back, and add the accepted dE / accept count with one atomic pair per block.
#pragma once
#include "smcx_common.cuh"

namespace smcxk {

constexpr int kWarpsPerBlock = 8;

__device__ __forceinline__ void sweep_origin(const Geom& G, uint32_t t, int& ox, int& oy, int& oz) {
  const Philox4 r = philox4x32_10(0u, 0u, t, TAG_SHIFT, G.key0, G.key1);
  ox = (int)mulhi_u32(r.x, (uint32_t)G.w);
  oy = (int)mulhi_u32(r.y, (uint32_t)G.w);
  oz = (int)mulhi_u32(r.z, (uint32_t)G.w);
}

// Global id of link cell (cx, cy, cz) (cz counted inside the slab when the handle holds one): ctr[0] of S4.
__device__ __forceinline__ uint32_t global_cell_id(const Geom& G, int cx, int cy, int cz) {
  return (uint32_t)(((cz + G.cz_global) * G.ncy + cy) * G.ncx + cx);
}
// First layer (conventional cell) of the tile of a cell of row cz.
__device__ __forceinline__ int tile_z0(const Geom& G, int oz, int cz) { return (oz + cz * G.w + G.z_bias) % G.Lz; }

// m-th cell of a colour -> cell coordinates; cells of one colour are enumerated x fastest.
__device__ __forceinline__ void colour_cell(const Geom& G, uint32_t m, int colour, int& cx, int& cy,
                                            int& cz) {
  const uint32_t hx = (uint32_t)(G.ncx >> 1), hy = (uint32_t)(G.ncy >> 1);
  const uint32_t ix = m % hx;
  const uint32_t r = m / hx;
  const uint32_t iy = r % hy;
  const uint32_t iz = r / hy + (uint32_t)G.iz_first;
  cx = (int)(2u * ix) + (colour & 1);
  cy = (int)(2u * iy) + ((colour >> 1) & 1);
  cz = (int)(2u * iz) + ((colour >> 2) & 1);
}

template <int B>
__global__ void __launch_bounds__(kWarpsPerBlock * 32)
sweep_warp_per_cell(const Geom G, uint8_t* __restrict__ species, const int32_t* __restrict__ epi,
                    const uint32_t* __restrict__ accept, DevState* __restrict__ st, int colour) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n2 = G.n_species * G.n_species;
  const int n_epi = G.n_shells * n2;
  int32_t* s_epi = reinterpret_cast<int32_t*>(smem);
  short* s_delta = reinterpret_cast<short*>(s_epi + n_epi);            // [B][ZT]
  unsigned char* s_shell = reinterpret_cast<unsigned char*>(s_delta + B * G.ZT);
  const int tile_sites = G.TW * G.TW * G.TW * B;
  const int tables_bytes = (n_epi * 4 + B * G.ZT * 2 + G.ZT + 15) & ~15;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  unsigned char* tile = smem + tables_bytes + warp * ((tile_sites + 15) & ~15);
  __shared__ long long s_dE[kWarpsPerBlock];
  __shared__ unsigned s_acc[kWarpsPerBlock];

  for (int k = threadIdx.x; k < n_epi; k += blockDim.x) s_epi[k] = epi[k];
  for (int k = threadIdx.x; k < B * G.ZT; k += blockDim.x) s_delta[k] = G.delta[k / G.ZT][k % G.ZT];
  for (int k = threadIdx.x; k < G.ZT; k += blockDim.x) s_shell[k] = G.shell_of[k];

  const uint32_t t = (uint32_t)st->sweep;
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);

  const uint32_t m = blockIdx.x * kWarpsPerBlock + warp;
  const bool active = m < G.cells_per_colour;
  long long sum_dE = 0;
  unsigned n_acc = 0;
  int cx = 0, cy = 0, cz = 0, t0x = 0, t0y = 0, t0z = 0;
  const int TW = G.TW, H = G.H, w = G.w;
  if (active) {
    colour_cell(G, m, colour, cx, cy, cz);
    // a3: stage the tile; its first conventional cell is (o + c w - H) mod L per axis.
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
  __syncthreads();  // tables + tiles visible

  if (active) {
    const uint32_t cell_id = global_cell_id(G, cx, cy, cz);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    const int ZT = G.ZT;
    uint32_t r_dir_even = 0, r_u_even = 0, r_dir_odd = 0, r_u_odd = 0;
    int k = 0;
    for (int lz = 0; lz < w; ++lz)
      for (int ly = 0; ly < w; ++ly)
        for (int lx = 0; lx < w; ++lx) {
          const int conv = ((lz + H) * TW + (ly + H)) * TW + (lx + H);
#pragma unroll
          for (int b = 0; b < B; ++b, ++k) {
            if ((k & 63) == 0) {  // a4: 32 Philox calls cover the next 64 slots
              const Philox4 r = philox4x32_10(cell_id, (uint32_t)(k >> 1) + lane, t, ctr3, G.key0, G.key1);
              r_dir_even = r.x; r_u_even = r.y; r_dir_odd = r.z; r_u_odd = r.w;
            }
            const int src = (k >> 1) & 31;
            const uint32_t w_dir = __shfl_sync(0xffffffffu, (k & 1) ? r_dir_odd : r_dir_even, src);
            const uint32_t u = __shfl_sync(0xffffffffu, (k & 1) ? r_u_odd : r_u_even, src);
            const int si = conv * B + b;
            const int dir = (int)mulhi_u32(w_dir, (uint32_t)G.Z0);
            const int sj = si + s_delta[b * ZT + dir];
            const int sa = tile[si], sb = tile[sj];
            if (sa == sb) continue;  // same species: counts as a trial only
            // a5: dE = sum over bonds of i (a->b) and of j (b->a), the i-j bond left out.
            const int bj = sj & (B - 1);
            int part = 0;
            for (int n = lane; n < 2 * ZT; n += 32) {
              const bool jside = n >= ZT;
              const int mm = jside ? n - ZT : n;
              const int base = jside ? sj : si;
              const int bb = jside ? bj : b;
              const int ns = base + s_delta[bb * ZT + mm];
              const int x = tile[ns];
              const int row = (int)s_shell[mm] * n2 + x;
              int dv = s_epi[row + sb * G.n_species] - s_epi[row + sa * G.n_species];
              if (ns == (jside ? si : sj)) dv = 0;
              part += jside ? -dv : dv;
            }
            const int dE = __reduce_add_sync(0xffffffffu, part);
            // a6: Eq. 3 in integer form.
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
    // a7: write back the sites a swap can have touched: positions within r0 of the cell.
    const int lo = 2 * H - G.r0, hi = 2 * (H + w) - 1 + G.r0;  // tile half-unit positions, inclusive
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
        if (px >= lo && px <= hi && py >= lo && py <= hi && pz >= lo && pz <= hi)
          species[g + b] = tile[idx * B + b];
      }
    }
  }
  // a8: one atomic pair per block.
  if (lane == 0) { s_dE[warp] = sum_dE; s_acc[warp] = n_acc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < kWarpsPerBlock; ++i) { e += s_dE[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

// S3.3: trace[t] = E_run, t += 1.  One thread.
__global__ void sweep_epilogue(DevState* st, long long* trace, int trace_capacity) {
  const unsigned long long t = st->sweep;
  trace[t % (unsigned long long)trace_capacity] = st->e_run;
  st->sweep = t + 1ull;
  for (int c = 0; c < 16; ++c) st->work[c] = 0u;
}

}  // namespace smcxk
