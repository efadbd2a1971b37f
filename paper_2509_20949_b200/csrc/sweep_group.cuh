// Sub-warp colour-pass kernel: L lanes (4, 8, 16 or 32) per link cell, uint8 species, any lattice /
// shell list / link-cell size ("sub-warp variants of the same path").
//
// Same steps a1-a8 and the same schedule as sweep_warp_per_cell, arranged for fewer instructions per
// trial:
//  * the serial part of a trial (slot -> site, direction, species of i and j, acceptance) is replicated
//    over L lanes instead of 32, and 32 / L cells share a warp;
//  * a neighbour visit is three shared-memory loads and two adds: one packed table word gives the
//    tile-index delta and the row of the difference table, the tile gives the species x, and
//    D[(a,b)][s][x] = V_s(b,x) - V_s(a,x) (built in shared memory when the block starts) gives the bond
//    term.  The sums over the neighbours of i and of j both include the i-j bond;
//    corr(a,b) = 2 V_0(a,b) - V_0(a,a) - V_0(b,b) takes it out again (exact integer identity);
//  * lane g of a group takes neighbours g, g + L, ... of both sites; one xor-shuffle tree over the group
//    sums the partial dE;
//  * Philox: lane g of a group computes the call of slot pair q0 + g, so a group draws 2 L slots at a
//    time and hands the words round with group-wide shuffles;
//  * control flow is uniform over the warp (a trial between equal species is computed and masked, the
//    neighbour loop has the same trip count in every lane), so the 32 / L cells of a warp never
//    serialise, and the acceptance test reads the two-level filter tables in shared memory (see
//    sweep_thread.cuh; the exact table in global memory only when u falls within E of the bound): a
//    lattice with few cells per colour is bound by the latency of one cell's chain of trials.
// Results are bit-identical to the other kernels (tests/test_gpu_parity.py).
#pragma once
#include "smcx_common.cuh"
#include "sweep_thread.cuh"   // two-level acceptance filter (kFilterTr, kFilterWords, build_accept_filter)
#include "sweep_warp.cuh"

namespace smcxk {

constexpr int kGroupWarpsPerBlock = 8;
// Tile layout in shared memory (bytes): site (tz, ty, tx, b) of the tile at tz * zpitch + ty * TW * B +
// tx * B + b with zpitch = TW * TW * B + kGroupZPad.  Without the pad a step in z is a multiple of 32
// words and neighbours that differ in z share a bank.  The tiles of the cells of a warp are
// kGroupSkew bytes further apart than a multiple of 128 bytes, so that the same site of different
// cells lies in different banks (ncu, FCC 128^3 before either: 71 % of the shared-memory wavefronts
// were bank conflicts).
constexpr int kGroupZPad = 12;
constexpr int kGroupSkew = 4;
__host__ __device__ inline int group_zpitch(int TW, int B) { return TW * TW * B + kGroupZPad; }

struct GroupSmem {
  int d_stride;        // ints per ordered pair in the difference table (odd: spreads the pairs over the banks)
  int d_bytes, nb_bytes, filt_bytes, tile_bytes, total;
};

inline GroupSmem group_smem_layout(const Geom& G, int lanes) {
  GroupSmem L;
  const int n = G.n_species;
  int stride = G.n_shells * n + 1;            // the last entry of a row is corr(a,b)
  if ((stride & 1) == 0) ++stride;
  L.d_stride = stride;
  L.d_bytes = (n * n * stride * 4 + 15) & ~15;
  L.nb_bytes = (G.B * G.ZT * 4 + 15) & ~15;
  L.tile_bytes = ((G.TW * group_zpitch(G.TW, G.B) + 127) & ~127) + kGroupSkew;
  const int cells_per_block = kGroupWarpsPerBlock * (32 / lanes);
  L.filt_bytes = kFilterWords * 4;
  L.total = (L.d_bytes + L.nb_bytes + L.filt_bytes + cells_per_block * L.tile_bytes + 15) & ~15;
  return L;
}

template <int B, int L>
__global__ void __launch_bounds__(kGroupWarpsPerBlock * 32)
sweep_group_per_cell(const Geom G, uint8_t* __restrict__ species, const int32_t* __restrict__ epi,
                     const uint32_t* __restrict__ accept, const uint32_t* __restrict__ filt, DevState* __restrict__ st,
                     int colour, int d_stride, int d_bytes, int nb_bytes, int tile_bytes) {
  constexpr int CPW = 32 / L;                                   // cells per warp
  extern __shared__ __align__(16) unsigned char smem[];
  int32_t* s_D = reinterpret_cast<int32_t*>(smem);              // [a * n + b][d_stride]
  uint32_t* s_nb = reinterpret_cast<uint32_t*>(smem + d_bytes); // [basis][ZT]: (delta & 0xffff) | (shell * n) << 16
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int grp = lane / L, g = lane % L;
  uint32_t* s_filt = reinterpret_cast<uint32_t*>(smem + d_bytes + nb_bytes);   // Tr[64] then Tq[1024]
  unsigned char* tile = smem + d_bytes + nb_bytes + kFilterWords * 4 + (warp * CPW + grp) * tile_bytes;
  __shared__ long long s_dE[kGroupWarpsPerBlock];
  __shared__ unsigned s_acc[kGroupWarpsPerBlock];

  const int n = G.n_species, ZT = G.ZT;
  for (int k = threadIdx.x; k < n * n * d_stride; k += blockDim.x) {
    const int pair = k / d_stride, e = k % d_stride;
    const int a = pair / n, b = pair % n;
    int v = 0;
    if (e < G.n_shells * n) {
      const int s = e / n, x = e % n;
      v = epi[(s * n + b) * n + x] - epi[(s * n + a) * n + x];
    } else if (e == G.n_shells * n) {
      v = 2 * epi[a * n + b] - epi[a * n + a] - epi[b * n + b];
    }
    s_D[k] = v;
  }
  if (G.filter_E >= 0)
    for (int k = threadIdx.x; k < kFilterWords; k += blockDim.x) s_filt[k] = filt[k];
  const int ypitch = G.TW * B, zpitch = group_zpitch(G.TW, B);
  for (int k = threadIdx.x; k < B * ZT; k += blockDim.x) {
    const int b = k / ZT, m = k % ZT;
    // position of neighbour m of a site with basis b, relative to the site's conventional cell (units of
    // a/2): basis position + offset; its parity gives the basis of the neighbour (S0)
    int q[3], dc[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const int bp = B == 2 ? b : (a == 0 ? ((b >> 1) & 1) : a == 1 ? (b & 1) : (b == 1 || b == 2 ? 1 : 0));
      q[a] = bp + G.off[m][a];
      dc[a] = q[a] >= 0 ? q[a] >> 1 : -((1 - q[a]) >> 1);
    }
    const int par = (q[0] & 1) | ((q[1] & 1) << 1) | ((q[2] & 1) << 2);
    const int nb = B == 2 ? (q[0] & 1) : (par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3);
    const int delta = dc[2] * zpitch + dc[1] * ypitch + dc[0] * B + (nb - b);
    s_nb[k] = ((uint32_t)(uint16_t)(short)delta) | ((uint32_t)(G.shell_of[m] * n) << 16);
  }

  const uint32_t t = (uint32_t)st->sweep;
  int ox, oy, oz;
  sweep_origin(G, t, ox, oy, oz);
  const uint32_t m = (blockIdx.x * kGroupWarpsPerBlock + warp) * CPW + grp;
  const bool active = m < G.cells_per_colour;
  long long sum_dE = 0;
  unsigned n_acc = 0;
  int cx = 0, cy = 0, cz = 0, t0x = 0, t0y = 0, t0z = 0;
  const int TW = G.TW, H = G.H, w = G.w;
  const int n_conv = TW * TW * TW;
  if (active) {
    colour_cell(G, m, colour, cx, cy, cz);
    t0x = (ox + cx * w - H + G.Lx) % G.Lx;
    t0y = (oy + cy * w - H + G.Ly) % G.Ly;
    t0z = (oz + cz * w - H + G.Lz) % G.Lz;
    for (int idx = g; idx < n_conv; idx += L) {
      const int tx = idx % TW, ty = (idx / TW) % TW, tz = idx / (TW * TW);
      int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
      int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
      int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
      const long long gi = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
      unsigned char* dst = tile + tz * zpitch + ty * ypitch + tx * B;
      if (B == 2) *reinterpret_cast<uint16_t*>(dst) = *reinterpret_cast<const uint16_t*>(species + gi);
      else        *reinterpret_cast<uint32_t*>(dst) = *reinterpret_cast<const uint32_t*>(species + gi);
    }
  } else {
    // a group without a cell runs the trial loop on an all-zero tile: every trial is a same-species no-op
    for (int idx = g; idx < (TW * zpitch) / 4; idx += L) reinterpret_cast<uint32_t*>(tile)[idx] = 0u;
  }
  __syncthreads();  // tables + tiles visible

  {
    const uint32_t cell_id = (uint32_t)((cz * G.ncy + cy) * G.ncx + cx);
    const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
    const int corr_at = G.n_shells * n;
    const int nit = (ZT + L - 1) / L;
    const int filter_E = G.filter_E;
    uint32_t r_dir_even = 0, r_u_even = 0, r_dir_odd = 0, r_u_odd = 0;
    int k = 0;
    for (int lz = 0; lz < w; ++lz)
      for (int ly = 0; ly < w; ++ly)
        for (int lx = 0; lx < w; ++lx) {
          const int conv = (lz + H) * zpitch + (ly + H) * ypitch + (lx + H) * B;   // byte offset of the conventional cell
#pragma unroll
          for (int b = 0; b < B; ++b, ++k) {
            if ((k & (2 * L - 1)) == 0) {  // a4: the L Philox calls of a group cover the next 2 L slots
              const Philox4 r = philox4x32_10(cell_id, (uint32_t)(k >> 1) + g, t, ctr3, G.key0, G.key1);
              r_dir_even = r.x; r_u_even = r.y; r_dir_odd = r.z; r_u_odd = r.w;
            }
            const int src = (k >> 1) & (L - 1);
            const uint32_t w_dir = __shfl_sync(0xffffffffu, (k & 1) ? r_dir_odd : r_dir_even, src, L);
            const uint32_t u = __shfl_sync(0xffffffffu, (k & 1) ? r_u_odd : r_u_even, src, L);
            const int si = conv + b;
            const int dir = (int)mulhi_u32(w_dir, (uint32_t)G.Z0);
            const int sj = si + (int)(short)(s_nb[b * ZT + dir] & 0xffffu);
            const int sa = tile[si], sb = tile[sj];
            // a5: partial sums over this lane's neighbours of i (a -> b) and of j (b -> a); a trial between
            // equal species runs through the same code (its row of D is all zeros) and is masked below
            const int32_t* Drow = s_D + (sa * n + sb) * d_stride;
            const uint32_t* nb_i = s_nb + b * ZT;
            const uint32_t* nb_j = s_nb + (sj & (B - 1)) * ZT;
            int part = 0;
#pragma unroll 3
            for (int it = 0; it < nit; ++it) {
              const int mm = g + it * L;
              const bool valid = mm < ZT;
              const int mc = valid ? mm : 0;
              const uint32_t ei = nb_i[mc], ej = nb_j[mc];
              const int xi = tile[si + (int)(short)(ei & 0xffffu)];
              const int xj = tile[sj + (int)(short)(ej & 0xffffu)];
              const int term = Drow[(ei >> 16) + xi] - Drow[(ej >> 16) + xj];
              part += valid ? term : 0;
            }
#pragma unroll
            for (int o = L >> 1; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o, L);
            const int dE = part + Drow[corr_at];
            // a6: Eq. 3 in integer form.  ta <= T[dE] <= ta + E (host-verified); dE <= 0 maps to entry 0.
            bool ok;
            if (filter_E >= 0) {
              const uint32_t dc = (uint32_t)min(max(dE, 0), kFilterDmax);
              const uint32_t ta = mulhi_u32(s_filt[kFilterTr + (dc >> 6)], s_filt[dc & 63u]);
              ok = u < ta;
              if (u - ta <= (uint32_t)filter_E) ok = dE <= 0 || (dE < G.accept_len && u < __ldg(accept + dE));
            } else {
              ok = dE <= 0 || (dE < G.accept_len && u < __ldg(accept + dE));
            }
            ok = ok && sa != sb;
            __syncwarp();
            if (ok) {
              if (g == 0) { tile[si] = (unsigned char)sb; tile[sj] = (unsigned char)sa; }
              sum_dE += dE;
              ++n_acc;
            }
            __syncwarp();
          }
        }
  }
  if (active) {
    // a7: write back the sites a swap can have touched: positions within r0 of the cell
    const int lo = 2 * H - G.r0, hi = 2 * (H + w) - 1 + G.r0;  // tile half-unit positions, inclusive
    for (int idx = g; idx < n_conv; idx += L) {
      const int tx = idx % TW, ty = (idx / TW) % TW, tz = idx / (TW * TW);
      int gx = t0x + tx; if (gx >= G.Lx) gx -= G.Lx;
      int gy = t0y + ty; if (gy >= G.Ly) gy -= G.Ly;
      int gz = t0z + tz; if (gz >= G.Lz) gz -= G.Lz;
      const long long gi = (((long long)gz * G.Ly + gy) * G.Lx + gx) * B;
#pragma unroll
      for (int b = 0; b < B; ++b) {
        int px, py, pz;
        if (B == 2) { px = 2 * tx + b; py = 2 * ty + b; pz = 2 * tz + b; }
        else { px = 2 * tx + ((b >> 1) & 1); py = 2 * ty + ((b == 1 || b == 3) ? 1 : 0); pz = 2 * tz + ((b == 1 || b == 2) ? 1 : 0); }
        if (px >= lo && px <= hi && py >= lo && py <= hi && pz >= lo && pz <= hi)
          species[gi + b] = tile[tz * zpitch + ty * ypitch + tx * B + b];
      }
    }
  }
  // a8: one atomic pair per block (every lane of a group holds the group's sums: count lane g == 0 only)
  if (g != 0) { sum_dE = 0; n_acc = 0; }
  for (int o = 16; o > 0; o >>= 1) {
    sum_dE += __shfl_down_sync(0xffffffffu, sum_dE, o);
    n_acc += __shfl_down_sync(0xffffffffu, n_acc, o);
  }
  if (lane == 0) { s_dE[warp] = sum_dE; s_acc[warp] = n_acc; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long e = 0; unsigned a = 0;
    for (int i = 0; i < kGroupWarpsPerBlock; ++i) { e += s_dE[i]; a += s_acc[i]; }
    if (a) {
      atomicAdd(reinterpret_cast<unsigned long long*>(&st->e_run), (unsigned long long)e);
      atomicAdd(&st->accepted, (unsigned long long)a);
    }
  }
}

template <int B, int L>
inline cudaError_t configure_group_kernel(int smem_bytes) {
  cudaError_t e = cudaFuncSetAttribute(sweep_group_per_cell<B, L>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(sweep_group_per_cell<B, L>, cudaFuncAttributePreferredSharedMemoryCarveout,
                              cudaSharedmemCarveoutMaxShared);
}

inline cudaError_t configure_group_per_cell(const Geom& G, int lanes) {
  const int sm = group_smem_layout(G, lanes).total;
  if (G.B == 2) {
    switch (lanes) {
      case 4: return configure_group_kernel<2, 4>(sm);
      case 8: return configure_group_kernel<2, 8>(sm);
      case 16: return configure_group_kernel<2, 16>(sm);
      default: return configure_group_kernel<2, 32>(sm);
    }
  }
  switch (lanes) {
    case 4: return configure_group_kernel<4, 4>(sm);
    case 8: return configure_group_kernel<4, 8>(sm);
    case 16: return configure_group_kernel<4, 16>(sm);
    default: return configure_group_kernel<4, 32>(sm);
  }
}

inline void launch_group_per_cell(const Geom& G, int lanes, uint8_t* species, const int32_t* epi, const uint32_t* accept,
                                  const uint32_t* filt, DevState* st, int colour, cudaStream_t stream) {
  const GroupSmem S = group_smem_layout(G, lanes);
  const unsigned cpb = kGroupWarpsPerBlock * (32 / lanes);
  const unsigned grid = (G.cells_per_colour + cpb - 1) / cpb;
  const int nt = kGroupWarpsPerBlock * 32;
#define SMCX_GROUP_LAUNCH(BB, LL)                                                                      \
  sweep_group_per_cell<BB, LL><<<grid, nt, S.total, stream>>>(G, species, epi, accept, filt, st, colour, S.d_stride, \
                                                              S.d_bytes, S.nb_bytes, S.tile_bytes)
  if (G.B == 2) {
    switch (lanes) {
      case 4: SMCX_GROUP_LAUNCH(2, 4); break;
      case 8: SMCX_GROUP_LAUNCH(2, 8); break;
      case 16: SMCX_GROUP_LAUNCH(2, 16); break;
      default: SMCX_GROUP_LAUNCH(2, 32); break;
    }
  } else {
    switch (lanes) {
      case 4: SMCX_GROUP_LAUNCH(4, 4); break;
      case 8: SMCX_GROUP_LAUNCH(4, 8); break;
      case 16: SMCX_GROUP_LAUNCH(4, 16); break;
      default: SMCX_GROUP_LAUNCH(4, 32); break;
    }
  }
#undef SMCX_GROUP_LAUNCH
}

}  // namespace smcxk
