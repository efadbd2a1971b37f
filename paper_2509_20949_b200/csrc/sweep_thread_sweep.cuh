// The eight colour passes of a sweep as ONE launch of the persistent thread-per-cell kernel (sweep_thread.cuh), the
// passes pipelined: a warp that has finished its batches of colour c goes on with colour c + 1 while other warps are
// still on colour c, so that the SMs stay full across the colour boundaries (BCC 800^3: a pass is only 10.6 rounds of
// batches, and a launch per colour leaves the SMs partly idle at its start and end).
//
// What may run when (S2-S3: the cells of a colour commute; a cell must see the final state of every NEIGHBOURING cell
// of the earlier colours of the sweep, and no cell may run while a neighbour of an earlier colour has not):
// cells are enumerated x fastest, then y, then z (colour_cell), cell (cx, cy, cz) = (2 ix + px, 2 iy + py, 2 iz + pz),
// colour = px | py << 1 | pz << 2.  The neighbours of a cell of colour c among the cells of colour c' < c lie
//   * in the same layer iz if c' has the same pz (colours 0-3 among themselves, 4-7 among themselves),
//   * in layers iz and iz + 1 (mod ncz / 2) if pz differs (c >= 4 > c'): cz = 2 iz + 1 has the even neighbours 2 iz, 2 iz + 2.
// A batch of colour c that touches layer iz therefore waits until colour c - 1 has completed layer iz (c = 4: layers
// iz and iz + 1 of colour 3).  That is enough for all earlier colours: the cells of colour c - 1 in those layers have
// themselves waited for colour c - 2 there, and so on.  Completion is counted per (colour, layer) and per colour in
// `progress` (cumulative over sweeps; progress[0] = whole-sweep launches so far, advanced by whole_sweep_epoch): a warp
// adds the cells of a batch with a release after its write-back; a warp that starts a batch reads the counters with
// acquire loads -- first the count of the whole previous colour, and once that is complete it asks no more.
// No deadlock: a wait always points to an earlier colour, colour 0 never waits, and all blocks are resident (one per
// SM, never more blocks than SMs; the host gives this mode to one handle per process at a time, so that two such
// launches never hold SMs while waiting for blocks of their own that cannot get one).
#pragma once
#include "sweep_thread.cuh"

namespace smcxk {

__global__ void whole_sweep_epoch(unsigned* progress) { progress[0] += 1u; }

// progress: [0] launches so far, [1 + c * (ncz / 2) + iz] cells of colour c completed in layer iz, then [c] per colour
inline size_t whole_sweep_progress_words(const Geom& G) { return 1 + 8 * (size_t)(G.ncz >> 1) + 8; }

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_add_u32(unsigned* p, unsigned v) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

template <bool PK>
__global__ void __launch_bounds__(kPersistMaxWarps * 32, 1)
sweep_thread_whole_sweep(const Geom G, uint32_t* __restrict__ lattice, const int4* __restrict__ coef,
                         const uint32_t* __restrict__ accept, DevState* __restrict__ st, unsigned* __restrict__ progress) {
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
  TrialEnv env;
  env.coef = smem_ptr(s_coef0) + (lane & 7) * 16;
  env.filt = smem_ptr(s_T);
  env.accept = accept;
  env.accept_len = G.accept_len;
  env.filter_E = 0;
  env.tmax4 = 4u * (uint32_t)G.accept_len;
  const uint32_t n_batches = (G.cells_per_colour + 31u) >> 5;
  const uint32_t cpl = (uint32_t)(G.ncx >> 1) * (uint32_t)(G.ncy >> 1);      // cells of a colour per layer iz
  const uint32_t nzh = (uint32_t)(G.ncz >> 1);
  const unsigned epoch1 = *reinterpret_cast<volatile unsigned*>(progress) + 1u;
  const unsigned layer_target = epoch1 * cpl;                   // a layer / a colour is complete in THIS sweep at these counts
  const unsigned colour_target = epoch1 * G.cells_per_colour;
  unsigned* const layer_done = progress + 1;                    // [colour][layer]
  unsigned* const colour_done = progress + 1 + 8u * nzh;        // [colour]
  __syncthreads();
#pragma unroll 1
  for (int colour = 0; colour < 8; ++colour) {
  const uint32_t ctr3 = TAG_TRIAL | ((uint32_t)colour << 8);
  bool prev_complete = colour == 0;                             // the whole previous colour has been seen complete
  // warp-major numbering, as in sweep_thread_persistent
#pragma unroll 1
  for (uint32_t batch = (uint32_t)warp * gridDim.x + blockIdx.x; batch < n_batches; batch += (uint32_t)n_warps * gridDim.x) {
    const uint32_t m_first = batch * 32u;
    const uint32_t m_last = min(m_first + 31u, G.cells_per_colour - 1u);
    const uint32_t iz0 = m_first / cpl, iz1 = m_last / cpl;     // the layers the batch touches (one or two unless the lattice is tiny)
    if (!prev_complete) {
      // a4 may start once the neighbouring cells of the earlier colours are complete (see the head of this file).  The
      // acquire loads order the plain loads of the staging below after the stores the other warps released (and drop
      // what this SM's L1 holds of them); __syncwarp carries that to the other lanes.
      unsigned all = 0u;
      if (lane == 0) {
        all = ld_acquire_u32(colour_done + (colour - 1));
        if ((int)(all - colour_target) < 0) {
          const unsigned* prev = layer_done + (uint32_t)(colour - 1) * nzh;
          const uint32_t last_needed = colour == 4 ? iz1 + 1u : iz1;          // colour 4: layers iz and iz + 1 of colour 3
          for (uint32_t z = iz0; z <= last_needed; ++z) {
            const unsigned* p = prev + (z >= nzh ? z - nzh : z);
            while ((int)(ld_acquire_u32(p) - layer_target) < 0) __nanosleep(200);
          }
        }
      }
      __syncwarp();                                            // memory ordering for the other lanes (a shuffle gives none)
      all = __shfl_sync(0xffffffffu, all, 0);
      prev_complete = (int)(all - colour_target) >= 0;
    }
    const uint32_t m = m_first + (uint32_t)lane;
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
    // publish: the cells of this batch are complete (release by one lane: the warp barrier orders the stores of the
    // other lanes before it)
    __syncwarp();
    if (lane == 0) {
      for (uint32_t z = iz0; z <= iz1; ++z)
        red_release_add_u32(layer_done + (uint32_t)colour * nzh + z, min(m_last + 1u, (z + 1u) * cpl) - max(m_first, z * cpl));
      red_release_add_u32(colour_done + colour, m_last + 1u - m_first);
    }
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


inline int configure_whole_sweep() {
  if (cudaFuncSetAttribute(sweep_thread_whole_sweep<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPersistSmemMax) != cudaSuccess) return -1;
  if (cudaFuncSetAttribute(sweep_thread_whole_sweep<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPersistSmemMax) != cudaSuccess) return -1;
  return 0;
}

// grid: one block per SM at most -- the warps of a block wait for other blocks, which must all be resident
inline int launch_whole_sweep(const Geom& G, uint32_t* lattice, const int32_t* d_coef, bool packed, const uint32_t* accept,
                              DevState* st, unsigned* progress, int warps, int sm_count, cudaStream_t stream) {
  const unsigned n_batches = (G.cells_per_colour + 31u) / 32u;
  const unsigned want = (n_batches + warps - 1) / warps;
  const unsigned grid = want < (unsigned)sm_count ? want : (unsigned)sm_count;
  if (packed)
    sweep_thread_whole_sweep<true><<<grid, warps * 32, persist_smem(warps, G.accept_len), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef + 16 * kCoefInts), accept, st, progress);
  else
    sweep_thread_whole_sweep<false><<<grid, warps * 32, persist_smem(warps, G.accept_len), stream>>>(
        G, lattice, reinterpret_cast<const int4*>(d_coef), accept, st, progress);
  whole_sweep_epoch<<<1, 1, 0, stream>>>(progress);
  return cudaGetLastError() == cudaSuccess ? 0 : -1;
}

}  // namespace smcxk
