// Shared device-side definitions of the SMC-X CUDA path (sm_100a).
// Independent of oracle/: its own Philox, geometry tables and schedule arithmetic.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace smcxk {

// Counter tags (low byte of ctr[3]), S4.
enum : uint32_t { TAG_SHIFT = 1u, TAG_TRIAL = 2u, TAG_INIT = 3u };

constexpr int kMaxShells = 5;
constexpr int kMaxNeighbours = 80;  // FCC, 5 shells: 12+6+24+12+24 = 78
constexpr int kMaxSpecies = 16;
constexpr int kMaxGroupSlots = 128;  // neighbour slots of the sub-warp kernel: lanes * visits >= neighbours

// Philox4x32-10 (Salmon et al., SC'11).  Round keys are recomputed from the key each call; the
// additions fold into immediates when the key is a kernel parameter.
__host__ __device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2,
                                                      uint32_t& c3, uint32_t k0, uint32_t k1) {
  const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;  // IMAD.WIDE.U32
  const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
  const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
  const uint32_t n0 = hi1 ^ c1 ^ k0;
  const uint32_t n2 = hi0 ^ c3 ^ k1;
  c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}

struct Philox4 { uint32_t x, y, z, w; };

__host__ __device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2,
                                                          uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    philox_round(c0, c1, c2, c3, k0, k1);
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return Philox4{c0, c1, c2, c3};
}

// Same generator with the ten round keys precomputed (Geom::rk0 / rk1).
__device__ __forceinline__ Philox4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                    const uint32_t* rk0, const uint32_t* rk1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) philox_round(c0, c1, c2, c3, rk0[r], rk1[r]);
  return Philox4{c0, c1, c2, c3};
}

__host__ __device__ __forceinline__ uint32_t mulhi_u32(uint32_t a, uint32_t b) {
#ifdef __CUDA_ARCH__
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * b) >> 32);
#endif
}

// Device-resident bookkeeping, one per handle.
struct DevState {
  unsigned long long sweep;      // sweeps completed
  long long e_run;               // running energy E_0 + sum of accepted dE
  unsigned long long accepted;   // accepted swaps
  unsigned long long bad_state;  // set by validation kernels
  unsigned flag[2];              // connected slabs (domain_api.inc): serial of the last message that arrived from the lower [0] / upper [1] neighbour, written by that neighbour
  unsigned work[16];             // per colour (+ 8 for the second launch of a split pass, Geom::work_base): batches of cells handed out so far in this sweep (sweep_fcc_thread); zeroed by sweep_epilogue
};

// Lattice + link-cell geometry and the shell-offset tables.  Passed to kernels by value, i.e. it
// lives in the constant bank (the "shell-offset table in constant memory").
struct Geom {
  int Lx, Ly, Lz;      // conventional cells
  int B;               // sites per conventional cell (2 BCC, 4 FCC)
  int lattice;
  int n_species, n_shells;
  int w;               // link-cell edge (conventional cells)
  int H;               // halo (conventional cells) = ceil((r0 + R)/2)
  int TW;              // tile edge = w + 2H
  int r0;              // per-axis reach of shell 0 (half-lattice units)
  int ncx, ncy, ncz;   // link cells per axis
  // Slab windows (lattice parallelism, domain_api.inc): a handle that holds one slab of a lattice cut along z stores
  // the layers of its window only (Lz = storage layers, never wrapped) and runs the link-cell rows it owns.
  //   z_bias     tile origin: first tile layer = (oz + cz w + z_bias) mod Lz; Lz - H for a whole (periodic) lattice,
  //              0 for a slab (storage layer 0 is H layers below its first row at origin 0);
  //   cz_global  first link-cell row of the slab in the whole lattice (cell ids are global: they key the Philox stream);
  //   iz_first   first row pair a launch works on (a pass may be split into the boundary row and the rest).
  int z_bias, cz_global, iz_first;
  // Fused ghost-layer message (domain_api.inc): while it writes its tile back, the boundary row of a slab also stores the
  // layers [peer_z0, peer_z1) of its window into the neighbour slab's storage (a device pointer in this process: the same
  // GPU, or a peer GPU over NVLink), at the same word index of `peer_lat` = neighbour storage shifted by the difference
  // of the two windows.  0 = no mirroring.
  unsigned long long peer_lat;
  int peer_z0, peer_z1;
  int pc_z0, pc_z1;    // pair-count kernels: layers [pc_z0, pc_z1) of the source sites (the whole lattice, or the layers a slab owns)
  int work_base;       // 0 or 8: which half of DevState::work a launch of sweep_fcc_thread draws its batches from
  unsigned cells_per_colour;
  int S;               // trials per cell = w^3 B
  int Z0;              // coordination number of shell 0
  int ZT;              // neighbours over all shells
  int ZH;              // positive-half offsets over all shells (ZT/2)
  uint32_t key0, key1; // Philox key = seed
  int accept_len;
  int trace_capacity;
  // Two-level acceptance filter of the thread-per-cell kernel (see sweep_thread.cuh): disabled when
  // filter_E < 0, else T[d] - mulhi(Tq[d>>6], Tr[d&63]) lies in [0, filter_E] for every d.
  int filter_E;
  int filter_nq;
  // Philox round keys key + r * (W0, W1), r = 0..9: operands taken straight from the constant
  // bank (no per-call key schedule)
  uint32_t rk0[10], rk1[10];
  // constants the thread-per-cell kernel wants as constant-bank operands rather than immediates
  // (an IMAD takes one immediate; "dx * c0 + c1" with both constant needs the other from here):
  // kc[0] = 1, kc[1] = 0x1111, kc[2 + slot] and kc[10 + slot] per-slot constants (sweep_thread.cuh)
  uint32_t kc[18];
  // all shells concatenated, shell by shell, each in ascending (dz,dy,dx) order
  signed char off[kMaxNeighbours][3];   // half-lattice units
  unsigned char shell_of[kMaxNeighbours];
  unsigned char half_idx[kMaxNeighbours / 2];  // indices (into off) of the positive half
  // tile-linear index delta of neighbour m for a site with basis index b, and its basis index
  short delta[4][kMaxNeighbours];
  // sub-warp kernel (sweep_group.cuh), chosen on the host by a model of the shared-memory banks:
  // gslot[slot] = neighbour visited by lane (slot % lanes) in its visit (slot / lanes), 255 = none;
  // tile index of position (px, py, pz) (units of a/2) = (px + gA py + gB pz) >> gshift: gshift 0 is a plain
  // pitched byte grid, gshift 1 a compact linear index over the lattice sites only; gskew = extra distance
  // between the tiles of a warp, gtile = bytes of one tile without the skew
  unsigned char gslot[kMaxGroupSlots];
  int gA, gB, gtile;
  short gshift, gskew;
  int gd16;   // every difference V_s(b,x) - V_s(a,x) fits a signed 16-bit word (table of the sub-warp kernel)
};

}  // namespace smcxk
