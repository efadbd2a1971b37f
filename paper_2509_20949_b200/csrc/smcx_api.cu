// C ABI of the SMC-X CUDA path (include/smcx.h): validation, host-side geometry tables,
// workspace layout, launch orchestration.  No CPU fallback: every step of the hot path runs in
// the kernels of this directory.
#include "../../include/smcx.h"

#include <algorithm>
#include <atomic>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>   // header-only; ranges cost nothing without a profiler attached

#include "ensemble_kernels.cuh"
#include "lattice_kernels.cuh"
#include "smcx_common.cuh"
#include "sweep_bcc4.cuh"
#include "sweep_fcc.cuh"
#include "sweep_group.cuh"
#include "sweep_local.cuh"
#include "sweep_thread.cuh"
#include "sweep_thread_sweep.cuh"
#include "sweep_warp.cuh"

using namespace smcxk;

struct smcx;
static std::atomic<smcx*> g_whole_sweep_owner{nullptr};   // see smcx_create
constexpr long long kWholeSweepMaxCells = 2400000;         // link cells per colour: about 25 rounds of batches

namespace {

constexpr long long kPackedMinCellsPerColour = 12000;   // AUTO: packed 4-bit kernels from this many link cells per colour
constexpr int kAcceptCapacity = 1 << 20;  // entries reserved on the device for the threshold table
constexpr int kStagingSlots = 4;
constexpr long long kChunkSites = 1ll << 26;  // bounce-buffer size for packed <-> uint8 transfers

struct ShellVec { int x, y, z, d2; };

// S0: lattice translations of BCC (all components of equal parity) and FCC (even component sum)
// in units of a/2, grouped by squared length; within a shell ascending (dz, dy, dx).
std::vector<std::vector<ShellVec>> build_shells(int lattice, int n_shells) {
  std::vector<ShellVec> all;
  const int R = 6;
  for (int z = -R; z <= R; ++z)
    for (int y = -R; y <= R; ++y)
      for (int x = -R; x <= R; ++x) {
        if (x == 0 && y == 0 && z == 0) continue;
        const bool ok = lattice == SMCX_BCC ? (((x ^ y) & 1) == 0 && ((y ^ z) & 1) == 0) : (((x + y + z) & 1) == 0);
        if (ok) all.push_back({x, y, z, x * x + y * y + z * z});
      }
  std::stable_sort(all.begin(), all.end(), [](const ShellVec& a, const ShellVec& b) {
    if (a.d2 != b.d2) return a.d2 < b.d2;
    if (a.z != b.z) return a.z < b.z;
    if (a.y != b.y) return a.y < b.y;
    return a.x < b.x;
  });
  std::vector<std::vector<ShellVec>> shells;
  for (size_t k = 0; k < all.size() && (int)shells.size() <= n_shells; ++k) {
    if (k == 0 || all[k].d2 != all[k - 1].d2) {
      if ((int)shells.size() == n_shells) break;
      shells.emplace_back();
    }
    shells.back().push_back(all[k]);
  }
  return shells;
}

void basis_pos(int lattice, int b, int p[3]) {
  if (lattice == SMCX_BCC) { p[0] = p[1] = p[2] = b; return; }
  static const int f[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};
  p[0] = f[b][0]; p[1] = f[b][1]; p[2] = f[b][2];
}

int basis_from_parity(int lattice, int px, int py, int pz) {
  if (lattice == SMCX_BCC) return px & 1;
  const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
  return par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3;
}

inline int floor_div2(int v) { return v >= 0 ? v / 2 : -((-v + 1) / 2); }

inline bool is_thread_kernel(int k) { return k == SMCX_KERNEL_THREAD_PER_CELL || k == SMCX_KERNEL_THREAD_PERSISTENT; }
// kernels whose write-back can mirror the layers of a slab's pass message into the neighbour's storage
inline bool has_fused_writeback(int k) { return is_thread_kernel(k) || k == SMCX_KERNEL_FCC_THREAD || k == SMCX_KERNEL_BCC4_THREAD; }

struct Layout {
  size_t species, epi, coef, gtable, fcc_lut, fcc_corr, quad, utab, ucount, accept, filter, trace, state, counts, progress, total;
};

struct Plan {
  Geom G;
  long long n_sites;
  long long n_cells;
  int storage;
  int kernel;
  int group_lanes;  // lanes per cell of the sub-warp kernel
  int group_warps;  // its warps per block
  int coef_class;   // build_thread_coefficients: 2 = the filter variant of the thread kernel applies
  bool coef_packed; // pack_thread_coefficients: the 16-bit coefficient rows are exact
  int fcc_rep;      // sweep_fcc_thread: replicas of the look-up rows in shared memory
  int accept_tail_from = 0;   // T[k] >= T[d] for every d > k holds for all k >= this (0 for a table that never increases)
  int accept_tail_floor = 0;  // replica of an ensemble: the same for the weakest of the ensemble's tables (they move on the device)
  FccTables fcc_tables;
  Bcc4Tables bcc4_tables;
  Layout lay;
  int model = SMCX_MODEL_EPI;
  int local_umax = 0;   // SMCX_MODEL_LOCAL: affected sites per (basis, direction, shell), at most
  // Slab window (params domain_count >= 2): this handle holds slab domain_index of the lattice cut along z
  // (domain_api.inc).  n_sites then counts the sites of the window's storage, n_global those of the whole lattice.
  bool window = false;
  int dom_count = 1, dom_index = 0;
  int row_first = 0, row_count = 0;   // link-cell rows owned
  int z_base = 0;                     // layer of the whole lattice held in storage layer 0 (mod Lz_global)
  int Lz_global = 0;
  long long n_global = 0;
  long long layer_sites = 0;          // sites per layer = Lx Ly B
};

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

size_t storage_bytes(int storage, long long n_sites) {
  if (storage == SMCX_STORAGE_U8) return (size_t)n_sites;
  if (storage == SMCX_STORAGE_2BIT) return (size_t)((n_sites + 15) / 16) * 4;
  return (size_t)((n_sites + 7) / 8) * 4;   // 4BIT
}


void build_local_utable(const Plan& P, int lattice, std::vector<LocalUEntry>& tab, std::vector<int>& count);

int make_plan(const smcx_params_t* p, Plan* plan) {
  if (!p || !plan) return SMCX_E_NULL_ARG;
  if (p->lattice != SMCX_BCC && p->lattice != SMCX_FCC) return SMCX_E_BAD_LATTICE;
  if (p->n_species < 2 || p->n_species > kMaxSpecies) return SMCX_E_BAD_SPECIES;
  if (p->n_shells < 1 || p->n_shells > kMaxShells) return SMCX_E_BAD_SHELLS;
  if (!p->epi) return SMCX_E_NULL_ARG;
  if (!p->accept || p->accept_len < 1 || p->accept_len > kAcceptCapacity) return SMCX_E_BAD_TABLE;
  const int n = p->n_species;
  if (p->model != SMCX_MODEL_EPI && p->model != SMCX_MODEL_LOCAL) return SMCX_E_UNSUPPORTED;
  const bool local = p->model == SMCX_MODEL_LOCAL;
  plan->model = p->model;
  if (local && !p->local_quad) return SMCX_E_NULL_ARG;
  if (local && n > kLocalMaxSpecies) return SMCX_E_UNSUPPORTED;
  for (int s = 0; s < p->n_shells && !local; ++s)
    for (int a = 0; a < n; ++a)
      for (int b = 0; b < a; ++b)
        if (p->epi[(s * n + a) * n + b] != p->epi[(s * n + b) * n + a]) return SMCX_E_EPI_NOT_SYMMETRIC;
  const int w = p->link_cell == 0 ? 4 : p->link_cell;
  if (w < 1 || w > 16) return SMCX_E_LINK_CELL_TOO_SMALL;

  Geom& G = plan->G;
  std::memset(&G, 0, sizeof(G));
  G.lattice = p->lattice;
  G.B = p->lattice == SMCX_BCC ? 2 : 4;
  G.n_species = n;
  G.n_shells = p->n_shells;
  G.w = w;
  const auto shells = build_shells(p->lattice, p->n_shells);
  int m = 0, R = 0, r0 = 0, nh = 0;
  for (int s = 0; s < p->n_shells; ++s)
    for (const ShellVec& v : shells[s]) {
      if (m >= kMaxNeighbours) return SMCX_E_BAD_SHELLS;
      G.off[m][0] = (signed char)v.x; G.off[m][1] = (signed char)v.y; G.off[m][2] = (signed char)v.z;
      G.shell_of[m] = (unsigned char)s;
      const int reach = std::max(std::abs(v.x), std::max(std::abs(v.y), std::abs(v.z)));
      R = std::max(R, reach);
      if (s == 0) r0 = std::max(r0, reach);
      const int first = v.z != 0 ? v.z : (v.y != 0 ? v.y : v.x);
      if (first > 0) G.half_idx[nh++] = (unsigned char)m;
      ++m;
    }
  G.ZT = m;
  G.ZH = nh;
  G.Z0 = (int)shells[0].size();
  G.r0 = r0;
  // S2: same-colour cells must not interact during a pass: 2w >= 2 r0 + R (w in conventional cells).
  // reading S12: a trial of the local model reads the neighbours of the neighbours of i and j (reach r0 + 2 R)
  const int reach = local ? r0 + 2 * R : r0 + R;
  if (2 * w < r0 + reach) return SMCX_E_LINK_CELL_TOO_SMALL;
  G.H = (reach + 1) / 2;
  G.TW = w + 2 * G.H;
  group_default_layout(G);     // until group_tune_layout() has run
  long long n_sites = G.B;
  for (int a = 0; a < 3; ++a) {
    const int L = p->dims[a];
    if (L <= 0 || L % (2 * w) != 0 || L < G.TW) return SMCX_E_BAD_DIMS;
    n_sites *= L;
    if (n_sites > (1ll << 40)) return SMCX_E_BAD_DIMS;
  }
  G.Lx = p->dims[0]; G.Ly = p->dims[1]; G.Lz = p->dims[2];
  G.ncx = G.Lx / w; G.ncy = G.Ly / w; G.ncz = G.Lz / w;
  const long long n_cells = (long long)G.ncx * G.ncy * G.ncz;
  if (n_cells > 0xffffffffll) return SMCX_E_BAD_DIMS;  // cell id is a 32-bit Philox counter word
  G.cells_per_colour = (unsigned)(n_cells / 8);
  G.z_bias = G.Lz - G.H;
  G.cz_global = 0;
  G.iz_first = 0;
  G.work_base = 0;
  G.pc_z0 = 0;
  G.pc_z1 = G.Lz;
  plan->Lz_global = G.Lz;
  plan->n_global = n_sites;
  plan->layer_sites = (long long)G.Lx * G.Ly * G.B;
  plan->window = false;
  plan->dom_count = 1;
  plan->dom_index = 0;
  plan->row_first = 0;
  plan->row_count = G.ncz;
  plan->z_base = 0;
  if (p->domain_count >= 2) {
    // reading S11: slabs on pairs of link-cell rows; the window holds the rows' layers for every origin oz < w plus
    // H ghost layers on either side, stored without wrap
    const int D = p->domain_count, k = p->domain_index;
    const int pairs = G.ncz / 2;
    if (k < 0 || k >= D || D > pairs) return SMCX_E_BAD_DIMS;
    int first = 0, count = 0;
    for (int q = 0; q <= k; ++q) { first += count; count = 2 * (pairs / D + (q < pairs % D ? 1 : 0)); }
    const int layers = count * w + w - 1 + 2 * G.H;
    if (layers > G.Lz) return SMCX_E_BAD_DIMS;
    plan->window = true;
    plan->dom_count = D;
    plan->dom_index = k;
    plan->row_first = first;
    plan->row_count = count;
    plan->z_base = ((first * w - G.H) % G.Lz + G.Lz) % G.Lz;
    G.Lz = layers;
    G.ncz = count;
    G.z_bias = 0;
    G.cz_global = first;
    G.cells_per_colour = (unsigned)((long long)G.ncx * G.ncy * count / 8);
    G.pc_z0 = G.H;
    G.pc_z1 = G.H + count * w;
    n_sites = plan->layer_sites * layers;
  }
  G.S = w * w * w * G.B;
  G.key0 = (uint32_t)(p->seed & 0xffffffffull);
  G.key1 = (uint32_t)(p->seed >> 32);
  G.accept_len = p->accept_len;
  G.trace_capacity = p->trace_capacity > 0 ? p->trace_capacity : 65536;
  G.filter_E = -1;
  set_thread_masks(G);  // needs key0/key1
  // tile-linear deltas
  for (int b = 0; b < G.B; ++b) {
    int bp[3];
    basis_pos(p->lattice, b, bp);
    for (int k = 0; k < G.ZT; ++k) {
      const int qx = bp[0] + G.off[k][0], qy = bp[1] + G.off[k][1], qz = bp[2] + G.off[k][2];
      const int nb = basis_from_parity(p->lattice, qx, qy, qz);
      const int dcx = floor_div2(qx), dcy = floor_div2(qy), dcz = floor_div2(qz);
      const int d = ((dcz * G.TW + dcy) * G.TW + dcx) * G.B + (nb - b);
      if (d < -32768 || d > 32767) return SMCX_E_LINK_CELL_TOO_SMALL;
      G.delta[b][k] = (short)d;
    }
  }
  plan->n_sites = n_sites;
  plan->n_cells = plan->window ? (long long)G.ncx * G.ncy * G.ncz : n_cells;

  // kernel / storage choice
  bool fast_ok = thread_kernel_supported(G);
  plan->coef_class = 0;
  plan->coef_packed = false;
  if (fast_ok) {  // the packed kernel computes dE in int32 from a coefficient table: magnitudes must fit
    int32_t coef[16 * kCoefInts];
    plan->coef_class = build_thread_coefficients(p->epi, n, coef);
    fast_ok = plan->coef_class > 0;
    int32_t pk[16 * 4];
    plan->coef_packed = fast_ok && pack_thread_coefficients(coef, pk);
  }
  // packed FCC kernel: geometry, and every EPI difference must fit the 16-bit look-up
  bool fcc_ok = fcc_kernel_supported(G);
  plan->fcc_rep = 1;
  if (fcc_ok) {
    std::vector<uint32_t> lut;
    std::vector<int32_t> corr;
    fcc_ok = fcc_build_lut(p->epi, n, p->n_shells, 1, lut, corr) && fcc_build_tables<32, kFccWinRows>(G, plan->fcc_tables);
    plan->fcc_rep = fcc_lut_rep(n);
  }
  // packed BCC kernel for up to 8 species (4-bit storage): geometry, and every EPI difference must fit the 16-bit look-up
  bool bcc4_ok = bcc4_kernel_supported(G);
  if (bcc4_ok) {
    std::vector<uint32_t> lut;
    std::vector<int32_t> corr;
    bcc4_ok = fcc_build_lut(p->epi, n, p->n_shells, 1, lut, corr) && bcc4_build_tables<32, kBcc4WinRows>(G, plan->bcc4_tables);
  }
  int kernel = p->kernel, storage = p->storage;
  if (local) bcc4_ok = false;
  if (local) {
    if (kernel == SMCX_KERNEL_AUTO) kernel = SMCX_KERNEL_LOCAL_WARP;
    if (kernel != SMCX_KERNEL_LOCAL_WARP) return SMCX_E_UNSUPPORTED;
    fast_ok = fcc_ok = false;
    // int32 arithmetic of the kernel: |eps| <= sum_s (Z_s max|W1| + Z_s^2 max|W2|), |dE| <= 2 |U| max|eps|
    long long m1 = 0, m2 = 0, eps = 0;
    for (int k = 0; k < p->n_shells * n * n; ++k) m1 = std::max(m1, std::llabs((long long)p->epi[k]));
    for (int k = 0; k < p->n_shells * n * n * n; ++k) m2 = std::max(m2, std::llabs((long long)p->local_quad[k]));
    for (int s = 0; s < p->n_shells; ++s) { const long long Z = (long long)shells[s].size(); eps += Z * m1 + Z * Z * m2; }
    if (2 * (2 + 2ll * G.ZT) * eps >= (1ll << 31)) return SMCX_E_EPI_RANGE;
  } else if (kernel == SMCX_KERNEL_LOCAL_WARP) {
    return SMCX_E_UNSUPPORTED;
  }
  if (kernel == SMCX_KERNEL_AUTO) {
    // The packed thread-per-cell kernels (a warp = 32 cells, a pass at least one cell's chain of trials long) against the
    // sub-warp kernel (several lanes per cell), measured on lattices of growing size (profiles/README.md): the packed
    // kernels win from about 12,000 link cells per colour on (2.5 batches of 32 cells per SM) -- FCC 192^3: 1.9e10 against
    // 1.6e10, FCC 256^3: 4.6e10 against 1.8e10; BCC with five species 256^3: 4.8e10 against 2.4e10 -- and lose below
    // (8,000 cells per colour: 1.06e10 against 1.3e10).
    if (fcc_ok && (storage == SMCX_STORAGE_4BIT || (storage == SMCX_STORAGE_AUTO && plan->n_cells / 8 >= kPackedMinCellsPerColour)))
      kernel = SMCX_KERNEL_FCC_THREAD;
    else if (bcc4_ok && (storage == SMCX_STORAGE_4BIT || (storage == SMCX_STORAGE_AUTO && !fast_ok && plan->n_cells / 8 >= kPackedMinCellsPerColour)))
      kernel = SMCX_KERNEL_BCC4_THREAD;
    else if (storage == SMCX_STORAGE_U8) kernel = SMCX_KERNEL_GROUP_PER_CELL;
    else if (!fast_ok) kernel = SMCX_KERNEL_GROUP_PER_CELL;
    // The persistent kernel (one block of 20 warps and ~220 KB of shared memory per SM) pays off once
    // every warp of every SM gets a batch of 32 cells.  Below that a colour pass is as long as one
    // cell's chain of trials with either kernel, and concurrent launches of the persistent kernel
    // (replica ensembles) cost ~20 us each where those of the block kernel overlap freely (measured:
    // 32 replicas of BCC 64^3, 0.416 ms against 0.238 ms per sweep of all replicas).
    else kernel = plan->n_cells / 8 >= 148ll * kPersistMaxWarps * 32 ? SMCX_KERNEL_THREAD_PERSISTENT : SMCX_KERNEL_THREAD_PER_CELL;
  }
  if (kernel == SMCX_KERNEL_THREAD_PER_CELL || kernel == SMCX_KERNEL_THREAD_PERSISTENT) {
    if (!fast_ok) return SMCX_E_UNSUPPORTED;
    if (storage == SMCX_STORAGE_AUTO) storage = SMCX_STORAGE_2BIT;
    if (storage != SMCX_STORAGE_2BIT) return SMCX_E_UNSUPPORTED;
  } else if (kernel == SMCX_KERNEL_FCC_THREAD) {
    if (!fcc_ok) return SMCX_E_UNSUPPORTED;
    if (storage == SMCX_STORAGE_AUTO) storage = SMCX_STORAGE_4BIT;
    if (storage != SMCX_STORAGE_4BIT) return SMCX_E_UNSUPPORTED;
  } else if (kernel == SMCX_KERNEL_BCC4_THREAD) {
    if (!bcc4_ok) return SMCX_E_UNSUPPORTED;
    if (storage == SMCX_STORAGE_AUTO) storage = SMCX_STORAGE_4BIT;
    if (storage != SMCX_STORAGE_4BIT) return SMCX_E_UNSUPPORTED;
    plan->fcc_rep = bcc4_lut_rep();
  } else if (kernel == SMCX_KERNEL_WARP_PER_CELL || kernel == SMCX_KERNEL_GROUP_PER_CELL || kernel == SMCX_KERNEL_LOCAL_WARP) {
    if (storage == SMCX_STORAGE_AUTO) storage = SMCX_STORAGE_U8;
    if (storage != SMCX_STORAGE_U8) return SMCX_E_UNSUPPORTED;
  } else {
    return SMCX_E_UNSUPPORTED;
  }
  if (storage == SMCX_STORAGE_4BIT && (G.Lx & 7) != 0) return SMCX_E_UNSUPPORTED;
  plan->kernel = kernel;
  plan->storage = storage;
  // sub-warp kernel: lanes per cell by the number of cells of a colour.  With few cells a pass is as long as
  // one cell's chain of trials, which more lanes shorten; with many, fewer lanes mean less replicated work.
  // Measured on FCC, 5 species, 3 shells (ms per sweep with 8 / 16 / 32 lanes): 128^3 (4,096 cells per colour)
  // 0.99 / 0.87 / 1.00; 400^3 (125,000 cells per colour) 14.9 / 15.5 / 21.9.
  plan->group_lanes = 32;
  if (group_smem_layout(G, 16, 2).total <= 227 * 1024 && (long long)G.cells_per_colour * 16 / 32 >= 148ll * 12)
    plan->group_lanes = 16;
  if (group_smem_layout(G, 8, 2).total <= 227 * 1024 && (long long)G.cells_per_colour * 8 / 32 >= 148ll * 48)
    plan->group_lanes = 8;
  if (p->group_lanes != 0) {
    const int v = p->group_lanes;
    if (v != 4 && v != 8 && v != 16 && v != 32) return SMCX_E_UNSUPPORTED;
    if (group_smem_layout(G, v, 2).total <= 227 * 1024) plan->group_lanes = v;
  }
  if (p->group_warps < 0 || p->group_warps > kGroupWarpsPerBlock) return SMCX_E_UNSUPPORTED;
  {
    // the generic kernels compute dE = sum over 2 ZT neighbours of D_s(x) + corr(a,b) in int32
    long long max_d = 0;   // largest |V_s(b,x) - V_s(a,x)|
    for (int s = 0; s < p->n_shells; ++s)
      for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b)
          for (int x = 0; x < n; ++x)
            max_d = std::max(max_d, std::llabs((long long)p->epi[(s * n + b) * n + x] - (long long)p->epi[(s * n + a) * n + x]));
    G.gd16 = max_d <= 32767 ? 1 : 0;
    if ((2ll * G.ZT + 2 * kMaxGroupSlots + 4) * max_d >= (1ll << 31)) return SMCX_E_EPI_RANGE;
  }
  group_tune_layout(G, plan->group_lanes);
  plan->group_warps = group_warps_per_block(G, plan->group_lanes, p->group_warps);
  if (kernel == SMCX_KERNEL_GROUP_PER_CELL && group_smem_layout(G, plan->group_lanes, 2).total > 227 * 1024)
    return SMCX_E_LINK_CELL_TOO_SMALL;

  Layout& L = plan->lay;
  size_t off = 0;
  L.species = off;
  off += align_up(storage_bytes(storage, n_sites), 256);
  L.epi = off;     off += align_up((size_t)p->n_shells * n * n * sizeof(int32_t), 256);
  L.coef = off;    off += align_up((size_t)16 * (kCoefInts + 4) * sizeof(int32_t), 256);
  L.gtable = off;  off += align_up((size_t)group_smem_layout(G, plan->group_lanes).d_bytes, 256);   // sub-warp kernel's difference table
  L.fcc_lut = off; off += align_up((size_t)64 * 3 * 8 * 16, 256);                                   // packed FCC kernel's look-up rows
  L.fcc_corr = off; off += align_up((size_t)64 * sizeof(int32_t), 256);
  {   // SMCX_MODEL_LOCAL: affected (site, shell) pairs per (basis, direction, shell), at most: i, j and 2 Z_s neighbours
    int zmax = 0;
    for (int s2 = 0; s2 < p->n_shells; ++s2) zmax = std::max(zmax, (int)shells[s2].size());
    // units of the flat list (build_local_utable): per shell at most 2 Z_s sites, each in ceil(Z_s / 12) chunks
    int units = 0;
    for (int s2 = 0; s2 < p->n_shells; ++s2) {
      const int z = (int)shells[s2].size();
      units += 2 * z * ((z + kLocalChunk - 1) / kLocalChunk);
      const int last = z % kLocalChunk == 0 ? kLocalChunk : z % kLocalChunk;     // length of the last (or only) chunk
      if (local && local_chunk_code(last) < 0) return SMCX_E_UNSUPPORTED;
    }
    (void)zmax;
    plan->local_umax = local ? units : 0;
    if (local) {
      // the exact length of the longest list (sites that see both i and j drop out): shared memory per block
      std::vector<LocalUEntry> tab;
      std::vector<int> count;
      build_local_utable(*plan, p->lattice, tab, count);
      int longest = 1;
      for (int c : count) longest = std::max(longest, c);
      plan->local_umax = longest;
    }
  }
  L.quad = off;    off += align_up(local ? (size_t)p->n_shells * n * n * n * sizeof(int32_t) : 0, 256);
  L.utab = off;    off += align_up((size_t)G.B * G.Z0 * plan->local_umax * sizeof(LocalUEntry), 256);
  L.ucount = off;  off += align_up(local ? (size_t)G.B * G.Z0 * sizeof(int) : 0, 256);
  if (local && local_smem_bytes(G, plan->local_umax) > 227 * 1024) return SMCX_E_LINK_CELL_TOO_SMALL;
  L.accept = off;  off += align_up(((size_t)kAcceptCapacity + 1) * sizeof(uint32_t), 256);   // T and the zero entry behind it
  L.filter = off;  off += align_up((size_t)kFilterWords * sizeof(uint32_t), 256);
  L.trace = off;   off += align_up((size_t)G.trace_capacity * sizeof(long long), 256);
  L.state = off;   off += align_up(sizeof(DevState), 256);
  L.counts = off;  off += align_up((size_t)kMaxShells * kMaxSpecies * kMaxSpecies * sizeof(unsigned long long), 256);
  L.progress = off; off += align_up(whole_sweep_progress_words(G) * sizeof(unsigned), 256);   // sweep_thread_whole_sweep
  L.total = off;
  return SMCX_OK;
}

// SMCX_MODEL_LOCAL: for every (basis b of i, direction, shell s), the sites whose shell-s term of the local energy the
// swap changes -- i, j, and the sites that see i or j in shell s, each once -- as tile-linear steps from i.
void build_local_utable(const Plan& P, int lattice, std::vector<LocalUEntry>& tab, std::vector<int>& count) {
  const Geom& G = P.G;
  const int umax = P.local_umax;
  tab.assign((size_t)G.B * G.Z0 * umax, LocalUEntry{0, 0});
  count.assign((size_t)G.B * G.Z0, 0);
  auto shell_of_vec = [&](int x, int y, int z) {
    for (int m = 0; m < G.ZT; ++m)
      if (G.off[m][0] == x && G.off[m][1] == y && G.off[m][2] == z) return (int)G.shell_of[m];
    return -1;
  };
  std::vector<int> start(G.n_shells + 1, G.ZT);
  for (int m = G.ZT - 1; m >= 0; --m) start[G.shell_of[m]] = m;
  for (int b = 0; b < G.B; ++b) {
    int bp[3];
    basis_pos(lattice, b, bp);
    for (int dir = 0; dir < G.Z0; ++dir) {
      const int jx = G.off[dir][0], jy = G.off[dir][1], jz = G.off[dir][2];
      std::vector<std::array<int, 3>> U;
      auto add = [&](int x, int y, int z) {
        for (const auto& v : U)
          if (v[0] == x && v[1] == y && v[2] == z) return;
        U.push_back({x, y, z});
      };
      for (int m = 0; m < G.ZT; ++m) {
        add(G.off[m][0], G.off[m][1], G.off[m][2]);
        add(jx + G.off[m][0], jy + G.off[m][1], jz + G.off[m][2]);
      }
      // units, longest chunks first so that the lanes of a round count about equally many neighbours
      std::vector<LocalUEntry> units[kLocalChunk + 1];
      for (int s = 0; s < G.n_shells; ++s) {
        const int zs = start[s + 1] - start[s];
        for (const auto& v : U) {
          const int vx = v[0], vy = v[1], vz = v[2];
          if ((vx == 0 && vy == 0 && vz == 0) || (vx == jx && vy == jy && vz == jz)) continue;   // i, j: the kernel's own round
          const bool sees_i = shell_of_vec(-vx, -vy, -vz) == s;              // i - u in shell s
          const bool sees_j = shell_of_vec(jx - vx, jy - vy, jz - vz) == s;  // j - u in shell s
          if (sees_i == sees_j) continue;                                     // sees neither, or both: its counts stay
          const int qx = bp[0] + vx, qy = bp[1] + vy, qz = bp[2] + vz;
          const int nb = basis_from_parity(lattice, qx, qy, qz);
          const int d = ((floor_div2(qz) * G.TW + floor_div2(qy)) * G.TW + floor_div2(qx)) * G.B + (nb - b);
          for (int c0 = 0; c0 < zs; c0 += kLocalChunk) {
            const int len = std::min(kLocalChunk, zs - c0);
            LocalUEntry e;
            e.delta = (short)d;
            e.bits = (unsigned short)((sees_j ? 1u : 0u) | (c0 == 0 ? 2u : 0u) | ((unsigned)nb << 2) | ((unsigned)s << 4) |
                                      ((unsigned)(start[s] + c0) << 7) | ((unsigned)local_chunk_code(len) << 14));
            units[len].push_back(e);
          }
        }
      }
      LocalUEntry* out = tab.data() + (size_t)(b * G.Z0 + dir) * umax;
      int k = 0;
      for (int len = kLocalChunk; len >= 1; --len)
        for (const LocalUEntry& e : units[len]) out[k++] = e;
      count[(size_t)b * G.Z0 + dir] = k;
    }
  }
}

}  // namespace

// kernels that read the two-level acceptance filter tables
inline bool uses_filter(const Plan& P) {
  return (is_thread_kernel(P.kernel) && P.coef_class == 2) || P.kernel == SMCX_KERNEL_GROUP_PER_CELL ||
         P.kernel == SMCX_KERNEL_FCC_THREAD || P.kernel == SMCX_KERNEL_BCC4_THREAD;
}

struct smcx {
  Plan plan;
  int device = 0;
  cudaStream_t stream = nullptr;
  char* ws = nullptr;
  bool owns_ws = false;
  long long graph_launches = 9;   // kernels per replay of sweep_graph
  bool whole_sweep = false;   // smcx_sweep runs the eight colour passes as one launch (sweep_thread_sweep.cuh)
  std::vector<int32_t> epi;
  int kT_units = 0;
  uint32_t* staging[kStagingSlots] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t staging_ev[kStagingSlots] = {nullptr, nullptr, nullptr, nullptr};
  size_t staging_cap = 0;
  int staging_next = 0;
  // packed <-> uint8 host transfers: two device bounce buffers of kChunkSites bytes (lazily allocated), a copy
  // stream, and per buffer the events "filled" / "free again"
  uint8_t* bounce[2] = {nullptr, nullptr};
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t bounce_full[2] = {nullptr, nullptr}, bounce_free[2] = {nullptr, nullptr};
  long long sweeps_enqueued = 0;
  long long trace_first = 0;  // first sweep whose energy the trace holds (smcx_set_sweep_counter moves it)
  long long launches = 0;
  // one sweep (8 colour passes + epilogue) captured as a CUDA graph; re-captured when the kernel
  // parameters change (new threshold table)
  cudaStream_t capture_stream = nullptr;
  cudaGraphExec_t sweep_graph = nullptr;
  long long params_epoch = 0, graph_epoch = -1;
  bool graphs_ok = true;
  int sm_count = 148;
  std::string err;
  // slab window: origin oz of the sweep begun last (0 after an initial state or an upload, when every layer of the
  // window is valid); the layers the slab owns are storage layers [H + win_oz, H + win_oz + row_count w)
  int win_oz = 0;

  uint8_t* d_species() const { return reinterpret_cast<uint8_t*>(ws + plan.lay.species); }
  int32_t* d_epi() const { return reinterpret_cast<int32_t*>(ws + plan.lay.epi); }
  int32_t* d_coef() const { return reinterpret_cast<int32_t*>(ws + plan.lay.coef); }
  int32_t* d_gtable() const { return reinterpret_cast<int32_t*>(ws + plan.lay.gtable); }
  uint32_t* d_fcc_lut() const { return reinterpret_cast<uint32_t*>(ws + plan.lay.fcc_lut); }
  int32_t* d_fcc_corr() const { return reinterpret_cast<int32_t*>(ws + plan.lay.fcc_corr); }
  int32_t* d_quad() const { return reinterpret_cast<int32_t*>(ws + plan.lay.quad); }
  LocalUEntry* d_utab() const { return reinterpret_cast<LocalUEntry*>(ws + plan.lay.utab); }
  int* d_ucount() const { return reinterpret_cast<int*>(ws + plan.lay.ucount); }
  int lattice_type = 0;
  uint32_t* d_accept() const { return reinterpret_cast<uint32_t*>(ws + plan.lay.accept); }
  uint32_t* d_filter() const { return reinterpret_cast<uint32_t*>(ws + plan.lay.filter); }
  long long* d_trace() const { return reinterpret_cast<long long*>(ws + plan.lay.trace); }
  DevState* d_state() const { return reinterpret_cast<DevState*>(ws + plan.lay.state); }
  unsigned long long* d_counts() const { return reinterpret_cast<unsigned long long*>(ws + plan.lay.counts); }
  unsigned* d_progress() const { return reinterpret_cast<unsigned*>(ws + plan.lay.progress); }
};

namespace {

#define SMCX_CUDA(h, call)                                                        \
  do {                                                                            \
    cudaError_t e_ = (call);                                                      \
    if (e_ != cudaSuccess) {                                                      \
      (h)->err = std::string(#call) + ": " + cudaGetErrorString(e_);              \
      return SMCX_E_CUDA;                                                         \
    }                                                                             \
  } while (0)

// Every entry point that touches CUDA runs on the handle's device whatever device the caller has made current
// (a process that drives several GPUs switches devices between calls) and restores the caller's device on return.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int device) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    else cudaGetLastError();
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// `Store` = accessor of the handle's device storage (lattice_kernels.cuh) inside the statement(s) given
#define SMCX_STORE_DISPATCH(P, ...)                                                              \
  do {                                                                                           \
    if ((P).storage == SMCX_STORAGE_U8) { using Store = StoreU8; __VA_ARGS__; }                  \
    else if ((P).storage == SMCX_STORAGE_2BIT) { using Store = Store2; __VA_ARGS__; }            \
    else if ((P).G.B == 2) { using Store = Store4<2>; __VA_ARGS__; }                             \
    else { using Store = Store4<4>; __VA_ARGS__; }                                               \
  } while (0)

int grid_for(const smcx* h, long long work_items, int block) {
  const long long want = (work_items + block - 1) / block;
  const long long cap = (long long)h->sm_count * 16;
  return (int)std::max(1ll, std::min(want, cap));
}

int launch_init(smcx* h) {
  const Plan& P = h->plan;
  int hh = 1;
  while ((1ull << (2 * hh)) < (unsigned long long)P.n_global) ++hh;
  const int grid = grid_for(h, (P.n_sites + 15) / 16, 256);
  SMCX_STORE_DISPATCH(P, init_species_kernel<Store><<<grid, 256, 0, h->stream>>>(h->d_species(), P.n_sites, P.G.n_species, hh,
                                                                                   P.G.key0, P.G.key1, (long long)P.z_base * P.layer_sites,
                                                                                   P.n_global));
  h->launches++;
  SMCX_CUDA(h, cudaGetLastError());
  return SMCX_OK;
}

// Runs the pair-count reduction and leaves M[s][x][y] (positive-half counts) in host_M.
int run_pair_counts(smcx* h, std::vector<unsigned long long>& host_M) {
  const Plan& P = h->plan;
  Geom G = P.G;
  if (P.window) {   // the bonds of the layers the slab owns under the current origin
    G.pc_z0 = G.H + h->win_oz;
    G.pc_z1 = G.pc_z0 + P.row_count * G.w;
  }
  const int n_hist = G.n_shells * G.n_species * G.n_species;
  zero_u64_kernel<<<1, 256, 0, h->stream>>>(h->d_counts(), n_hist);
  h->launches++;
  const long long n_conv = (long long)G.Lx * G.Ly * (G.pc_z1 - G.pc_z0);
  const int grid = grid_for(h, n_conv, 256);
  const size_t sm = (size_t)n_hist * sizeof(unsigned);
  if (P.storage == SMCX_STORAGE_2BIT && G.lattice == SMCX_BCC && G.n_shells == 2) {
    // bit-parallel reduction: one thread per packed word (16 sites)
    const int gridw = grid_for(h, n_conv / 8, 256);
    pair_count_bcc2_kernel<<<gridw, 256, 0, h->stream>>>(G, reinterpret_cast<const uint32_t*>(h->d_species()), h->d_counts());
  } else if (G.B == 2) {
    SMCX_STORE_DISPATCH(P, pair_count_kernel<Store, 2><<<grid, 256, sm, h->stream>>>(G, h->d_species(), h->d_counts()));
  } else {
    SMCX_STORE_DISPATCH(P, pair_count_kernel<Store, 4><<<grid, 256, sm, h->stream>>>(G, h->d_species(), h->d_counts()));
  }
  h->launches++;
  SMCX_CUDA(h, cudaGetLastError());
  host_M.assign((size_t)n_hist, 0ull);
  SMCX_CUDA(h, cudaMemcpyAsync(host_M.data(), h->d_counts(), (size_t)n_hist * sizeof(unsigned long long),
                               cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return SMCX_OK;
}

long long energy_from_counts(const smcx* h, const std::vector<unsigned long long>& M) {
  const Geom& G = h->plan.G;
  const int n = G.n_species;
  long long E = 0;
  for (int s = 0; s < G.n_shells; ++s)
    for (int a = 0; a < n; ++a)
      for (int b = 0; b < n; ++b)
        E += (long long)h->epi[(size_t)(s * n + a) * n + b] * (long long)M[(size_t)(s * n + a) * n + b];
  return E;
}

// SMCX_MODEL_LOCAL: H = sum of the local energies, by local_energy_kernel.
int run_local_energy(smcx* h, long long* E) {
  const Plan& P = h->plan;
  Geom G = P.G;
  if (P.window) {   // the local energies of the sites of the layers the slab owns under the current origin
    G.pc_z0 = G.H + h->win_oz;
    G.pc_z1 = G.pc_z0 + P.row_count * G.w;
  }
  zero_u64_kernel<<<1, 32, 0, h->stream>>>(h->d_counts(), 1);
  const size_t sm = ((size_t)G.n_shells * G.n_species * G.n_species * (1 + G.n_species)) * sizeof(int32_t);
  const int grid = grid_for(h, P.layer_sites * (G.pc_z1 - G.pc_z0), 256);
  if (G.B == 2) local_energy_kernel<2><<<grid, 256, sm, h->stream>>>(G, h->d_species(), h->d_epi(), h->d_quad(), h->d_counts());
  else local_energy_kernel<4><<<grid, 256, sm, h->stream>>>(G, h->d_species(), h->d_epi(), h->d_quad(), h->d_counts());
  h->launches += 2;
  SMCX_CUDA(h, cudaGetLastError());
  unsigned long long v = 0;
  SMCX_CUDA(h, cudaMemcpyAsync(&v, h->d_counts(), sizeof(v), cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  *E = (long long)v;
  return SMCX_OK;
}

// Recompute H from the lattice and store it as the running energy.
int reset_running_energy(smcx* h) {
  long long E = 0;
  if (h->plan.model == SMCX_MODEL_LOCAL) {
    const int rc = run_local_energy(h, &E);
    if (rc != SMCX_OK) return rc;
  } else {
    std::vector<unsigned long long> M;
    const int rc = run_pair_counts(h, M);
    if (rc != SMCX_OK) return rc;
    E = energy_from_counts(h, M);
  }
  SMCX_CUDA(h, cudaMemcpyAsync(&h->d_state()->e_run, &E, sizeof(E), cudaMemcpyHostToDevice, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return SMCX_OK;
}

int upload_table(smcx* h, const uint32_t* accept, int len) {
  if (!accept || len < 1 || len > kAcceptCapacity) return SMCX_E_BAD_TABLE;
  const int slot = h->staging_next;
  h->staging_next = (slot + 1) % kStagingSlots;
  SMCX_CUDA(h, cudaEventSynchronize(h->staging_ev[slot]));
  std::memcpy(h->staging[slot], accept, (size_t)len * sizeof(uint32_t));
  h->staging[slot][len] = 0u;    // dE >= len is a rejection (S5): kernels that clamp dE to len read this entry
  {
    // the table is input data and need not be monotone: from which entry on does T[k] bound everything behind it
    // (what sweep_fcc_thread<2> relies on when it holds only the head of T in shared memory)
    int m = len;
    uint32_t run_max = 0u;
    while (m > 0 && accept[m - 1] >= run_max) { run_max = accept[m - 1]; --m; }
    h->plan.accept_tail_from = std::max(m, h->plan.accept_tail_floor);
  }
  SMCX_CUDA(h, cudaMemcpyAsync(h->d_accept(), h->staging[slot], ((size_t)len + 1) * sizeof(uint32_t),
                               cudaMemcpyHostToDevice, h->stream));
  h->plan.G.filter_E = -1;
  h->plan.G.filter_nq = 0;
  if (uses_filter(h->plan)) {
    uint32_t* filt = h->staging[slot] + kAcceptCapacity + 1;
    int nq = 0;
    const int E = build_accept_filter(accept, len, filt, &nq);
    if (E >= 0) {
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_filter(), filt, (size_t)kFilterWords * sizeof(uint32_t),
                                   cudaMemcpyHostToDevice, h->stream));
      h->plan.G.filter_E = E;
      h->plan.G.filter_nq = nq;
    }
  }
  SMCX_CUDA(h, cudaEventRecord(h->staging_ev[slot], h->stream));
  h->plan.G.accept_len = len;
  h->params_epoch++;
  return SMCX_OK;
}

int ensure_bounce(smcx* h) {
  const size_t chunk = (size_t)std::min<long long>(kChunkSites, h->plan.n_sites);
  for (int k = 0; k < 2; ++k) {
    if (!h->bounce[k]) SMCX_CUDA(h, cudaMalloc(&h->bounce[k], chunk));
    if (!h->bounce_full[k]) SMCX_CUDA(h, cudaEventCreateWithFlags(&h->bounce_full[k], cudaEventDisableTiming));
    if (!h->bounce_free[k]) SMCX_CUDA(h, cudaEventCreateWithFlags(&h->bounce_free[k], cudaEventDisableTiming));
  }
  if (!h->copy_stream) SMCX_CUDA(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  return SMCX_OK;
}

// One colour pass with the geometry G: the handle's own (smcx_sweep), or a copy of it restricted to some of the
// link-cell rows of a slab (smcx_domain_pass).
int launch_colour_pass(smcx* h, const Geom& G, int colour) {
  const Plan& P = h->plan;
  if (P.kernel == SMCX_KERNEL_THREAD_PERSISTENT) {
    const int warps = persist_warps_for(G.accept_len);
    if (warps > 0) {
      const int rc = launch_thread_persistent(G, reinterpret_cast<uint32_t*>(h->d_species()), h->d_coef(), P.coef_packed,
                                              h->d_accept(), h->d_state(), colour, warps, h->sm_count, h->stream);
      h->launches++;
      if (rc != 0) { h->err = "persistent thread-per-cell launch failed"; return SMCX_E_CUDA; }
      return SMCX_OK;
    }
  }
  if (is_thread_kernel(P.kernel)) {
    const int rc = launch_thread_per_cell(G, reinterpret_cast<uint32_t*>(h->d_species()), h->d_coef(), h->d_accept(),
                                          h->d_filter(), h->d_state(), colour, h->stream);
    h->launches++;
    if (rc != 0) { h->err = "thread-per-cell launch failed"; return SMCX_E_CUDA; }
    return SMCX_OK;
  }
  if (P.kernel == SMCX_KERNEL_FCC_THREAD) {
    const int rc = launch_fcc_thread(G, P.fcc_tables, reinterpret_cast<uint32_t*>(h->d_species()), h->d_fcc_lut(), h->d_fcc_corr(),
                                     P.fcc_rep, h->d_accept(), h->d_filter(), h->d_state(), colour, h->sm_count, P.accept_tail_from, h->stream);
    h->launches++;
    if (rc != 0) { h->err = "packed FCC thread-per-cell launch failed"; return SMCX_E_CUDA; }
    return SMCX_OK;
  }
  if (P.kernel == SMCX_KERNEL_BCC4_THREAD) {
    const int rc = launch_bcc4_thread(G, P.bcc4_tables, reinterpret_cast<uint32_t*>(h->d_species()), h->d_fcc_lut(), h->d_fcc_corr(),
                                      P.fcc_rep, h->d_accept(), h->d_filter(), h->d_state(), colour, h->sm_count, P.accept_tail_from, h->stream);
    h->launches++;
    if (rc != 0) { h->err = "packed BCC (4-bit) thread-per-cell launch failed"; return SMCX_E_CUDA; }
    return SMCX_OK;
  }
  if (P.kernel == SMCX_KERNEL_LOCAL_WARP) {
    const LocalTables T{h->d_epi(), h->d_quad(), h->d_utab(), h->d_ucount(), P.local_umax};
    const size_t sm = local_smem_bytes(G, P.local_umax);
    const unsigned grid = (G.cells_per_colour + kLocalWarps - 1) / kLocalWarps;
    int zmax = 0;
    for (int s2 = 0, m2 = 0; s2 < G.n_shells; ++s2) {
      int z = 0;
      while (m2 < G.ZT && (int)G.shell_of[m2] == s2) { ++m2; ++z; }
      zmax = std::max(zmax, z);
    }
    const bool narrow = G.n_species <= kLocalNarrowSpecies && zmax <= kLocalNarrowMaxZ;   // 5-bit count fields in a 32-bit word
    if (G.B == 2 && narrow) sweep_local_warp<2, true><<<grid, kLocalWarps * 32, sm, h->stream>>>(G, h->d_species(), T, h->d_accept(), h->d_state(), colour);
    else if (G.B == 2) sweep_local_warp<2, false><<<grid, kLocalWarps * 32, sm, h->stream>>>(G, h->d_species(), T, h->d_accept(), h->d_state(), colour);
    else if (narrow) sweep_local_warp<4, true><<<grid, kLocalWarps * 32, sm, h->stream>>>(G, h->d_species(), T, h->d_accept(), h->d_state(), colour);
    else sweep_local_warp<4, false><<<grid, kLocalWarps * 32, sm, h->stream>>>(G, h->d_species(), T, h->d_accept(), h->d_state(), colour);
    h->launches++;
    SMCX_CUDA(h, cudaGetLastError());
    return SMCX_OK;
  }
  if (P.kernel == SMCX_KERNEL_GROUP_PER_CELL) {
    launch_group_per_cell(G, P.group_lanes, P.group_warps, h->d_species(), h->d_gtable(), h->d_accept(), h->d_filter(), h->d_state(), colour, h->stream);
    h->launches++;
    SMCX_CUDA(h, cudaGetLastError());
    return SMCX_OK;
  }
  const int n2 = G.n_species * G.n_species;
  const int tables = (G.n_shells * n2 * 4 + G.B * G.ZT * 2 + G.ZT + 15) & ~15;
  const int tile = (G.TW * G.TW * G.TW * G.B + 15) & ~15;
  const size_t sm = (size_t)tables + (size_t)kWarpsPerBlock * tile;
  const unsigned grid = (G.cells_per_colour + kWarpsPerBlock - 1) / kWarpsPerBlock;
  if (G.B == 2)
    sweep_warp_per_cell<2><<<grid, kWarpsPerBlock * 32, sm, h->stream>>>(G, h->d_species(), h->d_epi(), h->d_accept(), h->d_state(), colour);
  else
    sweep_warp_per_cell<4><<<grid, kWarpsPerBlock * 32, sm, h->stream>>>(G, h->d_species(), h->d_epi(), h->d_accept(), h->d_state(), colour);
  h->launches++;
  return SMCX_OK;
}

// One sweep on h->stream: 8 colour passes and the trace/counter epilogue.
int enqueue_sweep(smcx* h) {
  static const char* const kPassName[8] = {"smcx colour 0", "smcx colour 1", "smcx colour 2", "smcx colour 3",
                                           "smcx colour 4", "smcx colour 5", "smcx colour 6", "smcx colour 7"};
  nvtxRangePushA("smcx sweep");
  if (h->whole_sweep && persist_warps_for(h->plan.G.accept_len) > 0) {
    // the eight passes pipelined in one launch (+ the launch that advances its sweep count)
    const Plan& P = h->plan;
    const int rc = launch_whole_sweep(P.G, reinterpret_cast<uint32_t*>(h->d_species()), h->d_coef(), P.coef_packed, h->d_accept(),
                                      h->d_state(), h->d_progress(), persist_warps_for(P.G.accept_len), h->sm_count, h->stream);
    h->launches += 2;
    if (rc != 0) { h->err = "whole-sweep launch failed"; nvtxRangePop(); return SMCX_E_CUDA; }
    sweep_epilogue<<<1, 1, 0, h->stream>>>(h->d_state(), h->d_trace(), h->plan.G.trace_capacity);
    h->launches++;
    nvtxRangePop();
    return SMCX_OK;
  }
  for (int colour = 0; colour < 8; ++colour) {
    nvtxRangePushA(kPassName[colour]);
    const int rc = launch_colour_pass(h, h->plan.G, colour);
    nvtxRangePop();
    if (rc != SMCX_OK) { nvtxRangePop(); return rc; }
  }
  sweep_epilogue<<<1, 1, 0, h->stream>>>(h->d_state(), h->d_trace(), h->plan.G.trace_capacity);
  h->launches++;
  nvtxRangePop();
  return SMCX_OK;
}

}  // namespace

extern "C" {

const char* smcx_version(void) { return "smcx-b200 0.1 (sm_100a)"; }

const char* smcx_strerror(int code) {
  switch (code) {
    case SMCX_OK: return "ok";
    case SMCX_E_NULL_ARG: return "null argument";
    case SMCX_E_BAD_LATTICE: return "lattice must be SMCX_BCC or SMCX_FCC";
    case SMCX_E_BAD_DIMS: return "dims must be positive, divisible by 2*link_cell, at least link_cell+2*halo, and small enough";
    case SMCX_E_BAD_SPECIES: return "n_species must be in 2..16";
    case SMCX_E_BAD_SHELLS: return "n_shells must be in 1..5";
    case SMCX_E_EPI_NOT_SYMMETRIC: return "EPI table is not symmetric";
    case SMCX_E_LINK_CELL_TOO_SMALL: return "link cell violates 2w >= 2 r0 + R (or is out of range)";
    case SMCX_E_BAD_TABLE: return "acceptance table missing, empty or too long";
    case SMCX_E_BAD_STATE: return "species value >= n_species";
    case SMCX_E_NO_MEMORY: return "out of memory or workspace too small";
    case SMCX_E_CUDA: return "CUDA error (see smcx_last_error)";
    case SMCX_E_UNSUPPORTED: return "storage/kernel choice not valid for these parameters";
    case SMCX_E_RANGE: return "range not available";
    case SMCX_E_EPI_RANGE: return "EPI magnitudes too large: the int32 energy change of a trial could overflow";
    case SMCX_E_STATIC_SCRATCH: return "n_shells * n_species^2 exceeds SMCX_STATIC_PAIR_COUNTS_MAX (1024), the size of the library's static device scratch";
    default: return "unknown error";
  }
}

const char* smcx_last_error(smcx_t* h) { return h ? h->err.c_str() : "null handle"; }

int smcx_workspace_bytes(const smcx_params_t* p, size_t* bytes) {
  if (!p || !bytes) return SMCX_E_NULL_ARG;
  Plan plan;
  const int rc = make_plan(p, &plan);
  if (rc != SMCX_OK) return rc;
  *bytes = plan.lay.total;
  return SMCX_OK;
}

int smcx_create(smcx_t** out, const smcx_params_t* p) {
  if (!out || !p) return SMCX_E_NULL_ARG;
  smcx* h = new (std::nothrow) smcx();
  if (!h) return SMCX_E_NO_MEMORY;
  int rc = make_plan(p, &h->plan);
  if (rc != SMCX_OK) { delete h; return rc; }
  h->device = p->device;
  h->stream = reinterpret_cast<cudaStream_t>(p->stream);
  h->kT_units = p->kT_units;
  const int n = p->n_species;
  h->epi.assign(p->epi, p->epi + (size_t)p->n_shells * n * n);

  auto fail = [&](int code) { smcx_destroy(h); return code; };
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev <= 0 || p->device < 0 || p->device >= n_dev) {
    cudaGetLastError();
    return fail(SMCX_E_CUDA);
  }
  DeviceGuard on_device(p->device);     // the caller's current device is restored on return
  int now = -1;
  if (cudaGetDevice(&now) != cudaSuccess || now != p->device) return fail(SMCX_E_CUDA);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) return fail(SMCX_E_CUDA);
  h->sm_count = prop.multiProcessorCount;

  if (p->d_workspace) {
    if (p->workspace_bytes < h->plan.lay.total) return fail(SMCX_E_NO_MEMORY);
    h->ws = reinterpret_cast<char*>(p->d_workspace);
  } else {
    void* ws = nullptr;
    if (cudaMalloc(&ws, h->plan.lay.total) != cudaSuccess) { cudaGetLastError(); return fail(SMCX_E_NO_MEMORY); }
    h->ws = reinterpret_cast<char*>(ws);
    h->owns_ws = true;
  }
  h->staging_cap = ((size_t)kAcceptCapacity + 1 + kFilterWords) * sizeof(uint32_t);
  for (int s = 0; s < kStagingSlots; ++s) {
    if (cudaMallocHost(reinterpret_cast<void**>(&h->staging[s]), h->staging_cap) != cudaSuccess) return fail(SMCX_E_NO_MEMORY);
    if (cudaEventCreateWithFlags(&h->staging_ev[s], cudaEventDisableTiming) != cudaSuccess) return fail(SMCX_E_CUDA);
  }
  if (configure_thread_per_cell() != 0) return fail(SMCX_E_CUDA);
  if (h->plan.kernel == SMCX_KERNEL_THREAD_PERSISTENT && configure_whole_sweep() != 0) return fail(SMCX_E_CUDA);
  cudaFuncSetAttribute(whole_sweep_epoch, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (h->plan.kernel == SMCX_KERNEL_FCC_THREAD && configure_fcc_thread(h->plan.fcc_rep) != 0) return fail(SMCX_E_CUDA);
  if (h->plan.kernel == SMCX_KERNEL_BCC4_THREAD && configure_bcc4_thread(h->plan.fcc_rep) != 0) return fail(SMCX_E_CUDA);
  // every kernel of a sweep prefers the largest shared-memory carve-out: an SM whose carve-out must
  // change drains first, which serialises lattices that run concurrently (replica ensembles:
  // measured 45 us instead of 28 us per colour pass when the one-thread epilogue asked for the default)
  cudaFuncSetAttribute(sweep_epilogue, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(replica_exchange_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(replica_apply_tables_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_thread_per_cell<true>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_thread_per_cell<false>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_warp_per_cell<2>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaFuncSetAttribute(sweep_warp_per_cell<4>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  cudaGetLastError();
  if (cudaStreamCreateWithFlags(&h->capture_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); h->capture_stream = nullptr; }
  {
    const Geom& G = h->plan.G;
    const int n2 = G.n_species * G.n_species;
    const size_t sm = (size_t)((G.n_shells * n2 * 4 + G.B * G.ZT * 2 + G.ZT + 15) & ~15) +
                      (size_t)kWarpsPerBlock * ((G.TW * G.TW * G.TW * G.B + 15) & ~15);
    if (h->plan.kernel == SMCX_KERNEL_GROUP_PER_CELL) {
      const cudaError_t e = configure_group_per_cell(G, h->plan.group_lanes, h->plan.group_warps);
      if (e != cudaSuccess) { h->err = cudaGetErrorString(e); return fail(SMCX_E_CUDA); }
    }
    if (h->plan.kernel == SMCX_KERNEL_LOCAL_WARP) {
      const int lsm = (int)local_smem_bytes(G, h->plan.local_umax);
      cudaError_t e = cudaFuncSetAttribute(sweep_local_warp<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lsm);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_local_warp<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, lsm);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_local_warp<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lsm);
      if (e == cudaSuccess) e = cudaFuncSetAttribute(sweep_local_warp<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, lsm);
      if (e != cudaSuccess) { h->err = cudaGetErrorString(e); return fail(SMCX_E_CUDA); }
    }
    if (h->plan.kernel == SMCX_KERNEL_WARP_PER_CELL) {
      if (sm > 227 * 1024) return fail(SMCX_E_LINK_CELL_TOO_SMALL);
      cudaError_t e = G.B == 2
          ? cudaFuncSetAttribute(sweep_warp_per_cell<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm)
          : cudaFuncSetAttribute(sweep_warp_per_cell<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      if (e != cudaSuccess) { h->err = cudaGetErrorString(e); return fail(SMCX_E_CUDA); }
    }
  }

  rc = [&]() -> int {
    DevState zero{};
    SMCX_CUDA(h, cudaMemcpyAsync(h->d_state(), &zero, sizeof(zero), cudaMemcpyHostToDevice, h->stream));
    SMCX_CUDA(h, cudaMemcpyAsync(h->d_epi(), h->epi.data(), h->epi.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    int32_t coef[16 * (kCoefInts + 4)] = {0};   // 32-bit rows, then the packed 16-bit rows
    if (is_thread_kernel(h->plan.kernel)) {
      build_thread_coefficients(h->epi.data(), h->plan.G.n_species, coef);
      pack_thread_coefficients(coef, coef + 16 * kCoefInts);
    }
    SMCX_CUDA(h, cudaMemcpyAsync(h->d_coef(), coef, sizeof(coef), cudaMemcpyHostToDevice, h->stream));
    std::vector<int32_t> gtab;
    if (h->plan.kernel == SMCX_KERNEL_GROUP_PER_CELL) {
      group_build_table(h->plan.G, h->plan.group_lanes, h->epi.data(), gtab);
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_gtable(), gtab.data(), gtab.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    }
    std::vector<LocalUEntry> utab;
    std::vector<int> ucount;
    if (h->plan.model == SMCX_MODEL_LOCAL) {
      build_local_utable(h->plan, p->lattice, utab, ucount);
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_quad(), p->local_quad, (size_t)p->n_shells * n * n * n * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_utab(), utab.data(), utab.size() * sizeof(LocalUEntry), cudaMemcpyHostToDevice, h->stream));
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_ucount(), ucount.data(), ucount.size() * sizeof(int), cudaMemcpyHostToDevice, h->stream));
    }
    std::vector<uint32_t> flut;
    std::vector<int32_t> fcorr;
    if (h->plan.kernel == SMCX_KERNEL_FCC_THREAD || h->plan.kernel == SMCX_KERNEL_BCC4_THREAD) {
      fcc_build_lut(h->epi.data(), h->plan.G.n_species, h->plan.G.n_shells, h->plan.fcc_rep, flut, fcorr);
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_fcc_lut(), flut.data(), flut.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, h->stream));
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_fcc_corr(), fcorr.data(), fcorr.size() * sizeof(int32_t), cudaMemcpyHostToDevice, h->stream));
    }
    SMCX_CUDA(h, cudaMemsetAsync(h->d_trace(), 0, (size_t)h->plan.G.trace_capacity * sizeof(long long), h->stream));
    SMCX_CUDA(h, cudaMemsetAsync(h->d_progress(), 0, whole_sweep_progress_words(h->plan.G) * sizeof(unsigned), h->stream));
    SMCX_CUDA(h, cudaStreamSynchronize(h->stream));  // &zero and epi must stay valid until copied
    int r = upload_table(h, p->accept, p->accept_len);
    if (r != SMCX_OK) return r;
    r = launch_init(h);
    if (r != SMCX_OK) return r;
    return reset_running_energy(h);
  }();
  if (rc != SMCX_OK) return fail(rc);
  // The whole-sweep launch (its warps wait for other blocks of the same launch) goes to one handle per process at a
  // time: an undivided lattice on the persistent kernel with at most kWholeSweepMaxCells link cells per colour (beyond
  // that a pass is many rounds of batches, the colour boundaries cost little and the bookkeeping more: measured).  Two
  // such launches at once could each hold SMs while waiting for blocks of their own that find none free.
  if (h->plan.kernel == SMCX_KERNEL_THREAD_PERSISTENT && !h->plan.window && h->plan.G.iz_first == 0 &&
      h->plan.n_cells / 8 <= kWholeSweepMaxCells) {
    smcx* none = nullptr;
    h->whole_sweep = g_whole_sweep_owner.compare_exchange_strong(none, h);
  }
  *out = h;
  return SMCX_OK;
}

void smcx_destroy(smcx_t* h) {
  if (!h) return;
  {
    smcx* me = h;
    g_whole_sweep_owner.compare_exchange_strong(me, nullptr);
  }
  DeviceGuard on_device(h->device);
  if (h->stream || h->ws) cudaStreamSynchronize(h->stream);
  for (int s = 0; s < kStagingSlots; ++s) {
    if (h->staging[s]) cudaFreeHost(h->staging[s]);
    if (h->staging_ev[s]) cudaEventDestroy(h->staging_ev[s]);
  }
  if (h->sweep_graph) cudaGraphExecDestroy(h->sweep_graph);
  if (h->capture_stream) cudaStreamDestroy(h->capture_stream);
  for (int k = 0; k < 2; ++k) {
    if (h->bounce[k]) cudaFree(h->bounce[k]);
    if (h->bounce_full[k]) cudaEventDestroy(h->bounce_full[k]);
    if (h->bounce_free[k]) cudaEventDestroy(h->bounce_free[k]);
  }
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->owns_ws && h->ws) cudaFree(h->ws);
  cudaGetLastError();
  delete h;
}

// Did a validation kernel flag a value >= n_species since clear_bad_state()?  Synchronises.
static int clear_bad_state(smcx* h) {
  SMCX_CUDA(h, cudaMemsetAsync(&h->d_state()->bad_state, 0, sizeof(unsigned long long), h->stream));
  return SMCX_OK;
}
static int check_bad_state(smcx* h) {
  unsigned long long bad = 0;
  SMCX_CUDA(h, cudaMemcpyAsync(&bad, &h->d_state()->bad_state, sizeof(bad), cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return bad ? SMCX_E_BAD_STATE : SMCX_OK;
}

// Runs of sites that are contiguous both in a host array of the whole lattice (site-id order) and in the handle's
// storage: the whole lattice is one run; the storage layers [l0, l1) of a slab window are one or two (the window may
// wrap around the periodic lattice).
struct SiteRun { long long host_first, local_first, count; };
static std::vector<SiteRun> site_runs(const smcx* h, int l0, int l1) {
  const Plan& P = h->plan;
  std::vector<SiteRun> runs;
  if (!P.window) { runs.push_back({0, 0, P.n_sites}); return runs; }
  const long long ls = P.layer_sites;
  const int g0 = (P.z_base + l0) % P.Lz_global;
  const int first = std::min(l1 - l0, P.Lz_global - g0);
  runs.push_back({g0 * ls, l0 * ls, first * ls});
  if (first < l1 - l0) runs.push_back({0, (l0 + first) * ls, (l1 - l0 - first) * ls});
  return runs;
}

int smcx_set_species_device(smcx_t* h, const void* d_src) {
  if (!h || !d_src) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  const uint8_t* src = reinterpret_cast<const uint8_t*>(d_src);
  int rc = clear_bad_state(h);
  if (rc != SMCX_OK) return rc;
  // validated before anything is written: on SMCX_E_BAD_STATE the lattice is unchanged
  validate_u8_kernel<<<grid_for(h, P.n_sites, 256), 256, 0, h->stream>>>(src, P.n_sites, P.G.n_species, h->d_state());
  h->launches++;
  rc = check_bad_state(h);
  if (rc != SMCX_OK) return rc;
  if (P.storage == SMCX_STORAGE_U8) {
    SMCX_CUDA(h, cudaMemcpyAsync(h->d_species(), src, (size_t)P.n_sites, cudaMemcpyDeviceToDevice, h->stream));
  } else {
    SMCX_STORE_DISPATCH(P, pack_kernel<Store><<<grid_for(h, (P.n_sites + 15) / 16, 256), 256, 0, h->stream>>>(
                               src, h->d_species(), 0, P.n_sites, P.G.n_species, h->d_state()));
    h->launches++;
    SMCX_CUDA(h, cudaGetLastError());
  }
  return reset_running_energy(h);
}

// Host upload.  The values are validated on the device while they are packed (no pass over the array on the
// host): on SMCX_E_BAD_STATE the lattice has been overwritten with the low bits of the rejected array and must
// be set again.  Packed storage: chunks of 2^26 sites through two device bounce buffers, the copy of chunk k + 1
// on the copy stream overlapping the packing of chunk k.
int smcx_set_species(smcx_t* h, const uint8_t* host_src) {
  if (!h || !host_src) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  int rc = clear_bad_state(h);
  if (rc != SMCX_OK) return rc;
  // a slab window takes its layers (all of them, ghost layers included) out of the array of the whole lattice
  const std::vector<SiteRun> runs = site_runs(h, 0, P.G.Lz);
  if (P.storage == SMCX_STORAGE_U8) {
    for (const SiteRun& r : runs)
      SMCX_CUDA(h, cudaMemcpyAsync(h->d_species() + r.local_first, host_src + r.host_first, (size_t)r.count, cudaMemcpyHostToDevice, h->stream));
    validate_u8_kernel<<<grid_for(h, P.n_sites, 256), 256, 0, h->stream>>>(h->d_species(), P.n_sites, P.G.n_species, h->d_state());
    h->launches++;
  } else {
    rc = ensure_bounce(h);
    if (rc != SMCX_OK) return rc;
    SMCX_CUDA(h, cudaEventRecord(h->bounce_free[0], h->stream));   // the bounce buffers are free once earlier work is done
    SMCX_CUDA(h, cudaEventRecord(h->bounce_free[1], h->stream));
    int k = 0;
    for (const SiteRun& r : runs)
      for (long long first = 0; first < r.count; first += kChunkSites, k ^= 1) {
        const long long cnt = std::min(kChunkSites, r.count - first);
        SMCX_CUDA(h, cudaStreamWaitEvent(h->copy_stream, h->bounce_free[k], 0));
        SMCX_CUDA(h, cudaMemcpyAsync(h->bounce[k], host_src + r.host_first + first, (size_t)cnt, cudaMemcpyHostToDevice, h->copy_stream));
        SMCX_CUDA(h, cudaEventRecord(h->bounce_full[k], h->copy_stream));
        SMCX_CUDA(h, cudaStreamWaitEvent(h->stream, h->bounce_full[k], 0));
        SMCX_STORE_DISPATCH(P, pack_kernel<Store><<<grid_for(h, (cnt + 15) / 16, 256), 256, 0, h->stream>>>(
                                   h->bounce[k], h->d_species(), r.local_first + first, cnt, P.G.n_species, h->d_state()));
        h->launches++;
        SMCX_CUDA(h, cudaGetLastError());
        SMCX_CUDA(h, cudaEventRecord(h->bounce_free[k], h->stream));
      }
  }
  rc = check_bad_state(h);
  if (rc != SMCX_OK) return rc;
  h->win_oz = 0;   // slab window: every layer is valid again
  return reset_running_energy(h);
}

int smcx_storage_bytes(smcx_t* h, size_t* bytes) {
  if (!h || !bytes) return SMCX_E_NULL_ARG;
  *bytes = storage_bytes(h->plan.storage, h->plan.n_sites);
  return SMCX_OK;
}

int smcx_species_packed(smcx_t* h, void* host_dst) {
  if (!h || !host_dst) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;
  DeviceGuard on_device(h->device);
  SMCX_CUDA(h, cudaMemcpyAsync(host_dst, h->d_species(), storage_bytes(h->plan.storage, h->plan.n_sites),
                               cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return SMCX_OK;
}

int smcx_set_species_packed(smcx_t* h, const void* host_src) {
  if (!h || !host_src) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  int rc = clear_bad_state(h);
  if (rc != SMCX_OK) return rc;
  SMCX_CUDA(h, cudaMemcpyAsync(h->d_species(), host_src, storage_bytes(P.storage, P.n_sites), cudaMemcpyHostToDevice, h->stream));
  SMCX_STORE_DISPATCH(P, validate_storage_kernel<Store><<<grid_for(h, P.n_sites, 256), 256, 0, h->stream>>>(
                             h->d_species(), P.n_sites, P.G.n_species, h->d_state()));
  h->launches++;
  rc = check_bad_state(h);
  if (rc != SMCX_OK) return rc;
  return reset_running_energy(h);
}

int smcx_init_composition(smcx_t* h, const int64_t* counts) {
  if (!h || !counts) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  CompositionCum C{};
  long long sum = 0;
  for (int p = 0; p < P.G.n_species; ++p) {
    if (counts[p] < 0) return SMCX_E_BAD_STATE;
    sum += counts[p];
    C.cum[p] = sum;
  }
  if (sum != P.n_global) return SMCX_E_BAD_STATE;
  int hh = 1;
  while ((1ull << (2 * hh)) < (unsigned long long)P.n_global) ++hh;
  const int grid = grid_for(h, (P.n_sites + 15) / 16, 256);
  SMCX_STORE_DISPATCH(P, init_composition_kernel<Store><<<grid, 256, 0, h->stream>>>(h->d_species(), P.n_sites, P.G.n_species, hh,
                                                                                       P.G.key0, P.G.key1, C,
                                                                                       (long long)P.z_base * P.layer_sites, P.n_global));
  if (P.window) h->win_oz = 0;   // every layer of the window is valid again
  h->launches++;
  SMCX_CUDA(h, cudaGetLastError());
  return reset_running_energy(h);
}

int smcx_set_sweep_counter(smcx_t* h, int64_t t) {
  if (!h) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  if (t < 0 || t > 0xffffffffll) return SMCX_E_RANGE;
  const unsigned long long v = (unsigned long long)t;
  SMCX_CUDA(h, cudaMemcpyAsync(&h->d_state()->sweep, &v, sizeof(v), cudaMemcpyHostToDevice, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  h->sweeps_enqueued = t;
  h->trace_first = t;
  return SMCX_OK;
}

int smcx_set_temperature(smcx_t* h, int32_t kT_units, const uint32_t* accept, int32_t accept_len) {
  if (!h) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const int rc = upload_table(h, accept, accept_len);
  if (rc == SMCX_OK) h->kT_units = kT_units;
  return rc;
}

int smcx_sweep(smcx_t* h, int64_t n) {
  if (!h) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;   // a slab is stepped pass by pass through smcx_domain_*
  DeviceGuard on_device(h->device);
  if (n < 0 || h->sweeps_enqueued + n > 0xffffffffll) return SMCX_E_RANGE;  // t is a 32-bit counter word
  // Runs of sweeps at fixed parameters are replayed from a captured graph of one sweep (the kernels
  // read the sweep counter from device memory, so the same graph serves every sweep).
  if (n >= 3 && h->graphs_ok && h->capture_stream) {
    if (h->graph_epoch != h->params_epoch) {
      if (h->sweep_graph) { cudaGraphExecDestroy(h->sweep_graph); h->sweep_graph = nullptr; }
      cudaGraph_t graph = nullptr;
      cudaStream_t user = h->stream;
      bool ok = cudaStreamBeginCapture(h->capture_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
      if (ok) {
        const long long launches_before = h->launches;
        h->stream = h->capture_stream;
        ok = enqueue_sweep(h) == SMCX_OK;
        h->stream = user;
        h->graph_launches = h->launches - launches_before;     // kernels one replay of the graph launches
        h->launches = launches_before;
        ok = (cudaStreamEndCapture(h->capture_stream, &graph) == cudaSuccess) && ok && graph;
      }
      if (ok) ok = cudaGraphInstantiate(&h->sweep_graph, graph, 0) == cudaSuccess;
      if (graph) cudaGraphDestroy(graph);
      if (!ok) { cudaGetLastError(); h->graphs_ok = false; h->sweep_graph = nullptr; }
      else h->graph_epoch = h->params_epoch;
    }
    if (h->sweep_graph) {
      for (int64_t s = 0; s < n; ++s) {
        SMCX_CUDA(h, cudaGraphLaunch(h->sweep_graph, h->stream));
        h->launches += h->graph_launches;
        h->sweeps_enqueued++;
      }
      return SMCX_OK;
    }
  }
  for (int64_t s = 0; s < n; ++s) {
    const int rc = enqueue_sweep(h);
    if (rc != SMCX_OK) return rc;
    h->sweeps_enqueued++;
  }
  SMCX_CUDA(h, cudaGetLastError());
  return SMCX_OK;
}

int smcx_synchronize(smcx_t* h) {
  if (!h) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return SMCX_OK;
}

int smcx_energy(smcx_t* h, int64_t* E) {
  if (!h || !E) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  if (h->plan.model == SMCX_MODEL_LOCAL) {
    long long e = 0;
    const int rc = run_local_energy(h, &e);
    if (rc == SMCX_OK) *E = e;
    return rc;
  }
  std::vector<unsigned long long> M;
  const int rc = run_pair_counts(h, M);
  if (rc != SMCX_OK) return rc;
  *E = energy_from_counts(h, M);
  return SMCX_OK;
}

int smcx_running_energy(smcx_t* h, int64_t* E) {
  if (!h || !E) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  long long e = 0;
  SMCX_CUDA(h, cudaMemcpyAsync(&e, &h->d_state()->e_run, sizeof(e), cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  *E = e;
  return SMCX_OK;
}

int smcx_energy_trace(smcx_t* h, int64_t first_sweep, int64_t count, int64_t* dst) {
  if (!h || (!dst && count > 0)) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const long long cap = h->plan.G.trace_capacity;
  if (first_sweep < h->trace_first || count < 0 || first_sweep + count > h->sweeps_enqueued ||
      h->sweeps_enqueued - first_sweep > cap)
    return SMCX_E_RANGE;
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  int64_t done = 0;
  while (done < count) {
    const long long pos = (first_sweep + done) % cap;
    const long long run = std::min<long long>(count - done, cap - pos);
    SMCX_CUDA(h, cudaMemcpy(dst + done, h->d_trace() + pos, (size_t)run * sizeof(long long), cudaMemcpyDeviceToHost));
    done += run;
  }
  return SMCX_OK;
}

int smcx_species_device(smcx_t* h, void* d_dst) {
  if (!h || !d_dst) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  if (P.storage == SMCX_STORAGE_U8) {
    SMCX_CUDA(h, cudaMemcpyAsync(d_dst, h->d_species(), (size_t)P.n_sites, cudaMemcpyDeviceToDevice, h->stream));
  } else {
    SMCX_STORE_DISPATCH(P, unpack_kernel<Store><<<grid_for(h, (P.n_sites + 15) / 16, 256), 256, 0, h->stream>>>(
                               h->d_species(), reinterpret_cast<uint8_t*>(d_dst), 0, P.n_sites));
    h->launches++;
    SMCX_CUDA(h, cudaGetLastError());
  }
  return SMCX_OK;
}

// Packed storage: chunk k is unpacked into bounce buffer k & 1 on the handle's stream and copied to the host on
// the copy stream while chunk k + 1 is being unpacked; one synchronisation at the end.  A slab window writes the
// layers it owns (under the origin of the last sweep) into their place in the array of the whole lattice and leaves
// the rest of host_dst alone.
int smcx_species(smcx_t* h, uint8_t* host_dst) {
  if (!h || !host_dst) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const Plan& P = h->plan;
  const int l0 = P.window ? P.G.H + h->win_oz : 0;
  const std::vector<SiteRun> runs = site_runs(h, l0, P.window ? l0 + P.row_count * P.G.w : P.G.Lz);
  if (P.storage == SMCX_STORAGE_U8) {
    for (const SiteRun& r : runs)
      SMCX_CUDA(h, cudaMemcpyAsync(host_dst + r.host_first, h->d_species() + r.local_first, (size_t)r.count, cudaMemcpyDeviceToHost, h->stream));
    SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
    return SMCX_OK;
  }
  int rc = ensure_bounce(h);
  if (rc != SMCX_OK) return rc;
  SMCX_CUDA(h, cudaEventRecord(h->bounce_free[0], h->stream));
  SMCX_CUDA(h, cudaEventRecord(h->bounce_free[1], h->stream));
  int k = 0;
  for (const SiteRun& r : runs)
    for (long long first = 0; first < r.count; first += kChunkSites, k ^= 1) {
      const long long cnt = std::min(kChunkSites, r.count - first);
      SMCX_CUDA(h, cudaStreamWaitEvent(h->stream, h->bounce_free[k], 0));
      SMCX_STORE_DISPATCH(P, unpack_kernel<Store><<<grid_for(h, (cnt + 15) / 16, 256), 256, 0, h->stream>>>(
                                 h->d_species(), h->bounce[k], r.local_first + first, cnt));
      h->launches++;
      SMCX_CUDA(h, cudaGetLastError());
      SMCX_CUDA(h, cudaEventRecord(h->bounce_full[k], h->stream));
      SMCX_CUDA(h, cudaStreamWaitEvent(h->copy_stream, h->bounce_full[k], 0));
      SMCX_CUDA(h, cudaMemcpyAsync(host_dst + r.host_first + first, h->bounce[k], (size_t)cnt, cudaMemcpyDeviceToHost, h->copy_stream));
      SMCX_CUDA(h, cudaEventRecord(h->bounce_free[k], h->copy_stream));
    }
  SMCX_CUDA(h, cudaStreamSynchronize(h->copy_stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  return SMCX_OK;
}

// Eq. 8 from the positive-half counts M of a whole lattice of N sites.
static void sro_from_half_counts(const Geom& G, double N, const std::vector<unsigned long long>& M, double* alpha,
                                 int64_t* pair_counts) {
  const int n = G.n_species;
  std::vector<int> Z(G.n_shells, 0);
  for (int m = 0; m < G.ZT; ++m) Z[G.shell_of[m]]++;
  // ordered counts N_s(p',p) = M_s(p',p) + M_s(p,p'); species counts from the row sums of shell 0
  std::vector<long long> Ns((size_t)G.n_shells * n * n);
  for (int s = 0; s < G.n_shells; ++s)
    for (int a = 0; a < n; ++a)
      for (int b = 0; b < n; ++b)
        Ns[(size_t)(s * n + a) * n + b] = (long long)(M[(size_t)(s * n + a) * n + b] + M[(size_t)(s * n + b) * n + a]);
  std::vector<long long> n_of(n, 0);
  for (int a = 0; a < n; ++a) {
    long long row = 0;
    for (int b = 0; b < n; ++b) row += Ns[(size_t)a * n + b];
    n_of[a] = row / Z[0];
  }
  for (int s = 0; s < G.n_shells; ++s)
    for (int a = 0; a < n; ++a)
      for (int b = 0; b < n; ++b) {
        const size_t idx = (size_t)(s * n + a) * n + b;
        if (n_of[a] == 0 || n_of[b] == 0) { alpha[idx] = std::numeric_limits<double>::quiet_NaN(); continue; }
        // Eq. 8: alpha = 1 - P(p|p')/c_p, P = N_s(p',p)/(Z_s n_p'), c_p = n_p/N
        const double P = (double)Ns[idx] / ((double)Z[s] * (double)n_of[a]);
        const double c = (double)n_of[b] / N;
        alpha[idx] = 1.0 - P / c;
      }
  if (pair_counts) std::memcpy(pair_counts, Ns.data(), Ns.size() * sizeof(long long));
}

int smcx_sro(smcx_t* h, double* alpha, int64_t* pair_counts) {
  if (!h || !alpha) return SMCX_E_NULL_ARG;
  if (h->plan.window) return SMCX_E_UNSUPPORTED;   // partial counts: smcx_domain_pair_counts + smcx_sro_from_counts
  DeviceGuard on_device(h->device);
  std::vector<unsigned long long> M;
  const int rc = run_pair_counts(h, M);
  if (rc != SMCX_OK) return rc;
  sro_from_half_counts(h->plan.G, (double)h->plan.n_sites, M, alpha, pair_counts);
  return SMCX_OK;
}

int smcx_stats(smcx_t* h, int64_t* sweeps_done, int64_t* trials, int64_t* accepted) {
  if (!h) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  DevState st;
  SMCX_CUDA(h, cudaMemcpyAsync(&st, h->d_state(), sizeof(st), cudaMemcpyDeviceToHost, h->stream));
  SMCX_CUDA(h, cudaStreamSynchronize(h->stream));
  if (sweeps_done) *sweeps_done = (int64_t)st.sweep;
  if (trials) *trials = (int64_t)st.sweep * (h->plan.window ? h->plan.layer_sites * h->plan.row_count * h->plan.G.w : h->plan.n_sites);
  if (accepted) *accepted = (int64_t)st.accepted;
  return SMCX_OK;
}

int smcx_shell_offsets(smcx_t* h, int32_t shell, int32_t* xyz, int32_t max_offsets, int32_t* n_offsets) {
  if (!h || !n_offsets) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  const Geom& G = h->plan.G;
  if (shell < 0 || shell >= G.n_shells) return SMCX_E_BAD_SHELLS;
  int k = 0;
  for (int m = 0; m < G.ZT; ++m)
    if (G.shell_of[m] == shell) {
      if (xyz && k < max_offsets) { xyz[3 * k] = G.off[m][0]; xyz[3 * k + 1] = G.off[m][1]; xyz[3 * k + 2] = G.off[m][2]; }
      ++k;
    }
  *n_offsets = k;
  return SMCX_OK;
}

int smcx_get_config(smcx_t* h, int32_t* storage, int32_t* kernel, int64_t* n_sites, int64_t* n_cells) {
  if (!h) return SMCX_E_NULL_ARG;
  DeviceGuard on_device(h->device);
  if (storage) *storage = h->plan.storage;
  if (kernel) *kernel = h->plan.kernel;
  if (n_sites) *n_sites = h->plan.n_sites;
  if (n_cells) *n_cells = h->plan.n_cells;
  return SMCX_OK;
}

int64_t smcx_kernel_launches(smcx_t* h) { return h ? h->launches : 0; }

int smcx_group_layout(const smcx_params_t* p, int32_t* lanes, int32_t* A, int32_t* B, int32_t* shift,
                      int32_t* tile_bytes, int32_t* skew, uint8_t* slots) {
  if (!p) return SMCX_E_NULL_ARG;
  Plan plan;
  const int rc = make_plan(p, &plan);
  if (rc != SMCX_OK) return rc;
  const Geom& G = plan.G;
  if (lanes) *lanes = plan.group_lanes;
  if (A) *A = G.gA;
  if (B) *B = G.gB;
  if (shift) *shift = G.gshift;
  if (tile_bytes) *tile_bytes = G.gtile;
  if (skew) *skew = G.gskew;
  if (slots) std::memcpy(slots, G.gslot, kMaxGroupSlots);
  return SMCX_OK;
}

}  // extern "C"

#include "ensemble_api.inc"
#include "domain_api.inc"
#include "static_scratch_api.inc"
