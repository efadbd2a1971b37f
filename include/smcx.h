/* smcx.h -- C ABI of the B200-native SMC-X hot path (arxiv 2509.20949).
 *
 * What the library computes: parallel Metropolis atom-swap sweeps over a multicomponent
 * BCC/FCC lattice alloy with an effective-pair-interaction (EPI) Hamiltonian, scheduled by
 * dynamic link cells (LC):
 *   - canonical ensemble and Metropolis acceptance, Eq. 1-3;
 *   - one Monte Carlo step (sweep) = exactly one trial move per lattice site;
 *   - a trial move swaps two neighbouring lattice sites;
 *   - link cells are re-built every step so that every site is visited exactly once and
 *     distant cells update concurrently; each trial costs O(1) through the local interaction
 *     zone (LIZ / LIZ+), section "Distributed SMC-X" (Eq. 4);
 *   - the EPI model is pairwise (section "Results and discussion");
 *   - the Warren-Cowley short-range-order parameter, Eq. 8.
 * The paper defers the concrete schedule to its Ref. 22; the schedule implemented here (per-sweep
 * random LC origin, 2x2x2 colouring, raster order inside a cell, Philox4x32-10 keyed by
 * (seed, sweep, colour, cell), integer energies and table-driven integer acceptance) is the
 * reading S0-S8 listed in DESIGN.md.  Given that schedule the species array and the energy trace
 * after n sweeps are unique, and the library reproduces them bit for bit.
 *
 * Conventions
 *   - Every call returns SMCX_OK (0) or a negative SMCX_E_* code.  Nothing throws or aborts
 *     across this boundary.  Out-parameters are written only on success.
 *   - "host" pointers are ordinary CPU memory, "device" pointers are CUDA device memory on the
 *     handle's device.  The caller owns every pointer it passes; host tables are copied during
 *     the call.  Device buffers passed at creation must outlive the handle.
 *   - All GPU work is enqueued on the stream given at creation.  Calls that return results to
 *     the host synchronise that stream; smcx_sweep and smcx_set_temperature do not.
 *   - A handle is not thread-safe.  One handle drives one GPU; there is no CPU fallback:
 *     without a CUDA device smcx_create fails with SMCX_E_CUDA.
 *
 * Geometry (reading S0).  Lengths in units of a/2.  BCC: 2 sites per conventional cell at
 * (0,0,0),(1,1,1); FCC: 4 sites at (0,0,0),(0,1,1),(1,0,1),(1,1,0).  Site id
 * i = ((z*Ly + y)*Lx + x)*B + b (PAPER.md:165 writes lattices as nx*ny*nz*basis), periodic in
 * all three directions.  Shell s is the set of lattice vectors with the s-th smallest
 * non-zero length, in ascending (dz, dy, dx) order.
 */
#ifndef SMCX_H_
#define SMCX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct smcx smcx_t; /* opaque; one per (GPU, stream) */

enum { SMCX_BCC = 0, SMCX_FCC = 1 };

/* Device storage of the species array.  U8: one byte per site in site-id order.
 * 2BIT: 16 sites per 32-bit word in site-id order (n_species <= 4).
 * 4BIT: 8 sites per 32-bit word (n_species <= 16), sublattice-planar in groups of 8 conventional cells along x
 * (dims[0] must be a multiple of 8): group g = c >> 3 of conventional cell c = (z Ly + y) Lx + x holds B words
 * (B = 2 BCC, 4 FCC), word b = the sites with basis index b of its 8 cells, cell c & 7 in bits 4 (c & 7) .. + 3.
 * Results never depend on the storage (smcx_species always returns one byte per site in site-id order). */
enum { SMCX_STORAGE_AUTO = 0, SMCX_STORAGE_2BIT = 2, SMCX_STORAGE_4BIT = 4, SMCX_STORAGE_U8 = 8 };

/* Which sweep kernel runs.  WARP_PER_CELL: any lattice/shell list, U8 storage.
 * GROUP_PER_CELL: the same generality with 4, 8, 16 or 32 lanes per link cell (8, 16 or 32 by the number of
 * cells per colour; smcx_params_t::group_lanes overrides the choice) and a
 * per-pair difference table in shared memory; what AUTO picks whenever a thread kernel does not apply.
 * THREAD_PER_CELL: BCC, first two shells, link_cell = 4, n_species <= 4, 2BIT storage; one block per
 * 128 cells, two-level acceptance filter in shared memory.
 * THREAD_PERSISTENT: same restrictions; one block per SM whose warps walk over the cells of the
 * colour, the whole threshold table in shared memory.  While the current table is too long for that
 * (more than 15,871 entries next to 20 warps, 24,063 next to 16) passes run the THREAD_PER_CELL
 * kernel instead.
 * FCC_THREAD: FCC, the first 2..3 shells (tile of 8^3 cells), link_cell = 4, n_species <= 8, 4BIT storage, every
 * |V_s(b,x) - V_s(a,x)| < 32768: one thread per link cell on a packed tile (one 32-bit word per sublattice row of 8
 * cells), neighbours gathered by rotations and bit-selects, the EPI differences applied four neighbours at a time by
 * byte-permute look-ups (PRMT) and byte dot products (sweep_fcc.cuh).  What AUTO picks for such lattices when
 * a colour has at least 12,000 link cells (measured crossover; below that the sub-warp kernel's shorter chain per trial wins).
 * BCC4_THREAD: BCC, the first two shells, link_cell = 4, n_species <= 8, 4BIT storage, every |V_s(b,x) - V_s(a,x)| < 32768:
 * the BCC counterpart of FCC_THREAD (one thread per link cell on a 512-byte packed tile, nine row loads per site, the same
 * PRMT look-ups; sweep_bcc4.cuh).  What AUTO picks for BCC lattices with 5..8 species when a colour has at least
 * 12,000 link cells.
 * smcx_sweep runs the eight colour passes of THREAD_PERSISTENT as ONE launch, the passes pipelined through completion
 * counters in device memory (sweep_thread_sweep.cuh), for an undivided lattice of up to 2.4e6 link cells per colour --
 * for one handle per process at a time (the first such handle alive; the others launch per colour): two of these launches
 * at once could starve each other of SMs.  Same results either way.  The launch has one block per SM and its warps
 * wait for one another's results, so every block must become resident: run it on a whole GPU (not inside an MPS
 * partition that exposes fewer SMs than the device reports); other kernels that merely occupy SMs for a while only
 * delay it.
 * AUTO picks, when the parameters allow a thread kernel, THREAD_PERSISTENT for lattices that give every
 * warp of every SM a batch of cells (>= 148*20*32 link cells per colour) and THREAD_PER_CELL below that
 * (same speed there, and concurrent lattices of a replica ensemble overlap freely).  Results never
 * depend on it. */
enum { SMCX_KERNEL_AUTO = 0, SMCX_KERNEL_WARP_PER_CELL = 1, SMCX_KERNEL_THREAD_PER_CELL = 2,
       SMCX_KERNEL_THREAD_PERSISTENT = 3, SMCX_KERNEL_GROUP_PER_CELL = 4, SMCX_KERNEL_FCC_THREAD = 5,
       SMCX_KERNEL_LOCAL_WARP = 6, SMCX_KERNEL_BCC4_THREAD = 7 };

/* Energy model.  EPI: the pairwise effective-pair-interaction Hamiltonian (reading S1).
 * LOCAL: "a general nonlinear short-range model, where the local energies of all lattice sites within LIZ are
 * calculated to determine the energy change due to a MC move" (the role of the paper's qSRO model, whose
 * form and weights are its Ref. 22 and not available).  Reading S12: H = sum_i eps(sigma_i, n_i), n_i[s][x] = number of
 * neighbours of species x in shell s of site i, eps(a, n) = sum_s ( sum_x W1[s][a][x] n[s][x] + sum_{x <= y}
 * W2[s][a][x][y] n[s][x] n[s][y] ); int32 weights, int64 energies.  `epi` is then W1 (it need not be symmetric) and
 * `local_quad` W2.  With W2 = 0 and W1 symmetric the model is twice the EPI Hamiltonian.  A trial reads the
 * neighbours of the neighbours of i and j, so the link cell must satisfy 2w >= 2 r0 + 2 R; n_species <= 8; uint8
 * storage; kernel SMCX_KERNEL_LOCAL_WARP (one warp per link cell).  smcx_energy returns H of this model;
 * smcx_sro is unchanged.  On slabs (smcx_domain_*) the window has H = 3 ghost layers and a pass message 4 layers. */
enum { SMCX_MODEL_EPI = 0, SMCX_MODEL_LOCAL = 1 };

enum {
  SMCX_OK = 0,
  SMCX_E_NULL_ARG = -1,
  SMCX_E_BAD_LATTICE = -2,
  SMCX_E_BAD_DIMS = -3,            /* non-positive, not divisible by 2*link_cell, smaller than a
                                      cell plus its halo, or too many sites/cells */
  SMCX_E_BAD_SPECIES = -4,         /* n_species outside 2..16 */
  SMCX_E_BAD_SHELLS = -5,          /* n_shells outside 1..5 */
  SMCX_E_EPI_NOT_SYMMETRIC = -6,
  SMCX_E_LINK_CELL_TOO_SMALL = -7, /* violates 2w >= 2 r0 + R (reading S2) */
  SMCX_E_BAD_TABLE = -8,           /* acceptance table missing, empty or too long */
  SMCX_E_BAD_STATE = -9,           /* uploaded species value >= n_species */
  SMCX_E_NO_MEMORY = -10,          /* host or device allocation failed / workspace too small */
  SMCX_E_CUDA = -11,               /* CUDA error; text via smcx_last_error */
  SMCX_E_UNSUPPORTED = -12,        /* storage/kernel choice not valid for these parameters */
  SMCX_E_RANGE = -13,              /* trace range not retained, sweep counter overflow */
  SMCX_E_EPI_RANGE = -14,          /* EPI magnitudes / local-model weights so large that the int32 dE of a trial could overflow */
  SMCX_E_STATIC_SCRATCH = -15      /* smcx_pair_counts_static: n_shells * n_species^2 > SMCX_STATIC_PAIR_COUNTS_MAX */
};

typedef struct {
  int32_t lattice;          /* SMCX_BCC | SMCX_FCC */
  int32_t dims[3];          /* Lx, Ly, Lz conventional cells; each divisible by 2*link_cell */
  int32_t n_species;        /* 2..16; species values are 0..n_species-1 */
  int32_t n_shells;         /* the first n_shells neighbour shells, 1..5 */
  const int32_t *epi;       /* host, [n_shells][n_species][n_species], symmetric, 0.1 meV units */
  int32_t link_cell;        /* w, conventional cells per link-cell edge; 0 means 4 */
  int32_t kT_units;         /* kT in 0.1 meV; recorded for reports only (see accept) */
  const uint32_t *accept;   /* host, thresholds T[0..accept_len): a trial with dE = d > 0 is
                               accepted iff d < accept_len and u < T[d], u a 32-bit Philox word
                               (Eq. 3 in integer form); the library never evaluates exp() */
  int32_t accept_len;       /* 1 .. 2^20 (entries reserved on the device); longer tables: SMCX_E_BAD_TABLE */
  uint64_t seed;            /* Philox key */
  int32_t storage;          /* SMCX_STORAGE_* */
  int32_t kernel;           /* SMCX_KERNEL_* */
  int32_t device;           /* CUDA device ordinal */
  int32_t trace_capacity;   /* sweeps of energy trace retained (ring buffer); 0 means 65536 */
  void *stream;             /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = legacy default */
  void *d_workspace;        /* device, caller-owned, >= smcx_workspace_bytes(); NULL = library allocates */
  size_t workspace_bytes;   /* size of d_workspace */
  int32_t group_lanes;      /* GROUP_PER_CELL: lanes per link cell, 4 | 8 | 16 | 32; 0 = chosen from the cells per colour.
                               A value whose tiles do not fit shared memory is ignored (auto). */
  int32_t group_warps;      /* GROUP_PER_CELL: warps per block, 1..8; 0 = as many as leave room for four blocks per SM */
  int32_t domain_count;     /* 0 or 1: the handle holds the whole lattice.  Set by smcx_domain_create (>= 2: the handle holds */
  int32_t domain_index;     /* slab domain_index of dims cut into domain_count slabs along z); leave both 0 otherwise */
  int32_t model;            /* SMCX_MODEL_* */
  const int32_t *local_quad;/* host, SMCX_MODEL_LOCAL: W2[n_shells][n_species][n_species][n_species] (x <= y used) */
} smcx_params_t;

/* Bytes of device workspace a handle with these parameters needs (species array in its storage
 * format, tables, trace, counters).  Validates the parameters like smcx_create. */
int smcx_workspace_bytes(const smcx_params_t *p, size_t *bytes);

/* Validates, copies the tables, builds the shell-offset tables, and fills the lattice with the
 * seeded equiatomic initial state (reading S6: sigma_i = pi(i) mod n_species, pi a 4-round Feistel
 * permutation of [0,N) keyed by seed).  The sweep counter starts at 0. */
int smcx_create(smcx_t **out, const smcx_params_t *p);
void smcx_destroy(smcx_t *h);

/* Replace the lattice state (the configuration sigma of Eq. 1-2).  host_src / d_src: N bytes, one
 * species per site in site-id order.  Values are validated on the device (no pass over the array on the host):
 * SMCX_E_BAD_STATE if one is >= n_species -- the device path then leaves the lattice unchanged, the host path has
 * overwritten it with the low bits of the rejected array and it must be set again.  Host memory may be pageable
 * or pinned (pinned: the copy of one 2^26-site chunk overlaps the packing of the previous one).
 * The running energy is recomputed; the sweep counter and trace are kept.  Synchronises. */
int smcx_set_species(smcx_t *h, const uint8_t *host_src);
int smcx_set_species_device(smcx_t *h, const void *d_src);

/* The species array in the handle's device storage format, for checkpoints that move 1/4 (2BIT) or 1/2 (4BIT) byte
 * per site (3-million-step runs): smcx_storage_bytes() bytes of host memory, layout as
 * described at SMCX_STORAGE_*.  A packed checkpoint can only be loaded into a handle with the same storage, lattice
 * and dims.  smcx_set_species_packed validates like smcx_set_species (SMCX_E_BAD_STATE: set the state again),
 * recomputes the running energy and keeps the sweep counter.  Both synchronise. */
int smcx_storage_bytes(smcx_t *h, size_t *bytes);
int smcx_species_packed(smcx_t *h, void *host_dst);
int smcx_set_species_packed(smcx_t *h, const void *host_src);

/* Replace the lattice state by a seeded random solid solution of a given composition (reading S10;
 * the paper's alloy is Fe29Co29Ni28Al7Ti7): counts[p] >= 0 sites of species p,
 * p < n_species, summing to N; site i holds the species p with cum_p <= pi(i) < cum_{p+1}, pi the
 * permutation of S6 keyed by the handle's seed.  Host array.  SMCX_E_BAD_STATE if the counts are negative
 * or do not sum to N.  The running energy is recomputed; the sweep counter and trace are kept. */
int smcx_init_composition(smcx_t *h, const int64_t *counts);

/* Resume from a checkpoint.  The state of a run is (species array, sweep counter, seed, threshold
 * table); the random numbers depend on counters only (reading S4), so a handle created with the same
 * parameters, given the saved species (smcx_set_species) and the saved counter, continues the run bit for
 * bit (3-million-step runs as in PAPER.md:165 need this).  The next sweep is sweep t, 0 <= t < 2^32; the
 * energy trace restarts at t.  Synchronises. */
int smcx_set_sweep_counter(smcx_t *h, int64_t t);

/* New acceptance table (a new temperature) for the following sweeps.  Asynchronous with respect
 * to the host: the table is copied into library-owned pinned memory before the call returns. */
int smcx_set_temperature(smcx_t *h, int32_t kT_units, const uint32_t *accept, int32_t accept_len);

/* Enqueue n sweeps (reading S3).  Asynchronous.  The sweep counter is global to the handle:
 * sweep(a); sweep(b) is identical to sweep(a+b). */
int smcx_sweep(smcx_t *h, int64_t n);

/* Total energy H (reading S1: every unordered bond once, int64) recomputed from the lattice by the
 * pair-count reduction kernel.  Synchronises. */
int smcx_energy(smcx_t *h, int64_t *E);
/* Running energy E_0 + sum of accepted dE as kept by the sweep kernels.  Synchronises. */
int smcx_running_energy(smcx_t *h, int64_t *E);
/* Energy after every Monte Carlo step (the quantity a warm-up / measurement protocol watches, PAPER.md:65;
 * E_i of Eq. 6 for replica exchange): dst[k] = running energy after sweep first_sweep + k,
 * k < count.  SMCX_E_RANGE if a sweep is no longer (or not yet) in the ring of trace_capacity entries.
 * Synchronises. */
int smcx_energy_trace(smcx_t *h, int64_t first_sweep, int64_t count, int64_t *dst);

/* The configuration sigma itself (what the paper stores and post-processes: "configurations" for the SRO
 * average PAPER.md:163 and the atom-probe comparison PAPER.md:185; lattice order nx*ny*nz*basis):
 * N bytes, one species per site in site-id order whatever the device storage.  Synchronises. */
int smcx_species(smcx_t *h, uint8_t *host_dst);
int smcx_species_device(smcx_t *h, void *d_dst); /* asynchronous, on the handle's stream */

/* Warren-Cowley parameters, Eq. 8: alpha[(s*n + p')*n + p] = 1 - N_s(p',p) N / (Z_s n_p' n_p) in
 * fp64 from the exact ordered pair counts N_s(p',p) = #{(i,d): d in shell s, sigma_i = p',
 * sigma_{i+d} = p} (int64).  NaN where a species is absent.  pair_counts may be NULL.  Synchronises. */
int smcx_sro(smcx_t *h, double *alpha, int64_t *pair_counts);

/* Bookkeeping of the run: Monte Carlo steps done, trial moves made (= steps x N: one trial per site per step,
 * PAPER.md:65; the paper's throughput unit "atom step") and trials accepted by Eq. 3
 * (PAPER.md:60-63).  Every pointer may be NULL.  Synchronises. */
int smcx_stats(smcx_t *h, int64_t *sweeps_done, int64_t *trials, int64_t *accepted);
int smcx_synchronize(smcx_t *h);

/* Introspection for tests and benchmarks. */
int smcx_shell_offsets(smcx_t *h, int32_t shell, int32_t *xyz, int32_t max_offsets, int32_t *n_offsets);
int smcx_get_config(smcx_t *h, int32_t *storage, int32_t *kernel, int64_t *n_sites, int64_t *n_cells);
int64_t smcx_kernel_launches(smcx_t *h); /* kernels launched by this handle so far */
/* Shared-memory tile layout the host chose for the GROUP_PER_CELL kernel with these parameters (needs no
 * GPU): lanes per cell; the tile index of the site at tile position (px, py, pz), units of a/2, is
 * (px + A py + B pz) >> shift; tile_bytes per cell plus skew bytes between the tiles of a warp;
 * slots[k] = neighbour (index into the concatenated shell list) that lane k % lanes visits in its visit
 * k / lanes, 255 = none, k < 128.  Every pointer may be NULL. */
int smcx_group_layout(const smcx_params_t *p, int32_t *lanes, int32_t *A, int32_t *B, int32_t *shift,
                      int32_t *tile_bytes, int32_t *skew, uint8_t *slots);

/* ---- Temperature parallelism on one GPU: replica ensemble and replica exchange -----------------
 * "multiple replicas of the same system are simulated concurrently at different
 * temperatures.  Configurations between replicas are periodically exchanged according to a
 * Metropolis criterion", P_swap = min(1, exp(Delta)) (Eq. 5),
 * Delta = (1/kT_i - 1/kT_j)(E_i - E_j) (Eq. 6); the ladder spacing follows Eq. 7 (PAPER.md:99-102,
 * chosen by the caller).  Reading S9: in exchange round r the neighbouring slots
 * (p, p+1), p = parity, parity+2, ..., attempt an exchange; Delta is evaluated in fp64 from the
 * integer running energies and integer kT; accept iff Delta >= 0 or
 * u < min(floor(exp(Delta) 2^32), 2^32-1), u = philox4x32_10(ctr = (p, r_hi, r_lo, 6), key =
 * exchange_seed)[0].  An accepted exchange swaps the temperatures of the two replicas (each keeps
 * its lattice, seed, sweep counter and trace and gets the threshold table of its new slot), which is
 * the same Markov chain as swapping the configurations.  Decision and table switch run in kernels on
 * the device: no call below synchronises with the host except smcx_ensemble_state.
 *
 * An ensemble owns n_replicas handles, one CUDA stream each (so small lattices run concurrently),
 * all forked from / joined to the stream of `base` around every call: seen from that stream the
 * calls execute in order.  Replica r is created like smcx_create(base) with seed seeds[r] and starts
 * in slot r.  Every table is zero-padded to the longest one (T[d] = 0 for d >= len is the
 * definition of the table, so no decision changes). */
typedef struct smcx_ensemble smcx_ensemble_t;

/* kT_units, accept, accept_len, seeds: host arrays of n_replicas entries (accept[p] is the host
 * table of slot p, kT_units strictly positive).  base->accept / accept_len / seed / kT_units /
 * d_workspace are ignored (the library allocates device memory).  2 <= n_replicas <= 1024. */
int smcx_ensemble_create(smcx_ensemble_t **out, const smcx_params_t *base, int32_t n_replicas,
                         const int32_t *kT_units, const uint32_t *const *accept, const int32_t *accept_len,
                         const uint64_t *seeds, uint64_t exchange_seed);
void smcx_ensemble_destroy(smcx_ensemble_t *e);
/* Borrowed handle of replica r (valid until the ensemble is destroyed; do not smcx_destroy it, do
 * not call smcx_set_temperature on it).  Reading calls (smcx_species, smcx_energy, smcx_sro,
 * smcx_energy_trace, smcx_stats) are fine and synchronise that replica's stream only. */
smcx_t *smcx_ensemble_replica(smcx_ensemble_t *e, int32_t r);
/* n sweeps on every replica, each on its own stream.  Asynchronous. */
int smcx_ensemble_sweep(smcx_ensemble_t *e, int64_t n);
/* One exchange round with the given parity (0: pairs (0,1),(2,3),...; 1: (1,2),(3,4),...).
 * Asynchronous: decision kernel + table switch on the device. */
int smcx_ensemble_exchange(smcx_ensemble_t *e, int32_t parity);
/* rounds x (sweeps_per_round sweeps on every replica, then one exchange round whose parity is the
 * low bit of the ensemble's round counter).  Asynchronous. */
int smcx_ensemble_run(smcx_ensemble_t *e, int64_t rounds, int64_t sweeps_per_round);
/* Synchronises and reports (every pointer may be NULL): replica_at_slot[n], energy_at_slot[n]
 * (running energy of the replica in that slot), attempted[n-1] / accepted[n-1] per slot pair,
 * last_flags[n-1] (accept flags of the last round, 0 for pairs not attempted), rounds done. */
int smcx_ensemble_state(smcx_ensemble_t *e, int32_t *replica_at_slot, int64_t *energy_at_slot,
                        int64_t *attempted, int64_t *accepted, int32_t *last_flags, int64_t *rounds);
int smcx_ensemble_synchronize(smcx_ensemble_t *e);
int64_t smcx_ensemble_kernel_launches(smcx_ensemble_t *e); /* ensemble kernels + those of all replicas */

/* ---- Lattice parallelism: slabs with ghost layers, computation-communication overlap ---------------------------
 * PAPER.md:85 (section "Distributed SMC-X"): "the complete lattice is partitioned across multiple GPUs, with a ghost
 * layer used to exchange boundary information between neighboring sublattices" (Fig. 2); "We also
 * implemented a computing-communication overlap for EPI_GPU" (strong scaling 0.339 -> 0.679 on 16 GPUs).  The paper
 * gives no protocol; reading S11:
 *   - the lattice is cut along z into n_domains slabs on boundaries of PAIRS of link-cell rows: with
 *     pairs = dims[2] / link_cell / 2, slab k owns pairs / n + (k < pairs mod n) consecutive pairs (n <= pairs);
 *   - a slab owns link cells, not layers: in a sweep with origin oz its rows [r0, r1) cover the layers
 *     [a, b) = [oz + r0 w, oz + r1 w) (mod dims[2]).  It stores, without wrap, the layers r0 w - H .. r1 w + w - 2 + H
 *     (H = 2 ghost layers: the LIZ+ reaches r0 + R = 3 half-units): every window [a - H, b + H) for oz < w;
 *   - random numbers are keyed by the GLOBAL cell id, so the decomposed sweep reproduces the undivided one bit for bit;
 *   - start of a sweep: the window moves by oz - oz_prev layers and the layers entering it are fetched from the
 *     neighbour on that side; after colour pass c (rows of parity pz = (c >> 2) & 1 active) the slab's bottom row
 *     (pz = 0) sends the layers [a - 1, a + H) down, its top row (pz = 1) sends [b - H, b + 1) up: one message per slab
 *     and pass, H + 1 layers, contiguous in device storage (layers are the slowest index of every storage format);
 *   - overlap: a pass is launched as the boundary row first, then the message leaves on a copy stream while the
 *     other rows of the pass run.
 * Three ways to run it.  (1) Connected slabs, smcx_domain_ipc_* / smcx_domain_sweep_connected: one slab per process and
 * GPU, the neighbours' storage mapped with CUDA IPC, messages written by the sweep kernels into the neighbour's memory
 * and signalled through device flags -- no host code in the data path (see below).  (2) smcx_domain_group_*: all slabs
 * in one process, on one or several devices, ordered by events; the pass messages of the packed kernels are fused into
 * the boundary-row kernel (smcx_domain_pass_fused), which runs next to the other rows of the pass; only the window
 * shift is a copy.  (3) smcx_domain_begin_sweep / _pass / _pass_split / _end_sweep: one slab per handle stepped by the
 * caller, who moves the messages (e.g. torch.distributed send/recv over NCCL on the byte ranges the message calls
 * name) -- for slabs on different nodes.
 * Errors: the calls return SMCX_E_RANGE when used out of order (a pass outside begin/end_sweep, results asked for in
 * the middle of a sweep), SMCX_E_BAD_DIMS for a cut the lattice does not allow, SMCX_E_UNSUPPORTED where stated, and
 * otherwise what the underlying handle returns.  All pointers are the caller's; device pointers must be valid on the
 * slab's device (peer access enabled when they belong to another GPU). */
typedef struct smcx_domain smcx_domain_t;
typedef struct smcx_domain_group smcx_domain_group_t;

typedef struct {
  int32_t n_domains, index;
  int32_t lower, upper;          /* indices of the neighbouring slabs (periodic) */
  int32_t row_first, row_count;  /* link-cell rows along z this slab owns (both even) */
  int32_t z_base;                /* layer of the whole lattice held in storage layer 0 (mod dims[2]) */
  int32_t z_layers;              /* storage layers = row_count w + w - 1 + 2 ghost */
  int32_t ghost;                 /* H */
  int32_t storage;               /* SMCX_STORAGE_* of the slab */
  int64_t layer_bytes;           /* bytes of one layer in device storage */
  int64_t owned_sites;           /* row_count w dims[0] dims[1] B */
} smcx_domain_info_t;

/* One message: `bytes` bytes at byte offset `offset` of this slab's species storage (smcx_domain_storage), to / from
 * slab `peer`.  tag 0: the message travels downwards (to the lower neighbour), 1: upwards.  The message a slab sends
 * with tag T is the one its peer receives with tag T.  bytes = 0: no message. */
typedef struct { int32_t peer, tag; int64_t offset, bytes; } smcx_domain_msg_t;

/* The partition alone (host arithmetic, no GPU): what slab `index` of `n_domains` holds.  storage / layer_bytes are
 * those smcx_domain_create would choose.  SMCX_E_BAD_DIMS if dims[2] has fewer than n_domains pairs of rows. */
int smcx_domain_partition(const smcx_params_t *p, int32_t n_domains, int32_t index, smcx_domain_info_t *info);
/* The messages of a slab, from the seed and the sweep number alone (host arithmetic, no GPU): phase -1 = window shift at
 * the start of sweep `sweep` (needs the origins of sweeps sweep - 1 and sweep; none for sweep == first_sweep, when every
 * layer of a window is valid), phase 0..7 = after that colour pass. */
int smcx_domain_plan_messages(const smcx_params_t *p, int32_t n_domains, int32_t index, int64_t sweep, int64_t first_sweep,
                              int32_t phase, smcx_domain_msg_t *send, smcx_domain_msg_t *recv);

/* One slab.  p describes the WHOLE lattice (dims, seed, tables ...); p->d_workspace, if given, must hold
 * smcx_domain_workspace_bytes().  The initial state is the slab's part of the seeded state of the whole lattice. */
int smcx_domain_workspace_bytes(const smcx_params_t *p, int32_t n_domains, int32_t index, size_t *bytes);
int smcx_domain_create(smcx_domain_t **out, const smcx_params_t *p, int32_t n_domains, int32_t index);
void smcx_domain_destroy(smcx_domain_t *d);
int smcx_domain_info(smcx_domain_t *d, smcx_domain_info_t *info);
void *smcx_domain_storage(smcx_domain_t *d);   /* device pointer of the species storage: z_layers * layer_bytes bytes */
/* host arrays of the WHOLE lattice (N bytes, site-id order): the slab takes its window / fills in the layers it owns */
int smcx_domain_set_species(smcx_domain_t *d, const uint8_t *host_whole);
int smcx_domain_species(smcx_domain_t *d, uint8_t *host_whole);
int smcx_domain_init_composition(smcx_domain_t *d, const int64_t *counts);
int smcx_domain_set_temperature(smcx_domain_t *d, int32_t kT_units, const uint32_t *accept, int32_t accept_len);
int smcx_domain_set_sweep_counter(smcx_domain_t *d, int64_t t);
/* One sweep = begin_sweep, [move the shift messages], then for colour 0..7: pass (part 0 = every row of the colour;
 * or part 1 = the boundary row, then part 2 = the others), [move the pass messages], and end_sweep.  The caller must
 * have completed the incoming messages of a phase (and its own outgoing ones) on the slab's stream before the next
 * smcx_domain_pass.  send / recv may be NULL.  All asynchronous on the slab's stream. */
int smcx_domain_begin_sweep(smcx_domain_t *d, smcx_domain_msg_t *send, smcx_domain_msg_t *recv);
int smcx_domain_pass(smcx_domain_t *d, int32_t colour, int32_t part);
int smcx_domain_pass_messages(smcx_domain_t *d, int32_t colour, smcx_domain_msg_t *send, smcx_domain_msg_t *recv);
/* Parts 1 and 2 of a pass at the same time (computation-communication overlap): the boundary row on
 * `side_stream` (a cudaStream_t of the slab's device; it is made to wait for the slab's stream first), the other rows on
 * the slab's own stream, on disjoint sets of SMs where the kernel takes one block per SM.  The caller sends the pass
 * message from side_stream (its layers are complete when the work enqueued there so far is) and lets the slab's stream
 * wait for side_stream before the next pass. */
int smcx_domain_pass_split(smcx_domain_t *d, int32_t colour, void *side_stream);
/* The boundary row of a pass (part 1) with its message FUSED into the kernel: while a cell writes its tile back it also
 * stores the layers of the outgoing message straight into the neighbour's species storage -- only the bytes it modified,
 * no copy kernel, no copy engine (peer stores over NVLink when the neighbour is on another GPU of this process).
 * peer_storage = smcx_domain_storage() of the neighbour the pass sends to (a device pointer valid in this process, peer
 * access enabled if it is on another device), peer_offset = the byte offset its smcx_domain_pass_messages gives for the
 * incoming message.  The neighbour's next pass must wait for this launch (an event), nothing else.  SMCX_E_UNSUPPORTED
 * if the slab's kernel has no fused write-back (the packed kernels THREAD_* and FCC_THREAD have): use part 1 + a copy. */
int smcx_domain_pass_fused(smcx_domain_t *d, int32_t colour, void *peer_storage, int64_t peer_offset);
int smcx_domain_end_sweep(smcx_domain_t *d);
/* Connected slabs: one slab per PROCESS (one process per GPU), no host in the data path.  A slab is connected to the
 * species storage and the two message flags of its neighbours -- device pointers valid in this process: exported with
 * smcx_domain_ipc_export and mapped with CUDA IPC by smcx_domain_ipc_connect when the neighbour lives in another process
 * (same GPU or a peer GPU over NVLink), or given directly to smcx_domain_connect when it lives in this one.  Then
 * smcx_domain_sweep_connected(n) enqueues n whole sweeps: the window shift is pushed into the neighbour's storage by a
 * device-to-device copy, the message of a colour pass is written there by the boundary-row kernel itself (as
 * smcx_domain_pass_fused) while the other rows of the pass run concurrently, and every message is followed by a serial
 * number stored into the neighbour's flag; the receiver's stream waits for that number (a stream memory operation, no
 * kernel spins, no host thread is involved).  Slabs are connected once, all of them before any of them sweeps (a
 * barrier of the caller's), and must be given the same sweep counts.  Slabs that share a process (tests) must be stepped
 * in turns with small n, and there may be at most three of them: the device has 8 hardware work queues by default, and a
 * stream that waits for a flag must not share a hardware work queue with the stream whose work sets it
 * (smcx_domain_connect returns SMCX_E_UNSUPPORTED beyond that; one slab per process, the intended use, needs two queues).  The slab's workspace must be the library's own
 * allocation (smcx_params_t::d_workspace NULL) for smcx_domain_ipc_export. */
typedef struct {
  unsigned char handle[64];      /* cudaIpcMemHandle_t of the slab's workspace allocation */
  int64_t storage_offset;        /* of the species storage inside it */
  int64_t flags_offset;          /* of the two message flags (uint32: from the lower, from the upper neighbour) */
  int32_t index, device;         /* slab index; CUDA device ordinal in the exporting process */
} smcx_domain_ipc_t;
int smcx_domain_ipc_export(smcx_domain_t *d, smcx_domain_ipc_t *out);
int smcx_domain_ipc_connect(smcx_domain_t *d, const smcx_domain_ipc_t *lower, const smcx_domain_ipc_t *upper);
void *smcx_domain_flags(smcx_domain_t *d);     /* device pointer of this slab's two message flags */
int smcx_domain_connect(smcx_domain_t *d, void *lower_storage, void *lower_flags, void *upper_storage, void *upper_flags);
int smcx_domain_sweep_connected(smcx_domain_t *d, int64_t n);   /* asynchronous */

/* Partial results; their sums over the slabs are those of the whole lattice.  pair_counts: positive-half counts
 * M[s][x][y] of the bonds of the layers the slab owns; running energy / trace: the slab's share of H at the start plus
 * the dE its cells accepted.  Synchronise the slab's stream. */
int smcx_domain_pair_counts(smcx_domain_t *d, int64_t *half_counts);
int smcx_domain_running_energy(smcx_domain_t *d, int64_t *E);
int smcx_domain_energy_trace(smcx_domain_t *d, int64_t first_sweep, int64_t count, int64_t *dst);
int smcx_domain_stats(smcx_domain_t *d, int64_t *sweeps_done, int64_t *trials, int64_t *accepted);
int smcx_domain_synchronize(smcx_domain_t *d);
int64_t smcx_domain_kernel_launches(smcx_domain_t *d);
/* Eq. 8 from the positive-half counts of the whole lattice (the sum of the slabs'): alpha and ordered pair counts as
 * smcx_sro returns them.  Host arithmetic only. */
int smcx_sro_from_counts(const smcx_params_t *p, const int64_t *half_counts, double *alpha, int64_t *pair_counts);

/* All slabs in one process.  devices: n_domains device ordinals, or NULL = all on p->device (slabs of one GPU; what
 * the tests run).  Slabs on different devices need peer access (NVLink): SMCX_E_CUDA if a device cannot reach its
 * neighbours.  overlap: 0 = a pass is one launch per slab, then the messages are copied; 1 = boundary row first, its message
 * under way while the other rows run (CCO), fused into the boundary-row kernel where the slab's kernel can
 * (smcx_domain_pass_fused), else a copy on a second stream; 2 = as 1 but always by copy.  p->stream orders
 * the group's calls: they fork from it and join it.  p->d_workspace is ignored (the library allocates). */
int smcx_domain_group_create(smcx_domain_group_t **out, const smcx_params_t *p, int32_t n_domains, const int32_t *devices,
                             int32_t overlap);
void smcx_domain_group_destroy(smcx_domain_group_t *g);
smcx_domain_t *smcx_domain_group_member(smcx_domain_group_t *g, int32_t k);   /* borrowed */
int smcx_domain_group_sweep(smcx_domain_group_t *g, int64_t n);               /* asynchronous */
int smcx_domain_group_set_temperature(smcx_domain_group_t *g, int32_t kT_units, const uint32_t *accept, int32_t accept_len);
int smcx_domain_group_set_species(smcx_domain_group_t *g, const uint8_t *host_whole);
int smcx_domain_group_init_composition(smcx_domain_group_t *g, const int64_t *counts);
int smcx_domain_group_set_sweep_counter(smcx_domain_group_t *g, int64_t t);
int smcx_domain_group_species(smcx_domain_group_t *g, uint8_t *host_whole);
int smcx_domain_group_energy(smcx_domain_group_t *g, int64_t *E);             /* recomputed from the slabs' pair counts */
int smcx_domain_group_running_energy(smcx_domain_group_t *g, int64_t *E);
int smcx_domain_group_energy_trace(smcx_domain_group_t *g, int64_t first_sweep, int64_t count, int64_t *dst);
int smcx_domain_group_sro(smcx_domain_group_t *g, double *alpha, int64_t *pair_counts);
int smcx_domain_group_stats(smcx_domain_group_t *g, int64_t *sweeps_done, int64_t *trials, int64_t *accepted);
int smcx_domain_group_synchronize(smcx_domain_group_t *g);
int64_t smcx_domain_group_kernel_launches(smcx_domain_group_t *g);
int64_t smcx_domain_group_message_bytes(smcx_domain_group_t *g);              /* bytes moved between slabs by copies so far */
int64_t smcx_domain_group_fused_messages(smcx_domain_group_t *g);             /* pass messages written by the sweep kernels themselves */

/* ---- Pair counts without any device allocation (a9; Eq. 8; reading S7) ---------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it):
 * the ordered pair counts N_s(p',p) of a lattice the CALLER holds in device memory, with the accumulator of the
 * reduction in a file-scope device array of the library instead of a handle's workspace.  Calls no cudaMalloc,
 * cudaFree or allocating library routine, needs no smcx_t handle, and does not synchronise.
 *   lattice, dims, n_species, n_shells: as in smcx_params_t (dims[a] >= 2; no divisibility requirement).
 *   d_species:      device, N = B * dims[0] * dims[1] * dims[2] bytes, one uint8 species per site in the site order of
 *                   smcx_species (values >= n_species are not checked: undefined counts).  Read only.
 *   d_pair_counts:  device, [n_shells][n_species][n_species] int64, written by the call: the same values smcx_sro
 *                   returns in pair_counts for that lattice (bit-exact: integer counts).
 *   stream:         cudaStream_t the three kernels (clear, count, finish) are enqueued on; NULL = default stream.
 * Limit: n_shells * n_species^2 <= SMCX_STATIC_PAIR_COUNTS_MAX (1024 entries = 8 KB of device memory that every GPU
 * which loads the library holds until the process exits); beyond it SMCX_E_STATIC_SCRATCH (e.g. 5 shells x 16 species).
 * The array is shared by every call on a device and keeps the last call's contents; each call clears it first.  Calls
 * that overlap on one GPU (different streams, threads or processes' worth of streams in one process) RACE on it: issue
 * them on one stream or order them with events.  The device current at the call is the one used; the first call on a
 * device resolves the array's device address (cudaGetSymbolAddress).  Errors: SMCX_E_NULL_ARG, SMCX_E_BAD_LATTICE,
 * SMCX_E_BAD_SPECIES, SMCX_E_BAD_SHELLS, SMCX_E_BAD_DIMS, SMCX_E_STATIC_SCRATCH, SMCX_E_CUDA (launch failure). */
#define SMCX_STATIC_PAIR_COUNTS_MAX 1024
int smcx_pair_counts_static(int32_t lattice, const int32_t *dims, int32_t n_species, int32_t n_shells,
                            const uint8_t *d_species, int64_t *d_pair_counts, void *stream);

const char *smcx_last_error(smcx_t *h); /* text of the last CUDA error seen by this handle */
const char *smcx_strerror(int code);
const char *smcx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SMCX_H_ */
