// SMC-X oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded CPU implementation of the hot path of SMC-X
// (arxiv 2509.20949): Metropolis atom-swap sweeps over a BCC/FCC alloy with an
// effective-pair-interaction (EPI) Hamiltonian, scheduled by dynamic link cells (LC).
// It exists only so that tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference leg can check and time the CUDA path against it.  Nothing under
// paper_2509_20949_b200/ may include, link or call this file, and this file shares no
// code with the CUDA path (its own Philox, geometry, energy, schedule, SRO).
//
// The method is a stochastic iteration, so the oracle follows the algorithm step by step.
// What the paper fixes:
//   Eq. 1-3  PAPER.md:51-63   canonical ensemble, Metropolis acceptance
//   sweep    PAPER.md:65      exactly one trial move per lattice site
//   move     PAPER.md:23      swap of two neighbouring lattice sites
//   LC/LIZ   PAPER.md:71-81   dynamic link cells, every site visited once per step, O(1) trial
//   EPI      PAPER.md:118     pairwise interactions only
//   SRO      PAPER.md:159-163 Warren-Cowley parameter, Eq. 8
//   indexing PAPER.md:165     lattice written nx*ny*nz*basis
// What the paper leaves open (it defers the algorithm to its Ref. 22) is fixed by the
// readings S0-S8 of SURVEY.md 8(c), restated in DESIGN.md "Readings"; each function below
// names the step it follows.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers; shell coordination
// numbers; closed-form energies (single species, B2); dE against full recomputation;
// conservation; energy bookkeeping; order independence of same-colour cells and its failure
// for w=1; exact Boltzmann histogram on 16 sites; B2 SRO values and sum rules.
// Threads: single-threaded unless oracle_set_threads(n > 1) is called; then the cells of one colour
// (which commute, pin P7; the paper's own CPU mapping spreads link cells over OpenMP threads,
// PAPER.md:114) are spread over n OpenMP threads, each with its own tally of trials / accepted / sum dE
// added up after the loop.  Same arithmetic, same order inside a cell; pinned bit for bit against the
// one-thread run (tests/test_oracle_schedule.py).
// Also pinned: the decomposed sweep (S11, slabs with ghost layers) against the undivided one with poison
// outside every slab's window and negative controls (tests/test_oracle_domains.py); the nonlinear local-energy model
// (S12) against a numpy restatement, closed forms, brute-force dE, its linear limit (= twice the EPI
// trajectory) and the exact Boltzmann histogram (tests/test_oracle_local_model.py); replica exchange (S9) against
// rational arithmetic and exact histograms (tests/test_oracle_exchange.py).
// Parity unpinned: the authors' own trajectories and Fig. 6 curves (their EPI values and code are not available,
// PAPER.md:213-217); the paper's qSRO model itself (its Ref. 22: form and weights not available) -- S12 is a model of
// the same kind with synthetic weights, pinned as stated, not the authors'.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <random>
#include <vector>

namespace {

enum { LAT_BCC = 0, LAT_FCC = 1 };
enum { TAG_SHIFT = 1, TAG_TRIAL = 2, TAG_INIT = 3, TAG_SEQ = 5, TAG_EXCHANGE = 6 };

// ---------------------------------------------------------------------------------------
// Philox4x32-10, Salmon, Moraes, Dror, Shaw, SC'11 (reading Q5 / S4).
// ---------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

inline uint32_t mulhi32(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }

struct Vec3 { int x, y, z; };

struct Oracle {
  int lattice = 0;
  int L[3] = {0, 0, 0};      // conventional cells
  int P[3] = {0, 0, 0};      // period in half-lattice units = 2 L
  int B = 0;                 // sites per conventional cell
  int n_species = 0;
  int n_shells = 0;
  int w = 0;                 // link-cell edge in conventional cells
  uint64_t seed = 0;
  int64_t N = 0;
  std::vector<int32_t> epi;             // [s][a][b]
  std::vector<uint32_t> accept;         // threshold table T[d]
  std::vector<std::vector<Vec3>> shell; // offsets per shell, half-lattice units
  std::vector<uint8_t> sigma;           // species per site
  std::vector<uint32_t> visits;         // per-site primary-visit counter (optional)
  bool count_visits = false;
  int64_t sweeps_done = 0;
  int64_t trials = 0;
  int64_t accepted = 0;
  int64_t E_run = 0;
  bool E_valid = false;
  std::vector<int64_t> trace;           // E_run after each sweep, from sweep trace_first on
  int64_t trace_first = 0;              // resume (checkpointing): the sweep counter was set to this value
  int threads = 1;                      // OpenMP threads over the cells of a colour (1 = plain loop)
  mutable int64_t poison_reads = 0;     // S11: species values >= n_species met while evaluating energies
  // S12: nonlinear local-energy model.  model 0: pairwise EPI (S1).  model 1: H = sum_i eps_i with
  // eps_i a quadratic form of the neighbour species counts of site i; `epi` is then its linear part W1[s][a][x]
  // (need not be symmetric) and `quad` its quadratic part W2[s][a][x][y] (entries with x <= y are used).
  int model = 0;
  std::vector<int32_t> quad;
};

constexpr uint8_t kPoison = 255;

// What a run of trials adds to the bookkeeping; one per thread when the cells of a colour are spread
// over threads, summed into the Oracle after the loop.
struct Tally {
  int64_t trials = 0, accepted = 0, dE = 0;
};

// S0: basis positions in half-lattice units.
const int kBasisBCC[2][3] = {{0, 0, 0}, {1, 1, 1}};
const int kBasisFCC[4][3] = {{0, 0, 0}, {0, 1, 1}, {1, 0, 1}, {1, 1, 0}};

inline const int* basis_of(const Oracle& o, int b) {
  return o.lattice == LAT_BCC ? kBasisBCC[b] : kBasisFCC[b];
}

// S0: is the integer vector d (half-lattice units) a lattice translation?
bool is_lattice_vector(int lattice, int dx, int dy, int dz) {
  if (lattice == LAT_BCC) {
    const int px = dx & 1, py = dy & 1, pz = dz & 1;
    return px == py && py == pz;
  }
  return ((dx + dy + dz) & 1) == 0;
}

// S0: shell s = all lattice vectors with the s-th smallest non-zero |d|^2,
// listed in ascending (dz, dy, dx) order.
std::vector<std::vector<Vec3>> make_shells(int lattice, int n_shells) {
  const int R = 8;
  std::vector<int> d2s;
  for (int dz = -R; dz <= R; ++dz)
    for (int dy = -R; dy <= R; ++dy)
      for (int dx = -R; dx <= R; ++dx) {
        if (!(dx | dy | dz)) continue;
        if (!is_lattice_vector(lattice, dx, dy, dz)) continue;
        d2s.push_back(dx * dx + dy * dy + dz * dz);
      }
  std::sort(d2s.begin(), d2s.end());
  d2s.erase(std::unique(d2s.begin(), d2s.end()), d2s.end());
  std::vector<std::vector<Vec3>> out;
  for (int s = 0; s < n_shells; ++s) {
    const int want = d2s[s];
    std::vector<Vec3> v;
    for (int dz = -R; dz <= R; ++dz)
      for (int dy = -R; dy <= R; ++dy)
        for (int dx = -R; dx <= R; ++dx) {
          if (!is_lattice_vector(lattice, dx, dy, dz)) continue;
          if (dx * dx + dy * dy + dz * dz == want) v.push_back({dx, dy, dz});
        }
    out.push_back(v);
  }
  return out;
}

// S0: site id -> position (half-lattice units), and back.
inline void site_to_pos(const Oracle& o, int64_t i, int p[3]) {
  const int b = (int)(i % o.B);
  int64_t c = i / o.B;
  const int x = (int)(c % o.L[0]); c /= o.L[0];
  const int y = (int)(c % o.L[1]); c /= o.L[1];
  const int z = (int)c;
  const int* beta = basis_of(o, b);
  p[0] = 2 * x + beta[0];
  p[1] = 2 * y + beta[1];
  p[2] = 2 * z + beta[2];
}

// v is a site coordinate plus one shell offset, so it lies within one period of [0, period)
// whenever period >= 8; tiny lattices (the 16-site exact test) need the general form.
inline int wrap(int v, int period) {
  if (v >= 0 && v < period) return v;
  v %= period;
  return v < 0 ? v + period : v;
}

inline int64_t pos_to_site(const Oracle& o, int px, int py, int pz) {
  px = wrap(px, o.P[0]); py = wrap(py, o.P[1]); pz = wrap(pz, o.P[2]);
  int b;
  if (o.lattice == LAT_BCC) {
    b = px & 1;
  } else {
    const int par = (px & 1) | ((py & 1) << 1) | ((pz & 1) << 2);
    // (0,0,0)->0  (0,1,1)->1  (1,0,1)->2  (1,1,0)->3
    b = par == 0 ? 0 : par == 6 ? 1 : par == 5 ? 2 : 3;
  }
  const int x = px >> 1, y = py >> 1, z = pz >> 1;
  return (((int64_t)z * o.L[1] + y) * o.L[0] + x) * o.B + b;
}

inline int64_t neighbour(const Oracle& o, int64_t i, const Vec3& d) {
  int p[3];
  site_to_pos(o, i, p);
  return pos_to_site(o, p[0] + d.x, p[1] + d.y, p[2] + d.z);
}

inline int32_t V(const Oracle& o, int s, int a, int b) {
  // kPoison marks sites a slab of the decomposed sweep (S11) does not hold; reading one is a bug of the
  // decomposition (ghost layer too thin, exchange missing), counted and answered with 0
  if (a >= o.n_species || b >= o.n_species) { o.poison_reads++; return 0; }
  return o.epi[((size_t)s * o.n_species + a) * o.n_species + b];
}

// S1: H = sum over shells, sites and the "positive half" O_s^+ of each shell of
// V_s(sigma_i, sigma_{i+d}); every unordered bond once; int64.
bool in_positive_half(const Vec3& d) {
  if (d.z != 0) return d.z > 0;
  if (d.y != 0) return d.y > 0;
  return d.x > 0;
}

int64_t total_energy_local(const Oracle& o);

int64_t total_energy(const Oracle& o) {
  if (o.model == 1) return total_energy_local(o);
  int64_t H = 0;
  for (int s = 0; s < o.n_shells; ++s)
    for (const Vec3& d : o.shell[s]) {
      if (!in_positive_half(d)) continue;
      // an exact integer sum over sites: the threads' partial sums add up to the same H
#pragma omp parallel for reduction(+ : H) schedule(static) num_threads(o.threads) if (o.threads > 1)
      for (int64_t i = 0; i < o.N; ++i) H += V(o, s, o.sigma[i], o.sigma[neighbour(o, i, d)]);
    }
  return H;
}

// ---------------------------------------------------------------------------------------
// S12: a general nonlinear short-range model.  PAPER.md:118: "the qSRO model represents a general nonlinear
// short-range model, where the local energies of all lattice sites within LIZ are calculated to determine the
// energy change due to a MC move"; the model itself is the paper's Ref. 22 and its weights are not available.
// Reading S12: the energy is a sum of local energies, H = sum_i eps(sigma_i, n_i), where
// n_i[s][x] = number of neighbours of species x in shell s of site i (the local short-range order of the site) and
//   eps(a, n) = sum_s ( sum_x W1[s][a][x] n[s][x]  +  sum_{x <= y} W2[s][a][x][y] n[s][x] n[s][y] ),
// int32 weights, int64 energies.  The quadratic part couples pairs of neighbours of a site (three-body terms):
// it cannot be written as a pair interaction.  With W2 = 0 and W1 = V symmetric the model is twice the EPI
// Hamiltonian (every bond is seen from both ends).  A swap of i and j changes the own species of i and j and the
// counts of every site that has i or j as a neighbour: dE is the sum, over that set U = {i, j} + N(i) + N(j), of
// the local energies after the swap minus before -- evaluated here exactly that way, site by site from scratch.
// ---------------------------------------------------------------------------------------
int64_t site_energy(const Oracle& o, int64_t k) {
  const int n = o.n_species;
  const int a = o.sigma[k];
  if (a >= n) { o.poison_reads++; return 0; }
  int64_t e = 0;
  std::vector<int64_t> cnt((size_t)n);
  for (int s = 0; s < o.n_shells; ++s) {
    std::fill(cnt.begin(), cnt.end(), (int64_t)0);
    for (const Vec3& d : o.shell[s]) {
      const int x = o.sigma[neighbour(o, k, d)];
      if (x >= n) { o.poison_reads++; continue; }
      cnt[(size_t)x]++;
    }
    for (int x = 0; x < n; ++x) {
      e += (int64_t)o.epi[((size_t)s * n + a) * n + x] * cnt[(size_t)x];
      for (int y = x; y < n; ++y)
        e += (int64_t)o.quad[(((size_t)s * n + a) * n + x) * n + y] * cnt[(size_t)x] * cnt[(size_t)y];
    }
  }
  return e;
}

int64_t total_energy_local(const Oracle& o) {
  int64_t H = 0;
#pragma omp parallel for reduction(+ : H) schedule(static) num_threads(o.threads) if (o.threads > 1)
  for (int64_t k = 0; k < o.N; ++k) H += site_energy(o, k);
  return H;
}

// the sites whose local energy a swap of i and j can change, each once
void affected_sites(const Oracle& o, int64_t i, int64_t j, std::vector<int64_t>& U) {
  U.clear();
  U.push_back(i);
  U.push_back(j);
  for (int s = 0; s < o.n_shells; ++s)
    for (const Vec3& d : o.shell[s]) {
      // k has i as a neighbour at offset d  <=>  k = i - d; the shells are symmetric, so this is N(i) itself
      U.push_back(neighbour(o, i, d));
      U.push_back(neighbour(o, j, d));
    }
  std::sort(U.begin(), U.end());
  U.erase(std::unique(U.begin(), U.end()), U.end());
}

int64_t swap_delta_local(Oracle& o, int64_t i, int64_t j) {
  static thread_local std::vector<int64_t> U;
  affected_sites(o, i, j, U);
  int64_t before = 0, after = 0;
  for (int64_t k : U) before += site_energy(o, k);
  std::swap(o.sigma[i], o.sigma[j]);
  for (int64_t k : U) after += site_energy(o, k);
  std::swap(o.sigma[i], o.sigma[j]);
  return after - before;
}

// S1: the sites bonded to i and to j (one entry per shell offset, shells in order), with
// the i-j bond(s) kept on i's side only: an entry of nbr_j that is i itself is marked -1.
struct Bonds {
  std::vector<int64_t> nbr_i, nbr_j;
};

void collect_bonds(const Oracle& o, int64_t i, int64_t j, Bonds& bonds) {
  int pi[3], pj[3];
  site_to_pos(o, i, pi);
  site_to_pos(o, j, pj);
  bonds.nbr_i.clear();
  bonds.nbr_j.clear();
  for (int s = 0; s < o.n_shells; ++s)
    for (const Vec3& d : o.shell[s]) {
      bonds.nbr_i.push_back(pos_to_site(o, pi[0] + d.x, pi[1] + d.y, pi[2] + d.z));
      const int64_t n = pos_to_site(o, pj[0] + d.x, pj[1] + d.y, pj[2] + d.z);
      bonds.nbr_j.push_back(n == i ? -1 : n);  // that bond is counted from i's side
    }
}

// S1: energy of all bonds touching i or j (the i-j bond(s) counted once), as it stands.
int64_t local_energy(const Oracle& o, int64_t i, int64_t j, const Bonds& bonds) {
  int64_t e = 0;
  size_t k = 0;
  for (int s = 0; s < o.n_shells; ++s)
    for (size_t m = 0; m < o.shell[s].size(); ++m, ++k) {
      e += V(o, s, o.sigma[i], o.sigma[bonds.nbr_i[k]]);
      if (bonds.nbr_j[k] >= 0) e += V(o, s, o.sigma[j], o.sigma[bonds.nbr_j[k]]);
    }
  return e;
}

// S1: dE of swapping sigma_i and sigma_j = H(sigma') - H(sigma), the plain way:
// local energy after the swap minus before.  The state is left unchanged.
int64_t swap_delta(Oracle& o, int64_t i, int64_t j) {
  if (o.model == 1) return swap_delta_local(o, i, j);
  static thread_local Bonds bonds;
  collect_bonds(o, i, j, bonds);
  const int64_t before = local_energy(o, i, j, bonds);
  std::swap(o.sigma[i], o.sigma[j]);
  const int64_t after = local_energy(o, i, j, bonds);
  std::swap(o.sigma[i], o.sigma[j]);
  return after - before;
}

// S4: one trial with primary site i, direction word w_dir and acceptance word u.
void trial(Oracle& o, Tally& tally, int64_t i, uint32_t w_dir, uint32_t u) {
  const std::vector<Vec3>& nn = o.shell[0];
  const uint32_t dir = mulhi32(w_dir, (uint32_t)nn.size());
  const int64_t j = neighbour(o, i, nn[dir]);
  tally.trials++;
  if (o.count_visits) o.visits[i]++;
  const uint8_t a = o.sigma[i], b = o.sigma[j];
  if (a == b) return;  // Q8: same species, nothing changes
  const int64_t dE = swap_delta(o, i, j);
  // Eq. 3 in integer form (S5): P=1 for dE<=0, else u < T[dE].
  const bool ok = dE <= 0 || (dE < (int64_t)o.accept.size() && u < o.accept[(size_t)dE]);
  if (ok) {
    std::swap(o.sigma[i], o.sigma[j]);
    tally.dE += dE;
    tally.accepted++;
  }
}

void add_tally(Oracle& o, const Tally& tally) {
  o.trials += tally.trials;
  o.accepted += tally.accepted;
  o.E_run += tally.dE;
}

void ensure_energy(Oracle& o) {
  if (!o.E_valid) {
    o.E_run = total_energy(o);
    o.E_valid = true;
  }
}

// S3.2 + S4: the S = w^3 B trials of one link cell, slot by slot.
void run_cell(Oracle& o, Tally& tally, uint32_t cell_id, int colour, uint32_t t, int ox, int oy, int oz) {
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const int w = o.w;
  const int ncx = o.L[0] / w, ncy = o.L[1] / w;
  const int S = w * w * w * o.B;
  const int cx = (int)(cell_id % (uint32_t)ncx);
  const int cy = (int)((cell_id / (uint32_t)ncx) % (uint32_t)ncy);
  const int cz = (int)(cell_id / (uint32_t)(ncx * ncy));
  uint32_t r[4];
  for (int k = 0; k < S; ++k) {
    // S3.2: slot k -> local site ((lz*w + ly)*w + lx)*B + b.
    const int b = k % o.B;
    int rest = k / o.B;
    const int lx = rest % w; rest /= w;
    const int ly = rest % w; rest /= w;
    const int lz = rest;
    const int x = (ox + cx * w + lx) % o.L[0];
    const int y = (oy + cy * w + ly) % o.L[1];
    const int z = (oz + cz * w + lz) % o.L[2];
    const int64_t i = (((int64_t)z * o.L[1] + y) * o.L[0] + x) * o.B + b;
    // S4: one Philox call serves two consecutive slots.
    const uint32_t q = (uint32_t)(k >> 1);
    const uint32_t ct[4] = {cell_id, q, t, (uint32_t)TAG_TRIAL | ((uint32_t)colour << 8)};
    philox4x32_10(ct, key, r);
    if (k & 1) trial(o, tally, i, r[2], r[3]);
    else       trial(o, tally, i, r[0], r[1]);
  }
}

// S3 + S4: one link-cell sweep.  order_mode: 0 = cells in ascending id, 1 = descending,
// 2 = shuffled with std::mt19937(order_seed) (test-only; results must not depend on it).
void sweep_lc(Oracle& o, int order_mode, uint32_t order_seed) {
  ensure_energy(o);
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const uint32_t t = (uint32_t)o.sweeps_done;
  const int w = o.w;
  // S3.1: link-cell grid origin for this sweep.
  const uint32_t cs[4] = {0u, 0u, t, (uint32_t)TAG_SHIFT};
  uint32_t r[4];
  philox4x32_10(cs, key, r);
  const int ox = (int)mulhi32(r[0], (uint32_t)w);
  const int oy = (int)mulhi32(r[1], (uint32_t)w);
  const int oz = (int)mulhi32(r[2], (uint32_t)w);
  const int ncx = o.L[0] / w, ncy = o.L[1] / w, ncz = o.L[2] / w;
  std::vector<uint32_t> cells;
  for (int colour = 0; colour < 8; ++colour) {
    // S2: cells of this colour.
    cells.clear();
    for (int cz = 0; cz < ncz; ++cz)
      for (int cy = 0; cy < ncy; ++cy)
        for (int cx = 0; cx < ncx; ++cx)
          if (((cx & 1) | ((cy & 1) << 1) | ((cz & 1) << 2)) == colour)
            cells.push_back((uint32_t)((cz * ncy + cy) * ncx + cx));
    if (order_mode == 1) std::reverse(cells.begin(), cells.end());
    if (order_mode == 2) {
      std::mt19937 g(order_seed + (uint32_t)colour + 8u * t);
      std::shuffle(cells.begin(), cells.end(), g);
    }
    // The cells of one colour, in the order of `cells`: a plain loop, or spread over o.threads OpenMP
    // threads (same-colour cells touch disjoint sites, S2, so they commute: pin P7).
    Tally total;
    const int64_t n_cells = (int64_t)cells.size();
    if (o.threads <= 1) {
      for (int64_t c = 0; c < n_cells; ++c) run_cell(o, total, cells[(size_t)c], colour, t, ox, oy, oz);
    } else {
#ifdef _OPENMP
#pragma omp parallel num_threads(o.threads)
      {
        Tally mine;
#pragma omp for schedule(static)
        for (int64_t c = 0; c < n_cells; ++c) run_cell(o, mine, cells[(size_t)c], colour, t, ox, oy, oz);
#pragma omp critical
        { total.trials += mine.trials; total.accepted += mine.accepted; total.dE += mine.dE; }
      }
#else
      for (int64_t c = 0; c < n_cells; ++c) run_cell(o, total, cells[(size_t)c], colour, t, ox, oy, oz);
#endif
    }
    add_tally(o, total);
  }
  // S3.3
  o.trace.push_back(o.E_run);
  o.sweeps_done++;
}

// ---------------------------------------------------------------------------------------
// S11: lattice parallelism (section "Distributed SMC-X": "the complete lattice is
// partitioned across multiple GPUs, with a ghost layer used to exchange boundary information between
// neighboring sublattices", Fig. 2; scaling and computation-communication overlap PAPER.md:147).
// The paper gives no protocol.  Reading S11: the lattice is cut into D slabs along z on
// boundaries of PAIRS of link-cell rows (so the colour of a row does not depend on the slab):
//   pairs = (Lz / w) / 2;  slab k owns pairs/D + (k < pairs mod D) consecutive row pairs.
// A slab owns link cells, not layers: in sweep t with origin oz its rows [r0, r1) cover the layers
// [a, b) = [oz + r0 w, oz + r1 w) (mod Lz) and it holds a copy of the window [a - g, b + g), g = ghost
// layers (conventional cells).  Every trial draws its random numbers from the GLOBAL cell id, slot, sweep
// and colour (S4), so a decomposed sweep must reproduce the undivided one bit for bit; what the protocol
// has to get right is only which copies are refreshed when:
//   start of sweep t:  the window moves by oz(t) - oz(t-1); the layers that enter it are fetched from the
//                      neighbour on that side (whose old window held them up to date);
//   after colour pass c (rows of parity pz = (c >> 2) & 1 were active): a slab's bottom row (pz = 0)
//                      modified layers [a - wr, a + w + wr), wr = layers a swap partner can lie outside its
//                      cell = ceil(r0 / 2); the part inside the lower neighbour's window, [a - wr, a + g),
//                      is sent down.  For pz = 1 the top row sends [b - g, b + wr) up.  One message per slab
//                      and pass; no other row reaches a neighbour's window.
// The implementation below keeps one full-size array per slab in which everything outside the slab's window is
// kPoison, runs the slabs in a shuffled order inside every pass (they must commute), copies exactly the layers
// named above, and counts reads of poisoned sites.  It is pinned against the undivided sweep (tests/
// test_oracle_domains.py): equal arrays / traces / statistics and zero poison reads for g = H; poison reads or
// different arrays for a thinner ghost layer or without the exchanges.
// ---------------------------------------------------------------------------------------
struct Slab {
  int row_first = 0, row_count = 0;
  std::vector<uint8_t> sig;     // N bytes; valid inside the window only
};

std::vector<Slab> slab_partition(const Oracle& o, int D) {
  const int pairs = o.L[2] / o.w / 2;
  std::vector<Slab> slabs((size_t)D);
  int row = 0;
  for (int k = 0; k < D; ++k) {
    slabs[k].row_first = row;
    slabs[k].row_count = 2 * (pairs / D + (k < pairs % D ? 1 : 0));
    row += slabs[k].row_count;
  }
  return slabs;
}

inline int64_t layer_sites(const Oracle& o) { return (int64_t)o.L[0] * o.L[1] * o.B; }

// copy `count` layers starting at global layer z0 (any integer; taken mod Lz) from src to dst
void copy_layers(const Oracle& o, const std::vector<uint8_t>& src, std::vector<uint8_t>& dst, int z0, int count) {
  const int64_t ls = layer_sites(o);
  for (int k = 0; k < count; ++k) {
    const int z = wrap(z0 + k, o.L[2]);
    std::memcpy(dst.data() + (size_t)z * ls, src.data() + (size_t)z * ls, (size_t)ls);
  }
}

// everything outside the window [lo, lo + count) of the slab becomes kPoison
void poison_outside(const Oracle& o, Slab& s, int lo, int count) {
  const int64_t ls = layer_sites(o);
  std::vector<char> keep((size_t)o.L[2], 0);
  for (int k = 0; k < count; ++k) keep[(size_t)wrap(lo + k, o.L[2])] = 1;
  for (int z = 0; z < o.L[2]; ++z)
    if (!keep[(size_t)z]) std::memset(s.sig.data() + (size_t)z * ls, kPoison, (size_t)ls);
}

void shift_origin(const Oracle& o, uint32_t t, int& ox, int& oy, int& oz) {
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const uint32_t cs[4] = {0u, 0u, t, (uint32_t)TAG_SHIFT};
  uint32_t r[4];
  philox4x32_10(cs, key, r);
  ox = (int)mulhi32(r[0], (uint32_t)o.w);
  oy = (int)mulhi32(r[1], (uint32_t)o.w);
  oz = (int)mulhi32(r[2], (uint32_t)o.w);
}

// n sweeps of the state in o.sigma, decomposed into D slabs with `ghost` ghost layers; `exchange` = false leaves
// the per-pass messages out (negative control).  The result is gathered back into o.sigma.  Returns the
// number of poisoned reads, or -1 if the lattice cannot be cut into D slabs.
int64_t sweep_lc_slabs(Oracle& o, int64_t n, int D, int ghost, bool exchange, uint32_t order_seed) {
  const int w = o.w;
  if (D < 2 || o.L[2] % (2 * w) || D > o.L[2] / w / 2 || ghost < 0) return -1;
  ensure_energy(o);
  int r0_reach = 0;
  for (const Vec3& d : o.shell[0]) r0_reach = std::max(r0_reach, std::max(std::abs(d.x), std::max(std::abs(d.y), std::abs(d.z))));
  const int wr = (r0_reach + 1) / 2;
  std::vector<Slab> slabs = slab_partition(o, D);
  const int ncx = o.L[0] / w, ncy = o.L[1] / w;
  o.poison_reads = 0;
  if (n <= 0) return 0;
  int ox = 0, oy = 0, oz = 0, oz_prev = 0;
  std::mt19937 order_rng(order_seed);
  for (int64_t step = 0; step < n; ++step) {
    const uint32_t t = (uint32_t)o.sweeps_done;
    shift_origin(o, t, ox, oy, oz);
    if (step == 0) {
      // scatter: every slab gets its window of the first sweep and nothing else
      for (Slab& s : slabs) {
        s.sig = o.sigma;
        poison_outside(o, s, oz + s.row_first * w - ghost, s.row_count * w + 2 * ghost);
      }
    } else if (oz != oz_prev) {
      // the windows move by oz - oz_prev layers: fetch what enters them from the neighbour on that side
      const int sh = oz - oz_prev;
      for (int k = 0; k < D; ++k) {
        Slab& s = slabs[(size_t)k];
        const int a_old = oz_prev + s.row_first * w, b_old = a_old + s.row_count * w;
        if (sh > 0) copy_layers(o, slabs[(size_t)((k + 1) % D)].sig, s.sig, b_old + ghost, sh);
        else        copy_layers(o, slabs[(size_t)((k + D - 1) % D)].sig, s.sig, a_old - ghost + sh, -sh);
      }
      for (Slab& s : slabs) poison_outside(o, s, oz + s.row_first * w - ghost, s.row_count * w + 2 * ghost);
    }
    oz_prev = oz;
    for (int colour = 0; colour < 8; ++colour) {
      const int pz = (colour >> 2) & 1;
      std::vector<int> order((size_t)D);
      for (int k = 0; k < D; ++k) order[(size_t)k] = k;
      std::shuffle(order.begin(), order.end(), order_rng);
      Tally total;
      for (int k : order) {
        Slab& s = slabs[(size_t)k];
        std::swap(o.sigma, s.sig);               // the slab's private copy is the lattice while its cells run
        for (int cz = s.row_first; cz < s.row_first + s.row_count; ++cz)
          for (int cy = 0; cy < ncy; ++cy)
            for (int cx = 0; cx < ncx; ++cx)
              if (((cx & 1) | ((cy & 1) << 1) | ((cz & 1) << 2)) == colour)
                run_cell(o, total, (uint32_t)((cz * ncy + cy) * ncx + cx), colour, t, ox, oy, oz);
        std::swap(o.sigma, s.sig);
      }
      add_tally(o, total);
      if (!exchange) continue;
      // one message per slab: the active boundary row's modified layers that lie in the neighbour's window
      for (int k = 0; k < D; ++k) {
        const Slab& s = slabs[(size_t)k];
        const int a = oz + s.row_first * w, b = a + s.row_count * w;
        if (pz == 0) copy_layers(o, s.sig, slabs[(size_t)((k + D - 1) % D)].sig, a - wr, wr + ghost);
        else         copy_layers(o, s.sig, slabs[(size_t)((k + 1) % D)].sig, b - ghost, ghost + wr);
      }
    }
    o.trace.push_back(o.E_run);
    o.sweeps_done++;
  }
  // gather: every layer from the slab whose rows cover it under the last origin
  for (const Slab& s : slabs) copy_layers(o, s.sig, o.sigma, oz + s.row_first * w, s.row_count * w);
  return o.poison_reads;
}

// S8: plain single-site-sequential Metropolis (no link cells); used for the exact
// Boltzmann test and as the ensemble reference for the LC schedule.
void sweep_seq(Oracle& o) {
  ensure_energy(o);
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const uint32_t t = (uint32_t)o.sweeps_done;
  uint32_t r[4];
  Tally tally;
  for (int64_t i = 0; i < o.N; ++i) {
    const uint32_t ct[4] = {(uint32_t)((uint64_t)i & 0xffffffffu), (uint32_t)((uint64_t)i >> 32), t,
                            (uint32_t)TAG_SEQ};
    philox4x32_10(ct, key, r);
    trial(o, tally, i, r[0], r[1]);
  }
  add_tally(o, tally);
  o.trace.push_back(o.E_run);
  o.sweeps_done++;
}

// S6: seeded bijection of [0,N): 4-round balanced Feistel network over 2h bits with
// cycle walking; sigma_i = pi(i) mod n_species, so the species counts are exactly
// floor(N/n) + (p < N mod n).
uint64_t feistel_permute(const Oracle& o, uint64_t v, int h) {
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const uint64_t mask = (1ull << h) - 1ull;
  do {
    uint64_t left = v >> h, right = v & mask;
    for (uint32_t round = 0; round < 4; ++round) {
      const uint32_t ct[4] = {(uint32_t)right, round, 0u, (uint32_t)TAG_INIT};
      uint32_t r[4];
      philox4x32_10(ct, key, r);
      const uint64_t f = (uint64_t)r[0] & mask;
      const uint64_t new_right = left ^ f;
      left = right;
      right = new_right;
    }
    v = (left << h) | right;
  } while (v >= (uint64_t)o.N);
  return v;
}

void init_species(Oracle& o) {
  int h = 1;
  while ((1ull << (2 * h)) < (uint64_t)o.N) ++h;
#pragma omp parallel for schedule(static) num_threads(o.threads) if (o.threads > 1)   // sites are independent
  for (int64_t i = 0; i < o.N; ++i)
    o.sigma[i] = (uint8_t)(feistel_permute(o, (uint64_t)i, h) % (uint64_t)o.n_species);
  o.E_valid = false;
}

// S10: a given composition (the paper's alloy is Fe29Co29Ni28Al7Ti7, not
// equiatomic): counts n_0..n_{n-1} with sum N; sigma_i = p for cum_p <= pi(i) < cum_{p+1}, cum_p =
// n_0 + ... + n_{p-1}, pi the permutation of S6.  Exactly n_p sites of species p, placed uniformly
// at random.  Returns false (state unchanged) if the counts do not sum to N or one is negative.
bool init_composition(Oracle& o, const int64_t* counts) {
  int64_t sum = 0;
  for (int p = 0; p < o.n_species; ++p) {
    if (counts[p] < 0) return false;
    sum += counts[p];
  }
  if (sum != o.N) return false;
  int h = 1;
  while ((1ull << (2 * h)) < (uint64_t)o.N) ++h;
#pragma omp parallel for schedule(static) num_threads(o.threads) if (o.threads > 1)   // sites are independent
  for (int64_t i = 0; i < o.N; ++i) {
    const int64_t r = (int64_t)feistel_permute(o, (uint64_t)i, h);
    int p = 0;
    int64_t cum = counts[0];
    while (r >= cum) cum += counts[++p];
    o.sigma[i] = (uint8_t)p;
  }
  o.E_valid = false;
  return true;
}

// S7: ordered pair counts N_s(p',p) = sum_i [sigma_i=p'] sum_{d in O_s} [sigma_{i+d}=p].
void pair_counts(const Oracle& o, int64_t* counts) {
  const int n = o.n_species;
  std::fill(counts, counts + (size_t)o.n_shells * n * n, (int64_t)0);
  for (int s = 0; s < o.n_shells; ++s)
    for (const Vec3& d : o.shell[s]) {
      int64_t* row = counts + (size_t)s * n * n;
      // exact integer histogram: per-thread copies of the n x n counters are added up by the reduction
#pragma omp parallel for reduction(+ : row[: n * n]) schedule(static) num_threads(o.threads) if (o.threads > 1)
      for (int64_t i = 0; i < o.N; ++i) {
        const int pc = o.sigma[i];
        const int pn = o.sigma[neighbour(o, i, d)];
        row[(size_t)pc * n + pn]++;
      }
    }
}

// Eq. 8: alpha_s^{pp'} = 1 - P_s(p | p') / c_p with
// P_s(p|p') = N_s(p',p) / (Z_s n_{p'}) and c_p = n_p / N.  Stored at [s][p'][p].
void sro(const Oracle& o, const int64_t* counts, double* alpha) {
  const int n = o.n_species;
  std::vector<int64_t> n_of(n, 0);
  for (int64_t i = 0; i < o.N; ++i) n_of[o.sigma[i]]++;
  for (int s = 0; s < o.n_shells; ++s) {
    const double Z = (double)o.shell[s].size();
    for (int pc = 0; pc < n; ++pc)
      for (int pn = 0; pn < n; ++pn) {
        const size_t idx = ((size_t)s * n + pc) * n + pn;
        if (n_of[pc] == 0 || n_of[pn] == 0) {
          alpha[idx] = std::numeric_limits<double>::quiet_NaN();
          continue;
        }
        const double P = (double)counts[idx] / (Z * (double)n_of[pc]);
        const double c = (double)n_of[pn] / (double)o.N;
        alpha[idx] = 1.0 - P / c;
      }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------
// C entry points for the ctypes wrapper in oracle/__init__.py.
// ---------------------------------------------------------------------------------------
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  philox4x32_10(ctr, key, out);
}

// ---------------------------------------------------------------------------------------
// S9 replica exchange (parallel tempering), Eq. 5-6, PAPER.md:89-97:
//   P_swap = min(1, exp(Delta)),  Delta = (1/kT_i - 1/kT_j)(E_i - E_j).
// Energies are the integer H (0.1 meV), temperatures kT in the same units, so Delta is a pure
// number.  Integer form of the decision, like Eq. 3: accept iff Delta >= 0 or u < T, with
//   Delta = (double)(kT_j - kT_i) * (double)(E_i - E_j) / ((double)kT_i * (double)kT_j),
//   T = min(floor(exp(Delta) * 2^32), 2^32 - 1), u a 32-bit Philox word.
// ---------------------------------------------------------------------------------------
double oracle_exchange_delta(int64_t E_i, int64_t E_j, int32_t kT_i, int32_t kT_j) {
  const double a = (double)(kT_j - kT_i);
  const double c = (double)(E_i - E_j);
  const double b = (double)kT_i * (double)kT_j;
  return a * c / b;
}

int oracle_exchange_accept(int64_t E_i, int64_t E_j, int32_t kT_i, int32_t kT_j, uint32_t u) {
  const double delta = oracle_exchange_delta(E_i, E_j, kT_i, kT_j);
  if (delta >= 0.0) return 1;
  const double x = std::exp(delta) * 4294967296.0;
  const uint32_t T = x >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)std::floor(x);
  return u < T ? 1 : 0;
}

// The draw of the exchange attempt between temperature slots p and p + 1 in round r:
// philox(ctr = (p, r_hi, r_lo, TAG_EXCHANGE), key = seed)[0].
uint32_t oracle_exchange_draw(uint64_t seed, uint64_t round, uint32_t p) {
  const uint32_t ctr[4] = {p, (uint32_t)(round >> 32), (uint32_t)(round & 0xffffffffull), (uint32_t)TAG_EXCHANGE};
  const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32)};
  uint32_t out[4];
  philox4x32_10(ctr, key, out);
  return out[0];
}

// Writes up to max_out offsets (dx,dy,dz triples) of shell s; returns the shell size.
int oracle_shell(int lattice, int s, int* out_xyz, int max_out) {
  std::vector<std::vector<Vec3>> sh = make_shells(lattice, s + 1);
  const std::vector<Vec3>& v = sh[s];
  for (int k = 0; k < (int)v.size() && k < max_out; ++k) {
    out_xyz[3 * k + 0] = v[k].x;
    out_xyz[3 * k + 1] = v[k].y;
    out_xyz[3 * k + 2] = v[k].z;
  }
  return (int)v.size();
}

void* oracle_create(int lattice, const int* dims, int n_species, int n_shells, const int32_t* epi,
                    int link_cell, const uint32_t* accept, int accept_len, uint64_t seed) {
  if (lattice != LAT_BCC && lattice != LAT_FCC) return nullptr;
  if (n_species < 1 || n_species > 255 || n_shells < 1 || n_shells > 8) return nullptr;
  for (int a = 0; a < 3; ++a)
    if (dims[a] < 2) return nullptr;  // L=1 would make a 2nd-shell offset a self-bond
  Oracle* o = new Oracle();
  o->lattice = lattice;
  o->B = lattice == LAT_BCC ? 2 : 4;
  for (int a = 0; a < 3; ++a) { o->L[a] = dims[a]; o->P[a] = 2 * dims[a]; }
  o->N = (int64_t)dims[0] * dims[1] * dims[2] * o->B;
  o->n_species = n_species;
  o->n_shells = n_shells;
  o->epi.assign(epi, epi + (size_t)n_shells * n_species * n_species);
  o->w = link_cell;
  o->accept.assign(accept, accept + accept_len);
  o->seed = seed;
  o->shell = make_shells(lattice, n_shells);
  o->sigma.assign((size_t)o->N, 0);
  return o;
}

void oracle_destroy(void* h) { delete (Oracle*)h; }

// S12: switch the handle to the nonlinear local-energy model.  quad = W2[s][a][x][y], n_shells n^3 entries (x <= y
// used); the table given at creation becomes the linear part W1[s][a][x].  quad == NULL: back to pairwise EPI.
void oracle_set_local_model(void* h, const int32_t* quad) {
  Oracle& o = *(Oracle*)h;
  if (!quad) { o.model = 0; o.quad.clear(); }
  else {
    o.model = 1;
    o.quad.assign(quad, quad + (size_t)o.n_shells * o.n_species * o.n_species * o.n_species);
  }
  o.E_valid = false;
}

int64_t oracle_site_energy(void* h, int64_t k) {
  Oracle& o = *(Oracle*)h;
  return o.model == 1 ? site_energy(o, k) : 0;
}

int64_t oracle_n_sites(void* h) { return ((Oracle*)h)->N; }

void oracle_init_species(void* h) { init_species(*(Oracle*)h); }

int oracle_init_composition(void* h, const int64_t* counts) { return init_composition(*(Oracle*)h, counts) ? 0 : -1; }

// pi(i) itself, for the bijection pin.
uint64_t oracle_init_permutation(void* h, uint64_t i) {
  Oracle& o = *(Oracle*)h;
  int hh = 1;
  while ((1ull << (2 * hh)) < (uint64_t)o.N) ++hh;
  return feistel_permute(o, i, hh);
}

int oracle_set_species(void* h, const uint8_t* src) {
  Oracle& o = *(Oracle*)h;
  for (int64_t i = 0; i < o.N; ++i)
    if (src[i] >= o.n_species) return -1;
  std::memcpy(o.sigma.data(), src, (size_t)o.N);
  o.E_valid = false;
  return 0;
}

void oracle_get_species(void* h, uint8_t* dst) {
  Oracle& o = *(Oracle*)h;
  std::memcpy(dst, o.sigma.data(), (size_t)o.N);
}

void oracle_set_temperature(void* h, const uint32_t* accept, int accept_len) {
  ((Oracle*)h)->accept.assign(accept, accept + accept_len);
}

int64_t oracle_energy(void* h) { return total_energy(*(Oracle*)h); }

int64_t oracle_running_energy(void* h) {
  Oracle& o = *(Oracle*)h;
  ensure_energy(o);
  return o.E_run;
}

int64_t oracle_neighbour(void* h, int64_t i, int s, int k) {
  Oracle& o = *(Oracle*)h;
  return neighbour(o, i, o.shell[s][k]);
}

// dE of swapping site i with its shell-0 neighbour number dir (state unchanged).
int64_t oracle_delta_e(void* h, int64_t i, int dir) {
  Oracle& o = *(Oracle*)h;
  const int64_t j = neighbour(o, i, o.shell[0][dir]);
  return swap_delta(o, i, j);
}

int oracle_lc_valid(void* h) {
  // S2: 2w >= 2 r0 + R (per-axis reaches in half-lattice units; w in conventional cells
  // = 2 half-units), and every dimension divisible by 2w.
  Oracle& o = *(Oracle*)h;
  if (o.w < 1) return 0;
  for (int a = 0; a < 3; ++a)
    if (o.L[a] % (2 * o.w)) return 0;
  int r0 = 0, R = 0;
  for (int s = 0; s < o.n_shells; ++s)
    for (const Vec3& d : o.shell[s]) {
      const int m = std::max(std::abs(d.x), std::max(std::abs(d.y), std::abs(d.z)));
      if (s == 0) r0 = std::max(r0, m);
      R = std::max(R, m);
    }
  // S12: a trial of the local model reads the neighbours of the neighbours of i and j: reach r0 + 2 R
  return 2 * o.w >= 2 * r0 + (o.model == 1 ? 2 * R : R) ? 1 : 0;
}

// n link-cell sweeps.  The caller is responsible for oracle_lc_valid(); an invalid w is
// allowed on purpose so that a test can show the order dependence it causes.
int oracle_sweep_lc(void* h, int64_t n, int order_mode, uint32_t order_seed) {
  Oracle& o = *(Oracle*)h;
  if (o.w < 1) return -1;
  for (int a = 0; a < 3; ++a)
    if (o.L[a] % (2 * o.w)) return -1;
  for (int64_t s = 0; s < n; ++s) sweep_lc(o, order_mode, order_seed);
  return 0;
}

// Threads over the cells of a colour for the following oracle_sweep_lc calls (1 = plain loop).  Returns
// the number that will be used: 1 when the library was built without OpenMP.
int oracle_set_threads(void* h, int n) {
  Oracle& o = *(Oracle*)h;
#ifdef _OPENMP
  o.threads = n < 1 ? 1 : n;
#else
  (void)n;
  o.threads = 1;
#endif
  return o.threads;
}

// S11: n link-cell sweeps with the lattice cut into D slabs along z (ghost layers, exchanges after every colour
// pass).  Returns the number of reads of sites a slab did not hold (0 for a correct protocol), -1 if the
// lattice cannot be cut that way.
int64_t oracle_sweep_lc_slabs(void* h, int64_t n, int D, int ghost, int exchange, uint32_t order_seed) {
  return sweep_lc_slabs(*(Oracle*)h, n, D, ghost, exchange != 0, order_seed);
}

// The slab partition itself: rows[2 k] = first link-cell row of slab k, rows[2 k + 1] = its number of rows.
int oracle_slab_partition(void* h, int D, int* rows) {
  Oracle& o = *(Oracle*)h;
  if (D < 1 || o.L[2] % (2 * o.w) || D > o.L[2] / o.w / 2) return -1;
  const std::vector<Slab> slabs = slab_partition(o, D);
  for (int k = 0; k < D; ++k) { rows[2 * k] = slabs[(size_t)k].row_first; rows[2 * k + 1] = slabs[(size_t)k].row_count; }
  return 0;
}

void oracle_sweep_seq(void* h, int64_t n) {
  Oracle& o = *(Oracle*)h;
  for (int64_t s = 0; s < n; ++s) sweep_seq(o);
}

// The link-cell origin S3.1 draws for sweep t.
void oracle_shift(void* h, uint32_t t, int* oxyz) {
  Oracle& o = *(Oracle*)h;
  const uint32_t key[2] = {(uint32_t)(o.seed & 0xffffffffu), (uint32_t)(o.seed >> 32)};
  const uint32_t cs[4] = {0u, 0u, t, (uint32_t)TAG_SHIFT};
  uint32_t r[4];
  philox4x32_10(cs, key, r);
  for (int a = 0; a < 3; ++a) oxyz[a] = (int)mulhi32(r[a], (uint32_t)o.w);
}

void oracle_stats(void* h, int64_t* sweeps, int64_t* trials, int64_t* accepted) {
  Oracle& o = *(Oracle*)h;
  *sweeps = o.sweeps_done; *trials = o.trials; *accepted = o.accepted;
}

// Resume from a checkpoint (state = species array, sweep counter, seed; the RNG is counter-based, so the
// continuation is exact): the next sweep is sweep t.  The trace restarts there.
int oracle_set_sweep_counter(void* h, int64_t t) {
  Oracle& o = *(Oracle*)h;
  if (t < 0 || t > 0xffffffffll) return -1;
  o.sweeps_done = t;
  o.trials = t * o.N;
  o.trace.clear();
  o.trace_first = t;
  return 0;
}

int64_t oracle_trace(void* h, int64_t first, int64_t count, int64_t* dst) {
  Oracle& o = *(Oracle*)h;
  if (first < o.trace_first || first - o.trace_first + count > (int64_t)o.trace.size()) return -1;
  for (int64_t k = 0; k < count; ++k) dst[k] = o.trace[(size_t)(first - o.trace_first + k)];
  return count;
}

void oracle_count_visits(void* h, int on) {
  Oracle& o = *(Oracle*)h;
  o.count_visits = on != 0;
  o.visits.assign(on ? (size_t)o.N : 0, 0u);
}

void oracle_get_visits(void* h, uint32_t* dst) {
  Oracle& o = *(Oracle*)h;
  std::memcpy(dst, o.visits.data(), o.visits.size() * sizeof(uint32_t));
}

void oracle_pair_counts(void* h, int64_t* counts) { pair_counts(*(Oracle*)h, counts); }

void oracle_sro(void* h, double* alpha, int64_t* counts_or_null) {
  Oracle& o = *(Oracle*)h;
  std::vector<int64_t> c((size_t)o.n_shells * o.n_species * o.n_species);
  pair_counts(o, c.data());
  sro(o, c.data(), alpha);
  if (counts_or_null) std::memcpy(counts_or_null, c.data(), c.size() * sizeof(int64_t));
}

}  // extern "C"
