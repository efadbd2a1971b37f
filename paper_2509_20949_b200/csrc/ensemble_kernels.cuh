// Temperature parallelism on one GPU ("temperature parallelism" and Eq. 5-6):
// several replicas of the same system at different temperatures, replica exchange between
// neighbouring temperature slots decided and applied on the device (no host round trip, so a whole
// run of sweeps + exchanges can be enqueued asynchronously).
//
// Reading S9: slots p, p + 1 with p = parity, parity + 2, ... attempt an exchange in
// round r; Delta = (1/kT_p - 1/kT_{p+1}) (E_p - E_{p+1}) evaluated in fp64 as
// (kT_{p+1} - kT_p) * (E_p - E_{p+1}) / (kT_p * kT_{p+1}); accept iff Delta >= 0 or
// u < min(floor(exp(Delta) 2^32), 2^32 - 1), u = philox(ctr = (p, r_hi, r_lo, TAG_EXCHANGE), key =
// exchange seed)[0].  "Exchanging configurations" is done by exchanging temperatures: the two
// replicas keep their lattices and swap slots, and each gets the threshold table of its new slot.
#pragma once
#include "smcx_common.cuh"

namespace smcxk {

enum : uint32_t { TAG_EXCHANGE = 6u };

// Device-resident bookkeeping of an ensemble.  All arrays live in the ensemble's own device area.
struct EnsembleDev {
  int n;                              // replicas = temperature slots
  int len_max;                        // common (zero-padded) threshold-table length
  int has_filter;                     // per-slot two-level filter tables present
  const int32_t* kT;                  // [slot] temperature in 0.1 meV
  const uint32_t* tables;             // [slot][len_max]
  const uint32_t* filters;            // [slot][filter_words] (has_filter)
  int filter_words;
  DevState* const* states;            // [replica] bookkeeping of every replica (running energy)
  uint32_t* const* dst_accept;        // [replica] threshold table inside the replica's workspace
  uint32_t* const* dst_filter;        // [replica] filter tables inside the replica's workspace
  int* replica_at_slot;               // [slot]
  int* slot_of_replica;               // [replica]
  int* changed;                       // [replica] slot changed since the tables were last applied
  int* last_flags;                    // [n - 1] accept flags of the last round (0 for pairs not attempted)
  unsigned long long* attempted;      // [n - 1]
  unsigned long long* accepted;       // [n - 1]
  unsigned long long* round;          // exchange rounds done
};

// One block; thread k decides the pair (p, p + 1), p = parity + 2 k.  Pairs are disjoint, so the
// decisions of a round are independent of each other.
// parity < 0: the low bit of the round counter (smcx_ensemble_run; lets one captured graph serve every round).
__global__ void replica_exchange_kernel(const EnsembleDev E, int parity, uint32_t key0, uint32_t key1) {
  const unsigned long long r = *E.round;
  if (parity < 0) parity = (int)(r & 1ull);
  for (int p = threadIdx.x; p < E.n - 1; p += blockDim.x) E.last_flags[p] = 0;
  __syncthreads();
  for (int k = threadIdx.x; ; k += blockDim.x) {
    const int p = (parity & 1) + 2 * k;
    if (p >= E.n - 1) break;
    const int ri = E.replica_at_slot[p], rj = E.replica_at_slot[p + 1];
    const long long Ei = E.states[ri]->e_run, Ej = E.states[rj]->e_run;
    const int kTi = E.kT[p], kTj = E.kT[p + 1];
    const double a = (double)(kTj - kTi);
    const double c = (double)(Ei - Ej);
    const double b = (double)kTi * (double)kTj;
    const double delta = __ddiv_rn(__dmul_rn(a, c), b);
    bool ok = delta >= 0.0;
    if (!ok) {
      const Philox4 d = philox4x32_10((uint32_t)p, (uint32_t)(r >> 32), (uint32_t)(r & 0xffffffffull), TAG_EXCHANGE, key0, key1);
      const double x = __dmul_rn(exp(delta), 4294967296.0);
      const uint32_t T = x >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)floor(x);
      ok = d.x < T;
    }
    E.attempted[p] += 1ull;
    if (ok) {
      E.accepted[p] += 1ull;
      E.last_flags[p] = 1;
      E.replica_at_slot[p] = rj;
      E.replica_at_slot[p + 1] = ri;
      E.slot_of_replica[rj] = p;
      E.slot_of_replica[ri] = p + 1;
      E.changed[ri] = 1;
      E.changed[rj] = 1;
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) *E.round = r + 1ull;
}

// Block r gives replica r the tables of its slot if the slot changed.
__global__ void replica_apply_tables_kernel(const EnsembleDev E) {
  const int r = blockIdx.x;
  if (!E.changed[r]) return;
  const int slot = E.slot_of_replica[r];
  const uint32_t* src = E.tables + (size_t)slot * E.len_max;
  uint32_t* dst = E.dst_accept[r];
  for (int k = threadIdx.x; k < E.len_max; k += blockDim.x) dst[k] = src[k];
  if (E.has_filter) {
    const uint32_t* fs = E.filters + (size_t)slot * E.filter_words;
    uint32_t* fd = E.dst_filter[r];
    for (int k = threadIdx.x; k < E.filter_words; k += blockDim.x) fd[k] = fs[k];
  }
  __syncthreads();
  if (threadIdx.x == 0) E.changed[r] = 0;
}

}  // namespace smcxk
