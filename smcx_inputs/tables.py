"""EPI tables and acceptance-threshold tables (input data, see package docstring)."""
from __future__ import annotations

import math

import numpy as np

TAG_EPI = 4  # low byte of ctr[3]; SURVEY.md 8(c) S4 tag list

_M0 = 0xD2511F53
_M1 = 0xCD9E8D57
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    """Philox4x32-10 (Salmon et al., SC'11), pure-Python integers.

    Only used to draw the handful of EPI entries; the oracle and the CUDA path each carry
    their own implementation.  ``ctr`` is 4 and ``key`` 2 unsigned 32-bit integers.
    """
    c0, c1, c2, c3 = (int(c) & _MASK for c in ctr)
    k0, k1 = (int(k) & _MASK for k in key)
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> 32, p0 & _MASK
        hi1, lo1 = p1 >> 32, p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def make_epi(n_shells: int, n_species: int, amplitude: int, seed: int) -> np.ndarray:
    """Symmetric int32 EPI tables, shape [n_shells][n_species][n_species], 0.1 meV units."""
    key = (seed & _MASK, (seed >> 32) & _MASK)
    v = np.zeros((n_shells, n_species, n_species), dtype=np.int32)
    span = 2 * amplitude + 1
    for s in range(n_shells):
        for a in range(n_species):
            for b in range(a, n_species):
                r0 = philox4x32_10((a, b, s, TAG_EPI), key)[0]
                val = -amplitude + ((r0 * span) >> 32)
                v[s, a, b] = val
                v[s, b, a] = val
    return v


TAG_LOCAL = 7  # synthetic weights of the nonlinear local-energy model (reading S12)


def make_local_weights(n_shells: int, n_species: int, amp_linear: int, amp_quad: int, seed: int):
    """Synthetic integer weights of the nonlinear local-energy model (reading S12; the paper's qSRO weights, PAPER.md:118,
    are not published): (W1, W2) with W1[s][a][x] uniform in [-amp_linear, amp_linear] (not symmetric) and
    W2[s][a][x][y], x <= y, uniform in [-amp_quad, amp_quad] (0 for x > y), drawn like the EPI entries:
    -A + mulhi32(philox(ctr=(index, a, s, TAG_LOCAL), key=seed)[0], 2A + 1), index = x for W1, n + x n + y for W2."""
    key = (seed & _MASK, (seed >> 32) & _MASK)
    n = n_species
    w1 = np.zeros((n_shells, n, n), dtype=np.int32)
    w2 = np.zeros((n_shells, n, n, n), dtype=np.int32)
    for s in range(n_shells):
        for a in range(n):
            for x in range(n):
                r = philox4x32_10((x, a, s, TAG_LOCAL), key)[0]
                w1[s, a, x] = -amp_linear + ((r * (2 * amp_linear + 1)) >> 32)
                for y in range(x, n):
                    r = philox4x32_10((n + x * n + y, a, s, TAG_LOCAL), key)[0]
                    w2[s, a, x, y] = -amp_quad + ((r * (2 * amp_quad + 1)) >> 32)
    return w1, w2


def accept_table_len(kT_units: int) -> int:
    return int(math.floor(32.0 * math.log(2.0) * kT_units)) + 2


def make_accept_table(kT_units: int) -> np.ndarray:
    """uint32 thresholds: a trial with dE = d > 0 is accepted iff u < T[d] (u a 32-bit draw)."""
    n = accept_table_len(kT_units)
    d = np.arange(n, dtype=np.float64)
    x = np.exp(-d / float(kT_units)) * 4294967296.0
    t = np.where(x >= 4294967295.0, 4294967295.0, np.floor(x))
    return t.astype(np.uint32)


def anneal_kT_units(t: int, n_sweeps: int = 2000, kT_hi: int = 1720, kT_lo: int = 430) -> int:
    """Linear anneal of config 2: kT(t) = kT_hi - floor((kT_hi-kT_lo) * t / (n_sweeps-1))."""
    if n_sweeps <= 1:
        return kT_hi
    return kT_hi - ((kT_hi - kT_lo) * t) // (n_sweeps - 1)


def replica_ladder(kT_lo: int, n_replicas: int, n_sites: int, coeff: float) -> list:
    """Temperatures of a replica-exchange ladder spaced as Eq. 7 asks:
    delta kT = coeff / sqrt(n_sites) (0.1 meV units, rounded to integers, at least 1 apart)."""
    step = max(1, int(round(coeff / math.sqrt(float(n_sites)))))
    return [int(kT_lo) + r * step for r in range(n_replicas)]


def composition_counts(n_sites: int, parts) -> list:
    """Integer species counts for a composition given in parts (e.g. (29, 29, 28, 7, 7) for the paper's
    Fe29Co29Ni28Al7Ti7): floor(n_sites * part / sum), the remainder handed out one site at a
    time to the species with the largest fractional part (ties: lower index first).  Sums to n_sites."""
    total = int(sum(parts))
    base = [int(n_sites) * int(p) // total for p in parts]
    rem = [int(n_sites) * int(p) % total for p in parts]
    left = int(n_sites) - sum(base)
    for p in sorted(range(len(parts)), key=lambda q: (-rem[q], q))[:left]:
        base[p] += 1
    return base


def cooling_stages(kT_hi: int, kT_lo: int, n_stages: int) -> list:
    """Stage-wise cooling as the paper runs it ("decrease the temperature from 2000 K to 1000 K, with tens of
    thousands of MC steps at each temperature"): n_stages equally spaced temperatures from
    kT_hi down to kT_lo inclusive, in 0.1 meV units (integers)."""
    if n_stages <= 1:
        return [int(kT_hi)]
    return [int(kT_hi) - ((int(kT_hi) - int(kT_lo)) * s) // (n_stages - 1) for s in range(n_stages)]
