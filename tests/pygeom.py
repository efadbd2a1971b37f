"""Independent numpy restatement of the lattice geometry of SURVEY.md 8(c) S0/S1/S7, used by the
tests to pin the oracle by brute force on small lattices.  Shares no code with oracle/ or the
CUDA path; deliberately written differently (explicit coordinate tables, no site<->position
inverse by parity).
"""
from __future__ import annotations

import itertools

import numpy as np

BASIS = {
    0: np.array([[0, 0, 0], [1, 1, 1]]),
    1: np.array([[0, 0, 0], [0, 1, 1], [1, 0, 1], [1, 1, 0]]),
}


def lattice_points(lattice, R):
    """All lattice translations in [-R,R]^3 (half-lattice units): differences of site positions."""
    pts = set()
    basis = BASIS[lattice]
    rng = range(-R // 2 - 1, R // 2 + 2)
    for cx, cy, cz in itertools.product(rng, rng, rng):
        for beta in basis:
            p = (2 * cx + beta[0], 2 * cy + beta[1], 2 * cz + beta[2])
            if max(abs(v) for v in p) <= R and p != (0, 0, 0):
                pts.add(p)
    return pts


def shells(lattice, n_shells):
    """Shells by squared distance; within a shell ascending (dz, dy, dx)."""
    pts = lattice_points(lattice, 6)
    d2 = sorted({x * x + y * y + z * z for x, y, z in pts})
    out = []
    for s in range(n_shells):
        v = [p for p in pts if p[0] ** 2 + p[1] ** 2 + p[2] ** 2 == d2[s]]
        v.sort(key=lambda p: (p[2], p[1], p[0]))
        out.append(np.array(v, dtype=np.int64))
    return out, d2[:n_shells]


def site_positions(lattice, dims):
    """positions[i] for i = ((z*Ly + y)*Lx + x)*B + b."""
    Lx, Ly, Lz = dims
    basis = BASIS[lattice]
    B = len(basis)
    pos = np.zeros((Lx * Ly * Lz * B, 3), dtype=np.int64)
    i = 0
    for z in range(Lz):
        for y in range(Ly):
            for x in range(Lx):
                for b in range(B):
                    pos[i] = (2 * x + basis[b][0], 2 * y + basis[b][1], 2 * z + basis[b][2])
                    i += 1
    return pos


def neighbour_table(lattice, dims, offsets):
    """nbr[i, k] = site at P(i)+offsets[k] (periodic), found by dictionary lookup of positions."""
    pos = site_positions(lattice, dims)
    period = 2 * np.array(dims)
    index = {tuple(p): i for i, p in enumerate(pos)}
    nbr = np.zeros((len(pos), len(offsets)), dtype=np.int64)
    for i, p in enumerate(pos):
        for k, d in enumerate(offsets):
            q = tuple((p + d) % period)
            nbr[i, k] = index[q]
    return nbr


def positive_half(offsets):
    keep = []
    for d in offsets:
        dx, dy, dz = int(d[0]), int(d[1]), int(d[2])
        first = dz if dz != 0 else (dy if dy != 0 else dx)
        keep.append(first > 0)
    return np.array(keep)


class PyLattice:
    def __init__(self, lattice, dims, n_shells):
        self.lattice, self.dims, self.n_shells = lattice, tuple(dims), n_shells
        self.offsets, self.d2 = shells(lattice, n_shells)
        self.nbr = [neighbour_table(lattice, dims, o) for o in self.offsets]
        self.half = [positive_half(o) for o in self.offsets]
        self.n_sites = self.nbr[0].shape[0]

    def energy(self, sigma, epi):
        """H = sum_s sum_i sum_{d in O_s^+} V_s(sigma_i, sigma_{i+d})  (S1)."""
        sigma = np.asarray(sigma, dtype=np.int64)
        H = 0
        for s in range(self.n_shells):
            nb = self.nbr[s][:, self.half[s]]
            H += int(epi[s][sigma[:, None], sigma[nb]].sum())
        return H

    def pair_counts(self, sigma, n_species):
        sigma = np.asarray(sigma, dtype=np.int64)
        out = np.zeros((self.n_shells, n_species, n_species), dtype=np.int64)
        for s in range(self.n_shells):
            nb = self.nbr[s]
            a = np.repeat(sigma, nb.shape[1])
            b = sigma[nb].ravel()
            np.add.at(out[s], (a, b), 1)
        return out
