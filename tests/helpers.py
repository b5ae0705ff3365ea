"""Hand-built inputs for the pins and edge-case tests (inputs only: no method arithmetic here)."""
from __future__ import annotations

import numpy as np

from ephc_inputs import Problem, bose_einstein, fermi_dirac, KB_EV_PER_K  # noqa: F401


def manual_problem(grid, E, hw, pairs, g2, sigma, window=(-10.0, 10.0), ncut=3.0, g2_cut=0.0,
                   kfull=None, f=None, N=None, name="manual"):
    """All k of `kfull` (default: the whole grid) with energies E[nk, nb]; pairs = list of (ik, ikq)."""
    grid = tuple(int(g) for g in grid)
    nq = grid[0] * grid[1] * grid[2]
    E = np.ascontiguousarray(E, dtype=np.float64)
    nk, nb = E.shape
    hw = np.ascontiguousarray(hw, dtype=np.float64)
    nnu = hw.shape[1]
    assert hw.shape[0] == nq
    if kfull is None:
        assert nk == nq
        kfull = np.arange(nq)
    pairs = sorted(pairs)
    pik = np.array([p[0] for p in pairs], dtype=np.int32)
    pikq = np.array([p[1] for p in pairs], dtype=np.int32)
    g2 = np.ascontiguousarray(g2, dtype=np.float64).reshape(len(pairs), nnu, nb, nb)
    ns = nk * nb
    f = np.full(ns, 0.5) if f is None else np.ascontiguousarray(f, dtype=np.float64).reshape(ns)
    N = np.ones(nq * nnu) if N is None else np.ascontiguousarray(N, dtype=np.float64).reshape(nq * nnu)
    return Problem(name=name, seed=0, grid=grid, nk=nk, nb=nb, nnu=nnu,
                   kfull=np.asarray(kfull, dtype=np.int32), E=E, emin=float(window[0]), emax=float(window[1]),
                   hw=hw, sigma=float(sigma), ncut=float(ncut), g2_cut=float(g2_cut), pair_ik=pik,
                   pair_ikq=pikq, g2=g2, f=f, f0=f.copy(), N=N, v=np.zeros((3, ns)), temperature=300.0,
                   mu=0.0, pair_prob=1.0, meta={})


def neg_index(grid):
    n1, n2, n3 = grid
    idx = np.arange(n1 * n2 * n3)
    i1, i2, i3 = idx // (n2 * n3), (idx // n3) % n2, idx % n3
    return (((-i1) % n1) * n2 + ((-i2) % n2)) * n3 + ((-i3) % n3)


def exact_energy_problem(seed=7, grid=(3, 3, 4), nb=3, nnu=4, unit=2.0 ** -6, temperature=400.0, mu=None):
    """Energies and phonon energies are integer multiples of `unit` (a power of two, so sums and
    differences are exact) and sigma = unit/10, so 3*sigma < unit: a delta passes only when its
    argument is EXACTLY zero.  Every active channel then conserves energy exactly, which is the
    setting of the detailed-balance pin.  f = Fermi-Dirac, N = Bose-Einstein at one temperature."""
    rng = np.random.default_rng(seed)
    n1, n2, n3 = grid
    nq = n1 * n2 * n3
    E = rng.integers(0, 6, size=(nq, nb)).astype(np.float64) * unit
    c = rng.integers(1, 4, size=(nq, nnu))
    neg = neg_index(grid)
    canon = np.minimum(np.arange(nq), neg)
    hw = c[canon].astype(np.float64) * unit
    pairs = [(i, j) for i in range(nq) for j in range(i, nq)]
    g2 = rng.lognormal(-9.0, 1.0, size=(len(pairs), nnu, nb, nb))
    for p, (i, j) in enumerate(pairs):
        if i == j:
            g2[p] = 0.5 * (g2[p] + np.swapaxes(g2[p], 1, 2))
    if mu is None:
        mu = 2.5 * unit
    f = fermi_dirac(E, mu, temperature).reshape(-1)
    N = bose_einstein(hw, temperature).reshape(-1)
    return manual_problem(grid, E, hw, pairs, g2, sigma=unit / 10.0, f=f, N=N, name="exact")
