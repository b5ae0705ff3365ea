"""k-sharded evaluation across ranks ("k points are evenly distributed over different MPI processes";
PAPER.md:148-173: the strong-scaling experiment).  One process per GPU; every rank owns a contiguous range of
destination k points (ephc_build_channels_range) and computes the collision integral / transport update / RK stage of
its own states; after every evaluation the owned slices are exchanged with ONE all-gather (<= ns doubles), because the
next evaluation reads f (or F) of all states.  This module is plumbing only: ranges, the exchange and the call order;
all arithmetic runs in the library's kernels.
"""
from __future__ import annotations

import numpy as np

from . import build_channels


def balanced_k_ranges(prob, nparts: int):
    """nparts contiguous ranges of compact k indices with about the same number of ordered (k <- k') half-pairs,
    which is what a rank's store and work scale with.  Returns a list of (k_lo, k_hi) that partitions [0, nk)."""
    nk = int(prob.nk)
    ik = np.asarray(prob.pair_ik, dtype=np.int64)
    ikq = np.asarray(prob.pair_ikq, dtype=np.int64)
    load = np.bincount(ik, minlength=nk) + np.bincount(ikq[ikq != ik], minlength=nk)
    cum = np.concatenate([[0], np.cumsum(load)])
    bounds = [0]
    for r in range(1, nparts):
        goal = cum[-1] * r / nparts
        k = int(np.searchsorted(cum, goal, side="left"))
        bounds.append(min(max(k, bounds[-1]), nk))
    bounds.append(nk)
    return [(bounds[r], bounds[r + 1]) for r in range(nparts)]


class Exchange:
    """All-gather of the owned state slices of every rank into a full vector (in place)."""

    def __init__(self, dist, ranges, nb: int, device):
        import torch
        self.dist, self.torch = dist, torch
        self.world = len(ranges)
        self.rank = dist.get_rank() if dist is not None else 0
        self.lo = [r[0] * nb for r in ranges]
        self.hi = [r[1] * nb for r in ranges]
        self.maxlen = max(1, max(h - l for l, h in zip(self.lo, self.hi)))
        self.send = torch.zeros(self.maxlen, dtype=torch.float64, device=device)
        self.recv = [torch.zeros(self.maxlen, dtype=torch.float64, device=device) for _ in range(self.world)]
        self.bytes = 8 * self.maxlen * self.world

    def __call__(self, x, ncomp: int = 1):
        """x: [ncomp * ns] (component-major).  After the call every rank holds the owners' values of all states."""
        if self.dist is None or self.world == 1:
            return
        ns = x.numel() // ncomp
        for c in range(ncomp):
            xc = x[c * ns:(c + 1) * ns]
            lo, hi = self.lo[self.rank], self.hi[self.rank]
            self.send[:hi - lo].copy_(xc[lo:hi])
            self.dist.all_gather(self.recv, self.send)
            for r in range(self.world):
                if r != self.rank:
                    xc[self.lo[r]:self.hi[r]].copy_(self.recv[r][:self.hi[r] - self.lo[r]])


class ShardedSolver:
    """The hot path on a k-sharded handle: collision, transport solve and RK4 steps with the exchanges in place."""

    def __init__(self, prob, dist, device, flags: int = 0):
        import torch
        self.torch = torch
        world = dist.get_world_size() if dist is not None else 1
        rank = dist.get_rank() if dist is not None else 0
        self.ranges = balanced_k_ranges(prob, world)
        self.h = build_channels(prob, flags=flags, k_range=self.ranges[rank])
        self.ns = prob.nk * prob.nb
        self.x = Exchange(dist, self.ranges, prob.nb, device)
        self.y = [torch.empty(self.ns, dtype=torch.float64, device=device) for _ in range(2)]

    def collision(self, f, N, I, stream=None):
        self.h.collision(f, N, I, stream)
        self.x(I)

    def transport_solve(self, f0, N, v, niter, Gamma, tau, Fa, Fb, stream=None):
        self.h.transport_setup(f0, N, Gamma, stream)
        self.x(Gamma)
        self.h.transport_start(Gamma, v, tau, Fa, stream)
        for _ in range(niter):
            self.h.transport_iter(Fa, v, tau, Fb, stream)
            self.x(Fb, 3)
            Fa, Fb = Fb, Fa
        return Fa

    def rt_step(self, f, N, dt_fs, nsteps, stream=None):
        y0, y1 = self.y
        for _ in range(nsteps):
            self.h.rt_stage(f, f, N, dt_fs, 1, y0, stream)
            self.x(y0)
            self.h.rt_stage(f, y0, N, dt_fs, 2, y1, stream)
            self.x(y1)
            self.h.rt_stage(f, y1, N, dt_fs, 3, y0, stream)
            self.x(y0)
            self.h.rt_stage(f, y0, N, dt_fs, 4, None, stream)
            self.x(f)
