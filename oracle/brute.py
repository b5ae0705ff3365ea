"""oracle/brute.py -- TEST INFRASTRUCTURE ("oracle A").

Brute force over ALL ordered (k, q, n, m, nu) of Eq. 2 on tiny grids: no channel
list, no unordered trick, no sorting.  For every active k and every q of the full grid it forms
k+q (component-wise modulo, "commensurate grids"), looks the (k, k+q) pair up in the
candidate table and sums

    I[n,k] = -C sum_{q,m,nu} g2 [ delta_s(E_a - E_b + hw) F_abs + delta_s(E_a - E_b - hw) F_em ]

with the readings listed in oracle/ephc_oracle.c (S-1..S-10).  hw and N are read at the q of the
ORDERED term (so the mirror term reads them at -q): the evenness precondition (S-10) is therefore
tested, not assumed.  Independent of ephc_oracle.c: it shares no code with it and is written in
numpy with its own index arithmetic.  It also assembles the dense transport matrix W[a,b]
(S-16), used to pin the transport iteration against a library mat-vec.

Only tests/ may import this module.
"""
from __future__ import annotations

import numpy as np

HBAR_EV_FS = 0.6582119569


def _gauss(x, sigma, ncut):
    out = np.exp(-(x * x) / (2.0 * sigma * sigma)) / (sigma * np.sqrt(2.0 * np.pi))
    return np.where(np.abs(x) < ncut * sigma, out, 0.0)


def _tables(prob):
    n1, n2, n3 = prob.grid
    nq = n1 * n2 * n3
    comp = -np.ones(nq, dtype=np.int64)
    comp[prob.kfull.astype(np.int64)] = np.arange(prob.nk)
    pid = -np.ones((prob.nk, prob.nk), dtype=np.int64)
    pid[prob.pair_ik.astype(np.int64), prob.pair_ikq.astype(np.int64)] = np.arange(prob.npair)
    return comp, pid


def _ordered_terms(prob):
    """Yield, per active k, the arrays of every ordered term that leaves a state of k:
    (k, ikq[nt], iq[nt], G[nt, nnu, nb(m of b), nb(n of a)])."""
    n1, n2, n3 = prob.grid
    comp, pid = _tables(prob)
    q = np.arange(n1 * n2 * n3, dtype=np.int64)
    q1, q2, q3 = q // (n2 * n3), (q // n3) % n2, q % n3
    for k in range(prob.nk):
        kf = int(prob.kfull[k])
        k1, k2, k3 = kf // (n2 * n3), (kf // n3) % n2, kf % n3
        kq_full = (((k1 + q1) % n1) * n2 + ((k2 + q2) % n2)) * n3 + ((k3 + q3) % n3)
        ikq = comp[kq_full]
        ok = ikq >= 0
        lo = np.minimum(k, ikq)
        hi = np.maximum(k, ikq)
        p = np.where(ok, pid[lo.clip(0), hi.clip(0)], -1)
        ok &= p >= 0
        sel = np.nonzero(ok)[0]
        if sel.size == 0:
            continue
        ikq_s, p_s = ikq[sel], p[sel]
        G = prob.g2[p_s]                                   # [nt, nnu, m(at pair_ikq), n(at pair_ik)]
        swap = ikq_s < k                                   # k sits on the pair_ikq side
        G = np.where(swap[:, None, None, None], np.swapaxes(G, 2, 3), G)
        yield k, ikq_s, sel, G


def _term_weights(prob, k, ikq, iq, G):
    nb, nnu = prob.nb, prob.nnu
    Ea = prob.E[k][None, None, None, :]                    # n
    Eb = prob.E[ikq][:, None, :, None]                     # m
    hw = prob.hw[iq][:, :, None, None]                     # nu
    inwin = ((Ea >= prob.emin) & (Ea <= prob.emax)) & ((Eb >= prob.emin) & (Eb <= prob.emax))
    d = Ea - Eb
    da = _gauss(d + hw, prob.sigma, prob.ncut)
    de = _gauss(d - hw, prob.sigma, prob.ncut)
    keep = inwin & (G >= prob.g2_cut)
    C = 2.0 * np.pi / (HBAR_EV_FS * float(prob.nq))
    wa = np.where(keep, C * G * da, 0.0)
    we = np.where(keep, C * G * de, 0.0)
    assert wa.shape == (len(ikq), nnu, nb, nb)
    return wa, we


def collision_brute(prob, f, N):
    """I[ns] by the ordered sum of Eq. 2; also returns the number of non-zero ordered terms."""
    nb, nnu = prob.nb, prob.nnu
    f2 = np.asarray(f, dtype=np.float64).reshape(prob.nk, nb)
    N2 = np.asarray(N, dtype=np.float64).reshape(prob.nq, nnu)
    I = np.zeros((prob.nk, nb))
    nterms = 0
    for k, ikq, iq, G in _ordered_terms(prob):
        wa, we = _term_weights(prob, k, ikq, iq, G)
        fa = f2[k][None, None, None, :]
        fb = f2[ikq][:, None, :, None]
        Nq = N2[iq][:, :, None, None]
        Fabs = fa * (1.0 - fb) * Nq - fb * (1.0 - fa) * (Nq + 1.0)
        Fem = fa * (1.0 - fb) * (Nq + 1.0) - fb * (1.0 - fa) * Nq
        I[k] -= (wa * Fabs + we * Fem).sum(axis=(0, 1, 2))
        nterms += int(((wa != 0) | (we != 0)).sum())
    return I.reshape(-1), nterms


def transport_matrix_brute(prob, f0, N):
    """Dense W[a, b] = sum_{nu} W(a<-b) over every ordered term (q=0, n==m included), reading S-16."""
    nb, nnu = prob.nb, prob.nnu
    f2 = np.asarray(f0, dtype=np.float64).reshape(prob.nk, nb)
    N2 = np.asarray(N, dtype=np.float64).reshape(prob.nq, nnu)
    ns = prob.nk * nb
    W = np.zeros((ns, ns))
    for k, ikq, iq, G in _ordered_terms(prob):
        wa, we = _term_weights(prob, k, ikq, iq, G)
        fb = f2[ikq][:, None, :, None]
        Nq = N2[iq][:, :, None, None]
        Wab = (we * (1.0 + Nq - fb) + wa * (Nq + fb)).sum(axis=1)      # [nt, m, n]
        a = k * nb + np.arange(nb)
        for t in range(len(ikq)):
            b = int(ikq[t]) * nb + np.arange(nb)
            W[np.ix_(a, b)] += Wab[t].T                                 # rows a(n), cols b(m)
    return W
