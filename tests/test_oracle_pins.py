"""Pins of the CPU oracle: what the paper and the mathematics fix.

The paper prints no value of I(n,k) (PAPER.md has no worked numeric example), so the oracle is
pinned by brute force on tiny inputs, closed forms, invariants and special cases that reduce to a
library routine.  None of these tests touches the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import oracle
from ephc_inputs import make_problem, fermi_dirac, bose_einstein
from oracle import brute
from helpers import exact_energy_problem, manual_problem

HBAR = 0.6582119569


@pytest.fixture(scope="module")
def tiny():
    p = make_problem("tiny")
    return p, oracle.OracleList(p)


@pytest.fixture(scope="module")
def small_win():
    # 4x4x4, 2 bands, 3 modes, a window that cuts states out, a g2 cut-off, low hw so that q=0 diagonals exist
    p = make_problem("tiny", grid=(4, 4, 4), window=(0.08, 0.22), seed=99)
    p.g2_cut = float(np.quantile(p.g2, 0.2))
    p.hw[...] = p.hw * 0.5                                   # hw in [2.5, 30) meV, still even in q
    p.N = bose_einstein(p.hw, 300.0).reshape(-1)
    return p, oracle.OracleList(p)


# ----------------------------------------------------------------------------- P0: brute force
def test_p0_list_equals_brute_force_tiny(tiny):
    p, L = tiny
    IB = L.collision(p.f, p.N)
    IA, nterms = brute.collision_brute(p, p.f, p.N)
    assert nterms == 2 * L.nch + L.ndiag                       # every channel = two ordered terms
    assert np.abs(IA - IB).max() <= 1e-13 * np.abs(IA).max()
    assert 3e5 < L.nch < 7e5                                   # ~5e5 unordered channels


def test_p0_list_equals_brute_force_window_cut_diag(small_win):
    p, L = small_win
    assert p.nk < 64 and L.ndiag > 0 and L.nch > 100
    IA, nterms = brute.collision_brute(p, p.f, p.N)
    assert nterms == 2 * L.nch + L.ndiag
    IB = L.collision(p.f, p.N)
    assert np.abs(IA - IB).max() <= 1e-13 * np.abs(IA).max()
    # out-of-window states never receive a contribution
    out = ~((p.E.reshape(-1) >= p.emin) & (p.E.reshape(-1) <= p.emax))
    assert out.any() and np.all(IB[out] == 0.0)


def test_sampled_definition_equals_list(small_win, tiny):
    for p, L in (small_win, tiny):
        IB = L.collision(p.f, p.N)
        st = np.arange(0, p.ns, max(1, p.ns // 37), dtype=np.int32)
        Is = oracle.collision_sampled(p, p.f, p.N, st)
        assert np.abs(Is - IB[st]).max() <= 1e-13 * np.abs(IB).max()


def test_threaded_collision_equals_serial(tiny, small_win):
    # orc_collision_omp (the paper's Baseline-CPU shape: OpenMP over the list, atomic updates) is only
    # used to time the oracle on all host cores; it is pinned to the serial loop, which P0-P5 pin: same terms,
    # any order, so the two agree within 1e-13 of the sum of |T| that reaches a state
    rng = np.random.default_rng(17)
    for p, L in (tiny, small_win):
        for f, N in ((p.f, p.N), (rng.uniform(0, 1, p.ns), rng.uniform(0, 3, p.nq * p.nnu))):
            I1, I2 = L.collision(f, N), L.collision(f, N, omp=True)
            ch = L.export()
            fa, fb = f[ch["ik"] * p.nb + ch["n"]], f[ch["ikq"] * p.nb + ch["m"]]
            Nq = N[ch["iq"].astype(np.int64) * p.nnu + ch["nu"]]
            out_, in_ = fa * (1 - fb), fb * (1 - fa)
            absT = np.abs(ch["w_abs"] * (out_ * Nq - in_ * (Nq + 1))) + np.abs(ch["w_em"] * (out_ * (Nq + 1) - in_ * Nq))
            bound = np.zeros(p.ns)
            np.add.at(bound, ch["ik"] * p.nb + ch["n"], absT)
            np.add.at(bound, ch["ikq"] * p.nb + ch["m"], absT)
            assert np.abs(I1).max() > 0
            assert np.all(np.abs(I1 - I2) <= 1e-13 * bound + 1e-300)
            assert abs(I2.sum()) <= 1e-13 * absT.sum()


def test_canonical_list_structure(tiny):
    p, L = tiny
    ch = L.export()
    key = np.stack([ch["ik"], ch["ikq"], ch["nu"], ch["m"], ch["n"]]).astype(np.int64)
    # strictly increasing lexicographic order (ik, ikq, nu, m, n): unique and sorted
    d = np.diff(key, axis=1)
    first = (d != 0).argmax(axis=0)
    assert np.all(d[first, np.arange(d.shape[1])] > 0)
    assert np.all((ch["ik"] < ch["ikq"]) | ((ch["ik"] == ch["ikq"]) & (ch["n"] < ch["m"])))
    assert np.all((ch["w_abs"] > 0) | (ch["w_em"] > 0))
    # q index: kfull[ikq] - kfull[ik] on the 8x8x8 grid (all k active, kfull = identity)
    n = 8
    kf, kqf = ch["ik"].astype(np.int64), ch["ikq"].astype(np.int64)
    q = [((kqf // (n * n) - kf // (n * n)) % n), (((kqf // n) % n - (kf // n) % n) % n), ((kqf % n - kf % n) % n)]
    assert np.array_equal(ch["iq"], (q[0] * n + q[1]) * n + q[2])


# ----------------------------------------------------------------------------- P1: one channel by hand
def test_p1_single_channel_worked_example():
    # tests/golden/p1_single_channel.txt: Eq. 2 for one absorption channel with exact energy
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "p1_single_channel.txt")) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                k, v = line.split("=")
                vals[k.strip()] = float(v)
    hw = 0.03
    p = manual_problem((1, 1, 1), E=[[0.0, hw]], hw=[[hw]], pairs=[(0, 0)], g2=[[[[0.0, 1e-4], [1e-4, 0.0]]]],
                       sigma=0.010, f=[0.5, 0.25], N=[1.0])
    L = oracle.OracleList(p)
    assert L.nch == 1 and L.ndiag == 0
    ch = L.export()
    assert (ch["n"][0], ch["m"][0]) == (0, 1) and ch["w_em"][0] == 0.0
    I = L.collision(p.f, p.N)
    assert I[0] == pytest.approx(vals["I_a"], rel=1e-11)
    assert I[1] == -I[0]
    # the same number from the formula, written out: -(2 pi/hbar) g2 delta_sigma(0) F_abs
    expect = -(2 * math.pi / HBAR) * 1e-4 * (1.0 / (0.010 * math.sqrt(2 * math.pi))) * 0.125
    assert I[0] == pytest.approx(expect, rel=1e-14)


# ----------------------------------------------------------------------------- P2: f == c closed form
def test_p2_constant_occupation_closed_form(tiny):
    p, L = tiny
    ch = L.export()
    a = ch["ik"] * p.nb + ch["n"]
    b = ch["ikq"] * p.nb + ch["m"]
    # ordered terms of a: (w_abs, w_em); of b (mirror): (w_em, w_abs)  ->  I_s = -c(1-c) * S_s
    S = np.zeros(p.ns)
    np.add.at(S, a, ch["w_em"] - ch["w_abs"])
    np.add.at(S, b, ch["w_abs"] - ch["w_em"])
    for c in (0.3, 0.9):
        for Nscale in (1.0, 3.0):                      # independent of N
            I = L.collision(np.full(p.ns, c), p.N * Nscale)
            assert np.abs(I + c * (1 - c) * S).max() <= 1e-12 * np.abs(c * (1 - c) * S).max()
    assert np.all(L.collision(np.zeros(p.ns), p.N) == 0.0)
    assert np.abs(L.collision(np.ones(p.ns), p.N)).max() <= 1e-18


# ----------------------------------------------------------------------------- P3: particle number
def test_p3_particle_number_conservation(tiny, small_win):
    rng = np.random.default_rng(5)
    for p, L in (tiny, small_win):
        for _ in range(2):
            f = rng.uniform(0, 1, p.ns)
            N = rng.uniform(0, 3, p.nq * p.nnu)
            I = L.collision(f, N)
            assert abs(I.sum()) <= 1e-13 * np.abs(I).sum()
            assert np.abs(I).max() > 0


# ----------------------------------------------------------------------------- P4: detailed balance
def test_p4_detailed_balance_on_exact_energy_channels():
    p = exact_energy_problem()
    L = oracle.OracleList(p)
    assert L.nch > 500
    ch = L.export()
    # every surviving delta has argument exactly zero: weight = C g2 / (sigma sqrt(2 pi))
    I_eq = L.collision(p.f, p.N)
    scale = np.zeros(p.ns)
    a = ch["ik"] * p.nb + ch["n"]
    b = ch["ikq"] * p.nb + ch["m"]
    np.add.at(scale, a, ch["w_abs"] + ch["w_em"])
    np.add.at(scale, b, ch["w_abs"] + ch["w_em"])
    assert np.abs(I_eq).max() <= 1e-14 * scale.max()
    # ... and it is not zero away from equilibrium (the pin would pass trivially otherwise)
    f2 = p.f.copy(); f2[::3] *= 0.5
    assert np.abs(L.collision(f2, p.N)).max() > 1e-3 * scale.max() * 0.01
    # wrong phonon temperature breaks it
    N2 = bose_einstein(p.hw, 800.0).reshape(-1)
    assert np.abs(L.collision(p.f, N2)).max() > 1e-6 * scale.max()
    IA, _ = brute.collision_brute(p, p.f, p.N)
    assert np.abs(IA).max() <= 1e-14 * scale.max()


# ----------------------------------------------------------------------------- P5: structure
def test_p5_quadratic_in_f_linear_in_g2(small_win):
    p, L = small_win
    rng = np.random.default_rng(11)
    d = rng.uniform(-0.05, 0.05, p.ns)
    I = [L.collision(p.f + t * d, p.N) for t in range(4)]
    third = I[0] - 3 * I[1] + 3 * I[2] - I[3]
    second = I[0] - 2 * I[1] + I[2]
    assert np.abs(second).max() > 1e-9 * np.abs(I[0]).max()          # genuinely quadratic
    assert np.abs(third).max() <= 1e-12 * np.abs(I[0]).max()
    p2 = make_problem("tiny", grid=(4, 4, 4), window=(0.08, 0.22), seed=99)
    p2.hw[...] = p.hw; p2.N = p.N; p2.g2 = p.g2 * 2.0; p2.g2_cut = p.g2_cut * 2.0
    assert np.array_equal(oracle.OracleList(p2).collision(p.f, p.N), 2.0 * I[0])   # power of two: bit exact


# ----------------------------------------------------------------------------- P6: Gamma = -dI_a/df_a
def test_p6_gamma_is_minus_diagonal_derivative(small_win):
    p, L = small_win
    G = L.transport_setup(p.f0, p.N)
    h = 1e-3
    rng = np.random.default_rng(3)
    inw = np.nonzero(G > 0)[0]
    for s in rng.choice(inw, size=12, replace=False):
        fp, fm = p.f0.copy(), p.f0.copy()
        fp[s] += h; fm[s] -= h
        dIds = (L.collision(fp, p.N)[s] - L.collision(fm, p.N)[s]) / (2 * h)   # exact for a quadratic
        # the q=0, n==m diagonal term enters Gamma_a but cancels in I (W_aa F_a on both sides): remove it
        dg = L.export_diag()
        Wd = 0.0
        for j in np.nonzero(dg["s"] == s)[0]:
            Nq = p.N[dg["iq"][j] * p.nnu + dg["nu"][j]]
            Wd += dg["w_em"][j] * (1 + Nq - p.f0[s]) + dg["w_abs"][j] * (Nq + p.f0[s])
        assert -dIds == pytest.approx(G[s] - Wd, rel=1e-9)


# ----------------------------------------------------------------------------- P7: transport
def test_p7_transport_iteration_is_dense_matvec(small_win):
    p, L = small_win
    W = brute.transport_matrix_brute(p, p.f0, p.N)
    G = L.transport_setup(p.f0, p.N)
    assert np.abs(W.sum(axis=1) - G).max() <= 1e-13 * G.max()
    tau = np.where(G > 0, 1.0 / np.where(G > 0, G, 1.0), 0.0)
    rng = np.random.default_rng(8)
    F = rng.normal(size=(3, p.ns)); v = rng.normal(size=(3, p.ns))
    Fo = L.transport_iter(p.f0, p.N, F, v, tau)
    ref = tau[None, :] * (v + F @ W.T)
    assert np.abs(Fo - ref).max() <= 1e-12 * np.abs(ref).max()
    # F == const c  =>  F' = tau v + c  on every state that scatters (row sums of W are Gamma)
    c = 0.37
    Fc = L.transport_iter(p.f0, p.N, np.full((3, p.ns), c), v, tau)
    on = G > 0
    assert np.abs(Fc[:, on] - (tau[on] * v[:, on] + c)).max() <= 1e-12


def test_p7_detailed_balance_symmetry_of_W():
    p = exact_energy_problem(seed=21)
    W = brute.transport_matrix_brute(p, p.f, p.N)
    w = p.f * (1 - p.f)
    A = W * w[:, None]            # W(a<-b) f0_a (1 - f0_a) = W(b<-a) f0_b (1 - f0_b)
    assert np.abs(A - A.T).max() <= 1e-13 * np.abs(A).max() and np.abs(A).max() > 0
    L = oracle.OracleList(p)
    G = L.transport_setup(p.f, p.N)
    assert np.abs(W.sum(axis=1) - G).max() <= 1e-13 * G.max()


# ----------------------------------------------------------------------------- P8: two-state logistic
def _two_state(f_a, f_b, Nph):
    hw = 0.03
    p = manual_problem((1, 1, 1), E=[[0.0, hw]], hw=[[hw]], pairs=[(0, 0)], g2=[[[[0.0, 4e-3], [4e-3, 0.0]]]],
                       sigma=0.010, f=[f_a, f_b], N=[Nph])
    return p, oracle.OracleList(p)


def _logistic(fa0, c, Nph, R, t):
    # df/dt = R (f - r1)(f - r2),  r1,2 roots of f^2 - (2N+1+c) f + c(N+1)
    bq = 2 * Nph + 1 + c
    disc = math.sqrt(bq * bq - 4 * c * (Nph + 1))
    r1, r2 = (bq - disc) / 2, (bq + disc) / 2
    K = (fa0 - r1) / (fa0 - r2)
    e = K * math.exp(R * (r1 - r2) * t)
    return (r1 - r2 * e) / (1 - e)


def test_p8_rk4_two_state_closed_form():
    fa0, fb0, Nph = 0.8, 0.1, 0.6
    p, L = _two_state(fa0, fb0, Nph)
    R = L.export()["w_abs"][0]
    assert R == pytest.approx((2 * math.pi / HBAR) * 4e-3 / (0.010 * math.sqrt(2 * math.pi)), rel=1e-14)
    T = 2.0   # fs; R ~ 1.5 / fs, so the relaxation is well under way
    errs = []
    for nsteps in (20, 40, 80):
        f, sumf = L.rt_step(p.f, p.N, T / nsteps, nsteps)
        exact = _logistic(fa0, fa0 + fb0, Nph, R, T)
        errs.append(abs(f[0] - exact))
        assert f[0] + f[1] == pytest.approx(fa0 + fb0, abs=1e-15)
        assert np.abs(sumf - (fa0 + fb0)).max() <= 1e-15
    assert errs[0] < 1e-4 and 12 < errs[0] / errs[1] < 20 and 12 < errs[1] / errs[2] < 20   # 4th order
    assert abs(fa0 - _logistic(fa0, fa0 + fb0, Nph, R, T)) > 0.05


# ----------------------------------------------------------------------------- P9: conservation over many steps
def test_p9_rt_conserves_particle_number_and_is_reproducible(small_win):
    p, L = small_win
    f1, s1 = L.rt_step(p.f, p.N, 1.0, 200)
    f2, s2 = L.rt_step(p.f, p.N, 1.0, 200)
    assert np.array_equal(f1, f2) and np.array_equal(s1, s2)
    assert np.abs(s1 - s1[0]).max() <= 1e-12 * abs(s1[0])
    assert np.abs(f1 - p.f).max() > 1e-4          # the state did evolve


# ---- drift term of Eq. 1 and transport post-processing (readings R-25, R-26) -----------------------------------
def _full_grid_problem(grid, nb=2):
    nq = grid[0] * grid[1] * grid[2]
    return manual_problem(grid, E=np.zeros((nq, nb)), hw=np.full((nq, 1), 0.02), pairs=[], g2=np.zeros((0, 1, nb, nb)),
                          sigma=0.01)


def test_drift_closed_form_on_a_fourier_mode():
    # f = A + B cos(2 pi x_i): the central difference is exact up to the factor N_i sin(2 pi / N_i):
    # D = -(F_i / hbar) * (-B N_i sin(2 pi / N_i) sin(2 pi x_i))
    grid = (6, 5, 8)
    p = _full_grid_problem(grid)
    idx = np.arange(p.nk)
    c = [idx // (grid[1] * grid[2]), (idx // grid[2]) % grid[1], idx % grid[2]]
    for i in range(3):
        theta = 2 * np.pi * c[i] / grid[i]
        f = np.repeat(0.3 + 0.2 * np.cos(theta), p.nb)
        field = np.zeros(3); field[i] = 0.07
        D = oracle.drift(p, f, field)
        exp = np.repeat((0.07 / HBAR) * 0.2 * grid[i] * np.sin(2 * np.pi / grid[i]) * np.sin(theta), p.nb)
        assert np.abs(D - exp).max() <= 1e-14 * np.abs(exp).max()
        other = np.zeros(3); other[(i + 1) % 3] = 0.07               # a field along another axis sees no gradient
        assert np.abs(oracle.drift(p, f, other)).max() <= 1e-15
    # general f and field: linear in both, and the drift moves occupation without creating it (periodic grid)
    rng = np.random.default_rng(3)
    f = rng.uniform(0, 1, p.ns); g = rng.uniform(0, 1, p.ns)
    F1, F2 = np.array([0.01, -0.02, 0.03]), np.array([0.05, 0.0, -0.01])
    assert np.allclose(oracle.drift(p, 2 * f - g, F1 + F2), 2 * oracle.drift(p, f, F1) - oracle.drift(p, g, F1)
                       + 2 * oracle.drift(p, f, F2) - oracle.drift(p, g, F2), rtol=0, atol=1e-13)
    assert abs(oracle.drift(p, f, F1).sum()) <= 1e-12 * np.abs(oracle.drift(p, f, F1)).sum()


def test_drift_treats_missing_neighbours_as_empty():
    # active k = a slab of the grid: the neighbour outside it counts as f = 0 (reading R-25)
    grid = (4, 1, 1)
    p = manual_problem(grid, E=np.zeros((2, 1)), hw=np.full((4, 1), 0.02), pairs=[], g2=np.zeros((0, 1, 1, 1)), sigma=0.01,
                       kfull=[1, 2])
    D = oracle.drift(p, [0.5, 0.25], [0.1, 0.0, 0.0])
    # k = 1: neighbours 2 (f = 0.25) and 0 (inactive, 0);  k = 2: neighbours 3 (inactive) and 1 (0.5); N_1 / 2 = 2
    assert D[0] == pytest.approx(-(0.1 / HBAR) * 2 * (0.25 - 0.0), rel=1e-15)
    assert D[1] == pytest.approx(-(0.1 / HBAR) * 2 * (0.0 - 0.5), rel=1e-15)


def test_field_rk4_advects_a_fourier_mode():
    # no channels: df/dt = D[f]; cos(theta - w t) with w = F N sin(2 pi / N) / hbar solves the discretised equation
    # exactly, so RK4's error falls 16-fold when dt is halved
    grid = (12, 1, 1)
    p = _full_grid_problem(grid, nb=1)
    L = oracle.OracleList(p)
    assert L.nch == 0
    theta = 2 * np.pi * np.arange(12) / 12
    F = 0.2
    w = F * 12 * np.sin(2 * np.pi / 12) / HBAR
    errs = []
    for nsteps in (40, 80):
        dt = 4.0 / nsteps
        f, sumf = oracle.rt_step_field(L, p, 0.5 + 0.3 * np.cos(theta), p.N, [F, 0, 0], dt, nsteps)
        errs.append(np.abs(f - (0.5 + 0.3 * np.cos(theta - w * 4.0))).max())
        assert np.abs(sumf - sumf[0]).max() <= 1e-13 * sumf[0]
    assert errs[0] < 1e-4 and 12 < errs[0] / errs[1] < 20
    # with the field off the driver is the plain rt_step
    p2, L2 = make_problem("tiny", grid=(4, 4, 4), seed=5), None
    L2 = oracle.OracleList(p2)
    fa, sa = oracle.rt_step_field(L2, p2, p2.f, p2.N, [0, 0, 0], 1.0, 3)
    fb, sb = L2.rt_step(p2.f, p2.N, 1.0, 3)
    assert np.array_equal(fa, fb) and np.array_equal(sa, sb)


def test_transport_moments_closed_form():
    # states whose velocity points along one axis each, F = 2 v, f0 = 1/2: S = diag(count_al / 4 * 2), n = ns / 2
    ns = 12
    v = np.zeros((3, ns)); v[np.arange(ns) % 3, np.arange(ns)] = 1.0
    S, n = oracle.transport_moments(np.full(ns, 0.5), v, 2 * v)
    assert np.array_equal(S, np.diag([2.0, 2.0, 2.0])) and n == 6.0
    # F = c v with any v: S is symmetric; one state with v = (1, 2, 3), F = (4, 5, 6), f0 = 0.2: outer product
    rng = np.random.default_rng(5)
    v = rng.normal(size=(3, 40)); f0 = rng.uniform(0, 1, 40)
    S, _ = oracle.transport_moments(f0, v, 3.0 * v)
    assert np.allclose(S, S.T, rtol=0, atol=1e-13)
    S, n = oracle.transport_moments([0.2], [[1.0], [2.0], [3.0]], [[4.0], [5.0], [6.0]])
    assert np.allclose(S, 0.16 * np.outer([1, 2, 3], [4, 5, 6]), rtol=1e-15) and n == 0.2
