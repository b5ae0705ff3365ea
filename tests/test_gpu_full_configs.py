"""Full-size runs of BASELINE.json configs 3 (gaas, 1.9e8 channels) and 4 (bigcell, 5e7 channels, nb = 16, nnu = 36)
in the default launch configuration (-m gpu).  The channel list is compared bit for bit with the oracle's, every
element of I, Gamma, F' and f(t) with the list oracle, sampled states with the definition-level oracle; the timings
are printed (pytest -s)."""
import os
import time

import numpy as np
import pytest

import oracle
import paper_2511_03683_b200 as ephc
from ephc_inputs import make_problem

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-11
PEAK_GBS = 6543.1  # MEASURED_PEAKS.json hbm_gbs (context for the printed fractions only)


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1), device="cuda")


def _rel(a, b):
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(b).max())


def _time_us(fn, n=5):
    fn()
    torch.cuda.synchronize()
    s, e = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s.record()
    for _ in range(n):
        fn()
    e.record()
    torch.cuda.synchronize()
    return s.elapsed_time(e) / n * 1e3


def _assert_same_list(h, L):
    # north_star: channel lists and indices match the oracle bit for bit; weights within 4 ulp (two exp implementations)
    a, b = h.export_channels(), L.export()
    for k in ("ik", "ikq", "iq", "n", "m", "nu"):
        assert np.array_equal(a[k], b[k]), k
        a[k] = b[k] = None
    for k in ("w_abs", "w_em"):
        assert np.all(np.abs(a[k] - b[k]) <= 4 * np.spacing(np.maximum(np.abs(a[k]), np.abs(b[k])))), k
        assert np.array_equal(a[k] == 0.0, b[k] == 0.0), k
        a[k] = b[k] = None


@pytest.mark.parametrize("name", ["bigcell", "gaas"])
def test_full_size_config_matches_oracle(name):
    p = make_problem(name)
    t0 = time.perf_counter()
    h = ephc.build_channels(p)
    t_build = time.perf_counter() - t0
    q = h.query()
    L = oracle.OracleList(p)
    assert L.nch == q["nch"] > 4.0e7
    _assert_same_list(h, L)
    f, f0, N, v = _dev(p.f), _dev(p.f0), _dev(p.N), _dev(p.v)
    I = torch.empty(p.ns, device="cuda", dtype=torch.float64)
    h.collision(f, N, I)
    got = I.cpu().numpy()
    Io = L.collision(p.f, p.N)
    assert _rel(got, Io) <= TOL
    assert abs(got.sum()) <= 1e-12 * np.abs(got).sum()
    st = np.random.default_rng(3).choice(np.flatnonzero(Io != 0.0), 8, replace=False).astype(np.int32)
    assert np.abs(got[st] - oracle.collision_sampled(p, p.f, p.N, st)).max() <= TOL * np.abs(Io).max()
    us_c = _time_us(lambda: h.collision(f, N, I))
    G = torch.empty(p.ns, device="cuda", dtype=torch.float64)
    h.transport_setup(f0, N, G)
    Go = L.transport_setup(p.f0, p.N)
    assert _rel(G.cpu().numpy(), Go) <= TOL
    tau_o = np.where(Go > 0, 1.0 / np.where(Go > 0, Go, 1.0), 0.0)
    Fr = tau_o[None, :] * p.v
    Fa, Fb, tau = _dev(Fr), torch.empty(3 * p.ns, device="cuda", dtype=torch.float64), _dev(tau_o)
    h.transport_iter(Fa, v, tau, Fb)
    assert _rel(Fb.cpu().numpy().reshape(3, -1), L.transport_iter(p.f0, p.N, Fr, p.v, tau_o)) <= TOL
    us_t = _time_us(lambda: h.transport_iter(Fa, v, tau, Fb))
    fr = _dev(p.f)
    sumf = torch.zeros(3, device="cuda", dtype=torch.float64)
    h.rt_step(fr, N, 1.0, 2, sumf)
    fo, so = L.rt_step(p.f, p.N, 1.0, 2)
    assert _rel(fr.cpu().numpy(), fo) <= TOL
    assert np.abs(sumf.cpu().numpy() - so).max() <= 1e-12 * abs(so[0])
    print(f"\n{name}: nch={q['nch']:.4g} build {t_build:.1f} s, variants {h.get_variant()}/{h.get_transport_variant()}; "
          f"collision {us_c:.0f} us = {q['alg_bytes_collision'] / us_c / 1e3 / PEAK_GBS:.3f} of the roofline, "
          f"transport_iter {us_t:.0f} us = {q['alg_bytes_transport'] / us_t / 1e3 / PEAK_GBS:.3f}")


def test_config5_thousand_steps_conserve_particle_number():
    # BASELINE.json configs[4]: config[1]'s channel set, hot-electron initial f, RK4 dt = 1 fs, 1000 steps (4000 collision
    # evaluations); electron number checked after EVERY step; a second run gives the same bits
    p = make_problem("rt")
    h = ephc.build_channels(p)
    N = _dev(p.N)
    nsteps = 1000
    out = []
    for _ in range(2):
        f = _dev(p.f)
        sumf = torch.zeros(nsteps + 1, device="cuda", dtype=torch.float64)
        t0 = time.perf_counter()
        h.rt_step(f, N, 1.0, nsteps, sumf)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        out.append((f.cpu().numpy(), sumf.cpu().numpy()))
    fa, sa = out[0]
    assert np.isfinite(fa).all() and np.abs(fa - p.f).max() > 1e-3
    assert sa[0] == pytest.approx(p.f.sum(), rel=1e-13)
    assert np.abs(sa - sa[0]).max() <= 1e-12 * abs(sa[0])
    assert np.array_equal(fa, out[1][0]) and np.array_equal(sa, out[1][1])
    print(f"\nrt: 1000 RK4 steps in {dt:.2f} s, max |sum f - sum f0| / sum f0 = {np.abs(sa - sa[0]).max() / abs(sa[0]):.2e}")
    # the first 50 steps, every element, against the oracle (about 20 s of CPU)
    L = oracle.OracleList(p)
    assert L.nch == h.query()["nch"]
    _assert_same_list(h, L)
    f = _dev(p.f)
    s50 = torch.zeros(51, device="cuda", dtype=torch.float64)
    h.rt_step(f, N, 1.0, 50, s50)
    fo, so = L.rt_step(p.f, p.N, 1.0, 50)
    assert _rel(f.cpu().numpy(), fo) <= TOL
    assert np.abs(s50.cpu().numpy() - so).max() <= 1e-12 * abs(so[0])
    assert np.array_equal(s50.cpu().numpy(), sa[:51])


def test_config5_thousand_steps_match_oracle_on_a_small_copy():
    # the whole 1000-step trajectory, element by element, where the oracle takes seconds (14^3 copy of the rt config)
    p = make_problem("rt", grid=(14, 14, 14), pair_prob=0.3, seed=8)
    L = oracle.OracleList(p)
    fo, so = L.rt_step(p.f, p.N, 1.0, 1000)
    for variant in (-1, 2, 3):
        h = ephc.build_channels(p)
        h.set_variant(variant)
        f = _dev(p.f)
        sumf = torch.zeros(1001, device="cuda", dtype=torch.float64)
        h.rt_step(f, _dev(p.N), 1.0, 1000, sumf)
        assert _rel(f.cpu().numpy(), fo) <= TOL
        assert np.abs(sumf.cpu().numpy() - so).max() <= 1e-12 * abs(so[0])
        assert np.abs(sumf.cpu().numpy() - so[0]).max() <= 1e-12 * abs(so[0])
