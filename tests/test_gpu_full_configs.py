"""Full-size runs of BASELINE.json configs 3 (gaas) and 4 (bigcell) in the default launch configuration (-m gpu).
bigcell (5e7 channels, nb = 16, nnu = 36) runs always; gaas (1.9e8 channels, 36 GB of host memory, about two
minutes) only with EPHC_FULL_CONFIGS=1.  Every element of I, Gamma, F' and f(t) is compared with the list oracle;
the timings are printed (pytest -s) and recorded in profiles/r1e_launches.md."""
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


@pytest.mark.parametrize("name", ["bigcell", "gaas"])
def test_full_size_config_matches_oracle(name):
    if name == "gaas" and os.environ.get("EPHC_FULL_CONFIGS") != "1":
        pytest.skip("set EPHC_FULL_CONFIGS=1 (needs 36 GB of host memory and about two minutes)")
    p = make_problem(name)
    t0 = time.perf_counter()
    h = ephc.build_channels(p)
    t_build = time.perf_counter() - t0
    q = h.query()
    L = oracle.OracleList(p)
    assert L.nch == q["nch"] > 4.0e7
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
