"""Host logic of the library, no GPU: the C ABI loads and exports what include/ephc.h declares, channel
selection reproduces the oracle's canonical list bit for bit, the two-sided store covers every ordered
term exactly once, and bad input is rejected with the documented error codes."""
import os
import re

import numpy as np
import pytest

import oracle
import paper_2511_03683_b200 as ephc
from ephc_inputs import make_problem, bose_einstein
from helpers import manual_problem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _ulp_close(a, b, ulps):
    a = np.asarray(a); b = np.asarray(b)
    return np.all(np.abs(a - b) <= ulps * np.spacing(np.maximum(np.abs(a), np.abs(b))))


def test_abi_exports_every_declared_symbol():
    import ctypes
    hdr = open(os.path.join(ROOT, "include", "ephc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(ephc_[a-z_]+)\s*\(", hdr))
    assert {"ephc_build_channels", "ephc_collision", "ephc_transport_iter", "ephc_rt_step"} <= names
    lib = ctypes.CDLL(ephc.lib_path())
    for n in sorted(names):
        assert hasattr(lib, n), f"{n} declared in include/ephc.h but not exported"
    assert "sm_100a" in ephc.version()


def _small_problems():
    out = [make_problem("tiny", grid=(4, 4, 4), seed=5)]
    p = make_problem("tiny", grid=(4, 4, 4), window=(0.08, 0.22), seed=99)
    p.g2_cut = float(np.quantile(p.g2, 0.2))
    p.hw[...] = p.hw * 0.5
    p.N = bose_einstein(p.hw, 300.0).reshape(-1)
    out.append(p)
    out.append(make_problem("si", grid=(12, 12, 12), pair_prob=0.3, seed=3))
    out.append(make_problem("gaas", grid=(24, 24, 24), pair_prob=0.5, seed=4, window=(0.0, 0.5)))
    out.append(make_problem("bigcell", grid=(3, 3, 3), pair_prob=0.2, seed=6))
    return out


@pytest.fixture(scope="module", params=range(5), ids=["tiny4", "window_cut_diag", "si12", "gaas24", "bigcell3"])
def prob(request):
    return _small_problems()[request.param]


def test_canonical_list_matches_oracle_bit_exact(prob):
    L = oracle.OracleList(prob)
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    q = h.query()
    assert q["nch"] == L.nch and q["ndiag"] == L.ndiag and q["nw"] == L.nw and q["ns"] == prob.ns
    assert L.nch > 0
    a, b = h.export_channels(), L.export()
    for k in ("ik", "ikq", "iq", "n", "m", "nu"):
        assert np.array_equal(a[k], b[k]), k
    for k in ("w_abs", "w_em"):
        assert np.array_equal(a[k] == 0.0, b[k] == 0.0), k       # the decision "delta is cut" is exact
        assert _ulp_close(a[k], b[k], 4), k
    da, db = h.export_diag(), L.export_diag()
    for k in ("s", "iq", "nu"):
        assert np.array_equal(da[k], db[k]), k
    assert _ulp_close(da["w_abs"], db["w_abs"], 4) and _ulp_close(da["w_em"], db["w_em"], 4)


def test_gather_store_holds_every_ordered_term_once(prob):
    L = oracle.OracleList(prob)
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    g = h.export_gather()                      # also checks: every entry covered by exactly one task
    q = h.query()
    ch, dg = L.export(), L.export_diag()
    nw_d = int((dg["w_abs"] != 0).sum() + (dg["w_em"] != 0).sum())
    assert q["gather_entries"] == 2 * L.nw + nw_d
    # multiset of ordered terms expected from the oracle's list: (dest, partner, iq, nu, kind, diag, w)
    a = ch["ik"] * prob.nb + ch["n"]
    b = ch["ikq"] * prob.nb + ch["m"]
    rows = []
    for wk, kd in (("w_abs", 0), ("w_em", 1)):
        sel = ch[wk] != 0
        rows.append(np.stack([a[sel], b[sel], ch["iq"][sel], ch["nu"][sel], np.full(sel.sum(), kd), np.zeros(sel.sum(), int)]))
        rows.append(np.stack([b[sel], a[sel], ch["iq"][sel], ch["nu"][sel], np.full(sel.sum(), 1 - kd), np.zeros(sel.sum(), int)]))
        seld = dg[wk] != 0
        rows.append(np.stack([dg["s"][seld], dg["s"][seld], dg["iq"][seld], dg["nu"][seld], np.full(seld.sum(), kd), np.ones(seld.sum(), int)]))
    exp = np.concatenate(rows, axis=1).astype(np.int64)
    got = np.stack([g[k] for k in ("dest", "partner", "iq", "nu", "kind", "diag")]).astype(np.int64)
    assert exp.shape == got.shape
    oe = np.lexsort(exp[::-1]); og = np.lexsort(got[::-1])
    assert np.array_equal(exp[:, oe], got[:, og])
    # rows are contiguous runs per task; destinations never decrease inside a work unit's round order is not
    # required, but a destination state must be owned by exactly one work unit: checked by export_gather.
    # The store, evaluated with numpy, reproduces the oracle's collision integral and transport rates.
    f, N = prob.f, prob.N
    fa, fb, Nq = f[g["dest"]], f[g["partner"]], N[g["iq"].astype(np.int64) * prob.nnu + g["nu"]]
    out_, in_ = fa * (1 - fb), fb * (1 - fa)
    F = np.where(g["kind"] == 1, out_ * (Nq + 1) - in_ * Nq, out_ * Nq - in_ * (Nq + 1))
    I = np.zeros(prob.ns)
    np.add.at(I, g["dest"], np.where(g["diag"] == 1, 0.0, -g["w"] * F))
    Io = L.collision(f, N)
    assert np.abs(I - Io).max() <= 1e-12 * np.abs(Io).max()
    f0 = prob.f0
    W = np.where(g["kind"] == 1, g["w"] * (1 + Nq - f0[g["partner"]]), g["w"] * (Nq + f0[g["partner"]]))
    G = np.zeros(prob.ns)
    np.add.at(G, g["dest"], W)
    Go = L.transport_setup(f0, N)
    assert np.abs(G - Go).max() <= 1e-12 * Go.max()


@pytest.mark.parametrize("rows,ctas", [(None, None), (8, 5), (16, 64), (2048, 1)])
def test_tile_store_holds_every_channel_once(prob, rows, ctas, monkeypatch):
    if rows is not None:
        monkeypatch.setenv("EPHC_TILE_ROWS", str(rows))
        monkeypatch.setenv("EPHC_TILE_CTAS", str(ctas))
    L = oracle.OracleList(prob)
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    q = h.query()
    if prob.nb > 4 or prob.nnu > 8:
        assert q["scatter_entries"] == 0 and h.get_variant() == 0       # no tile store; small problem: gather store
        with pytest.raises(ephc.EphcError):
            h.set_variant(1)
        return
    h.set_variant(1)
    assert h.get_variant() == 1
    t = h.export_tiles()      # also checks tickets, slots, lane order and that every entry is covered once
    ch, dg = L.export(), L.export_diag()
    nw_d = int((dg["w_abs"] != 0).sum() + (dg["w_em"] != 0).sum())
    assert q["scatter_entries"] == L.nw + nw_d
    a = ch["ik"] * prob.nb + ch["n"]
    b = ch["ikq"] * prob.nb + ch["m"]
    rows_, ws = [], []
    for wk, kd in (("w_abs", 0), ("w_em", 1)):
        sel = ch[wk] != 0
        rows_.append(np.stack([a[sel], b[sel], ch["iq"][sel], ch["nu"][sel], np.full(sel.sum(), kd), np.zeros(sel.sum(), int)]))
        ws.append(ch[wk][sel])
        seld = dg[wk] != 0
        rows_.append(np.stack([dg["s"][seld], dg["s"][seld], dg["iq"][seld], dg["nu"][seld], np.full(seld.sum(), kd), np.ones(seld.sum(), int)]))
        ws.append(dg[wk][seld])
    exp = np.concatenate(rows_, axis=1).astype(np.int64)
    expw = np.concatenate(ws)
    got = np.stack([t[k] for k in ("a", "b", "iq", "nu", "kind", "diag")]).astype(np.int64)
    assert exp.shape == got.shape
    oe = np.lexsort(exp[::-1]); og = np.lexsort(got[::-1])
    assert np.array_equal(exp[:, oe], got[:, og])
    assert _ulp_close(t["w"][og], expw[oe], 4)
    # the store, evaluated with numpy in Eq. 2's printed form, reproduces the oracle's collision integral
    f, N = prob.f, prob.N
    fa, fb, Nq = f[t["a"]], f[t["b"]], N[t["iq"].astype(np.int64) * prob.nnu + t["nu"]]
    out_, in_ = fa * (1 - fb), fb * (1 - fa)
    T = t["w"] * np.where(t["kind"] == 1, out_ * (Nq + 1) - in_ * Nq, out_ * Nq - in_ * (Nq + 1))
    T = np.where(t["diag"] == 1, 0.0, T)
    I = np.zeros(prob.ns)
    np.add.at(I, t["a"], -T)
    np.add.at(I, t["b"], T)
    Io = L.collision(f, N)
    assert np.abs(I - Io).max() <= 1e-12 * np.abs(Io).max()


@pytest.mark.parametrize("rows,fine,ctas", [(None, None, None), (16, 4, 3), (64, 8, 40), (2048, 128, 1)])
def test_stream_store_holds_every_channel_once(prob, rows, fine, ctas, monkeypatch):
    if rows is not None:
        monkeypatch.setenv("EPHC_STREAM_ROWS", str(rows))
        monkeypatch.setenv("EPHC_STREAM_ROWS_B", str(rows))
        monkeypatch.setenv("EPHC_STREAM_FINE", str(fine))
        monkeypatch.setenv("EPHC_STREAM_CTAS", str(ctas))
    L = oracle.OracleList(prob)
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    t = h.export_stream()     # also checks chunk limits, row tasks, permutations, slots and coverage
    ch = L.export()
    assert len(t["w"]) == L.nw
    a = ch["ik"] * prob.nb + ch["n"]
    b = ch["ikq"] * prob.nb + ch["m"]
    rows_, ws = [], []
    for wk, kd in (("w_abs", 0), ("w_em", 1)):
        sel = ch[wk] != 0
        rows_.append(np.stack([a[sel], b[sel], ch["iq"][sel], ch["nu"][sel], np.full(sel.sum(), kd)]))
        ws.append(ch[wk][sel])
    exp = np.concatenate(rows_, axis=1).astype(np.int64)
    expw = np.concatenate(ws)
    got = np.stack([t[k] for k in ("a", "b", "iq", "nu", "kind")]).astype(np.int64)
    assert exp.shape == got.shape
    oe = np.lexsort(exp[::-1]); og = np.lexsort(got[::-1])
    assert np.array_equal(exp[:, oe], got[:, og])
    assert _ulp_close(t["w"][og], expw[oe], 4)
    # the store, evaluated with numpy in Eq. 2's printed form, reproduces the oracle's collision integral
    f, N = prob.f, prob.N
    fa, fb, Nq = f[t["a"]], f[t["b"]], N[t["iq"].astype(np.int64) * prob.nnu + t["nu"]]
    out_, in_ = fa * (1 - fb), fb * (1 - fa)
    T = t["w"] * np.where(t["kind"] == 1, out_ * (Nq + 1) - in_ * Nq, out_ * Nq - in_ * (Nq + 1))
    I = np.zeros(prob.ns)
    np.add.at(I, t["a"], -T)
    np.add.at(I, t["b"], T)
    Io = L.collision(f, N)
    assert np.abs(I - Io).max() <= 1e-12 * np.abs(Io).max()


@pytest.mark.parametrize("rows,fine,smem,hcap,mode", [(None, None, None, None, None), (16, 4, 16000, 1, 1), (64, 8, 24000, 2, 4),
                                                      (512, 128, None, 3, 6), (32, 32, 20000, 200, 2)])
def test_res_store_holds_every_weight_once(prob, rows, fine, smem, hcap, mode, monkeypatch):
    # resident-tile store (variant 3): default geometry, and forced geometries with many tiny tiles, tiles split by
    # the shared-memory budget, rows cut into many one- to three-element pieces (several lanes per row), other launch modes
    if rows is not None:
        monkeypatch.setenv("EPHC_RES_ROWS", str(rows))
        monkeypatch.setenv("EPHC_RES_ROWS_B", str(rows))
        monkeypatch.setenv("EPHC_RES_FINE", str(fine))
    for k, v in (("EPHC_RES_SMEM", smem), ("EPHC_RES_HCAP", hcap), ("EPHC_RES_MODE", mode)):
        if v is not None:
            monkeypatch.setenv(k, str(v))
    if mode in (1, 4, 6):
        # the schedule re-cut that device handles do from measured tile times (res_reschedule), here with pseudo-random
        # costs: the export below checks runs, flags, slots and slot lists of the new shares
        monkeypatch.setenv("EPHC_RES_TEST_RECUT", str(mode))
    L = oracle.OracleList(prob)
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    t = h.export_res()        # also checks the tile images: slabs of both phases, padding, gather lists, slots, coverage
    ch = L.export()
    assert len(t["w"]) == L.nw
    a = ch["ik"] * prob.nb + ch["n"]
    b = ch["ikq"] * prob.nb + ch["m"]
    rows_, ws = [], []
    for wk, kd in (("w_abs", 0), ("w_em", 1)):
        sel = ch[wk] != 0
        rows_.append(np.stack([a[sel], b[sel], ch["iq"][sel], ch["nu"][sel], np.full(sel.sum(), kd)]))
        ws.append(ch[wk][sel])
    exp = np.concatenate(rows_, axis=1).astype(np.int64)
    expw = np.concatenate(ws)
    got = np.stack([t[k] for k in ("a", "b", "iq", "nu", "kind")]).astype(np.int64)
    assert exp.shape == got.shape
    oe = np.lexsort(exp[::-1]); og = np.lexsort(got[::-1])
    assert np.array_equal(exp[:, oe], got[:, og])
    assert _ulp_close(t["w"][og], expw[oe], 4)
    # evaluated with numpy in Eq. 2's printed form, the store reproduces the oracle's collision integral
    f, N = prob.f, prob.N
    fa, fb, Nq = f[t["a"]], f[t["b"]], N[t["iq"].astype(np.int64) * prob.nnu + t["nu"]]
    out_, in_ = fa * (1 - fb), fb * (1 - fa)
    T = t["w"] * np.where(t["kind"] == 1, out_ * (Nq + 1) - in_ * Nq, out_ * Nq - in_ * (Nq + 1))
    I = np.zeros(prob.ns)
    np.add.at(I, t["a"], -T)
    np.add.at(I, t["b"], T)
    Io = L.collision(f, N)
    assert np.abs(I - Io).max() <= 1e-12 * np.abs(Io).max()


@pytest.mark.parametrize("rng_rows,strips,sparse", [(None, None, None), (32, 1, None), (64, 3, None), (32, 40, None), (32, 5, 1),
                                                    (64, 40, 1), (None, None, 1)])
def test_row_store_is_a_regrouping_of_the_gather_store(prob, rng_rows, strips, sparse, monkeypatch):
    # the store transport_iter runs on: same ordered terms as the gather store (dest, partner), every gather position
    # exactly once; strips / tiles / segments (and, with sparse staging, the strips' partner lists) checked in C
    # (ephc_export_rows)
    if rng_rows is not None:
        monkeypatch.setenv("EPHC_ROW_RANGE", str(rng_rows))
        monkeypatch.setenv("EPHC_ROW_STRIPS", str(strips))
    if sparse is not None:
        monkeypatch.setenv("EPHC_ROW_SPARSE", str(sparse))
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY)
    g, r = h.export_gather(), h.export_rows()
    assert len(r["dest"]) == len(g["dest"]) > 0
    assert np.array_equal(np.sort(r["gather_pos"]), np.arange(len(g["dest"])))
    assert np.array_equal(g["dest"][r["gather_pos"]], r["dest"])
    assert np.array_equal(g["partner"][r["gather_pos"]], r["partner"])
    # destination-sorted at strip granularity: the destinations of the store are non-decreasing across strips
    inside = (prob.E.reshape(-1) >= prob.emin) & (prob.E.reshape(-1) <= prob.emax)
    assert inside[r["dest"]].all() and inside[r["partner"]].all()


@pytest.mark.parametrize("rng_rows,strips", [(None, None), (32, 3), (64, 40), (-32, 7)])
def test_collapsed_row_store_sums_every_ordered_term_once(prob, rng_rows, strips, monkeypatch):
    # mode-collapsed specialisation: one entry per (destination, partner) state pair of a segment; the counts are the
    # multiplicities of the pairs in the row store; coverage and adjacency checked in C (ephc_export_rows_collapsed)
    if rng_rows is not None:
        if rng_rows < 0:     # negative: the same range with sparse staging forced
            monkeypatch.setenv("EPHC_ROW_SPARSE", "1")
        monkeypatch.setenv("EPHC_ROW_RANGE", str(abs(rng_rows)))
        monkeypatch.setenv("EPHC_ROW_STRIPS", str(strips))
    h = ephc.build_channels(prob, flags=ephc.HOST_ONLY | ephc.TRANSPORT_COLLAPSE)
    r, c = h.export_rows(), h.export_rows_collapsed()
    assert 0 < len(c["dest"]) <= len(r["dest"]) and c["count"].sum() == len(r["dest"])
    ns = prob.nk * prob.nb
    key_r = r["dest"].astype(np.int64) * ns + r["partner"]
    key_c = c["dest"].astype(np.int64) * ns + c["partner"]
    uniq, cnt = np.unique(key_r, return_counts=True)
    order = np.argsort(key_c, kind="stable")
    assert np.array_equal(key_c[order], uniq) and np.array_equal(c["count"][order], cnt)   # one entry per state pair
    with pytest.raises(ephc.EphcError):
        ephc.build_channels(prob, flags=ephc.HOST_ONLY).export_rows_collapsed()


def test_launch_geometry_limits():
    # a segment with more half-pairs than one round can stage (tiny 8x8x8: 512 partners per k, 5 doubles each)
    # and a dense many-band block: both must split into rounds/tasks within the kernel's limits
    p = make_problem("tiny")
    h = ephc.build_channels(p, flags=ephc.HOST_ONLY)
    q = h.query()
    assert q["n_workunits"] >= 1 and q["n_rounds"] >= q["n_workunits"] and q["n_tasks"] >= q["n_rounds"]
    g = h.export_gather()
    assert len(g["w"]) == q["gather_entries"] and q["nch"] > 3e5
    # every state is owned by one work unit: destinations of a work unit are a contiguous k range (checked in C)
    assert np.all(np.diff(np.unique(g["dest"])) > 0)


def test_segments_split_over_several_rounds(monkeypatch):
    # force the multi-round path (a k segment whose half-pairs exceed one round's staging buffer), as the
    # full-size GaAs-like config does, on a small problem: 7 half-pairs per round
    monkeypatch.setenv("EPHC_ROUND_PAIRS", "7")
    monkeypatch.setenv("EPHC_WU_ENTRIES", "300")
    for p in _small_problems()[:4]:
        L = oracle.OracleList(p)
        h = ephc.build_channels(p, flags=ephc.HOST_ONLY)
        q = h.query()
        assert q["n_rounds"] > 2 * q["n_workunits"] and q["n_workunits"] == p.nk
        g = h.export_gather()
        f, N = p.f, p.N
        fa, fb, Nq = f[g["dest"]], f[g["partner"]], N[g["iq"].astype(np.int64) * p.nnu + g["nu"]]
        out_, in_ = fa * (1 - fb), fb * (1 - fa)
        F = np.where(g["kind"] == 1, out_ * (Nq + 1) - in_ * Nq, out_ * Nq - in_ * (Nq + 1))
        I = np.zeros(p.ns)
        np.add.at(I, g["dest"], np.where(g["diag"] == 1, 0.0, -g["w"] * F))
        Io = L.collision(f, N)
        assert np.abs(I - Io).max() <= 1e-12 * np.abs(Io).max()


def test_empty_and_degenerate_inputs():
    # no candidate pairs at all
    p = manual_problem((2, 1, 1), E=[[0.0], [0.1]], hw=[[0.02], [0.02]], pairs=[], g2=np.zeros((0, 1, 1, 1)), sigma=0.01)
    h = ephc.build_channels(p, flags=ephc.HOST_ONLY)
    q = h.query()
    assert q["nch"] == 0 and q["gather_entries"] == 0 and q["ns"] == 2
    # candidate pairs but nothing conserves energy
    p = manual_problem((2, 1, 1), E=[[0.0], [1.0]], hw=[[0.02], [0.02]], pairs=[(0, 1)], g2=np.ones((1, 1, 1, 1)), sigma=0.01)
    assert ephc.build_channels(p, flags=ephc.HOST_ONLY).query()["nch"] == 0
    # only a diagonal term (q = 0, n == m): hw < 3 sigma
    p = manual_problem((1, 1, 1), E=[[0.0]], hw=[[0.02]], pairs=[(0, 0)], g2=np.ones((1, 1, 1, 1)), sigma=0.01)
    q = ephc.build_channels(p, flags=ephc.HOST_ONLY).query()
    assert q["nch"] == 0 and q["ndiag"] == 1 and q["gather_entries"] == 2
    assert oracle.OracleList(p).ndiag == 1


def test_error_codes():
    p = make_problem("tiny", grid=(2, 2, 2), seed=1)
    bad = make_problem("tiny", grid=(2, 2, 2), seed=1); bad.hw[0, 0] = -1.0
    with pytest.raises(ephc.EphcError) as e:
        ephc.build_channels(bad, flags=ephc.HOST_ONLY)
    assert e.value.code == -1
    bad = make_problem("tiny", grid=(2, 2, 2), seed=1); bad.E[0, 0] = np.nan
    with pytest.raises(ephc.EphcError):
        ephc.build_channels(bad, flags=ephc.HOST_ONLY)
    bad = make_problem("tiny", grid=(2, 2, 2), seed=1); bad.pair_ik = bad.pair_ik[::-1].copy()
    with pytest.raises(ephc.EphcError) as e:
        ephc.build_channels(bad, flags=ephc.HOST_ONLY)
    assert e.value.code == -1 and "pair list" in str(e.value)
    bad = make_problem("tiny", grid=(2, 2, 2), seed=1); bad.kfull = bad.kfull[::-1].copy()
    with pytest.raises(ephc.EphcError):
        ephc.build_channels(bad, flags=ephc.HOST_ONLY)
    bad = make_problem("tiny", grid=(2, 2, 2), seed=1); bad.sigma = 0.0
    with pytest.raises(ephc.EphcError):
        ephc.build_channels(bad, flags=ephc.HOST_ONLY)
    # format limit
    big = manual_problem((1, 1, 1), E=np.zeros((1, 17)), hw=[[0.02]], pairs=[], g2=np.zeros((0, 1, 17, 17)), sigma=0.01)
    with pytest.raises(ephc.EphcError) as e:
        ephc.build_channels(big, flags=ephc.HOST_ONLY)
    assert e.value.code == -5
    # compute on a host-only handle fails loudly (no CPU fallback)
    h = ephc.build_channels(p, flags=ephc.HOST_ONLY)
    with pytest.raises(ephc.EphcError) as e:
        h.collision_host(p.f, p.N, np.zeros(p.ns))
    assert e.value.code == -4
    with pytest.raises(TypeError):
        h.collision(p.f, p.N, np.zeros(p.ns))            # device entry points refuse host arrays


def test_no_device_means_error_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    p = make_problem("tiny", grid=(2, 2, 2), seed=1)
    with pytest.raises(ephc.EphcError) as e:
        ephc.build_channels(p)
    assert e.value.code == -3
