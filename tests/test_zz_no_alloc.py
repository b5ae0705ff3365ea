"""Allocation-free entry point (ephc_sum_states_noalloc): the conservation scalar sum_s f_s with its scratch in a fixed
device array of the library instead of cudaMalloc'ed memory.  Collected last on purpose (the suite runs with pytest -x).
Checked against the existing path (ephc_rt_step's sumf_dev) on two calls in a row."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
import paper_2511_03683_b200 as ephc
from ephc_inputs import make_problem

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64).reshape(-1), device="cuda")


def test_sum_states_noalloc_matches_rt_step_sum_on_two_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    # two problems of different size: the second call is smaller, so stale partial sums of the first would show
    big = make_problem("si", grid=(30, 30, 30), pair_prob=0.05, seed=21)     # 10 228 states: three blocks of partial sums
    small = make_problem("tiny", grid=(4, 4, 4), seed=5)
    assert big.ns > 4096 > small.ns              # several blocks of partial sums, then a single one
    ephc.noalloc_init()
    ephc.noalloc_init()                          # idempotent
    expected = []
    for p in (big, small):                       # the existing path: sumf[0] of ephc_rt_step (no step taken)
        h = ephc.build_channels(p)
        s = torch.zeros(1, device="cuda", dtype=torch.float64)
        h.rt_step(_dev(p.f), _dev(p.N), 1.0, 0, s)
        expected.append(float(s.cpu()[0]))
        h.close()
    fb, fs = _dev(big.f), _dev(small.f)
    out = torch.full((2,), float("nan"), device="cuda", dtype=torch.float64)
    warm = torch.zeros(1, device="cuda", dtype=torch.float64)
    ephc.sum_states_noalloc(fs, warm)            # first launch of the kernels (the driver loads their code lazily)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ephc.sum_states_noalloc(fb, out[0:1])        # two calls in a row on one stream: ordered, no race on the scratch
    ephc.sum_states_noalloc(fs, out[1:2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0  # nothing was allocated on the device
    got = out.cpu().numpy()
    for g, e, p in zip(got, expected, (big, small)):
        assert abs(g - e) <= 1e-12 * abs(e)                      # tolerance of the sumf checks in test_gpu_parity.py
        assert abs(g - float(np.sum(p.f))) <= 1e-12 * abs(e)
    # repeated: the same bits (fixed order), also after the other call used the scratch in between
    out2 = torch.full((2,), float("nan"), device="cuda", dtype=torch.float64)
    ephc.sum_states_noalloc(fs, out2[1:2])
    ephc.sum_states_noalloc(fb, out2[0:1])
    assert torch.equal(out, out2)
    # a prefix, n = 0, and a non-default stream
    st = torch.cuda.Stream()
    o3 = torch.full((2,), float("nan"), device="cuda", dtype=torch.float64)
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        ephc.sum_states_noalloc(fb, o3[0:1], n=5000, stream=st)
        ephc.sum_states_noalloc(fb, o3[1:2], n=0, stream=st)
    st.synchronize()
    r = o3.cpu().numpy()
    assert abs(r[0] - float(np.sum(big.f.reshape(-1)[:5000]))) <= 1e-12 * abs(expected[0]) and r[1] == 0.0


def test_sum_states_noalloc_rejects_sizes_beyond_the_fixed_scratch():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    nmax = ephc.noalloc_max_states()
    assert nmax == 4096 * 4096
    f = torch.ones(8, device="cuda", dtype=torch.float64)
    out = torch.full((1,), -1.0, device="cuda", dtype=torch.float64)
    with pytest.raises(ephc.EphcError) as ei:
        ephc.sum_states_noalloc(f, out, n=nmax + 1)   # rejected before anything is read or launched
    assert ei.value.code == -5 and "exceeds" in str(ei.value)
    with pytest.raises(ephc.EphcError):
        ephc.sum_states_noalloc(f, out, n=-1)
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == -1.0
