"""The allocation-free entry point qmc_batch_stats_static (fixed file-scope device scratch) against the existing
qmc_batch_stats, through the C ABI.  Collected last on purpose: the suite runs with `pytest -x`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def test_batch_stats_static_matches_batch_stats_on_two_calls_in_a_row():
    import torch
    from oracle import binding as ob
    from paper_2506_09743_b200 import binding as qb
    assert torch.cuda.is_available()
    rng = np.random.default_rng(41)
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    # two calls in a row on different data and sizes (the shared scratch keeps the first call's contents), then ragged
    # and tiny sizes; tolerances of tests/test_gpu_parity.py::test_batch_stats
    for M, shift in ((100003, -40.0), (65537, 17.5), (1, 2.0), (255, -3.0), (257, 1e3), (1 << 20, -79.6)):
        x = rng.standard_normal(M) * 3 + shift
        xg = torch.from_numpy(x).cuda()
        m0, s0 = qb.batch_stats(xg)                      # the existing path
        out.fill_(float("nan"))
        qb.batch_stats_static(xg, out)
        torch.cuda.synchronize()
        m, s = (float(v) for v in out.cpu())
        assert abs(m - m0) <= 1e-12 * abs(m0), (M, m, m0)
        assert abs(s - s0) <= 1e-10 * max(s0, 1e-300), (M, s, s0)
        mo, so = ob.batch_stats(x)                       # and the oracle
        assert abs(m - mo) <= 1e-12 * abs(mo) and abs(s - so) <= 1e-10 * max(so, 1e-300)
    # repeatable bit for bit
    a = qb.batch_stats_static(xg, torch.empty(2, dtype=torch.float64, device="cuda")).clone()
    b = qb.batch_stats_static(xg, torch.empty(2, dtype=torch.float64, device="cuda")).clone()
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    # beyond the fixed scratch's limit: a clear error, nothing launched
    L = qb.lib()
    rc = L.qmc_batch_stats_static(xg.data_ptr(), (1 << 26) + 1, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    assert rc == qb.QMC_ETOOLARGE and b"67108864" in L.qmc_status_string(rc)
    assert L.qmc_batch_stats_static(xg.data_ptr(), 0, out.data_ptr(), None) == qb.QMC_EINVAL
    assert L.qmc_static_scratch_init(0) == qb.QMC_OK


def test_batch_stats_static_allocates_nothing_and_can_be_captured():
    import torch
    from paper_2506_09743_b200 import binding as qb
    x = torch.from_numpy(np.random.default_rng(42).standard_normal(50021) - 5.0).cuda()
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    assert qb.lib().qmc_static_scratch_init(torch.cuda.current_device()) == qb.QMC_OK
    qb.batch_stats_static(x, out)
    torch.cuda.synchronize()
    want = out.clone()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        qb.batch_stats_static(x, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0            # device memory in use did not change
    # under stream capture (where cudaMalloc is not allowed), replayed twice in sequence
    st = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    out.zero_()
    with torch.cuda.stream(st):
        g.capture_begin()
        qb.batch_stats_static(x, out, stream=st)
        g.capture_end()
    for _ in range(2):
        out.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, want)
