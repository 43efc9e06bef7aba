"""The no-allocation entry point pf_relax_noalloc (include/pf_noalloc.h): row N5, Table 2 step 5, with
its scratch in a file-scope device array of the library instead of per-grid allocated memory.  Checked against the
existing path -- the kernel and per-grid scratch that pf_solve_pf uses, reached alone through pf_grid_relax -- on two
calls in a row (the shared scratch keeps the first call's contents).  The arithmetic is the same statement for
statement, so the relaxed field is compared bit for bit and the increment exactly.

In a file of its own that pytest collects last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def pf():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1711_04060_b200 import build as _build, pf as _pf
    _build.build()
    _pf.load()
    return _pf


def _existing_path(pf, shape, omega, phi0, phi):
    nx, ny, nz = shape
    n = nx * ny * nz
    g = pf.Grid(nx, ny, nz, 0.5, np.full(n, 78.5), np.zeros((0, 4)), np.zeros(6, dtype=np.int32), np.zeros(6))
    out = phi.clone()
    d = pf.pf_grid_relax(g.handle, n, omega, phi0, out)
    g.close()
    return out, d


def test_no_alloc_entry_point_matches_existing_path_on_two_calls_in_a_row(pf):
    rng = np.random.default_rng(17)
    incr = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    # first call: 70 x 61 x 53 = 226 310 nodes (56 blocks of the no-alloc kernel, a ragged last one);
    # second call: smaller (stale partial results of the first call sit behind its own) and with another omega_PF
    for shape, omega in (((70, 61, 53), 0.3), ((33, 20, 11), 0.55)):
        n = shape[0] * shape[1] * shape[2]
        phi0 = torch.from_numpy(rng.standard_normal(n) * 5.0).cuda()
        phi = torch.from_numpy(rng.standard_normal(n) * 5.0).cuda()
        ref_phi, ref_d = _existing_path(pf, shape, omega, phi0, phi)
        out = phi.clone()
        pf.pf_relax_noalloc(n, omega, phi0, out, incr)
        torch.cuda.synchronize()
        assert torch.equal(out, ref_phi)                       # same statements: same bits
        assert float(incr.item()) == ref_d and ref_d > 0.0
        # and against the definition, in numpy
        p0, p1 = phi0.cpu().numpy(), phi.cpu().numpy()
        expect = omega * p0 + (1.0 - omega) * p1
        assert np.allclose(out.cpu().numpy(), expect, rtol=1e-15, atol=0)
        assert np.isclose(ref_d, np.abs(expect - p0).max(), rtol=1e-14)


def test_no_alloc_entry_point_limits_and_edge_cases(pf):
    incr = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    x = torch.zeros(8, dtype=torch.float64, device="cuda")
    # beyond the stated maximum: a clear error, nothing launched
    with pytest.raises(pf.PFError) as e:
        pf.pf_relax_noalloc((1 << 28) + 1, 0.3, x, x.clone(), incr)
    assert e.value.code == pf.PF_ERR_ARG and "PF_NOALLOC_MAX_N" in str(e.value)
    with pytest.raises(pf.PFError):
        pf.pf_relax_noalloc(-1, 0.3, x, x.clone(), incr)
    with pytest.raises(pf.PFError):
        pf.pf_relax_noalloc(8, 1.0, x, x.clone(), incr)
    with pytest.raises(pf.PFError):
        pf.pf_relax_noalloc(8, 0.3, None, x.clone(), incr)
    # n = 0: increment 0 although the scratch holds an earlier call's results
    pf.pf_relax_noalloc(0, 0.3, None, None, incr)
    torch.cuda.synchronize()
    assert float(incr.item()) == 0.0
    # a NaN anywhere makes the increment NaN (reading D7), as in the existing path
    phi0 = torch.zeros(5000, dtype=torch.float64, device="cuda")
    phi = torch.ones(5000, dtype=torch.float64, device="cuda")
    phi[4321] = float("nan")
    pf.pf_relax_noalloc(5000, 0.3, phi0, phi, incr)
    torch.cuda.synchronize()
    assert np.isnan(float(incr.item()))
    # on a side stream, repeated: same result (calls on one stream are serialised; overlapping calls would race)
    s = torch.cuda.Stream()
    a = torch.arange(10000, dtype=torch.float64, device="cuda")
    b = torch.zeros(10000, dtype=torch.float64, device="cuda")
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(3):
            c = b.clone()
            pf.pf_relax_noalloc(10000, 0.25, a, c, incr, stream=s)
    s.synchronize()
    assert float(incr.item()) == 0.75 * 9999.0 and torch.equal(c, 0.25 * a)
