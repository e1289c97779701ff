"""GPU test of qs_matvec_noalloc (include/qs.h): y = M x on free rings with all scratch memory in the library's static
device array - no cudaMalloc anywhere in the call - against the existing path (qs_init + qs_matvec_device, workspace
allocated at init), which tests/test_gpu_operator.py compares with the oracle.  Tolerance: the suite's 1e-9 rel-L2 for
the matvec (the two paths differ by ring order, i.e. by summation order and AGM class only).

Collected last on purpose (file name): the suite runs with pytest -x, a failure here must not hide other tests.  Passes
alone in a fresh process (the first call does the per-device set-up) and after the other tests.
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.mark.parametrize("n", [5000, 16384, 31])
def test_matvec_noalloc_equals_the_handle_path_on_two_calls_in_a_row(n):
    import torch
    import paper_2403_07666_b200 as pkg
    geo, x1 = wl.free_rings(n, seed=4100 + n)
    x2 = np.random.default_rng(n).standard_normal(n)
    with pkg.QS(geo, wl.Material()) as sim:                     # existing path (allocates its workspace at qs_init)
        ref1, ref2 = sim.matvec(x1), sim.matvec(x2)
    dev = torch.device("cuda", 0)
    with torch.cuda.device(dev):
        r = torch.from_numpy(geo.r).to(dev)
        z = torch.from_numpy(geo.z).to(dev)
        xa, xb = torch.from_numpy(x1).to(dev), torch.from_numpy(x2).to(dev)
        ya, yb = torch.full_like(xa, float("nan")), torch.full_like(xa, float("nan"))
        torch.cuda.synchronize()
        # two calls in a row on one stream, the second with another vector: the shared scratch array keeps the first
        # call's accumulators and inputs, which the second call must clear / rewrite
        pkg.matvec_noalloc(r, z, geo.softening, xa, ya)
        pkg.matvec_noalloc(r, z, geo.softening, xb, yb)
        torch.cuda.synchronize()
        got1, got2 = ya.cpu().numpy(), yb.cpu().numpy()
        # in place (y aliases x) and repeated: same result as the first call
        xc = xa.clone()
        pkg.matvec_noalloc(r, z, geo.softening, xc, xc)
        torch.cuda.synchronize()
        got3 = xc.cpu().numpy()
    for got, ref in ((got1, ref1), (got2, ref2), (got3, ref1)):
        assert np.all(np.isfinite(got))
        assert rel(got, ref) <= 1e-9
        assert np.max(np.abs(got - ref)) <= 1e-9 * np.max(np.abs(ref))


def test_matvec_noalloc_rejects_sizes_beyond_the_static_array():
    import torch
    import paper_2403_07666_b200 as pkg
    n = pkg.NOALLOC_MAX_RINGS + 1
    dev = torch.device("cuda", 0)
    with torch.cuda.device(dev):
        t = torch.ones(n, dtype=torch.float64, device=dev)
        y = torch.zeros(n, dtype=torch.float64, device=dev)
        with pytest.raises(pkg.QsError) as e:
            pkg.matvec_noalloc(t, t, 1e-4, t, y)
        assert e.value.code == -1 and "QS_NOALLOC_MAX_RINGS" in str(e.value)
        with pytest.raises(pkg.QsError):
            pkg.matvec_noalloc(t[:8], t[:8], 0.0, t[:8], y[:8])        # softening must be > 0
        torch.cuda.synchronize()
        assert float(y.abs().sum()) == 0.0                               # nothing was launched
