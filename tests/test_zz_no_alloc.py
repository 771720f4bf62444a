"""jxs_mse_tangent_noalloc (include/jxs.h): the allocation-free variant of jxs_mse_tangent, whose partial sums live in a
file-scope device array of the library.  Same launches, same summation order: its output must EQUAL the existing
path's (the tolerance of the MSE tests, rel 1e-12, is kept as the stated bar; equality is what is observed), on two
calls in a row (the second one finds the first one's partial sums in the shared array), on a second size (fewer partial
sums than the call before left behind), and it must allocate nothing and reject sizes beyond its stated limit.
Collected last on purpose (pytest -x must not hide other tests behind it)."""
import numpy as np
import pytest
import torch

from paper_2601_04400_b200 import jxs, workloads as wl

pytestmark = pytest.mark.gpu


def fields(case, seed):
    rng = np.random.default_rng(seed)
    U = torch.tensor(case["U0"], device="cuda")
    Udot = torch.tensor(rng.normal(size=case["U0"].shape), device="cuda")
    Ut = torch.tensor(case["U0"] * (1.0 + 1e-2 * rng.normal(size=case["U0"].shape)), device="cuda")
    return U, Udot, Ut


def test_noalloc_equals_the_existing_path_twice_in_a_row():
    torch.cuda.set_device(0)
    big = wl.shock_cylinder(256, 128, Ms=2.0)        # 131 072 entries: 512 partial sums
    small = wl.sod1d(200)                            # 800 entries: 4 partial sums, after the 512 of the call before
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    for case, seed in ((big, 1), (big, 2), (small, 3), (big, 4)):
        s = jxs.Solver.from_case(case)
        U, Udot, Ut = fields(case, seed)
        want = s.mse_tangent(U, Udot, Ut)            # the existing path (allocates its buffer on first use)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        free_before = torch.cuda.mem_get_info()[0]
        for call in range(2):                        # two calls in a row on the same inputs
            out.fill_(float("nan"))
            s.mse_tangent_noalloc(U, Udot, Ut, out)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
            assert got[0] == pytest.approx(want[0], rel=1e-12) and got[1] == pytest.approx(want[1], rel=1e-12, abs=1e-300)
            assert got[0] == want[0] and got[1] == want[1], (call, got, want)   # same launches: same bits
        assert torch.cuda.memory_allocated() == before
        assert torch.cuda.mem_get_info()[0] == free_before          # nothing was taken from the device either
        # and against the definition (Eq. 14), in numpy
        r = (U - Ut).cpu().numpy()
        assert got[0] == pytest.approx(float((r * r).mean()), rel=1e-12)
        assert got[1] == pytest.approx(float((2.0 * r * Udot.cpu().numpy()).mean()), rel=1e-9, abs=1e-15)


def test_noalloc_rejects_what_it_is_not_stated_for():
    torch.cuda.set_device(0)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    # 4 x 8192 x 2056 = 67 371 008 entries > 2^26: rejected before anything is launched (no state is allocated for
    # the call: the pointers only have to be non-NULL)
    nx, ny = 8192, 2056
    assert 4 * nx * ny > jxs.MSE_NOALLOC_MAX_N
    s = jxs.Solver(nx, ny, 1.0 / nx, 1.0 / nx, bc=wl.sod1d(200)["bc"])
    dummy = torch.zeros(8, dtype=torch.float64, device="cuda")
    rc = jxs.lib().jxs_mse_tangent_noalloc(s._h, dummy.data_ptr(), dummy.data_ptr(), dummy.data_ptr(), out.data_ptr())
    assert rc == jxs.EINVAL
    assert b"JXS_MSE_NOALLOC_MAX_N" in jxs.lib().jxs_last_error(s._h)
    del s
    # an fp32 handle and NULL pointers
    case = wl.sod1d(200)
    f = jxs.Solver.from_case(case, dtype=torch.float32)
    assert jxs.lib().jxs_mse_tangent_noalloc(f._h, dummy.data_ptr(), dummy.data_ptr(), dummy.data_ptr(), out.data_ptr()) == jxs.EINVAL
    d = jxs.Solver.from_case(case)
    assert jxs.lib().jxs_mse_tangent_noalloc(d._h, None, dummy.data_ptr(), dummy.data_ptr(), out.data_ptr()) == jxs.EINVAL
    assert jxs.lib().jxs_mse_tangent_noalloc(d._h, dummy.data_ptr(), dummy.data_ptr(), dummy.data_ptr(), None) == jxs.EINVAL
