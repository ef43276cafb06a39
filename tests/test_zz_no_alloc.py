"""The allocation-free entry point fg_eval_points_dd_noalloc (include/fg.h): the double-double evaluation of given points
with the kernel's scratch in a static device array, against the existing path fg_eval_points(mode 2), on two calls in a row
(the array keeps the contents of the first call).  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from paper_1909_08015_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fg():
    import torch
    assert torch.cuda.is_available()
    from paper_1909_08015_b200 import build, fg as m
    build.build()
    return m


def _run(fg, plan, z):
    import torch
    n = len(z)
    zd = torch.from_numpy(np.ascontiguousarray(z)).cuda()
    Id = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    Ed = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    Fd = torch.full((n,), 255, dtype=torch.uint8, device="cuda")          # the entry point must clear the flags itself
    torch.cuda.synchronize()
    plan.eval_points_dd_noalloc(zd.data_ptr(), n, Id.data_ptr(), Ed.data_ptr(), Fd.data_ptr(), stream=torch.cuda.current_stream())
    torch.cuda.synchronize()
    return Id.cpu().numpy(), Ed.cpu().numpy(), Fd.cpu().numpy()


def _check(fg, plan, z):
    I, err, fl = _run(fg, plan, z)
    ref = plan.eval_points(z, mode=2)                # existing path: double-double for every point, quad-double for the rest
    to_qd = (ref["flags"] & 8) != 0                  # points the existing path handed on to the quad-double rung
    assert np.array_equal((fl & 4) != 0, to_qd)      # ... are exactly the ones double-double alone leaves unresolved
    assert np.array_equal(fl & 2, ref["flags"] & 2)
    ok = ~to_qd & ((fl & 2) == 0)
    assert ok.sum() > 0.5 * len(z)
    assert np.all(np.isfinite(I[ok]))
    assert np.all(np.abs(I[ok] - ref["I"][ok]) <= 1e-12 * np.abs(ref["I"][ok]))        # the per-sample tolerance of the parity tests
    assert np.all(err[ok] >= 0)
    return I


def test_no_alloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row(fg):
    scratch_bytes, max_points = fg.noalloc_limits()
    assert scratch_bytes == 32 << 20 and max_points == 1 << 20
    fg.noalloc_setup(0)
    x, ph = inputs.all_graphs(3)[18]
    plan = fg.plan_for(x, ph, rel_tol=1e-12)
    za = plan.sample_dump(0, 700 + 13, 7, words=False)["z"]
    zb = plan.sample_dump(5000, 300, 8, words=False)["z"]
    Ia = _check(fg, plan, za)                        # first call
    _check(fg, plan, zb)                             # second call, other points, fewer of them: stale scratch must not matter
    Ia2 = _check(fg, plan, za)                       # and the first set again
    assert np.array_equal(Ia, Ia2)
    # a second plan (other graph, other scratch layout) shares the same array
    x2, ph2 = 2, [(0, 4), (1, 3)]
    plan2 = fg.plan_for(x2, ph2, rel_tol=1e-12)
    _check(fg, plan2, plan2.sample_dump(0, 1000, 3, words=False)["z"])
    _check(fg, plan, zb)


def test_no_alloc_entry_point_rejects_sizes_beyond_the_maximum(fg):
    import torch
    plan = fg.plan_for(1, [(0, 2)])
    _, max_points = fg.noalloc_limits()
    buf = torch.zeros(8, dtype=torch.float64, device="cuda")
    with pytest.raises(fg.FgError) as e:
        plan.eval_points_dd_noalloc(buf.data_ptr(), max_points + 1, buf.data_ptr(), 0, buf.data_ptr())
    assert e.value.code == -8 and "2^20" in str(e.value)
    with pytest.raises(fg.FgError):
        plan.eval_points_dd_noalloc(0, 4, buf.data_ptr(), 0, buf.data_ptr())
