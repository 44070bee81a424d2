"""GPU test of afsat_check_static (include/afsat.h): the discrete check with its scratch in the library's file-scope
device array instead of cudaMalloc'ed workspace.  Collected LAST (file name), runs alone or after the other tests.

The output is integer (satisfied counts, solution flags), so the comparison with the existing path (afsat_check) is
bit-exact -- the bar the other check tests use -- and the oracle is consulted as well."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2606_06641_b200 import binding as Bd
from paper_2606_06641_b200 import build as Build
from paper_2606_06641_b200 import instances as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    Build.build()
    assert torch.cuda.is_available()


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _outputs(B):
    # poisoned, so that a call that wrote nothing cannot pass
    return (torch.full((B,), -7, dtype=torch.int32, device="cuda"), torch.full((B,), 9, dtype=torch.uint8, device="cuda"))


@pytest.mark.parametrize("dtype", [32, 64])
def test_check_static_matches_check_on_two_calls_in_a_row(dtype):
    """Two calls in a row on DIFFERENT contexts and sizes (the second smaller than the first, so that whatever the first
    left in the shared array lies under and beyond the second's footprint), then the first again: each equals
    afsat_check bit for bit and the oracle's check.  Ragged batches, every type, k up to 30, a partial assignment."""
    Bd.static_setup(0)
    npdt = np.float32 if dtype == 32 else np.float64
    big = I.make_mixed(n=90, m=700, kmin=1, kmax=30, seed=4401, batch=300, with_fixed=True)
    small = I.make_mixed(n=33, m=150, kmin=1, kmax=12, seed=4402, batch=70)
    cases = []
    for inst, seed in ((big, 1), (small, 2)):
        B = inst.batch
        x = I.make_x0(inst, seed=seed, batch=B)
        x[2, : B // 3] = 0.0
        x[3, : B // 3] = -0.0
        ctx = Bd.Context.from_instance(inst, batch=B, ldb=x.shape[1], dtype=dtype)
        cases.append((inst, B, x, ctx, dev(x.astype(npdt))))
    for inst, B, x, ctx, xd in cases + cases[:1]:
        sat_ref, sol_ref = ctx.check(xd)                               # the existing path
        sat, sol = _outputs(B)
        ctx.check_static(xd, sat, sol)
        torch.cuda.synchronize()
        assert torch.equal(sat, sat_ref) and torch.equal(sol, sol_ref)
        so, lo = O.check(inst, x.astype(np.float64), B)
        assert np.array_equal(sat.cpu().numpy(), so) and np.array_equal(sol.cpu().numpy(), lo)
    # back to back on ONE stream without a sync in between: stream order is all the sharing needs
    (i0, B0, x0, c0, d0), (i1, B1, x1, c1, d1) = cases
    s0, l0 = _outputs(B0)
    s1, l1 = _outputs(B1)
    c0.check_static(d0, s0, l0)
    c1.check_static(d1, s1, l1)
    c0.check_static(d0, s0, l0)
    torch.cuda.synchronize()
    assert np.array_equal(s0.cpu().numpy(), O.check(i0, x0.astype(np.float64), B0)[0])
    assert np.array_equal(s1.cpu().numpy(), O.check(i1, x1.astype(np.float64), B1)[0])
    for c in cases:
        c[3].close()


def test_check_static_allocates_nothing_and_rejects_what_does_not_fit():
    inst = I.make_config(1, scale=0.02, batch=256)
    x = dev(I.make_x0(inst, batch=256))
    ctx = Bd.Context.from_instance(inst, batch=256)
    sat, sol = _outputs(256)
    Bd.static_setup(0)
    ctx.check_static(x, sat, sol)                                      # warm: module loaded, address resolved
    torch.cuda.synchronize()
    ws = ctx.query(Bd.Q_WORKSPACE_BYTES)
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        ctx.check_static(x, sat, sol)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and ctx.query(Bd.Q_WORKSPACE_BYTES) == ws    # no device memory taken, by the library or anyone
    ctx.close()
    # a context whose scratch exceeds AFSAT_STATIC_SCRATCH_BYTES: a clear error, and the ordinary path still serves it
    n, B = 3000, 32768                                                  # 3000 x 1024 words x 4 B = 12.3 MB > 8 MiB
    wide = I.make_mixed(n=n, m=50, kmin=2, kmax=5, seed=4403, batch=B)
    xw = dev(I.make_x0(wide, seed=3, batch=B))
    cw = Bd.Context.from_instance(wide, batch=B)
    sw, lw = _outputs(B)
    with pytest.raises(Bd.AfsatError) as ei:
        cw.check_static(xw, sw, lw)
    assert ei.value.code == -7 and "AFSAT_STATIC_SCRATCH_BYTES" in str(ei.value) and str(Bd.STATIC_SCRATCH_BYTES) in str(ei.value)
    assert int(sw[0]) == -7                                            # nothing was launched
    sat_ref, _ = cw.check(xw)
    torch.cuda.synchronize()
    assert sat_ref.shape[0] == B
    cw.close()
