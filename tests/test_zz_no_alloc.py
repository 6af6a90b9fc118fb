"""qmcd_invert_static: the entry point that allocates nothing (its scratch is a file-scope
`static __device__` array of the library, resolved per device with cudaGetSymbolAddress) against
the existing qmcd_invert path with a caller-provided scratch buffer -- same kernel, so the bar
is the one the other inversion tests use (1e-10 on the inverse, 1e-8 on the residual) and the
results are in fact bit-identical.  Two calls in a row share the array and must not see each
other's leftovers.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes

import numpy as np
import pytest

from paper_1708_00744_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_INV = 1e-10
TOL_RESID = 1e-8


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("N,batch", [(130, 5), (512, 16)])
def test_invert_static_matches_invert_on_two_calls_in_a_row(qmcd, N, batch):
    import torch
    q = qmcd.Qmcd(N, 1, batch)
    assert qmcd.load().qmcd_invert_scratch_bytes(N, batch) <= qmcd.load().qmcd_invert_static_max_bytes()
    wl1 = inputs.make_workload(batch, N, n_moves=1, seed=21)
    wl2 = inputs.make_workload(batch, N, n_moves=1, seed=22)
    A1 = wl1.A.copy()
    A1[0, 0, 0] = 0.0                                   # walker 0 needs a row exchange at the first step
    A2 = wl2.A.copy()
    A2[batch - 1] = np.eye(N)
    A2[batch - 1, 3, 3] = 0.0                           # last walker exactly singular: info = 4
    refs = []
    for A in (A1, A2):                                  # the existing path: caller's scratch buffer
        X, info = q.invert(_dev(A))
        torch.cuda.synchronize()
        refs.append((X.clone(), info.clone()))
    # the new path, two calls in a row on the shared static array; the second call is the singular
    # batch FIRST and the regular one after it, so stale info words / pivots would show
    order = [(A2, refs[1]), (A1, refs[0]), (A2, refs[1])]
    X = torch.empty((batch, N, N), dtype=torch.float64, device="cuda")
    info = torch.full((batch,), -7, dtype=torch.int32, device="cuda")
    for call, (A, (Xref, iref)) in enumerate(order):
        Ad = _dev(A)
        X.fill_(float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        q.invert_static(Ad, X, info)
        torch.cuda.synchronize()
        if call > 0:                                    # (the first call may page the kernel's code in)
            assert torch.cuda.mem_get_info()[0] == free_before, "qmcd_invert_static changed the free device memory"
        assert torch.equal(info, iref), (call, info.cpu().numpy(), iref.cpu().numpy())
        ok = (iref == 0).cpu().numpy()
        Xh, Xr = X.cpu().numpy(), Xref.cpu().numpy()
        for w in np.nonzero(ok)[0]:
            assert np.max(np.abs(Xh[w] - Xr[w])) <= TOL_INV * max(1.0, np.abs(Xr[w]).max()), (call, w)
            assert np.max(np.abs(A[w] @ Xh[w] - np.eye(N))) <= TOL_RESID, (call, w)
        assert np.array_equal(Xh[ok], Xr[ok])           # same kernel, same launch shape: bit-identical
    assert info.cpu().numpy()[batch - 1] == 4 and int(refs[0][1].abs().max()) == 0
    q.close()


def test_invert_static_rejects_sizes_beyond_the_static_array(qmcd):
    import torch
    L = qmcd.load()
    N, batch = 512, 600                                  # 600 * 512 * 4 B of pivots alone > 1 MiB
    assert L.qmcd_invert_static_max_bytes() == 1 << 20
    assert L.qmcd_invert_scratch_bytes(N, batch) > L.qmcd_invert_static_max_bytes()
    q = qmcd.Qmcd(N, 1, batch)
    tiny = torch.zeros(8, dtype=torch.float64, device="cuda")    # never read: the size check comes first
    info = torch.zeros(batch, dtype=torch.int32, device="cuda")
    rc = L.qmcd_invert_static(q._h, ctypes.c_void_p(tiny.data_ptr()), ctypes.c_void_p(tiny.data_ptr()),
                              ctypes.c_void_p(info.data_ptr()))
    assert rc == qmcd.ELIMIT
    msg = L.qmcd_strerror(rc)
    assert b"qmcd_invert_static" in msg and b"1048576" in msg
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0 and float(tiny.abs().max()) == 0.0
    q.close()
