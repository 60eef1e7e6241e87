"""tsm_loops_local_noalloc: the entry point that allocates nothing (its reduction scratch is a 4 MiB file-scope
`static __device__` array, csrc/contract.cu) against the existing path (tsm_loops_source, whose scratch is carved from
the workspace), on two calls in a row that share the array, within the tolerances the other GPU tests use for the
loops (1e-12 for an fp64 solution, 1e-6 for an fp32 one) -- and in fact bit for bit.  In a file of its own that
pytest collects last; it owns its contexts, so it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import oracle
from paper_1211_0126_b200 import workloads as W

pytestmark = pytest.mark.gpu

F64, F32 = 0, 1


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def _loops_of(out):
    """[nrhs][16][Lt][2] float64 device tensor -> complex numpy [nrhs][16][Lt]"""
    a = out.cpu().numpy()
    return a[..., 0] + 1j * a[..., 1]


@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (6, 10, 4, 6), (16, 16, 16, 4)])
def test_noalloc_loops_match_the_existing_path_on_two_calls_in_a_row(dims):
    import torch
    from paper_1211_0126_b200 import tsm
    wl = W.WORKLOADS[1]
    U = W.random_su3_links(dims, 0.4, 4242)
    t = tsm.Tsm(dims, t_boundary=-1, max_nrhs=4)
    t.set_params(wl.kappa, wl.mu)
    t.set_gauge(U, 18)
    t.loops_reset(False)
    assert t.lib.tsm_noalloc_scratch_bytes() == 4 << 20
    seed = 0x1211012600000009
    batches = {}
    for prec, ids, k in ((F64, [3, 4, 5], 9), (F32, [11, 12, 13, 14], 6)):
        rc, _ = t.solve(seed, ids, prec, 0.0, k, slot=0)
        assert rc == 0
        want = np.stack([t.loops_source(0, j) for j in range(len(ids))])            # the existing path
        sol = np.stack([t.get_solution(0, j) for j in range(len(ids))])
        batches[prec] = (ids, want, t.pack(prec, sol))                               # exact: the slot's own values
    # the new entry point (it touches neither the workspace nor the slots): three calls in a row, of different
    # precisions and numbers of sources, so that each later call finds an earlier call's partials in the shared array
    outs = {}
    for prec in (F64, F32, F64):
        ids, want, field = batches[prec]
        out = torch.full((len(ids), 16, dims[3], 2), float("nan"), dtype=torch.float64, device="cuda")
        t.loops_local_noalloc(prec, field, seed, ids, out)
        outs[prec] = out
    torch.cuda.synchronize()
    for prec, tol in ((F64, 1e-12), (F32, 1e-6)):
        ids, want, _ = batches[prec]
        got = _loops_of(outs[prec])
        assert np.isfinite(got.view(np.float64)).all()
        assert rel(got, want) < tol, (dims, prec)
        assert np.array_equal(got, want), (dims, prec)            # same arithmetic, same reduction order
    # and against the oracle directly for the fp64 batch (the existing path is itself tested that way elsewhere)
    ids, want, _ = batches[F64]
    eta = oracle.noise(dims, seed, ids[1])
    s1 = t.unpack(F64, len(ids), batches[F64][2])[1]
    assert rel(_loops_of(outs[F64])[1], oracle.loops(dims, eta, s1)) < 1e-12
    t.close()


def test_noalloc_rejects_what_does_not_fit_and_bad_arguments():
    import torch
    from paper_1211_0126_b200 import tsm
    dims = (4, 4, 4, 1024)                       # 16 sources x 1024 timeslices x 2 x 1 x 32 doubles = 8 MiB > 4 MiB
    t = tsm.Tsm(dims, t_boundary=-1, max_nrhs=1)
    field = torch.zeros(t.field_bytes(F64, 16) * 2, dtype=torch.uint8, device="cuda")
    out = torch.zeros((16, 16, dims[3], 2), dtype=torch.float64, device="cuda")
    with pytest.raises(tsm.TsmError) as e:
        t.loops_local_noalloc(F64, field, 1, list(range(16)), out)
    assert e.value.code == tsm.EINVAL and "4 MiB" in str(e.value)
    t.loops_local_noalloc(F64, field, 1, list(range(8)), out)       # 8 sources fit exactly
    torch.cuda.synchronize()
    assert float(out[:8].abs().max()) == 0.0                         # zero solution, zero loops
    with pytest.raises(tsm.TsmError) as e:
        t.loops_local_noalloc(2, field, 1, [0], out)                 # bf16 is not a solution precision
    assert e.value.code == tsm.EINVAL
    t.close()
