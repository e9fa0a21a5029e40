"""bsr_lambda_noalloc (include/bsr_amg.h): the power iteration behind omega with all of its work space in the library's
fixed device array -- nothing allocated, by the library or by torch, during the call.  Checked against the existing
path (prolongator_smooth_lambda, which allocates its work vectors at first use) and the oracle, on two calls in a row
that leave different contents in the shared array.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr

pytestmark = pytest.mark.gpu
TOL = 1e-11            # the tolerance of the lambda tests in tests/test_gpu_next_rows.py


@pytest.fixture(scope="module")
def bsr():
    import torch
    assert torch.cuda.is_available()
    from paper_2606_24748_b200 import bsr as m
    m.lib()
    return m


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def as_host(M):
    return pr.HostBSR(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx, M.vals)


def test_lambda_noalloc_two_calls_in_a_row(bsr):
    import torch
    # problem 1: config 0, 3x3 blocks; problem 2: its Galerkin coarse operator, 6x6 blocks (another layout of the array)
    g = pr.make_generator(0)
    g.build_prolongator(0)
    A, Pt, P = g.A(0), g.P_tent(0), g.P(0)
    Ac = as_host(orc.ptap(A, P))
    v0 = pr.uniform(g.seed, pr.PURPOSE_POWER, A.nbrows * 3)
    v1 = pr.uniform(g.seed, pr.PURPOSE_POWER + 16, Ac.nbrows * 6)
    GA, GT, GAc = bsr.Bsr.from_host(A), bsr.Bsr.from_host(Pt), bsr.Bsr.from_host(Ac)
    dv0, dv1 = dev(v0), dev(v1)
    # the existing path: work vectors owned by a smoothing plan
    ref0 = bsr.ProlongatorSmoother(GA, GT).lambda_estimate(dv0, 20)
    assert abs(ref0 / orc.power_lambda(A, v0, 20) - 1) < TOL
    ref1 = orc.power_lambda(Ac, v1, 20)
    # outputs are the caller's; everything is resident before the counters are read
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    st = torch.full((2,), -1, dtype=torch.int32, device="cuda")
    assert bsr.lambda_noalloc_scratch_bytes(A.nbrows, 3) <= bsr.NOALLOC_SCRATCH_BYTES
    torch.cuda.synchronize()
    lib_allocs = bsr.counters()[1]
    torch_allocs = torch.cuda.memory_stats()["allocation.all.allocated"]
    torch_segments = torch.cuda.memory_stats()["segment.all.allocated"]
    bsr.lambda_noalloc(GA, dv0, 20, out[0:1], st[0:1])        # call 1
    bsr.lambda_noalloc(GAc, dv1, 20, out[1:2], st[1:2])       # call 2: same array, other sizes and block shape
    torch.cuda.synchronize()
    assert bsr.counters()[1] == lib_allocs
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == torch_allocs
    assert torch.cuda.memory_stats()["segment.all.allocated"] == torch_segments
    got = out.cpu().numpy()
    assert st.cpu().tolist() == [0, 0]
    assert abs(got[0] / ref0 - 1) < TOL and got[0] == ref0    # same kernels, same order: the same bits
    assert abs(got[1] / ref1 - 1) < TOL
    # and once more the first problem over what the second call left behind
    again = torch.zeros(1, dtype=torch.float64, device="cuda")
    bsr.lambda_noalloc(GA, dv0, 20, again)
    assert again.item() == ref0


def test_lambda_noalloc_status_and_limit(bsr):
    import torch
    # a singular diagonal block is reported through d_status, and the flag does not stick to the next call
    g = pr.make_generator(0)
    A = g.A(0)
    vals = A.vals.copy()
    kd = A.rowptr[7] + np.searchsorted(A.colidx[A.rowptr[7]:A.rowptr[8]], 7)
    vals[kd] = 0.0
    Gbad = bsr.Bsr.from_host(pr.HostBSR(A.nbrows, A.nbcols, 3, 3, A.rowptr, A.colidx, vals))
    Ggood = bsr.Bsr.from_host(A)
    v0 = dev(pr.uniform(g.seed, pr.PURPOSE_POWER, A.nbrows * 3))
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    bsr.lambda_noalloc(Gbad, v0, 3, out, st)
    assert st.item() == 1
    bsr.lambda_noalloc(Ggood, v0, 3, out, st)
    assert st.item() == 0
    # a matrix whose work space exceeds the fixed array is refused (block-diagonal, 300,000 rows of 3x3 blocks)
    nb = 300_000
    assert bsr.lambda_noalloc_scratch_bytes(nb, 3) > bsr.NOALLOC_SCRATCH_BYTES
    big = pr.HostBSR(nb, nb, 3, 3, np.arange(nb + 1, dtype=np.int32), np.arange(nb, dtype=np.int32),
                     np.tile(np.eye(3), (nb, 1, 1)))
    Gbig = bsr.Bsr.from_host(big)
    vb = torch.ones(nb * 3, dtype=torch.float64, device="cuda")
    launches = bsr.counters()[0]
    with pytest.raises(bsr.BsrError) as e:
        bsr.lambda_noalloc(Gbig, vb, 2, out)
    assert e.value.code == 10 and "BSR_NOALLOC_SCRATCH_BYTES" in str(e.value)
    assert bsr.counters()[0] == launches                       # nothing was enqueued
    # the largest size that fits still works: 279,000 block rows, lambda of D^-1 A = 1 for a block-diagonal matrix
    nb = 279_000
    assert bsr.lambda_noalloc_scratch_bytes(nb, 3) <= bsr.NOALLOC_SCRATCH_BYTES
    fit = pr.HostBSR(nb, nb, 3, 3, np.arange(nb + 1, dtype=np.int32), np.arange(nb, dtype=np.int32),
                     np.tile(2.0 * np.eye(3), (nb, 1, 1)))
    bsr.lambda_noalloc(bsr.Bsr.from_host(fit), vb[:nb * 3], 2, out, st)
    assert abs(out.item() - 1.0) < 1e-12 and st.item() == 0
