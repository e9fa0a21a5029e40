"""Test doubles for paper_2606_24748_b200/shard.py: an in-process communicator (one thread per rank, queues) and an
`ops` provider backed by the CPU oracle, so that the sharding bookkeeping can be checked without GPUs."""
import queue
import threading
import types

import numpy as np
import torch

from oracle import oracle as orc


class LoopbackWorld:
    def __init__(self, world):
        self.world = world
        self.q = {(s, d): queue.Queue() for s in range(world) for d in range(world)}

    def comm(self, rank):
        return LoopbackComm(self, rank)

    def run(self, fn, timeout=600):
        """fn(comm) on one thread per rank; returns the list of results, re-raising the first failure."""
        out, err = [None] * self.world, [None] * self.world

        def work(r):
            try:
                out[r] = fn(self.comm(r))
            except BaseException as e:  # noqa: BLE001
                err[r] = e
        th = [threading.Thread(target=work, args=(r,), daemon=True) for r in range(self.world)]
        for t in th:
            t.start()
        for t in th:
            t.join(timeout)
        real = [e for e in err if e is not None and not isinstance(e, queue.Empty)]
        if real:
            raise real[0]            # a rank that only timed out waiting for a failed peer is not the cause
        for e in err:
            if e is not None:
                raise e
        assert not any(t.is_alive() for t in th), "a rank is stuck in an exchange"
        return out


class LoopbackComm:
    def __init__(self, w, rank):
        self.w, self.rank, self.world = w, rank, w.world

    def exchange(self, sends, recvs):
        for q, t in sorted(sends.items()):
            if t.numel():
                if t.is_cuda:
                    torch.cuda.current_stream().synchronize()
                self.w.q[(self.rank, q)].put(t.clone())
        for q, t in sorted(recvs.items()):
            if t.numel():
                t.copy_(self.w.q[(q, self.rank)].get(timeout=30))

    def exchange_arrays(self, sends, dtype):
        for q in range(self.world):
            if q != self.rank:
                self.w.q[(self.rank, q)].put(np.ascontiguousarray(sends.get(q, np.zeros(0, dtype)), dtype).copy())
        got = {q: self.w.q[(q, self.rank)].get(timeout=30) for q in range(self.world) if q != self.rank}
        return {q: a for q, a in got.items() if a.shape[0]}

    def exchange_ids(self, sends):
        return self.exchange_arrays(sends, np.int64)

    def exchange_host_values(self, sends):
        return self.exchange_arrays(sends, np.float64)


class OracleOps:
    """The `ops` interface of shard.py on CPU tensors, every numeric step by the oracle (tests only)."""

    def zeros(self, n):
        return torch.zeros(int(n), dtype=torch.float64)

    def int_tensor(self, a):
        return torch.from_numpy(np.ascontiguousarray(a, np.int32))

    def _mat(self, nbrows, nbcols, bs_r, bs_c, rowptr, colidx, vals):
        m = types.SimpleNamespace(nbrows=nbrows, nbcols=nbcols, bs_r=bs_r, bs_c=bs_c, rowptr=np.asarray(rowptr, np.int32),
                                  colidx=np.asarray(colidx, np.int32), tvals=vals)
        m.host = lambda: types.SimpleNamespace(nbrows=m.nbrows, nbcols=m.nbcols, bs_r=m.bs_r, bs_c=m.bs_c, rowptr=m.rowptr,
                                               colidx=m.colidx, vals=m.tvals.numpy().reshape(-1, m.bs_r, m.bs_c))
        return m

    def matrix(self, M):
        return self._mat(M.nbrows, M.nbcols, M.bs_r, M.bs_c, M.rowptr, M.colidx,
                         torch.from_numpy(np.ascontiguousarray(M.vals, np.float64).reshape(-1).copy()))

    def alias(self, M, nbrows, nbcols, rowptr):
        return self._mat(nbrows, nbcols, M.bs_r, M.bs_c, rowptr, M.colidx, M.tvals)

    def slice_rows(self, M, row0, nrows, rowptr, blk0):
        n, bb = int(rowptr[-1]), M.bs_r * M.bs_c
        return self._mat(nrows, M.nbcols, M.bs_r, M.bs_c, rowptr, M.colidx[blk0:blk0 + n], M.tvals[blk0 * bb:(blk0 + n) * bb])

    def values(self, M):
        return M.tvals

    def values_changed(self, M):
        pass

    def spmv(self, M, x, y):
        y.copy_(torch.from_numpy(orc.spmv(M.host(), x.numpy())))

    def spmv_t(self, M, x, y):
        y.copy_(torch.from_numpy(orc.spmv_t(M.host(), x.numpy())))

    def gather(self, idx, bs, src):
        return src.reshape(-1, bs)[idx.long()].reshape(-1).clone()

    def scatter_add(self, idx, bs, src, dst):
        dst.reshape(-1, bs)[idx.long()] += src.reshape(-1, bs)

    def ptap_plan(self, A, P):
        return types.SimpleNamespace(A=A, P=P, st=orc.ptap_symbolic(A.host(), P.host())[1])

    def plan_structure(self, plan):
        return plan.st

    def ptap_numeric(self, plan, out):
        out.copy_(torch.from_numpy(orc.ptap(plan.A.host(), plan.P.host(), structure=plan.st).vals.reshape(-1)))

    def bcoo_plan(self, brow, bcol, nbrows, nbcols, bs_r, bs_c):
        z = np.zeros((brow.shape[0], bs_r, bs_c))
        M = orc.bcoo_assemble(brow, bcol, z, nbrows, nbcols)
        return types.SimpleNamespace(brow=brow, bcol=bcol, nbrows=nbrows, nbcols=nbcols, bs_r=bs_r, bs_c=bs_c,
                                     st=(M.rowptr, M.colidx))

    def bcoo_nnzb(self, plan):
        return int(plan.st[1].shape[0])

    def bcoo_structure(self, plan):
        return plan.st

    def bcoo_set_values(self, plan, stream, out):
        M = orc.bcoo_assemble(plan.brow, plan.bcol, stream.numpy().reshape(-1, plan.bs_r, plan.bs_c), plan.nbrows,
                              plan.nbcols, structure=plan.st)
        out.copy_(torch.from_numpy(M.vals.reshape(-1)))


def check_shard(comm, ops, A, P, agg, x, xc, Ac_ref, to_dev=lambda t: t, tol=1e-13):
    """One rank of the sharded hot path against the single-rank oracle results (x, xc global vectors; Ac_ref the
    global A_c).  Returns a dict of facts for the caller to compare across ranks."""
    from paper_2606_24748_b200 import shard
    sh = shard.RowShard(A, P, agg, comm, ops)
    bs, bc = A.bs_r, P.bs_c
    rows = slice(sh.r0 * bs, sh.r1 * bs)
    crow = slice(sh.c0 * bc, sh.c1 * bc)
    res = {"rank": comm.rank, "rows": (sh.r0, sh.r1), "crows": (sh.c0, sh.c1), "ghosts": sh.next - sh.nloc}
    # y = A x: only the local part of x is given; the ghosts arrive through the halo exchange
    x_ext = sh.new_fine_ext()
    sh.fine_local(x_ext).copy_(to_dev(torch.from_numpy(x[rows])))
    y = ops.zeros(sh.nloc * bs)
    sh.spmv_A(x_ext, y)
    ref = orc.spmv(A, x)[rows]
    res["spmv_A"] = float(np.abs(y.cpu().numpy() - ref).max() / np.abs(ref).max())
    # y = P x_c
    xc_ext = sh.new_coarse_ext()
    sh.coarse_local(xc_ext).copy_(to_dev(torch.from_numpy(xc[crow])))
    sh.spmv_P(xc_ext, y)
    ref = orc.spmv(P, xc)[rows]
    res["spmv_P"] = float(np.abs(y.cpu().numpy() - ref).max() / np.abs(ref).max())
    # y_c = P^T x (owned coarse rows)
    yc_ext = sh.new_coarse_ext()
    sh.spmv_Pt(sh.fine_local(x_ext), yc_ext)
    ref = orc.spmv_t(P, x)[crow]
    res["spmv_Pt"] = float(np.abs(sh.coarse_local(yc_ext).cpu().numpy() - ref).max() / np.abs(ref).max())
    # A_c: owned rows, global columns
    rp, ci = sh.ptap_symbolic()
    g0, g1 = Ac_ref.rowptr[sh.c0], Ac_ref.rowptr[sh.c1]
    res["structure"] = bool(np.array_equal(rp, Ac_ref.rowptr[sh.c0:sh.c1 + 1] - g0) and np.array_equal(ci, Ac_ref.colidx[g0:g1]))
    vals = sh.ptap_numeric().cpu().numpy().reshape(-1, bc, bc)
    refv = Ac_ref.vals[g0:g1]
    res["ptap"] = float(np.abs(vals - refv).max() / np.abs(refv).max())
    # state gate on P_oth: untouched P -> no gather; after the local rows of P moved -> exactly one
    n0 = sh.n_poth_gathers
    sh.ptap_numeric()
    res["gate_idle"] = sh.n_poth_gathers - n0
    ops.values(sh.P_loc).mul_(2.0)
    sh.p_values_changed()
    vals2 = sh.ptap_numeric().cpu().numpy().reshape(-1, bc, bc)
    res["gate_moved"] = sh.n_poth_gathers - n0
    res["ptap_scaled"] = float(np.abs(vals2 - 4.0 * refv).max() / np.abs(refv).max())
    res["bytes"] = sh.exchange_bytes()
    return res
