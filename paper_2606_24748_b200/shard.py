"""Row sharding of the hot path over several GPUs: one process per GPU, contiguous slabs of
block rows cut on aggregate boundaries, the paper's distribution ("one rank per GPU").

What crosses ranks, and nothing else:
  * y = A x        halo of x at the ghost columns of the local rows (the "blocked SpMV halo"), whole bs-blocks;
  * y = P x_c      halo of the coarse vector at the ghost coarse columns;
  * y = P^T x      partial sums for the coarse rows a neighbour owns, added by the owner in a fixed order;
  * P_oth          the prolongator rows of the ghost fine nodes, whole bs_r x bs_c blocks, gathered ONCE and cached;
                   re-gathered (values only) when P's state moves -- the state gate of PAPER.md:103;
  * A_c            every rank runs the single-GPU ptap_numeric on its LOCAL rows (A extended by empty ghost rows, P
                   stacked with P_oth: "the stacked operand"); the coarse rows it computed for a neighbour are sent to
                   their owner, which sums own and received blocks through ONE blocked COO plan ("local triple-product
                   contributions plus off-process contributions routed to their owning ranks").
Everything numeric runs in the library's kernels through an `ops` object (LibOps below: bsr_spmv, bsr_gather_blocks,
bsr_scatter_add_blocks, ptap_numeric, bcoo_set_values); the exchange is `comm.exchange` (torch.distributed point to
point: NCCL over NVLink on GPUs, gloo in the CPU tests).  This module holds index bookkeeping only.

The partition works on any ordering in which a prefix of the block rows is exactly the set of rows of a prefix of the
aggregates (box aggregates in lexicographic order: z-slabs cut at multiples of three node planes)."""
from __future__ import annotations

import dataclasses

import numpy as np


# ------------------------------------------------------------------ partition
def slab_cuts(agg: np.ndarray, world: int):
    """Cuts (fine, coarse) of `world` contiguous slabs: fine rows [f[k], f[k+1]) are exactly the rows whose aggregate
    lies in [c[k], c[k+1]).  Balanced by fine rows among the admissible cut points."""
    agg = np.asarray(agg)
    n = agg.shape[0]
    pmax = np.maximum.accumulate(agg)
    smin = np.minimum.accumulate(agg[::-1])[::-1]
    ok = np.nonzero(pmax[:-1] < smin[1:])[0] + 1            # admissible fine cut points r (rows [0, r) | [r, n))
    f, c = [0], [0]
    for k in range(1, world):
        if ok.size == 0:
            raise ValueError("no aggregate-aligned cut: the row ordering does not follow the aggregates")
        r = int(ok[np.argmin(np.abs(ok - k * n / world))])
        if r <= f[-1]:
            raise ValueError(f"cannot cut {n} rows into {world} aggregate-aligned slabs")
        f.append(r)
        c.append(int(pmax[r - 1]) + 1)
    f.append(n)
    c.append(int(agg.max()) + 1)
    return np.asarray(f, np.int64), np.asarray(c, np.int64)


@dataclasses.dataclass
class HostMat:
    """A host block-CSR matrix (numpy arrays), as handed to an `ops` provider."""
    nbrows: int
    nbcols: int
    bs_r: int
    bs_c: int
    rowptr: np.ndarray
    colidx: np.ndarray
    vals: np.ndarray

    @property
    def nnzb(self):
        return int(self.colidx.shape[0])


def _ext_ids(cols: np.ndarray, lo: int, hi: int):
    """Ascending extended numbering [ghosts below | lo..hi-1 | ghosts above] of the columns a slab touches."""
    u = np.unique(cols)
    return np.concatenate([u[u < lo], np.arange(lo, hi, dtype=u.dtype), u[u >= hi]]).astype(np.int64)


class _Halo:
    """Who sends which block entries of a distributed vector to whom.  ghosts: global ids this rank needs (ascending);
    cuts: ownership ranges.  The owners learn what to send from one request exchange at setup (cold)."""

    def __init__(self, comm, ghosts: np.ndarray, cuts: np.ndarray, lo: int, off_lo: int, off_hi: int):
        self.comm = comm
        owner = np.searchsorted(cuts, ghosts, side="right") - 1
        self.recv = {}                                        # peer -> (offset in the extended vector, count)
        reqs = {}
        pos_lo, pos_hi = off_lo, off_hi
        for q in np.unique(owner):
            ids = ghosts[owner == q]
            if q < comm.rank:
                self.recv[int(q)] = (pos_lo, ids.shape[0]); pos_lo += ids.shape[0]
            else:
                self.recv[int(q)] = (pos_hi, ids.shape[0]); pos_hi += ids.shape[0]
            reqs[int(q)] = ids
        got = comm.exchange_ids(reqs)                          # peer -> global ids the peer wants from this rank
        self.send = {q: (ids - lo).astype(np.int32) for q, ids in sorted(got.items()) if ids.shape[0]}
        self.recv = {q: v for q, v in sorted(self.recv.items()) if v[1]}


class RowShard:
    """One rank's slab of (A, P) and the cached exchange plans.  A, P: the GLOBAL host matrices (this harness
    generates the whole problem on every rank and slices it -- a stand-in for a distributed assembly; only this rank's
    rows of A and P are used, P's ghost rows arrive through the communicator)."""

    def __init__(self, A, P, agg, comm, ops):
        self.comm, self.ops = comm, ops
        k, W = comm.rank, comm.world
        self.fcuts, self.ccuts = slab_cuts(agg, W)
        r0, r1, c0, c1 = int(self.fcuts[k]), int(self.fcuts[k + 1]), int(self.ccuts[k]), int(self.ccuts[k + 1])
        self.r0, self.r1, self.c0, self.c1 = r0, r1, c0, c1
        self.bs, self.bc, self.ncoarse = A.bs_r, P.bs_c, P.nbcols
        self.nloc, self.ncloc = r1 - r0, c1 - c0
        # ---- A: local rows, extended column numbering [ghost below | local | ghost above]
        a0, a1 = int(A.rowptr[r0]), int(A.rowptr[r1])
        acols = np.asarray(A.colidx[a0:a1], np.int64)
        self.ext = _ext_ids(acols, r0, r1)
        # the library wants 16-byte aligned vectors: when the ghosts below hold an odd number of doubles, one unused
        # pad node (id -1) is put in front so that the local part of an extended vector starts on a 16-byte boundary
        if (int(np.searchsorted(self.ext, r0)) * A.bs_c) % 2:
            self.ext = np.concatenate([[-1], self.ext])
        self.nglo = int(np.searchsorted(self.ext, r0))
        self.next = int(self.ext.shape[0])
        rp = (np.asarray(A.rowptr[r0:r1 + 1], np.int64) - a0).astype(np.int32)
        ci = np.searchsorted(self.ext, acols).astype(np.int32)
        va = np.ascontiguousarray(A.vals[a0:a1])
        self.A_loc = ops.matrix(HostMat(self.nloc, self.next, A.bs_r, A.bs_c, rp, ci, va))
        # the same arrays as a SQUARE matrix whose ghost rows are empty: the operand of the local triple product
        rpx = np.concatenate([np.zeros(self.nglo, np.int32), rp, np.full(self.next - self.nglo - self.nloc, rp[-1], np.int32)])
        self.A_ext = ops.alias(self.A_loc, self.next, self.next, rpx)
        fpad = int(self.ext[0] < 0)
        self.halo = _Halo(comm, np.concatenate([self.ext[fpad:self.nglo], self.ext[self.nglo + self.nloc:]]), self.fcuts, r0,
                          fpad, self.nglo + self.nloc)
        # ---- P: local rows + P_oth (rows of the ghost fine nodes), gathered once
        self._P = P
        self._gather_P_oth_structure()
        self.plan = None
        self.P_state = 0                                      # bumped by p_values_changed()
        self._poth_state = 0

    # ------------------------------------------------------------------ vectors
    def new_fine_ext(self):
        return self.ops.zeros(self.next * self.bs)

    def new_coarse_ext(self):
        return self.ops.zeros(self.ncext * self.bc)

    def fine_local(self, x_ext):
        return x_ext[self.nglo * self.bs:(self.nglo + self.nloc) * self.bs]

    def coarse_local(self, xc_ext):
        return xc_ext[self.ncglo * self.bc:(self.ncglo + self.ncloc) * self.bc]

    def _exchange_halo(self, halo, x_ext, loc_off, bs):
        ops = self.ops
        loc = x_ext[loc_off * bs:]
        sends = {q: ops.gather(self._idx(halo, q), bs, loc) for q in halo.send}
        recvs = {q: x_ext[o * bs:(o + n) * bs] for q, (o, n) in halo.recv.items()}
        self.comm.exchange(sends, recvs)

    def _idx(self, halo, q):
        key = (id(halo), q)
        if key not in self.__dict__.setdefault("_idx_cache", {}):
            self._idx_cache[key] = self.ops.int_tensor(halo.send[q])
        return self._idx_cache[key]

    # ------------------------------------------------------------------ SpMV family
    def spmv_A(self, x_ext, y_loc):
        """y_loc = (A x)[local rows]; the ghost entries of x_ext are filled by the halo exchange first."""
        self._exchange_halo(self.halo, x_ext, self.nglo, self.bs)
        self.ops.spmv(self.A_loc, x_ext, y_loc)
        return y_loc

    def spmv_P(self, xc_ext, y_loc):
        """y_loc = (P x_c)[local rows] (prolongation): coarse halo, then the local rows of the stacked P."""
        self._exchange_halo(self.chalo, xc_ext, self.ncglo, self.bc)
        self.ops.spmv(self.P_loc, xc_ext, y_loc)
        return y_loc

    def spmv_Pt(self, x_loc, yc_ext):
        """local part of yc_ext = (P^T x)[owned coarse rows] (restriction): every rank forms P_loc^T x_loc, ships the
        partial sums of the coarse rows a neighbour owns, and the owner adds them in peer order."""
        ops = self.ops
        ops.spmv_t(self.P_loc, x_loc, yc_ext)
        sends = {q: yc_ext[o * self.bc:(o + n) * self.bc] for q, (o, n) in self.chalo.recv.items()}
        recvs = {q: ops.zeros(self.chalo.send[q].shape[0] * self.bc) for q in self.chalo.send}
        self.comm.exchange(sends, recvs)
        loc = self.coarse_local(yc_ext)
        for q in sorted(recvs):
            ops.scatter_add(self._idx(self.chalo, q), self.bc, recvs[q], loc)
        return yc_ext

    # ------------------------------------------------------------------ P_oth
    def _gather_P_oth_structure(self):
        P, comm, ops = self._P, self.comm, self.ops
        r0, r1 = self.r0, self.r1
        p0, p1 = int(P.rowptr[r0]), int(P.rowptr[r1])
        # what the peers want from this rank: rows halo.send[q] of P_loc -> their slot lists (blocks), sent whole
        self._poth_slots = {}
        sends_i, sends_v = {}, {}
        for q, rows in self.halo.send.items():
            g = rows.astype(np.int64) + r0
            cnt = (P.rowptr[g + 1] - P.rowptr[g]).astype(np.int64)
            slots = np.concatenate([np.arange(P.rowptr[i], P.rowptr[i + 1]) for i in g]) if g.size else np.zeros(0, np.int64)
            self._poth_slots[q] = (slots - p0).astype(np.int32)
            sends_i[q] = np.concatenate([cnt, np.asarray(P.colidx[slots], np.int64)])
            sends_v[q] = np.ascontiguousarray(P.vals[slots]).reshape(-1)
        got_i = comm.exchange_ids(sends_i)
        got_v = comm.exchange_host_values(sends_v)
        # stack: [ghost rows below | local rows | ghost rows above]
        bb = P.bs_r * P.bs_c
        parts_cnt, parts_col, parts_val = [], [], []
        self._poth_recv = {}                                   # peer -> (block offset in P_ext.vals, blocks)
        blk = 0

        def add_peer(q):
            nonlocal blk
            n = self.halo.recv[q][1]
            cnt, col = got_i[q][:n], got_i[q][n:]
            parts_cnt.append(cnt); parts_col.append(col); parts_val.append(got_v[q].reshape(-1, P.bs_r, P.bs_c))
            self._poth_recv[q] = (blk, int(col.shape[0]))
            blk += int(col.shape[0])

        if self.ext[0] < 0:                                    # the pad node: an empty row
            parts_cnt.append(np.zeros(1, np.int64))
        for q in [q for q in self.halo.recv if q < comm.rank]:
            add_peer(q)
        loc_cnt = (P.rowptr[r0 + 1:r1 + 1] - P.rowptr[r0:r1]).astype(np.int64)
        parts_cnt.append(loc_cnt); parts_col.append(np.asarray(P.colidx[p0:p1], np.int64)); parts_val.append(P.vals[p0:p1])
        self._ploc_blk = (blk, p1 - p0)
        blk += p1 - p0
        for q in [q for q in self.halo.recv if q > comm.rank]:
            add_peer(q)
        cnt, col = np.concatenate(parts_cnt), np.concatenate(parts_col)
        assert cnt.shape[0] == self.next
        self.cext = _ext_ids(col, self.c0, self.c1)
        if (int(np.searchsorted(self.cext, self.c0)) * P.bs_c) % 2:     # same alignment pad for coarse vectors
            self.cext = np.concatenate([[-1], self.cext])
        self.ncglo = int(np.searchsorted(self.cext, self.c0))
        self.ncext = int(self.cext.shape[0])
        rp = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
        ci = np.searchsorted(self.cext, col).astype(np.int32)
        va = np.ascontiguousarray(np.concatenate(parts_val))
        self.P_ext = ops.matrix(HostMat(self.next, self.ncext, P.bs_r, P.bs_c, rp, ci, va))
        lo = int(rp[self.nglo])
        self.P_loc = ops.slice_rows(self.P_ext, self.nglo, self.nloc, rp[self.nglo:self.nglo + self.nloc + 1] - lo, lo)
        cpad = int(self.cext[0] < 0)
        self.chalo = _Halo(comm, np.concatenate([self.cext[cpad:self.ncglo], self.cext[self.ncglo + self.ncloc:]]),
                           self.ccuts, self.c0, cpad, self.ncglo + self.ncloc)
        self.n_poth_gathers = 1

    def p_values_changed(self):
        """The caller rewrote the local rows of P in place (ops.values(P_loc)): P_oth is stale."""
        self.P_state += 1
        self.ops.values_changed(self.P_loc)

    def ensure_P_oth(self):
        """State gate: P_oth is re-gathered (values only, packed on the device) iff P moved."""
        if self._poth_state == self.P_state:
            return
        ops, bb = self.ops, self._P.bs_r * self._P.bs_c
        vals = ops.values(self.P_ext)
        loc = vals[self._ploc_blk[0] * bb:]
        sends = {q: ops.gather(self._slot_idx(q), bb, loc) for q in self._poth_slots}
        recvs = {q: vals[o * bb:(o + n) * bb] for q, (o, n) in self._poth_recv.items()}
        self.comm.exchange(sends, recvs)
        ops.values_changed(self.P_ext)
        self._poth_state = self.P_state
        self.n_poth_gathers += 1

    def _slot_idx(self, q):
        c = self.__dict__.setdefault("_slot_cache", {})
        if q not in c:
            c[q] = self.ops.int_tensor(self._poth_slots[q])
        return c[q]

    # ------------------------------------------------------------------ Galerkin product
    def ptap_symbolic(self):
        """Cold: the local plan (single-GPU ptap_symbolic on the extended operands), the exchange of the structure of
        the coarse rows computed for a neighbour, and the blocked COO plan that sums own and received blocks."""
        ops, comm = self.ops, self.comm
        self.plan = ops.ptap_plan(self.A_ext, self.P_ext)
        rp, ci = ops.plan_structure(self.plan)                 # numpy; ncext x ncext, extended coarse numbering
        bb = self.bc * self.bc
        gcol = self.cext[ci]                                   # global coarse columns
        grow = np.repeat(self.cext, np.diff(rp))
        sends, self._c_send = {}, {}
        for q, (o, n) in self.chalo.recv.items():              # coarse ghost rows [o, o+n) belong to peer q
            b0, b1 = int(rp[o]), int(rp[o + n])
            self._c_send[q] = (b0, b1 - b0)
            sends[q] = np.concatenate([grow[b0:b1], gcol[b0:b1]])
        got = comm.exchange_ids(sends)
        own0, own1 = int(rp[self.ncglo]), int(rp[self.ncglo + self.ncloc])
        brow = np.full(ci.shape[0], -1, np.int64)              # blocks of ghost rows: declared, not owned -> ignored
        brow[own0:own1] = grow[own0:own1] - self.c0
        bcol = gcol.copy()
        self._c_recv, off = {}, ci.shape[0]
        for q in sorted(got):
            m = got[q].shape[0] // 2
            if not m:
                continue
            brow = np.concatenate([brow, got[q][:m] - self.c0])
            bcol = np.concatenate([bcol, got[q][m:]])
            self._c_recv[q] = (off, m)
            off += m
        self._npart, self._nstream = int(ci.shape[0]), int(off)
        self.coo = ops.bcoo_plan(brow.astype(np.int32), bcol.astype(np.int32), self.ncloc, self.ncoarse, self.bc, self.bc)
        self._stream = ops.zeros(self._nstream * bb)
        self.vals_c = ops.zeros(ops.bcoo_nnzb(self.coo) * bb)
        return ops.bcoo_structure(self.coo)                    # (rowptr, colidx) of the owned rows, GLOBAL columns

    def ptap_numeric(self):
        """Hot: local triple product -> neighbour exchange of the cut rows -> one blocked COO summation."""
        ops, bb = self.ops, self.bc * self.bc
        self.ensure_P_oth()
        part = self._stream[:self._npart * bb]
        ops.ptap_numeric(self.plan, part)
        sends = {q: part[b0 * bb:(b0 + n) * bb] for q, (b0, n) in self._c_send.items() if n}
        recvs = {q: self._stream[o * bb:(o + n) * bb] for q, (o, n) in self._c_recv.items()}
        self.comm.exchange(sends, recvs)
        ops.bcoo_set_values(self.coo, self._stream, self.vals_c)
        return self.vals_c

    def exchange_bytes(self) -> dict:
        """Bytes this rank SENDS per hot call (the communication profile)."""
        bb = self.bc * self.bc
        return {"spmv_A": 8 * self.bs * sum(v.shape[0] for v in self.halo.send.values()),
                "spmv_P": 8 * self.bc * sum(v.shape[0] for v in self.chalo.send.values()),
                "spmv_Pt": 8 * self.bc * sum(n for _, n in self.chalo.recv.values()),
                "ptap_numeric": 8 * bb * sum(n for _, n in getattr(self, "_c_send", {}).values()),
                "P_oth_gather": 8 * self._P.bs_r * self._P.bs_c * sum(v.shape[0] for v in self._poth_slots.values())}


# ------------------------------------------------------------------ communicators
class DistComm:
    """torch.distributed point-to-point (NCCL between GPUs, gloo on the CPU).  exchange(): tensors of known sizes,
    posted as one batch; exchange_ids() / exchange_host_values(): cold, variable-size host arrays (sizes first)."""

    def __init__(self, device):
        import torch.distributed as dist
        self.dist, self.device = dist, device
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def exchange(self, sends: dict, recvs: dict):
        dist = self.dist
        ops = [dist.P2POp(dist.irecv, t, q) for q, t in sorted(recvs.items()) if t.numel()]
        ops += [dist.P2POp(dist.isend, t.contiguous(), q) for q, t in sorted(sends.items()) if t.numel()]
        if ops:
            for r in dist.batch_isend_irecv(ops):
                r.wait()

    def exchange_arrays(self, sends: dict, dtype):
        """Cold: variable-size host arrays; any rank may talk to any other, so the sizes are agreed through an
        all-gather of a size matrix first.  Collective: every rank calls it, in the same order."""
        import torch
        tdt = torch.int64 if dtype == np.int64 else torch.float64
        counts = torch.zeros(self.world, dtype=torch.int64, device=self.device)
        for q, a in sends.items():
            counts[q] = a.shape[0]
        allc = [torch.zeros_like(counts) for _ in range(self.world)]
        self.dist.all_gather(allc, counts)
        mat = torch.stack(allc).cpu().numpy()                  # mat[src, dst]
        peers = [q for q in range(self.world) if q != self.rank]
        out = {q: torch.from_numpy(np.ascontiguousarray(sends[q], dtype)).to(self.device) for q in peers if mat[self.rank, q]}
        inn = {q: torch.empty(int(mat[q, self.rank]), dtype=tdt, device=self.device) for q in peers if mat[q, self.rank]}
        self.exchange(out, inn)
        return {q: t.cpu().numpy() for q, t in inn.items()}

    def exchange_ids(self, sends: dict):
        return self.exchange_arrays(sends, np.int64)

    def exchange_host_values(self, sends: dict):
        return self.exchange_arrays(sends, np.float64)


class SoloComm:
    """World of one rank (no neighbours): every exchange is empty."""
    rank, world = 0, 1

    def exchange(self, sends, recvs):
        assert not sends and not recvs

    def exchange_arrays(self, sends, dtype):
        return {}

    def exchange_ids(self, sends):
        return {}

    def exchange_host_values(self, sends):
        return {}


class LibOps:
    """The library behind the sharded path: every numeric step is one of libbsramg.so's kernels."""

    def __init__(self, device):
        import torch
        from . import bsr
        self.t, self.b, self.device = torch, bsr, device

    def zeros(self, n):
        return self.t.zeros(int(n), dtype=self.t.float64, device=self.device)

    def int_tensor(self, a):
        return self.t.from_numpy(np.ascontiguousarray(a, np.int32)).to(self.device)

    def matrix(self, M: HostMat):
        t = self.t
        return self.b.Bsr(M.nbrows, M.nbcols, M.bs_r, M.bs_c, self.int_tensor(M.rowptr), self.int_tensor(M.colidx),
                          t.from_numpy(np.ascontiguousarray(M.vals, np.float64).reshape(-1)).to(self.device))

    def alias(self, M, nbrows, nbcols, rowptr):
        return self.b.Bsr(nbrows, nbcols, M.bs_r, M.bs_c, self.int_tensor(rowptr), M.colidx, M.vals)

    def slice_rows(self, M, row0, nrows, rowptr, blk0):
        n = int(rowptr[-1])
        bb = M.bs_r * M.bs_c
        return self.b.Bsr(nrows, M.nbcols, M.bs_r, M.bs_c, self.int_tensor(rowptr), M.colidx[blk0:blk0 + n],
                          M.vals[blk0 * bb:(blk0 + n) * bb])

    def values(self, M):
        return M.vals

    def values_changed(self, M):
        M.values_changed()

    def spmv(self, M, x, y):
        M.spmv(x, y)

    def spmv_t(self, M, x, y):
        M.spmv_t(x, y)

    def gather(self, idx, bs, src):
        return self.b.gather_blocks(idx, bs, src)

    def scatter_add(self, idx, bs, src, dst):
        self.b.scatter_add_blocks(idx, bs, src, dst)

    def ptap_plan(self, A, P):
        return self.b.PtapPlan(A, P)

    def plan_structure(self, plan):
        return plan.rowptr_c.cpu().numpy(), plan.colidx_c.cpu().numpy()

    def ptap_numeric(self, plan, out):
        plan.numeric(out)

    def bcoo_plan(self, brow, bcol, nbrows, nbcols, bs_r, bs_c):
        return self.b.BcooPlan(self.int_tensor(brow), self.int_tensor(bcol), nbrows, nbcols, bs_r, bs_c)

    def bcoo_nnzb(self, plan):
        return plan.nnzb

    def bcoo_structure(self, plan):
        return plan.rowptr.cpu().numpy(), plan.colidx.cpu().numpy()

    def bcoo_set_values(self, plan, stream, out):
        plan.set_values(stream, out)
