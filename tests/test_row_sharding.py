"""SURVEY.md 8(f) row f3 on the CPU: the row-sharded hot path (paper_2606_24748_b200/shard.py) with the oracle as the
local kernel provider.  Every rank sees only its slab's part of the vectors; halo, P_oth and cut-row exchanges go
through a communicator -- in-process (threads) for 2 and 3 ranks, and torch.distributed gloo with world_size 2 under
torchrun.  The sharded results must reproduce the single-rank oracle: structure bit for bit, values to rounding."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr, shard
from tests.shard_util import LoopbackWorld, OracleOps, check_shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _problem(d, ne, seed):
    g = pr.Generator(d, ne, seed=seed, modulus_mode=1)
    g.build_prolongator(0)
    A, P = g.A(0), g.P(0)
    agg = g.level_arrays(0)["agg"].copy()
    x = pr.uniform(seed, pr.PURPOSE_FINE, A.nbrows * A.bs_r)
    xc = pr.uniform(seed, pr.PURPOSE_COARSE, P.nbcols * P.bs_c)
    return g, A, P, agg, x, xc, orc.ptap(A, P)


def test_slab_cuts_follow_aggregates():
    g, A, P, agg, *_ = _problem(3, 11, 1)            # 12^3 nodes, 4^3 aggregates
    f, c = shard.slab_cuts(agg, 2)
    assert f.tolist() == [0, 6 * 144, 12 ** 3] and c.tolist() == [0, 32, 64]      # cut after 6 node planes = 2 coarse planes
    f, c = shard.slab_cuts(agg, 4)
    assert np.diff(f).tolist() == [3 * 144] * 4 and np.diff(c).tolist() == [16] * 4
    for k in range(4):
        assert set(agg[f[k]:f[k + 1]].tolist()) == set(range(c[k], c[k + 1]))
    with pytest.raises(ValueError):
        shard.slab_cuts(agg, 5)                       # only 4 coarse planes
    gg = pr.Generator(3, 8, seed=6, agg_mode=1); gg.build_prolongator(0)
    with pytest.raises(ValueError):                   # greedy aggregates do not follow the row ordering
        shard.slab_cuts(gg.level_arrays(0)["agg"], 2)


@pytest.mark.parametrize("d,ne,world", [(3, 11, 2), (3, 11, 3), (3, 8, 3), (2, 26, 3)])
def test_sharded_hot_path_in_process(d, ne, world):
    g, A, P, agg, x, xc, Ac = _problem(d, ne, 2)
    res = LoopbackWorld(world).run(lambda comm: check_shard(comm, OracleOps(), A, P, agg, x, xc, Ac))
    assert [r["rows"][0] for r in res] == sorted(r["rows"][0] for r in res)
    assert res[0]["rows"][0] == 0 and res[-1]["rows"][1] == A.nbrows and res[-1]["crows"][1] == P.nbcols
    for r in res:
        assert r["structure"], r
        assert r["spmv_A"] == 0.0 and r["spmv_P"] == 0.0          # same blocks, same order, long double: bit-equal
        assert r["spmv_Pt"] < 1e-14 and r["ptap"] < 1e-14 and r["ptap_scaled"] < 1e-14, r
        assert r["gate_idle"] == 0 and r["gate_moved"] == 1, r
        assert r["ghosts"] > 0
    # the communication profile: one node plane of x per cut, whole blocks
    plane = (ne + 1) ** (d - 1)
    inner = res[1] if world > 2 else None
    assert res[0]["bytes"]["spmv_A"] == 8 * A.bs_r * plane
    if inner:
        assert inner["bytes"]["spmv_A"] == 2 * 8 * A.bs_r * plane


WORKER = r'''
import json, os, sys
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from oracle import oracle as orc
from paper_2606_24748_b200 import problems as pr, shard
from tests.shard_util import OracleOps, check_shard
dist.init_process_group("gloo")
g = pr.Generator(3, 11, seed=2, modulus_mode=1); g.build_prolongator(0)
A, P = g.A(0), g.P(0)
agg = g.level_arrays(0)["agg"].copy()
x = pr.uniform(2, pr.PURPOSE_FINE, A.nbrows * 3); xc = pr.uniform(2, pr.PURPOSE_COARSE, P.nbcols * 6)
res = check_shard(shard.DistComm(torch.device("cpu")), OracleOps(), A, P, agg, x, xc, orc.ptap(A, P))
out = [None] * dist.get_world_size()
dist.all_gather_object(out, res)
if dist.get_rank() == 0:
    print(json.dumps(out))
dist.destroy_process_group()
'''


def test_sharded_hot_path_two_gloo_ranks(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER.format(root=ROOT))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", "29547", str(w)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT, env=dict(os.environ, OMP_NUM_THREADS="2"))
    assert r.returncode == 0, r.stderr[-3000:]
    res = json.loads([ln for ln in r.stdout.splitlines() if ln.startswith("[")][-1])
    assert len(res) == 2 and res[0]["rows"][1] == res[1]["rows"][0]
    for q in res:
        assert q["structure"] and q["spmv_A"] == 0.0 and q["spmv_P"] == 0.0
        assert q["spmv_Pt"] < 1e-14 and q["ptap"] < 1e-14 and q["gate_idle"] == 0 and q["gate_moved"] == 1
