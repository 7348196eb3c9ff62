"""Datapoint sharding over ranks: the host-side plan and the two collectives of
paper_1909_10547_b200/sharded.py under a world-size-2 gloo group on CPU.  The per-rank arithmetic is done by the
oracle here (tests may call it; on GPUs it is the C-ABI library's): the sharded forward + gather and the sharded
VJP + all-reduce must reproduce the unsharded oracle."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, os.environ["FK_ROOT"])
import numpy as np, torch
import torch.distributed as dist
from paper_1909_10547_b200 import sharded, synth
from oracle import fk_oracle as O
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
case = synth.hadronic_case(12, 37, 9, 11, 3, sub=4)          # N = 37: uneven split
g = synth.rng_for(12, synth.T_G, 5).standard_normal(size=(case.N, 3))
n0, n1 = sharded.shard_rows(case.N, world, rank)
sig_local, _ = O.hadronic(case.fk[n0:n1], case.pairs, case.f)
sig = sharded.gather_sigma(torch.from_numpy(sig_local), case.N).numpy()
df_part, _ = O.hadronic_vjp(case.fk[n0:n1], case.pairs, case.f, g[n0:n1])
df = sharded.allreduce_df(torch.from_numpy(df_part)).numpy()
ref, scale = O.hadronic(case.fk, case.pairs, case.f)
dref, D = O.hadronic_vjp(case.fk, case.pairs, case.f, g)
e1 = float(np.max(np.abs(sig - ref) / scale)); e2 = float(np.max(np.abs(df - dref) / np.maximum(D, 1e-300)))
# ragged group, whole tables to ranks (GroupPlan): forward pieces and per-table df assembled by the one all-reduce
shapes = synth.small_ragged_shapes(T=5)
R = 2
params = synth.pdf_params(synth.rng_for(4, synth.T_PDF), R)
cases = [synth.config4_table(t, shapes, R, params) for t in range(shapes.T)]
plan = sharded.GroupPlan([(c.N, c.nx, c.nfl, c.C) for c in cases], world)
fo, so = plan.offsets(R)
mine = plan.owner_tables[rank]
sig_p = [torch.from_numpy(O.hadronic(cases[t].fk, cases[t].pairs, cases[t].f)[0]) for t in mine]
df_p = [torch.from_numpy(O.hadronic_vjp(cases[t].fk, cases[t].pairs, cases[t].f, cases[t].g)[0]) for t in mine]
sig_cat = sharded.allreduce_cat(plan.scatter_local(sig_p, rank, so)).numpy()
df_cat = sharded.allreduce_cat(plan.scatter_local(df_p, rank, fo)).numpy()
ref_sig = np.concatenate([O.hadronic(c.fk, c.pairs, c.f)[0].ravel() for c in cases])
ref_df = np.concatenate([O.hadronic_vjp(c.fk, c.pairs, c.f, c.g)[0].ravel() for c in cases])
grp_exact = bool(np.array_equal(sig_cat, ref_sig) and np.array_equal(df_cat, ref_df))
dist.barrier()
print(json.dumps({"rank": rank, "rows": [n0, n1], "exact_sigma": bool(np.array_equal(sig, ref)), "e1": e1, "e2": e2,
                  "group_exact": grp_exact, "owned": mine}))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_row_sharded_forward_and_vjp_with_gloo_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port, FK_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    outs.sort(key=lambda o: o["rank"])
    assert outs[0]["rows"] == [0, 18] and outs[1]["rows"] == [18, 37]
    for o in outs:
        assert o["exact_sigma"]            # rows are independent: the gathered forward is the unsharded one, bit for bit
        assert o["e1"] == 0.0 and o["e2"] <= 1e-15   # df: one extra add per element (sum of two partials)
        assert o["group_exact"]            # whole-table sharding: x + 0 assembly, bit-identical to the unsharded group
    assert sorted(outs[0]["owned"] + outs[1]["owned"]) == [0, 1, 2, 3, 4] and outs[0]["owned"] and outs[1]["owned"]


def test_shard_plans():
    sys.path.insert(0, ROOT)
    from paper_1909_10547_b200 import sharded
    for N in (1, 7, 512, 12437):
        for world in (1, 2, 3, 8):
            if world > N:
                continue
            cuts = [sharded.shard_rows(N, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == N
            assert all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
    cost = [5, 1, 9, 3, 3, 8, 2]
    plan = sharded.shard_tables(cost, 3)
    assert sorted(t for p in plan for t in p) == list(range(len(cost)))
    loads = [sum(cost[t] for t in p) for p in plan]
    assert max(loads) - min(loads) <= max(cost) and plan == sharded.shard_tables(cost, 3)
    with pytest.raises(ValueError):
        sharded.shard_rows(5, 0, 0)
