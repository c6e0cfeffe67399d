"""N > 1 path on CPU: two gloo ranks run the replica bookkeeping of paper_2605_26261_b200.replicas
(chain assignment, gather of the per-chain Lanczos coefficients, max-over-ranks timing, broadcast of
the kernel choice) with the host-only C-ABI entry points standing in for the device work."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
import numpy as np
import torch.distributed as dist
from paper_2605_26261_b200 import ftlm, replicas

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
chains = replicas.chain_list([8, 9, 10], 3)                    # 9 chains
mine = replicas.assign_chains(len(chains), world, rank)
local = {}
for k in mine:
    n_up, r = chains[k]
    rng = np.random.default_rng(1000 * n_up + r)               # stands in for the device chain
    alpha, beta = rng.standard_normal(6), np.abs(rng.standard_normal(5)) + 0.1
    theta, weight = ftlm.ftlm_tridiag_eig(alpha, beta)          # host-only entry point of the C ABI
    local[k] = {"rank": rank, "n_up": n_up, "r": r, "theta0": float(theta[0]), "wsum": float(np.sum(weight))}
allr = replicas.gather_chain_results(local, dist)
t = replicas.max_over_ranks(1.0 + rank, dist)
choice = replicas.broadcast_choice("tmlr+passb" if rank == 0 else "unset", dist)
if rank == 0:
    print(json.dumps({"n": len(allr), "keys": list(allr.keys()), "ranks": [v["rank"] for v in allr.values()],
                      "wsum": [v["wsum"] for v in allr.values()], "t": t, "choice": choice}))
else:
    assert allr == {} and choice == "tmlr+passb" and t == float(world)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_assignment_covers_every_chain_once():
    from paper_2605_26261_b200 import replicas
    for world in (1, 2, 3, 8):
        got = sorted(k for r in range(world) for k in replicas.assign_chains(10, world, r))
        assert got == list(range(10))
    assert replicas.chain_list([8, 9], 2) == [(8, 0), (8, 1), (9, 0), (9, 1)]


def test_two_gloo_ranks_gather_chain_results():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), [o[1][-1500:] for o in outs]
    d = json.loads(outs[0][0].strip().splitlines()[-1])
    assert d["n"] == 9 and d["keys"] == list(range(9))
    assert d["ranks"] == [k % 2 for k in range(9)]              # round-robin
    assert np.allclose(d["wsum"], 1.0, atol=1e-12)              # sum_k w_k = 1 for every chain
    assert d["t"] == 2.0 and d["choice"] == "tmlr+passb"


def test_chain_checkpoint_round_trip(tmp_path):
    """Resume between chains: coefficients survive JSON exactly, a foreign file is refused, the rest list is right."""
    import numpy as np
    from paper_2605_26261_b200 import replicas
    rng = np.random.default_rng(0)
    res = {k: {"alpha": rng.standard_normal(7), "beta": np.abs(rng.standard_normal(6)), "m_eff": 7} for k in (0, 2, 5)}
    path = str(tmp_path / "chains.json")
    assert replicas.load_chain_results(path) == {}
    meta = {"workload": "ring16", "seed": 20260526, "mode": "clt"}
    replicas.save_chain_results(path, res, meta)
    back = replicas.load_chain_results(path, meta)
    assert sorted(back) == [0, 2, 5]
    for k in res:
        assert back[k]["alpha"] == [float(x) for x in res[k]["alpha"]] and back[k]["m_eff"] == 7
        assert np.array_equal(np.array(back[k]["beta"]), res[k]["beta"])          # bit-exact round trip
    assert replicas.remaining_chains(6, back) == [1, 3, 4]
    import pytest
    with pytest.raises(ValueError):
        replicas.load_chain_results(path, dict(meta, seed=1))
