"""Multi-GPU mode of the FTLM hot path: replicas only.

Every Lanczos chain (sector, start vector r) is independent until the host-side trace assembly
(Eq. 7: the sum over r and over sectors happens on the Ritz values), so N
GPUs run N chains with no data-path collective.  This module holds the host bookkeeping only:
which rank runs which chain, and how the per-chain coefficients and the timing come back to rank 0
through `torch.distributed` (NCCL on GPUs, gloo in the CPU tests).  No arithmetic of the method.
"""
from __future__ import annotations

from typing import Dict, List, Sequence, Tuple


def chain_list(sectors: Sequence[int], R: int) -> List[Tuple[int, int]]:
    """All chains of a run in a fixed order: (N_up, r) for every sector, r = 0..R-1."""
    return [(int(n_up), r) for n_up in sectors for r in range(R)]


def assign_chains(n_chains: int, world: int, rank: int) -> List[int]:
    """Round-robin: chain k runs on rank k mod world (equal sectors first: consecutive r of the largest
    sector land on different ranks)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    return list(range(rank, n_chains, world))


def gather_chain_results(local: Dict[int, dict], dist=None) -> Dict[int, dict]:
    """Rank 0 receives {chain id: result} from every rank (objects are small: <= 2 n_steps doubles per
    chain); other ranks get {}.  Without a process group the local dict is returned."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return dict(local)
    box = [None] * dist.get_world_size() if dist.get_rank() == 0 else None
    dist.gather_object(local, box, dst=0)
    if dist.get_rank() != 0:
        return {}
    out: Dict[int, dict] = {}
    for part in box:
        for k, v in part.items():
            if k in out:
                raise RuntimeError(f"chain {k} was run twice")
            out[k] = v
    return dict(sorted(out.items()))


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """The job's time is the slowest rank's device time."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def broadcast_choice(choice, dist=None):
    """Rank 0's kernel configuration (bench.py's probe) is applied by every rank."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return choice
    box = [choice]
    dist.broadcast_object_list(box, src=0)
    return box[0]


def save_chain_results(path: str, results: Dict[int, dict], meta: dict | None = None) -> None:
    """Checkpoint between chains (only alpha, beta survive a chain, L45): the coefficients of the
    finished chains as JSON - {chain id: {"alpha": [...], "beta": [...], "m_eff": m}} plus free-form `meta` (workload,
    seed, index mode) - written to a temporary file and renamed, so that an interrupted run leaves the previous file."""
    import json
    import os
    doc = {"meta": meta or {}, "chains": {str(k): {"alpha": [float(x) for x in v["alpha"]], "beta": [float(x) for x in v["beta"]],
                                                   "m_eff": int(v["m_eff"])} for k, v in sorted(results.items())}}
    tmp = path + ".tmp"
    with open(tmp, "w") as f:
        json.dump(doc, f)
    os.replace(tmp, path)


def load_chain_results(path: str, meta: dict | None = None) -> Dict[int, dict]:
    """The chains a previous run finished ({} if there is no file); with `meta`, a file written for another workload /
    seed is refused.  float -> JSON -> float is exact for IEEE doubles (repr round trip)."""
    import json
    import os
    if not os.path.exists(path):
        return {}
    with open(path) as f:
        doc = json.load(f)
    if meta is not None and doc.get("meta") != meta:
        raise ValueError(f"{path} belongs to another run: {doc.get('meta')}")
    return {int(k): v for k, v in doc["chains"].items()}


def remaining_chains(n_chains: int, done: Dict[int, dict]) -> List[int]:
    """Chain ids still to run after a resume."""
    return [k for k in range(n_chains) if k not in done]
