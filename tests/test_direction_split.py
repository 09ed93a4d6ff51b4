"""Direction split of the staple over ranks: host logic on CPU with gloo, world_size 2.

The per-direction compute is injected (the oracle's literal eq. 2.3, one direction at a time), so this test covers what the
multi-rank path adds to the single-GPU one: which rank owns which direction, the order of the all-gathered series, and that
every rank ends up with the same four staples as the four-direction oracle."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent

WORKER = r"""
import sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import oracle
from paper_2001_02835_b200 import parallel, workloads as wl
rank = int(sys.argv[1])
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=2)
Un, z = wl.config_staple(4, 3, seed=11, twist_k=1)
U = [torch.from_numpy(u) for u in Un]
calls = []
def compute(U, z, mu):
    # literal eq. 2.3 for one direction: oracle.staple evaluates all four, keep mu (CPU stand-in for nspt_staple_dir)
    calls.append(mu)
    return torch.from_numpy(oracle.staple([u.numpy() for u in U], z)[mu])
S = parallel.staple_direction_split(U, z, compute=compute)
ref = oracle.staple(Un, z)
err = max(float(np.abs(S[mu].numpy() - ref[mu]).max()) for mu in range(4))
dist.barrier()
dist.destroy_process_group()
print(json.dumps({{"rank": rank, "calls": calls, "err": err}}))
"""


def test_owned_directions_partition():
    from paper_2001_02835_b200 import parallel
    for world in (1, 2, 4):
        owned = [parallel.owned_directions(r, world) for r in range(world)]
        assert sorted(mu for o in owned for mu in o) == [0, 1, 2, 3]
        assert all(len(o) == 4 // world for o in owned)
    assert parallel.owned_directions(1, 2) == [1, 3]
    with pytest.raises(ValueError):
        parallel.owned_directions(0, 3)
    with pytest.raises(ValueError):
        parallel.owned_directions(2, 2)


def test_single_rank_needs_no_process_group():
    import numpy as np
    import torch
    import oracle
    from paper_2001_02835_b200 import parallel, workloads as wl
    Un, z = wl.config_staple(4, 2, seed=12, twist_k=1)
    U = [torch.from_numpy(u) for u in Un]
    S = parallel.staple_direction_split(U, z, rank=0, world=1,
                                        compute=lambda U, z, mu: torch.from_numpy(oracle.staple([u.numpy() for u in U], z)[mu]))
    ref = oracle.staple(Un, z)
    assert all(np.array_equal(S[mu].numpy(), ref[mu]) for mu in range(4))


def test_staple_direction_split_two_ranks_gloo(tmp_path):
    port = 31500 + (os.getpid() % 2000)
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT), port=port))
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, text=True) for r in range(2)]
    outs = [p.communicate(timeout=300)[0] for p in procs]
    assert all(p.returncode == 0 for p in procs)
    res = {d["rank"]: d for d in (json.loads(o.strip().splitlines()[-1]) for o in outs)}
    assert res[0]["calls"] == [0, 2] and res[1]["calls"] == [1, 3]     # each rank computes only the directions it owns
    assert res[0]["err"] == 0.0 and res[1]["err"] == 0.0                 # and every rank holds all four staples, in order
