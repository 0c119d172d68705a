"""Space decomposition (P:37-39, S:8(e), S:8(f4)), host logic on CPU: the slab plan, the halo index sets and the message
routing of paper_1401_4350_b200/dd.py against the oracle's pair set -- every Verlet pair that involves a particle a rank
owns must have both members in that rank's local set (owned + ghosts).  World size 2 over gloo exercises the
torch.distributed transport; 1, 3 and 4 ranks run through the in-process transport."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _messages(pos, plan, rank):
    """(to_left, to_right) of `rank` built with the numpy twin of md_dd_select: [rows of pos, global ids]."""
    from paper_1401_4350_b200.dd import select_np
    x = pos[:, 0]
    owned = np.nonzero(plan.owner(x) == rank)[0]
    out = []
    for zone in (plan.zone_to_left(rank), plan.zone_to_right(rank)):
        k = owned[select_np(x[owned], *zone)]
        out.append([torch.from_numpy(pos[k].copy()), torch.from_numpy(k.astype(np.float32).reshape(-1, 1))])
    return owned, out[0], out[1]


def _check_rank(pos, pairs, plan, rank, owned, from_left, from_right):
    from paper_1401_4350_b200.dd import local_sets_np
    ghosts = np.concatenate([from_left[1].numpy().ravel(), from_right[1].numpy().ravel()]).astype(np.int64)
    own_ref, ghost_ref = local_sets_np(pos, plan, rank)
    assert np.array_equal(owned, own_ref) and np.array_equal(ghosts, ghost_ref)      # routing = the reference sets, in order
    assert np.array_equal(np.concatenate([from_left[0].numpy(), from_right[0].numpy()]), pos[ghosts])
    local = np.zeros(pos.shape[0], dtype=bool)
    local[owned] = True
    assert not local[ghosts].any() and np.unique(ghosts).size == ghosts.size          # ghosts are foreign and unique
    local[ghosts] = True
    mine = np.zeros(pos.shape[0], dtype=bool)
    mine[owned] = True
    touch = mine[pairs[:, 0]] | mine[pairs[:, 1]]
    assert touch.any()
    assert local[pairs[touch, 0]].all() and local[pairs[touch, 1]].all()             # the slab + its halo is self-sufficient
    return int(touch.sum())


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    from oracle import Oracle
    from paper_1401_4350_b200.dd import DistTransport, SlabPlan
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.lj_fluid(2048, 2.5)
    plan = SlabPlan(w.box, world, w.rcut + w.skin)
    owned, to_left, to_right = _messages(w.pos, plan, rank)
    tr = DistTransport(plan, dist, torch.device("cpu"))
    from_left, from_right = tr.exchange({rank: (to_left, to_right)})[rank]
    pairs = Oracle().pair_set(w.pos, w.box, w.rcut, w.skin)
    n = _check_rank(w.pos, pairs, plan, rank, owned, from_left, from_right)
    flag = tr.any_flag({rank: 1 if rank == 1 else 0})
    dist.barrier()
    Path(out + f".{rank}").write_text(f"{n} {int(flag)} {len(owned)}")
    dist.destroy_process_group()


def test_halo_sets_cover_the_pair_set_world2(tmp_path):
    out = str(tmp_path / "dd")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = [Path(out + f".{r}").read_text().split() for r in range(2)]
    assert all(int(r[0]) > 0 and r[1] == "1" for r in res)          # the max-reduced rebuild flag reached both ranks
    assert sum(int(r[2]) for r in res) == 2048                        # the slabs partition the particles


@pytest.mark.parametrize("nranks", [1, 3, 4])
def test_halo_sets_cover_the_pair_set_in_process(oracle, nranks):
    from paper_1401_4350_b200.dd import LocalTransport, SlabPlan
    w = W.lj_fluid(2 ** 14, 2.5)                                      # cubic box 27.4: three slabs of 9.1, four of 6.8 >= 2 x 2.8
    plan = SlabPlan(w.box, nranks, w.rcut + w.skin)
    pairs = oracle.pair_set(w.pos, w.box, w.rcut, w.skin)
    msgs = {r: _messages(w.pos, plan, r) for r in range(nranks)}
    if nranks == 1:
        owned = msgs[0][0]
        assert owned.size == w.N
        return
    inc = LocalTransport(plan).exchange({r: (m[1], m[2]) for r, m in msgs.items()})
    seen = 0
    for r in range(nranks):
        seen += _check_rank(w.pos, pairs, plan, r, msgs[r][0], *inc[r])
    assert seen >= len(pairs)                                         # pairs across a face are seen by both ranks
    assert sum(m[0].size for m in msgs.values()) == w.N


def test_plan_rejects_slabs_thinner_than_two_halos():
    from paper_1401_4350_b200.dd import SlabPlan
    with pytest.raises(ValueError):
        SlabPlan([13.68, 13.68, 13.68], 4, 2.8)
    p = SlabPlan([16.0, 16.0, 16.0], 2, 2.8)
    assert p.slab(0) == (0.0, 8.0) and p.slab(1) == (8.0, 16.0) and p.left(0) == 1 and p.right(1) == 0
    assert list(p.owner(np.array([0.0, 7.999, 8.0, 15.99], dtype=np.float32))) == [0, 0, 1, 1]
