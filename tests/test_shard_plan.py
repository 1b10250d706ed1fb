"""Host logic of the intra-mesh sharding (ep_shard_plan, no GPU): ownership, halos, exchange lists; the N > 1 plumbing is
exercised with two gloo processes on the CPU (each rank plans its own part and the ranks cross-check their lists)."""
import os
import subprocess
import sys

import numpy as np
import pytest

from ep_inputs import make
from ep_inputs import meshes as M

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _stencil_reach(tets, cells):
    """Cells whose Vm an update of `cells` reads: all cells around the nodes of the cells and of their face neighbours
    (brute force, the definition in)."""
    nc = tets.shape[0]
    node_cells = {}
    for c in range(nc):
        for n in tets[c]:
            node_cells.setdefault(int(n), []).append(c)
    faces = {}
    for c in range(nc):
        for j in range(4):
            key = tuple(sorted(int(x) for k, x in enumerate(tets[c]) if k != j))
            faces.setdefault(key, []).append(c)
    nbrs = {c: set() for c in range(nc)}
    for lst in faces.values():
        if len(lst) == 2:
            nbrs[lst[0]].add(lst[1]); nbrs[lst[1]].add(lst[0])
    need = set()
    for c in cells:
        nodes = set(int(n) for n in tets[c])
        for d in nbrs[c]:
            nodes |= set(int(n) for n in tets[d])
        for n in nodes:
            need |= set(node_cells[n])
    return need


@pytest.mark.parametrize("n_parts", [2, 3, 5])
def test_plan_covers_the_stencil_and_lists_match(n_parts):
    import paper_2112_12854_b200 as ep
    m = M.kuhn_slab(7, 5, 3, 0.3)
    M.jitter_interior(m, 0.05, 3)
    nc = m.n_tets
    plans = [ep.shard_plan(m.xyz, m.tets, p, n_parts) for p in range(n_parts)]
    owned = [pl["local_cells"][: pl["n_owned"]] for pl in plans]
    allc = np.sort(np.concatenate(owned))
    assert np.array_equal(allc, np.arange(nc))                              # a partition of the cells
    sizes = [o.size for o in owned]
    assert max(sizes) - min(sizes) <= 1                                     # balanced ranges of the curve
    for p, pl in enumerate(plans):
        local = set(pl["local_cells"].tolist())
        assert np.all(np.diff(owned[p]) > 0) and np.all(np.diff(pl["local_cells"][pl["n_owned"]:]) > 0)
        need = _stencil_reach(m.tets, owned[p].tolist())
        assert need <= local                                                # everything an owned update reads is local
        halo = pl["local_cells"][pl["n_owned"]:]
        assert not (set(halo.tolist()) & set(owned[p].tolist()))
        # every halo cell is received from exactly one peer: its owner
        assert np.array_equal(np.sort(pl["recv_global"]), halo)
        for q in range(n_parts):
            seg = pl["recv_global"][pl["recv_ptr"][q]: pl["recv_ptr"][q + 1]]
            assert set(seg.tolist()) <= set(owned[q].tolist())
            # ... and q's send segment to p is the same list in the same order
            other = plans[q]["send_global"][plans[q]["send_ptr"][p]: plans[q]["send_ptr"][p + 1]]
            assert np.array_equal(seg, other)
        assert pl["send_ptr"][p + 1] == pl["send_ptr"][p] and pl["recv_ptr"][p + 1] == pl["recv_ptr"][p]


def test_plan_on_a_carved_shell_and_errors():
    import paper_2112_12854_b200 as ep
    m = make(3, coarsen=5.0).mesh
    pl = [ep.shard_plan(m.xyz, m.tets, p, 4) for p in range(4)]
    halo_frac = [(p_["local_cells"].size - p_["n_owned"]) / p_["n_owned"] for p_ in pl]
    assert sum(p_["n_owned"] for p_ in pl) == m.n_tets and max(halo_frac) < 1.5
    with pytest.raises(ep.EpError):
        ep.shard_plan(m.xyz, m.tets, 4, 4)
    with pytest.raises(ep.EpError):
        ep.shard_plan(m.xyz, m.tets, 0, 65)


_WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.environ["EP_ROOT"])
import paper_2112_12854_b200 as ep
from ep_inputs import meshes as M
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
m = M.kuhn_slab(8, 6, 3, 0.25)
pl = ep.shard_plan(m.xyz, m.tets, rank, world)
# every rank announces what it will send to each peer; the peer checks it against what it expects to receive
for src in range(world):
    for dst in range(world):
        if src == dst:
            continue
        if rank == src:
            seg = pl["send_global"][pl["send_ptr"][dst]: pl["send_ptr"][dst + 1]]
            dist.send(torch.tensor([seg.size], dtype=torch.int64), dst)
            dist.send(torch.from_numpy(seg.copy()), dst)
        if rank == dst:
            n = torch.zeros(1, dtype=torch.int64); dist.recv(n, src)
            buf = torch.zeros(int(n.item()), dtype=torch.int64); dist.recv(buf, src)
            want = pl["recv_global"][pl["recv_ptr"][src]: pl["recv_ptr"][src + 1]]
            assert np.array_equal(buf.numpy(), want), (src, dst)
# a halo exchange of a field defined by global id, through the same lists: received values must be the owners' values
field = lambda ids: 1000.0 * np.sin(ids) + ids
mine = field(pl["local_cells"].astype(np.float64))
got = np.full(pl["recv_global"].size, np.nan)
for src in range(world):
    for dst in range(world):
        if src == dst:
            continue
        if rank == src:
            seg = pl["send_global"][pl["send_ptr"][dst]: pl["send_ptr"][dst + 1]]
            dist.send(torch.from_numpy(field(seg.astype(np.float64))), dst)
        if rank == dst:
            a, b = pl["recv_ptr"][src], pl["recv_ptr"][src + 1]
            buf = torch.zeros(int(b - a), dtype=torch.float64); dist.recv(buf, src)
            got[a:b] = buf.numpy()
assert np.array_equal(got, field(pl["recv_global"].astype(np.float64)))
tot = torch.tensor([pl["n_owned"]], dtype=torch.int64); dist.all_reduce(tot)
assert int(tot.item()) == m.n_tets
if rank == 0:
    print("shard plan ok", world)
dist.destroy_process_group()
"""


def test_two_ranks_agree_on_their_exchange_lists_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, EP_ROOT=ROOT, MASTER_ADDR="127.0.0.1")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr",
                        "127.0.0.1", "--master-port", "29517", str(script)], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "shard plan ok 2" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]
