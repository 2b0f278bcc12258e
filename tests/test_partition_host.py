"""Host side of the element-partitioned (multi-GPU) path, on the CPU: the partitioner's send / receive lists, and the halo
exchange as paper_2502_17805_b200.partition routes it -- pack by send list, all_to_all_single with per-peer split sizes, unpack
by receive list -- run with torch.distributed (gloo) at world sizes 2 and 3 on face data whose value names its global face."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2502_17805_b200 import inputs as I          # noqa: E402
from paper_2502_17805_b200.partition import route_offsets   # noqa: E402

W = 5        # doubles per face in this test


def _mesh():
    return I.cubed_sphere_shell(4, 3, 0.7, 0.95, I.lobatto_abscissae(3))


def _face_value(g, f):
    """Every (global element, face) has its own block of W numbers."""
    return (np.asarray(g)[..., None] * 6 + np.asarray(f)[..., None]) * 10.0 + np.arange(W)


@pytest.mark.parametrize("P", [1, 2, 3, 7])
def test_partition_lists_cover_exactly_the_boundary_faces(P):
    m = _mesh()
    parts = I.partition_mesh(m, P)
    E = m["n_elem"]
    assert sorted(np.concatenate([p["elems"][:p["n_owned"]] for p in parts]).tolist()) == list(range(E))      # every element owned once
    owner = np.concatenate([np.full(p["n_owned"], p["rank"]) for p in parts])
    n_cross = 0
    for p in parts:
        n, el, pm = p["n_owned"], p["elems"], p["mesh"]
        assert np.all(np.diff(el[n:]) > 0) and np.all(owner[el[n:]] != p["rank"])                             # ghosts: off-rank, sorted
        for i in range(n):
            for f in range(6):
                g = int(m["nbr_elem"][el[i], f])
                assert (pm["nbr_elem"][i, f] == g) if g < 0 else (el[pm["nbr_elem"][i, f]] == g)               # connectivity kept
                n_cross += g >= 0 and owner[g] != p["rank"]
        np.testing.assert_array_equal(pm["xyz"], m["xyz"][el])
        assert p["send_counts"][p["rank"]] == 0 and p["send_counts"].sum() == p["send_elem"].size == p["recv_elem"].size
        # a received face is exactly a face some owned element looks at
        looked = {(int(pm["nbr_elem"][i, f]), int(pm["nbr_face"][i, f])) for i in range(n) for f in range(6) if pm["nbr_elem"][i, f] >= n}
        assert looked == set(zip(p["recv_elem"].tolist(), p["recv_face"].tolist()))
    assert n_cross == sum(p["send_elem"].size for p in parts)
    # sender's group for q and q's group from the sender name the same global faces in the same order
    for p in parts:
        so = route_offsets(p["send_counts"])
        for q in parts:
            ro = route_offsets(q["recv_counts"])
            s = list(zip(p["elems"][p["send_elem"][so[q["rank"]]:so[q["rank"] + 1]]].tolist(), p["send_face"][so[q["rank"]]:so[q["rank"] + 1]].tolist()))
            r = list(zip(q["elems"][q["recv_elem"][ro[p["rank"]]:ro[p["rank"] + 1]]].tolist(), q["recv_face"][ro[p["rank"]]:ro[p["rank"] + 1]].tolist()))
            assert s == r


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        p = I.partition_mesh(_mesh(), world, rank)
        el, n = p["elems"], p["n_owned"]
        # local face data [n_local][6][W]: owned faces hold their global value, ghost faces a poison value
        data = np.full((el.size, 6, W), -1.0)
        data[:n] = _face_value(el[:n, None], np.arange(6)[None, :])
        send = torch.from_numpy(np.ascontiguousarray(data[p["send_elem"], p["send_face"]]))               # pack
        recv = torch.empty((p["recv_elem"].size, W), dtype=torch.float64)
        dist.all_to_all_single(recv, send, output_split_sizes=[int(c) for c in p["recv_counts"]],
                               input_split_sizes=[int(c) for c in p["send_counts"]])
        data[p["recv_elem"], p["recv_face"]] = recv.numpy()                                               # unpack
        ok = True
        for k, (g, f) in enumerate(zip(p["recv_elem"], p["recv_face"])):
            ok &= bool(np.array_equal(data[g, f], _face_value(el[g], f)))
        untouched = np.ones((el.size, 6), bool)
        untouched[:n] = False
        untouched[p["recv_elem"], p["recv_face"]] = False
        ok &= bool(np.all(data[untouched] == -1.0))                                                      # nothing else was written
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)                                         # the CFL max-allreduce
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        out.put((rank, ok, float(t.item()), int(p["recv_elem"].size)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_halo_exchange_routing_gloo(world):
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=180)
        assert p.exitcode == 0
    for rank, ok, mx, nrecv in res:
        assert ok and mx == float(world) and nrecv > 0
