"""The N > 1 path of bench.py on CPU: 2 gloo ranks (events shard, no data-path collective).

Each rank transports its own shard of events (here with the CPU oracle standing in for the GPU library),
the run-level scoring is one sum over ranks and the timing is the max over ranks; the result must equal
the single-process run over all events."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
E_PER_RANK = 3


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _edep_of_events(first_event, n):
    from oracle import binding as ob
    from paper_2209_15445_b200.inputs import field, geometry, materials, primaries
    g = geometry.calorimeter()
    _, tabs, scal = materials.build_material_set(g.material_names)
    o = ob.Oracle(g, tabs, scal, field.no_field())
    prim = primaries.beam(n, 500.0, spread=1.0, seed=1, first_event=first_event)
    e, led, st = o.run(o.make_tracks(prim))
    return e, prim["event"], sum(st.steps)


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    first = bench.shard_first_event(rank, E_PER_RANK)
    e, events, steps = _edep_of_events(first, E_PER_RANK)
    assert list(events) == list(range(rank * E_PER_RANK, (rank + 1) * E_PER_RANK))
    (t_max, _), (steps_all,) = bench.reduce_over_ranks(dist, torch.device("cpu"), [1.0 + rank, 0.0], [steps])
    tot = torch.from_numpy(e.copy())
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)          # the one run-level scoring reduction
    if rank == 0:
        np.save(out, np.concatenate([[t_max, steps_all], tot.numpy()]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_events_and_reduce(tmp_path):
    out = str(tmp_path / "r0.npy")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    got = np.load(out)
    e_all, events, steps = _edep_of_events(0, 2 * E_PER_RANK)
    assert got[0] == 2.0                                # max over ranks of the per-rank time
    assert got[1] == steps                              # sum over ranks of the per-rank step counts
    np.testing.assert_allclose(got[2:], e_all, rtol=1e-12, atol=1e-12)
