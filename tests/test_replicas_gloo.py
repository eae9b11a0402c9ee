"""Multi-GPU path of bench.py ("replicas only"): N independent simulations, one process per
GPU, no data-path collective.  The only collectives are the barrier around the timed region and the reductions in
`bench.aggregate` (MAX of the device time, SUM of the vehicle-updates).  Covered here with world_size = 2 on the
`gloo` backend (CPU); `--impl reference` under a multi-rank launch lets rank 0 alone work."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r: 10 + 5 r ms for (r + 1) million updates
    ms_max, upd_all, value = bench.aggregate(10.0 + 5.0 * rank, 1.0e6 * (rank + 1), world, "cpu")
    dist.barrier()
    out[rank] = (ms_max, upd_all, value)
    dist.destroy_process_group()


def test_aggregate_world_size_2_gloo():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for r in (0, 1):
        ms_max, upd_all, value = res[r]
        assert ms_max == 15.0                      # MAX over ranks
        assert upd_all == 3.0e6                    # SUM over ranks
        assert value == pytest.approx(3.0e6 / 15.0e-3)


def test_aggregate_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(4.0, 2000.0, 1, "cpu") == (4.0, 2000.0, 2000.0 / 4.0e-3)


def test_reference_arm_other_ranks_exit_without_work():
    """`bench.py --impl reference` under torchrun: ranks other than 0 print nothing and exit 0."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""
