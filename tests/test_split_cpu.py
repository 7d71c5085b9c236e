"""CPU tests of the host-side bookkeeping of a divided lattice (paper_1310_7087_b200/split.py):
the partition into even, possibly unequal parts, who sends which boundary layer to whom, and -- with two gloo ranks, each
owning one part and an oracle-backed stand-in for the GPU slab -- that the schedule (one-site halos of the array a sub-step
wrote, refreshed after every sub-step) reproduces the undivided oracle bit for bit.  Everything a rank does not own or hold
as a halo copy is NaN, so any read beyond the halo poisons the result."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _split():
    sys.path.insert(0, ROOT)
    import importlib.util
    spec = importlib.util.spec_from_file_location("qcd_split_host", os.path.join(ROOT, "paper_1310_7087_b200", "split.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_partition_even_unequal_and_weighted():
    sp = _split()
    assert sp.partition(32, 1) == [(0, 32)]
    assert sp.partition(32, 2) == [(0, 16), (16, 16)]
    assert sp.partition(12, 4) == [(0, 4), (4, 4), (8, 2), (10, 2)] or sorted(e for _, e in sp.partition(12, 4)) == [2, 2, 4, 4]
    for extent, n, w in [(48, 5, None), (64, 8, None), (32, 3, [1, 2, 1]), (20, 2, [3, 1]), (16, 8, None)]:
        parts = sp.partition(extent, n, w)
        assert len(parts) == n and parts[0][0] == 0
        assert all(o % 2 == 0 and e % 2 == 0 and e >= 2 for o, e in parts)
        assert all(parts[k][0] + parts[k][1] == parts[k + 1][0] for k in range(n - 1)) and parts[-1][0] + parts[-1][1] == extent
    w = sp.partition(32, 3, [1, 2, 1])
    assert w[1][1] > w[0][1] and w[1][1] > w[2][1]           # the faster device gets the larger part
    with pytest.raises(ValueError):
        sp.partition(8, 5)
    with pytest.raises(ValueError):
        sp.partition(7, 2)


def test_neighbours_messages_and_schedule():
    sp = _split()
    assert sp.neighbours(0, 4) == (3, 1) and sp.neighbours(3, 4) == (2, 0) and sp.neighbours(0, 1) == (0, 0)
    # first own layer -> previous part's copy of "next part's first layer"; last own layer -> next part's copy of "previous ... last"
    assert sp.halo_messages(1, 4) == [(0, 0, 1), (1, 2, 0)]
    assert sp.halo_messages(0, 2) == [(0, 1, 1), (1, 1, 0)]
    sched = sp.sweep_schedule(4, 1, 4)
    assert len(sched) == 40 and sched[0] == (0, 0, 0, 0) and sched[7] == (0, 0, 1, 3) and sched[8] == (1, 0, 0, 0) and sched[-1] == (1, 0, 1, 3)
    assert sp.sweep_schedule(3, 2, 0)[6] == (0, 1, 0, 0)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("case", ["su3_4d", "su2_3d_unequal"])
def test_two_ranks_reproduce_the_undivided_oracle_gloo(case):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_split_rank_helper.py"), case]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-3000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("SPLIT ")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0][6:])
    assert out["parts"][0][0] == 0 and sum(e for _, e in out["parts"]) == out["split_extent"]
    assert out["links_equal"] is True and out["nan_free_owned"] is True
    assert out["max_measure_diff"] < 1e-13
    assert out["messages_per_substep_per_rank"] == 2
