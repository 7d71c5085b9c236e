"""Host-side logic of the N > 1 path of bench.py on CPU (gloo, world_size 2).  The path does not shard (DESIGN.md sec 9:
replicas only), so what there is to test is: one independent lattice per rank with its own seed, the MAX over ranks of the
timed region, the whole-job value, and that only rank 0 of the reference arm works and prints."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replicas_max_over_ranks_and_value_gloo():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_rank_helper.py")]
    env = dict(os.environ, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("RANKS ")]
    assert len(lines) == 1, r.stdout
    ranks = json.loads(lines[0][6:])
    assert [x["rank"] for x in ranks] == [0, 1] and all(x["world"] == 2 for x in ranks)
    assert ranks[0]["seed"] != ranks[1]["seed"] and ranks[0]["seed"] == 42          # independent lattices, rank 0 = config 3
    assert ranks[0]["ms_max"] == ranks[1]["ms_max"] == 125.0                         # the slowest rank's time, on every rank
    want = 2 * (4 * 32 ** 4) * 10 / 0.125                                            # all replicas' links / that time
    assert abs(ranks[0]["value"] - want) < 1e-6 * want and ranks[0]["value"] == ranks[1]["value"]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1", CUDA_VISIBLE_DEVICES="")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=120, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == "", (r.returncode, r.stdout, r.stderr[-500:])
