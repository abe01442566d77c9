"""world_size-2 gloo test of the multi-GPU host logic: the path shards by template
with no data-path collective; ranks only agree on the slowest device time."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_two_ranks_gloo():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29653", os.path.join(ROOT, "tests", "_gloo_worker.py")]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("{")][-1]
    r = json.loads(line)
    assert r["world"] == 2
    assert r["digests"][0] != r["digests"][1]                      # disjoint template shards (different banks)
    assert r["ranges"] == [[0, 512], [512, 1024]]                  # contiguous cover of the template range
    assert r["slow"] == 11.0                                        # max over ranks
    assert r["total_updates"] == 2 * r["per_rank_updates"]         # weak scaling: units add up


def test_shard_templates_covers_everything():
    from paper_1702_02256_b200 import inputs
    for T in (1, 7, 1024, 16384):
        for world in (1, 2, 3, 8):
            spans = [inputs.shard_templates(T, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == T
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
