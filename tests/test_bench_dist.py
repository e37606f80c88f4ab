"""Host logic of the N>1 bench path on CPU (gloo, world_size 2): walker sharding has no
data-path collective; the only exchange is the max-over-ranks of the step time."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_walkers_partitions_the_batch():
    sys.path.insert(0, ROOT)
    import bench
    for total, world in ((64, 1), (64, 2), (64, 8), (7, 3), (2, 4)):
        spans = [bench.shard_walkers(total, world, r) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == total
        for a, b in zip(spans, spans[1:]):
            assert a[1] == b[0]
        sizes = [hi - lo for lo, hi in spans]
        assert max(sizes) - min(sizes) <= 1


def test_dist_max_over_two_gloo_ranks(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys
        sys.path.insert(0, {ROOT!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        r = dist.get_rank()
        lo, hi = bench.shard_walkers(5, dist.get_world_size(), r)
        m = bench.dist_max(10.0 + r, dist, None)
        assert m == 11.0, m
        # aggregate = units of all ranks / max time: identical on every rank
        open(os.path.join({str(tmp_path)!r}, f"rank{{r}}.txt"), "w").write(f"{{lo}} {{hi}} {{m}}")
        dist.destroy_process_group()
    """))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29531")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                          "--master-addr", "127.0.0.1", "--master-port", "29531", str(script)],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    assert (tmp_path / "rank0.txt").read_text() == "0 3 11.0"
    assert (tmp_path / "rank1.txt").read_text() == "3 5 11.0"
