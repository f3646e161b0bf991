"""The N > 1 host logic (query sharding, max-over-ranks timing) on CPU with the gloo backend, world_size 2."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_partitions_exactly():
    from paper_2606_08469_b200.dist import shard_range
    for n in (0, 1, 7, 1048576, 921600):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def test_gloo_world_size_2_reduce(tmp_path):
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent("""
        import os, sys
        sys.path.insert(0, %r)
        import torch
        from paper_2606_08469_b200 import dist as D
        rank, local, world = D.env_rank_world()
        D.init_process_group("gloo")
        lo, hi = D.shard_range(1000001, rank, world)
        (mx,), (tot,) = D.reduce_max_sum([1.0 + rank], [hi - lo], torch.device("cpu"))
        assert mx == 2.0 and tot == 1000001, (mx, tot)
        # the optional RGB all-gather: ragged shards (7 rows over 2 ranks = 4 + 3) come back in query order on every rank
        full = torch.arange(21, dtype=torch.float32).reshape(7, 3)
        a, b = D.shard_range(7, rank, world)
        got = D.all_gather_rows(full[a:b].clone(), 7)
        assert torch.equal(got, full), got
        if rank == 0:
            print("OK", mx, tot)
    """ % ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29533", str(script)], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "OK 2.0 1000001" in r.stdout
