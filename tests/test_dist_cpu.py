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


def _bench(*flags, env_drop=("WORLD_SIZE", "RANK", "LOCAL_RANK")):
    env = {k: v for k, v in os.environ.items() if k not in env_drop}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + list(flags), capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout                      # ONE JSON line on stdout, whatever the ranks and NCCL/gloo print elsewhere
    import json
    return json.loads(lines[0])


def test_bench_gpus_n_from_a_plain_shell_starts_n_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment re-launches itself under torch.distributed.run with two
    ranks; --dry-run-dist runs the product arm's N > 1 host logic on CPU (gloo): per-rank frames for weak scaling, shard_range
    slices + all_gather_rows for strong scaling (which must rebuild the one-rank frame exactly: same checksum)."""
    one = _bench("--dry-run-dist")
    assert one["n_gpus"] == 1 and one["queries"] == one["frame"]
    weak = _bench("--gpus", "2", "--dry-run-dist")
    assert weak["n_gpus"] == 2 and weak["scaling"] == "weak" and weak["queries"] == 2 * one["frame"] and weak["max_ms"] == 2.0
    assert one["dist_ranks"] is None and weak["dist_ranks"] == 2          # what the process group itself reports, not the flag
    assert weak["checksum"] != 2 * one["checksum"]        # rank 1 rendered its own frame, not a copy of rank 0's
    strong = _bench("--gpus", "2", "--dry-run-dist", "--scaling", "strong")
    assert strong["n_gpus"] == 2 and strong["scaling"] == "strong" and strong["queries"] == one["frame"]
    assert strong["checksum"] == one["checksum"]
    three = _bench("--gpus", "3", "--dry-run-dist", "--scaling", "strong")      # ragged shards
    assert three["n_gpus"] == 3 and three["checksum"] == one["checksum"] and three["dist_ranks"] == 3


def test_traffic_json_is_refused_when_the_kernel_sources_changed(tmp_path, monkeypatch):
    """bench.py reads the ncu facts of the dominant kernel from profiles/traffic.json only if they were captured from the
    same kernel sources (hash stamp); --ingest-ncu writes that stamp from an ncu launch list."""
    import importlib
    import json
    import shutil
    bench = importlib.import_module("bench")
    root = tmp_path / "repo"
    (root / "profiles").mkdir(parents=True)
    shutil.copytree(os.path.join(ROOT, "paper_2606_08469_b200", "csrc"), root / "paper_2606_08469_b200" / "csrc")
    monkeypatch.setattr(bench, "ROOT", str(root))
    csv = tmp_path / "l.csv"
    head = '"ID","Process ID","Process Name","Host Name","Kernel Name","Context","Stream","Block Size","Grid Size","Device","CC","Section Name","Metric Name","Metric Unit","Metric Value"\n'
    row = '"%d","1","python","h","%s","1","7","(640, 1, 1)","(148, 1, 1)","0","10.0","Command line profiler metrics","%s","%s","%s"\n'
    body = ""
    for i, (k, vals) in enumerate([("oo::pad_atlas_kernel(int)", (1, 2, 3, 4)), ("void oo::fused_tm_kernel<4, 8>(int)", (10, 20, 30, 40)),
                                   ("void oo::fused_tm_kernel<4, 8>(int)", ("54,000,000", 849792, 29900000, 58080))]):
        for m, u, v in zip(("dram__bytes_read.sum", "dram__bytes_write.sum", "smsp__inst_executed.sum", "gpu__time_duration.sum"), ("byte", "byte", "inst", "ns"), vals):
            body += row % (i, k, m, u, v)
    csv.write_text("==PROF== Connected\n" + head + body)

    class A:
        ingest_ncu, ingest_kernel, config = str(csv), "fused", 1
    assert bench.ingest_ncu(A) == 0
    facts, why = bench.ncu_facts(1)
    assert why is None and facts["dram_bytes_per_launch"] == 54849792 and facts["warp_instructions_per_launch"] == 29900000
    assert bench.ncu_facts(2)[0] is None
    with open(root / "paper_2606_08469_b200" / "csrc" / "oo_device.cuh", "a") as f:
        f.write("// changed\n")
    facts, why = bench.ncu_facts(1)
    assert facts is None and "stale" in why
