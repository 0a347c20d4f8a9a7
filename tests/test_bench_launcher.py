"""-m "not gpu": `bench.py --gpus N` starts N ranks itself (PAPER.md:177-183 is the paper's multi-GPU claim).

The --dry-run flag runs the launcher, the rendezvous, the source partition and the one gather of the loops on CPU over gloo;
no kernel runs and nothing is timed."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _run(args, env=None):
    e = dict(os.environ)
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        e.pop(k, None)
    e.update(env or {})
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py")] + args, capture_output=True, text=True, env=e, timeout=300)


def test_bare_gpus_2_launches_two_ranks():
    r = _run(["--gpus", "2", "--dry-run"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1  # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["ranks_reported"] == [0, 1]
    assert out["gather_in_source_order"] is True and out["sources"] == 24 and out["max_over_ranks"] == 2.0


def test_single_rank_needs_no_launcher():
    r = _run(["--dry-run"])
    assert r.returncode == 0, r.stderr[-2000:]
    out = json.loads([l for l in r.stdout.splitlines() if l.startswith("{")][0])
    assert out["n_gpus"] == 1 and out["ranks_reported"] == [0]


def test_rank_count_must_match_gpus():
    r = _run(["--gpus", "2", "--dry-run"], env={"WORLD_SIZE": "3", "RANK": "0", "LOCAL_RANK": "0"})
    assert r.returncode != 0 and "must equal --gpus" in (r.stderr + r.stdout)


def test_traffic_record_is_tied_to_the_kernel_signature(tmp_path, monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    rec = tmp_path / "t.json"
    rec.write_text(json.dumps({"signature": "k<1>", "dram_bytes_per_launch": 2.5e9, "source": "x.md"}))
    monkeypatch.setattr(bench, "TRAFFIC_RECORD", str(rec))
    v, src = bench.ncu_traffic("k<1>")
    assert v == 2.5e9
    v, src = bench.ncu_traffic("k<2>")
    assert v is None and "stale" in src
    monkeypatch.setattr(bench, "TRAFFIC_RECORD", str(tmp_path / "missing.json"))
    assert bench.ncu_traffic("k<1>")[0] is None
