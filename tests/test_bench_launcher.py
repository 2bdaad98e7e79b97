"""-m "not gpu": bench.py's N > 1 plumbing without a GPU.  `--dry-run` keeps the launcher, the
rank / world checks, the seed partition, the ragged reward all-gather, the max-over-ranks timing and the JSON line,
and replaces the CUDA step with a stub over gloo."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
BENCH = os.path.join(ROOT, "bench.py")


def _run(cmd, env=None, timeout=300):
    e = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    e.update(env or {})
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=e, cwd=ROOT)


def _json_lines(stdout):
    return [json.loads(l) for l in stdout.splitlines() if l.startswith("{")]


@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_gpus_flag_starts_that_many_ranks(scaling):
    """`python bench.py --gpus 2` (no torchrun around it) must run TWO ranks and print ONE line with n_gpus 2."""
    r = _run([sys.executable, BENCH, "--gpus", "2", "--dry-run", "--steps", "2", "--warmup", "1", "--scaling", scaling])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    line = lines[0]
    assert line["n_gpus"] == 2 and line["scaling"] == scaling and line["dry_run"] is True
    assert line["config"]["parallelism"].startswith("dp2 " + scaling)
    assert line["rewards_gathered"] == (32 if scaling == "weak" else 16)       # cfg3: 16 sequences per rank / in the one batch
    assert "starting 2 ranks" in r.stderr


def test_driver_style_torchrun_launch():
    """The driver's own command line: torch.distributed.run around bench.py --gpus N."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    r = _run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
              "--master-port", str(port), BENCH, "--gpus", "2", "--dry-run", "--steps", "2", "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2
    assert "starting 2 ranks" not in r.stderr                       # no second level of ranks


def test_mismatched_world_size_and_missing_devices_fail_loudly():
    r = _run([sys.executable, BENCH, "--gpus", "2", "--dry-run"], env={"WORLD_SIZE": "3", "RANK": "0"})
    assert r.returncode != 0 and "WORLD_SIZE=3" in r.stderr and not _json_lines(r.stdout)
    import torch
    if torch.cuda.device_count() < 8:
        r = _run([sys.executable, BENCH, "--gpus", "8"])
        assert r.returncode != 0 and "CUDA device(s) are visible" in r.stderr and not _json_lines(r.stdout)


def test_job_seeds_partition():
    sys.path.insert(0, ROOT)
    import bench
    from synth import CONFIGS
    s = CONFIGS[3]
    weak = [bench.job_seeds(s, "weak", r, 4) for r in range(4)]
    flat = [v for w in weak for v in w]
    assert all(len(w) == s.n_seqs for w in weak) and len(set(flat)) == 4 * s.n_seqs      # disjoint seed groups
    assert weak[0] == list(s.seeds)                                                     # rank 0 = the 1-GPU job
    assert all(bench.job_seeds(s, "strong", r, 4) == list(s.seeds) for r in range(4))   # one batch, sliced by explore_sharded
