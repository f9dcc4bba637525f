"""N > 1 path of bench.py on the CPU: world size 2, gloo.  The data path has no collective (replicas
only); what is multi-rank is host logic: per-rank fluence sequences, the max-over-ranks
reduction of the timed region, whole-job aggregation, rank-0-only output."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _torchrun(script_args, tmp_path, extra_env=None):
    env = dict(os.environ, VMAT_TEST_OUT=str(tmp_path / "out"), **(extra_env or {}))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", "29581"] + script_args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=300)


def test_two_rank_reduction_and_seeds(tmp_path):
    r = _torchrun([os.path.join(ROOT, "tests", "_dist_worker.py")], tmp_path)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                     # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["t"] == [11.0, 20.0]                            # max over ranks of each timed region
    assert out["ms_per_step"] == 11.0 / 50 and abs(out["value"] - 2 * 50 / 11.0e-3) < 1e-6   # whole-job throughput
    other = json.load(open(str(tmp_path / "out") + ".1"))
    assert not set(out["idx0"]) & set(other["idx"])            # ranks draw different x sequences


def test_reference_arm_runs_on_rank0_only(tmp_path):
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--gpus", "2",
                   "--steps", "2", "--warmup", "1"], tmp_path)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    out = json.loads(lines[0])
    assert out["impl"] == "reference" and out["n_gpus"] == 2 and out["cpu_baseline"]["kind"] == "oracle"
    assert out["e2e"]["h2d_bytes_per_step"] == 0 and out["value"] > 0
