"""The N > 1 path of bench.py is "replicas only": no data-path
collective, but a barrier and a max-over-ranks of the device time.  That host
logic is covered here with world_size 2 on the gloo backend (no GPU), and the
reference arm's rule that only rank 0 runs and prints."""
import json
import socket
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(script_args, nproc=2, timeout=300):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), *script_args]
    return subprocess.run(cmd, cwd=str(ROOT), capture_output=True, text=True, timeout=timeout)


def _json_lines(text):
    """Every top-level JSON object in `text` (two ranks may interleave their lines on one stdout)."""
    out, dec, i = [], json.JSONDecoder(), 0
    while True:
        i = text.find("{", i)
        if i < 0:
            return out
        try:
            obj, end = dec.raw_decode(text, i)
            out.append(obj)
            i = end
        except json.JSONDecodeError:
            i += 1


def test_replica_timing_logic_world2_gloo():
    r = _torchrun([str(ROOT / "tests" / "_dist_worker.py")])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert sorted(d["rank"] for d in lines) == [0, 1]
    for d in lines:
        assert d["world"] == 2
        assert d["t_max"] == 11.0                      # max over ranks of {10, 11}
        assert abs(d["value"] - 2 * 200 / 11.0) < 1e-12  # whole-job aggregate over both replicas


def test_reference_arm_only_rank0_prints():
    r = _torchrun([str(ROOT / "bench.py"), "--impl", "reference", "--config", "C1", "--gpus", "2", "--steps", "1",
                   "--warmup", "1"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["d2h_bytes_per_step"] == 0


def test_native_arm_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        return
    r = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--config", "C1", "--steps", "1", "--warmup", "1"],
                       cwd=str(ROOT), capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "no CPU fallback" in r.stderr
