"""The N > 1 path of bench.py on CPU: world_size 2 over gloo (replicas only -- no data-path collective;
the only traffic is the barrier and the max-over-ranks of the device-timed region), and the reference arm under a 2-rank launch
(rank 0 alone runs and prints, the other rank exits 0 without work)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=world)
dist.barrier()
secs = [0.30, 0.42][rank]                      # the slower rank decides
ms_step, ms_eval = bench.replicas_step_time(secs, 3, world, dist, torch, torch.device("cpu"))
dist.barrier()
print("RESULT", rank, repr(ms_step), repr(ms_eval), flush=True)
dist.destroy_process_group()
"""


def _spawn(code, port, extra_env=None):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        env.update(extra_env or {})
        procs.append(subprocess.Popen([sys.executable, "-c", code], cwd=ROOT, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


def test_step_time_is_the_max_over_ranks_and_replicas_divide_it():
    res = _spawn(_WORKER.format(root=ROOT), 29541)
    got = {}
    for rc, out, err in res:
        assert rc == 0, err[-2000:]
        for line in out.splitlines():
            if line.startswith("RESULT"):
                _, r, a, b = line.split()
                got[int(r)] = (float(a), float(b))
    assert set(got) == {0, 1}
    for r in (0, 1):                            # both ranks hold the same, max-reduced numbers
        assert abs(got[r][0] - 0.42 / 3 * 1e3) < 1e-9 and abs(got[r][1] - 0.42 / 3 * 1e3 / 2) < 1e-9
    import bench                                # N = 1: no collective, no division
    assert bench.replicas_step_time(0.5, 5, 1) == (100.0, 100.0)


def test_reference_arm_under_a_two_rank_launch_runs_on_rank_0_only():
    code = "import sys; sys.argv = ['bench.py', '--impl', 'reference', '--workload', 'cfg1', '--steps', '1', '--warmup', '0']; import bench; bench.main()"
    res = _spawn(code, 29542)
    (rc0, out0, err0), (rc1, out1, err1) = res
    assert rc0 == 0 and rc1 == 0, (err0[-1500:], err1[-1500:])
    lines = [l for l in out0.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and out1.strip() == ""
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "ms_per_gw_sigma_evaluation" and d["higher_is_better"] is False
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
