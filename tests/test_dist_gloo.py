"""World-size-2 host logic of bench.py on CPU (gloo): rendezvous on 127.0.0.1, barrier, max-over-ranks timing and
the whole-job value of the session-sharded replicas (no data-path collective), and the
reference arm's rule that rank 0 alone runs and prints."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

RANK_SNIPPET = r"""
import json, os, sys
sys.path.insert(0, {root!r})
import torch
import bench
d = bench.Dist(2)
assert d.on and d.world == 2
d.init("gloo")
d.barrier()
mine = 1.0 + d.rank            # this rank's device time for K steps, ms
worst = d.max(mine, torch.device("cpu"))
d.barrier()
n_sess, steps = 3, 4
value = (worst / steps) * 1e3 / (n_sess * d.world)   # us per session over the whole job (weak scaling)
print(json.dumps({{"rank": d.rank, "worst": worst, "value": value}}))
d.close()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _launch(code, port, extra_args=()):
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable] + list(code) + list(extra_args), env=env, cwd=ROOT,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=240) for p in procs]
    return [(p.returncode, o, e) for p, (o, e) in zip(procs, outs)]


def test_two_ranks_barrier_and_max_over_ranks():
    res = _launch(["-c", RANK_SNIPPET.format(root=ROOT)], _free_port())
    lines = []
    for rc, out, err in res:
        assert rc == 0, err[-2000:]
        lines.append(json.loads(out.strip().splitlines()[-1]))
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["worst"] == 2.0                       # the slower rank's time, on both ranks
        assert abs(l["value"] - (2.0 / 4) * 1e3 / 6) < 1e-9


def test_reference_arm_only_rank0_prints():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the one JSON line, rank 1 exits 0 silently."""
    res = _launch([os.path.join(ROOT, "bench.py")], _free_port(),
                  ["--impl", "reference", "--gpus", "2", "--config", "c1", "--steps", "1", "--warmup", "1"])
    (rc0, out0, err0), (rc1, out1, err1) = res
    assert rc0 == 0, err0[-2000:]
    assert rc1 == 0, err1[-2000:]
    line = json.loads([x for x in out0.splitlines() if x.startswith("{")][-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "us/session"
    assert not [x for x in out1.splitlines() if x.startswith("{")]
