"""Multi-GPU plumbing on CPU: world_size 2 over gloo (the data path has no collective)."""
import os
import socket
import subprocess
import sys

import numpy as np

from paper_1607_03884_b200 import shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, sys.argv[1])
import numpy as np
from paper_1607_03884_b200 import shard, synth
rank, world = shard.init_process_group("gloo")
n_total = 1001
lo, hi = shard.shard_range(n_total, rank, world)
mech = synth.make_mechanism("h2co", synth.MECH_SEED)
y = synth.make_states(mech, n_total, "uniform", 7)[lo:hi]          # each rank works on its own block only
shard.barrier()
t, units = shard.reduce_max_sum(0.5 + rank, float(hi - lo))
checksum, _ = shard.reduce_max_sum(0.0, float(y[:, 0].sum()))
print(json.dumps({"rank": rank, "lo": lo, "hi": hi, "t": t, "units": units, "tsum": _}))
"""


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 1000, 1048576):
        for world in (1, 2, 3, 8):
            blocks = [shard.shard_range(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [b[1] - b[0] for b in blocks]
            assert max(sizes) - min(sizes) <= 1


def test_two_ranks_over_gloo(tmp_path):
    import json
    port = free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env, stdout=subprocess.PIPE, text=True))
    outs = [json.loads(p.communicate(timeout=120)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    outs.sort(key=lambda o: o["rank"])
    assert (outs[0]["lo"], outs[0]["hi"], outs[1]["lo"], outs[1]["hi"]) == (0, 501, 501, 1001)
    for o in outs:
        assert o["t"] == 1.5 and o["units"] == 1001.0          # max over ranks, sum over ranks
    from paper_1607_03884_b200 import synth
    mech = synth.make_mechanism("h2co", synth.MECH_SEED)
    assert np.isclose(outs[0]["tsum"], synth.make_states(mech, 1001, "uniform", 7)[:, 0].sum())


def test_bench_reference_arm_runs_on_cpu():
    """`bench.py --impl reference` (the oracle on host cores) prints one JSON line with the contract's keys"""
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "1",
                          "--config", "0"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["unit"] == "states/s"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
