"""N > 1 path on CPU: two replicas over gloo (world size 2), host halves of the path only.

The D-instance KV path shards by request with no exchange step, so `bench.py --gpus N`
is N independent replicas; what crosses ranks is the barrier, MAX of the time and SUM of the units
(paper_2511_20982_b200/replicas.py).  Each rank here drives a host-only pool (allocator + planner,
a1 / a6 and the work-list half of a4) through the decode schedule bench.py uses, with its own salt,
and the test checks the whole-job aggregate against what the two ranks reported individually."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import json, os, sys, time
sys.path.insert(0, os.environ["KV_ROOT"])
import numpy as np
from paper_2511_20982_b200 import replicas, workloads as W, binding as B
from paper_2511_20982_b200.engine import build_schedule

rep = replicas.init("gloo")
w = W.CONFIGS["cfg3_8b_gqa"].scaled(num_layers=2, batch=32, ingest_per_step=4)
steps = 6
sch = build_schedule(w, steps, bank_steps=2, salt=rep.salt)
cfg = B.PoolConfig(num_layers=w.num_layers, num_q_heads=w.num_q_heads, num_kv_heads=w.num_kv_heads,
                   head_dim=w.head_dim, num_blocks=sch.peak_blocks + 64, max_requests=w.batch + 16,
                   max_blocks_per_request=(w.max_len + steps + 16) // 16 + 1, alloc_seed=w.seed + rep.salt)
pool = B.KVPool(cfg, device=None)                       # host-only: kernels refused, allocator + planner work
pool.reserve(np.arange(w.batch), sch.n0.astype(np.int32))
pool.reserve(sch.prime.arrive, sch.bank_lens[sch.prime.arrive_bank].astype(np.int32))
rep.barrier()
t0 = time.perf_counter()
units = 0
items = 0
for sp in sch.steps:
    pool.free(sp.retire)                                                          # a6
    pool.reserve(sp.arrive, sch.bank_lens[sp.arrive_bank].astype(np.int32))       # a1 (arrivals)
    pool.reserve(sp.batch, np.ones(len(sp.batch), np.int32))                      # a1 (append)
    plan, chunk = pool.plan(sp.batch)                                             # a4, host half
    # every logical block of every request covered exactly once per kv head
    assert int(plan[:, 3].sum()) == int(((sp.lens_after + 15) // 16).sum()) * w.num_kv_heads
    for i, n in zip(sp.batch, sp.lens_after):
        assert pool.block_table(int(i))[1] == int(n)
    units += sp.attn_bytes_layer * w.num_layers + sp.ingest_bytes + sp.append_bytes
    items += len(plan)
ms = (time.perf_counter() - t0) * 1e3 + 1.0 + rep.rank     # ranks report different times on purpose
try:
    B.paged_decode_attention(pool.handle, 0, sch.steps[-1].batch, 4096, 8192)  # dummy non-null addresses: refused before any use
    refused = False
except B.KVError as e:
    refused = e.status == B.KV_ERR_NO_DEVICE
rep.barrier()
value, ms_max = rep.throughput(units, ms)
print("RANK_LINE " + json.dumps({"rank": rep.rank, "world": rep.world, "units": units, "ms": ms, "value": value,
                                  "ms_max": ms_max, "first_len": int(sch.n0[0]), "items": items,
                                  "refused": refused, "stats": pool.stats()}), flush=True)
pool.close()
rep.close()
"""


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_over_gloo(tmp_path):
    port = _free_port()
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), KV_ROOT=ROOT, CUDA_VISIBLE_DEVICES="", OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    lines = []
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        lines += [json.loads(l[len("RANK_LINE "):]) for l in out.splitlines() if l.startswith("RANK_LINE ")]
    assert sorted(l["rank"] for l in lines) == [0, 1] and all(l["world"] == 2 for l in lines)
    a, b = sorted(lines, key=lambda l: l["rank"])
    # weak scaling: each replica draws its OWN requests ...
    assert a["first_len"] != b["first_len"] or a["units"] != b["units"]
    # ... the whole-job value is sum(units) / max(time), identical on every rank
    ms_max = max(a["ms"], b["ms"])
    want = (a["units"] + b["units"]) / (ms_max * 1e-3)
    for l in (a, b):
        assert np.isclose(l["ms_max"], ms_max) and np.isclose(l["value"], want, rtol=1e-12)
        assert l["refused"], "a host-only pool must refuse kernel calls (no CPU fallback)"
        assert l["stats"]["live_requests"] > 0 and l["items"] > 0


def test_single_process_needs_no_group():
    from paper_2511_20982_b200 import replicas
    env_backup = {k: os.environ.pop(k, None) for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    try:
        rep = replicas.init("gloo")
        assert rep.world == 1 and rep.backend is None
        assert rep.max(3.5) == 3.5 and rep.sum(2.0) == 2.0
        v, ms = rep.throughput(10.0, 2.0)
        assert v == 5000.0 and ms == 2.0
        rep.barrier()
        rep.close()
    finally:
        for k, v in env_backup.items():
            if v is not None:
                os.environ[k] = v
