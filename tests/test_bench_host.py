"""Host-side logic of bench.py without a GPU: the drive schedule (Q8, S1), the N > 1 aggregation over a
world_size-2 `gloo` group (replicas: time = max over ranks, work = sum), and the reference arm's rank behaviour."""
import json
import os
import subprocess
import sys

import numpy as np
import torch.multiprocessing as mp

import asd_inputs as ai

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_planes_per_shift_follow_the_travel_accumulator():
    for a in (0.3, 0.2725):
        p = [ai.planes_for_shift(q, a) for q in range(1, 201)]
        assert set(p) <= {3, 4}
        assert sum(p) == int(np.floor(200 * 1.0 / a + 1e-9))      # never drifts from the 1 nm-per-shift travel
    assert [ai.planes_for_shift(q, 0.3) for q in (1, 2, 3)] == [3, 3, 4]
    assert [ai.planes_for_shift(q, 0.2725) for q in (1, 2, 3)] == [3, 4, 4]


def test_field_scale_ramp_and_drive():
    import bench
    bits = np.array([1.0, -1.0, -1.0, 1.0])
    assert ai.field_scale_at(0, bits, 100) == 1.0
    assert ai.field_scale_at(100, bits, 100) == 1.0            # start of the ramp towards -1
    assert abs(ai.field_scale_at(150, bits, 100) - 0.0) < 1e-12
    assert ai.field_scale_at(250, bits, 100) == -1.0           # same polarity: no ramp
    assert ai.field_scale_at(10 ** 9, bits, 100) == 1.0

    class W:                                                   # the three fields _drive reads
        bit_seed, bit_steps, shift_every, spacing_nm = 3, 100000, 5000, (0.3, 0.3, 0.3)
    nxt = bench._drive(W, 50)
    shifts = [nxt()[1] for _ in range(400)]                    # 20 000 Heun steps
    assert [i for i, p in enumerate(shifts) if p] == [99, 199, 299, 399]
    assert [p for p in shifts if p] == [3, 3, 4, 3]


def _rank_main(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, upd = bench.reduce_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1), dist, "cpu")
    w = bench._workload(0, seed_offset=rank)                   # replicas differ only by their Philox seed
    out.put((rank, ms, upd, w.seed))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    assert [(r[1], r[2]) for r in res] == [(15.0, 3000.0), (15.0, 3000.0)]   # max of times, sum of work, on every rank
    assert [r[3] for r in res] == [1, 2]


def test_reference_arm_prints_one_line_on_rank_0_only():
    env = dict(os.environ, WORLD_SIZE="2")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "2",
           "--warmup", "1"]
    r0 = subprocess.run(cmd, env=dict(env, RANK="0"), capture_output=True, text=True, timeout=300)
    r1 = subprocess.run(cmd, env=dict(env, RANK="1"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0 and r1.returncode == 0
    assert r1.stdout.strip() == ""
    d = json.loads(r0.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0
    assert d["unit"] == "spin-updates/s" and d["config"]["workload"].startswith("cfg0")
