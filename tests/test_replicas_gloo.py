"""N > 1 is replicas only: covers the host logic of `bench.py --gpus N` with world_size 2 on
gloo (CPU): distinct time frames per rank, max-over-ranks time, summed work, and the reference arm's rank rule."""
import json
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, {root!r})
    import torch.distributed as dist
    import bench
    from tpc_synth import generate_config
    rank = int(os.environ["RANK"]); world = int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo")
    tf = generate_config("cfg3", n_collisions=1, seed=bench.replica_seed("cfg3", rank))
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    out = bench.aggregate_over_ranks(ms, 2.0 * ms, tf.n, world)
    dist.barrier()
    print("RESULT " + json.dumps({{"rank": rank, "n": tf.n, "out": out, "z0": float(tf.z[0]) if tf.n else 0.0}}), flush=True)
    dist.destroy_process_group()
""")


def test_two_replicas_max_time_sum_work(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29531", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in range(2)]
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err[-2000:]
        line = [ln for ln in out.splitlines() if ln.startswith("RESULT ")][-1]
        d = json.loads(line[7:])
        res[d["rank"]] = d
    assert res[0]["n"] > 0 and res[1]["n"] > 0
    assert (res[0]["n"], res[0]["z0"]) != (res[1]["n"], res[1]["z0"])          # different time frames per rank
    for r in (0, 1):
        ms, ms_e2e, n_total = res[r]["out"]
        assert ms == 15.0 and ms_e2e == 30.0                                    # MAX over ranks
        assert n_total == res[0]["n"] + res[1]["n"]                             # SUM of the work


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.0, 4.0, 7, 1) == (3.0, 4.0, 7)
    assert bench.replica_seed("cfg5", 0) == 5 and bench.replica_seed("cfg5", 3) == 3005


def test_reference_arm_runs_on_rank_zero_only():
    """`bench.py --impl reference` under torchrun: ranks != 0 exit 0 without work and print nothing."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_reference_arm_line_has_the_contract_keys():
    """`bench.py --impl reference` (the oracle as the reference arm) on the small cfg1 workload: one JSON line."""
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload", "cfg1", "--steps", "2",
                        "--warmup", "1"], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "clusters/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1 and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"] == {"value": d["value"], "unit": "clusters/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["config"]["workload"] == "cfg1" and d["steps"] == 2 and d["warmup"] == 1
