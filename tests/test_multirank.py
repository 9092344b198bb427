"""The N>1 host logic of bench.py on CPU: two ranks over `gloo` (world_size 2, 127.0.0.1).

The path has no exchange step ("replicas only"): what N>1 adds is the
per-rank replica seed, the max-over-ranks of the device time and the sum-over-ranks of the
work, plus the rule that only rank 0 of `--impl reference` runs and prints.  No GPU needed."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    import bench
    import meshgen

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank times its own replica: rank r reports (10 + r) ms and its own work
        m = meshgen.make_config("cfg1", bench.rank_seed("cfg1", rank))
        samples = bench.candidate_samples(m)
        dist.barrier()
        tmax, ssum, tsum = bench.reduce_over_ranks(dist, 10.0 + rank, samples, m.T, "cpu")
        q.put((rank, tmax, ssum, tsum, samples, m.T, int(m.verts.astype("int64").sum())))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_reduce_and_replica_seeds():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, s0, n0, own0, T0, sum0), (r1, t1, s1, n1, own1, T1, sum1) = got
    assert (r0, r1) == (0, 1)
    assert t0 == t1 == 11.0                      # max over ranks
    assert s0 == s1 == float(own0 + own1)        # whole-job work = sum over ranks
    assert n0 == n1 == float(T0 + T1)
    assert sum0 != sum1                          # different seeds: replicas are different meshes
    assert own0 > 0 and own1 > 0


def test_single_rank_reduce_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_over_ranks(None, 3.5, 7, 9, "cpu") == (3.5, 7.0, 9.0)


def test_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--workload", "cfg1", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_reference_arm_line_on_small_workload():
    env = dict(os.environ, RANK="0", WORLD_SIZE="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                          "--workload", "cfg2", "--steps", "2", "--warmup", "1"],
                         capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "Gvoxel-samples/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert line["higher_is_better"] is True and line["steps"] == 2 and line["warmup"] == 1


def test_both_arms_print_the_same_config_keys_and_the_capture_guard_reads_its_column():
    """The driver compares the `config` objects of the CUDA arm and of --impl reference: one function builds both.
    profiles/traffic.csv names, per capture, the hash of the kernel sources it was taken from; bench.py nulls
    roofline.frac when that differs from kernel_source_sha256() of the tree being timed."""
    import bench
    import meshgen

    m = meshgen.make_config("cfg1")
    a = bench.workload_config(m, "tets", 1234, 1, 1024)
    b = bench.workload_config(m, "tets", 1234, 1, 1024)
    assert a == b and a["workload"] == m.name and a["bounded_sample_stride"] == 1 and "l2" in a
    src = open(os.path.join(ROOT, "bench.py")).read()
    assert src.count('"config": workload_config(') == 2  # both arms, nothing hand-built beside it
    sha = bench.kernel_source_sha256()
    assert len(sha) == 64 and sha == bench.kernel_source_sha256()
    row = bench.ncu_traffic("cfg4", "k4_flat")
    assert row and len(row["capture_sha256"]) == 64
