"""N > 1 path on CPU: two gloo processes aggregate replica throughput exactly as bench.py does
(sum of chain-steps over ranks / max of elapsed over ranks)."""
import os
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    from paper_2310_20103_b200 import runtime
    rank, local_rank, world = runtime.dist_env()
    dist.init_process_group("gloo")
    units = 1000.0 * (rank + 1)           # replicas may differ only in the test
    elapsed = 2.0 + rank                  # rank 1 is slower: the max must win
    u, t = runtime.aggregate_throughput(units, elapsed)
    v = runtime.whole_job_value(units, elapsed)
    dist.barrier()
    if rank == 0:
        print("RESULT", world, u, t, v)
    dist.destroy_process_group()
""" % ROOT)


def test_two_rank_gloo_aggregation(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", "29511", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("RESULT")][0].split()
    assert int(line[1]) == 2
    assert float(line[2]) == 3000.0 and float(line[3]) == 3.0 and abs(float(line[4]) - 1000.0) < 1e-9


def test_single_process_passthrough():
    from paper_2310_20103_b200 import runtime
    assert runtime.aggregate_throughput(10.0, 2.0) == (10.0, 2.0)
    assert runtime.whole_job_value(10.0, 2.0) == 5.0
    assert runtime.dist_env()[2] >= 1


def test_reference_arm_prints_contract_line():
    """bench.py --impl reference runs the oracle on the host and prints the base-contract JSON line."""
    import json
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    d = json.loads(r.stdout.strip().splitlines()[-1])
    assert d["impl"] == "reference" and d["metric"] == "lanczos_chain_steps_per_s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"].startswith("BASELINE.json:configs[0]")


SHARD_WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, %r)
    import numpy as np, torch
    import torch.distributed as dist
    from oracle import gw_oracle as orc
    from paper_2310_20103_b200 import runtime, synth
    dist.init_process_group("gloo")
    rank = dist.get_rank()
    p = synth.make_custom(3, 4, 12, seed=1)
    omega = np.linspace(-20, 20, 21)
    m, L = 2, 5
    def local(lo, hi):       # stands in for the per-GPU run: the oracle on this rank's slice of n
        out = torch.zeros(len(omega), 2, dtype=torch.float64)
        if hi > lo:
            n = np.arange(lo, hi, dtype=np.int32)
            r = orc.run_chains(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, n, np.full_like(n, m), L, omega, 0.1)
            out[:, 0] = torch.from_numpy(r["sigma_sum"].real.copy()); out[:, 1] = torch.from_numpy(r["sigma_sum"].imag.copy())
        return out
    tot = runtime.sharded_sigma_state(local, 7)
    ref = orc.sigma_state(p.phi_v, p.phi_c, p.eps_v, p.eps_c, p.V, m, L, omega, 0.1)
    err = max(np.abs(tot[:, 0].numpy() - ref.real).max(), np.abs(tot[:, 1].numpy() - ref.imag).max())
    lo, hi = runtime.shard_range(7, rank, dist.get_world_size())
    print("SHARD", rank, lo, hi, err)
    dist.barrier()
    dist.destroy_process_group()
""" % ROOT)


def test_chain_sharded_sigma_state_two_ranks(tmp_path):
    """7 chains over 2 ranks (4 + 3), one all-reduce of the omega grid = Eq. 10."""
    script = tmp_path / "shard_worker.py"
    script.write_text(SHARD_WORKER)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", "29513", str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    rows = sorted(l.split() for l in r.stdout.splitlines() if l.startswith("SHARD"))
    assert [(int(x[2]), int(x[3])) for x in rows] == [(0, 4), (4, 7)]
    assert all(float(x[4]) <= 1e-12 for x in rows)


def test_shard_range_covers_everything():
    from paper_2310_20103_b200 import runtime
    for n in (0, 1, 7, 32, 1280):
        for w in (1, 2, 3, 8):
            cuts = [runtime.shard_range(n, r, w) for r in range(w)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            assert max(h - l for l, h in cuts) - min(h - l for l, h in cuts) <= 1


def test_tile_aligned_shards():
    """runtime.shard_range with quantum = 128 (the GEMM column tile): cuts at multiples of 128, whole tiles balanced to +-1,
    everything covered once, and the largest tile count of any rank is the optimum ceil(tiles / world) -- for the chain
    counts of config 2 (1280), config 3 (5120) and the Si86H76-shaped state (1730) on 8 / 8 / 4 ranks."""
    from paper_2310_20103_b200 import runtime
    q = 128
    for n, w in ((1280, 8), (5120, 8), (1730, 4), (160, 8), (100, 3), (0, 2), (129, 2)):
        cuts = [runtime.shard_range(n, r, w, q) for r in range(w)]
        assert cuts[0][0] == 0 and cuts[-1][1] == n
        assert all(cuts[i][1] == cuts[i + 1][0] for i in range(w - 1))
        assert all((lo % q == 0 or lo == hi == n) and (hi % q == 0 or hi == n) for lo, hi in cuts)   # empty slices sit at n
        tiles = [-(-(hi - lo) // q) for lo, hi in cuts]
        assert max(tiles) == -(-(-(-n // q)) // w) and max(tiles) - min(tiles) <= 1
    assert [hi - lo for lo, hi in (runtime.shard_range(1280, r, 8, q) for r in range(8))] == [256, 256, 128, 128, 128, 128, 128, 128]
    assert [hi - lo for lo, hi in (runtime.shard_range(1730, r, 4, q) for r in range(4))] == [512, 512, 384, 322]
    # the +-1-chain cut of config 2 on 8 ranks pays two tiles for 160 chains on every rank: 62.5 %; the aligned cut, with
    # the same two-tile critical path, is honest about it, and 5120 chains on 8 ranks lose nothing
    assert abs(runtime.tile_efficiency(1280, 8, q) - 0.625) < 1e-12 and runtime.tile_efficiency(5120, 8, q) == 1.0
    assert runtime.shard_range(10, 1, 3) == (4, 7)                              # quantum 1: the old balanced cut
