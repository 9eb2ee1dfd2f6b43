"""CPU tests of bench.py's host logic: the N > 1 path ("replicas only") with world-size-2 gloo, the flop
model, and the reference arm's rank handling."""
import json
import os
import socket
import subprocess
import sys
import textwrap

import bench

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_whole_job_value_and_flop_model():
    assert bench.whole_job_value(4, 1000, 10, 2.0) == 20000.0
    # regrouped Taylor series on harmonically reduced moments (m2p.cuh, tables.cuh): W_{m,e} counts, more terms with
    # order, Yukawa = Laplace + exp
    assert bench.m2p_nw(6) == 84 and bench.m2p_nw(8) == 165 and bench.m2p_nw(0) == 1
    f = [bench.m2p_flops(P, False) for P in (1, 2, 6, 8)]
    assert all(b > a for a, b in zip(f, f[1:]))
    assert bench.m2p_flops(6, True) == bench.m2p_flops(6, False) + 2
    # P = 6: 11 + 48 monomials + 2 * 84 + 6 + 20 + 14 = 267 for one region; twin regions share offsets and monomials
    assert bench.m2p_flops(6, False) == 267 and bench.m2p_flops(6, (False, True)) == 477
    assert bench.m2p_flops(8, True) == 11 + 80 + 2 * 165 + 8 + 28 + 18
    assert bench.m2p_flops(6, (False, True)) < bench.m2p_flops(6, False) + bench.m2p_flops(6, True)
    assert bench.m2p_lap_flops(8) == 344
    assert bench.P2P_FLOPS_FUSED < bench.P2P_FLOPS[False] + bench.P2P_FLOPS[True]


def test_richardson_formulas():
    """eq. (16)-(17), on a manufactured sequence f(h) = f* + C h^p."""
    from paper_1309_4018_b200.richardson import observed_order, extrapolate
    fstar, C, p, r = -41.2465, 0.8, 1.013, 4.0
    f = [fstar + C * h ** p for h in (1.0 / 16, 1.0 / 4, 1.0)]          # fine, medium, coarse
    assert abs(observed_order(f[0], f[1], f[2], r) - p) < 1e-12
    assert abs(extrapolate(f[0], f[1], r, p) - fstar) < 1e-12


def test_max_over_ranks_gloo_world2(tmp_path):
    """Two processes, gloo: every rank must get the slowest rank's time; the aggregate counts both replicas."""
    script = tmp_path / "w.py"
    script.write_text(textwrap.dedent(f"""
        import os, sys, json
        sys.path.insert(0, {ROOT!r})
        import torch.distributed as dist
        import bench
        dist.init_process_group("gloo")
        rank = dist.get_rank()
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")
        v = bench.whole_job_value(dist.get_world_size(), 100, 2, ms * 1e-3)
        dist.barrier()
        open(os.path.join({str(tmp_path)!r}, f"rank{{rank}}.json"), "w").write(json.dumps({{"rank": rank, "ms": ms, "value": v}}))
        dist.destroy_process_group()
    """))
    port = _free_port()
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.load(open(tmp_path / f"rank{r}.json")) for r in (0, 1)]
    assert sorted(l["rank"] for l in lines) == [0, 1]
    for l in lines:
        assert l["ms"] == 15.0 and abs(l["value"] - 2 * 100 * 2 / 0.015) < 1e-6


def test_reference_arm_prints_one_line_from_rank0_only():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "born_l3",
           "--steps", "1", "--warmup", "0"]
    r0 = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=dict(env, RANK="0", WORLD_SIZE="2"))
    r1 = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=dict(env, RANK="1", WORLD_SIZE="2"))
    assert r0.returncode == 0 and r1.returncode == 0 and r1.stdout.strip() == ""
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0 and line["unit"] == bench.UNIT
