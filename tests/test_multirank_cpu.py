"""World-size-2 gloo test (CPU) of the N > 1 bookkeeping bench.py uses: the path shards by
independent segments, so ranks exchange nothing but a barrier and the MAX of
their timings; whole-job throughput = images of all ranks / max time."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys
    sys.path.insert(0, {root!r})
    import numpy as np
    import torch, torch.distributed as dist
    import oracle as O, workloads as W
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    cfg = W.get_config("tiny")
    f, uvw, dms = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg), W.dm_list(cfg)
    cell = W.default_cell_rad(cfg, uvw)
    # each rank searches its own segment (different noise rows), no data-path collective
    vis = W.noise_rows(cfg, range(1000 * rank, 1000 * rank + cfg.nint))
    delays = O.delay_table(f, dms, cfg.inttime_s)
    n_img = sum(O.n_images(cfg.nint, int(delays[d].max()), dt) for d in range(cfg.ndm) for dt in cfg.dt_list)
    cands = O.search(vis, f, uvw, cfg.inttime_s, cfg.npix, cell, dms[:2], cfg.dt_list, 4.0)
    dist.barrier()
    t = torch.tensor([10.0 + 5.0 * rank, float(n_img), float(len(cands))], dtype=torch.float64)
    tmax = t.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    tsum = t.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    if rank == 0:
        assert tmax[0].item() == 10.0 + 5.0 * (world - 1)
        assert tsum[1].item() == world * n_img
        value = tsum[1].item() / (tmax[0].item() * 1e-3)
        print("OK", world, int(tsum[1].item()), value)
    dist.destroy_process_group()
""")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_replicas(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    line = [l for l in out.stdout.splitlines() if l.startswith("OK")]
    assert line and line[0].split()[1] == "2" and int(line[0].split()[2]) == 2 * 388
