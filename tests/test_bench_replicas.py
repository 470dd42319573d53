"""bench.py's N > 1 path is "replicas only": no data-path collective, one max-over-ranks
of the device-timed durations.  Covered here with two gloo processes on CPU; plus the algorithmic byte counts."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    ms = bench.reduce_max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")
    out.put((rank, ms, bench.job_throughput(1_000_000, 10, world, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks see the slower rank's 15 ms; the job assembled 2 x 1M cells x 10 steps in it
    assert [g[1] for g in got] == [15.0, 15.0]
    assert got[0][2] == pytest.approx(2 * 1e6 * 10 / 15e-3 / 1e6)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.reduce_max_over_ranks(3.5, 1) == 3.5
    assert bench.job_throughput(1_000_000, 10, 1, 30.0) == pytest.approx(1e6 * 10 / 30e-3 / 1e6)


def test_algorithmic_bytes_match_design():
    """11 596 B per interior cell for k_assemble, about 890 B for k_gradient_limiter."""
    import bench
    nc, nnzb, nst = 1_000_000, 3_997_000, 12_400_000
    asm, grad = bench.algorithmic_bytes(nc, nnzb, nst)
    assert asm == nnzb * 2592 + nc * (3 * 144 + 144 + 432 + 192 + 28)
    assert grad == nc * (144 + 4 + 64 + 432) + nst * 20
    # quadrilateral meshes: 4 face slots (576 B of face states, 256 B of geometry, 16 + 32 B of tables per cell)
    asm4, grad4 = bench.algorithmic_bytes(262144, 5 * 262144, 8 * 262144, F=4)
    assert asm4 == 5 * 262144 * 2592 + 262144 * (3 * 144 + 144 + 576 + 256 + 48)
    assert grad4 == 262144 * (144 + 4 + 80 + 576) + 8 * 262144 * 20
    # packed Jacobian: full diagonal blocks, 114 entries per off-diagonal block
    asm_p, _ = bench.algorithmic_bytes(nc, nnzb, nst, packed=True)
    assert asm - asm_p == (nnzb - nc) * (2592 - 912)
    # SURVEY 8(d)'s own per-step figures: 11.19 KB / 12.05 KB per interior triangle
    fused, stored = bench.survey_bytes(nc, 4 * nc)
    assert fused == nc * (10368 + 432 + 144 + 250) and stored - fused == nc * 864
