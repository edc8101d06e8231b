"""N > 1 path of bench.py on CPU (gloo, world_size 2): "replicas only" -- each rank times its own
replica, the job time is the MAX over ranks and the value is the aggregate over all replicas.  No data-path
collective exists to test; this covers the rendezvous, the max-over-ranks reduction and the aggregation."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = [10.0 + 5.0 * rank, 100.0 - 7.0 * rank]            # rank 1 is slower on the first, rank 0 on the second
    ms_max, e2e_max = bench.max_over_ranks(local_ms, world, "cpu")
    dist.barrier()
    q.put((rank, ms_max, e2e_max, bench.job_value(world, 1000, 4, ms_max * 1e-3)))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_and_aggregate_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_max, e2e_max, value in res:
        assert ms_max == 15.0 and e2e_max == 100.0                 # every rank sees the max over ranks
        assert value == pytest.approx(2 * 1000 * 4 / 15.0e-3)      # aggregate of 2 replicas over the slowest rank's time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([3.0, 4.0], 1, "cpu") == [3.0, 4.0]
    assert bench.job_value(1, 16777216, 120, 0.6) == pytest.approx(16777216 * 120 / 0.6)


def test_reference_arm_non_zero_ranks_do_no_work(monkeypatch, capsys):
    """`bench.py --impl reference` under torchrun: only rank 0 runs and prints."""
    sys.path.insert(0, ROOT)
    import argparse
    import bench
    bench.run_reference(argparse.Namespace(config=3, steps=1, warmup=0, gpus=2), rank=1)
    assert capsys.readouterr().out == ""


def test_ncu_table_is_readable_and_covers_the_headline_variant():
    """bench.py takes its ncu-only counters (DRAM bytes, FP64 warp-instructions, pipe utilisation) from the committed
    summary profiles/r2_ncu_kernels.csv: the table must parse, carry the sha of the sources it was taken at, and hold
    the three sweep classes of the headline variant (config 3, fp64, WENO7, nf = 4) and of the variants with a claim."""
    sys.path.insert(0, ROOT)
    import bench
    for variant in ("cfg3_f64_w7_nf4_lim0", "cfg3_f64_w5_nf4_lim0", "cfg3_f32_w7_nf4_lim0", "cfg3_f64_w7_nf4_lim1",
                    "cfg4_f64_w7_nf5_lim0"):
        rows = bench.ncu_rows(variant)
        assert {"sweep_x", "sweep_y", "sweep_z", "prim"} <= set(rows), variant
        shas = {r["csrc_sha"] for rs in rows.values() for r in rs}
        assert len(shas) == 1 and len(next(iter(shas))) == 16
        traffic = bench.ncu_pass_mean(rows, "dram_read_B") + bench.ncu_pass_mean(rows, "dram_write_B")
        cells = 512 ** 3 if variant.startswith("cfg4") else 256 ** 3
        nf, esz = (5 if "nf5" in variant else 4), (4 if "f32" in variant else 8)
        floor = 8.0 * nf * esz * cells / 9.0                  # unique bytes of a fused stage, per pass
        assert 2.0 * floor < traffic < 6.0 * floor, (variant, traffic / floor)
    # a 5-field fp64 pass is two kernels (fields 0..3 + baryon density): their counters add up per pass
    rows = bench.ncu_rows("cfg4_f64_w7_nf5_lim0")
    assert len(rows["sweep_y"]) == 2 and len(rows["sweep_x"]) == 4
    assert bench.variant_key(3, 64, 7, 4, False) == "cfg3_f64_w7_nf4_lim0"
