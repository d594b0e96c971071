"""Host-side logic of bench.py (no GPU): the cost model of SURVEY.md 8(d), the replica aggregation and the
max-over-ranks timing rule under a world_size-2 gloo group (replicas only, no data-path collective)."""
import os
import socket

import pytest

import bench
from harness import synth


def test_cost_model_textbook_numbers():
    # SU(3) fundamental: 1320 flops per hopping site (textbook Wilson dslash), 1368 with the mass term (A15)
    cm = bench.cost_model(synth.CONFIGS["C2"], "f64")
    V = synth.CONFIGS["C2"].volume
    assert cm["F_hop"] == 1320 and cm["S"] == 192 and cm["K"] == 144
    assert cm["ops"]["Dphi_eo"][0] == 1320 * V / 2
    assert cm["ops"]["Dphi"][0] == 1368 * V
    assert cm["ops"]["Dphi_eo"][1] == 1536 * V / 2          # 2S + 8K per output site
    assert cm["ops"]["Dphi_hat"][1] == (5 * 192 + 16 * 144) * V / 2


@pytest.mark.parametrize("name,prec,F,bytes_site", [("C1", "f64", 624, 768), ("C3", "f64", 744, 960), ("C3", "f32", 744, 480),
                                                   ("C4", "f64", 4944, 5376), ("C5", "f64", 80360, 82880), ("C5", "f32", 80360, 41440)])
def test_cost_model_table(name, prec, F, bytes_site):
    cm = bench.cost_model(synth.CONFIGS[name], prec)
    assert cm["F_hop"] == F and 2 * cm["S"] + 8 * cm["K"] == bytes_site


def test_cost_model_rebuild_bytes():
    cm = bench.cost_model(synth.CONFIGS["C4"], "f64", rebuild=True)
    assert 2 * cm["S"] + 8 * cm["K"] == 2816                  # C4 rebuilt = 2S + 8 K_F
    cm = bench.cost_model(synth.CONFIGS["C5"], "f32", rebuild=True)
    assert 2 * cm["S"] + 8 * cm["K"] == 4544


def _worker(rank, world, port, values, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = bench.max_over_ranks(values[rank], dist)
        out.put((rank, ms, bench.aggregate_value(1e9, world, ms)))
    finally:
        dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    values = [2.0, 5.0]
    procs = [ctx.Process(target=_worker, args=(r, 2, port, values, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks see the slower replica's time; the job value counts the units of both replicas over that time
    assert [g[1] for g in got] == [5.0, 5.0]
    assert got[0][2] == pytest.approx(2 * 1e9 / 5e-3 / 1e9)
    assert bench.max_over_ranks(3.5, None) == 3.5
