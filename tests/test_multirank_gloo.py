"""N > 1 on CPU (gloo, world size 2): the path shards as independent populations, so the
multi-rank logic is bench.py's rank seeding and its max-over-ranks time / sum-over-ranks work reduction.
The oracle stands in for the per-rank population here (no GPU in this test): two ranks anneal different
seeds, and the whole-job throughput is (sum of updates) / (max of times)."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist            # noqa: E402
import torch.multiprocessing as mp          # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from oracle import pa_oracle as po
    from paper_1703_03676_b200.workloads import CONFIGS
    wl = CONFIGS[1]
    seed = bench.rank_seed(wl, rank)
    o = po.Oracle(wl.L, 64, seed)
    betas = wl.betas()
    o.resample(betas[0], betas[1]); o.sweep(betas[1], 2)
    E, _ = o.energies()
    units = o.population * wl.N * 2
    ms = 10.0 * (rank + 1)                                   # rank 1 is the slow one
    t, u = bench.reduce_over_ranks(ms, units, "cpu", dist)
    # Eq. 6-7: the ranks' runs combined by their free-energy estimates
    ob = o.observables(betas[1])
    comb = bench.combine_over_ranks(o.lnZ, ob, "cpu", dist, po.weighted_average)
    # Adaptive mode: the first run -- rank 0 -- decides every temperature step, the others keep its sequence,
    # so that Eq. 6-7 may combine the runs at every temperature.  8 bytes broadcast per step.
    from paper_1703_03676_b200.workloads import Workload
    wa = Workload("adaptive_small", 8, 96, 40, 0.0, 1.0, None, 2, target_overlap=0.8)
    a = po.Oracle(wa.L, wa.R, bench.rank_seed(wa, rank))
    own = a.adapt_dbeta(wa.target_overlap, 0.0, wa.beta_f)           # what this rank would have chosen on its own
    sched, beta = [], 0.0
    for i in range(1, 4):
        new = bench.next_beta(a, wa, None, i, beta, dist)
        a.resample(beta, new); a.sweep(new, wa.theta)
        sched.append(new); beta = new
    comb_a = bench.combine_over_ranks(a.lnZ, a.observables(beta), "cpu", dist, po.weighted_average)
    allu = [None] * world
    dist.all_gather_object(allu, (seed, int(units), int(E.sum()), o.lnZ, ob["e"], comb, own, sched, comb_a))
    dist.barrier()
    if rank == 0:
        q.put((t, u, allu))
    dist.destroy_process_group()


def test_two_ranks_independent_populations_and_reduction():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    t, u, allu = q.get()
    assert t == 20.0                                         # max over ranks
    assert u == float(sum(x[1] for x in allu))               # sum over ranks
    assert allu[0][0] != allu[1][0]                          # different seeds ...
    assert allu[0][2] != allu[1][2]                          # ... different populations
    # the weighted average: both ranks hold the same result; weights follow exp(lnZ_m); e~ = sum omega_m e_m
    import math
    c0, c1 = allu[0][5], allu[1][5]
    assert c0 == c1 and c0["runs"] == 2
    w0 = 1.0 / (1.0 + math.exp(allu[1][3] - allu[0][3]))
    assert c0["omega"][0] == pytest.approx(w0, rel=1e-12) and sum(c0["omega"]) == pytest.approx(1.0, rel=1e-14)
    assert c0["e"] == pytest.approx(w0 * allu[0][4] + (1 - w0) * allu[1][4], rel=1e-12)


    # adaptive protocol: both ranks walked rank 0's temperatures although their own bisections differ
    assert allu[0][6] != allu[1][6]
    assert allu[0][7] == allu[1][7] and allu[0][7][0] == allu[0][6] and len(allu[0][7]) == 3
    assert all(b > a for a, b in zip(allu[0][7], allu[0][7][1:]))
    assert allu[0][8] == allu[1][8] and allu[0][8]["runs"] == 2


def test_single_rank_reduction_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.5, 7, "cpu", None) == (3.5, 7.0)
    from oracle import pa_oracle as po
    ob = {"e": -1.0, "C": 0.5, "absm": 0.2, "m2": 0.1, "m4": 0.05}
    c = bench.combine_over_ranks(12.0, ob, "cpu", None, po.weighted_average)
    assert c["runs"] == 1 and c["omega"] == [1.0] and all(c[k] == ob[k] for k in ob)
