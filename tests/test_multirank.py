"""World-size-2 gloo test (CPU) of the N > 1 path of bench.py: rank sharding and the cross-rank reduction.
The hot path itself has no collective; this covers the only multi-rank logic there is."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2606_28831_b200 import accounting, sharding
    wl = sharding.rank_workload(2, rank, B=2, n0=np.array([700, 900], np.int32), max_ctx=1024, k_cap=128,
                                l_upper=np.array([568, 768], np.int32), cond_cap=8)
    K0, _ = wl.prefill_unit(0, 0)
    # a fake measurement per rank: bytes from the shared accounting module, time rank-dependent
    nb = accounting.algorithmic_bytes(wl, wl.n0 + 1, np.full(wl.B, wl.sink), np.full(wl.B * wl.Hkv, 100),
                                      np.zeros(wl.B * wl.Hkv))["total"]
    ms, e2e, tot = sharding.reduce_run(10.0 + rank, 20.0 - rank, nb, "cpu")
    dist.barrier()
    q.put((rank, wl.seed, tuple(K0.shape), float(K0[0, 0]), nb, ms, e2e, tot))
    dist.destroy_process_group()


def test_two_ranks_shard_and_reduce():
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, sh0, v0, nb0, ms0, e0, t0), (r1, s1, sh1, v1, nb1, ms1, e1, t1) = res
    assert (r0, r1) == (0, 1)
    assert s1 == s0 + 1000 and sh0 == sh1 and v0 != v1          # same shapes, different data
    assert ms0 == ms1 == 11.0 and e0 == e1 == 20.0              # max over ranks
    assert t0 == t1 == nb0 + nb1                                # bytes of the whole job
    from paper_2606_28831_b200 import sharding
    assert abs(sharding.job_throughput_gbs(ms0, t0) - (nb0 + nb1) / 11e-3 / 1e9) < 1e-9


def _tp_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle.batch import OracleBatch
    from paper_2606_28831_b200 import sharding
    from workloads.synth import make_workload
    full = make_workload(2, B=2, n0=np.array([700, 900], np.int32), max_ctx=1024, k_cap=256,
                         l_upper=np.array([568, 768], np.int32), cond_cap=8)
    sh = sharding.head_shard(full, rank, world)
    assert (sh.Hkv, sh.Hq, sh.G) == (full.Hkv // world, full.Hq // world, full.G)
    ob = OracleBatch(sh, {(b, h): sh.prefill_unit(b, h) for b in range(sh.B) for h in range(sh.Hkv)})
    outs = []
    for t in range(3):
        kn, vn = sh.step_kv(t, None)
        ob.step(sh.step_q(t), kn, vn, sh.p)
        local = torch.from_numpy(ob.sel_count().reshape(sh.B, sh.Hkv))
        counts = sharding.gather_head_counts(local, world)          # the one exchange of the TP deployment (L562)
        outs.append((counts.numpy().copy(), ob.out().copy()))
    dist.barrier()
    q.put((rank, outs))
    dist.destroy_process_group()


def test_kv_head_sharding_gathers_the_single_gpu_counts():
    """Width sharding: two ranks take half the KV heads each, select on their own heads, and
    all-gather the per-head counts.  The gathered [B][Hkv] counts on every rank, and each rank's outputs, equal what one
    process computes for the whole batch (units are independent: no other exchange exists)."""
    from oracle.batch import OracleBatch
    from workloads.synth import make_workload
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_tp_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = dict(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = make_workload(2, B=2, n0=np.array([700, 900], np.int32), max_ctx=1024, k_cap=256,
                         l_upper=np.array([568, 768], np.int32), cond_cap=8)
    ob = OracleBatch(full, {(b, h): full.prefill_unit(b, h) for b in range(full.B) for h in range(full.Hkv)})
    for t in range(3):
        kn, vn = full.step_kv(t, None)
        ob.step(full.step_q(t), kn, vn, full.p)
        want = ob.sel_count().reshape(full.B, full.Hkv)
        assert want.min() >= 1 and len(set(want.reshape(-1).tolist())) > 4      # head-adaptive budgets, not a constant
        for r in range(2):
            np.testing.assert_array_equal(res[r][t][0], want)                   # every rank holds all heads' counts
            hq = full.Hq // 2
            np.testing.assert_array_equal(res[r][t][1], ob.out()[:, r * hq:(r + 1) * hq])


def test_single_process_reduce_is_identity():
    from paper_2606_28831_b200 import sharding
    assert sharding.reduce_run(1.5, 2.5, 100.0, "cpu") == (1.5, 2.5, 100.0)
