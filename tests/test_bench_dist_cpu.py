"""Host-side logic of the multi-rank bench path on CPU: world_size 2, gloo.  The path does not shard in
this build (replicas only), so the only cross-rank logic is the aggregation: max over ranks of
the device time, sum over ranks of the units."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, units = bench.aggregate(dist, 10.0 + 5.0 * rank, 1000 * (rank + 1))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, units))


def test_aggregate_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in res:
        assert ms == 15.0 and units == 3000.0


def test_aggregate_single():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(None, 3.5, 7) == (3.5, 7.0)


def test_accounting_matches_kernel_op_counts():
    """flop accounting (roofline numerator) against the op counts in the SASS of k_m2p<P, pot> as built:
    one FFMA2 / FMUL2 / FADD2 per counted ffma / fmul / fadd (the body is straight-line, inlined once)."""
    import shutil
    import subprocess
    from paper_1407_2600_b200 import accounting, build
    assert accounting.m2p_ops(4, pot=True) == (103, 43, 3)
    assert accounting.p2p_flops(pot=True) == 19
    assert accounting.m2p_flops(4) > accounting.m2p_flops(2) and accounting.m2p_flops(8) > accounting.m2p_flops(6)
    assert abs(accounting.fp32_peak_flops(148, 1965.0) - 74.45e12) < 0.1e12
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    obj = os.path.join(os.path.dirname(build.LIB), "build", "m2p.o")
    if not (os.path.exists(cuobjdump) and os.path.exists(obj)):
        pytest.skip("cuobjdump or build/m2p.o missing: the SASS half of this test did not run")
    sass = subprocess.run([cuobjdump, "-sass", obj], capture_output=True, text=True).stdout
    for mode, dip in ((0, False), (2, True)):               # isolated rows; periodic rows with the dipole block (background subtraction)
        for p in (2, 3, 4, 5, 6):                           # the packed (f32x2) instantiations: <P, pot, MODE>
            fn = [b for b in sass.split("Function : ")[1:] if b.startswith(f"_Z5k_m2pILi{p}ELb1ELi{mode}EE")]
            assert len(fn) == 1
            ffma, fmul, fadd = accounting.m2p_ops(p, pot=True, dip=dip)
            assert fn[0].count(" FFMA2 ") == ffma, (p, mode, fn[0].count(" FFMA2 "), ffma)
            assert fn[0].count(" FMUL2 ") == fmul, (p, mode, fn[0].count(" FMUL2 "), fmul)
            # + the packed TwoSum fold of the tile sums into the two-float accumulators: 6 adds x 4 components
            # (a few more where the compiler packs scalar pairs itself, e.g. the sinks' offsets from the group centre)
            assert fadd + 24 <= fn[0].count(" FADD2 ") <= fadd + 32, (p, mode, fn[0].count(" FADD2 "), fadd)
    assert accounting.m2p_flops(4, dip=True) - accounting.m2p_flops(4) == 2 * 6 - 1


def _shard_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import numpy as np
    import torch.distributed as dist
    from paper_1407_2600_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(5)                      # the same "tree" on every rank
    ng = 5000
    count = rng.integers(1, 193, ng)
    first = np.concatenate([[0], np.cumsum(count)[:-1]])
    n = int(count.sum())
    w = sharding.group_work(count, rng.integers(500, 4000, ng), rng.integers(1000, 9000, ng), 252)
    cut = sharding.cut_points(w, world)
    full = torch.from_numpy(rng.standard_normal((n, 3)).astype(np.float32))      # what a full evaluation would give
    order = torch.from_numpy(rng.permutation(n))                                  # sorted rank -> caller index
    acc = torch.zeros((n, 3))
    r_lo = int(first[cut[rank]]) if cut[rank] < ng else n
    r_hi = int(first[cut[rank + 1]]) if cut[rank + 1] < ng else n
    mine = order[r_lo:r_hi]
    acc[mine] = full[mine]                              # this rank's shard, caller order; the rest stays zero
    sharding.assemble(dist, acc)
    ok = bool(torch.equal(acc, full))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ok, cut, float(w[cut[rank]:cut[rank + 1]].sum()) / float(w.sum())))


def test_shard_assembly_world2_gloo():
    """N > 1 path of bench.py --shard on CPU: both ranks derive the same cut from the same tree, fill disjoint shards that
    cover every particle once, and the sum-reduction leaves the full result on both."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(ok for _, ok, _, _ in res)
    assert res[0][2] == res[1][2] and res[0][2][0] == 0 and res[0][2][-1] == 5000
    assert abs(res[0][3] - 0.5) < 0.01 and abs(res[1][3] - 0.5) < 0.01


def test_shard_cut_balances_clustered_weights():
    """the cut rule on weights shaped like configs[3]'s (a few heavy groups next to halos among many light ones): every group
    in exactly one shard, shards balanced to 5 % for 2, 4 and 8 ranks"""
    import numpy as np
    from paper_1407_2600_b200 import sharding
    rng = np.random.default_rng(1)
    ng = 400000
    w = sharding.group_work(rng.integers(1, 193, ng), (2000 * rng.lognormal(0.0, 0.5, ng)).astype(np.int64),
                            (4000 * rng.lognormal(0.0, 0.8, ng)).astype(np.int64), 682)
    for nr in (1, 2, 4, 8, 7):
        cut = sharding.cut_points(w, nr)
        assert cut[0] == 0 and cut[-1] == ng and all(cut[i] <= cut[i + 1] for i in range(nr))
        share = np.array([float(w[cut[i]:cut[i + 1]].sum()) for i in range(nr)]) / float(w.sum())
        assert np.max(np.abs(share * nr - 1.0)) < 0.05, (nr, share)
    assert sharding.cut_points([5], 3) == [0, 0, 1, 1] or sharding.cut_points([5], 3)[-1] == 1
