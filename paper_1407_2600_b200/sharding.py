"""Host-side bookkeeping of sink-group sharding over ranks ("cut the sorted list into N_p pieces
weighted by work").  The cut itself is made on the device by dsk_accel_shard (walk.cu); `cut_points` states the same rule in numpy for the
tests and for planning, `assemble` is the exchange step: every rank zero-fills, fills its own shard, and a sum-reduction over the ranks
puts the full result on all of them.  No force arithmetic lives here."""
import numpy as np


def group_work(count, m2p_len, p2p_src, flop_m2p, flop_p2p=19):
    """w_g = ((n_sinks (len_M2P flop_M2P + src_P2P flop_P2P)) >> 10) + 1, the weight dsk_accel_shard gives group g"""
    v = np.asarray(count, np.uint64) * (np.asarray(m2p_len, np.uint64) * np.uint64(flop_m2p) + np.asarray(p2p_src, np.uint64) * np.uint64(flop_p2p))
    return (v >> np.uint64(10)) + np.uint64(1)


def cut_points(weights, nranks):
    """cut[k] = first group whose exclusive prefix sum of the weights is >= k total / nranks (cut[nranks] = number of groups):
    rank r takes groups [cut[r], cut[r+1])."""
    w = np.asarray(weights, dtype=np.uint64)
    off = np.concatenate([[0], np.cumsum(w, dtype=np.uint64)]).astype(object)       # exact integers
    total = int(off[-1])
    return [_first_at_least(off, total * k // nranks, len(w), k == nranks) for k in range(nranks + 1)]


def _first_at_least(off, target, ng, last):
    if last:
        return ng
    lo, hi = 0, ng
    while lo < hi:
        mid = (lo + hi) // 2
        if off[mid] < target:
            lo = mid + 1
        else:
            hi = mid
    return lo


def assemble(dist, acc):
    """sum-reduction of the zero-filled, shard-filled result over the ranks (NCCL on GPUs, gloo in the CPU tests)"""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(acc, op=dist.ReduceOp.SUM)
    return acc
