"""dsk_sort_keys_noalloc: the key + sort steps with their scratch in a fixed device array of the library (no cudaMalloc, no
workspace) against the existing path (dsk_build_tree + dsk_get_keys), bit for bit, on calls in a row.
Collected last on purpose (the suite runs with pytest -x)."""
import gc

import numpy as np
import pytest

from paper_1407_2600_b200 import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dsk():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1407_2600_b200 import dsk as m
    m.load_library()          # fails loudly if libdsk.so is missing: no CPU fallback
    return m


def _existing(dsk, pos_d, mass_d, box, periodic):
    d = dsk.Dsk(pos_d.shape[0], box, periodic, 1e-3, 0.5, 2)
    d.build_tree(pos_d, mass_d)
    k, o = d.get_keys()
    k, o = k.clone(), o.clone()
    d.close()
    return k, o


def test_sort_keys_noalloc_equals_existing_path_on_calls_in_a_row(dsk):
    rng = np.random.default_rng(11)
    cases = [
        (workloads.make(2, 1 / 4)[0], 1.0, False),                                  # clustered Plummer sphere, 2^18: 128 tiles
        (workloads.uniform_box(5003)[0], 1.0, False),                               # ragged, smaller than the call before it
        ((rng.random((70001, 3), dtype=np.float32) * 3.0 - 1.0), 1.0, True),        # periodic wrap, ragged tail
        (np.tile(np.array([[0.3, 0.4, 0.5]], np.float32), (3000, 1)), 1.0, False),  # all keys equal: order = identity
        (workloads.make(2, 1 / 4)[0], 1.0, False),                                  # the first input again
    ]
    first = None
    for i, (pos, box, periodic) in enumerate(cases):
        n = len(pos)
        pos_d = torch.from_numpy(np.ascontiguousarray(pos, dtype=np.float32)).cuda()
        mass_d = torch.full((n,), 1.0 / n, dtype=torch.float32, device="cuda")
        k_ref, o_ref = _existing(dsk, pos_d, mass_d, box, periodic)
        keys = torch.full((n,), -1, dtype=torch.int64, device="cuda")
        order = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        for rep in range(2):                                                        # two calls in a row on the same input
            gc.collect()                                                            # tensors of earlier tests die here, not inside the bracket
            torch.cuda.synchronize()
            free0 = torch.cuda.mem_get_info()[0]
            alloc0 = torch.cuda.memory_allocated()
            dsk.sort_keys_noalloc(pos_d, box, periodic, keys, order)
            torch.cuda.synchronize()
            if i > 0 or rep > 0:                                                    # the first launch loads the kernels
                assert torch.cuda.memory_allocated() <= alloc0                     # nothing new from torch's allocator either
                assert free0 - torch.cuda.mem_get_info()[0] < (1 << 20)
            assert torch.equal(keys, k_ref), (i, rep)
            assert torch.equal(order, o_ref), (i, rep)
            keys.fill_(-1); order.fill_(-1)
        if i == 0:
            first = (k_ref, o_ref)
        if i == len(cases) - 1:
            assert torch.equal(k_ref, first[0]) and torch.equal(o_ref, first[1])
        if i == 3:
            assert torch.equal(o_ref, torch.arange(n, dtype=torch.int32, device="cuda"))


def test_sort_keys_noalloc_on_a_side_stream_and_at_the_maximum(dsk):
    n = dsk.NOALLOC_NMAX
    pos, mass = workloads.make(2)                                                   # configs[1]: N = 2^20 = the maximum
    assert len(pos) == n
    pos_d, mass_d = torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda()
    k_ref, o_ref = _existing(dsk, pos_d, mass_d, 1.0, False)
    keys = torch.empty(n, dtype=torch.int64, device="cuda")
    order = torch.empty(n, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        for _ in range(2):
            dsk.sort_keys_noalloc(pos_d, 1.0, False, keys, order)
            assert torch.equal(keys, k_ref) and torch.equal(order, o_ref)
    torch.cuda.current_stream().wait_stream(s)


def test_sort_keys_noalloc_rejects(dsk):
    n = dsk.NOALLOC_NMAX + 1
    pos = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    keys = torch.full((n,), 7, dtype=torch.int64, device="cuda")
    order = torch.full((n,), 7, dtype=torch.int32, device="cuda")
    with pytest.raises(dsk.DskError) as e:
        dsk.sort_keys_noalloc(pos, 1.0, False, keys, order)
    assert e.value.code == -9 and "maximum" in str(e.value)
    assert bool((keys == 7).all()) and bool((order == 7).all())                     # nothing was launched
    # the errors of the existing path: a position outside an isolated box, a NaN
    p = torch.rand((1000, 3), dtype=torch.float32, device="cuda")
    k, o = keys[:1000].contiguous(), order[:1000].contiguous()
    p[17, 1] = 1.5
    with pytest.raises(dsk.DskError) as e:
        dsk.sort_keys_noalloc(p, 1.0, False, k, o)
    assert e.value.code == -4
    dsk.sort_keys_noalloc(p, 1.0, True, k, o)                                       # periodic: wrapped, fine; status was cleared
    p[17, 1] = float("nan")
    with pytest.raises(dsk.DskError) as e:
        dsk.sort_keys_noalloc(p, 1.0, True, k, o)
    assert e.value.code == -5
    p[17, 1] = 0.5
    dsk.sort_keys_noalloc(p, 1.0, False, k, o)                                      # and the array is usable after an error
    kk = k.cpu().numpy().view(np.uint64)
    assert np.all(kk[1:] >= kk[:-1]) and np.array_equal(np.sort(o.cpu().numpy()), np.arange(1000))
