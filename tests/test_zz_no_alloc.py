"""pvg_sort_pairs_static (include/pvg.h): the onesweep sort with its scratch in a static device array of the library,
for callers that may not allocate. Collected last on purpose (the suite runs with pytest -x).

The results are integers: the bar is bit-equality with pvg_sort_pairs, the existing path, on the same inputs."""
import os
import subprocess
import sys

import numpy as np
import pytest

import paper_2311_18561_b200 as pvg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _pairs(n, seed, bits=64):
    import torch
    rng = np.random.default_rng(seed)
    k = rng.integers(0, 2 ** 63, size=n, dtype=np.int64)
    if bits < 64:
        k &= np.int64((1 << bits) - 1)
    # duplicates, so that stability shows: a tenth of the keys repeat an earlier one
    if n > 10:
        k[rng.integers(0, n, size=n // 10)] = k[rng.integers(0, n, size=n // 10)]
    return torch.from_numpy(k).cuda(), torch.arange(n, dtype=torch.int32, device="cuda")


@pytest.mark.gpu
def test_static_sort_matches_sort_pairs_on_two_calls_in_a_row():
    import torch
    assert pvg.sort_pairs_static_max_n() == 1 << 20
    # two calls back to back on one stream, no synchronisation between them: the second starts from the scratch the
    # first one left (other tile count, other passes, other bit range), then a third at the maximum size
    cases = [(300_003, 0, 64, 1), (70_001, 32, 46, 2), (1 << 20, 3, 40, 3), (5, 0, 64, 4), (0, 0, 64, 5), (4096, 17, 17, 6)]
    ins, outs = [], []
    for n, b0, b1, seed in cases:
        k, v = _pairs(n, seed)
        ins.append((k.clone(), v.clone()))
        ko, vo = torch.empty_like(k), torch.empty_like(v)
        pvg.sort_pairs_static(k, v, ko, vo, b0, b1)
        outs.append((ko, vo))
    torch.cuda.synchronize()
    for (n, b0, b1, seed), (k, v), (ko, vo) in zip(cases, ins, outs):
        rk, rv = pvg.sort_pairs(k.clone(), v.clone(), b0, b1)
        assert torch.equal(ko, rk) and torch.equal(vo, rv), (n, b0, b1)
        if b1 > b0 and n:
            # and against the definition: a stable sort on the bit field
            field = (k.cpu().numpy().view(np.uint64) >> np.uint64(b0)) & np.uint64((1 << (b1 - b0)) - 1 if b1 - b0 < 64 else 2 ** 64 - 1)
            order = np.argsort(field, kind="stable")
            assert np.array_equal(vo.cpu().numpy(), order.astype(np.int32)), (n, b0, b1)


@pytest.mark.gpu
def test_static_sort_rejects_sizes_beyond_its_scratch():
    import torch
    n = pvg.sort_pairs_static_max_n() + 1
    k = torch.zeros(n, dtype=torch.int64, device="cuda")
    v = torch.zeros(n, dtype=torch.int32, device="cuda")
    ko, vo = torch.full_like(k, -1), torch.full_like(v, -1)
    with pytest.raises(pvg.PvgError) as e:
        pvg.sort_pairs_static(k, v, ko, vo)
    assert e.value.code == -9 and "exceeds the static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert int(ko[0]) == -1 and int(vo[-1]) == -1   # nothing was enqueued
    # the library is still usable
    k, v = _pairs(1000, 9)
    ko, vo = torch.empty_like(k), torch.empty_like(v)
    pvg.sort_pairs_static(k.clone(), v.clone(), ko, vo)
    rk, rv = pvg.sort_pairs(k, v)
    assert torch.equal(ko, rk) and torch.equal(vo, rv)


@pytest.mark.gpu
def test_static_sort_allocates_nothing():
    """Through counting allocator hooks (pvg_set_allocator), in a process of its own: pvg_sort_pairs asks the hooks for
    its scratch, the static entry point never does -- and the device's free memory does not move."""
    code = r'''
import sys
sys.path.insert(0, %r)
import ctypes as C
import numpy as np, torch
import paper_2311_18561_b200 as pvg
L = pvg.load_library()
count = {"alloc": 0, "free": 0}
def _alloc(nbytes, stream, _user):
    count["alloc"] += 1
    return torch.cuda.caching_allocator_alloc(int(nbytes))
def _free(ptr, _user):
    count["free"] += 1
    torch.cuda.caching_allocator_delete(ptr)
a, f = pvg.ALLOC_FN(_alloc), pvg.FREE_FN(_free)
assert L.pvg_set_allocator(C.cast(a, C.c_void_p), C.cast(f, C.c_void_p), None) == 0
n = 200_000
k = torch.randint(0, 2 ** 62, (n,), dtype=torch.int64, device="cuda")
v = torch.arange(n, dtype=torch.int32, device="cuda")
rk, rv = pvg.sort_pairs(k.clone(), v.clone())
assert count["alloc"] >= 3 and count["free"] == count["alloc"], count   # the hooks do see the existing path
ko, vo = torch.empty_like(k), torch.empty_like(v)
k2, v2 = k.clone(), v.clone()
torch.cuda.synchronize()
before = dict(count)
free0 = torch.cuda.mem_get_info()[0]
for rep in range(2):
    k2.copy_(k); v2.copy_(v)
    pvg.sort_pairs_static(k2, v2, ko, vo)
torch.cuda.synchronize()
assert count == before, (before, count)
assert torch.cuda.mem_get_info()[0] == free0
assert torch.equal(ko, rk) and torch.equal(vo, rv)
print("ok")
''' % ROOT
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and r.stdout.strip().endswith("ok"), r.stdout + r.stderr
