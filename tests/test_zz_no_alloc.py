"""The allocation-free entry point (hot_sort_keys_noalloc: the radix sort of hot_build with its scratch in a fixed device
array of the library) against the existing path (hot_build -> hot_export_keys), bit-exact, on two calls in a row.
Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_1310_4502_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _existing_path(hot, w):
    """Sorted keys and permutation of hot_build, and the unsorted keys they imply (key[perm[i]] = key_sorted[i])."""
    import torch

    hot.hot_set_params(16, 64)
    hot.hot_build(torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda(), w.lo, w.size, w.periodic)
    skey, perm = hot.hot_export_keys()
    key = np.empty_like(skey)
    key[perm] = skey
    return key, skey, perm


def _noalloc(hot, key):
    import torch

    n = key.shape[0]
    dk = torch.from_numpy(key.view(np.int64).copy()).cuda()
    dp = torch.empty(n, dtype=torch.int32, device="cuda")
    kw = torch.empty(n, dtype=torch.int64, device="cuda")
    iw = torch.empty(n, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    hot.hot_sort_keys_noalloc(dk, dp, kw, iw)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    return dk.cpu().numpy().view(np.uint64), dp.cpu().numpy().view(np.uint32), free0 - free1


def test_noalloc_sort_matches_hot_build_on_two_calls_in_a_row(hot):
    from paper_1310_4502_b200 import HotError

    # two different problems, the larger first: the second call finds the first one's counts, tickets and look-back
    # words in the shared scratch and must clear them; duplicates (ties keep ascending input position) in both
    w1 = W.config(2, 18)
    w1.pos[1000:3000] = w1.pos[0:2000]
    w2 = W.config(1, 15)
    w2.pos[5:2000] = w2.pos[4]
    ref = [_existing_path(hot, w) for w in (w1, w2)]
    hot.hot_free()  # the new entry point needs nothing of the library's context
    _noalloc(hot, ref[1][0][:4097].copy())  # first use on this device: module load, symbol address
    leaks = []
    for key, skey, perm in ref:  # the two calls in a row
        gk, gp, leak = _noalloc(hot, key)
        assert np.array_equal(gk, skey), "sorted keys"
        assert np.array_equal(gp, perm), "stable permutation"
        leaks.append(leak)
    assert max(leaks) <= 0, f"device memory in use grew across a call: {leaks}"
    # sizes at and beyond the fixed scratch
    import torch

    nmax = 1 << 22
    rng = np.random.default_rng(22)
    big = rng.integers(0, 1 << 63, nmax, dtype=np.uint64) | np.uint64(1 << 63)
    gk, gp, _ = _noalloc(hot, big)
    assert np.array_equal(gk, big[gp]) and (gk[1:] >= gk[:-1]).all()
    too = torch.empty(nmax + 1, dtype=torch.int64, device="cuda")
    idx = torch.empty(nmax + 1, dtype=torch.int32, device="cuda")
    with pytest.raises(HotError) as e:
        hot.hot_sort_keys_noalloc(too, idx, too.clone(), idx.clone())
    assert e.value.code == -1 and "2^22" in str(e.value)
    # and the small call still works after the rejected one
    gk, gp, _ = _noalloc(hot, ref[1][0])
    assert np.array_equal(gk, ref[1][1]) and np.array_equal(gp, ref[1][2])
