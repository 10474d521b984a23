"""-m gpu, collected last: tpcStartHitsNoAlloc (include/tpc_abi.h, csrc/tpc_noalloc.cu), the entry point that allocates
nothing -- its scratch is a static device array of the library -- against the existing path (the start_hits output of
tpcRun, itself bit-exact against the oracle in test_gpu_parity.py), bit for bit, on calls in a row that share the scratch.

Integer work: the tolerance is zero, as everywhere in this suite.  The file is named to be collected after every other
test (the suite runs with pytest -x) and passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

from paper_1910_12214_b200 import datagen

pytestmark = pytest.mark.gpu


def _existing_path(ev):
    """link_up, link_dn (device tensors, global input indices) and start_hits of the existing path: one tpcRun."""
    from paper_1910_12214_b200 import tpc
    trk = tpc.TpcTracker.from_event(ev)
    off, y, z = trk.upload(ev)
    res = trk.run(off, y, z, stages=True)
    assert res.status.status == 0
    up, dn = res.stages["link_up"].clone(), res.stages["link_dn"].clone()
    want = res.stages["start_hits"].cpu().numpy().view(np.uint32).copy()
    assert len(want) == res.status.n_start_hits
    trk.close()
    return up, dn, want


def _no_alloc(up, dn, cap, out=None, cnt=None, stream=None):
    """One tpcStartHitsNoAlloc on device tensors; returns (count, list) after synchronising."""
    import torch
    from paper_1910_12214_b200 import tpc
    n = int(up.shape[0])
    dev = up.device
    if out is None:
        out = torch.full((max(cap, 1),), -7, dtype=torch.int32, device=dev)
    if cnt is None:
        cnt = torch.full((1,), -7, dtype=torch.int64, device=dev)
    s = stream if stream is not None else torch.cuda.current_stream(dev)
    tpc.tpcStartHitsNoAlloc(dev.index or 0, n, up.data_ptr() if n else 0, dn.data_ptr() if n else 0,
                            out.data_ptr() if cap else 0, cap, cnt.data_ptr(), s.cuda_stream)
    s.synchronize()
    return int(cnt.item()), out.cpu().numpy().view(np.uint32)


def test_two_calls_in_a_row_equal_the_existing_path():
    """A large event, then a small one (its tiles are a prefix of the stale scratch of the first call), then the large
    one again: every list equals tpcRun's start_hits, and the calls allocate no device memory."""
    import torch
    from paper_1910_12214_b200 import tpc
    tpc.tpcNoAllocSetup(0)
    tpc.tpcNoAllocSetup(0)                                                   # idempotent
    big = _existing_path(datagen.make_event(1, scale=0.5))                   # 732 176 clusters: 358 tiles of the scratch
    small = _existing_path(datagen.make_event(1, scale=0.05))                #  72 524 clusters:  36 tiles
    assert len(big[2]) > 4 * 2048 > len(small[2]) > 0 and big[0].shape[0] > 8 * small[0].shape[0]
    bufs = {}
    for name, (up, dn, want) in (("big", big), ("small", small)):
        bufs[name] = (torch.full((len(want) + 5,), -7, dtype=torch.int32, device=up.device),
                      torch.full((1,), -7, dtype=torch.int64, device=up.device))
    _no_alloc(*big[:2], len(big[2]) + 5, *bufs["big"])                       # first call: lazy module load happens here
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for name, (up, dn, want) in (("big", big), ("small", small), ("big", big), ("small", small)):
        out, cnt = bufs[name]
        out.fill_(-7)
        cnt.fill_(-7)
        n, got = _no_alloc(up, dn, len(want) + 5, out, cnt)
        assert n == len(want), name
        assert np.array_equal(got[:n], want), name
        assert np.all(got[n:].view(np.int32) == -7), name                    # nothing written beyond the list
        # restated apart from both paths: ascending indices of the clusters with an up link and no down link
        u, d = up.cpu().numpy(), dn.cpu().numpy()
        assert np.array_equal(got[:n], np.nonzero((d == -1) & (u != -1))[0].astype(np.uint32)), name
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                             # no device allocation by any of the calls


def test_truncation_empty_input_unaligned_pointers_and_the_limit():
    import torch
    from paper_1910_12214_b200 import tpc
    up, dn, want = _existing_path(datagen.make_event(3, scale=0.01))
    assert len(want) > 100
    # cap smaller than the list: the count is the required capacity, only cap entries are written
    out = torch.full((60,), -7, dtype=torch.int32, device=up.device)
    cnt = torch.zeros(1, dtype=torch.int64, device=up.device)
    n, got = _no_alloc(up, dn, 50, out, cnt)
    assert n == len(want) and np.array_equal(got[:50], want[:50]) and np.all(got[50:].view(np.int32) == -7)
    # cap 0 with no output array: the count alone
    n, _ = _no_alloc(up, dn, 0)
    assert n == len(want)
    # no clusters: count 0 (and the stale tile counts of the call before are not read)
    n, _ = _no_alloc(up[:0], dn[:0], 4)
    assert n == 0
    # link arrays that start 4 bytes into a 16-byte line (the scalar load path) and end mid-tile
    u1, d1 = up[1:-3], dn[1:-3]
    assert u1.data_ptr() % 16 == 4
    n, got = _no_alloc(u1, d1, len(want))
    ref = np.nonzero((d1.cpu().numpy() == -1) & (u1.cpu().numpy() != -1))[0].astype(np.uint32)
    assert n == len(ref) and np.array_equal(got[:n], ref)
    # and the existing path's answer once more after all of that
    n, got = _no_alloc(up, dn, len(want))
    assert n == len(want) and np.array_equal(got[:n], want)
    # beyond the stated maximum: refused with its own code, nothing launched (the pointers are never touched)
    limit = tpc.tpcNoAllocMaxClusters()
    assert limit == 1 << 24
    cnt.fill_(-3)
    with pytest.raises(tpc.TpcError) as e:
        tpc.tpcStartHitsNoAlloc(0, limit + 1, up.data_ptr(), dn.data_ptr(), out.data_ptr(), 10, cnt.data_ptr(), 0)
    assert e.value.code == tpc.TPC_ERR_NOALLOC_LIMIT and "TPC_NOALLOC_MAX_CLUSTERS" in str(e.value)
    with pytest.raises(tpc.TpcError) as e:
        tpc.tpcStartHitsNoAlloc(0, 10, 0, dn.data_ptr(), out.data_ptr(), 10, cnt.data_ptr(), 0)
    assert e.value.code == tpc.TPC_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int(cnt.item()) == -3


def test_at_the_stated_maximum():
    """n_clusters == TPC_NOALLOC_MAX_CLUSTERS exactly (all 8192 tile counts of the scratch in use), synthetic links."""
    import torch
    from paper_1910_12214_b200 import tpc
    n = tpc.tpcNoAllocMaxClusters()
    g = torch.Generator(device="cuda").manual_seed(5)
    r = torch.randint(0, 8, (n,), generator=g, device="cuda", dtype=torch.int32)
    up = torch.where(r < 6, torch.arange(n, device="cuda", dtype=torch.int32), torch.full_like(r, -1))
    dn = torch.where((r & 1) == 0, torch.full_like(r, -1), torch.arange(n, device="cuda", dtype=torch.int32))
    ref = torch.nonzero((dn == -1) & (up != -1)).flatten().to(torch.int32).cpu().numpy().view(np.uint32)
    for _ in range(2):
        cnt, got = _no_alloc(up, dn, len(ref) + 1)
        assert cnt == len(ref) and np.array_equal(got[:cnt], ref)
    assert got.view(np.int32)[-1] == -7
