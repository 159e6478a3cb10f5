"""gm_scan_counts_static: the zone-count prefix sum for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is off limits: inside a host application whose memory pool has taken
the whole GPU and forbids allocations behind its back, or in a latency-bound loop that cannot take cudaMalloc's
device-wide synchronisation.  They cannot create a library context (gm_create / gm_prepare allocate), so the header
gives them one context-free call whose only scratch -- one partial sum per 1024 zones -- is a fixed 32 KiB array that
is part of the library itself.  Consequences checked here:

  * the result is the same, bit for bit, as the prefix sum gm_prepare forms with its own allocated scratch (integer
    work: the tolerance of every integer comparison in this suite is zero);
  * the array is shared and keeps the previous call's contents, so a second call right after the first, on an input of
    ANOTHER size (fewer tiles: most of the array is then stale), must still be right, and so must a third on the first
    input again;
  * a size beyond GM_SCAN_STATIC_MAX_ZONES is refused with a message that names the limit, and nothing is launched.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here must not hide other tests), and it
builds everything it needs itself, so it gives the same verdict run alone in a fresh process or after the whole suite.
"""
import ctypes

import numpy as np
import pytest

from paper_2602_13198_b200 import workloads as wl


def _existing_path(gm, p, prim):
    """Zone counts and their prefix sum as the ordinary, allocating path computes them (gm_create .. gm_prepare)."""
    g = gm.GPUMonty(p)
    g.set_grid(prim)
    n = g.prepare()
    counts, offsets = g.zone_counts(), g.zone_offsets()
    g.close()
    assert offsets[-1] == n and offsets[0] == 0
    return counts, offsets


@pytest.mark.gpu
def test_static_scratch_scan_equals_the_allocating_path_on_two_calls_in_a_row():
    import torch
    from paper_2602_13198_b200 import binding as gm
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    # (a) 256 x 256 zones = 256 full tiles; (b) 75 x 41 = 3 tiles + a ragged tail of 3 zones, many empty zones
    pa, prim_a = wl.config2(Ns=1e6)
    pb, prim_b = wl.config2(Ns=3e4, n1=75, n2=41)
    ca, oa = _existing_path(gm, pa, prim_a)
    cb, ob = _existing_path(gm, pb, prim_b)
    assert ca.size == 65536 and cb.size == 3075 and (cb == 0).sum() > 100
    # the caller's own buffers: inputs and outputs only, made before the calls under test
    d_ca, d_cb = torch.from_numpy(ca).cuda(), torch.from_numpy(cb).cuda()
    d_oa = torch.full((ca.size + 1,), -1, dtype=torch.int64, device="cuda")
    d_ob = torch.full((cb.size + 1,), -1, dtype=torch.int64, device="cuda")
    d_oa2 = torch.full_like(d_oa, -1)
    # three calls back to back on one stream, no synchronisation in between: large, small (stale tail in the scratch), large
    gm.scan_counts_static(d_ca, d_oa)
    gm.scan_counts_static(d_cb, d_ob)
    gm.scan_counts_static(d_ca, d_oa2)
    torch.cuda.synchronize()
    for got, want, cnt in ((d_oa, oa, ca), (d_ob, ob, cb), (d_oa2, oa, ca)):
        got = got.cpu().numpy()
        assert np.array_equal(got, want)
        # and both equal the definition, independent of either implementation
        assert np.array_equal(got, np.concatenate(([0], np.cumsum(cnt.astype(np.int64)))))
    # empty input: only the total is written
    d_o0 = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    gm.scan_counts_static(d_ca, d_o0, n_zones=0)
    assert int(d_o0.cpu()[0]) == 0


@pytest.mark.gpu
def test_static_scratch_scan_at_its_maximum_size():
    """Every tile of the built-in array in use: counts with a known sum over GM_SCAN_STATIC_MAX_ZONES zones."""
    import torch
    from paper_2602_13198_b200 import binding as gm
    torch.cuda.set_device(0)
    n = gm.SCAN_STATIC_MAX_ZONES
    g = torch.Generator(device="cuda").manual_seed(13198)
    c = torch.randint(0, 2000, (n,), dtype=torch.int32, device="cuda", generator=g)   # sum ~ 4e9: beyond int32
    out = torch.full((n + 1,), -1, dtype=torch.int64, device="cuda")
    gm.scan_counts_static(c, out)
    torch.cuda.synchronize()
    want = np.concatenate(([0], np.cumsum(c.cpu().numpy().astype(np.int64))))
    assert want[-1] > 2**31 and np.array_equal(out.cpu().numpy(), want)


def test_static_scratch_scan_refuses_sizes_beyond_its_fixed_array():
    """No GPU needed: the size is checked before the device is touched and before anything is launched."""
    from paper_2602_13198_b200 import binding as gm
    L = gm.load_library()
    dummy_in, dummy_out = (ctypes.c_int32 * 4)(), (ctypes.c_int64 * 4)()     # never dereferenced: the call is refused first
    for n in (gm.SCAN_STATIC_MAX_ZONES + 1, 2**40, -1):
        rc = L.gm_scan_counts_static(ctypes.addressof(dummy_in), n, ctypes.addressof(dummy_out), None)
        assert rc == -1, n                                                    # GM_ERR_PARAM
        msg = L.gm_last_error(None).decode()
        assert str(gm.SCAN_STATIC_MAX_ZONES) in msg and "GM_SCAN_STATIC_MAX_ZONES" in msg, msg
    assert L.gm_scan_counts_static(None, 8, ctypes.addressof(dummy_out), None) == -1
    assert "NULL" in L.gm_last_error(None).decode()


def test_static_scratch_scan_has_no_cpu_path():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2602_13198_b200 import binding as gm
    L = gm.load_library()
    dummy_in, dummy_out = (ctypes.c_int32 * 4)(), (ctypes.c_int64 * 5)()
    rc = L.gm_scan_counts_static(ctypes.addressof(dummy_in), 4, ctypes.addressof(dummy_out), None)
    assert rc == -3 and "no CPU path" in L.gm_last_error(None).decode()     # GM_ERR_CUDA
