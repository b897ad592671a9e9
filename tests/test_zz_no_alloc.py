"""bh_domain_box_static: the S0 domain box for callers that cannot allocate device memory.

Everything else in this library works inside a workspace the caller allocates.  A caller that cannot allocate -- its host
application's allocator already owns the whole card, it runs under a fixed device-memory budget where a cudaMalloc in the
middle of a run may fail, or it sits in a loop that cannot take the device-wide stall of cudaMalloc / cudaFree -- gets this
one entry point, whose intermediates live in an array built into the library (256 KiB per GPU, n <= 2^25 particles).

The tests compare it with the path that already exists (bh_tree_build + bh_sync_status: bh_stats.lo / hi / domain_exp and the
deferred status), bit for bit, which is the bar tests/test_gpu_parity.py sets for S0.  Calls come in pairs on purpose: the
built-in array is shared and keeps the previous call's contents, so a second call on different particles is what shows that
nothing stale leaks into a result.

This file is named to be collected last: under `pytest -x` a failure here cannot hide any other test.
"""
import ctypes as C

import numpy as np
import pytest

import bh_inputs


def _existing_path(pm, front_mode=0):
    """(lo, hi, domain_exp, status) as bh_tree_build reports them for the same particles."""
    from paper_1106_1900_b200 import BarnesHut
    bh = BarnesHut(pm.shape[0], front_mode=front_mode)
    bh.set_particles(pm)
    bh.tree_build()
    st = bh.sync_status(check=False)
    out = (np.array(st.lo, np.float32), np.array(st.hi, np.float32), int(st.domain_exp), int(st.status))
    bh.close()
    return out


def _same_bits(a, b):
    return np.array_equal(np.asarray(a, np.float32).view(np.uint32), np.asarray(b, np.float32).view(np.uint32))


def _check(box, ref):
    lo, hi, e, status = ref
    assert _same_bits(np.array(box.lo, np.float32), lo), (list(box.lo), lo)
    assert _same_bits(np.array(box.hi, np.float32), hi), (list(box.hi), hi)
    assert box.domain_exp == e and box.status == status, (box.domain_exp, e, box.status, status)


def test_size_beyond_the_built_in_scratch_is_refused():
    """Host-side check only (runs without a GPU): n above the limit is refused before any pointer is looked at."""
    import __graft_entry__ as g
    g.build()
    from paper_1106_1900_b200 import domain_box_static_max_n, load_library
    lib = load_library()
    mx = domain_box_static_max_n()
    assert mx == 1 << 25
    fake = C.c_void_p(256)                       # never dereferenced: the size check comes first
    assert lib.bh_domain_box_static(fake, mx + 1, fake, None) == -7
    assert lib.bh_domain_box_static(fake, 1 << 40, fake, None) == -7
    assert b"BH_DOMAIN_STATIC_MAX_N" in lib.bh_status_string(-7)
    assert lib.bh_domain_box_static(None, 16, fake, None) == -1 and lib.bh_domain_box_static(fake, 0, fake, None) == -1


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_existing_path():
    """Call 1 on a wide set (25 blocks, ragged tail), call 2 on a narrow, shifted set (2 blocks) through the same built-in
    array, then call 1's input again: each result equals bh_tree_build's, so nothing of an earlier call survives in it."""
    import torch
    from paper_1106_1900_b200 import decode_domain_box, domain_box_static
    wide, _, _ = bh_inputs.make("c1", n=100_003, seed=5)
    narrow, _, _ = bh_inputs.make("c1", n=4097, seed=6)
    narrow = narrow.copy()
    narrow[:, :3] = narrow[:, :3] * np.float32(1e-3) + np.array([3.0, -2.0, 0.5], np.float32)   # strictly inside the wide box
    d_wide, d_narrow = torch.from_numpy(wide).cuda(), torch.from_numpy(narrow).cuda()
    outs = [torch.full((8,), -1, dtype=torch.int32, device="cuda") for _ in range(3)]           # the caller's outputs
    domain_box_static(d_wide, outs[0])           # first call on this device: also the set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    domain_box_static(d_narrow, outs[1])         # back to back on one stream, no synchronisation between them
    domain_box_static(d_wide, outs[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before          # the library took no device memory for them
    ref_wide, ref_narrow = _existing_path(wide), _existing_path(narrow)
    assert ref_wide[3] == 0 and ref_narrow[3] == 0
    assert np.all(ref_narrow[0] > ref_wide[0]) and np.all(ref_narrow[1] < ref_wide[1])          # a stale partial would show
    _check(decode_domain_box(outs[0]), ref_wide)
    _check(decode_domain_box(outs[1]), ref_narrow)
    _check(decode_domain_box(outs[2]), ref_wide)
    # the other front end of the existing path (k_bbox + k_domain, one launch per stage) says the same
    _check(decode_domain_box(outs[1]), _existing_path(narrow, front_mode=1))


@pytest.mark.gpu
@pytest.mark.parametrize("n", [1, 2, 4096, 4097, 65_536, 1_000_003])
def test_sizes_around_the_block_tile(n):
    """One particle, one full block, one particle more, many blocks: twice each, against bh_tree_build."""
    import torch
    from paper_1106_1900_b200 import decode_domain_box, domain_box_static
    pm, _, _ = bh_inputs.make("c2", n=n, seed=41)
    d = torch.from_numpy(pm).cuda()
    a = torch.zeros(8, dtype=torch.int32, device="cuda")
    b = torch.zeros(8, dtype=torch.int32, device="cuda")
    domain_box_static(d, a)
    domain_box_static(d, b)
    ref = _existing_path(pm)
    _check(decode_domain_box(a), ref)
    _check(decode_domain_box(b), ref)


@pytest.mark.gpu
def test_bad_input_is_reported_and_does_not_stick():
    """A NaN coordinate / a non-positive mass gives BH_ERR_NONFINITE like the deferred status of bh_tree_build, and the call
    after it on clean particles is clean again."""
    import torch
    from paper_1106_1900_b200 import BhError, decode_domain_box, domain_box_static
    pm, _, _ = bh_inputs.make("c1", n=20_000, seed=9)
    for row, col, val in [(12_345, 1, np.nan), (19_999, 3, 0.0), (0, 0, np.inf)]:
        bad = pm.copy()
        bad[row, col] = val
        o_bad = torch.zeros(8, dtype=torch.int32, device="cuda")
        o_ok = torch.zeros(8, dtype=torch.int32, device="cuda")
        domain_box_static(torch.from_numpy(bad).cuda(), o_bad)
        domain_box_static(torch.from_numpy(pm).cuda(), o_ok)
        got = decode_domain_box(o_bad)
        assert got.status == -5 and _existing_path(bad)[3] == -5
        _check(decode_domain_box(o_ok), _existing_path(pm))
    with pytest.raises(BhError):                                   # host memory is refused, not dereferenced
        load = torch.zeros(8, dtype=torch.int32, device="cuda")
        from paper_1106_1900_b200 import load_library
        rc = load_library().bh_domain_box_static(C.c_void_p(pm.ctypes.data), pm.shape[0], C.c_void_p(load.data_ptr()), None)
        if rc != 0:
            raise BhError(rc, "host pointer")
