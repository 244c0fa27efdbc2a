"""cfgms_deinterleave_host_static — the de-interleave for callers that cannot allocate device memory.

A serving process may be unable to call cudaMalloc by the time a request finishes and its codes have to be
de-interleaved: the engine has given all free HBM to its cache pool (the allocation fails), or an allocation's
device-wide synchronisation would stall the decode streams.  The library therefore has one entry point that takes
no context and allocates nothing; its staging is a fixed 8 MiB array inside the library (CFGMS_STATIC_SCRATCH_BYTES)
that every call shares and that keeps the previous call's bytes.

What is checked: bit-equal grids (integer work: the tolerance every de-interleave test here uses) against the
existing paths (cfgms_deinterleave on device buffers, cfgms_deinterleave_host) and the oracle, on calls made back
to back so that the second one runs on an array still full of the first one's data; the size limit is enforced
with its own status and leaves the output alone.

The file is named so that pytest collects it last: a failure here cannot hide another test behind `-x`.  In a
fresh process the static call below is the first thing the library does on the device (no context exists yet);
after the rest of the suite it runs on a device that has seen everything else — both orders must pass."""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2607_02119_b200 as pkg


def _delayed(n, T, S, seed, lo=-5, hi=5000):
    g = torch.Generator().manual_seed(seed)
    return torch.randint(lo, hi, (n, T, S), generator=g, dtype=torch.int32)


@pytest.mark.gpu
def test_static_scratch_calls_in_a_row_match_the_existing_paths():
    import oracle
    import workloads
    from parity_util import DeviceWorkload

    dev = torch.device("cuda:0")
    # call 1: S = 64 needs the shared-memory opt-in the one-time set-up makes; call 2 is smaller with S % 4 != 0, so
    # it runs over call 1's leftovers on the scalar path; call 3 repeats call 1's shape with other data
    cases = [_delayed(2, 200, 64, 1), _delayed(3, 40, 9, 2), _delayed(2, 200, 64, 3), _delayed(5, 513, 16, 4)]
    got = [pkg.deinterleave_host_static(c) for c in cases]                 # back to back, nothing else in between
    # an output buffer the caller owns, pre-filled: every element must be overwritten
    mine = torch.full((3, 32, 9), -77, dtype=torch.int32)
    assert pkg.deinterleave_host_static(cases[1], grid_out=mine) is mine
    got.append(mine)
    cases.append(cases[1])

    ctx = DeviceWorkload(workloads.make_config(1), dev).ctx                # the existing paths need a context
    for delayed, g in zip(cases, got):
        n, T, S = delayed.shape
        assert g.device.type == "cpu" and g.shape == (n, T - S + 1, S)
        on_device = ctx.deinterleave(delayed.to(dev))
        torch.cuda.synchronize()
        assert torch.equal(g, on_device.cpu())                             # cfgms_deinterleave
        assert torch.equal(g, ctx.deinterleave(delayed))                   # cfgms_deinterleave_host
        assert np.array_equal(g.numpy(), oracle.deinterleave(delayed.numpy()))
    # and once more after the context's own kernels have run
    assert torch.equal(pkg.deinterleave_host_static(cases[0]), got[0])


@pytest.mark.gpu
def test_static_scratch_limit_is_enforced_and_exact():
    import oracle
    # S = 1: grid == delayed and both halves are n*T*4 bytes; 2 x 4 MiB is exactly the limit
    T_max = pkg.CFGMS_STATIC_SCRATCH_BYTES // 8
    at_limit = _delayed(1, T_max, 1, 7)
    assert torch.equal(pkg.deinterleave_host_static(at_limit), at_limit)
    over = _delayed(1, T_max + 64, 1, 8)
    out = torch.full((1, T_max + 64, 1), -3, dtype=torch.int32)
    with pytest.raises(pkg.CfgmsError) as e:
        pkg.deinterleave_host_static(over, grid_out=out)
    assert e.value.status == pkg.CFGMS_ERR_LIMIT and "scratch" in str(e.value)
    assert bool((out == -3).all())                                         # refused before anything was copied
    # the paper-shaped example of the header fits: 64 requests x 1024 steps x 16 streams
    big = _delayed(64, 1024, 16, 9, 0, 2049)
    assert np.array_equal(pkg.deinterleave_host_static(big).numpy(), oracle.deinterleave(big.numpy()))
    # a call after a refused one is unaffected
    small = _delayed(2, 9, 9, 10)
    assert np.array_equal(pkg.deinterleave_host_static(small).numpy(), oracle.deinterleave(small.numpy()))


def test_static_entry_point_validates_before_touching_a_device():
    """Runs anywhere: argument and size checks come first, and without a GPU the call fails loudly (no fallback)."""
    lib = pkg.library()
    buf = (C.c_int32 * 64)()
    f = lib.cfgms_deinterleave_host_static
    assert f(buf, 0, 8, 4, buf, None) == 0                                 # n == 0: nothing to do
    assert f(buf, 1, 3, 4, buf, None) == 1                                 # T < S
    assert f(None, 1, 8, 4, buf, None) == 1
    assert f(buf, 1, 80, 65, buf, None) == 2                               # S > 64
    assert f(buf, 1, (8 << 20) // 8 + 64, 1, buf, None) == pkg.CFGMS_ERR_LIMIT
    assert b"scratch" in lib.cfgms_strerror(pkg.CFGMS_ERR_LIMIT)
    if not torch.cuda.is_available():
        assert f(buf, 1, 8, 4, buf, None) not in (0, pkg.CFGMS_ERR_LIMIT)
