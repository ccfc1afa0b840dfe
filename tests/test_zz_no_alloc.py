"""-m gpu: mcrt_get_cell_temperature_noalloc against mcrt_get_cell_temperature.

Why the entry point exists: reading temperatures to the host needs a device array for the
conversion kernel's output, and the ordinary getter cudaMallocs it on first use.  A caller whose
device memory is already owned in full by another pool or capped by a quota, a caller that runs
beside a thread recording a CUDA graph, or a loop that cannot take an allocation's stall cannot
have that happen between batches.  The no-alloc getter writes into a fixed 4 MiB array that is
part of libmcrt.so instead (up to mcrt.NOALLOC_MAX_SLOTS leaf slots) and allocates nothing.

What is checked: the two getters run the same kernels on the same stored rows, so their outputs
must be equal bit for bit (stricter than the 1e-3 the parity tests allow against the oracle) --
on two calls in a row, with the temperatures changed in between and the no-alloc call made
first the second time, so an answer left in the shared array by the previous call would be
caught; on a second, smaller, two-level grid right after the larger one (the array still holds
the first grid's values); and that a grid beyond the limit is refused with a message that names
the limit.  This file sorts last on purpose: `pytest -x` stops at the first failure, and a
failure here must not hide the parity tests.  It makes no assumption about what ran before it
in the process (the array may be fresh or may hold an earlier call's output)."""
import numpy as np
import pytest

from paper_1201_3588_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "-m gpu tests need a CUDA device"
    from paper_1201_3588_b200 import build, mcrt
    build.build_library()
    mcrt.lib()
    return mcrt


def test_noalloc_temperatures_equal_the_ordinary_getter_twice_in_a_row(M):
    wl = W.c0()
    ctx = M.from_workload(wl)
    batches = list(wl.batches(3 * wl.batch, wl.batch))
    ctx.run_batch(wl.seed, *batches[0])
    T_ref1 = ctx.get_cell_temperature()
    T_na1 = ctx.get_cell_temperature_noalloc()
    assert T_na1.dtype == np.float32 and T_na1.shape == (ctx.slots,)
    assert np.array_equal(T_na1, T_ref1)
    assert (T_ref1 > T_ref1.min()).sum() > 100          # a real temperature field, not the floor

    ctx.run_batch(wl.seed, *batches[1])
    T_na2 = ctx.get_cell_temperature_noalloc()            # first this time: the array holds call 1's answer
    T_ref2 = ctx.get_cell_temperature()
    assert np.array_equal(T_na2, T_ref2)
    assert not np.array_equal(T_na2, T_na1)               # the batch moved the temperatures

    # into the caller's own buffer, a third call in a row
    buf = np.full(ctx.slots, -1.0, dtype=np.float32)
    assert ctx.get_cell_temperature_noalloc(out=buf) is buf
    assert np.array_equal(buf, T_ref2)

    # a smaller, two-level grid straight after (root cells and sub-cells take different kernels)
    wl2 = W.c2(n_root=8, n_packets=20000, batch=20000)
    ctx2 = M.run_workload(wl2)
    assert ctx.slots > ctx2.slots > 8 ** 3
    T2 = ctx2.get_cell_temperature_noalloc()
    assert np.array_equal(T2, ctx2.get_cell_temperature())
    assert (T2 > T2.min()).sum() > 10
    # ... and the first context again: nothing of ctx2's read-out leaks into it
    assert np.array_equal(ctx.get_cell_temperature_noalloc(), T_ref2)


def test_noalloc_refuses_grids_beyond_its_fixed_array(M):
    wl = W.c1(n_root=104, n_packets=10, batch=10)         # 104^3 = 1 124 864 leaf slots > 2^20
    ctx = M.from_workload(wl)
    assert ctx.slots > M.NOALLOC_MAX_SLOTS
    with pytest.raises(M.McrtError, match="MCRT_NOALLOC_MAX_SLOTS = 1048576"):
        ctx.get_cell_temperature_noalloc()
    assert ctx.get_cell_temperature().shape == (ctx.slots,)   # the ordinary getter still serves it
