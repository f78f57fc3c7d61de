"""u1gf_paper_count_static: the one entry point of libu1gf.so that needs no device memory from anybody.

Who it is for: code that receives its input and output device buffers from a host application and cannot get more --
a plug-in in a program that handed out all of HBM at start-up, a step in a latency-critical loop that must not sit
through the device-wide stall of a cudaMalloc/cudaFree, an embedding that may only enqueue stream work.  Such a caller
can neither bring the workspace u1gf_paper_count asks for nor use a *_host call (those allocate inside).  The scratch of
this variant is a 32 MiB `static __device__` array inside the library, good for at most 2^20 records per call.

What is checked: the count equals u1gf_paper_count's (the existing path; integer output, so bit-exact -- the bar every
integer output has in these tests) on two calls in a row that share the array, the second with fewer records than the
first so that stale keys of the first call sit behind its data; the full 2^20 records fit the array; one record more is
refused; the second call leaves the amount of free device memory where it was.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It has to pass alone in a fresh process (then its first call is the per-device set-up) and after all
other tests (then the library's device code is long loaded).
"""
import ctypes as C

import pytest


@pytest.fixture(scope="module")
def b():
    from paper_1403_0555_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def test_static_limit_is_refused_before_any_device_work(b):
    """Argument checks come first, so they can be seen on a machine without a GPU: a batch over the limit is an
    U1GF_EINVAL whose text names the limit and the call to use instead."""
    L = b.lib()
    assert b.PAPER_COUNT_STATIC_MAX_N == 1 << 20
    dummy = C.c_void_p(256)          # never dereferenced: the size check fails first
    rc = L.u1gf_paper_count_static(b.PAPER_COUNT_STATIC_MAX_N + 1, dummy, dummy, 1e8, dummy, None)
    msg = L.u1gf_last_error().decode()
    assert rc == -1 and "U1GF_PAPER_COUNT_STATIC_MAX_N = 1048576" in msg and "u1gf_paper_count " in msg
    assert L.u1gf_paper_count_static(4, dummy, dummy, 1e8, None, None) == -1        # NULL n_keys
    assert L.u1gf_paper_count_static(4, dummy, dummy, 0.0, dummy, None) == -1       # scale <= 0
    assert L.u1gf_paper_count_static(4, None, dummy, 1e8, dummy, None) == -1        # NULL input


def _records(n, seed, n_values):
    """Seeded synthetic records: F/(dV) drawn from n_values distinct levels in (0.3, 0.9) (so keys repeat, as the
    functional values of a real batch do), about one record in eight flagged as not converged."""
    import torch
    gen = torch.Generator(device="cuda")
    gen.manual_seed(seed)
    level = torch.randint(0, n_values, (n,), generator=gen, device="cuda", dtype=torch.int64)
    F = 0.3 + 0.6 * (level.to(torch.float64) + 0.5) / n_values
    status = (torch.randint(0, 8, (n,), generator=gen, device="cuda", dtype=torch.int64) == 0).to(torch.uint8)
    return F, status


@pytest.mark.gpu
def test_static_scratch_count_equals_workspace_count_on_consecutive_calls(b):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    out = torch.empty(1, dtype=torch.int64, device="cuda")       # the caller's output buffer, reused by every call

    # set-up call: n = 0 finds the array on this device and returns a zero count
    e = torch.zeros(0, dtype=torch.float64, device="cuda")
    out.fill_(-7)
    assert int(b.paper_count_static(e, torch.zeros(0, dtype=torch.uint8, device="cuda"), out=out).item()) == 0

    # two calls in a row on the shared array: a large batch, then a small one with different records
    batches = [_records(300_001, 11, 70_000), _records(4_097, 12, 900)]
    expected = [int(b.paper_count(F, st).item()) for F, st in batches]          # existing path, caller workspace
    assert 0 < expected[1] < expected[0]
    torch.cuda.synchronize()
    got = []
    for k, (F, st) in enumerate(batches):
        if k == 1:
            free_before = torch.cuda.mem_get_info()[0]
        got.append(int(b.paper_count_static(F, st, out=out).item()))            # .item() drains the stream
        assert b.last_launch_count() == 2
    assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"
    assert got == expected
    # and once more in the other order, with another scale, same stream, no synchronisation in between
    o0, o1 = torch.empty_like(out), torch.empty_like(out)
    b.paper_count_static(*batches[1], scale=1e3, out=o1)
    b.paper_count_static(*batches[0], scale=1e3, out=o0)
    assert [int(o0.item()), int(o1.item())] == [int(b.paper_count(F, st, 1e3).item()) for F, st in batches]

    # all records flagged: nothing to count
    F, st = batches[1]
    assert int(b.paper_count_static(F, torch.ones_like(st), out=out).item()) == 0

    # the limit itself fits the array; one more record is refused and the message says what to do
    n_max = b.PAPER_COUNT_STATIC_MAX_N
    F, st = _records(n_max + 1, 13, 1 << 19)
    assert int(b.paper_count_static(F[:n_max], st[:n_max], out=out).item()) == int(b.paper_count(F[:n_max], st[:n_max]).item())
    with pytest.raises(b.U1gfError) as err:
        b.paper_count_static(F, st, out=out)
    assert err.value.code == -1 and "U1GF_PAPER_COUNT_STATIC_MAX_N" in str(err.value)
    # a refused call leaves the array usable
    F, st = batches[1]
    assert int(b.paper_count_static(F, st, out=out).item()) == expected[1]
