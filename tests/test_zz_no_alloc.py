"""catapult_estimate_static: the Monte-Carlo estimate (Eq. 2) for callers that must not allocate.

Who needs it: a program that gave all of its GPU memory to its own memory manager at start-up and cannot let a
library go to the driver for more, a loop with a latency budget in which an allocation may block or fail at the wrong
moment, or a driver set-up without memory pools (no cudaMallocAsync).  catapult_estimate takes its per-block partial
sums from the stream-ordered allocator on every call; the static variant keeps them in a 16 KiB array that is part
of the library's device image, for at most CATAPULT_ESTIMATE_STATIC_MAX_N = 2,097,152 particles.

What is checked here: the static entry point returns what catapult_estimate returns (it uses the same block partition
and summation order, so the comparison is exact, which is inside the 1e-12 / exact-count tolerance of
test_estimate_parity), on two calls in a row -- the second call finds the first call's partial sums in the shared
array and must not be disturbed by them, including when it needs fewer blocks than the first --, on another
measurement g, and up to the size limit; that a size beyond the limit is refused with a message that names it; and
that the calls leave the device's memory pool and free memory as they found them.

The file name sorts last on purpose: `pytest -x` stops at the first failure, so this extra entry point cannot hide a
failure of the parity tests.  It depends on nothing the other tests do: it passes alone in a fresh process (where
its first call is the one that looks the array up on the device) and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def K():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    from paper_2604_07617_b200 import binding
    binding.load()
    return binding


def _inputs(n, seed):
    rng = np.random.default_rng(seed)
    status = torch.from_numpy(rng.integers(0, 3, size=n).astype(np.int32)).cuda()
    tstop = torch.from_numpy(rng.random(n) * 1e-3).cuda()
    return status, tstop, tstop * tstop


def _same(got, want, kind):
    got, want = got.cpu().numpy(), np.asarray(want)
    if kind == 0:
        assert got[2] == want[2] and got[0] == want[0]          # the lost count and the loss fraction: exact
    assert np.allclose(got, want, rtol=1e-12, atol=1e-300)       # the tolerance of test_estimate_parity
    assert np.array_equal(got, want)                             # and in fact the same bits: same summation order


def test_static_estimate_equals_the_allocating_one_on_two_calls_in_a_row(K):
    out = torch.empty(4, dtype=torch.float64, device="cuda")     # the caller's result buffer, made once
    # first call: 300,001 particles = 147 blocks of partial sums left behind in the shared array
    s1, t1, u1 = _inputs(300_001, 5)
    want1 = K.catapult_estimate(0, d_status=s1, d_tstop=t1, d_g_user=u1)
    got1 = K.catapult_estimate_static(0, d_status=s1, d_tstop=t1, d_g_user=u1, out=out)
    assert got1.data_ptr() == out.data_ptr()
    _same(got1, want1, 0)
    # second call straight after it, fewer particles (3 blocks) and other values: must not see the leftovers
    s2, t2, u2 = _inputs(5_000, 6)
    for kind in (0, 1, 2):
        want2 = K.catapult_estimate(kind, d_status=s2, d_tstop=t2, d_g_user=u2)
        _same(K.catapult_estimate_static(kind, d_status=s2, d_tstop=t2, d_g_user=u2, out=out), want2, kind)
    # and the first inputs again give the first answer again
    _same(K.catapult_estimate_static(0, d_status=s1, d_tstop=t1, d_g_user=u1, out=out), want1, 0)


@pytest.mark.parametrize("n", [1, 2, 31, 2048, 2049, 1_000_000])
def test_static_estimate_sizes(K, n):
    s, t, u = _inputs(n, 100 + n % 97)
    for kind in (0, 1, 2):
        _same(K.catapult_estimate_static(kind, d_status=s, d_tstop=t, d_g_user=u),
              K.catapult_estimate(kind, d_status=s, d_tstop=t, d_g_user=u), kind)


def test_static_estimate_size_limit_and_bad_arguments(K):
    nmax = K.ESTIMATE_STATIC_MAX_N
    assert nmax == 2_097_152
    s = torch.ones(nmax + 1, dtype=torch.int32, device="cuda")
    got = K.catapult_estimate_static(0, d_status=s[:nmax])        # exactly the limit: all 1024 slots in use
    assert got[2].item() == float(nmax) and got[0].item() == 1.0
    _same(got, K.catapult_estimate(0, d_status=s[:nmax]), 0)
    with pytest.raises(K.CatapultError) as e:                     # one more: refused, with the limit in the message
        K.catapult_estimate_static(0, d_status=s)
    assert e.value.status == K.EINVAL and "CATAPULT_ESTIMATE_STATIC_MAX_N" in str(e.value) and "2097152" in str(e.value)
    with pytest.raises(K.CatapultError):                          # same argument rules as catapult_estimate
        K.catapult_estimate_static(1, d_status=s[:8])
    # an empty ensemble is allowed, as in catapult_estimate: all four numbers zero
    z = K.catapult_estimate_static(0, d_status=s[:0])
    assert np.array_equal(z.cpu().numpy(), np.zeros(4))


def test_static_estimate_takes_no_device_memory(K):
    """Neither the driver's free memory nor the device's stream-ordered pool changes across calls of the static entry
    point (the result tensor is made before the measurement; the first call of this process has already happened in
    the warm-up line, because looking the array up may load the library's device image)."""
    s, t, u = _inputs(100_000, 9)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    K.catapult_estimate_static(0, d_status=s, out=out)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    reserved0 = torch.cuda.memory_reserved()
    for kind in (0, 1, 2):
        K.catapult_estimate_static(kind, d_status=s, d_tstop=t, d_g_user=u, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.cuda.memory_reserved() == reserved0
