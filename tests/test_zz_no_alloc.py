"""sk_frame_noalloc against sk_frame.

sk_frame_noalloc (include/sk_b200.h) is the fused path for callers that cannot allocate device
memory: a stage inside a real-time pipeline gets every buffer from the host framework's start-up
pool and has no allocator of its own, and a frame loop that is already running cannot take the
device-wide stall of a cudaMalloc.  Instead of a caller-supplied workspace it uses a 4 MiB array
built into the library, shared by all calls on a device and never cleared behind the caller's back
except by the call itself.  What has to hold, and what this file checks on the GPU:

  * its outputs equal those of the existing sk_frame path on the same bytes (S1, S2, mask and
    excised bytes bit for bit, SK within the 1e-6 relative bound every parity test here uses);
  * that stays true for calls made back to back with no synchronisation in between, on shapes
    that lay the shared array out differently, i.e. what one call leaves behind never leaks into
    the next;
  * a frame that needs more than the built-in array is refused, and nothing is launched.

The file name keeps it last in pytest's collection order on purpose: the suite runs with -x, and a
failure here must not hide the parity tests.  It does not depend on anything the earlier files
do (it resets the test-only plan override and uses its own buffers), so it passes alone in a fresh
process as well as at the end of the whole run.
"""
import ctypes as C

import numpy as np
import pytest
import torch

import sk_synth

SK_RTOL = 1e-6          # the bar of tests/test_gpu_parity.py: |a - b| <= 1e-6 * max(1, |b|)


@pytest.fixture(scope="module")
def sk():
    import paper_1808_10365_b200 as m
    from paper_1808_10365_b200 import build
    build.build()
    m.lib()
    return m


def _i32(t):
    return t.view(torch.int32) if t.dtype in (torch.uint32, torch.float32) else t


def _empty_result(sk, T, F, E, M, dev, sums):
    B = T // M
    return sk.SKResult(torch.empty((B, F), dtype=torch.float32, device=dev),
                       torch.empty((B, F), dtype=torch.uint8, device=dev),
                       torch.empty((B, F, E), dtype=torch.uint32, device=dev) if sums else None,
                       torch.empty((B, F, E), dtype=torch.uint32, device=dev) if sums else None)


def _assert_same(got, got_data, want, want_data, what):
    assert torch.equal(got.mask, want.mask), f"{what}: mask"
    if want.S1 is not None:
        assert torch.equal(_i32(got.S1), _i32(want.S1)), f"{what}: S1"
        assert torch.equal(_i32(got.S2), _i32(want.S2)), f"{what}: S2"
    assert torch.equal(got_data, want_data), f"{what}: frame bytes after excision"
    a = got.SK.double().cpu().numpy()
    b = want.SK.double().cpu().numpy()
    assert np.array_equal(np.isnan(a), np.isnan(b)), f"{what}: NaN pattern"
    ok = ~np.isnan(b)
    err = np.abs(a[ok] - b[ok])
    assert (err <= SK_RTOL * np.maximum(1.0, np.abs(b[ok]))).all(), f"{what}: max SK error {err.max():.3e}"


# (host frame, M, keyword arguments common to both paths, with S1/S2): three shapes whose scratch
# layouts differ (cells x slabs), the middle one the 2048-input CHIME frame of BASELINE config 1
def _cases():
    cfg0 = sk_synth.config(0)
    return [
        ("toy, excised", sk_synth.make_frame(cfg0), cfg0.M, dict(n_sigma=3.0, sk_mean=0.941, zero_flagged=True), True),
        ("chime frame", sk_synth.random_bytes(49152, 1, 2048, seed=41), 256, dict(n_sigma=3.0, sk_mean=0.4), False),
        ("3 freq, first 1000, excised", sk_synth.random_bytes(2048, 3, 2048, seed=42), 128,
         dict(n_sigma=2.0, sk_mean=0.4, first_n=1000, zero_flagged=True), False),
        ("odd width (scalar kernel)", sk_synth.random_bytes(96, 2, 50, seed=43), 32, dict(n_sigma=1.0, sk_mean=0.4), True),
    ]


@pytest.mark.gpu
def test_noalloc_equals_sk_frame_back_to_back(sk):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sk.plan_override(0, 0)
    dev = torch.device("cuda", torch.cuda.current_device())
    cases = _cases()
    # the existing path first, each frame on its own copy and with its own workspace
    want = []
    for what, host, M, kw, sums in cases:
        d = host.to(dev)
        want.append((sk.sk_frame(d, M, want_sums=sums, **kw), d))
    torch.cuda.synchronize()
    # then every frame through sk_frame_noalloc, twice round, all calls enqueued one after the other
    # on one stream with no synchronisation: call k+1 starts from whatever call k left in the array
    got = []
    for rnd in range(2):
        for what, host, M, kw, sums in cases:
            T, F, E = host.shape
            d = host.to(dev)
            out = _empty_result(sk, T, F, E, M, dev, sums)
            n0 = sk.sk_launch_count()
            sk.sk_frame_noalloc(d, M, out, **kw)
            assert sk.sk_launch_count() - n0 == 1, "one fused kernel per call, as for sk_frame"
            got.append((f"round {rnd}, {what}", out, d))
    torch.cuda.synchronize()
    for i, (what, out, d) in enumerate(got):
        ref, ref_data = want[i % len(cases)]
        _assert_same(out, d, ref, ref_data, what)
    # the checks above are not vacuous: both mask values occur, and excision changed bytes
    assert 0 < int(want[0][0].mask.sum().item()) < want[0][0].mask.numel()
    assert not torch.equal(want[0][1].cpu(), cases[0][1])


@pytest.mark.gpu
def test_noalloc_same_frame_twice_in_a_row(sk):
    """The plainest form of the requirement: one frame, two calls in a row, both equal to sk_frame."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    sk.plan_override(0, 0)
    dev = torch.device("cuda", torch.cuda.current_device())
    host = sk_synth.random_bytes(4096, 4, 1024, seed=44)
    d = host.to(dev)
    kw = dict(n_sigma=2.5, sk_mean=0.4)
    ref = sk.sk_frame(d, 256, want_sums=True, **kw)
    a = sk.sk_frame_noalloc(d, 256, _empty_result(sk, 4096, 4, 1024, 256, dev, True), **kw)
    b = sk.sk_frame_noalloc(d, 256, _empty_result(sk, 4096, 4, 1024, 256, dev, True), **kw)
    torch.cuda.synchronize()
    _assert_same(a, d, ref, d, "first call")
    _assert_same(b, d, ref, d, "second call")


@pytest.mark.gpu
def test_noalloc_refuses_oversize_then_still_works(sk):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    dev = torch.device("cuda", torch.cuda.current_device())
    # 64 blocks x 80 frequencies x 128 slabs x 8 B = 5 MiB of scratch > 4 MiB (the frame itself is 160 MiB)
    T, F, E, M = 1024, 80, 2048, 16
    assert sk.sk_frame_workspace_bytes(T, F, E, M) > sk.SK_NOALLOC_SCRATCH_BYTES
    big = torch.zeros((T, F, E), dtype=torch.uint8, device=dev)
    n0 = sk.sk_launch_count()
    with pytest.raises(sk.SKError, match="SK_NOALLOC_SCRATCH_BYTES"):
        sk.sk_frame_noalloc(big, M, _empty_result(sk, T, F, E, M, dev, False))
    assert sk.sk_launch_count() == n0
    del big
    host = sk_synth.random_bytes(512, 1, 256, seed=45)
    d = host.to(dev)
    ref = sk.sk_frame(d, 64, sk_mean=0.4)
    out = sk.sk_frame_noalloc(d, 64, _empty_result(sk, 512, 1, 256, 64, dev, False), sk_mean=0.4)
    torch.cuda.synchronize()
    _assert_same(out, d, ref, d, "after a refused call")


def test_noalloc_size_and_argument_errors_need_no_device(sk):
    """Refusals come before the library touches the device (so they can be checked on a CPU box)."""
    L = sk.lib()
    one = C.c_void_p(256)              # never dereferenced
    assert sk.SK_NOALLOC_SCRATCH_BYTES == 4 << 20
    # config 4 of BASELINE.json needs 16 MiB of scratch: refused
    assert L.sk_frame_noalloc(one, 65536, 64, 2048, 256, None, 2048, 3.0, 1.0, 0, one, one, None, None, None) == -7
    # the largest configs that fit: config 2 (2 MiB + 8 KiB) is not refused for its size (-4: first_n > E)
    assert sk.sk_frame_workspace_bytes(32768, 16, 2048, 256) <= sk.SK_NOALLOC_SCRATCH_BYTES
    assert L.sk_frame_noalloc(one, 32768, 16, 2048, 256, None, 4096, 3.0, 1.0, 0, one, one, None, None, None) == -4
    assert L.sk_frame_noalloc(None, 8, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, one, None, None, None) == -1
    assert L.sk_frame_noalloc(one, 9, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, one, None, None, None) == -2
    assert L.sk_frame_noalloc(one, 8, 1, 16, 4, None, 16, float("nan"), 1.0, 0, one, one, None, None, None) == -5
    assert L.sk_frame_noalloc(one, 8, 1, 16, 4, None, 16, 3.0, 1.0, 0, one, one, one, None, None) == -1
    assert "SK_NOALLOC_SCRATCH_BYTES" in sk.sk_strerror(-7)
