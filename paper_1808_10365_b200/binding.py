"""Thin ctypes binding of libsk_b200.so (include/sk_b200.h): argument marshalling only.

Every step of the SK path (arXiv 1808.10365: Eq. 7, 9-11, 14, flag, excision) runs in the CUDA
kernels under csrc/.  PyTorch is used here for device memory and streams, nothing else.  There
is no CPU fallback: a missing library or a non-CUDA tensor raises.
"""
import ctypes as C
import os
from typing import NamedTuple, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsk_b200.so")

SYMBOLS = ("sk_power_sums", "sk_combine", "sk_flag", "sk_frame_workspace_bytes", "sk_frame",
           "sk_frame_noalloc",
           "sk_frame_multi_workspace_bytes", "sk_frame_multi", "sk_frame_host", "sk_frames_host", "sk_rebin_sums", "sk_single",
           "sk_significance", "sk_sim_digitised", "sk_sim_common_mode", "sk_moments", "sk_strerror", "sk_version",
           "sk_launch_count", "sk_frame_plan")

# bits of sk_frame's `flags` (include/sk_b200.h)
SK_FRAME_ZERO_FLAGGED, SK_FRAME_INPUTS_READY, SK_FRAME_EQ13 = 1, 2, 4
SK_FRAME_PLAN_LDG, SK_FRAME_PLAN_NO_TMAP = 1 << 8, 1 << 9
SK_PLAN_AUTO, SK_PLAN_LDG, SK_PLAN_NO_TMAP = 0, 1, 2      # arguments of plan_override (Python side only)

_lib = None


class SKError(RuntimeError):
    pass


def lib() -> C.CDLL:
    """Load the C-ABI library (built in-tree by `python -m paper_1808_10365_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        # a fresh checkout: compile the library in-tree (nvcc), then load it; there is no other path
        try:
            from . import build as _build
            _build.build()
        except Exception as e:
            raise SKError(f"{LIB_PATH} is missing and could not be built ({e}): run "
                          "`python -m paper_1808_10365_b200.build` (there is no CPU fallback)") from e
    L = C.CDLL(LIB_PATH)
    u32, vp, f32, i32, sz = C.c_uint32, C.c_void_p, C.c_float, C.c_int, C.c_size_t
    L.sk_power_sums.argtypes = [vp, u32, u32, u32, u32, vp, vp, vp]
    L.sk_combine.argtypes = [vp, vp, u32, u32, u32, u32, vp, u32, vp, vp]
    L.sk_flag.argtypes = [vp, u32, u32, u32, u32, f32, f32, vp, vp]
    L.sk_frame_workspace_bytes.argtypes = [u32, u32, u32, u32]
    L.sk_frame_workspace_bytes.restype = sz
    L.sk_frame.argtypes = [vp, u32, u32, u32, u32, vp, u32, f32, f32, i32, vp, vp, vp, vp, vp, sz, vp]
    L.sk_frame_noalloc.argtypes = [vp, u32, u32, u32, u32, vp, u32, f32, f32, i32, vp, vp, vp, vp, vp]
    L.sk_frame_noalloc.restype = i32
    L.sk_frame_host.argtypes = [vp, u32, u32, u32, u32, vp, u32, f32, f32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
    L.sk_frames_host.argtypes = [vp, u32, u32, u32, u32, u32, vp, u32, f32, f32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
    L.sk_frames_host.restype = i32
    L.sk_frame_multi_workspace_bytes.argtypes = [u32, u32, u32, u32, u32]
    L.sk_frame_multi_workspace_bytes.restype = sz
    L.sk_frame_multi.argtypes = [vp, u32, u32, u32, u32, u32, vp, u32, f32, vp, i32, vp, vp, vp, sz, vp]
    L.sk_frame_plan.argtypes = [u32, u32, u32, u32, u32, i32, u32, vp]
    L.sk_frame_plan.restype = i32
    L.sk_rebin_sums.argtypes = [vp, vp, u32, u32, u32, u32, u32, vp, vp, vp]
    L.sk_single.argtypes = [vp, vp, u32, u32, u32, u32, vp, vp]
    L.sk_significance.argtypes = [vp, u32, u32, u32, u32, f32, vp, vp]
    L.sk_sim_digitised.argtypes = [vp, u32, u32, u32, vp, C.c_uint64, C.c_uint64, vp]
    L.sk_moments.argtypes = [vp, u32, u32, vp, vp, vp]
    L.sk_sim_common_mode.argtypes = [u32, u32, u32, C.c_double, C.c_uint64, vp, vp]
    L.sk_strerror.argtypes = [i32]
    L.sk_strerror.restype = C.c_char_p
    L.sk_version.restype = i32
    L.sk_launch_count.restype = C.c_ulonglong
    for name in ("sk_power_sums", "sk_combine", "sk_flag", "sk_frame", "sk_frame_multi", "sk_frame_host", "sk_rebin_sums",
                 "sk_single", "sk_significance", "sk_sim_digitised", "sk_moments", "sk_sim_common_mode"):
        getattr(L, name).restype = i32
    _lib = L
    return L


def sk_strerror(code: int) -> str:
    return lib().sk_strerror(int(code)).decode()


def sk_version() -> int:
    return int(lib().sk_version())


def sk_launch_count() -> int:
    return int(lib().sk_launch_count())


_plan_flags = 0      # SK_FRAME_PLAN_* bits added to the flags of every fused call made through this module


def plan_flags(path: int = SK_PLAN_AUTO, lanes: int = 0) -> int:
    """The SK_FRAME_PLAN_* bits of include/sk_b200.h for a kernel path and a slab width of 16*lanes inputs."""
    f = SK_FRAME_PLAN_LDG if path == SK_PLAN_LDG else SK_FRAME_PLAN_NO_TMAP if path == SK_PLAN_NO_TMAP else 0
    if lanes in (1, 2, 4, 8, 16):
        f |= lanes << 12
    return f


def plan_override(path: int = SK_PLAN_AUTO, lanes: int = 0) -> None:
    """Tests and A/B timing only: from now on every sk_frame / sk_frame_multi / sk_frame_host /
    sk_frame_noalloc call made through THIS module passes the SK_FRAME_PLAN_* bits for `path` and `lanes`
    (the direct-load kernel, a refused tensor map, a narrower slab) in its flags.  The C library itself keeps
    no such state: the override is per call.  (0, 0) restores the automatic choice."""
    global _plan_flags
    _plan_flags = plan_flags(path, lanes)


def sk_frame_plan(T: int, F: int, E: int, M: int, first_n=None, inputs_ready: bool = False, nlev: int = 1,
                  flags=None):
    """(lanes, slabs, chunk_rows or 0 for the direct-load kernel, blocks_per_unit) the fused path
    would use for this shape (aligned data, no subset) under the current plan_override (or `flags`)."""
    plan = (C.c_uint32 * 4)()
    fl = (_plan_flags if flags is None else int(flags)) | (SK_FRAME_INPUTS_READY if inputs_ready else 0)
    _check(lib().sk_frame_plan(T, F, E, M, int(first_n or E), fl, nlev, C.cast(plan, C.c_void_p)), "sk_frame_plan")
    return tuple(int(x) for x in plan)


def _check(rc: int, what: str):
    if rc != 0:
        raise SKError(f"{what} failed ({rc}): {sk_strerror(rc)}")


def _dev(t: torch.Tensor, dtype, what: str) -> torch.Tensor:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise SKError(f"{what} must be a CUDA tensor (there is no CPU path)")
    if t.dtype != dtype or not t.is_contiguous():
        raise SKError(f"{what} must be a contiguous {dtype} tensor")
    return t


def _cur() -> int:
    """The raw handle of torch's current stream (inside `with torch.cuda.stream(...)`)."""
    return torch.cuda.current_stream().cuda_stream


def _torch_stream(stream, device):
    """The torch.cuda.Stream the call will run on (a raw handle is wrapped): temporaries are
    allocated, filled and released in its order, so the caching allocator cannot hand them to
    another stream while the kernel is pending."""
    if stream is None:
        return torch.cuda.current_stream(device)
    if isinstance(stream, torch.cuda.Stream):
        return stream
    return torch.cuda.ExternalStream(int(stream), device=device)


def _subset(subset, E, device):
    """Receiver subset -> E bytes on the device (uploaded on the current stream: callers hold
    `with torch.cuda.stream(...)` around this and the launch)."""
    if subset is None:
        return None
    if (isinstance(subset, torch.Tensor) and subset.is_cuda and subset.dtype == torch.uint8
            and subset.is_contiguous() and tuple(subset.shape) == (E,)):
        return subset
    s = torch.as_tensor(subset)
    s = (s != 0).to(torch.uint8).to(device).contiguous()
    if s.shape != (E,):
        raise SKError("subset must have E entries")
    return s


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else t.data_ptr()


class SKResult(NamedTuple):
    SK: torch.Tensor
    mask: torch.Tensor
    S1: Optional[torch.Tensor]
    S2: Optional[torch.Tensor]


_ws_cache = {}


def sk_frame_workspace_bytes(T: int, F: int, E: int, M: int) -> int:
    return int(lib().sk_frame_workspace_bytes(T, F, E, M))


def sk_frame_multi_workspace_bytes(T: int, F: int, E: int, M: int, nlev: int) -> int:
    return int(lib().sk_frame_multi_workspace_bytes(T, F, E, M, nlev))


def workspace_for(T, F, E, M, device, stream_id=0, nlev=1) -> torch.Tensor:
    """A zero-filled device workspace for sk_frame / sk_frame_multi, cached per (device, stream,
    size).  The library leaves a workspace zero-filled after every call, so it is cleared only
    when created — on the CURRENT torch stream: call this under `with torch.cuda.stream(s)` for
    the stream s the workspace will be used on (sk_frame does), and never use one workspace on
    two streams."""
    n = sk_frame_multi_workspace_bytes(T, F, E, M, nlev)
    if n == 0:
        raise SKError("bad shape for sk_frame")
    key = (str(device), stream_id, n)
    ws = _ws_cache.get(key)
    if ws is None:
        ws = torch.zeros((n + 7) // 8, dtype=torch.int64, device=device)
        _ws_cache[key] = ws
    return ws


def sk_power_sums(data: torch.Tensor, M: int, stream=None):
    """PAPER.md:77 Eq. 7.  data uint8 [T][F][E] (CUDA) -> S1, S2 uint32 [T/M][F][E]."""
    _dev(data, torch.uint8, "data")
    with torch.cuda.stream(_torch_stream(stream, data.device)):   # outputs are allocated in stream order
        T, F, E = data.shape
        B = T // M if M else 0
        S1 = torch.empty((B, F, E), dtype=torch.uint32, device=data.device)
        S2 = torch.empty_like(S1)
        _check(lib().sk_power_sums(data.data_ptr(), T, F, E, M, S1.data_ptr(), S2.data_ptr(), _cur()), "sk_power_sums")
        return S1, S2


def sk_combine(S1: torch.Tensor, S2: torch.Tensor, M: int, subset=None, first_n=None, stream=None):
    """PAPER.md:84-88 Eq. 9-11, :108-113 Eq. 14.  S1, S2 uint32 [B][F][E] -> SK float32 [B][F]."""
    _dev(S1, torch.uint32, "S1")
    _dev(S2, torch.uint32, "S2")
    with torch.cuda.stream(_torch_stream(stream, S1.device)):   # outputs are allocated in stream order
        B, F, E = S1.shape
        sub = _subset(subset, E, S1.device)
        if sub is None and first_n is None:
            first_n = E
        SK = torch.empty((B, F), dtype=torch.float32, device=S1.device)
        _check(lib().sk_combine(S1.data_ptr(), S2.data_ptr(), B, F, E, M, _ptr(sub), int(first_n or 0),
                                SK.data_ptr(), _cur()), "sk_combine")
        return SK


def sk_flag(SK: torch.Tensor, M: int, N: int, n_sigma: float, sk_mean: float = 1.0, stream=None):
    """PAPER.md:183 / :119 Eq. 16.  SK float32 [B][F] -> mask uint8 [B][F]."""
    _dev(SK, torch.float32, "SK")
    with torch.cuda.stream(_torch_stream(stream, SK.device)):   # outputs are allocated in stream order
        B, F = SK.shape
        mask = torch.empty((B, F), dtype=torch.uint8, device=SK.device)
        _check(lib().sk_flag(SK.data_ptr(), B, F, M, N, n_sigma, sk_mean, mask.data_ptr(), _cur()),
               "sk_flag")
        return mask


def sk_rebin_sums(S1: torch.Tensor, S2: torch.Tensor, M: int, factor: int, stream=None):
    """sums at block length M re-binned to M*factor.  [B][F][E] -> [B/factor][F][E]."""
    _dev(S1, torch.uint32, "S1")
    _dev(S2, torch.uint32, "S2")
    with torch.cuda.stream(_torch_stream(stream, S1.device)):   # outputs are allocated in stream order
        B, F, E = S1.shape
        Bo = B // factor if factor else 0
        O1 = torch.empty((Bo, F, E), dtype=torch.uint32, device=S1.device)
        O2 = torch.empty_like(O1)
        _check(lib().sk_rebin_sums(S1.data_ptr(), S2.data_ptr(), B, F, E, M, factor, O1.data_ptr(), O2.data_ptr(),
                                   _cur()), "sk_rebin_sums")
        return O1, O2


def sk_single(S1: torch.Tensor, S2: torch.Tensor, M: int, stream=None):
    """PAPER.md:80 Eq. 8 per receiver.  S1, S2 uint32 [B][F][E] -> SKi float32 [B][F][E]."""
    _dev(S1, torch.uint32, "S1")
    _dev(S2, torch.uint32, "S2")
    with torch.cuda.stream(_torch_stream(stream, S1.device)):   # outputs are allocated in stream order
        B, F, E = S1.shape
        SKi = torch.empty((B, F, E), dtype=torch.float32, device=S1.device)
        _check(lib().sk_single(S1.data_ptr(), S2.data_ptr(), B, F, E, M, SKi.data_ptr(), _cur()), "sk_single")
        return SKi


def sk_significance(SK: torch.Tensor, M: int, N: int, sk_mean: float = 1.0, stream=None):
    """PAPER.md:183 detection significance.  SK float32 [B][F] -> float32 [B][F]."""
    _dev(SK, torch.float32, "SK")
    with torch.cuda.stream(_torch_stream(stream, SK.device)):   # outputs are allocated in stream order
        B, F = SK.shape
        sig = torch.empty((B, F), dtype=torch.float32, device=SK.device)
        _check(lib().sk_significance(SK.data_ptr(), B, F, M, N, sk_mean, sig.data_ptr(), _cur()),
               "sk_significance")
        return sig


def sk_sim_digitised(T: int, F: int, E: int, thr: torch.Tensor, seed: int, frame: int = 0, out=None, stream=None):
    """PAPER.md:276-284 (App. B): seeded 4+4-bit round-and-clip Gaussian frame uint8 [T][F][E] on
    thr's device; thr uint32 [E][14] (sk_synth.digitiser_thresholds)."""
    _dev(thr, torch.uint32, "thr")
    if tuple(thr.shape) != (E, 14):
        raise SKError("thr must be [E][14]")
    with torch.cuda.stream(_torch_stream(stream, thr.device)):   # outputs are allocated in stream order
        if out is None:
            out = torch.empty((T, F, E), dtype=torch.uint8, device=thr.device)
        _dev(out, torch.uint8, "out")
        _check(lib().sk_sim_digitised(out.data_ptr(), T, F, E, thr.data_ptr(), seed, frame, _cur()),
               "sk_sim_digitised")
        return out


def sk_sim_common_mode(D: int, M: int, N: int, amp: float, seed: int, device="cuda", stream=None):
    """PAPER.md:262-272 (App. A): SK~ of D simulated datasets (M samples x N receivers, common-mode
    amplitude amp): float32 [D][1] on `device` (shape ready for sk_moments)."""
    dev = torch.device(device)
    if dev.type != "cuda":
        raise SKError("sk_sim_common_mode needs a CUDA device (there is no CPU fallback)")
    with torch.cuda.stream(_torch_stream(stream, dev)):
        SK = torch.empty((D, 1), dtype=torch.float32, device=dev)
        _check(lib().sk_sim_common_mode(D, M, N, float(amp), seed, SK.data_ptr(), _cur()), "sk_sim_common_mode")
        return SK


def sk_moments(SK: torch.Tensor, stream=None):
    """Mean and unbiased variance of SK float32 [B][F] over the blocks: float64 [F] each."""
    _dev(SK, torch.float32, "SK")
    with torch.cuda.stream(_torch_stream(stream, SK.device)):   # outputs are allocated in stream order
        B, F = SK.shape
        mean = torch.empty(F, dtype=torch.float64, device=SK.device)
        var = torch.empty(F, dtype=torch.float64, device=SK.device)
        _check(lib().sk_moments(SK.data_ptr(), B, F, mean.data_ptr(), var.data_ptr(), _cur()), "sk_moments")
        return mean, var


def sk_frame(data: torch.Tensor, M: int, subset=None, first_n=None, n_sigma: float = 3.0,
             sk_mean: float = 1.0, zero_flagged: bool = False, want_sums: bool = False,
             out: Optional[SKResult] = None, workspace: Optional[torch.Tensor] = None,
             stream=None, inputs_ready: bool = False, eq13: bool = False) -> SKResult:
    """The fused path (one pass over HBM).  `data` is modified in place only if zero_flagged.
    inputs_ready = SK_FRAME_INPUTS_READY (include/sk_b200.h): nothing enqueued on the stream since
    its last synchronisation (or the last call without the flag) writes `data`/`subset`, so the
    kernel may overlap the previous one.  eq13 = SK_FRAME_EQ13."""
    _dev(data, torch.uint8, "data")
    T, F, E = data.shape
    B = T // M if M else 0
    dev = data.device
    ts = _torch_stream(stream, dev)
    with torch.cuda.stream(ts):                 # outputs, subset upload, workspace fill: in stream order
        sub = _subset(subset, E, dev)
        if sub is None and first_n is None:
            first_n = E
        if out is None:
            SK = torch.empty((B, F), dtype=torch.float32, device=dev)
            mask = torch.empty((B, F), dtype=torch.uint8, device=dev)
            S1 = torch.empty((B, F, E), dtype=torch.uint32, device=dev) if want_sums else None
            S2 = torch.empty((B, F, E), dtype=torch.uint32, device=dev) if want_sums else None
            out = SKResult(SK, mask, S1, S2)
        if workspace is None:
            workspace = workspace_for(T, F, E, M, dev, ts.cuda_stream)
        flags = ((SK_FRAME_ZERO_FLAGGED if zero_flagged else 0) | (SK_FRAME_INPUTS_READY if inputs_ready else 0)
                 | (SK_FRAME_EQ13 if eq13 else 0) | _plan_flags)
        _check(lib().sk_frame(data.data_ptr(), T, F, E, M, _ptr(sub), int(first_n or 0), n_sigma, sk_mean,
                              flags, out.SK.data_ptr(), out.mask.data_ptr(), _ptr(out.S1), _ptr(out.S2),
                              workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                              ts.cuda_stream), "sk_frame")
    return out


SK_NOALLOC_SCRATCH_BYTES = 4 << 20     # include/sk_b200.h


def sk_frame_noalloc(data: torch.Tensor, M: int, out: SKResult, subset: Optional[torch.Tensor] = None, first_n=None,
                     n_sigma: float = 3.0, sk_mean: float = 1.0, zero_flagged: bool = False, stream=None,
                     eq13: bool = False) -> SKResult:
    """sk_frame for code that must not allocate on the device (include/sk_b200.h, sk_frame_noalloc):
    a pipeline stage whose buffers all come from the host framework's start-up pool, or a real-time
    loop that cannot take the device-wide stall of a cudaMalloc.  The scratch is a 4 MiB array inside
    the library, so frames whose sk_frame_workspace_bytes exceeds SK_NOALLOC_SCRATCH_BYTES raise.

    Nothing is allocated here either, which is why `out` (SK, mask and optionally S1, S2, all
    pre-allocated CUDA tensors of the right shape) is required and `subset`, if given, must already
    be a uint8 [E] CUDA tensor.  All calls on one device share the one scratch array: keep them on
    one stream.  Make the first call on a device before any stream capture (it looks up the array's
    device address)."""
    _dev(data, torch.uint8, "data")
    T, F, E = data.shape
    B = T // M if M else 0
    _dev(out.SK, torch.float32, "out.SK")
    _dev(out.mask, torch.uint8, "out.mask")
    if tuple(out.SK.shape) != (B, F) or tuple(out.mask.shape) != (B, F):
        raise SKError("out.SK and out.mask must be [T/M][F]")
    for t, what in ((out.S1, "out.S1"), (out.S2, "out.S2")):
        if t is not None:
            _dev(t, torch.uint32, what)
            if tuple(t.shape) != (B, F, E):
                raise SKError(f"{what} must be [T/M][F][E]")
    if subset is not None:
        _dev(subset, torch.uint8, "subset")
        if tuple(subset.shape) != (E,):
            raise SKError("subset must have E entries")
    elif first_n is None:
        first_n = E
    ts = _torch_stream(stream, data.device)
    flags = (SK_FRAME_ZERO_FLAGGED if zero_flagged else 0) | (SK_FRAME_EQ13 if eq13 else 0) | _plan_flags
    with torch.cuda.device(data.device):        # the scratch's address is looked up on the current device
        _check(lib().sk_frame_noalloc(data.data_ptr(), T, F, E, M, _ptr(subset), int(first_n or 0), n_sigma, sk_mean,
                                      flags, out.SK.data_ptr(), out.mask.data_ptr(), _ptr(out.S1), _ptr(out.S2),
                                      ts.cuda_stream), "sk_frame_noalloc")
    return out


class SKMultiResult(NamedTuple):
    SK: list        # per integration length M << l: float32 [T / (M << l)][F]
    mask: list      # uint8, same shapes


def sk_frame_multi(data: torch.Tensor, M: int, nlev: int, subset=None, first_n=None, n_sigma: float = 3.0,
                   sk_means=None, zero_flagged: bool = False, out: Optional[SKMultiResult] = None,
                   workspace: Optional[torch.Tensor] = None, stream=None,
                   inputs_ready: bool = False) -> SKMultiResult:
    """SK and mask at the integration lengths M, 2M, ..., M << (nlev-1) from one
    pass over the data.  sk_means: one flag centre per length (default 1.0 each)."""
    _dev(data, torch.uint8, "data")
    T, F, E = data.shape
    dev = data.device
    nlev = int(nlev)
    if not 1 <= nlev <= 4:
        raise SKError("nlev must be in [1, 4]")
    means = [1.0] * nlev if sk_means is None else [float(x) for x in sk_means]
    if len(means) != nlev:
        raise SKError("sk_means must have nlev entries")
    ts = _torch_stream(stream, dev)
    with torch.cuda.stream(ts):
        sub = _subset(subset, E, dev)
        if sub is None and first_n is None:
            first_n = E
        if out is None:
            shapes = [((T // (M << l)) if M else 0, F) for l in range(nlev)]
            out = SKMultiResult([torch.empty(s, dtype=torch.float32, device=dev) for s in shapes],
                                [torch.empty(s, dtype=torch.uint8, device=dev) for s in shapes])
        if workspace is None:
            workspace = workspace_for(T, F, E, M, dev, ts.cuda_stream, nlev)
        c_means = (C.c_float * nlev)(*means)
        c_SK = (C.c_void_p * nlev)(*[t.data_ptr() for t in out.SK])
        c_mask = (C.c_void_p * nlev)(*[t.data_ptr() for t in out.mask])
        flags = (SK_FRAME_ZERO_FLAGGED if zero_flagged else 0) | (SK_FRAME_INPUTS_READY if inputs_ready else 0) | _plan_flags
        _check(lib().sk_frame_multi(data.data_ptr(), T, F, E, M, nlev, _ptr(sub), int(first_n or 0), n_sigma,
                                    C.cast(c_means, C.c_void_p), flags, C.cast(c_SK, C.c_void_p),
                                    C.cast(c_mask, C.c_void_p), workspace.data_ptr(),
                                    workspace.numel() * workspace.element_size(), ts.cuda_stream), "sk_frame_multi")
    return out


def sk_frame_host(h_data: torch.Tensor, M: int, h_SK: torch.Tensor, h_mask: torch.Tensor,
                  d_data: torch.Tensor, d_SK: torch.Tensor, d_mask: torch.Tensor, subset=None,
                  first_n=None, n_sigma: float = 3.0, sk_mean: float = 1.0, zero_flagged: bool = False,
                  workspace: Optional[torch.Tensor] = None, stream=None):
    """End-to-end form: host buffers in and out (pinned recommended), copies inside the call."""
    if h_data.is_cuda or h_SK.is_cuda or h_mask.is_cuda:
        raise SKError("h_* tensors must live in host memory")
    T, F, E = h_data.shape
    _dev(d_data, torch.uint8, "d_data")
    ts = _torch_stream(stream, d_data.device)
    with torch.cuda.stream(ts):
        sub = _subset(subset, E, d_data.device)
        if sub is None and first_n is None:
            first_n = E
        if workspace is None:
            workspace = workspace_for(T, F, E, M, d_data.device, ts.cuda_stream)
        _check(lib().sk_frame_host(h_data.data_ptr(), T, F, E, M, _ptr(sub), int(first_n or 0), n_sigma,
                                   sk_mean, int(bool(zero_flagged)) | _plan_flags, h_SK.data_ptr(), h_mask.data_ptr(),
                                   d_data.data_ptr(), d_SK.data_ptr(), d_mask.data_ptr(), workspace.data_ptr(),
                                   workspace.numel() * workspace.element_size(), ts.cuda_stream), "sk_frame_host")
    return h_SK, h_mask


def sk_frames_host(h_frames, M: int, h_SK: torch.Tensor, h_mask: torch.Tensor, d_data: torch.Tensor,
                   d_SK: torch.Tensor, d_mask: torch.Tensor, subset=None, first_n=None, n_sigma: float = 3.0,
                   sk_mean: float = 1.0, zero_flagged: bool = False, workspace: Optional[torch.Tensor] = None, stream=None):
    """sk_frame_host for a queue of frames (include/sk_b200.h): h_frames is a list of host tensors uint8
    [T][F][E] (pinned recommended), h_SK float32 / h_mask uint8 [len(h_frames)][T/M][F] receive the results;
    uploads, kernels and read-backs are enqueued back to back and the call waits once at the end."""
    n = len(h_frames)
    if n == 0 or any(t.is_cuda or t.dtype != torch.uint8 or not t.is_contiguous() or t.shape != h_frames[0].shape
                     for t in h_frames) or h_SK.is_cuda or h_mask.is_cuda:
        raise SKError("h_frames must be equal-shaped contiguous uint8 host tensors, h_SK / h_mask host tensors")
    T, F, E = h_frames[0].shape
    B = T // M if M else 0
    if (tuple(h_SK.shape) != (n, B, F) or tuple(h_mask.shape) != (n, B, F) or h_SK.dtype != torch.float32
            or h_mask.dtype != torch.uint8 or not h_SK.is_contiguous() or not h_mask.is_contiguous()):
        raise SKError("h_SK float32 / h_mask uint8 must be contiguous [nframes][T/M][F]")
    _dev(d_data, torch.uint8, "d_data")
    ts = _torch_stream(stream, d_data.device)
    with torch.cuda.stream(ts):
        sub = _subset(subset, E, d_data.device)
        if sub is None and first_n is None:
            first_n = E
        if workspace is None:
            workspace = workspace_for(T, F, E, M, d_data.device, ts.cuda_stream)
        ptrs = (C.c_void_p * n)(*[t.data_ptr() for t in h_frames])
        _check(lib().sk_frames_host(C.cast(ptrs, C.c_void_p), n, T, F, E, M, _ptr(sub), int(first_n or 0), n_sigma, sk_mean,
                                    int(bool(zero_flagged)) | _plan_flags, h_SK.data_ptr(), h_mask.data_ptr(),
                                    d_data.data_ptr(), d_SK.data_ptr(), d_mask.data_ptr(), workspace.data_ptr(),
                                    workspace.numel() * workspace.element_size(), ts.cuda_stream), "sk_frames_host")
    return h_SK, h_mask
