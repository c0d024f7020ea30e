"""ctypes binding of libsk_b200_bench.so (csrc/bench/sk_bench.h): MEASUREMENT ONLY.

bench.py (--op ceiling, --op memonly, the roofline's sm_ceiling extra) and one GPU test use it.  It is
not part of the product: libsk_b200.so and include/sk_b200.h contain none of these entry points.
"""
import ctypes as C
import os

import torch

from .binding import SKError, sk_strerror

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsk_b200_bench.so")
SYMBOLS = ("skb_loop_ceiling", "skb_pipe_rate", "skb_stream_workspace_bytes", "skb_stream", "skb_frame_loop",
           "skb_launch_count")
VAR_PRODUCT, VAR_MEMONLY, VAR_NO_SUB, VAR_NO_PICK, VAR_NO_UNPACK = 0, 1, 2, 3, 4
VARIANTS = {"product": VAR_PRODUCT, "memonly": VAR_MEMONLY, "no_fadd2": VAR_NO_SUB, "no_prmt": VAR_NO_PICK,
            "no_unpack": VAR_NO_UNPACK}
PIPE_MODES = ("FFMA", "FFMA2", "FADD2", "IDP.4A", "PRMT", "IDP+FFMA2", "IDP+FFMA", "PRMT+FFMA2", "IDP+PRMT")

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        try:
            from . import build as _build
            _build.build_one(_build.BENCH_LIB)
        except Exception as e:
            raise SKError(f"{LIB_PATH} is missing and could not be built ({e})") from e
    L = C.CDLL(LIB_PATH)
    u32, vp, i32, sz = C.c_uint32, C.c_void_p, C.c_int, C.c_size_t
    L.skb_loop_ceiling.argtypes = [i32, u32, u32, vp, vp, vp, vp]
    L.skb_loop_ceiling.restype = i32
    L.skb_pipe_rate.argtypes = [i32, u32, vp, vp, vp, vp]
    L.skb_pipe_rate.restype = i32
    L.skb_stream_workspace_bytes.argtypes = [u32, u32, u32, u32]
    L.skb_stream_workspace_bytes.restype = sz
    L.skb_stream.argtypes = [i32, vp, u32, u32, u32, u32, vp, vp, vp, sz, i32, vp]
    L.skb_stream.restype = i32
    L.skb_frame_loop.argtypes = [vp, vp, u32, u32, u32, u32, u32, C.c_float, C.c_float, i32, vp, vp, vp, sz, u32, vp, vp]
    L.skb_frame_loop.restype = i32
    L.skb_launch_count.restype = C.c_ulonglong
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != 0:
        raise SKError(f"{what} failed ({rc}): {sk_strerror(rc)}")


def _cur() -> int:
    return torch.cuda.current_stream().cuda_stream


def launch_count() -> int:
    return int(lib().skb_launch_count())


def loop_ceiling(warps_per_sm: int = 12, rounds: int = 200, device="cuda", variant: int = VAR_PRODUCT) -> float:
    """Sub-partition cycles per 32 samples of the hot loop (or of a removal variant of it) on a fixed
    shared-memory tile, no global-memory traffic.  Synchronises."""
    dev = torch.device(device)
    if dev.type != "cuda":
        raise SKError("loop_ceiling needs a CUDA device")
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sink = torch.empty(sms * warps_per_sm * 32, dtype=torch.int32, device=dev)
    cycles = torch.zeros(1, dtype=torch.int64, device=dev)
    spl = C.c_double(0.0)
    _check(lib().skb_loop_ceiling(variant, warps_per_sm, rounds, sink.data_ptr(), cycles.data_ptr(),
                                  C.cast(C.pointer(spl), C.c_void_p), _cur()), "skb_loop_ceiling")
    torch.cuda.synchronize(dev)
    return float(cycles.item()) / (spl.value * warps_per_sm / 4.0)


def pipe_rate(mode: int, warps_per_sm: int = 16, device="cuda") -> float:
    """Sub-partition cycles per warp instruction of PIPE_MODES[mode].  Synchronises."""
    dev = torch.device(device)
    if dev.type != "cuda":
        raise SKError("pipe_rate needs a CUDA device")
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    io = torch.full((2048 + sms * warps_per_sm * 32,), 0x3F800011, dtype=torch.int32, device=dev)
    cycles = torch.zeros(1, dtype=torch.int64, device=dev)
    n = C.c_double(0.0)
    _check(lib().skb_pipe_rate(mode, warps_per_sm, io.data_ptr(), cycles.data_ptr(),
                               C.cast(C.pointer(n), C.c_void_p), _cur()), "skb_pipe_rate")
    torch.cuda.synchronize(dev)
    return float(cycles.item()) / (n.value * warps_per_sm / 4.0)


def stream_workspace(T: int, F: int, E: int, M: int, device) -> torch.Tensor:
    n = int(lib().skb_stream_workspace_bytes(T, F, E, M))
    if n == 0:
        raise SKError("skb_stream: needs E % 256 == 0, M % 32 == 0, 32 <= M <= 256")
    return torch.zeros((n + 7) // 8, dtype=torch.int64, device=device)


def stream(variant: int, data: torch.Tensor, M: int, SK: torch.Tensor, mask: torch.Tensor, workspace: torch.Tensor,
           inputs_ready: bool = False, stream=None) -> None:
    """The product's TMA stream kernel with the loop body of `variant` (VAR_PRODUCT / VAR_MEMONLY) on
    data uint8 [T][F][E]; SK float32 / mask uint8 [T/M][F] are written (meaningless with VAR_MEMONLY)."""
    T, F, E = data.shape
    st = _cur() if stream is None else stream.cuda_stream
    _check(lib().skb_stream(variant, data.data_ptr(), T, F, E, M, SK.data_ptr(), mask.data_ptr(), workspace.data_ptr(),
                            workspace.numel() * workspace.element_size(), int(bool(inputs_ready)), st), "skb_stream")


def frame_loop(frames, M: int, SK: torch.Tensor, mask: torch.Tensor, workspace: torch.Tensor, calls: int, flags: int = 0,
               n_sigma: float = 5.0, sk_mean: float = 1.0, stream=None) -> float:
    """`calls` plain back-to-back sk_frame calls (the PRODUCT library's entry point) issued from a C loop, call i on
    frames[i % len(frames)]: what a C caller without a CUDA graph gets.  Returns the host seconds the loop took."""
    from . import binding
    T, F, E = frames[0].shape
    ptrs = (C.c_void_p * len(frames))(*[f.data_ptr() for f in frames])
    host_s = C.c_double(0.0)
    st = _cur() if stream is None else stream.cuda_stream
    fn = C.cast(binding.lib().sk_frame, C.c_void_p)
    _check(lib().skb_frame_loop(fn, C.cast(ptrs, C.c_void_p), len(frames), T, F, E, M, n_sigma, sk_mean, int(flags),
                                SK.data_ptr(), mask.data_ptr(), workspace.data_ptr(),
                                workspace.numel() * workspace.element_size(), calls,
                                C.cast(C.pointer(host_s), C.c_void_p), st), "skb_frame_loop")
    return host_s.value
