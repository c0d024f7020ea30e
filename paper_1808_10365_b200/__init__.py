"""B200-native spectral-kurtosis (SK) RFI detector — the hot path of arXiv 1808.10365.

The product is the C-ABI library built from csrc/ (declared in include/sk_b200.h); this package is
its thin Python binding.  See DESIGN.md.
"""
from .binding import (SKError, SKResult, SKMultiResult, LIB_PATH, SYMBOLS, SK_PLAN_AUTO, SK_PLAN_LDG, SK_PLAN_NO_TMAP, lib, sk_combine,
                      sk_frame_plan, plan_override, plan_flags, sk_flag, sk_frame, sk_frame_multi, sk_frame_multi_workspace_bytes,
                      sk_frame_noalloc, SK_NOALLOC_SCRATCH_BYTES,
                      sk_frame_host, sk_frames_host, sk_frame_workspace_bytes, sk_launch_count, sk_power_sums,
                      sk_moments, sk_rebin_sums, sk_significance, sk_sim_common_mode, sk_sim_digitised, sk_single, sk_strerror, sk_version, workspace_for)

__all__ = ["SKError", "SKResult", "SKMultiResult", "LIB_PATH", "SYMBOLS", "SK_PLAN_AUTO", "SK_PLAN_LDG", "SK_PLAN_NO_TMAP", "lib",
           "sk_combine", "sk_frame_plan", "plan_override", "plan_flags", "sk_flag", "sk_frame", "sk_frame_multi", "sk_frame_multi_workspace_bytes",
           "sk_frame_noalloc", "SK_NOALLOC_SCRATCH_BYTES",
           "sk_frame_host", "sk_frames_host", "sk_frame_workspace_bytes", "sk_launch_count", "sk_power_sums",
           "sk_moments", "sk_rebin_sums", "sk_significance", "sk_sim_common_mode", "sk_sim_digitised", "sk_single",
           "sk_strerror", "sk_version", "workspace_for"]
