"""ctypes binding of oracle/libsk_oracle.so — TEST INFRASTRUCTURE, not the product.

Argument marshalling only (numpy arrays in, numpy arrays out); all arithmetic is in
oracle/sk_oracle.cpp, which cites the passage of PAPER.md each function follows.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.sk_oracle_single.restype = C.c_double
        _lib.sk_oracle_single.argtypes = [C.c_double] * 3
    return _lib


def _p(a, ty):
    return None if a is None else a.ctypes.data_as(C.POINTER(ty))


def _subset(subset, E):
    if subset is None:
        return None
    s = np.ascontiguousarray(np.asarray(subset) != 0, dtype=np.uint8)
    assert s.shape == (E,)
    return s


def _n(subset, first_n, E):
    return int(first_n if subset is None else np.count_nonzero(subset))


def _check(rc, what):
    if rc != 0:
        raise ValueError(f"{what}: oracle rejected the arguments (rc={rc})")


def power_sums(data, M):
    """PAPER.md:77 Eq. 7.  data uint8 [T][F][E] -> S1, S2 uint32 [T/M][F][E]."""
    data = np.ascontiguousarray(data, dtype=np.uint8)
    T, F, E = data.shape
    S1 = np.empty((T // M if M else 0, F, E), np.uint32)
    S2 = np.empty_like(S1)
    _check(lib().sk_oracle_power_sums(_p(data, C.c_uint8), T, F, E, M, _p(S1, C.c_uint32),
                                      _p(S2, C.c_uint32)), "power_sums")
    return S1, S2


def combine(S1, S2, M, subset=None, first_n=None, want64=False):
    """PAPER.md:84-88 Eq. 9-11, :108-113 Eq. 14.  -> SK float32 [B][F] (and float64 if want64)."""
    S1 = np.ascontiguousarray(S1, dtype=np.uint32)
    S2 = np.ascontiguousarray(S2, dtype=np.uint32)
    B, F, E = S1.shape
    sub = _subset(subset, E)
    if sub is None and first_n is None:
        first_n = E
    SK = np.empty((B, F), np.float32)
    SK64 = np.empty((B, F), np.float64)
    _check(lib().sk_oracle_combine(_p(S1, C.c_uint32), _p(S2, C.c_uint32), B, F, E, M,
                                   _p(sub, C.c_uint8), int(first_n or 0), _p(SK, C.c_float),
                                   _p(SK64, C.c_double)), "combine")
    return (SK, SK64) if want64 else SK


def flag(SK, M, N, n_sigma, sk_mean=1.0):
    """PAPER.md:183 with PAPER.md:119 Eq. 16.  SK float32 [B][F] -> mask uint8 [B][F]."""
    SK = np.ascontiguousarray(SK, dtype=np.float32)
    B, F = SK.shape
    mask = np.empty((B, F), np.uint8)
    _check(lib().sk_oracle_flag(_p(SK, C.c_float), B, F, M, N, C.c_float(n_sigma),
                                C.c_float(sk_mean), _p(mask, C.c_uint8)), "flag")
    return mask


def frame(data, M, subset=None, first_n=None, n_sigma=3.0, sk_mean=1.0, zero_flagged=False):
    """The whole path.  Returns dict(SK, mask, S1, S2, data) — data is a copy, excised if asked."""
    data = np.array(data, dtype=np.uint8, order="C", copy=True)
    T, F, E = data.shape
    sub = _subset(subset, E)
    if sub is None and first_n is None:
        first_n = E
    B = T // M if M else 0
    SK = np.empty((B, F), np.float32)
    mask = np.empty((B, F), np.uint8)
    S1 = np.empty((B, F, E), np.uint32)
    S2 = np.empty_like(S1)
    t1 = np.empty_like(S1)
    t2 = np.empty_like(S1)
    _check(lib().sk_oracle_frame(_p(data, C.c_uint8), T, F, E, M, _p(sub, C.c_uint8),
                                 int(first_n or 0), C.c_float(n_sigma), C.c_float(sk_mean),
                                 int(bool(zero_flagged)), _p(SK, C.c_float), _p(mask, C.c_uint8),
                                 _p(S1, C.c_uint32), _p(S2, C.c_uint32), _p(t1, C.c_uint32),
                                 _p(t2, C.c_uint32)), "frame")
    return dict(SK=SK, mask=mask, S1=S1, S2=S2, data=data)


def single(S1, S2, M):
    """PAPER.md:48 Eq. 2 / :80 Eq. 8 for one receiver (scalars)."""
    return lib().sk_oracle_single(float(S1), float(S2), float(M))


def singles(S1, S2, M):
    """PAPER.md:80 Eq. 8 per receiver as an output: float32 [B][F][E] (0 where S1 == 0)."""
    S1 = np.ascontiguousarray(S1, dtype=np.uint32)
    S2 = np.ascontiguousarray(S2, dtype=np.uint32)
    B, F, E = S1.shape
    out = np.empty((B, F, E), dtype=np.float32)
    _check(lib().sk_oracle_singles(_p(S1, C.c_uint32), _p(S2, C.c_uint32), B, F, E, int(M), _p(out, C.c_float)),
           "sk_oracle_singles")
    return out


def significance(SK, M, N, sk_mean=1.0):
    """PAPER.md:183 detection significance: (SK - sk_mean) / sqrt(4/(M N)), float32 [B][F]."""
    SK = np.ascontiguousarray(SK, dtype=np.float32)
    B, F = SK.shape
    out = np.empty((B, F), dtype=np.float32)
    _check(lib().sk_oracle_significance(_p(SK, C.c_float), B, F, int(M), int(N), C.c_float(sk_mean),
                                        _p(out, C.c_float)), "sk_oracle_significance")
    return out


def average_of_singles(S1, S2, M, subset=None, first_n=None):
    """PAPER.md:112 Eq. 14, third line: the mean of the per-receiver Eq. 8 estimates (float64)."""
    S1 = np.ascontiguousarray(S1, dtype=np.uint32)
    S2 = np.ascontiguousarray(S2, dtype=np.uint32)
    B, F, E = S1.shape
    sub = _subset(subset, E)
    if sub is None and first_n is None:
        first_n = E
    out = np.empty((B, F), np.float64)
    _check(lib().sk_oracle_average_of_singles(_p(S1, C.c_uint32), _p(S2, C.c_uint32), B, F, E, M,
                                              _p(sub, C.c_uint8), int(first_n or 0),
                                              _p(out, C.c_double)), "average_of_singles")
    return out


def eq13_and_s1bar(S1, S2, M, subset=None, first_n=None):
    """PAPER.md:97 Eq. 13 (un-rescaled), :86 Eq. 10 S1bar, :88 Eq. 11 S2bar (all float64)."""
    S1 = np.ascontiguousarray(S1, dtype=np.uint32)
    S2 = np.ascontiguousarray(S2, dtype=np.uint32)
    B, F, E = S1.shape
    sub = _subset(subset, E)
    if sub is None and first_n is None:
        first_n = E
    sk13 = np.empty((B, F), np.float64)
    s1bar = np.empty((B, F), np.float64)
    s2bar = np.empty((B, F), np.float64)
    _check(lib().sk_oracle_eq13_and_s1bar(_p(S1, C.c_uint32), _p(S2, C.c_uint32), B, F, E, M,
                                          _p(sub, C.c_uint8), int(first_n or 0),
                                          _p(sk13, C.c_double), _p(s1bar, C.c_double),
                                          _p(s2bar, C.c_double)), "eq13_and_s1bar")
    return sk13, s1bar, s2bar


def frame_float(re, im, M, subset=None, first_n=None):
    """Float-input path (no quantisation): re, im float64 [T][F][E] -> SK float64 [B][F], S1, S2."""
    re = np.ascontiguousarray(re, dtype=np.float64)
    im = np.ascontiguousarray(im, dtype=np.float64)
    T, F, E = re.shape
    assert im.shape == re.shape
    sub = _subset(subset, E)
    if sub is None and first_n is None:
        first_n = E
    B = T // M if M else 0
    SK = np.empty((B, F), np.float64)
    S1 = np.empty((B, F, E), np.float64)
    S2 = np.empty_like(S1)
    _check(lib().sk_oracle_frame_float(_p(re, C.c_double), _p(im, C.c_double), T, F, E, M,
                                       _p(sub, C.c_uint8), int(first_n or 0), _p(SK, C.c_double),
                                       _p(S1, C.c_double), _p(S2, C.c_double)), "frame_float")
    return SK, S1, S2


def philox(ctr, key):
    """Philox4x32-10 (Salmon et al., SC'11): 4 counter words, 2 key words -> 4 output words."""
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.empty(4, dtype=np.uint32)
    _check(lib().sk_oracle_philox(_p(ctr, C.c_uint32), _p(key, C.c_uint32), _p(out, C.c_uint32)), "sk_oracle_philox")
    return out


def sim_digitised(T, F, E, thr, seed, frame=0):
    """PAPER.md:276-284 (App. B): seeded 4+4-bit round-and-clip Gaussian bytes [T][F][E] from the
    per-receiver thresholds thr uint32 [E][14]."""
    thr = np.ascontiguousarray(thr, dtype=np.uint32)
    assert thr.shape == (E, 14)
    data = np.empty((T, F, E), dtype=np.uint8)
    _check(lib().sk_oracle_sim_digitised(_p(data, C.c_uint8), T, F, E, _p(thr, C.c_uint32),
                                         C.c_uint64(seed), C.c_uint64(frame)), "sk_oracle_sim_digitised")
    return data


def moments(SK):
    """Mean and unbiased variance of SK over the blocks, per frequency (float64 [F] each)."""
    SK = np.ascontiguousarray(SK, dtype=np.float32)
    B, F = SK.shape
    mean = np.empty(F, dtype=np.float64)
    var = np.empty(F, dtype=np.float64)
    _check(lib().sk_oracle_moments(_p(SK, C.c_float), B, F, _p(mean, C.c_double), _p(var, C.c_double)),
           "sk_oracle_moments")
    return mean, var


def gauss_pair(w0, w1):
    """Box-Muller: two 32-bit words -> one circular complex Gaussian (re, im), unit variance each."""
    out = np.empty(2, dtype=np.float64)
    _check(lib().sk_oracle_gauss_pair(C.c_uint32(int(w0)), C.c_uint32(int(w1)), _p(out, C.c_double)), "gauss_pair")
    return out


def sim_common_mode(D, M, N, amp, seed, want_x=False):
    """PAPER.md:262-272 (App. A): D datasets of M samples x N receivers of unit Gaussian noise plus
    amp x a common-mode Gaussian; returns SK~ per dataset (float64 [D]) and optionally the samples
    complex128 [D][M][N]."""
    SK = np.empty(D, dtype=np.float64)
    x = np.empty((D, M, N, 2), dtype=np.float64) if want_x else None
    _check(lib().sk_oracle_sim_common_mode(D, M, N, C.c_double(amp), C.c_uint64(seed), _p(SK, C.c_double),
                                           _p(x, C.c_double)), "sk_oracle_sim_common_mode")
    return (SK, x[..., 0] + 1j * x[..., 1]) if want_x else SK
