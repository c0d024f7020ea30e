"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test is chosen so that a plausible mistake in oracle/sk_oracle.cpp (a dropped term, a wrong
sign, index or offset, un-normalised pooling, Eq. 13 instead of Eq. 14) fails at least one.
PAPER.md line numbers refer to /root/reference/PAPER.md (arXiv 1808.10365).
"""
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def enc(re, im):
    """Encode integer components in [-8, 7] (test-side helper; the inverse of the method's a1)."""
    return (((np.asarray(re) + 8) << 4) | (np.asarray(im) + 8)).astype(np.uint8)


# ---------------------------------------------------------------------------------------- P7
def test_hand_example_golden(oracle):
    """Hand-worked sums, tests/golden/hand_example.txt (PAPER.md:77 Eq. 7, :108-113 Eq. 14)."""
    kv = {}
    for line in open(os.path.join(GOLDEN, "hand_example.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        kv[k] = v
    M, E = int(kv["M"][0]), int(kv["E"][0])
    data = np.array([int(x, 16) for x in kv["data"]], np.uint8).reshape(M, 1, E)
    S1, S2 = oracle.power_sums(data, M)
    assert S1.ravel().tolist() == [int(x) for x in kv["S1"]]
    assert S2.ravel().tolist() == [int(x) for x in kv["S2"]]
    sk2, sk64 = oracle.combine(S1, S2, M, want64=True)
    assert sk64[0, 0] == float(kv["SK_N2"][0])          # 0.3125 is exact in binary
    assert sk2[0, 0] == np.float32(kv["SK_N2"][0])
    assert oracle.combine(S1, S2, M, first_n=1)[0, 0] == np.float32(kv["SK_input0"][0])
    assert oracle.combine(S1, S2, M, subset=[0, 1])[0, 0] == np.float32(kv["SK_input1"][0])
    assert oracle.single(8, 22, 4) == 0.625             # Eq. 2 on the same sums


def test_decode_offsets(oracle):
    """a1: value = nibble - 8, nibble 0 decodes to -8 (reading A3), 0x88 is zero."""
    M = 2
    for byte, p in [(0x88, 0), (0x00, 128), (0xFF, 98), (0x80, 64), (0x08, 64), (0x8F, 49),
                    (0xF8, 49), (0x97, 2), (0x11, 98), (0x10, 49 + 64)]:
        data = np.full((M, 1, 1), byte, np.uint8)
        S1, S2 = oracle.power_sums(data, M)
        assert (S1[0, 0, 0], S2[0, 0, 0]) == (M * p, M * p * p), hex(byte)


# ---------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("M,E", [(4, 1), (64, 16), (256, 256), (1024, 48)])
def test_constant_modulus_gives_exactly_zero(oracle, M, E):
    """A constant-modulus signal has M*S2/S1^2 = 1 exactly, so Eq. 2 / Eq. 14 give 0 exactly."""
    rng = np.random.default_rng(1)
    pts = np.array([(5, 0), (-5, 0), (0, 5), (0, -5), (3, 4), (-3, 4), (3, -4), (-3, -4),
                    (4, 3), (-4, 3), (4, -3), (-4, -3)])
    k = rng.integers(0, len(pts), size=(3 * M, 2, E))
    data = enc(pts[k, 0], pts[k, 1])
    r = oracle.frame(data, M)
    assert (r["S1"] == 25 * M).all() and (r["S2"] == 625 * M).all()
    assert (r["SK"] == 0.0).all()
    # |0 - 1| is outside 3 sigma exactly when 3*sqrt(4/(MN)) < 1
    assert (r["mask"] == (1 if 3 * math.sqrt(4 / (M * E)) < 1 else 0)).all()


# ---------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("scale,lim", [(2, 3), (3, 2)])
def test_scale_invariance_is_exact(oracle, scale, lim):
    """'overall-scaling-invariant': S2/S1^2 is a ratio of degree-4 forms, and on the
    integer grid scaling by k multiplies both exactly, so SK64 is bit-identical."""
    rng = np.random.default_rng(2)
    M, F, E = 32, 3, 24
    re = rng.integers(-lim, lim + 1, size=(4 * M, F, E))
    im = rng.integers(-lim, lim + 1, size=(4 * M, F, E))
    re[:, :, 0] = np.where(re[:, :, 0] == 0, 1, re[:, :, 0])     # keep every input's power > 0
    a = oracle.frame(enc(re, im), M)
    b = oracle.frame(enc(scale * re, scale * im), M)
    assert (b["S1"] == scale ** 2 * a["S1"]).all() and (b["S2"] == scale ** 4 * a["S2"]).all()
    ska = oracle.combine(a["S1"], a["S2"], M, want64=True)[1]
    skb = oracle.combine(b["S1"], b["S2"], M, want64=True)[1]
    # the quotient M^2 S2 / S1^2 is the same real number; both operand pairs are exact in double
    np.testing.assert_array_equal(ska, skb)


# ---------------------------------------------------------------------------- P3, P4, P5, Eq. 12
def test_paper_identities(oracle):
    """S1bar = nN (Eq. 10), Eq. 12, Eq. 14's second and third lines agree, Eq. 13/14 ratio."""
    rng = np.random.default_rng(3)
    M, F, E = 64, 2, 40
    data = rng.integers(0, 256, size=(5 * M, F, E), dtype=np.uint8)
    S1, S2 = oracle.power_sums(data, M)
    for kw in (dict(), dict(first_n=7), dict(subset=(np.arange(E) % 3 == 1))):
        N = E if not kw else (7 if "first_n" in kw else int(np.count_nonzero(kw["subset"])))
        sk32, sk = oracle.combine(S1, S2, M, want64=True, **kw)
        avg = oracle.average_of_singles(S1, S2, M, **kw)
        sk13, s1bar, s2bar = oracle.eq13_and_s1bar(S1, S2, M, **kw)
        np.testing.assert_allclose(s1bar, M * N, rtol=1e-13)                       # Eq. 10
        np.testing.assert_allclose(sk, avg, rtol=1e-12, atol=1e-14)                # Eq. 14 l.2 = l.3
        np.testing.assert_allclose(s2bar, M * (M - 1) / (M + 1) * N * avg + M * N,
                                   rtol=1e-12)                                     # Eq. 12
        ratio = (M * N + 1) * (M - 1) / ((M * N - 1) * (M + 1))
        np.testing.assert_allclose(sk13, ratio * sk, rtol=1e-12)                   # Eq. 13 vs 14
        np.testing.assert_array_equal(sk32, sk.astype(np.float32))


def test_n1_reduces_to_single_receiver(oracle):
    """N = 1: Eq. 14 is Eq. 2."""
    rng = np.random.default_rng(4)
    M = 16
    data = rng.integers(0, 256, size=(3 * M, 1, 5), dtype=np.uint8)
    S1, S2 = oracle.power_sums(data, M)
    for e in range(5):
        sub = np.arange(5) == e
        sk = oracle.combine(S1, S2, M, subset=sub, want64=True)[1]
        for b in range(3):
            assert sk[b, 0] == pytest.approx(oracle.single(S1[b, 0, e], S2[b, 0, e], M), rel=1e-14)


def test_singles_output(oracle):
    """NEXT-4: the per-receiver output is Eq. 8 element by element: the hand example's 0.625 and 0
    (tests/golden/hand_example.txt), exact Fractions on random bytes, N = 1 combine, and its mean
    over the receivers is Eq. 14 (PAPER.md:112 third line)."""
    from fractions import Fraction
    M = 4
    data = np.array([[0x98, 0x99], [0x99, 0x99], [0x86, 0x99], [0x87, 0x99]], dtype=np.uint8).reshape(4, 1, 2)
    S1, S2 = oracle.power_sums(data, M)
    np.testing.assert_array_equal(oracle.singles(S1, S2, M)[0, 0], np.float32([0.625, 0.0]))
    rng = np.random.default_rng(8)
    M, E = 12, 7
    data = rng.integers(0, 256, size=(2 * M, 2, E), dtype=np.uint8)
    data[:M, 0, 3] = 0x88                                   # a dead receiver: 0 (reading A4)
    S1, S2 = oracle.power_sums(data, M)
    got = oracle.singles(S1, S2, M)
    for b in range(2):
        for f in range(2):
            for e in range(E):
                s1, s2 = int(S1[b, f, e]), int(S2[b, f, e])
                want = Fraction(0) if s1 == 0 else Fraction(M + 1, M - 1) * (Fraction(M * s2, s1 * s1) - 1)
                assert got[b, f, e] == np.float32(float(want))
    assert got[0, 0, 3] == 0.0
    sk64 = oracle.combine(S1, S2, M, want64=True)[1]
    np.testing.assert_allclose(got.astype(np.float64).mean(axis=2), sk64, rtol=0, atol=2e-7)


def test_significance(oracle):
    """a value k spreads away from the mean has significance k; the flag at
    threshold a is |significance| > a (same cells as oracle.flag away from the boundary)."""
    M, N, mean = 256, 2048, 0.94
    sd = np.sqrt(4.0 / (M * N))
    k = np.array([[-7.5, -3.0, -0.25, 0.0, 0.5, 2.999, 3.001, 12.0]])
    SK = (mean + k * sd).astype(np.float32)
    sig = oracle.significance(SK, M, N, sk_mean=mean)
    np.testing.assert_allclose(sig, k, rtol=0, atol=2e-4)          # float32 SK carries ~1e-4 sigma
    assert np.array_equal(np.abs(sig) > 3.0, oracle.flag(SK, M, N, 3.0, sk_mean=mean).astype(bool))
    assert np.isnan(oracle.significance(np.float32([[np.nan]]), M, N)[0, 0])


def test_integration_lengths_from_sums(oracle):
    """NEXT-2 ("a variety of integration lengths"): Eq. 7's sums over a block of
    k*M samples are the sums of its k sub-blocks, so S1, S2 at M re-binned by k equal S1, S2
    computed at k*M from the data: exact integers."""
    rng = np.random.default_rng(9)
    M, F, E = 8, 2, 5
    data = rng.integers(0, 256, size=(12 * M, F, E), dtype=np.uint8)
    S1, S2 = oracle.power_sums(data, M)
    for k in (2, 3, 4, 6):
        T1, T2 = oracle.power_sums(data, k * M)
        np.testing.assert_array_equal(S1.reshape(12 // k, k, F, E).sum(axis=1, dtype=np.uint64), T1)
        np.testing.assert_array_equal(S2.reshape(12 // k, k, F, E).sum(axis=1, dtype=np.uint64), T2)


def test_two_level_closed_form(oracle):
    """A receiver alternating between powers a and b has M S2/S1^2 = 2(a^2+b^2)/(a+b)^2:
    with a=1 (0x98), b=4 (0xA8): 2*17/25 = 1.36, SK = (M+1)/(M-1)*0.36."""
    M = 10
    data = np.array([0x98, 0xA8] * (M // 2), np.uint8).reshape(M, 1, 1)
    sk = oracle.frame(data, M)["SK"][0, 0]
    assert sk == np.float32(11 / 9 * 0.36)


# --------------------------------------------------------------------------------------- P12
def brute(data, M, sel):
    """Differently structured: per-input Eq. 8 with Python ints/Fractions, then the average."""
    from fractions import Fraction
    T, F, E = data.shape
    out = np.zeros((T // M, F))
    for b in range(T // M):
        for f in range(F):
            tot = Fraction(0)
            for e in sel:
                ps = []
                for t in range(b * M, (b + 1) * M):
                    byte = int(data[t, f, e])
                    hi, lo = divmod(byte, 16)
                    ps.append((hi - 8) ** 2 + (lo - 8) ** 2)
                s1, s2 = sum(ps), sum(p * p for p in ps)
                if s1:
                    tot += Fraction(M + 1, M - 1) * (Fraction(M * s2, s1 * s1) - 1)
            out[b, f] = float(tot / len(sel))
    return out


@pytest.mark.parametrize("M,E", [(2, 1), (3, 4), (8, 8), (5, 7)])
def test_brute_force_tiny(oracle, M, E):
    rng = np.random.default_rng(100 + M)
    data = rng.integers(0, 256, size=(4 * M, 2, E), dtype=np.uint8)
    data[:, 0, 0] = 0x88                  # a dead input (reading A4)
    data[:M, 1, :] = rng.choice([0x00, 0x08, 0x80, 0x88, 0xFF], size=(M, E))  # nibble 0 = -8
    for sel in (list(range(E)), list(range(0, E, 2))):
        sub = np.isin(np.arange(E), sel)
        sk = oracle.combine(*oracle.power_sums(data, M), M, subset=sub, want64=True)[1]
        np.testing.assert_allclose(sk, brute(data, M, sel), rtol=1e-13, atol=1e-14)


def test_all_zero_cell_is_zero_and_flagged(oracle):
    """Reading A4: an all-0x88 cell gives SK = 0 exactly (no NaN) and is flagged."""
    data = np.full((128, 2, 16), 0x88, np.uint8)
    r = oracle.frame(data, 64)
    assert (r["SK"] == 0).all() and (r["mask"] == 1).all() and not np.isnan(r["SK"]).any()


# --------------------------------------------------------------------------------------- P11
def test_permutations(oracle):
    rng = np.random.default_rng(5)
    M, F, E = 32, 2, 64
    data = rng.integers(0, 256, size=(2 * M, F, E), dtype=np.uint8)
    S1, S2 = oracle.power_sums(data, M)
    shuf = data.copy()
    for b in range(2):
        shuf[b * M:(b + 1) * M] = data[b * M + rng.permutation(M)]
    S1s, S2s = oracle.power_sums(shuf, M)
    assert (S1 == S1s).all() and (S2 == S2s).all()          # time order inside a block is irrelevant
    perm = rng.permutation(E)
    a = oracle.combine(S1, S2, M, want64=True)[1]
    b = oracle.combine(S1[:, :, perm], S2[:, :, perm], M, want64=True)[1]
    np.testing.assert_allclose(a, b, rtol=1e-13)             # input order: only rounding changes
    swapped = data.copy()
    swapped[:M], swapped[M:] = data[M:], data[:M]            # blocks are independent (A10)
    c = oracle.frame(swapped, M)["SK"]
    np.testing.assert_array_equal(c[::-1], oracle.frame(data, M)["SK"])


# ---------------------------------------------------------------------------------------- P8
def _gauss(rng, T, F, E, sig):
    return rng.standard_normal((T, F, E)) * sig, rng.standard_normal((T, F, E)) * sig


@pytest.mark.parametrize("M,N,cells", [(64, 8, 20000), (256, 4, 6000)])
def test_null_moments_float_input(oracle, M, N, cells):
    """Circular Gaussian input: mean(SK~) = 1 (Eq. 15), var(SK~) = 4/(nN) + O(1/(n^2 N)) (Eq. 16).
    Per-input sigma varies by 2.3x, so pooling un-normalised sums would fail this test."""
    rng = np.random.default_rng(8)
    sig = rng.uniform(1.5, 3.5, size=N)
    re, im = _gauss(rng, M * cells, 1, N, sig)
    sk = oracle.frame_float(re, im, M)[0].ravel()
    first = 4.0 / (M * N)
    se_mean = math.sqrt(first / cells)
    assert abs(sk.mean() - 1.0) < 4 * se_mean
    # exact Gaussian-input variance is 4 M^2 / ((M-1)(M+2)(M+3) N): first order minus O(1/M)
    ratio = sk.var(ddof=1) / first
    expected = M ** 3 / ((M - 1) * (M + 2) * (M + 3))
    assert abs(ratio - expected) < 4 * math.sqrt(2.0 / cells) + 0.01
    assert abs(ratio - 1.0) < 6.0 / M + 4 * math.sqrt(2.0 / cells)      # "to first order"
    # the wrong estimator (Eq. 13, un-rescaled) is biased low by (nN+1)(n-1)/((nN-1)(n+1))
    assert abs(sk.mean() * (M * N + 1) * (M - 1) / ((M * N - 1) * (M + 1)) - 1.0) > 4 * se_mean


def test_unnormalised_pooling_would_fail(oracle):
    """Control for P8: pooling raw S1, S2 across receivers of unequal power is NOT mean-1."""
    rng = np.random.default_rng(9)
    M, N, cells = 64, 8, 4000
    sig = np.linspace(1.0, 4.0, N)
    re, im = _gauss(rng, M * cells, 1, N, sig)
    sk, S1, S2 = oracle.frame_float(re, im, M)
    pooled = (M * N + 1) / (M * N - 1) * (M * N * S2.sum(-1) / S1.sum(-1) ** 2 - 1)
    assert abs(pooled.mean() - 1.0) > 0.3 and abs(sk.mean() - 1.0) < 0.01


def test_frame_float_layout_at_several_frequencies(oracle):
    """The float-input entry at F > 1 (its [t][f][e] indexing): integer-valued doubles decoded from
    random bytes with numpy (not with the oracle) must reproduce the byte entry's S1, S2 exactly
    (exact integers in float64) and its SK, subset included; and a frequency must see only its own
    samples (changing f = 1 leaves f = 0 and f = 2 bit-identical)."""
    rng = np.random.default_rng(21)
    T, F, E, M = 96, 3, 10, 24
    data = rng.integers(0, 256, size=(T, F, E), dtype=np.uint8)
    re = (data >> 4).astype(np.float64) - 8.0
    im = (data & 15).astype(np.float64) - 8.0
    S1, S2 = oracle.power_sums(data, M)
    for kw in ({}, {"first_n": 7}, {"subset": np.arange(E) % 3 != 0}):
        sk, f1, f2 = oracle.frame_float(re, im, M, **kw)
        assert np.array_equal(f1, S1.astype(np.float64)) and np.array_equal(f2, S2.astype(np.float64))
        ref = oracle.combine(S1, S2, M, want64=True, **kw)[1]
        assert np.array_equal(sk, ref)
    # hand sums of one cell from the definition (Eq. 7), straight from re/im
    b, f, e = 2, 1, 4
    pw = re[b * M:(b + 1) * M, f, e] ** 2 + im[b * M:(b + 1) * M, f, e] ** 2
    sk, f1, f2 = oracle.frame_float(re, im, M)
    assert f1[b, f, e] == pw.sum() and f2[b, f, e] == (pw ** 2).sum()
    re2, im2 = re.copy(), im.copy()
    re2[:, 1, :] += 1.0
    sk2 = oracle.frame_float(re2, im2, M)[0]
    assert np.array_equal(sk2[:, 0], sk[:, 0]) and np.array_equal(sk2[:, 2], sk[:, 2])
    assert not np.array_equal(sk2[:, 1], sk[:, 1])


# ---------------------------------------------------------------------------------------- P9
def test_skew_and_kurtosis_single_receiver(oracle):
    """N = 1: skew ~ 10/sqrt(M), excess kurtosis ~ 246/M to first order."""
    rng = np.random.default_rng(10)
    M, cells = 128, 100000
    re, im = _gauss(rng, M * cells // 50, 1, 50, 2.0)      # 50 independent receivers, used singly
    _, S1, S2 = oracle.frame_float(re, im, M)
    sk = (M + 1) / (M - 1) * (M * S2 / S1 ** 2 - 1)
    sk = sk.ravel()
    assert sk.size == cells
    d = sk - sk.mean()
    skew = (d ** 3).mean() / (d ** 2).mean() ** 1.5
    kurt = (d ** 4).mean() / (d ** 2).mean() ** 2 - 3.0
    assert abs(sk.mean() - 1) < 4 * math.sqrt(4 / M / cells)
    assert abs(sk.var() / (4 / M) - 1) < 0.08
    assert abs(skew / (10 / math.sqrt(M)) - 1) < 0.30
    assert abs(kurt / (246 / M) - 1) < 0.35


# --------------------------------------------------------------------------------------- P10
def test_digitised_offset_is_constant_in_N(oracle):
    """App. B: 4+4-bit data, RMS 1.52 LSB, clipped to +-7: the mean of SK~
    converges to a constant slightly off 1 for all N, the variance to the float-input value."""
    rng = np.random.default_rng(11)
    M, E, cells = 256, 64, 1500
    re = np.clip(np.rint(rng.standard_normal((M * cells, 1, E)) * 1.52), -7, 7).astype(int)
    im = np.clip(np.rint(rng.standard_normal((M * cells, 1, E)) * 1.52), -7, 7).astype(int)
    S1, S2 = oracle.power_sums(enc(re, im), M)
    means = {}
    for N in (4, 16, 64):
        sk = oracle.combine(S1, S2, M, first_n=N, want64=True)[1].ravel()
        means[N] = sk.mean()
        se = math.sqrt(4 / (M * N) / cells)
        assert abs(sk.mean() - 1) < 0.01                      # "slightly offset from unity"
        assert abs(sk.var() / (4 / (M * N)) - 1) < 0.15       # variance as in the float case
        assert abs(means[N] - means[4]) < 5 * math.sqrt(4 / (M * 4) / cells) + se
    assert means[64] < 1.0                                    # the offset is real (about -1e-3)
    # large-M limit from the quantised pmf alone: E[p^2]/E[p]^2 - 1 (finite-M bias is O(1/M))
    assert abs(means[64] - _quantised_limit(1.52)) < 4 * math.sqrt(4 / (M * 64) / cells) + 2.0 / M


def _quantised_limit(sigma):
    """E[p^2]/E[p]^2 - 1 for p = re^2 + im^2 with re, im iid rounded-and-clipped N(0, sigma^2):
    computed from the normal cdf, with no reference to the estimator's code."""
    k = np.arange(-7, 8)
    cdf = lambda x: 0.5 * (1 + np.vectorize(math.erf)(x / (sigma * math.sqrt(2))))
    pmf = cdf(k + 0.5) - cdf(k - 0.5)
    pmf[0] += cdf(-7.5)
    pmf[-1] += 1 - cdf(7.5)
    m2, m4 = (pmf * k ** 2).sum(), (pmf * k ** 4).sum()
    return (2 * m4 + 2 * m2 * m2) / (2 * m2) ** 2 - 1


def test_digitised_mean_matches_pmf_prediction(oracle):
    """sigma = 2.5 LSB clipped at +-7 (configs 0 and 3): the null mean of SK~ on 4-bit data sits
    well below 1 (about 0.94); its large-M limit follows from the quantised pmf."""
    rng = np.random.default_rng(13)
    M, E, cells = 256, 128, 400
    re = np.clip(np.rint(rng.standard_normal((M * cells, 1, E)) * 2.5), -7, 7).astype(int)
    im = np.clip(np.rint(rng.standard_normal((M * cells, 1, E)) * 2.5), -7, 7).astype(int)
    sk = oracle.frame(enc(re, im), M)["SK"].ravel().astype(np.float64)
    lim = _quantised_limit(2.5)
    assert 0.92 < lim < 0.96
    assert abs(sk.mean() - lim) < 4 * math.sqrt(4 / (M * E) / cells) + 2.0 / M


# -------------------------------------------------------------------------------------- flag
def test_flag_interval(oracle):
    """flagged iff outside mean +- a*sqrt(var); var = 4/(nN) (Eq. 16); strict; NaN."""
    M, N, a = 256, 2048, 5.0
    s = math.sqrt(4.0 / (M * N))
    mean = 0.9985
    SK = np.array([[mean, mean + 4.99 * s, mean + 5.01 * s, mean - 4.99 * s, mean - 5.01 * s,
                    np.nan, np.inf, 0.0, 2.0]], np.float32)
    m = oracle.flag(SK, M, N, a, sk_mean=mean)
    assert m.tolist() == [[0, 0, 1, 0, 1, 1, 1, 1, 1]]
    thr = np.float32(a * s)
    edge = np.array([[np.float32(1.0) + thr, np.float32(1.0) - thr]], np.float32)
    dev = np.abs(edge - np.float32(1.0))
    assert (oracle.flag(edge, M, N, a, sk_mean=1.0) == (dev > thr)).all()     # strict, in float32
    # the width scales as 1/sqrt(N): 4x the receivers, half the interval
    assert oracle.flag(np.array([[1 + 2.6 * s]], np.float32), M, N, a)[0, 0] == 0
    assert oracle.flag(np.array([[1 + 2.6 * s]], np.float32), M, 4 * N, a)[0, 0] == 1


def test_frame_excision(oracle):
    """Reading A11: flagged cells (all E inputs, all M rows) become 0x88, others are untouched;
    mask and SK come from the data before excision; a second pass is idempotent (A4)."""
    rng = np.random.default_rng(12)
    M, F, E = 64, 3, 32
    re = np.clip(np.rint(rng.standard_normal((4 * M, F, E)) * 1.5), -7, 7).astype(int)
    im = np.clip(np.rint(rng.standard_normal((4 * M, F, E)) * 1.5), -7, 7).astype(int)
    re[M:2 * M, 1, :] = 5
    im[M:2 * M, 1, :] = 0                                     # cell (1,1): constant modulus
    data = enc(re, im)
    null_mean = float(oracle.frame(data, M)["SK"][[0, 2, 3]].mean())
    r = oracle.frame(data, M, n_sigma=6.0, sk_mean=null_mean, zero_flagged=True)
    assert r["mask"][1, 1] == 1 and r["mask"].sum() == 1
    expect = data.copy()
    expect[M:2 * M, 1, :] = 0x88
    np.testing.assert_array_equal(r["data"], expect)
    plain = oracle.frame(data, M, n_sigma=6.0, sk_mean=null_mean)
    np.testing.assert_array_equal(plain["SK"], r["SK"])
    np.testing.assert_array_equal(plain["data"], data)
    again = oracle.frame(r["data"], M, n_sigma=6.0, sk_mean=null_mean, zero_flagged=True)
    assert again["SK"][1, 1] == 0 and again["mask"][1, 1] == 1
    np.testing.assert_array_equal(again["data"], r["data"])


def test_bad_arguments(oracle):
    d = np.zeros((8, 1, 4), np.uint8)
    with pytest.raises(ValueError):
        oracle.power_sums(d, 3)            # T % M != 0
    with pytest.raises(ValueError):
        oracle.power_sums(d, 1)            # M < 2
    S1, S2 = oracle.power_sums(d, 4)
    with pytest.raises(ValueError):
        oracle.combine(S1, S2, 4, first_n=5)   # N > E
    with pytest.raises(ValueError):
        oracle.combine(S1, S2, 4, subset=[0, 0, 0, 0])   # N == 0


# ---- App. B digitisation simulation ---------------------
def _philox_py(ctr, key):
    """Philox4x32-10 written out independently of the oracle (Salmon et al., SC'11, section 3.3):
    ten rounds of two 32x32->64 multiplies by fixed constants, crossed with the key, which is
    bumped by the Weyl constants every round."""
    c = [int(x) for x in ctr]
    k = [int(x) for x in key]
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_philox_known_answers(oracle):
    """The published known-answer vectors of Philox4x32-10 (Random123 distribution, kat_vectors:
    zero counter and key; all-ones; the digits of pi)."""
    kat = [
        ([0, 0, 0, 0], [0, 0], [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]),
        ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2, [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]),
        ([0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344], [0xA4093822, 0x299F31D0],
         [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]),
    ]
    for ctr, key, want in kat:
        assert [int(x) for x in oracle.philox(ctr, key)] == want
        assert _philox_py(ctr, key) == want


def test_sim_digitised_layout_and_pmf(oracle):
    """Counter layout and threshold rule element by element (independent Philox), then the
    empirical distribution against the model's exact probabilities and RMS."""
    import sk_synth
    T, F, E = 6, 2, 5
    sig = np.array([0.7, 1.52, 2.5, 3.5, 9.0])
    thr = sk_synth.digitiser_thresholds(sig).numpy().astype(np.uint32)
    seed, frame = 0x123456789ABCDEF, 3
    data = oracle.sim_digitised(T, F, E, thr, seed, frame)
    for t in range(T):
        for f in range(F):
            for e in range(E):
                w = _philox_py([e // 2, t * F + f, frame & 0xFFFFFFFF, frame >> 32], [seed & 0xFFFFFFFF, seed >> 32])
                re = -7 + sum(int(w[2 * (e & 1)] >= x) for x in thr[e])
                im = -7 + sum(int(w[2 * (e & 1) + 1] >= x) for x in thr[e])
                assert data[t, f, e] == ((re + 8) << 4) | (im + 8)
    assert not np.array_equal(data, oracle.sim_digitised(T, F, E, thr, seed, frame + 1))
    # statistics: 2 x 400k components per receiver
    T = 100000
    data = oracle.sim_digitised(T, 4, 3, thr[1:4], seed=7)
    comp = np.stack([(data >> 4).astype(int) - 8, (data & 15).astype(int) - 8])       # [2][T][4][3]
    assert comp.min() >= -7 and comp.max() <= 7
    from math import erf, sqrt
    for i, s_ in enumerate(sig[1:4]):
        cdf = [0.0] + [0.5 * (1 + erf((j - 6.5) / s_ / sqrt(2))) for j in range(14)] + [1.0]
        pmf = np.diff(cdf)
        x = comp[..., i].ravel()
        n = x.size
        freq = np.bincount(x + 7, minlength=15) / n
        assert (np.abs(freq - pmf) < 5 * np.sqrt(pmf * (1 - pmf) / n) + 2e-9).all()
        rms_model = np.sqrt((pmf * np.arange(-7, 8) ** 2).sum())
        assert abs(np.sqrt((x.astype(float) ** 2).mean()) - rms_model) < 0.01
    # the paper's operating point: RMS ~1.52 LSB per component
    pmf152 = np.diff([0.0] + [0.5 * (1 + erf((j - 6.5) / 1.52 / sqrt(2))) for j in range(14)] + [1.0])
    assert abs(np.sqrt((pmf152 * np.arange(-7, 8) ** 2).sum()) - 1.52) < 0.04


def test_digitiser_thresholds_exact():
    """sk_synth.digitiser_thresholds is App. B's input model (components rounded to the
    nearest level and bounded to [-7, 7]) and feeds BOTH simulators, so neither parity test can see a
    mistake in it.  Pin it on its own, exactly: thr[e][k] = floor(2^32 Phi((k - 6.5) / sigma_e)), Phi from
    math.erfc (not the torch routine the table is built with).  An edge off by one level (k - 7.5,
    k - 5.5) moves a threshold by ~1e8; the comparison allows 1 count for the last bit of Phi."""
    import sk_synth
    from math import erfc, floor, sqrt
    sig = [0.7, 1.0, 1.52, 2.5, 3.5, 9.0]
    thr = sk_synth.digitiser_thresholds(sig).numpy().astype(np.int64)
    assert thr.shape == (len(sig), 14)
    exact = 0
    for e, s_ in enumerate(sig):
        for k in range(14):
            want = floor(4294967296.0 * 0.5 * erfc(-(k - 6.5) / s_ / sqrt(2.0)))
            assert abs(int(thr[e, k]) - want) <= 1, (s_, k, int(thr[e, k]), want)
            exact += int(thr[e, k]) == want
        assert (np.diff(thr[e]) >= 0).all() and (np.diff(thr[e, 3:11]) > 0).all()   # ascending (the tails saturate for a small sigma)
        assert (thr[e] + thr[e][::-1] - 4294967296 >= -2).all() and (thr[e] + thr[e][::-1] - 4294967296 <= 0).all()   # symmetric levels
    assert exact >= len(sig) * 14 - 2
    # sigma = 1: a textbook value, Phi(0.5) = 0.6914624612740131 -> level 0 ends at floor(2^32 * 0.69146...)
    assert abs(int(thr[1, 7]) - 2969808657) <= 1 and abs(int(thr[1, 6]) - (4294967296 - 2969808657)) <= 1
    # the clamps: sigma -> 0 puts everything on level 0 (thresholds 0 below the centre, 2^32 - 1 above, never
    # 2^32, which would not fit); a huge sigma gives the two outer levels half the mass each
    tiny = sk_synth.digitiser_thresholds([1e-6]).numpy().astype(np.int64)[0]
    assert (tiny[:7] == 0).all() and (tiny[7:] == 4294967295).all()
    huge = sk_synth.digitiser_thresholds([1e9]).numpy().astype(np.int64)[0]
    assert (np.abs(huge - 2147483648) < 64).all() and (np.diff(huge) >= 0).all()


def test_app_b_mean_offset_constant_variance_converges(oracle):
    """PAPER.md:282-284 on the simulator's data (sigma = 1.52): the mean of SK~ is offset from 1 by
    a constant that does not depend on N and equals the model's E[p^2]/E[p]^2 - 1; the variance
    approaches the un-digitised 4/(MN) (here within 15 %)."""
    import sk_synth
    M, E, B = 64, 256, 400
    thr = sk_synth.digitiser_thresholds(np.full(E, 1.52)).numpy().astype(np.uint32)
    data = oracle.sim_digitised(M * B, 1, E, thr, seed=11)
    lim = _quantised_limit(1.52)
    means = {}
    for N in (16, 64, 256):
        sk = oracle.frame(data, M, first_n=N)["SK"]
        mean, var = oracle.moments(sk)
        means[N] = mean[0]
        assert abs(mean[0] - lim) < 4 * np.sqrt(4 / (M * N * B)) + 2.0 / M ** 2 + 1e-3
        assert 0.85 < var[0] / (4 / (M * N)) < 1.15
    assert abs(means[16] - means[256]) < 5 * np.sqrt(4 / (M * 16 * B))


def test_moments(oracle):
    rng = np.random.default_rng(13)
    SK = rng.normal(0.94, 0.003, size=(500, 3)).astype(np.float32)
    mean, var = oracle.moments(SK)
    np.testing.assert_allclose(mean, SK.astype(np.float64).mean(axis=0), rtol=1e-13)
    np.testing.assert_allclose(var, SK.astype(np.float64).var(axis=0, ddof=1), rtol=1e-10)
    assert np.isnan(oracle.moments(SK[:1])[1]).all()


# ---- App. A common-mode simulation ----------------------
def test_gauss_pair_and_common_mode_samples(oracle):
    """Box-Muller against its definition at chosen words, then the simulated samples: unit variance
    per component, E|z|^4 = 8 (circular Gaussian, variance 2), independent receivers when amp = 0,
    correlation amp^2/(1+amp^2) between receivers otherwise, and the counter layout (receiver pairs
    share one Philox call; the common-mode term is the same for every receiver)."""
    z = oracle.gauss_pair(0x7FFFFFFF, 0)                        # u1 = 0.5 - 2^-33 + ..., u2 = 2^-33
    assert z[0] == pytest.approx(math.sqrt(-2 * math.log((0x7FFFFFFF + 0.5) / 2 ** 32)) * math.cos(2 * math.pi * 0.5 / 2 ** 32), rel=1e-14)
    assert abs(z[1]) < 1e-8
    z = oracle.gauss_pair(0, 0x40000000)                        # u2 ~ 1/4: on the imaginary axis
    assert abs(z[0]) < 1e-7 and z[1] == pytest.approx(math.sqrt(-2 * math.log(0.5 / 2 ** 32)), rel=1e-9)
    D, M, N = 40, 64, 16
    sk0, x0 = oracle.sim_common_mode(D, M, N, 0.0, seed=5, want_x=True)
    sk1, x1 = oracle.sim_common_mode(D, M, N, 1.5, seed=5, want_x=True)
    n = x0.size
    assert abs(x0.real.var() - 1) < 5 * math.sqrt(2 / n) and abs(x0.imag.var() - 1) < 5 * math.sqrt(2 / n)
    assert abs((np.abs(x0) ** 4).mean() - 8) < 5 * math.sqrt((384 - 64) / n)
    assert abs(x0.mean()) < 5 * math.sqrt(2 / n)
    c = (x1 - x0) / 1.5                                           # the common-mode term
    assert np.allclose(c, c[:, :, :1], atol=1e-12) and abs(c[:, :, 0].real.var() - 1) < 0.1
    a = x0.reshape(-1, N)
    corr0 = (a[:, 0] * np.conj(a[:, 1])).mean() / 2
    assert abs(corr0) < 5 / math.sqrt(a.shape[0])
    b = x1.reshape(-1, N)
    corr1 = ((b[:, 0] * np.conj(b[:, 1])).mean() / (np.abs(b[:, 0]) ** 2).mean()).real
    assert corr1 == pytest.approx(1.5 ** 2 / (1 + 1.5 ** 2), abs=0.06)
    # Eq. 14 of these samples, recomputed with numpy from the returned x
    p = np.abs(x1) ** 2
    S1, S2 = p.sum(axis=1), (p ** 2).sum(axis=1)
    want = (M + 1) / (M - 1) * ((M * M * S2 / S1 ** 2).sum(axis=1) / (M * N) - 1)
    np.testing.assert_allclose(sk1, want, rtol=1e-12)


def test_app_a_effective_receivers(oracle):
    """PAPER.md:266-272 (Fig. 5): with no common mode var(SK~) = 4/(nN) (N_eff = N); as the
    common-mode amplitude grows the variance rises towards the single-receiver value (N_eff -> 1);
    a larger array loses a larger share of its receivers at the same amplitude."""
    M, D = 64, 600
    exact = lambda N: 4.0 * M * M / ((M - 1) * (M + 2) * (M + 3) * N)      # Gaussian value of 4/(nN)
    neff = {}
    for N in (8, 64):
        for amp in (0.0, 0.5, 4.0):
            sk = oracle.sim_common_mode(D, M, N, amp, seed=17 + N)
            neff[N, amp] = exact(1) / sk.var(ddof=1)
            assert abs(sk.mean() - 1) < 5 * math.sqrt(exact(1) / D)
    for N in (8, 64):
        assert neff[N, 0.0] == pytest.approx(N, rel=0.25)
        assert neff[N, 0.0] > neff[N, 0.5] > neff[N, 4.0]
        assert neff[N, 4.0] < 1.6                                   # effectively a single receiver
    assert neff[64, 0.5] / 64 < neff[8, 0.5] / 8                    # larger arrays suffer first
