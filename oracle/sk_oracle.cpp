// sk_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded, float64 CPU statement of what the spectral-kurtosis (SK) hot
// path computes, written from the paper's equations (arXiv 1808.10365, /root/reference/PAPER.md).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call it.  It shares no code, header, table or constant with the CUDA path under
// paper_1808_10365_b200/csrc/ and neither side includes the other.
//
// Every function below is the paper's definition written out: no blocking, fusion or reordering.
// Loops run block -> frequency -> input -> time; sums over inputs run in ascending input order.
//
// Notation (PAPER.md uses n for the block length in §2.2 and M in §2.1; BASELINE.json uses M):
//   T  time samples in the buffer, F frequencies, E inputs in the buffer
//   M  time samples per SK block ("n" of PAPER.md:73-80), B = T/M blocks
//   N  receivers combined, chosen by `subset` (E bytes, 0/1) or the first `first_n`
//   data[t][f][e] uint8: high nibble = re + 8, low nibble = im + 8 (4+4-bit offset encoding,
//                 PAPER.md:278 "4+4-bit complex"; bit layout from BASELINE.json config 0)
//
// Readings of silent points are listed in DESIGN.md ("Readings"); the ones used here:
//   A3  nibble 0 decodes to -8 (no clamp)            A4  S1 == 0  =>  term = M (SK_i = 0)
//   A5  flag centre is the parameter sk_mean         A6  flag width sqrt(4/(M N))
//   A7  strict '>' and NaN => flagged                A11 excision writes 0x88 to all E inputs
//
// Pins: tests/test_oracle_pins.py (all functions here are pinned, incl. sk_oracle_singles and
// sk_oracle_significance of SURVEY.md section 8(f)).
// Build: g++ -O2 -ffp-contract=off -shared -fPIC (oracle/build.py); no -ffast-math, no OpenMP.

#include <cmath>
#include <cstddef>
#include <cstdint>

namespace {

// PAPER.md:278 + BASELINE.json: value = nibble - 8.
inline int decode_re(uint8_t byte) { return (int)(byte >> 4) - 8; }
inline int decode_im(uint8_t byte) { return (int)(byte & 15) - 8; }

// Is input e one of the N combined receivers?  (reading A9)
inline bool in_subset(const uint8_t* subset, uint32_t first_n, uint32_t e) {
    return subset ? subset[e] != 0 : e < first_n;
}

inline uint32_t count_subset(const uint8_t* subset, uint32_t first_n, uint32_t E) {
    if (!subset) return first_n;
    uint32_t n = 0;
    for (uint32_t e = 0; e < E; ++e) n += subset[e] != 0;
    return n;
}

// PAPER.md:88 Eq. 11 summand, written as Eq. 11's right-hand form n^2 (S2)_i / ((S1)_i)^2.
// Reading A4: a receiver with zero power contributes n (its SK_i is taken as 0).
inline double eq11_term(double M, double S1, double S2) {
    if (S1 == 0.0) return M;
    return (M * M * S2) / (S1 * S1);
}

}  // namespace

extern "C" {

// ---------------------------------------------------------------------------------------------
// PAPER.md:77 Eq. 7 (and :45 Eq. 1): (S1)_i = sum_j |x_j|^2, (S2)_i = sum_j |x_j|^4 over the
// M samples of each block, for every (block, frequency, input).  Exact integers.
// S1, S2: uint32 [B][F][E].  Returns 0, or -1 on a bad argument.
int sk_oracle_power_sums(const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                         uint32_t* S1, uint32_t* S2) {
    if (!data || !S1 || !S2 || M < 2 || T == 0 || T % M != 0 || F == 0 || E == 0) return -1;
    const uint32_t B = T / M;
    for (uint32_t b = 0; b < B; ++b)
        for (uint32_t f = 0; f < F; ++f)
            for (uint32_t e = 0; e < E; ++e) {
                uint64_t s1 = 0, s2 = 0;
                for (uint32_t j = 0; j < M; ++j) {
                    const size_t t = (size_t)b * M + j;
                    const uint8_t byte = data[(t * F + f) * E + e];
                    const int re = decode_re(byte), im = decode_im(byte);
                    const uint64_t p = (uint64_t)(re * re + im * im);  // |x|^2
                    s1 += p;
                    s2 += p * p;
                }
                const size_t o = ((size_t)b * F + f) * E + e;
                S1[o] = (uint32_t)s1;
                S2[o] = (uint32_t)s2;
            }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// PAPER.md:84-88 Eq. 9-11 and :108-113 Eq. 14 (second line):
//   mu_i = (S1)_i / n;  S2bar = sum_i (S2)_i / mu_i^2 = sum_i n^2 (S2)_i / (S1)_i^2
//   SK~ = (n+1)/(n-1) * (S2bar/(nN) - 1)
// SK64 (optional) receives the float64 value, SK its float32 rounding (round-to-nearest-even).
int sk_oracle_combine(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E,
                      uint32_t M, const uint8_t* subset, uint32_t first_n, float* SK,
                      double* SK64) {
    if (!S1 || !S2 || !SK || M < 2 || B == 0 || F == 0 || E == 0) return -1;
    const uint32_t N = count_subset(subset, first_n, E);
    if (N == 0 || N > E) return -1;
    const double n = (double)M;
    for (uint32_t b = 0; b < B; ++b)
        for (uint32_t f = 0; f < F; ++f) {
            const size_t c = (size_t)b * F + f;
            double S2bar = 0.0;
            for (uint32_t e = 0; e < E; ++e) {
                if (!in_subset(subset, first_n, e)) continue;
                S2bar += eq11_term(n, (double)S1[c * E + e], (double)S2[c * E + e]);
            }
            const double sk = (n + 1.0) / (n - 1.0) * (S2bar / (n * (double)N) - 1.0);
            if (SK64) SK64[c] = sk;
            SK[c] = (float)sk;
        }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// flag data outside mean(SK~) +- a*sqrt(var(SK~)); var from PAPER.md:119 Eq. 16
// to first order, 4/(nN); centre = sk_mean (1 by Eq. 15, or the simulated value of
// PAPER.md:284).  Decision taken in float32 (reading D2): thr = (float)(a*sqrt(4/(nN))),
// mask = fabsf(SK - sk_mean) > thr, strict; NaN => 1.
int sk_oracle_flag(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N, float n_sigma,
                   float sk_mean, uint8_t* mask) {
    if (!SK || !mask || M < 2 || N == 0 || B == 0 || F == 0) return -1;
    const float thr = (float)((double)n_sigma * std::sqrt(4.0 / ((double)M * (double)N)));
    for (size_t c = 0; c < (size_t)B * F; ++c) {
        const float dev = std::fabs(SK[c] - sk_mean);  // float32 subtract, float32 abs
        mask[c] = (dev > thr || std::isnan(dev)) ? 1 : 0;
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// The whole path: Eq. 7 -> Eq. 9-11, 14 -> flag -> optional excision ("detection and
// excision"; reading A11: every byte of every flagged cell, all E inputs, becomes 0x88 = 0+0i).
// The mask is computed from the data as it was before excision.  S1out/S2out may be NULL.
int sk_oracle_frame(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                    const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean,
                    int zero_flagged, float* SK, uint8_t* mask, uint32_t* S1out, uint32_t* S2out,
                    uint32_t* S1tmp, uint32_t* S2tmp) {
    if (!S1tmp || !S2tmp) return -1;
    int rc = sk_oracle_power_sums(data, T, F, E, M, S1tmp, S2tmp);
    if (rc) return rc;
    const uint32_t B = T / M;
    rc = sk_oracle_combine(S1tmp, S2tmp, B, F, E, M, subset, first_n, SK, nullptr);
    if (rc) return rc;
    const uint32_t N = count_subset(subset, first_n, E);
    rc = sk_oracle_flag(SK, B, F, M, N, n_sigma, sk_mean, mask);
    if (rc) return rc;
    const size_t cells = (size_t)B * F * E;
    if (S1out) for (size_t i = 0; i < cells; ++i) S1out[i] = S1tmp[i];
    if (S2out) for (size_t i = 0; i < cells; ++i) S2out[i] = S2tmp[i];
    if (zero_flagged)
        for (uint32_t b = 0; b < B; ++b)
            for (uint32_t f = 0; f < F; ++f)
                if (mask[(size_t)b * F + f])
                    for (uint32_t j = 0; j < M; ++j)
                        for (uint32_t e = 0; e < E; ++e)
                            data[(((size_t)b * M + j) * F + f) * E + e] = 0x88;
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Companion definitions used only to pin the above against the paper's identities.

// PAPER.md:48 Eq. 2 / :80 Eq. 8: SK^_i = (n+1)/(n-1) * (n (S2)_i / (S1)_i^2 - 1).
double sk_oracle_single(double S1, double S2, double M) {
    return (M + 1.0) / (M - 1.0) * (M * S2 / (S1 * S1) - 1.0);
}

// PAPER.md:112 Eq. 14 third line ("average the individual estimates"):
// SK~ = (1/N) sum_i SK^_i, per (block, frequency).  Zero-power receivers count as SK^_i = 0 (A4).
int sk_oracle_average_of_singles(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F,
                                 uint32_t E, uint32_t M, const uint8_t* subset, uint32_t first_n,
                                 double* SK64) {
    if (!S1 || !S2 || !SK64 || M < 2) return -1;
    const uint32_t N = count_subset(subset, first_n, E);
    if (N == 0 || N > E) return -1;
    for (size_t c = 0; c < (size_t)B * F; ++c) {
        double acc = 0.0;
        for (uint32_t e = 0; e < E; ++e) {
            if (!in_subset(subset, first_n, e)) continue;
            const double s1 = (double)S1[c * E + e], s2 = (double)S2[c * E + e];
            acc += (s1 == 0.0) ? 0.0 : sk_oracle_single(s1, s2, (double)M);
        }
        SK64[c] = acc / (double)N;
    }
    return 0;
}

// Per-receiver estimates as an output (Eq. 8, the
// "independent SK estimates" of PAPER.md:73, 145-151): SKi[b][f][e] = SK^_e rounded to float32.
// A zero-power receiver gives 0 (reading A4).
int sk_oracle_singles(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E,
                      uint32_t M, float* SKi) {
    if (!S1 || !S2 || !SKi || M < 2) return -1;
    for (size_t i = 0; i < (size_t)B * F * E; ++i) {
        const double s1 = (double)S1[i], s2 = (double)S2[i];
        SKi[i] = (float)((s1 == 0.0) ? 0.0 : sk_oracle_single(s1, s2, (double)M));
    }
    return 0;
}

// Detection significance ("detection significance", the distance from the expected
// mean in units of the expected spread): sig = (SK - sk_mean) / sqrt(4/(n N)) (Eq. 16), evaluated
// in float64 from the float32 SK and rounded to float32.  |sig| > a is the flag of sk_oracle_flag.
int sk_oracle_significance(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N,
                           float sk_mean, float* sig) {
    if (!SK || !sig || M < 2 || N == 0) return -1;
    const double sd = std::sqrt(4.0 / ((double)M * (double)N));
    for (size_t c = 0; c < (size_t)B * F; ++c) sig[c] = (float)(((double)SK[c] - (double)sk_mean) / sd);
    return 0;
}

// PAPER.md:97-99 Eq. 13 (first two lines), the un-rescaled multi-receiver estimator, and
// PAPER.md:86 Eq. 10, S1bar = sum_i (S1)_i / mu_i (which must equal nN).
int sk_oracle_eq13_and_s1bar(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F,
                             uint32_t E, uint32_t M, const uint8_t* subset, uint32_t first_n,
                             double* SKhat13, double* S1bar_out, double* S2bar_out) {
    if (!S1 || !S2 || M < 2) return -1;
    const uint32_t N = count_subset(subset, first_n, E);
    if (N == 0 || N > E) return -1;
    const double n = (double)M, nN = n * (double)N;
    for (size_t c = 0; c < (size_t)B * F; ++c) {
        double S1bar = 0.0, S2bar = 0.0;
        for (uint32_t e = 0; e < E; ++e) {
            if (!in_subset(subset, first_n, e)) continue;
            const double s1 = (double)S1[c * E + e], s2 = (double)S2[c * E + e];
            const double mu = s1 / n;                       // Eq. 9
            S1bar += (s1 == 0.0) ? n : s1 / mu;             // Eq. 10
            S2bar += (s1 == 0.0) ? n : s2 / (mu * mu);      // Eq. 11, first form
        }
        if (S1bar_out) S1bar_out[c] = S1bar;
        if (S2bar_out) S2bar_out[c] = S2bar;
        if (SKhat13)  // Eq. 13 first line: M_eff = nN, with S1bar and S2bar as the cumulants
            SKhat13[c] = (nN + 1.0) / (nN - 1.0) * (nN * S2bar / (S1bar * S1bar) - 1.0);
    }
    return 0;
}

// Float-input entry (not quantised): x[t][f][e] = re[..] + i im[..] as doubles.  Same Eq. 7,
// 9-11, 14 with float64 sums, used for the null-moment pins and for
// the "non-digitized" arm of PAPER.md:278.  S1f/S2f (optional): double [B][F][E].
int sk_oracle_frame_float(const double* re, const double* im, uint32_t T, uint32_t F, uint32_t E,
                          uint32_t M, const uint8_t* subset, uint32_t first_n, double* SK64,
                          double* S1f, double* S2f) {
    if (!re || !im || !SK64 || M < 2 || T == 0 || T % M != 0) return -1;
    const uint32_t N = count_subset(subset, first_n, E);
    if (N == 0 || N > E) return -1;
    const uint32_t B = T / M;
    const double n = (double)M;
    for (uint32_t b = 0; b < B; ++b)
        for (uint32_t f = 0; f < F; ++f) {
            double S2bar = 0.0;
            for (uint32_t e = 0; e < E; ++e) {
                double s1 = 0.0, s2 = 0.0;
                for (uint32_t j = 0; j < M; ++j) {
                    const size_t i = (((size_t)b * M + j) * F + f) * E + e;
                    const double p = re[i] * re[i] + im[i] * im[i];
                    s1 += p;
                    s2 += p * p;
                }
                const size_t o = ((size_t)b * F + f) * E + e;
                if (S1f) S1f[o] = s1;
                if (S2f) S2f[o] = s2;
                if (in_subset(subset, first_n, e)) S2bar += eq11_term(n, s1, s2);
            }
            SK64[(size_t)b * F + f] = (n + 1.0) / (n - 1.0) * (S2bar / (n * (double)N) - 1.0);
        }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// the digitisation simulation of PAPER.md:276-284 (App. B).
// "a set of sample data was generated which mimicked the properties of CHIME's intermediate data
// products - 4+4-bit complex Gaussian data (bounded between -7 and 7) with an RMS of ~1.52
// least-significant bits in each component."
//
// Random numbers: the counter-based generator Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel
// random numbers: as easy as 1, 2, 3", SC'11), restated here from the paper's description; the
// CUDA path has its own copy.  Pinned by the published known-answer vectors (tests).
static inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

int sk_oracle_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    if (!ctr || !key || !out) return -1;
    philox4x32_10(ctr, key, out);
    return 0;
}

// One digitised component from one 32-bit uniform u and the receiver's 14 ascending thresholds
// thr[j] = 2^32 * P(value <= j - 7) (the caller's model of round-and-clip to [-7, 7]):
// value = -7 + #{ j : u >= thr[j] }.
static inline int digitise(uint32_t u, const uint32_t* thr) {
    int v = -7;
    for (int j = 0; j < 14; ++j) v += (u >= thr[j]) ? 1 : 0;
    return v;
}

// data[t][f][e]: for row r = t*F + f and receiver pair j = e/2 the generator is called with
// counter (j, r, frame_lo, frame_hi) and key (seed_lo, seed_hi); words 0, 1 give (re, im) of
// receiver 2j, words 2, 3 give (re, im) of receiver 2j+1.  byte = (re+8)<<4 | (im+8).
int sk_oracle_sim_digitised(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, const uint32_t* thr,
                            uint64_t seed, uint64_t frame) {
    if (!data || !thr || T == 0 || F == 0 || E == 0) return -1;
    if ((uint64_t)T * F > 0xFFFFFFFFull) return -1;
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (uint64_t r = 0; r < (uint64_t)T * F; ++r) {
        for (uint32_t e = 0; e < E; ++e) {
            const uint32_t ctr[4] = {e / 2, (uint32_t)r, (uint32_t)frame, (uint32_t)(frame >> 32)};
            uint32_t w[4];
            philox4x32_10(ctr, key, w);
            const int re = digitise(w[2 * (e & 1)], thr + (size_t)e * 14);
            const int im = digitise(w[2 * (e & 1) + 1], thr + (size_t)e * 14);
            data[r * E + e] = (uint8_t)(((re + 8) << 4) | (im + 8));
        }
    }
    return 0;
}

// Mean and unbiased variance of the estimates over the blocks, per frequency (the "statistics of
// those estimates"): two passes in float64, NaN if B < 2 for the variance.
int sk_oracle_moments(const float* SK, uint32_t B, uint32_t F, double* mean, double* var) {
    if (!SK || !mean || !var || B == 0 || F == 0) return -1;
    for (uint32_t f = 0; f < F; ++f) {
        double m = 0.0;
        for (uint32_t b = 0; b < B; ++b) m += (double)SK[(size_t)b * F + f];
        m /= (double)B;
        double v = 0.0;
        for (uint32_t b = 0; b < B; ++b) {
            const double d = (double)SK[(size_t)b * F + f] - m;
            v += d * d;
        }
        mean[f] = m;
        var[f] = (B > 1) ? v / (double)(B - 1) : std::nan("");
    }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// the common-mode simulation of PAPER.md:262-272 (App. A, Fig. 5).
// "a number of independent Gaussian datasets, representing the noise-dominated receiver
// timestreams, are augmented by a common-mode Gaussian signal representing the 'source'."
//
// One complex circular Gaussian (unit variance per component) from two 32-bit words: Box-Muller,
// u1 = (w0 + 0.5) / 2^32 in (0, 1), u2 = (w1 + 0.5) / 2^32:
//   z = sqrt(-2 ln u1) * (cos 2 pi u2, sin 2 pi u2).
static inline void gauss_pair(uint32_t w0, uint32_t w1, double& re, double& im) {
    const double u1 = ((double)w0 + 0.5) / 4294967296.0, u2 = ((double)w1 + 0.5) / 4294967296.0;
    const double rad = std::sqrt(-2.0 * std::log(u1)), ang = 6.283185307179586476925286766559 * u2;
    re = rad * std::cos(ang);
    im = rad * std::sin(ang);
}

int sk_oracle_gauss_pair(uint32_t w0, uint32_t w1, double* out) {
    if (!out) return -1;
    gauss_pair(w0, w1, out[0], out[1]);
    return 0;
}

// Sample (dataset d, time t, receiver e): x = z + amp * c, with
//   z from Philox counter (e/2, t, d, 0), words 0,1 (even e) or 2,3 (odd e),
//   c from Philox counter (0,   t, d, 1), words 0,1 (the same for all receivers),
// key (seed_lo, seed_hi).  x_out (optional): [D][M][N][2] doubles, for tests.
// SK64[d] = Eq. 14 over the N receivers and the M samples of dataset d (float64 sums, Eq. 7, 9-11).
int sk_oracle_sim_common_mode(uint32_t D, uint32_t M, uint32_t N, double amp, uint64_t seed,
                              double* SK64, double* x_out) {
    if (!SK64 || D == 0 || M < 2 || N == 0) return -1;
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    const double n = (double)M;
    for (uint32_t d = 0; d < D; ++d) {
        double S2bar = 0.0;
        for (uint32_t e = 0; e < N; ++e) {
            double s1 = 0.0, s2 = 0.0;
            for (uint32_t t = 0; t < M; ++t) {
                const uint32_t cz[4] = {e / 2, t, d, 0u}, cc[4] = {0u, t, d, 1u};
                uint32_t wz[4], wc[4];
                philox4x32_10(cz, key, wz);
                philox4x32_10(cc, key, wc);
                double zr, zi, cr, ci;
                gauss_pair(wz[2 * (e & 1)], wz[2 * (e & 1) + 1], zr, zi);
                gauss_pair(wc[0], wc[1], cr, ci);
                const double xr = zr + amp * cr, xi = zi + amp * ci;
                if (x_out) {
                    const size_t i = (((size_t)d * M + t) * N + e) * 2;
                    x_out[i] = xr;
                    x_out[i + 1] = xi;
                }
                const double p = xr * xr + xi * xi;       // Eq. 7
                s1 += p;
                s2 += p * p;
            }
            const double mu = s1 / n;                      // Eq. 9
            S2bar += (s1 == 0.0) ? n : s2 / (mu * mu);     // Eq. 11
        }
        SK64[d] = (n + 1.0) / (n - 1.0) * (S2bar / (n * (double)N) - 1.0);   // Eq. 14
    }
    return 0;
}

int sk_oracle_version(void) { return 4; }

}  // extern "C"
