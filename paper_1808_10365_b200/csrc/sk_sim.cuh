// sk_sim.cuh — SURVEY.md section 8(f) NEXT-1: the digitisation simulation of PAPER.md:276-284
// (App. B) on the device: seeded 4+4-bit round-and-clip Gaussian frames generated straight into
// HBM, and the mean / variance of the SK estimates.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "sk_kernels.cuh"

namespace sk {

// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): counter-based, so every (row, receiver pair)
// draws its four words independently of the launch shape.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// value + 8 = 1 + #{ j : u >= thr[j] }  (value = -7 + count).  The thresholds ascend (the caller's table is a
// CDF), so the count is found by a 4-step branch-free binary search.  The table lives in shared memory as
// col[k * kSimStride] (k = 0..14, entry 14 = 0xFFFFFFFF), one column per thread and receiver, so that a warp's
// reads never conflict whatever the indices are; the ALU pipe (ISETP / SEL at half rate) is what bounds this
// kernel, and the search costs it 3 instructions per step instead of the 23 per component of a search over
// registers (select chains).  Equal neighbouring thresholds are fine: the count is the number of thresholds <= u.
constexpr int kSimThreads = 128;
constexpr int kSimStride = 2 * kSimThreads;     // words between consecutive thresholds of one column

__device__ __forceinline__ uint32_t digitise_nibble(uint32_t u, const uint32_t* col) {
    uint32_t n = (u >= col[7 * kSimStride]) ? 8u : 0u;
    n += (u >= col[(n + 3u) * kSimStride]) ? 4u : 0u;
    n += (u >= col[(n + 1u) * kSimStride]) ? 2u : 0u;
    n += (u >= col[n * kSimStride]) ? 1u : 0u;           // n = 14 reads the pad: u = 2^32 - 1 would count it
    return 1u + (n < 14u ? n : 14u);
}

constexpr int kSimRows = 64;              // rows per thread (at least)

// Thread = one receiver pair (2j, 2j+1) for rpt rows r = t*F + f; counter (j, r, frame), key seed.
__global__ void __launch_bounds__(kSimThreads)
sk_sim_kernel(uint8_t* __restrict__ data, uint64_t rows, uint32_t rpt, uint32_t E, const uint32_t* __restrict__ thr,
              uint32_t seed_lo, uint32_t seed_hi, uint32_t frame_lo, uint32_t frame_hi) {
    const uint32_t j = blockIdx.x * kSimThreads + threadIdx.x;
    const uint32_t e = 2 * j;
    if (e >= E) return;
    const bool two = e + 1 < E;
    __shared__ uint32_t table[15 * kSimStride];
    uint32_t* const ta = table + threadIdx.x;                      // receiver 2j
    uint32_t* const tb = table + kSimThreads + threadIdx.x;        // receiver 2j + 1
#pragma unroll
    for (int i = 0; i < 15; ++i) {
        ta[i * kSimStride] = i < 14 ? __ldg(thr + (size_t)e * 14 + i) : 0xFFFFFFFFu;
        tb[i * kSimStride] = (i < 14 && two) ? __ldg(thr + (size_t)(e + 1) * 14 + i) : 0xFFFFFFFFu;
    }
    const uint64_t r0 = (uint64_t)blockIdx.y * rpt;
    const uint64_t r1 = r0 + rpt < rows ? r0 + rpt : rows;
    for (uint64_t r = r0; r < r1; ++r) {
        uint32_t w[4];
        philox4x32_10(j, (uint32_t)r, frame_lo, frame_hi, seed_lo, seed_hi, w);
        const uint32_t a = (digitise_nibble(w[0], ta) << 4) | digitise_nibble(w[1], ta);
        uint8_t* q = data + r * E + e;
        if (two) {
            const uint32_t b = (digitise_nibble(w[2], tb) << 4) | digitise_nibble(w[3], tb);
            if ((reinterpret_cast<uintptr_t>(q) & 1u) == 0) *reinterpret_cast<uint16_t*>(q) = (uint16_t)(a | (b << 8));
            else { q[0] = (uint8_t)a; q[1] = (uint8_t)b; }
        } else {
            q[0] = (uint8_t)a;
        }
    }
}

// Mean and unbiased variance of SK over the blocks, per frequency: one CTA per frequency, two
// passes in float64, fixed order (thread-strided partial sums, then a shared-memory tree).
constexpr int kMomThreads = 256;

__device__ __forceinline__ double block_sum(double x, double* red) {
    red[threadIdx.x] = x;
    __syncthreads();
    for (int o = kMomThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + o]);
        __syncthreads();
    }
    const double s = red[0];
    __syncthreads();
    return s;
}

__global__ void __launch_bounds__(kMomThreads)
sk_moments_kernel(const float* __restrict__ SK, uint32_t B, uint32_t F, double* __restrict__ mean,
                  double* __restrict__ var) {
    __shared__ double red[kMomThreads];
    const uint32_t f = blockIdx.x;
    double s = 0.0;
    for (uint32_t b = threadIdx.x; b < B; b += kMomThreads) s = __dadd_rn(s, (double)SK[(size_t)b * F + f]);
    const double m = __ddiv_rn(block_sum(s, red), (double)B);
    double v = 0.0;
    for (uint32_t b = threadIdx.x; b < B; b += kMomThreads) {
        const double d = __dsub_rn((double)SK[(size_t)b * F + f], m);
        v = __fma_rn(d, d, v);
    }
    v = block_sum(v, red);
    if (threadIdx.x == 0) {
        mean[f] = m;
        var[f] = B > 1 ? __ddiv_rn(v, (double)(B - 1)) : __longlong_as_double(0x7ff8000000000000ll);
    }
}

// ------------------------------------------------------------------ SURVEY 8(f) NEXT-3 (App. A)
// Common-mode simulation (Fig. 5): dataset d holds M samples of N receivers,
// x = z + amp * c, z independent unit circular Gaussians, c one common circular Gaussian per time
// sample.  One CTA per dataset; the samples never touch HBM: Philox words -> Box-Muller -> float64
// sums S1, S2 per receiver (Eq. 7) -> Eq. 11 terms -> canonical tree -> Eq. 14.
__device__ __forceinline__ void gauss_pair(uint32_t w0, uint32_t w1, double& re, double& im) {
    const double u1 = ((double)w0 + 0.5) * (1.0 / 4294967296.0), u2 = ((double)w1 + 0.5) * (1.0 / 4294967296.0);
    const double rad = sqrt(-2.0 * log(u1));
    double sn, cs;
    sincos(6.283185307179586476925286766559 * u2, &sn, &cs);
    re = rad * cs;
    im = rad * sn;
}

constexpr int kCmThreads = 256;

__global__ void __launch_bounds__(kCmThreads)
sk_sim_common_mode_kernel(uint32_t M, uint32_t N, double amp, uint32_t seed_lo, uint32_t seed_hi,
                          float* __restrict__ SK) {
    extern __shared__ double2 cm[];                 // amp * c(t), t < M
    __shared__ double red[kCmThreads];
    const uint32_t d = blockIdx.x;
    for (uint32_t t = threadIdx.x; t < M; t += kCmThreads) {
        uint32_t w[4];
        philox4x32_10(0u, t, d, 1u, seed_lo, seed_hi, w);
        double cr, ci;
        gauss_pair(w[0], w[1], cr, ci);
        cm[t] = make_double2(amp * cr, amp * ci);
    }
    __syncthreads();
    const double Md = (double)M, MM = Md * Md;
    TreeMerge tm;
    for (uint32_t e0 = 0; e0 < N; e0 += 2 * kCmThreads) {          // 512 receivers per pass
        const uint32_t j = e0 / 2 + threadIdx.x, e = 2 * j;
        double term = 0.0;
        if (e < N) {
            double a1 = 0.0, a2 = 0.0, b1 = 0.0, b2 = 0.0;
            for (uint32_t t = 0; t < M; ++t) {
                uint32_t w[4];
                philox4x32_10(j, t, d, 0u, seed_lo, seed_hi, w);
                double zr, zi;
                gauss_pair(w[0], w[1], zr, zi);
                const double2 c = cm[t];
                double xr = zr + c.x, xi = zi + c.y;
                double pw = xr * xr + xi * xi;
                a1 += pw;
                a2 += pw * pw;
                gauss_pair(w[2], w[3], zr, zi);
                xr = zr + c.x;
                xi = zi + c.y;
                pw = xr * xr + xi * xi;
                b1 += pw;
                b2 += pw * pw;
            }
            term = a1 == 0.0 ? Md : MM * a2 / (a1 * a1);
            if (e + 1 < N) term += (b1 == 0.0 ? Md : MM * b2 / (b1 * b1));
        }
        red[threadIdx.x] = term;
        __syncthreads();
        for (int o = 1; o < kCmThreads; o <<= 1) {
            if ((threadIdx.x & (2 * o - 1)) == 0) red[threadIdx.x] += red[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) tm.push(red[0]);
        __syncthreads();
    }
    if (threadIdx.x == 0)
        SK[d] = (float)((Md + 1.0) / (Md - 1.0) * (tm.total() / (Md * (double)N) - 1.0));
}

}  // namespace sk
