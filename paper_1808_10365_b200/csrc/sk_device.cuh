// sk_device.cuh — device-side building blocks of the SK hot path (sm_100a).
//
// Steps (equations of arXiv 1808.10365, lines of PAPER.md):
//   a1 unpack 4+4-bit offset samples      a2 |x|^2
//   a3 S1 = sum |x|^2, S2 = sum |x|^4 (Eq. 7)
//   a4 term_e = M^2 S2_e / S1_e^2 (Eq. 9, 11)
// This file shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sk {

// ---------------------------------------------------------------------------------- loads
// Streaming 128-bit load: read-only path, do not allocate in L1 (every byte is used once).
__device__ __forceinline__ uint4 ldg_stream(const uint8_t* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// The same load without .nc, for a kernel that also WRITES the buffer it reads (in-place excision):
// PTX allows ld.global.nc only on memory that stays read-only for the kernel's whole lifetime.
__device__ __forceinline__ uint4 ldg_stream_rw(const uint8_t* p) {
    uint4 r;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

// Scheduling fence for a batch of loads: every register of the batch passes through one empty
// volatile asm, so all loads of the batch are issued before the first sample is unpacked
// (keeps kUnroll 128-bit loads in flight per lane instead of one).
template <int U>
__device__ __forceinline__ void loads_issued(uint4 (&v)[U]) {
#pragma unroll
    for (int u = 0; u < U; u += 2) {
        asm volatile("" : "+r"(v[u].x), "+r"(v[u].y), "+r"(v[u].z), "+r"(v[u].w),
                          "+r"(v[u + 1].x), "+r"(v[u + 1].y), "+r"(v[u + 1].z), "+r"(v[u + 1].w));
    }
}

// ------------------------------------------------------------------------- a1 + a2, packed
// One 32-bit word holds 4 samples: byte = (re+8)<<4 | (im+8).
//   hi(w) = (w & 0xF0F0F0F0) ^ 0x80808080 : four signed bytes 16*re   (one LOP3)
//   lo(w) = (rotl(w,4) & 0xF0F0F0F0) ^ 0x80808080 : four signed bytes 16*im (SHF + LOP3)
// Flipping the top bit of the offset nibble turns it into two's complement, and leaving it in
// the high nibble of its byte sign-extends it for free (scaled by 16).  Nibble 0 -> -128 = 16*(-8).
// The two masks live in registers (LOP3 takes one immediate only; with both as literals ptxas
// emits two LOP3 per word instead of one).
struct UnpackConsts {
    uint32_t f0, x80;
    __device__ __forceinline__ void init() {
        asm volatile("mov.u32 %0, 0xF0F0F0F0;" : "=r"(f0));
        asm volatile("mov.u32 %0, 0x80808080;" : "=r"(x80));
    }
};
__device__ __forceinline__ uint32_t and_xor(uint32_t a, uint32_t b, uint32_t c) {   // (a & b) ^ c
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, 0x6a;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t re16(uint32_t w, const UnpackConsts& k) { return and_xor(w, k.f0, k.x80); }
// The shift is written as a rotate (SHF.L.W on the ALU pipe; the bits that wrap around land in a low
// nibble and are masked off): a plain `w << 4` becomes IMAD.SHL on the fmaheavy pipe, which the
// IDP and the packed FP32 instructions already fill.
__device__ __forceinline__ uint32_t rotl4(uint32_t w) {
    uint32_t d;
    asm("shf.l.wrap.b32 %0, %1, %1, 4;" : "=r"(d) : "r"(w));
    return d;
}
__device__ __forceinline__ uint32_t im16(uint32_t w, const UnpackConsts& k) { return and_xor(rotl4(w), k.f0, k.x80); }

// ------------------------------------------------------------------------------ a3 variants
// Accumulators for TWO adjacent inputs (one 64-bit register pair of state each), three exact
// strategies with one interface: add2(c0, c1) adds one sample to each input, c = [16re,16im,16re,16im]
// (pick<K>); read(i, n, S1, S2) returns the sums of input i in {0, 1} after n samples each.
//
// AccPlain2: S1 += p; S2 += p*p in 32-bit registers (shift, add, IMAD per sample).  Any n.
//
// AccWide2 : ONE 64-bit multiply-add per sample.  With q = 512 p + 2^31 (the 2^31 comes free as the
//   DP4A addend), q*q = 2^18 p^2 + 2^41 p + 2^62, so a 64-bit accumulator collects
//   sum p^2 in bits 18..40 and sum p in bits 41..61; the constant n*2^62 (n = samples added) wraps
//   mod 2^64 and is removed at read-out.  Exact while sum p^2 < 2^23, i.e. n <= 511 samples
//   (p^2 <= 2^14).
//
// AccChain2: S1 on the IDP addend chain, S2 on the FP32 pipes with Blackwell's packed FP32.
//   r starts as the bit pattern of the float 2^23 and every IDP adds 512 p to it:
//   r_k = IDP(C, C, r_{k-1}).  While 512 sum(p) <= 2^23 the float view of r is exactly
//   2^23 + 512 sum(p), so d = float(r_k) - float(r_{k-1}) = 512 p_k exactly and
//   s2 = fma(d, d, s2) = 2^18 sum(p^2) exactly (sum p^2 < 2^24).  The two inputs' r sit in one
//   aligned register pair and their s2 in another, so ONE sub.rn.f32x2 (SASS FADD2) and ONE
//   fma.rn.f32x2 (SASS FFMA2) serve both: 3 issue slots per sample (PRMT, IDP, half of each packed
//   op) instead of 4.  S1 = (r - 2^23 pattern) >> 9.
//   Limit: sum(p) <= 16384, i.e. n <= 128 samples per lane and unit (p <= 128).
//   Why not AccWide2 everywhere: IMAD.WIDE costs 4 cycles of the half-rate fmaheavy pipe, the
//   bottleneck of an all-AccWide kernel (ncu: sm__pipe_fmaheavy_cycles_active 78 %).
struct AccPlain2 {
    uint32_t s1[2], s2[2];
    __device__ __forceinline__ void reset() { s1[0] = s1[1] = s2[0] = s2[1] = 0; }
    __device__ __forceinline__ void add1(int i, uint32_t c) {
        const uint32_t p = (uint32_t)__dp4a((int)c, (int)c, 0) >> 9;
        s1[i] += p;
        s2[i] += p * p;
    }
    __device__ __forceinline__ void add2(uint32_t c0, uint32_t c1) { add1(0, c0); add1(1, c1); }
    __device__ __forceinline__ void read(int i, uint32_t /*n*/, uint32_t& S1, uint32_t& S2) const { S1 = s1[i]; S2 = s2[i]; }
};

struct AccWide2 {
    unsigned long long a[2];
    static constexpr uint32_t kMaxSamples = 511;
    __device__ __forceinline__ void reset() { a[0] = a[1] = 0ull; }
    __device__ __forceinline__ void add1(int i, uint32_t c) {
        const uint32_t q = (uint32_t)__dp4a((int)c, (int)c, (int)0x80000000u);
        a[i] += (unsigned long long)q * q;
    }
    __device__ __forceinline__ void add2(uint32_t c0, uint32_t c1) { add1(0, c0); add1(1, c1); }
    __device__ __forceinline__ void read(int i, uint32_t n, uint32_t& S1, uint32_t& S2) const {
        const unsigned long long v = a[i] - ((unsigned long long)(n & 3u) << 62);
        S1 = (uint32_t)(v >> 41);
        S2 = (uint32_t)((v & ((1ull << 41) - 1ull)) >> 18);
    }
};

__device__ __forceinline__ unsigned long long pack2(uint32_t lo, uint32_t hi) {
    unsigned long long v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "r"(lo), "r"(hi));
    return v;
}
__device__ __forceinline__ void unpack2(unsigned long long v, uint32_t& lo, uint32_t& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(v));
}

struct AccChain2 {
    uint32_t r0, r1;               // the two IDP chains (float view: 2^23 + 512 sum p)
    unsigned long long s2;         // two floats: 2^18 sum p^2 of input 0 (low word) and input 1
    static constexpr uint32_t kMagic = 0x4B000000u;
    static constexpr uint32_t kMaxSamples = 128;
    __device__ __forceinline__ void reset() { r0 = r1 = kMagic; s2 = 0ull; }
    // NOSUB (measurement builds only, see kVar* below): leave the FADD2 out; the sums are then wrong.
    template <bool NOSUB = false>
    __device__ __forceinline__ void add2(uint32_t c0, uint32_t c1) {
        const uint32_t n0 = (uint32_t)__dp4a((int)c0, (int)c0, (int)r0);
        const uint32_t n1 = (uint32_t)__dp4a((int)c1, (int)c1, (int)r1);
        unsigned long long d = pack2(n0, n1);
        if (!NOSUB) asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pack2(n0, n1)), "l"(pack2(r0, r1)));
        asm("fma.rn.f32x2 %0, %1, %1, %2;" : "=l"(s2) : "l"(d), "l"(s2));
        r0 = n0;
        r1 = n1;
    }
    __device__ __forceinline__ void read(int i, uint32_t /*n*/, uint32_t& S1, uint32_t& S2) const {
        uint32_t lo, hi;
        unpack2(s2, lo, hi);
        S1 = ((i ? r1 : r0) - kMagic) >> 9;
        S2 = __float2uint_rn(__uint_as_float(i ? hi : lo) * (1.0f / 262144.0f));
    }
};

// [16re_k, 16im_k, 16re_k, 16im_k] of sample K of a word (one PRMT); C.C = 512 |x_k|^2 (one IDP.4A).
template <int K>
__device__ __forceinline__ uint32_t pick(uint32_t r16, uint32_t i16) {
    constexpr uint32_t sel = (uint32_t)K | ((4u + K) << 4) | ((uint32_t)K << 8) | ((4u + K) << 12);
    return __byte_perm(r16, i16, sel);
}

// Measurement variants of the loop body.  The product library instantiates
// kVarProduct only; the others exist in the bench library (csrc/bench/), give WRONG sums by design and
// answer one question each: what does the loop cost without this instruction?
//   kVarMemOnly  : no arithmetic at all, the loaded words are XORed into the accumulators (is memory the limit?)
//   kVarNoSub    : without the FADD2 (sub.rn.f32x2)          kVarNoPick : without the PRMTs (pick<K>)
//   kVarNoUnpack : without the LOP3 / SHF / LOP3 of re16 / im16
enum { kVarProduct = 0, kVarMemOnly = 1, kVarNoSub = 2, kVarNoPick = 3, kVarNoUnpack = 4 };

// Add the 16 samples of one 128-bit load to the lane's 16 inputs (8 pair accumulators).
template <class Acc2, int VAR = kVarProduct>
__device__ __forceinline__ void accumulate16(Acc2 (&acc)[8], const uint4& v, const UnpackConsts& kc) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    if constexpr (VAR == kVarProduct) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t r = re16(w[i], kc), m = im16(w[i], kc);
            acc[2 * i + 0].add2(pick<0>(r, m), pick<1>(r, m));
            acc[2 * i + 1].add2(pick<2>(r, m), pick<3>(r, m));
        }
    } else if constexpr (VAR == kVarMemOnly) {
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[i].r0 ^= w[i];
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const uint32_t r = VAR == kVarNoUnpack ? w[i] : re16(w[i], kc);
            const uint32_t m = VAR == kVarNoUnpack ? w[(i + 1) & 3] : im16(w[i], kc);
            if constexpr (VAR == kVarNoPick) {
                acc[2 * i + 0].add2(r, m);
                acc[2 * i + 1].add2(m, r);
            } else {
                acc[2 * i + 0].template add2<VAR == kVarNoSub>(pick<0>(r, m), pick<1>(r, m));
                acc[2 * i + 1].template add2<VAR == kVarNoSub>(pick<2>(r, m), pick<3>(r, m));
            }
        }
    }
}

// S1, S2 of the lane's 16 inputs after n samples each.
template <class Acc2>
__device__ __forceinline__ void read16(const Acc2 (&acc)[8], uint32_t n, uint32_t (&S1)[16], uint32_t (&S2)[16]) {
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k / 2].read(k % 2, n, S1[k], S2[k]);
}

// Scalar a1-a2 for the fallback kernel.
__device__ __forceinline__ uint32_t power_scalar(uint8_t byte) {
    const int re = (int)(byte >> 4) - 8, im = (int)(byte & 15) - 8;
    return (uint32_t)(re * re + im * im);
}

// ------------------------------------------------------------------------------------- a4
// uint32 -> float64 without the conversion unit: the integer is the low word of 2^52 + u.
__device__ __forceinline__ double u32_to_f64(uint32_t u) {
    return __dsub_rn(__hiloint2double(0x43300000, (int)u), 4503599627370496.0);
}

// n / y for finite n >= 0 and positive normal y (here 1 <= y < 2^53, n < 2^60, and the flag
// spread sqrt(4/(M N))): hardware reciprocal seed, two Newton steps, one
// correction of the quotient.  Branch-free; the result is within one ulp of n / y (normally the
// correctly rounded quotient).  Every kernel divides through this one function, so all paths
// agree bit for bit; against the oracle's IEEE division the difference is <= 2.2e-16 relative
// per term, nine orders of magnitude inside the 1e-6 tolerance on SK.
__device__ __forceinline__ double div_f64(double n, double y) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
    double e = __fma_rn(-y, r, 1.0);               // seed: ~2^-20 relative (upper mantissa word only)
    r = __fma_rn(r, e, r);                         // 2^-40
    e = __fma_rn(-y, r, 1.0);
    r = __fma_rn(r, e, r);                         // 2^-80: r is the rounded reciprocal
    const double q = __dmul_rn(n, r);
    return __fma_rn(__fma_rn(-y, q, n), r, q);
}

// term = M^2 S2 / S1^2 in float64 (MM = M*M, exact).  S1^2 < 2^53 for M <= 65536 only up to S1 < 2^26.5 and
// M^2 S2 exceeds 2^53 from M ~ 2900 on: each product is then rounded once (round to nearest even), exactly
// as the oracle's (double)M*M*S2 and (double)S1*S1 are, so the quotient still matches it to one division
// rounding.  A receiver with S1 == 0 contributes M (header: "A receiver whose S1 is 0").
__device__ __forceinline__ double eq11_term(double M, double MM, uint32_t S1, uint32_t S2) {
    const double s1 = u32_to_f64(S1), s2 = u32_to_f64(S2);
    const double t = div_f64(__dmul_rn(MM, s2), __dmul_rn(s1, s1));
    return S1 == 0u ? M : t;
}

// a6: SK~ = (M+1)/(M-1) * (S2bar/(M N) - 1)  (Eq. 14, second line), then float32.
__device__ __forceinline__ float eq14_sk(double S2bar, double M, double N) {
    const double a = __ddiv_rn(__dadd_rn(M, 1.0), __dsub_rn(M, 1.0));
    const double c = __ddiv_rn(S2bar, __dmul_rn(M, N));
    return __double2float_rn(__dmul_rn(a, __dsub_rn(c, 1.0)));
}

// Optional estimator: the un-rescaled SK^ = (MN+1)/(MN-1) * (S2bar/(M N) - 1)  (Eq. 13,
// second line), then float32.
__device__ __forceinline__ float eq13_sk(double S2bar, double M, double N) {
    const double mn = __dmul_rn(M, N);
    const double a = __ddiv_rn(__dadd_rn(mn, 1.0), __dsub_rn(mn, 1.0));
    const double c = __ddiv_rn(S2bar, mn);
    return __double2float_rn(__dmul_rn(a, __dsub_rn(c, 1.0)));
}

// a7: flagged iff fabsf(SK - sk_mean) > thr in float32, strict; NaN => flagged.
__device__ __forceinline__ uint8_t flag_decision(float SK, float sk_mean, float thr) {
    const float dev = fabsf(__fsub_rn(SK, sk_mean));
    return (dev > thr || dev != dev) ? 1 : 0;
}

// thr = (float)(n_sigma * sqrt(4/(M N))) — float64 inside, as the header states.
__host__ __device__ __forceinline__ float flag_threshold(float n_sigma, double M, double N) {
#ifdef __CUDA_ARCH__
    return __double2float_rn(__dmul_rn((double)n_sigma, __dsqrt_rn(__ddiv_rn(4.0, __dmul_rn(M, N)))));
#else
    return (float)((double)n_sigma * sqrt(4.0 / (M * N)));
#endif
}

__device__ __forceinline__ double warp_sum_fixed(double x) {
    // fixed butterfly: the same association order on every run
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = __dadd_rn(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
}

}  // namespace sk
