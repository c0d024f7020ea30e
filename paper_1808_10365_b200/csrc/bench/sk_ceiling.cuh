// sk_ceiling.cuh — measurement only: the SM-side ceiling of the hot loop.
//
// The stream kernel's tile loop (accumulate16 of sk_device.cuh: a1-a3 for 16 samples per lane and
// 128-bit shared-memory read) run on a shared-memory tile that never changes: no global-memory
// traffic, no TMA, no barrier waits, no epilogue.  One CTA per SM, `warps` warps per CTA (warp i
// sits on sub-partition i % 4), every warp on its own 8 KiB tile, the accumulators read out every
// 8 tiles (128 samples per lane: AccChain2's limit) as in the kernel.  The elapsed SM cycles of
// CTA 0 give the cycles one sub-partition needs per 32 samples (one sample per lane) — what the
// instruction mix costs when nothing else is in the way.  bench.py reports it beside the roofline
// (DESIGN.md section 6).  VAR = kVarProduct is the product's loop body; kVarNoSub / kVarNoPick /
// kVarNoUnpack leave one kind of instruction out (sk_device.cuh), which is how DESIGN.md section 6.3
// attributes the loop's cycles to pipes.  Part of the bench library only (libsk_b200_bench.so): the
// product library contains none of this.
#pragma once
#include "../sk_tma.cuh"

namespace sk {

constexpr int kCeilingMaxWarps = 16;
constexpr int kCeilingTilesPerReadout = 8;

template <int VAR>
__global__ void __launch_bounds__(kCeilingMaxWarps * 32)
sk_loop_ceiling_kernel(uint32_t* __restrict__ sink, unsigned long long* __restrict__ cycles, uint32_t rounds) {
    constexpr int L = 16, RPW = 32 / L, W = 16 * L, NLD = kTileBytes / W / RPW;
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (uint32_t i = threadIdx.x; i < blockDim.x / 32 * (kTileBytes / 4); i += blockDim.x)
        reinterpret_cast<uint32_t*>(smem)[i] = 0x9a7b5c88u + 0x01010101u * (i % 7u);     // arbitrary samples
    __syncthreads();
    const uint32_t src = smem_addr(smem) + warp * kTileBytes + (lane / L) * W + (lane % L) * 16;
    UnpackConsts kc;
    kc.init();
    AccChain2 acc[8];
    uint32_t tot = 0;
    const long long t0 = clock64();
    for (uint32_t r = 0; r < rounds; ++r) {
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k].reset();
        for (int g = 0; g < kCeilingTilesPerReadout; ++g) {
#pragma unroll
            for (int i = 0; i < NLD; ++i) accumulate16<AccChain2, VAR>(acc, lds128(src + i * RPW * W), kc);
            __syncwarp();
        }
        uint32_t S1[16], S2[16];
        read16(acc, 0u, S1, S2);
#pragma unroll
        for (int i = 0; i < 16; ++i) tot += S1[i] ^ S2[i];
    }
    __syncthreads();
    const long long t1 = clock64();
    sink[blockIdx.x * blockDim.x + threadIdx.x] = tot;
    if (blockIdx.x == 0 && threadIdx.x == 0) *cycles = (unsigned long long)(t1 - t0);
}

// Issue rate of the loop's instructions, alone and in pairs (the pipe model of DESIGN.md section 6.3):
// 8 independent chains per lane, 2048 x 8 instructions (or pairs), operands from memory so that nothing
// folds.  mode: 0 FFMA, 1 FFMA2, 2 FADD2, 3 IDP.4A, 4 PRMT, 5 IDP + FFMA2, 6 IDP + FFMA, 7 PRMT + FFMA2,
// 8 IDP + PRMT.  *cycles = elapsed SM clocks of CTA 0.
constexpr int kPipeModes = 9;
constexpr int kPipeIters = 2048;

template <int MODE>
__global__ void __launch_bounds__(kCeilingMaxWarps * 32)
sk_pipe_rate_kernel(uint32_t* __restrict__ io, unsigned long long* __restrict__ cycles) {
    uint32_t a[8], b[8];
    unsigned long long p[8], q[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i] = io[i * 32 + (threadIdx.x & 31)];
        b[i] = io[256 + i * 32 + (threadIdx.x & 31)];
        p[i] = pack2(io[512 + i * 32 + (threadIdx.x & 31)], io[768 + i * 32 + (threadIdx.x & 31)]);
        q[i] = pack2(io[1024 + i * 32 + (threadIdx.x & 31)], io[1280 + i * 32 + (threadIdx.x & 31)]);
    }
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kPipeIters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE == 3 || MODE == 5 || MODE == 6 || MODE == 8) asm volatile("dp4a.s32.s32 %0, %1, %1, %0;" : "+r"(a[i]) : "r"(b[i]));
            if (MODE == 4 || MODE == 7) asm volatile("prmt.b32 %0, %0, %1, 0x5140;" : "+r"(a[i]) : "r"(b[i]));
            if (MODE == 8) asm volatile("prmt.b32 %0, %0, %1, 0x5140;" : "+r"(b[i]) : "r"(a[(i + 3) & 7]));
            if (MODE == 0) asm volatile("fma.rn.f32 %0, %1, %1, %0;" : "+r"(a[i]) : "r"(b[i]));
            if (MODE == 6) asm volatile("fma.rn.f32 %0, %1, %1, %0;" : "+r"(b[i]) : "r"(a[i]));
            if (MODE == 1 || MODE == 5 || MODE == 7) asm volatile("fma.rn.f32x2 %0, %1, %1, %0;" : "+l"(p[i]) : "l"(q[i]));
            if (MODE == 2) asm volatile("sub.rn.f32x2 %0, %1, %0;" : "+l"(p[i]) : "l"(q[i]));
        }
    }
    __syncthreads();
    const long long t1 = clock64();
    uint32_t x = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t lo, hi;
        unpack2(p[i], lo, hi);
        x ^= a[i] ^ b[i] ^ lo ^ hi;
    }
    io[2048 + blockIdx.x * blockDim.x + threadIdx.x] = x;
    if (blockIdx.x == 0 && threadIdx.x == 0) *cycles = (unsigned long long)(t1 - t0);
}

}  // namespace sk
