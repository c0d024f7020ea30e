// sk_ceiling.cuh — measurement only: the SM-side ceiling of the hot loop.
//
// The stream kernel's tile loop (accumulate16 of sk_device.cuh: a1-a3 for 16 samples per lane and
// 128-bit shared-memory read) run on a shared-memory tile that never changes: no global-memory
// traffic, no TMA, no barrier waits, no epilogue.  One CTA per SM, `warps` warps per CTA (warp i
// sits on sub-partition i % 4), every warp on its own 8 KiB tile, the accumulators read out every
// 8 tiles (128 samples per lane: AccChain2's limit) as in the kernel.  The elapsed SM cycles of
// CTA 0 give the cycles one sub-partition needs per 32 samples (one sample per lane) — what the
// instruction mix costs when nothing else is in the way.  bench.py reports it beside the roofline
// (DESIGN.md section 6); no product path calls this.
#pragma once
#include "sk_tma.cuh"

namespace sk {

constexpr int kCeilingMaxWarps = 16;
constexpr int kCeilingTilesPerReadout = 8;

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
            for (int i = 0; i < NLD; ++i) accumulate16(acc, lds128(src + i * RPW * W), kc);
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

}  // namespace sk
