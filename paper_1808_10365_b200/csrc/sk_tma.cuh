// sk_tma.cuh — the fused SK kernel with TMA staging (sm_100a): the hot path for wide arrays.
//
// Every warp is an independent worker with a private shared-memory ring of kStages tiles.  A tile
// is kRows time rows x 256 contiguous inputs of one cell, fetched by ONE 2-D TMA bulk copy
// (cp.async.bulk.tensor -> SASS UTMALDG) that signals an mbarrier when its bytes have landed.
// Lane 0 keeps the ring kStages tiles ahead of the arithmetic, across unit boundaries, so the
// bytes in flight per SM (warps x kStages x tile) do not depend on registers or occupancy and the
// lanes only ever wait on shared memory.  Units (cell, 256-input slab) are dealt to warps
// round-robin over CTAs first, so every SM gets the same number of units to within one.
// The arithmetic, the per-unit float64 partial and the finalisation are those of sk_kernels.cuh.
#pragma once
#include <cuda.h>

#include "sk_kernels.cuh"

namespace sk {

constexpr int kTmaWarps = 8;                       // workers per CTA
constexpr int kTmaRows = 16;                       // time rows per tile
constexpr int kTmaStages = 3;                      // tiles in flight per warp
constexpr int kTmaSlab = 256;                      // inputs (bytes) per row of a tile
constexpr int kTmaTileBytes = kTmaRows * kTmaSlab;
constexpr int kTmaCtasPerSm = 2;
constexpr size_t kTmaSmemBytes = (size_t)kTmaWarps * kTmaStages * kTmaTileBytes + kTmaWarps * kTmaStages * 8;

__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
// 2-D tiled TMA load: box (kTmaSlab bytes, kTmaRows rows) at (x = byte in row, y = time row).
__device__ __forceinline__ void tma_load_tile(uint32_t dst, const CUtensorMap* tmap, uint32_t x, uint32_t y,
                                              uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tmap), "r"(x), "r"(y), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}

template <class Acc>
__global__ void __launch_bounds__(kTmaWarps * 32, kTmaCtasPerSm)
sk_frame_tma_kernel(const __grid_constant__ CUtensorMap tmap, const FrameParams p) {
    constexpr int L = 16, RPW = 2;
    extern __shared__ __align__(128) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t ring = smem_addr(smem) + warp * (kTmaStages * kTmaTileBytes);
    const uint32_t bars = smem_addr(smem) + kTmaWarps * kTmaStages * kTmaTileBytes + warp * (kTmaStages * 8);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kTmaStages; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();

    const int cl = lane & 15, r0 = lane >> 4;
    const uint32_t ustep = gridDim.x * kTmaWarps;
    const uint32_t ufirst = blockIdx.x + gridDim.x * warp;      // CTA-major dealing: balanced per SM
    const uint32_t tiles = (p.M + kTmaRows - 1) / kTmaRows;     // tiles per unit

    // ---- producer state (lane 0 only): next tile to request
    uint32_t pu = ufirst, pt = 0, pslot = 0;
    auto issue_one = [&]() {
        if (pu >= p.nunits) return;
        const uint32_t slab = pu % p.slabs, cell = pu / p.slabs;
        const uint32_t b = cell / p.F, f = cell % p.F;
        const uint32_t bar = bars + 8 * pslot;
        mbar_expect_tx(bar, kTmaTileBytes);
        tma_load_tile(ring + pslot * kTmaTileBytes, &tmap, f * p.E + slab * kTmaSlab, b * p.M + pt * kTmaRows, bar);
        pslot = (pslot + 1 == kTmaStages) ? 0 : pslot + 1;
        if (++pt == tiles) { pt = 0; pu += ustep; }
    };
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kTmaStages; ++s) issue_one();
    }

    UnpackConsts kc;
    kc.init();
    uint32_t cslot = 0, cparity = 0;
    for (uint32_t u = ufirst; u < p.nunits; u += ustep) {
        const uint32_t slab = u % p.slabs, cell = u / p.slabs;
        const uint32_t e0 = (slab * L + cl) * 16u;
        const bool active = e0 < p.E;
        Acc acc[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) acc[k].reset();
        uint32_t n = 0;
        for (uint32_t t = 0; t < tiles; ++t) {
            mbar_wait(bars + 8 * cslot, cparity);
            const uint32_t rows = min((uint32_t)kTmaRows, p.M - t * kTmaRows);
            const uint32_t src = ring + cslot * kTmaTileBytes + r0 * kTmaSlab + cl * 16;
            if (rows == kTmaRows) {
                uint4 v[kTmaRows / RPW];
#pragma unroll
                for (int i = 0; i < kTmaRows / RPW; ++i) v[i] = lds128(src + i * RPW * kTmaSlab);
#pragma unroll
                for (int i = 0; i < kTmaRows / RPW; ++i) accumulate16(acc, v[i], kc);
                n += kTmaRows / RPW;
            } else {
                for (uint32_t r = r0; r < rows; r += RPW) {
                    accumulate16(acc, lds128(src + (r - r0) * kTmaSlab), kc);
                    ++n;
                }
            }
            __syncwarp();                      // every lane has consumed this slot: refill it
            if (lane == 0) issue_one();
            if (++cslot == kTmaStages) { cslot = 0; cparity ^= 1; }
        }
        uint32_t S1[16], S2[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            acc[k].read(n, S1[k], S2[k]);
            if (!active) { S1[k] = 0; S2[k] = 0; }
        }
        const int base = reduce_scatter_rows<L>(S1, S2, r0);
        constexpr int kOwn = Owned<L>::value;
        const uint32_t e_first = e0 + base;
        if (p.S1out && active) {
            uint4* o1 = reinterpret_cast<uint4*>(p.S1out + (size_t)cell * p.E + e_first);
            uint4* o2 = reinterpret_cast<uint4*>(p.S2out + (size_t)cell * p.E + e_first);
#pragma unroll
            for (int i = 0; i < kOwn / 4; ++i) {
                o1[i] = make_uint4(S1[4 * i], S1[4 * i + 1], S1[4 * i + 2], S1[4 * i + 3]);
                o2[i] = make_uint4(S2[4 * i], S2[4 * i + 1], S2[4 * i + 2], S2[4 * i + 3]);
            }
        }
        if (p.SK) publish_and_finalize(p, cell, slab, lane, unit_partial<L>(p, active, true, e_first, S1, S2));
    }
}

}  // namespace sk
