// sk_tma.cuh — the fused SK kernel with TMA staging (sm_100a): the hot path.
//
// One WARP per unit, one warp per CTA.  A unit is one (cell, slab): M time rows x W = 16*L
// contiguous inputs.  The warp streams its unit through a private shared-memory ring of kStages
// tiles; a tile is kTileBytes = R rows x W bytes (R = kTileBytes / W) fetched by ONE 2-D TMA bulk
// copy (cp.async.bulk.tensor -> SASS UTMALDG) that signals an mbarrier when its bytes have landed.
// Lane 0 refills a slot as soon as the warp has consumed it, so the bytes in flight per SM are
// (resident warps) x kStages x kTileBytes, independent of registers, and the lanes only ever read
// shared memory.  No CTA-wide barrier exists anywhere: warps never wait for one another, and the
// hardware block scheduler deals units to SMs one warp at a time (even to within one unit).
// The arithmetic, the per-unit float64 partial and the finalisation are those of sk_kernels.cuh.
#pragma once
#include <cuda.h>

#include "sk_kernels.cuh"

namespace sk {

#ifndef SK_TILE_BYTES
#define SK_TILE_BYTES 4096
#endif
#ifndef SK_STAGES
#define SK_STAGES 2
#endif
#ifndef SK_MINCTAS
#define SK_MINCTAS 24
#endif
constexpr int kTileBytes = SK_TILE_BYTES;          // bytes per TMA tile (R rows x W inputs)
constexpr int kStages = SK_STAGES;                 // tiles in flight per warp
constexpr int kStreamMinCtas = SK_MINCTAS;         // resident warps per SM the register budget allows
constexpr size_t kStreamSmemBytes = (size_t)kStages * kTileBytes + kStages * 8;

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
// 2-D tiled TMA load: box (W bytes, R rows) at (x = byte in row, y = time row).
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

template <int L>
__global__ void __launch_bounds__(32, kStreamMinCtas)
sk_stream_kernel(const __grid_constant__ CUtensorMap tmap, const FrameParams p) {
    constexpr int RPW = 32 / L;                    // rows covered by one warp-wide 128-bit read
    constexpr int W = 16 * L;                      // slab width in inputs (= bytes)
    constexpr int R = kTileBytes / W;              // rows per tile
    constexpr int NLD = R / RPW;                   // 128-bit reads per lane per tile
    static_assert(R % RPW == 0 && NLD >= 1, "tile shape");
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x;
    const uint32_t ring = smem_addr(smem);
    const uint32_t bars = ring + kStages * kTileBytes;

    // grid = (slabs, F, B): no integer division on the way to the first load
    const uint32_t slab = blockIdx.x, f = blockIdx.y, b = blockIdx.z;
    const uint32_t cell = b * p.F + f;
    const uint32_t x0 = f * p.E + slab * W, y0 = b * p.M;
    const uint32_t full = p.M / R;                 // tiles with all R rows inside the block
    const uint32_t tiles = (p.M + R - 1) / R;

    // Programmatic dependent launch: let the next grid on the stream start filling SM slots as
    // they free up; wait for the previous grid before the first read unless the caller promised
    // that nothing upstream writes our inputs (then only before the first write, below).
    asm volatile("griddepcontrol.launch_dependents;");
    if (!p.inputs_ready) asm volatile("griddepcontrol.wait;" ::: "memory");

    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            if ((uint32_t)s < tiles) {
                mbar_expect_tx(bars + 8 * s, kTileBytes);
                tma_load_tile(ring + s * kTileBytes, &tmap, x0, y0 + s * R, bars + 8 * s);
            }
        }
    }
    __syncwarp();

    const int cl = lane % L, r0 = lane / L;
    const uint32_t e0 = (slab * L + cl) * 16u;
    const bool active = e0 < p.E;
    const uint32_t lane_off = r0 * W + cl * 16;

    UnpackConsts kc;
    kc.init();
    AccSplit acc;
    acc.reset();
    uint32_t n = 0, t = 0, parity = 0;
    uint32_t ynext = y0 + kStages * R;             // first row of the tile the next refill fetches
    // rounds of kStages full tiles: slot numbers are compile-time constants
    while (t + kStages <= full) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            const uint32_t bar = bars + 8 * s;
            const uint32_t src = ring + s * kTileBytes + lane_off;
            mbar_wait(bar, parity);
#pragma unroll
            for (int i = 0; i < NLD; ++i) acc.add16(lds128(src + i * RPW * W), kc);
            __syncwarp();                          // every lane has consumed this slot: refill it
            if (lane == 0 && t + s + kStages < tiles) {
                mbar_expect_tx(bar, kTileBytes);
                tma_load_tile(ring + s * kTileBytes, &tmap, x0, ynext + s * R, bar);
            }
        }
        t += kStages;
        ynext += kStages * R;
        parity ^= 1;
        n += kStages * NLD;
    }
    // what is left (fewer than kStages full tiles, then a ragged one) is already on its way
    for (uint32_t s = 0; t < tiles; ++t, ++s) {
        const uint32_t src = ring + s * kTileBytes + lane_off;
        mbar_wait(bars + 8 * s, parity);
        const uint32_t rows = min((uint32_t)R, p.M - t * R);
        for (uint32_t r = r0; r < rows; r += RPW) {
            acc.add16(lds128(src + (r - r0) * W), kc);
            ++n;
        }
    }

    if (p.inputs_ready) asm volatile("griddepcontrol.wait;" ::: "memory");   // before the first write

    uint32_t S1[16], S2[16];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            acc.read(i, k, n, S1[4 * i + k], S2[4 * i + k]);
            if (!active) { S1[4 * i + k] = 0; S2[4 * i + k] = 0; }
        }
    }
    const int base = reduce_scatter_rows<L>(S1, S2, r0);
    constexpr int kOwn = Owned<L>::value;
    const bool owner = (RPW <= 16) || (r0 < 16);
    const uint32_t e_first = e0 + base;
    if (p.S1out && active && owner) {
        uint32_t* o1 = p.S1out + (size_t)cell * p.E + e_first;
        uint32_t* o2 = p.S2out + (size_t)cell * p.E + e_first;
        if (kOwn % 4 == 0) {
#pragma unroll
            for (int i = 0; i < kOwn / 4; ++i) {
                reinterpret_cast<uint4*>(o1)[i] = make_uint4(S1[4 * i], S1[4 * i + 1], S1[4 * i + 2], S1[4 * i + 3]);
                reinterpret_cast<uint4*>(o2)[i] = make_uint4(S2[4 * i], S2[4 * i + 1], S2[4 * i + 2], S2[4 * i + 3]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < kOwn; ++i) { o1[i] = S1[i]; o2[i] = S2[i]; }
        }
    }
    if (p.SK) publish_and_finalize(p, cell, slab, lane, unit_partial<L>(p, active, owner, e_first, S1, S2));
}

}  // namespace sk
