// sk_tma.cuh — the fused SK kernel with TMA staging (sm_100a): the hot path.
//
// One WARP per unit, one warp per CTA.  A unit is one (row range, frequency, slab): p.bpu
// consecutive M-row blocks x W = 16*L contiguous inputs.  bpu = 1 (one cell) for the plain
// sk_frame at M >= 256; a multiple of 2^(NLEV-1), so that a unit holds whole cells of the longest
// of the NLEV integration lengths asked for; and several short blocks when M < 256, so that the
// unit's set-up is paid once per 256 rows.  The warp streams its rows through a
// private shared-memory ring of kStages tiles; a tile is kTileBytes = R rows x W bytes
// (R = kTileBytes / W) fetched by ONE 2-D TMA bulk copy (cp.async.bulk.tensor -> SASS UTMALDG)
// that signals an mbarrier when its bytes have landed.  Lane 0 refills a slot as soon as the warp
// has consumed it, so the bytes in flight per SM are (resident warps) x kStages x kTileBytes,
// independent of registers, and the lanes only ever read shared memory.  No CTA-wide barrier
// exists anywhere: warps never wait for one another, and the hardware block scheduler deals units
// to SMs one warp at a time (even to within one unit).
//
// The rows are consumed in chunks of p.chunk rows (a divisor of M, at most 128 rows per lane: the
// exactness limit of AccChain2).  After each chunk the lane's 16 x (S1, S2) are read out of the
// packed accumulators, the row groups are reduce-scattered (integers, exact) and, with CHUNKED,
// added to the running sums of the current M-row block.  When a block is complete its Eq. 11 terms
// go into the unit's float64 partial of length M; with NLEV > 1 the block's integer sums are also
// added to the running sums of lengths 2M, 4M, ... ("a variety of integration
// lengths"), each of which is published when its last block has been added.  The TMA ring never
// drains between chunks or blocks.
// The arithmetic, the per-unit float64 partial and the finalisation are those of sk_kernels.cuh.
#pragma once
#include <cuda.h>

#include "sk_kernels.cuh"

namespace sk {

// 8 KiB tiles x 2 stages x 13 resident warps per SM = 208 KiB in flight per SM.  Measured on B200
// (config 2, GB/s burst / power-capped): 4 KiB x 2 x 24 warps 4760 / 4160 (80 registers: the paired
// accumulators spill), 4 KiB x 2 x 20 5930 / 4820, 4 KiB x 3 x 16 6060 / 4970, 8 KiB x 2 x 13 6290 / 5140.
constexpr int kTileBytes = 8192;                   // bytes per TMA tile (R rows x W inputs)
constexpr int kStages = 2;                         // tiles in flight per warp
constexpr int kStreamMinCtas = 13;                 // resident warps per SM (16 KiB + barriers of shared memory each)
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

// 2-D tiled TMA store of one box from shared memory (bulk async-group completion).
__device__ __forceinline__ void tma_store_tile(const CUtensorMap* tmap, uint32_t x, uint32_t y, uint32_t src) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];"
                 ::"l"(tmap), "r"(x), "r"(y), "r"(src) : "memory");
}

// a8 for the stream kernel ("excision"): every byte of a flagged cell becomes 0x88.  The
// cell is rows [row0, row0 + rows) of frequency f, all E inputs; the whole warp calls.  A finalizer
// excises the WHOLE cell (512 KiB on config 1) while it holds an SM slot, so how it writes decides the
// kernel's tail when many cells are flagged.  When the warp's TMA ring is idle (ring_free: the unit's
// last tile has been consumed) and the cell is a whole number of boxes (E % W == 0; rows % R == 0 holds
// for this kernel), one ring slot is filled with 0x88 and the cell is written as rows/R x E/W bulk tensor
// stores of 8 KiB through the same tensor map the loads use: 64 instructions per config-1 cell instead
// of 1024 128-bit stores with their address arithmetic.  Otherwise (a cell that completes in the middle
// of a unit, a ragged last slab) the lanes store the bytes themselves.
template <int L>
__device__ __forceinline__ void excise_cell_stream(const CUtensorMap* tmap, const FrameParams& p, uint32_t ring,
                                                   bool ring_free, uint32_t row0, uint32_t rows, uint32_t f, int lane) {
    constexpr uint32_t W = 16 * L, R = kTileBytes / W;
    if (!ring_free || p.E % W != 0u || rows % R != 0u) {
        excise_cell<true>(p, row0, rows, f, (uint32_t)lane, 32u);
        return;
    }
#pragma unroll
    for (int i = 0; i < kTileBytes / (32 * 16); ++i)
        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(ring + (uint32_t)(i * 32 + lane) * 16u), "r"(0x88888888u)
                     : "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // the fill, visible to the TMA engine
    __syncwarp();
    const uint32_t nx = p.E / W, n = nx * (rows / R);
    for (uint32_t k = (uint32_t)lane; k < n; k += 32u) {
        const uint32_t iy = k / nx, ix = k - iy * nx;
        tma_store_tile(tmap, f * p.E + ix * W, row0 + iy * R, ring);
    }
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");         // written, not only read: the slot may be reused or freed
    __syncwarp();
}

// 128 registers = 13 resident warps.  Several integration lengths keep 16 more running sums per
// length and lane (touched once per M-row block) in registers: a higher limit, fewer resident warps.
// Measured on config 2 with 4 lengths (us per frame; 210 for one length): all in registers,
// 232-register limit = 8 warps 257; sums in the warp's shared memory, 168 registers = 9 warps 272;
// 128 registers with the sums spilled to local memory 409.
constexpr int stream_max_regs(int nlev) { return nlev == 1 ? 128 : nlev == 2 ? 200 : 232; }

// VAR: kVarProduct in the product library; the bench library instantiates kVarMemOnly (sk_device.cuh).
template <int L, int NLEV, bool CHUNKED, int VAR = kVarProduct>
__global__ void __maxnreg__(stream_max_regs(NLEV))
sk_stream_kernel(const __grid_constant__ CUtensorMap tmap, const FrameParams p) {
    constexpr int RPW = 32 / L;                    // rows covered by one warp-wide 128-bit read
    constexpr int W = 16 * L;                      // slab width in inputs (= bytes)
    constexpr int R = kTileBytes / W;              // rows per tile
    constexpr int NLD = R / RPW;                   // 128-bit reads per lane per tile
    constexpr int kOwn = Owned<L>::value;          // inputs a lane owns after the reduce-scatter
    static_assert(R % RPW == 0 && NLD >= 1, "tile shape");
    static_assert(NLEV >= 1 && NLEV <= kMaxLevels, "levels");
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x;
    const uint32_t ring = smem_addr(smem);
    const uint32_t bars = ring + kStages * kTileBytes;

    // grid = (slabs, F, B / bpu): no integer division on the way to the first load
    const uint32_t slab = blockIdx.x, f = blockIdx.y;
    const uint32_t x0 = f * p.E + slab * W;
    const uint32_t tpc = p.chunk / R;              // tiles per chunk (the host makes chunks of whole tiles)
    const uint32_t total = p.unit_tiles;           // tiles of this unit: M * bpu / R (from the host: no division here)
    const uint32_t y0 = blockIdx.z * p.M * p.bpu;

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
            if ((uint32_t)s < total) {
                mbar_expect_tx(bars + 8 * s, kTileBytes);
                tma_load_tile(ring + s * kTileBytes, &tmap, x0, y0 + s * R, bars + 8 * s);
            }
        }
    }
    __syncwarp();

    const uint32_t lane_off = (lane / L) * W + (lane % L) * 16;

    UnpackConsts kc;
    kc.init();
    AccChain2 acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k].reset();
    uint32_t run1[CHUNKED ? kOwn : 1], run2[CHUNKED ? kOwn : 1];          // the current block, chunk by chunk
    uint32_t up1[NLEV > 1 ? NLEV - 1 : 1][kOwn], up2[NLEV > 1 ? NLEV - 1 : 1][kOwn];   // lengths 2M, 4M, ...
    if (CHUNKED) {
#pragma unroll
        for (int i = 0; i < kOwn; ++i) run1[i] = run2[i] = 0;
    }
#pragma unroll
    for (int l = 0; l < NLEV - 1; ++l)
#pragma unroll
        for (int i = 0; i < kOwn; ++i) up1[l][i] = up2[l][i] = 0;

    uint32_t s = 0, parity = 0, tc = 0, cq = 0, blk = 0;
    for (uint32_t g = 0; g < total; ++g) {
        const uint32_t src = ring + s * kTileBytes + lane_off;
        mbar_wait(bars + 8 * s, parity);
#pragma unroll
        for (int i = 0; i < NLD; ++i) accumulate16<AccChain2, VAR>(acc, lds128(src + i * RPW * W), kc);
        __syncwarp();                              // every lane has consumed this slot: refill it
        if (lane == 0 && g + kStages < total) {
            mbar_expect_tx(bars + 8 * s, kTileBytes);
            tma_load_tile(ring + s * kTileBytes, &tmap, x0, y0 + (g + kStages) * R, bars + 8 * s);
        }
        if (++s == kStages) { s = 0; parity ^= 1; }
        if (++tc < tpc) continue;
        tc = 0;

        // ---- chunk read-out: integer sums of the lane's 16 inputs, row groups reduce-scattered
        // (what the tile loop does not need is recomputed here, to keep its registers free)
        const uint32_t sb = blockIdx.z;
        const int cl = lane % L, r0 = lane / L;
        const uint32_t e0 = (slab * L + cl) * 16u;
        const bool active = e0 < p.E;
        const bool owner = (RPW <= 16) || (r0 < 16);
        const uint32_t q = p.M / p.chunk;          // chunks per block
        uint32_t S1[16], S2[16];
        read16(acc, 0u, S1, S2);
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k].reset();
        if (p.E % W != 0u) {                       // a ragged last slab (warp-uniform test): its lanes beyond E add nothing
            if (!active) {
#pragma unroll
                for (int k = 0; k < 16; ++k) { S1[k] = 0; S2[k] = 0; }
            }
        }
        const int base = reduce_scatter_rows<L>(S1, S2, r0);
        const uint32_t e_first = e0 + base;
        if (CHUNKED) {
#pragma unroll
            for (int i = 0; i < kOwn; ++i) { run1[i] += S1[i]; run2[i] += S2[i]; }
            if (++cq < q) continue;
            cq = 0;
#pragma unroll
            for (int i = 0; i < kOwn; ++i) { S1[i] = run1[i]; S2[i] = run2[i]; run1[i] = run2[i] = 0; }
        }

        // ---- a block of M rows is complete
        if (p.inputs_ready) asm volatile("griddepcontrol.wait;" ::: "memory");   // before the first write
        const uint32_t b0 = sb * p.bpu + blk;
        if (p.S1out && active && owner) {
            const size_t cell = (size_t)b0 * p.F + f;
            uint32_t* o1 = p.S1out + cell * p.E + e_first;
            uint32_t* o2 = p.S2out + cell * p.E + e_first;
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
        const bool ring_free = g + 1u == total;    // the unit's last tile: nothing is in flight into the ring any more
        if (p.lev[0].SK) {
            if (publish_and_finalize<true>(p, 0, b0, f, slab, lane,
                                           unit_partial<L>(p, (double)p.M, active, owner, e_first, S1, S2)))
                excise_cell_stream<L>(&tmap, p, ring, ring_free, b0 * p.M, p.M, f, lane);
        }
        ++blk;
#pragma unroll
        for (int l = 1; l < NLEV; ++l) {
#pragma unroll
            for (int i = 0; i < kOwn; ++i) { up1[l - 1][i] += S1[i]; up2[l - 1][i] += S2[i]; }
            if ((blk & ((1u << l) - 1u)) == 0u) {  // the last block of a cell of length M << l
                if (publish_and_finalize<true>(p, l, (b0 >> l), f, slab, lane,
                                               unit_partial<L>(p, (double)(p.M << l), active, owner, e_first, up1[l - 1], up2[l - 1])))
                    excise_cell_stream<L>(&tmap, p, ring, ring_free, (b0 >> l) * (p.M << l), p.M << l, f, lane);
#pragma unroll
                for (int i = 0; i < kOwn; ++i) up1[l - 1][i] = up2[l - 1][i] = 0;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The same kernel for a block length that is NOT a whole number of tiles (M = 250, 1000, ...): a
// block is tpb = ceil(M / R) tiles, the last of them partial.  Every block's first tile starts at the
// block's first row (a TMA box may start at any row), the partial tile is fetched whole (its surplus
// rows belong to the next block, or lie beyond T and come back as zeros) and only its first
// M - (tpb-1) R rows are added; the accumulators are read out every 8 tiles (128 samples per lane)
// and at every block end.  One integration length, chunked running sums; everything after the
// row loop is the code of sk_stream_kernel.  The host uses it when M >= 2 R (at most a third of
// the fetched rows are surplus); shorter ragged blocks take the direct-load kernel.
constexpr int kRaggedTilesPerReadout = 8;

template <int L>
__global__ void __maxnreg__(128)
sk_stream_ragged_kernel(const __grid_constant__ CUtensorMap tmap, const FrameParams p) {
    constexpr int RPW = 32 / L;
    constexpr int W = 16 * L;
    constexpr int R = kTileBytes / W;
    constexpr int NLD = R / RPW;
    constexpr int kOwn = Owned<L>::value;
    static_assert(kRaggedTilesPerReadout * NLD <= (int)AccChain2::kMaxSamples, "read-out interval");
    extern __shared__ __align__(128) uint8_t smem[];
    const int lane = threadIdx.x;
    const uint32_t ring = smem_addr(smem);
    const uint32_t bars = ring + kStages * kTileBytes;
    const uint32_t slab = blockIdx.x, f = blockIdx.y;
    const uint32_t x0 = f * p.E + slab * W;
    const uint32_t tpb = p.tpb, total = p.unit_tiles;          // tiles per block, tiles of this unit (tpb * bpu)
    const uint32_t last_rows = p.M - (tpb - 1u) * R;            // rows of a block's last tile that belong to it

    asm volatile("griddepcontrol.launch_dependents;");
    if (!p.inputs_ready) asm volatile("griddepcontrol.wait;" ::: "memory");

    // producer (lane 0): the next tile to request is tile pk of the block that starts at row py
    uint32_t pk = 0, py = blockIdx.z * p.M * p.bpu;
    auto request = [&](uint32_t stage) {
        mbar_expect_tx(bars + 8 * stage, kTileBytes);
        tma_load_tile(ring + stage * kTileBytes, &tmap, x0, py + pk * R, bars + 8 * stage);
        if (++pk == tpb) { pk = 0; py += p.M; }
    };
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) mbar_init(bars + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
#pragma unroll
        for (int s = 0; s < kStages; ++s)
            if ((uint32_t)s < total) request(s);
    }
    __syncwarp();

    const int cl = lane % L, r0 = lane / L;
    const uint32_t lane_off = r0 * W + cl * 16;
    const uint32_t e0 = (slab * L + cl) * 16u;
    const bool active = e0 < p.E;
    const bool owner = (RPW <= 16) || (r0 < 16);

    UnpackConsts kc;
    kc.init();
    AccChain2 acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k].reset();
    uint32_t run1[kOwn], run2[kOwn];
#pragma unroll
    for (int i = 0; i < kOwn; ++i) run1[i] = run2[i] = 0;

    uint32_t s = 0, parity = 0, tc = 0, k = 0, blk = 0;
    for (uint32_t g = 0; g < total; ++g) {
        const uint32_t src = ring + s * kTileBytes + lane_off;
        mbar_wait(bars + 8 * s, parity);
        if (k + 1u < tpb || last_rows == (uint32_t)R) {
#pragma unroll
            for (int i = 0; i < NLD; ++i) accumulate16(acc, lds128(src + i * RPW * W), kc);
        } else {
            // the block's last tile: row i * RPW + r0 of the tile counts only while it is below last_rows
            for (uint32_t i = 0; i * RPW + (uint32_t)r0 < last_rows; ++i) accumulate16(acc, lds128(src + i * RPW * W), kc);
        }
        __syncwarp();
        if (lane == 0 && g + kStages < total) request(s);
        if (++s == kStages) { s = 0; parity ^= 1; }
        const bool block_end = ++k == tpb;
        if (++tc < (uint32_t)kRaggedTilesPerReadout && !block_end) continue;
        tc = 0;

        uint32_t S1[16], S2[16];
        read16(acc, 0u, S1, S2);
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[i].reset();
        if (!active) {
#pragma unroll
            for (int i = 0; i < 16; ++i) { S1[i] = 0; S2[i] = 0; }
        }
        const int base = reduce_scatter_rows<L>(S1, S2, r0);
        const uint32_t e_first = e0 + base;
#pragma unroll
        for (int i = 0; i < kOwn; ++i) { run1[i] += S1[i]; run2[i] += S2[i]; }
        if (!block_end) continue;
        k = 0;

        // ---- a block of M rows is complete
        if (p.inputs_ready) asm volatile("griddepcontrol.wait;" ::: "memory");   // before the first write
        const uint32_t b0 = blockIdx.z * p.bpu + blk;
        if (p.S1out && active && owner) {
            const size_t cell = (size_t)b0 * p.F + f;
            uint32_t* o1 = p.S1out + cell * p.E + e_first;
            uint32_t* o2 = p.S2out + cell * p.E + e_first;
#pragma unroll
            for (int i = 0; i < kOwn; ++i) { o1[i] = run1[i]; o2[i] = run2[i]; }
        }
        if (p.lev[0].SK)
            publish_and_finalize(p, 0, b0, f, slab, lane, unit_partial<L>(p, (double)p.M, active, owner, e_first, run1, run2));
#pragma unroll
        for (int i = 0; i < kOwn; ++i) run1[i] = run2[i] = 0;
        ++blk;
    }
}

}  // namespace sk
