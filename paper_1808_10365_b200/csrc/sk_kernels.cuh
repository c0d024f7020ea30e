// sk_kernels.cuh — the kernels of the SK hot path (sm_100a).  See sk_device.cuh for the arithmetic.
//
// Work decomposition (vector path, E % 16 == 0, 16-byte aligned data):
//   unit  = one (cell, slab): M rows x W = 16*L contiguous inputs, handled by ONE warp.
//   lane  = (row group r0 = lane / L, column cl = lane % L): 16 inputs e0..e0+15 of every
//           RPW-th row (RPW = 32/L rows are covered by one warp-wide 128-bit load).
//   After the row loop the RPW row groups are summed with shuffles (integers: exact), each lane
//   evaluates Eq. 11's term for its share of the 16 inputs in float64, the warp adds them with a
//   canonical tree (below), and the unit's partial S2bar goes to the workspace.  The last unit of a
//   cell to arrive (one atomic counter per cell) merges the partials in the same tree, evaluates
//   Eq. 14, rounds to float32, takes the flag decision, and resets the counter.
//   The order of every floating-point sum is fixed, so results are bit-reproducible.
#pragma once
#include "sk_device.cuh"

namespace sk {

constexpr int kMaxLevels = 4;     // integration lengths M, 2M, 4M, 8M from one pass (sk_frame_multi)

// Outputs of one integration length M << l: arrays [B >> l][F]; workspace of that length.
struct LevelOut {
    float* SK;                // nullptr at level 0 = power sums only
    uint8_t* mask;            // or nullptr
    double* partial;          // workspace: [cells of this length][slabs]
    uint32_t* counter;        // workspace: [cells of this length], zero on entry, zero on exit
    float sk_mean;            // flag centre at this length
};

struct FrameParams {
    const uint8_t* data;      // [T][F][E]
    uint8_t* excise;          // == data when flagged cells are to be overwritten with 0x88, else nullptr
    uint32_t T, F, E, M, B;   // M = the shortest integration length, B = T / M
    const uint8_t* subset;    // E bytes or nullptr
    uint32_t first_n;         // used when subset == nullptr
    float n_sigma;
    LevelOut lev[kMaxLevels];
    uint32_t nlev;            // 1 for every call but sk_frame_multi
    uint32_t eq13;            // estimator: 0 = Eq. 14 (SK~), 1 = Eq. 13 (un-rescaled SK^)
    uint32_t* S1out;          // [B][F][E] or nullptr (length M only)
    uint32_t* S2out;
    const uint32_t* S1in;     // combine: read sums instead of data
    const uint32_t* S2in;
    uint32_t inputs_ready;    // stream kernel: read data before waiting for the previous grid
    uint32_t chunk;           // stream kernel: rows per accumulator read-out (divides M)
    uint32_t bpu;             // stream kernel: M-row blocks per unit (a multiple of 1 << (nlev-1))
    uint32_t unit_tiles;      // stream kernel: TMA tiles per unit = M * bpu / (rows per tile)
    uint32_t tpb;             // ragged stream kernel: tiles per block = ceil(M / rows per tile); unit_tiles = tpb * bpu
    uint32_t slabs;           // units per cell that are launched
    uint32_t nunits;          // cells * slabs
};

constexpr int kWarpsPerCta = 4;
constexpr int kUnroll = 8;     // 128-bit loads in flight per lane
constexpr int kMinCtasPerSm = 4;   // with this hint ptxas keeps a batch of loads in flight (<= 128 regs)

// Number of combined receivers N: first_n, or the count of non-zero subset bytes (whole warp).
__device__ __forceinline__ uint32_t count_receivers(const FrameParams& p, int lane) {
    if (!p.subset) return p.first_n;
    uint32_t n = 0;
    for (uint32_t e = lane; e < p.E; e += 32) n += (__ldg(p.subset + e) != 0);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n += __shfl_xor_sync(0xffffffffu, n, o);
    return n;
}

__device__ __forceinline__ bool selected(const FrameParams& p, uint32_t e) {
    return p.subset ? (__ldg(p.subset + e) != 0) : (e < p.first_n);
}

// Sum the RPW row groups of a warp and scatter the result (recursive halving): on return lane
// (r0, cl) holds kOwned<L> fully summed inputs starting at input offset `base` of its 16, in
// v[0..kOwned).  Integers: exact in any order.  Costs 16 shuffles per array instead of 16*log2(RPW).
template <int L> struct Owned { static constexpr int value = (16 * L / 32) > 0 ? (16 * L / 32) : 1; };

template <int L>
__device__ __forceinline__ int reduce_scatter_rows(uint32_t (&v1)[16], uint32_t (&v2)[16], int r0) {
    constexpr int RPW = 32 / L;
    int base = 0;
    int c = 16;
#pragma unroll
    for (int s = 0; (1 << s) < RPW; ++s) {
        const int o = L << s;
        const bool bit = (r0 >> s) & 1;
        if (c > 1) {
            const int h = c / 2;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (i < h) {
                    const uint32_t k1 = bit ? v1[i + h] : v1[i], g1 = bit ? v1[i] : v1[i + h];
                    const uint32_t k2 = bit ? v2[i + h] : v2[i], g2 = bit ? v2[i] : v2[i + h];
                    v1[i] = k1 + __shfl_xor_sync(0xffffffffu, g1, o);
                    v2[i] = k2 + __shfl_xor_sync(0xffffffffu, g2, o);
                }
            }
            base += bit ? h : 0;
            c = h;
        } else {                       // RPW = 32: two row groups share the last input
            v1[0] += __shfl_xor_sync(0xffffffffu, v1[0], o);
            v2[0] += __shfl_xor_sync(0xffffffffu, v2[0], o);
        }
    }
    return base;
}

// ---- a5: the canonical order of the sum over inputs -------------------------------------------
// S2bar = Tree(0, P), P = the power of two >= E, with
//   Tree(lo, 1) = term of input lo (0.0 if lo >= E or the input is not selected),
//   Tree(lo, n) = Tree(lo, n/2) + Tree(lo + n/2, n/2).
// The order is a property of the input indices alone: it does not depend on the slab width, the
// kernel, the launch flags or the SM count, so every path gives the same float64 S2bar (adding an
// absent subtree's 0.0 is exact, and a + b = b + a).  A lane adds its aligned block pairwise, the
// warp climbs the remaining levels of the unit's subtree with one xor-shuffle per level (the lane
// bit that holds each input bit follows from reduce_scatter_rows), and the finalizer merges the
// units' subtrees like a binary counter.

// a4 + a5 within a unit: Tree(unit's first input, 16 L), identical on all lanes on return.
// Md = the integration length the sums v1/v2 cover.
// v1/v2[0..kOwned) are the sums of inputs e_first ..; `owner` is false for the duplicate lanes
// when RPW = 32.  Called by both fused kernels and by the combine kernel.
template <int L>
__device__ __forceinline__ double unit_partial(const FrameParams& p, double Md, bool active, bool owner,
                                               uint32_t e_first, const uint32_t* v1, const uint32_t* v2) {
    constexpr int kOwn = Owned<L>::value;
    constexpr int RPW = 32 / L;
    const double MM = __dmul_rn(Md, Md);
    // which of the lane's inputs are combined: decided once, so that the kOwn divisions below
    // are straight-line code the scheduler can interleave
    uint32_t sel = 0;
    if (active && owner) {
        if (p.subset) {
#pragma unroll
            for (int i = 0; i < kOwn; ++i) sel |= (uint32_t)(__ldg(p.subset + e_first + i) != 0) << i;
        } else {
#pragma unroll
            for (int i = 0; i < kOwn; ++i) sel |= (uint32_t)(e_first + i < p.first_n) << i;
        }
    }
    double t[kOwn];
#pragma unroll
    for (int i = 0; i < kOwn; ++i) {
        const double x = eq11_term(Md, MM, v1[i], v2[i]);
        t[i] = ((sel >> i) & 1u) ? x : 0.0;
    }
#pragma unroll
    for (int h = 1; h < kOwn; h *= 2)
#pragma unroll
        for (int i = 0; i + h < kOwn; i += 2 * h) t[i] = __dadd_rn(t[i], t[i + h]);
    double x = t[0];
    // input bits log2(kOwn) .. 3 live in the row-group bits of the lane, highest stage first
#pragma unroll
    for (int o = 16; o >= L; o >>= 1)
        if (o < 32 && (RPW <= 16 || o < 16)) x = __dadd_rn(x, __shfl_xor_sync(0xffffffffu, x, o));
    // input bits 4 .. live in the column bits of the lane
#pragma unroll
    for (int o = 1; o < L; o <<= 1) x = __dadd_rn(x, __shfl_xor_sync(0xffffffffu, x, o));
    if (RPW == 32) x = __dadd_rn(x, __shfl_xor_sync(0xffffffffu, x, 16));   // duplicates hold 0.0
    return x;
}

// a5 across units: merge equal-sized subtrees in index order, like a binary counter: neighbours
// are added as soon as both exist; what is left at the end is folded from the smallest up (its
// missing siblings are absent inputs, i.e. 0.0).  Slots are indexed by unrolled constants only,
// so they stay in registers.
struct TreeMerge {
    static constexpr int kLevels = 20;
    double v[kLevels];
    uint32_t n = 0;                                 // subtrees pushed so far
    __device__ __forceinline__ void push(double x) {
        const uint32_t k = n++;
        bool placed = false;
#pragma unroll
        for (int l = 0; l < kLevels; ++l) {
            if (!placed) {
                if ((k >> l) & 1u) x = __dadd_rn(v[l], x);
                else { v[l] = x; placed = true; }
            }
        }
    }
    __device__ __forceinline__ double total() const {
        double x = 0.0;
        bool have = false;
#pragma unroll
        for (int l = 0; l < kLevels; ++l) {
            if ((n >> l) & 1u) {
                x = have ? __dadd_rn(v[l], x) : v[l];
                have = true;
            }
        }
        return x;
    }
};

// A unit's partial travels through the workspace without any fence: the slot is written by one
// relaxed 64-bit store whose bit pattern is never zero (a partial of +0.0 is stored as -0.0, which
// adds like 0.0), and the finalizer polls a slot until it is non-zero.  The arrival counter only
// elects the finalizer; it does not have to be ordered against the stores.
__device__ __forceinline__ void store_partial(double* slot, double x) {
    unsigned long long bits = (unsigned long long)__double_as_longlong(x);
    if (bits == 0ull) bits = 0x8000000000000000ull;
    asm volatile("st.relaxed.gpu.global.b64 [%0], %1;" ::"l"(slot), "l"(bits) : "memory");
}
__device__ __forceinline__ double poll_partial(const double* slot) {
    unsigned long long bits;
    do {
        asm volatile("ld.relaxed.gpu.global.b64 %0, [%1];" : "=l"(bits) : "l"(slot) : "memory");
    } while (bits == 0ull);
    return __longlong_as_double((long long)bits);
}

// a8: every byte of a flagged cell becomes 0x88 (the encoded 0+0i; "excision").  The
// cell is rows [row0, row0 + rows) of frequency f, all E inputs.  Called by `nthreads` threads
// (rank tid) once every unit of the cell has published its partial, i.e. after the cell's last
// read.  VEC: E % 16 == 0 and data 16-byte aligned.
template <bool VEC>
__device__ __forceinline__ void excise_cell(const FrameParams& p, uint32_t row0, uint32_t rows, uint32_t f,
                                            uint32_t tid, uint32_t nthreads) {
    const size_t rstride = (size_t)p.F * p.E;
    uint8_t* base = p.excise + ((size_t)row0 * p.F + f) * p.E;
    if (VEC) {
        const uint32_t vec_per_row = p.E / 16;
        const uint4 z = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
        for (uint32_t j = 0; j < rows; ++j) {
            uint4* row = reinterpret_cast<uint4*>(base + (size_t)j * rstride);
            for (uint32_t c = tid; c < vec_per_row; c += nthreads) row[c] = z;
        }
    } else {
        for (uint32_t j = 0; j < rows; ++j) {
            uint8_t* row = base + (size_t)j * rstride;
            for (uint32_t c = tid; c < p.E; c += nthreads) row[c] = 0x88;
        }
    }
}

// a6: the estimator from S2bar.  Eq. 14 (what CHIME runs) unless the caller asked for Eq. 13.
__device__ __forceinline__ float estimator(const FrameParams& p, double S2bar, double Md, double Nd) {
    return p.eq13 ? eq13_sk(S2bar, Md, Nd) : eq14_sk(S2bar, Md, Nd);
}

// a5 (across units) + a6 + a7 for one cell of integration length M << l; whole warp calls, lane 0
// writes; returns the flag decision on every lane.  32 units at a time: an aligned group of 32
// subtrees is summed with the canonical butterfly, groups are merged.
// POLL: the partials are workspace slots that may still be in flight (fused kernels); otherwise
// they are plain memory that is already complete (combine kernel: shared memory).
template <bool POLL>
__device__ __forceinline__ uint32_t finalize_cell(const FrameParams& p, int l, uint32_t cell, int lane,
                                                  const double* partials) {
    const uint32_t N = count_receivers(p, lane);
    auto load = [&](uint32_t s) -> double {
        if (s >= p.slabs) return 0.0;
        return POLL ? poll_partial(partials + s) : partials[s];
    };
    double S2bar = load(lane);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) S2bar = __dadd_rn(S2bar, __shfl_xor_sync(0xffffffffu, S2bar, o));
    if (p.slabs > 32) {                             // more than one group of 32 units: merge groups
        TreeMerge tm;
        tm.push(S2bar);
        for (uint32_t s0 = 32; s0 < p.slabs; s0 += 32) {
            double x = load(s0 + lane);
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) x = __dadd_rn(x, __shfl_xor_sync(0xffffffffu, x, o));
            tm.push(x);
        }
        S2bar = tm.total();
    }
    const double Md = (double)(p.M << l);
    const float sk = estimator(p, S2bar, Md, (double)N);
    const uint32_t flagged = flag_decision(sk, p.lev[l].sk_mean, flag_threshold(p.n_sigma, Md, (double)N));
    if (lane == 0) {
        p.lev[l].SK[cell] = sk;
        if (p.lev[l].mask) p.lev[l].mask[cell] = (uint8_t)flagged;
    }
    return p.lev[l].mask ? flagged : 0u;
}

// Fused kernels: publish the unit's partial of cell (b, f) at length M << l; the last unit of the
// cell to arrive finalizes it and, if asked to, excises it (every unit has finished reading the
// cell by then).
// DEFER: do not excise here; return 1 (on every lane) when the cell is flagged and has to be excised,
// so that the caller can do it its own way (the stream kernel: TMA bulk stores).  Otherwise returns 0.
template <bool DEFER = false>
__device__ __forceinline__ uint32_t publish_and_finalize(const FrameParams& p, int l, uint32_t b, uint32_t f,
                                                         uint32_t slab, int lane, double part) {
    const uint32_t cell = b * p.F + f;
    double* slots = p.lev[l].partial + (size_t)cell * p.slabs;
    uint32_t last = 0;
    if (lane == 0) {
        store_partial(slots + slab, part);
        last = (atomicAdd(p.lev[l].counter + cell, 1u) == p.slabs - 1u);
    }
    last = __shfl_sync(0xffffffffu, last, 0);
    if (!last) return 0u;
    const uint32_t flagged = finalize_cell<true>(p, l, cell, lane, slots);
    __syncwarp();
    // leave the workspace all-zero: partials and counter (header contract)
    for (uint32_t s = lane; s < p.slabs; s += 32) slots[s] = 0.0;
    if (lane == 0) p.lev[l].counter[cell] = 0u;
    if (flagged && p.excise) {
        if (DEFER) return 1u;
        excise_cell<true>(p, b * (p.M << l), p.M << l, f, lane, 32);
    }
    return 0u;
}

// --------------------------------------------------------------------------- fused a1..a7
// Direct-load fallback of the stream kernel (sk_tma.cuh): the same unit decomposition, 128-bit global
// loads, one integration length.  Acc2 = AccChain2 / AccWide2 / AccPlain2 by block length.
// EXC = the launch excises flagged cells in place (p.excise != nullptr): the data is then read with
// plain ld.global instead of ld.global.nc, because another warp of this grid may be overwriting a
// neighbouring cell of the same 32-byte sector while this one loads (E = 16).
template <int L, class Acc2, bool EXC>
__global__ void __launch_bounds__(kWarpsPerCta * 32, kMinCtasPerSm)
sk_frame_kernel(const FrameParams p) {
    constexpr int RPW = 32 / L;
    const int lane = threadIdx.x & 31;
    const uint32_t unit = blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    if (unit >= p.nunits) return;
    const uint32_t slab = unit % p.slabs, cell = unit / p.slabs;
    const uint32_t b = cell / p.F, f = cell % p.F;
    const int cl = lane % L, r0 = lane / L;
    const uint32_t e0 = (slab * L + cl) * 16u;
    const bool active = e0 < p.E;

    uint32_t S1[16], S2[16];
    {
        Acc2 acc[8];
        UnpackConsts kc;
        kc.init();
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k].reset();
        const size_t rstride = (size_t)p.F * p.E;
        const uint8_t* base = p.data + ((size_t)b * p.M * p.F + f) * p.E + e0;
        uint32_t n = 0;
        if (active) {
            // rows r0, r0+RPW, ...: full batches of kUnroll independent 128-bit loads, then a tail
            const uint32_t mine = (p.M > (uint32_t)r0) ? (p.M - r0 + RPW - 1) / RPW : 0u;
            const uint8_t* q = base + (size_t)r0 * rstride;
            const size_t step = (size_t)RPW * rstride;
            uint32_t i = 0;
            for (; i + kUnroll <= mine; i += kUnroll) {
                uint4 v[kUnroll];
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) v[u] = EXC ? ldg_stream_rw(q + (size_t)u * step) : ldg_stream(q + (size_t)u * step);
                q += (size_t)kUnroll * step;
                loads_issued(v);
#pragma unroll
                for (int u = 0; u < kUnroll; ++u) accumulate16(acc, v[u], kc);
            }
            for (; i < mine; ++i) {
                const uint4 v = EXC ? ldg_stream_rw(q) : ldg_stream(q);
                q += step;
                accumulate16(acc, v, kc);
            }
            n = mine;
        }
        read16(acc, n, S1, S2);
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
    if (p.lev[0].SK)
        publish_and_finalize(p, 0, b, f, slab, lane, unit_partial<L>(p, (double)p.M, active, owner, e_first, S1, S2));
}

// ------------------------------------------------------------------ a4..a6 from stored sums
// One CTA per cell; its warps walk the cell's slabs with the same lane mapping as the fused
// kernel, keep the per-slab partials in shared memory, and warp 0 finalizes: bit-identical SK.
template <int L>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
sk_combine_kernel(const FrameParams p) {
    extern __shared__ double partials[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t cell = blockIdx.x;
    const int cl = lane % L;
    for (uint32_t slab = warp; slab < p.slabs; slab += kWarpsPerCta) {
        const uint32_t e0 = (slab * L + cl) * 16u;
        const bool active = e0 < p.E;
        constexpr int RPW = 32 / L;
        constexpr int kOwn = Owned<L>::value;
        const int r0 = lane / L;
        // the same ownership as after the fused kernel's reduce-scatter: bit s of r0 picks the half
        int base = 0;
        {
            int c = 16;
#pragma unroll
            for (int s = 0; (1 << s) < RPW; ++s)
                if (c > 1) { c /= 2; base += ((r0 >> s) & 1) ? c : 0; }
        }
        const bool owner = (RPW <= 16) || (r0 < 16);
        const uint32_t e_first = e0 + base;
        uint32_t S1[16], S2[16];
#pragma unroll
        for (int i = 0; i < kOwn; ++i) {
            S1[i] = (active && owner) ? __ldg(p.S1in + (size_t)cell * p.E + e_first + i) : 0u;
            S2[i] = (active && owner) ? __ldg(p.S2in + (size_t)cell * p.E + e_first + i) : 0u;
        }
        const double part = unit_partial<L>(p, (double)p.M, active, owner, e_first, S1, S2);
        if (lane == 0) partials[slab] = part;
    }
    __syncthreads();
    if (warp == 0) finalize_cell<false>(p, 0, cell, lane, partials);
}

// ------------------------------------------------------------- scalar fallback (any E, alignment)
// One CTA per cell.  Inputs are taken 256 at a time (thread t owns input 256 c + t); a chunk's
// terms are added with the canonical adjacent-first tree in shared memory, chunks are merged by
// thread 0: the same S2bar as the vector kernels, bit for bit.
constexpr int kScalarThreads = 256;

__global__ void __launch_bounds__(kScalarThreads) sk_cell_kernel_scalar(const FrameParams p) {
    __shared__ double red[kScalarThreads];
    __shared__ uint32_t cnt[kScalarThreads];
    const uint32_t cell = blockIdx.x;
    const uint32_t b = cell / p.F, f = cell % p.F;
    const double Md = (double)p.M, MM = __dmul_rn(Md, Md);
    TreeMerge tm;
    uint32_t nsel = 0;
    for (uint32_t c0 = 0; c0 < p.E; c0 += kScalarThreads) {
        const uint32_t e = c0 + threadIdx.x;
        double term = 0.0;
        if (e < p.E) {
            uint32_t s1 = 0, s2 = 0;
            if (p.S1in) {
                s1 = p.S1in[(size_t)cell * p.E + e];
                s2 = p.S2in[(size_t)cell * p.E + e];
            } else {
                const uint8_t* q = p.data + ((size_t)b * p.M * p.F + f) * p.E + e;
                const size_t rstride = (size_t)p.F * p.E;
                for (uint32_t j = 0; j < p.M; ++j) {
                    const uint32_t pw = power_scalar(q[(size_t)j * rstride]);
                    s1 += pw;
                    s2 += pw * pw;
                }
                if (p.S1out) {
                    p.S1out[(size_t)cell * p.E + e] = s1;
                    p.S2out[(size_t)cell * p.E + e] = s2;
                }
            }
            if (p.lev[0].SK && selected(p, e)) {
                term = eq11_term(Md, MM, s1, s2);
                ++nsel;
            }
        }
        if (!p.lev[0].SK) continue;
        red[threadIdx.x] = term;
        __syncthreads();
        for (int o = 1; o < kScalarThreads; o <<= 1) {
            if ((threadIdx.x & (2 * o - 1)) == 0) red[threadIdx.x] = __dadd_rn(red[threadIdx.x], red[threadIdx.x + o]);
            __syncthreads();
        }
        if (threadIdx.x == 0) tm.push(red[0]);
        __syncthreads();
    }
    if (!p.lev[0].SK) return;
    cnt[threadIdx.x] = nsel;
    __syncthreads();
    for (int o = kScalarThreads / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) cnt[threadIdx.x] += cnt[threadIdx.x + o];
        __syncthreads();
    }
    __shared__ uint32_t flagged;
    if (threadIdx.x == 0) {
        const double N = (double)cnt[0];
        const float sk = estimator(p, tm.total(), Md, N);
        p.lev[0].SK[cell] = sk;
        flagged = 0;
        if (p.lev[0].mask) {
            flagged = flag_decision(sk, p.lev[0].sk_mean, flag_threshold(p.n_sigma, Md, N));
            p.lev[0].mask[cell] = (uint8_t)flagged;
        }
    }
    __syncthreads();
    if (flagged && p.excise) excise_cell<false>(p, b * p.M, p.M, f, threadIdx.x, kScalarThreads);
}

// ------------------------------------------------------------------------------------- a7
__global__ void sk_flag_kernel(const float* __restrict__ SK, uint8_t* __restrict__ mask, size_t cells,
                               float sk_mean, float thr) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < cells) mask[i] = flag_decision(SK[i], sk_mean, thr);
}

// ------------------------------------------------------------------ SURVEY 8(f) NEXT-2 / NEXT-4
// Re-binned sums ("a variety of integration lengths"): Eq. 7 over k*M samples is
// the sum of k adjacent M-sample blocks.  in [B][FE] -> out [B/k][FE]; VEC: 4 inputs per thread.
template <bool VEC>
__global__ void __launch_bounds__(256)
sk_rebin_kernel(const uint32_t* __restrict__ A1, const uint32_t* __restrict__ A2, uint32_t* __restrict__ O1,
                uint32_t* __restrict__ O2, size_t FE, uint32_t k) {
    const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * (VEC ? 4 : 1);
    if (i >= FE) return;
    const size_t bo = blockIdx.y;
    const uint32_t* p1 = A1 + bo * k * FE + i;
    const uint32_t* p2 = A2 + bo * k * FE + i;
    if (VEC) {
        uint4 s1 = make_uint4(0, 0, 0, 0), s2 = s1;
        for (uint32_t j = 0; j < k; ++j) {
            const uint4 a = __ldg(reinterpret_cast<const uint4*>(p1 + (size_t)j * FE));
            const uint4 b = __ldg(reinterpret_cast<const uint4*>(p2 + (size_t)j * FE));
            s1.x += a.x; s1.y += a.y; s1.z += a.z; s1.w += a.w;
            s2.x += b.x; s2.y += b.y; s2.z += b.z; s2.w += b.w;
        }
        *reinterpret_cast<uint4*>(O1 + bo * FE + i) = s1;
        *reinterpret_cast<uint4*>(O2 + bo * FE + i) = s2;
    } else {
        uint32_t s1 = 0, s2 = 0;
        for (uint32_t j = 0; j < k; ++j) { s1 += __ldg(p1 + (size_t)j * FE); s2 += __ldg(p2 + (size_t)j * FE); }
        O1[bo * FE + i] = s1;
        O2[bo * FE + i] = s2;
    }
}

// Per-receiver estimate (Eq. 8): SKi = (M+1)/(M-1) * (M S2 / S1^2 - 1) in float64,
// rounded to float32; a zero-power receiver gives 0 (A4).  `a` = (M+1)/(M-1) from the host.
__device__ __forceinline__ float eq8_single(uint32_t u1, uint32_t u2, double M, double a) {
    const double s1 = u32_to_f64(u1), s2 = u32_to_f64(u2);
    const double q = div_f64(__dmul_rn(M, s2), __dmul_rn(s1, s1));
    return u1 == 0u ? 0.0f : __double2float_rn(__dmul_rn(a, __dsub_rn(q, 1.0)));
}

template <bool VEC>
__global__ void __launch_bounds__(256)
sk_single_kernel(const uint32_t* __restrict__ S1, const uint32_t* __restrict__ S2, float* __restrict__ SKi,
                 size_t n, double M, double a) {
    const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * (VEC ? 4 : 1);
    if (i >= n) return;
    if (VEC) {
        const uint4 u1 = __ldg(reinterpret_cast<const uint4*>(S1 + i));
        const uint4 u2 = __ldg(reinterpret_cast<const uint4*>(S2 + i));
        *reinterpret_cast<float4*>(SKi + i) = make_float4(eq8_single(u1.x, u2.x, M, a), eq8_single(u1.y, u2.y, M, a),
                                                          eq8_single(u1.z, u2.z, M, a), eq8_single(u1.w, u2.w, M, a));
    } else {
        SKi[i] = eq8_single(__ldg(S1 + i), __ldg(S2 + i), M, a);
    }
}

// Detection significance: (SK - sk_mean) / sd, sd = sqrt(4/(M N)) from the host.
__global__ void sk_significance_kernel(const float* __restrict__ SK, float* __restrict__ sig, size_t cells,
                                       double sk_mean, double sd) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= cells) return;
    const double d = __dsub_rn((double)SK[i], sk_mean);
    // div_f64 wants a positive divisor and a finite non-negative dividend: divide |d|, restore the sign
    const double q = div_f64(fabs(d), sd);
    sig[i] = (d != d || fabs(d) == __longlong_as_double(0x7ff0000000000000ll))
                 ? __double2float_rn(d) : __double2float_rn(d < 0.0 ? -q : q);
}

// ------------------------------------------------------------------------------------- a8
// Excision as a pass of its own (the fused kernels excise in their finalizer; this one serves
// sk_frame_multi when it has to take one pass per length): every byte of every flagged cell of
// length M becomes 0x88.  grid = (cells, row chunks); a CTA whose cell is clean exits at once.
constexpr int kExciseRows = 32;

template <bool VEC>
__global__ void __launch_bounds__(256)
sk_excise_kernel(const FrameParams p, const uint8_t* __restrict__ mask, uint32_t M) {
    const uint32_t cell = blockIdx.x;
    if (mask[cell] == 0) return;
    const uint32_t b = cell / p.F, f = cell % p.F;
    const uint32_t j0 = blockIdx.y * kExciseRows;
    excise_cell<VEC>(p, b * M + j0, min(M - j0, (uint32_t)kExciseRows), f, threadIdx.x, 256);
}

}  // namespace sk
