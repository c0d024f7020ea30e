// sk_api.cu — the C ABI of include/sk_b200.h: argument checks, shape -> kernel choice, launches.
// Nothing here allocates device memory or synchronises (sk_frame_host waits for its own copies).
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstring>

#include "../../include/sk_b200.h"
#include "sk_kernels.cuh"
#include "sk_tma.cuh"
#include "sk_sim.cuh"

namespace {

std::atomic<unsigned long long> g_launches{0};      // the library's only mutable process-wide state

// The SK_FRAME_PLAN_* bits of a call's `flags` (tests and A/B timing): they override the kernel
// choice for that call only.  Default-constructed = automatic.
struct Force {
    bool ldg = false;        // never the stream kernel
    bool no_tmap = false;    // behave as if the driver had refused to encode the tensor map
    int lanes = 0;           // != 0: a slab width of 16 * lanes inputs
};

Force force_of(int flags) {
    Force fc;
    fc.ldg = (flags & SK_FRAME_PLAN_LDG) != 0;
    fc.no_tmap = (flags & SK_FRAME_PLAN_NO_TMAP) != 0;
    const int l = (flags >> 12) & 31;
    if (l >= 1 && l <= 16 && (l & (l - 1)) == 0) fc.lanes = l;
    return fc;
}

inline int launch_status() {
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SK_OK : (int)e;
}

constexpr int kMaxDevices = 64;

int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
    return dev;
}

int sm_count() {
    static std::atomic<int> cache[kMaxDevices];
    const int dev = current_device();
    int v = cache[dev].load(std::memory_order_relaxed);
    if (v == 0) {
        if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0) v = 148;
        (void)cudaGetLastError();
        cache[dev].store(v, std::memory_order_relaxed);
    }
    return v;
}

// Lanes per row for the vector path (slab width = 16*L inputs).  The sum over inputs follows a
// canonical tree over the input indices (sk_kernels.cuh), so the choice affects speed only, never
// a result: wide 256-byte slabs (fewest units, least per-unit work) when that still gives every
// SM enough warps; otherwise narrower slabs.  A lone frame needs ~16 warps per SM of its own;
// frames that overlap their neighbours on the stream (SK_FRAME_INPUTS_READY) share the SM with
// them and run best on wide slabs from 8 warps per SM up (measured on config 1: 16.3 vs 17.0 us).
inline int lanes_per_row(uint32_t E, unsigned long long units_per_slab_column, bool overlapped, const Force& fc) {
    const uint32_t vecs = E / 16;            // 128-bit vectors per row
    int L = 16;
    while (L > 1 && (uint32_t)L > vecs) L >>= 1;
    const unsigned long long want = (unsigned long long)sm_count() * (overlapped ? 8u : 16u);
    while (L > 4 && units_per_slab_column * ((E + 16u * L - 1) / (16u * L)) < want) L >>= 1;
    const int v = fc.lanes;
    if (v >= 1 && (uint32_t)v <= (vecs < 16u ? vecs : 16u) && (v & (v - 1)) == 0) L = v;
    return L;
}

inline bool vector_ok(const void* data, uint32_t E) {
    return E % 16 == 0 && (reinterpret_cast<uintptr_t>(data) & 15u) == 0;
}

int check_shape(uint32_t T, uint32_t F, uint32_t E, uint32_t M) {
    if (M < 2 || M > 65536) return SK_ERR_M;
    if (T == 0 || F == 0 || E == 0 || T % M != 0) return SK_ERR_SHAPE;
    const unsigned long long total = (unsigned long long)T * F * E;
    if (total >= (1ull << 40)) return SK_ERR_SHAPE;
    if ((unsigned long long)(T / M) * F >= (1ull << 31)) return SK_ERR_SHAPE;
    if (E > (1u << 20)) return SK_ERR_SHAPE;
    return SK_OK;
}

// Rows per accumulator read-out of the stream kernel: the largest divisor of M that is a whole
// number of TMA tiles and keeps a lane within AccChain2's 128 samples (rows <= 128 * RPW).
// 0 = none (ragged or very short blocks): the direct-load kernel runs instead.
uint32_t chunk_rows(uint32_t M, int L) {
    const uint32_t RPW = 32u / L, cap = sk::AccChain2::kMaxSamples * RPW;
    const uint32_t R = sk::kTileBytes / (16u * L);
    if (M % R) return 0;
    for (uint32_t d = (M < cap ? M : cap) / R * R; d >= R; d -= R)
        if (M % d == 0) return d >= cap / 4 || d == M ? d : 0;
    return 0;
}

struct Plan {
    bool vec;
    int L;
    uint32_t slabs;       // launched slabs per cell
    bool wide;            // AccWide2 usable by the direct-load kernel (samples per lane <= 511)
    bool chain;           // AccChain2 usable by the direct-load kernel (samples per lane <= 128)
    uint32_t chunk;       // stream kernel: rows per read-out, 0 = stream kernel not usable
    uint32_t bpu;         // stream kernel: M-row blocks per unit (a power of two dividing B, >= 1 << (nlev-1))
    uint32_t ragged_tpb;  // != 0: the ragged stream kernel runs, with this many tiles per block (chunk == 0)
};

// nlev = integration lengths wanted (M << 0 .. M << (nlev-1)); B % (1 << (nlev-1)) == 0.
Plan make_plan(const void* data, uint32_t E, uint32_t M, uint32_t B, uint32_t F, const uint8_t* subset,
               uint32_t first_n, bool need_all_inputs, bool overlapped, uint32_t nlev, const Force& fc = Force{}) {
    Plan pl{};
    pl.vec = vector_ok(data, E);
    // blocks per unit: the longest length's worth, and for short blocks as many as make a unit
    // of >= 256 rows while every SM still gets its share of units
    uint32_t bpu = 1u << (nlev - 1);
    const unsigned long long want = (unsigned long long)sm_count() * 48u;
    while (M * bpu < 256u && B % (2u * bpu) == 0 &&
           (unsigned long long)(B / (2u * bpu)) * F * ((E + 255u) / 256u) >= want)
        bpu *= 2u;
    pl.bpu = bpu;
    pl.L = lanes_per_row(E, (unsigned long long)(B / bpu) * F, overlapped, fc);
    uint32_t cover = E;
    if (!subset && !need_all_inputs) cover = first_n;    // inputs beyond first_n are never read
    // a few receivers only: one slab no wider than needed (64 bytes at least), so that the rest of the row is not fetched
    while (pl.L > 4 && 8u * pl.L >= cover && fc.lanes == 0) pl.L >>= 1;
    const uint32_t W = 16u * pl.L;
    pl.slabs = (cover + W - 1) / W;
    const uint32_t RPW = 32u / pl.L;
    const uint32_t iters = (M + RPW - 1) / RPW;
    pl.wide = iters <= sk::AccWide2::kMaxSamples;
    pl.chain = iters <= sk::AccChain2::kMaxSamples;
    // the stream kernel's grid is (slabs, F, B / bpu) and its tensor map has a row of F*E bytes.  The
    // coordinates of a TMA box are SIGNED 32-bit: the last box of a row starts below F*E and a ragged
    // one reaches at most 256 bytes past it, so F*E + 256 <= 2^31 keeps every x (and B*M < 2^31 every
    // y) non-negative; a wider frame would have its upper boxes read as negative coordinates and
    // zero-filled.  Such frames take the direct-load kernel.
    const bool grid_ok = B / bpu <= 65535u && F <= 65535u && (unsigned long long)F * E + 256ull <= (1ull << 31) &&
                         (unsigned long long)B * M < (1ull << 31);
    pl.chunk = (pl.vec && grid_ok && pl.L >= 4) ? chunk_rows(M, pl.L) : 0u;
    if (pl.chunk == 0u && pl.vec && grid_ok && fc.lanes == 0) {
        // the block length is not a whole number of tiles at this slab width (a tile is 8 KiB: 32 rows of
        // 256 B, 64 of 128 B, 128 of 64 B): a wider slab has shorter tiles; take the first width that fits
        int widest = 16;                                  // ... but no wider than the receivers asked for justify
        while (widest > 4 && 8u * widest >= cover) widest >>= 1;
        for (int L2 = widest; L2 >= 4; L2 >>= 1) {
            if ((uint32_t)L2 > E / 16 || L2 == pl.L || chunk_rows(M, L2) == 0u) continue;
            pl.L = L2;
            pl.slabs = (cover + 16u * L2 - 1) / (16u * L2);
            const uint32_t it2 = (M + 32u / L2 - 1) / (32u / L2);
            pl.wide = it2 <= sk::AccWide2::kMaxSamples;
            pl.chain = it2 <= sk::AccChain2::kMaxSamples;
            pl.chunk = chunk_rows(M, L2);
            break;
        }
    }
    if (pl.chunk == 0u && pl.vec && grid_ok && nlev == 1) {
        // no slab width makes the block a whole number of tiles: the ragged stream kernel, at the widest
        // slab (shortest tiles), as long as the block is at least two tiles long
        int L2 = fc.lanes ? pl.L : 16;
        while (L2 > 1 && (uint32_t)L2 > E / 16) L2 >>= 1;
        while (L2 > 4 && 8u * L2 >= cover && fc.lanes == 0) L2 >>= 1;
        const uint32_t R = sk::kTileBytes / (16u * (uint32_t)L2);
        const uint32_t it2 = (M + 32u / L2 - 1) / (32u / L2);            // samples a lane adds per block
        // worth it for long blocks only: up to 128 samples per lane the direct-load kernel keeps the packed
        // accumulators and is as fast (measured: M = 100, 250: 4.2-4.7 TB/s either way; M = 1000: 5.0 against 3.7)
        if (L2 >= 4 && M >= 2u * R && it2 > sk::AccChain2::kMaxSamples) {
            pl.L = L2;
            pl.slabs = (cover + 16u * L2 - 1) / (16u * L2);
            pl.wide = it2 <= sk::AccWide2::kMaxSamples;
            pl.chain = false;
            pl.ragged_tpb = (M + R - 1) / R;
        }
    }
    return pl;
}

template <class Acc2, bool EXC>
void launch_vec_LX(int L, const sk::FrameParams& p, cudaStream_t st) {
    const unsigned grid = (p.nunits + sk::kWarpsPerCta - 1) / sk::kWarpsPerCta;
    const unsigned block = sk::kWarpsPerCta * 32;
    switch (L) {
        case 16: sk::sk_frame_kernel<16, Acc2, EXC><<<grid, block, 0, st>>>(p); break;
        case 8:  sk::sk_frame_kernel<8, Acc2, EXC><<<grid, block, 0, st>>>(p); break;
        case 4:  sk::sk_frame_kernel<4, Acc2, EXC><<<grid, block, 0, st>>>(p); break;
        case 2:  sk::sk_frame_kernel<2, Acc2, EXC><<<grid, block, 0, st>>>(p); break;
        default: sk::sk_frame_kernel<1, Acc2, EXC><<<grid, block, 0, st>>>(p); break;
    }
    ++g_launches;
}

// A launch that excises in place reads `data` without .nc (see sk_frame_kernel).
template <class Acc2>
void launch_vec_L(int L, const sk::FrameParams& p, cudaStream_t st) {
    if (p.excise) launch_vec_LX<Acc2, true>(L, p, st);
    else          launch_vec_LX<Acc2, false>(L, p, st);
}

// ---- TMA path ---------------------------------------------------------------------------
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled() {
    // resolved through the runtime, so the library has no link-time dependency on libcuda.so
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            f = nullptr;
        (void)cudaGetLastError();
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}

// The stream kernel runs whenever it applies; SK_FRAME_PLAN_LDG turns it off for the call.
bool stream_wanted(const Plan& pl, const Force& fc) {
    if (fc.ldg) return false;
    return (pl.chunk != 0 || pl.ragged_tpb != 0) && encode_tiled() != nullptr;
}

template <int L, int NLEV, bool CHUNKED>
int launch_stream_K(const CUtensorMap& tmap, const sk::FrameParams& p, uint32_t zblocks, cudaStream_t st) {
    // per device: the opt-in attributes belong to the device's copy of the function
    static std::atomic<bool> attr_set[kMaxDevices];
    const int dev = current_device();
    if (!attr_set[dev].load(std::memory_order_acquire)) {
        cudaFuncSetAttribute(sk::sk_stream_kernel<L, NLEV, CHUNKED>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sk::kStreamSmemBytes);
        cudaFuncSetAttribute(sk::sk_stream_kernel<L, NLEV, CHUNKED>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
        attr_set[dev].store(true, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.slabs, p.F, zblocks);
    cfg.blockDim = dim3(32);
    cfg.dynamicSmemBytes = sk::kStreamSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, sk::sk_stream_kernel<L, NLEV, CHUNKED>, tmap, p);
    return e == cudaSuccess ? SK_OK : (int)e;
}

template <int L>
int launch_ragged_L(const CUtensorMap& tmap, const sk::FrameParams& p, uint32_t zblocks, cudaStream_t st) {
    static std::atomic<bool> attr_set[kMaxDevices];
    const int dev = current_device();
    if (!attr_set[dev].load(std::memory_order_acquire)) {
        cudaFuncSetAttribute(sk::sk_stream_ragged_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sk::kStreamSmemBytes);
        cudaFuncSetAttribute(sk::sk_stream_ragged_kernel<L>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
        attr_set[dev].store(true, std::memory_order_release);
    }
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.slabs, p.F, zblocks);
    cfg.blockDim = dim3(32);
    cfg.dynamicSmemBytes = sk::kStreamSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, sk::sk_stream_ragged_kernel<L>, tmap, p);
    return e == cudaSuccess ? SK_OK : (int)e;
}

template <int L>
int launch_stream_L(const CUtensorMap& tmap, const sk::FrameParams& p, bool chunked, uint32_t zblocks,
                    cudaStream_t st) {
    switch (p.nlev) {
        case 1: return chunked ? launch_stream_K<L, 1, true>(tmap, p, zblocks, st)
                               : launch_stream_K<L, 1, false>(tmap, p, zblocks, st);
        case 2: return launch_stream_K<L, 2, true>(tmap, p, zblocks, st);
        case 3: return launch_stream_K<L, 3, true>(tmap, p, zblocks, st);
        default: return launch_stream_K<L, 4, true>(tmap, p, zblocks, st);
    }
}

// launch_stream could not build the tensor map for this pointer / shape (nothing was launched): the
// callers fall back to the direct-load kernels, whose results are identical.  Never returned to a user.
constexpr int kEncodeFailed = -1000;

int launch_stream(const Plan& pl, const sk::FrameParams& p, cudaStream_t st, const Force& fc) {
    CUtensorMap tmap;
    const uint32_t W = 16u * pl.L;
    const cuuint64_t gdim[2] = {(cuuint64_t)p.F * p.E, (cuuint64_t)p.T};
    const cuuint64_t gstride[1] = {(cuuint64_t)p.F * p.E};
    const cuuint32_t box[2] = {(cuuint32_t)W, (cuuint32_t)(sk::kTileBytes / W)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode_tiled()(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t*>(p.data), gdim,
                                      gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS || fc.no_tmap) return kEncodeFailed;
    const bool chunked = pl.chunk != p.M;
    const uint32_t zblocks = p.B / pl.bpu;
    int rc;
    if (pl.ragged_tpb) {
        switch (pl.L) {
            case 16: rc = launch_ragged_L<16>(tmap, p, zblocks, st); break;
            case 8:  rc = launch_ragged_L<8>(tmap, p, zblocks, st); break;
            default: rc = launch_ragged_L<4>(tmap, p, zblocks, st); break;
        }
        if (rc == SK_OK) ++g_launches;
        return rc;
    }
    switch (pl.L) {
        case 16: rc = launch_stream_L<16>(tmap, p, chunked, zblocks, st); break;
        case 8:  rc = launch_stream_L<8>(tmap, p, chunked, zblocks, st); break;
        default: rc = launch_stream_L<4>(tmap, p, chunked, zblocks, st); break;
    }
    if (rc == SK_OK) ++g_launches;
    return rc;
}

int launch_cells(const Plan& pl, sk::FrameParams& p, cudaStream_t st, const Force& fc = Force{}) {
    const uint32_t cells = p.B * p.F;
    if (pl.vec) {
        p.slabs = pl.slabs;
        p.nunits = cells * pl.slabs;
        int rc = kEncodeFailed;                                    // "no stream kernel": also when it is not wanted
        if (stream_wanted(pl, fc)) {
            p.chunk = pl.chunk;
            p.bpu = pl.bpu;
            p.tpb = pl.ragged_tpb;
            p.unit_tiles = pl.ragged_tpb ? pl.ragged_tpb * pl.bpu : p.M * pl.bpu / (sk::kTileBytes / (16u * pl.L));
            rc = launch_stream(pl, p, st, fc);
            if (rc != SK_OK && rc != kEncodeFailed) return rc;
            if (rc == kEncodeFailed && p.nlev > 1) return rc;      // frame_impl takes one pass per length instead
        }
        if (rc == kEncodeFailed) {
            // the direct-load kernel at this slab width: one cell per unit, accumulators by block length
            const uint32_t iters = (p.M + 32u / pl.L - 1) / (32u / pl.L);
            if (iters <= sk::AccChain2::kMaxSamples)     launch_vec_L<sk::AccChain2>(pl.L, p, st);
            else if (iters <= sk::AccWide2::kMaxSamples) launch_vec_L<sk::AccWide2>(pl.L, p, st);
            else                                         launch_vec_L<sk::AccPlain2>(pl.L, p, st);
        }
    } else {
        sk::sk_cell_kernel_scalar<<<cells, sk::kScalarThreads, 0, st>>>(p);
        ++g_launches;
    }
    return launch_status();
}

size_t level_bytes(uint32_t cells, uint32_t slabs_max) {
    return (size_t)cells * slabs_max * sizeof(double) + (((size_t)cells * sizeof(uint32_t) + 7u) & ~(size_t)7u);
}

// Workspace of integration length l: partials [cells_l][slabs_max] then counters [cells_l]; the
// lengths follow one another.  The place of every array depends on the shape alone (not on
// first_n or on the slab width), so a workspace stays clean across calls.
size_t workspace_bytes(uint32_t B, uint32_t F, uint32_t E, uint32_t nlev) {
    size_t n = 0;
    for (uint32_t l = 0; l < nlev; ++l) n += level_bytes((B >> l) * F, (E + 15u) / 16u);
    return n;
}

int check_frame_args(const uint8_t* subset, uint32_t E, uint32_t first_n, float n_sigma, const float* sk_means,
                     uint32_t nlev, bool with_mask) {
    if (!subset && (first_n == 0 || first_n > E)) return SK_ERR_N;
    if (with_mask) {
        if (!std::isfinite(n_sigma) || n_sigma < 0) return SK_ERR_PARAM;
        for (uint32_t l = 0; l < nlev; ++l)
            if (!std::isfinite(sk_means[l])) return SK_ERR_PARAM;
    }
    return SK_OK;
}

// The fused path for nlev integration lengths (sk_frame: nlev = 1).  All argument checks happen
// before the first launch.
int frame_impl(const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t nlev,
               const uint8_t* subset, uint32_t first_n, float n_sigma, const float* sk_means, int flags,
               float* const* SK, uint8_t* const* mask, uint32_t* S1o, uint32_t* S2o, void* workspace,
               size_t workspace_bytes_given, cudaStream_t st) {
    if (int rc = check_shape(T, F, E, M)) return rc;
    const uint32_t B = T / M;
    if (nlev < 1 || nlev > (uint32_t)sk::kMaxLevels) return SK_ERR_SHAPE;
    if (B % (1u << (nlev - 1)) != 0) return SK_ERR_SHAPE;
    if (((unsigned long long)M << (nlev - 1)) > 65536ull) return SK_ERR_M;
    bool any_mask = false;
    for (uint32_t l = 0; l < nlev; ++l) {
        if (!SK[l]) return SK_ERR_NULL;
        any_mask = any_mask || mask[l] != nullptr;
    }
    if ((flags & SK_FRAME_ZERO_FLAGGED) && !mask[0]) return SK_ERR_NULL;
    if (int rc = check_frame_args(subset, E, first_n, n_sigma, sk_means, nlev, any_mask)) return rc;
    if ((S1o == nullptr) != (S2o == nullptr)) return SK_ERR_NULL;
    const Force fc = force_of(flags);
    Plan pl = make_plan(data, E, M, B, F, subset, first_n, S1o != nullptr, (flags & SK_FRAME_INPUTS_READY) != 0, nlev, fc);
    if (S1o && ((reinterpret_cast<uintptr_t>(S1o) | reinterpret_cast<uintptr_t>(S2o)) & 15u)) pl.vec = false;
    sk::FrameParams p{};
    p.data = data; p.T = T; p.F = F; p.E = E; p.M = M; p.B = B;
    p.excise = (flags & SK_FRAME_ZERO_FLAGGED) ? const_cast<uint8_t*>(data) : nullptr;
    p.subset = subset; p.first_n = subset ? 0 : first_n;
    p.n_sigma = n_sigma;
    p.nlev = nlev;
    p.eq13 = (flags & SK_FRAME_EQ13) ? 1u : 0u;
    p.inputs_ready = (flags & SK_FRAME_INPUTS_READY) ? 1u : 0u;
    p.S1out = S1o; p.S2out = S2o;
    const bool one_launch = nlev == 1 || (pl.vec && stream_wanted(pl, fc));
    if (pl.vec) {
        if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7u) ||
            workspace_bytes_given < workspace_bytes(B, F, E, nlev))
            return SK_ERR_WORKSPACE;
    }
    const uint32_t slabs_max = (E + 15u) / 16u;
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    for (uint32_t l = 0; l < nlev; ++l) {
        const uint32_t cells = (B >> l) * F;
        p.lev[l].SK = SK[l];
        p.lev[l].mask = mask[l];
        p.lev[l].sk_mean = sk_means[l];
        if (pl.vec) {
            p.lev[l].partial = reinterpret_cast<double*>(ws);
            p.lev[l].counter = reinterpret_cast<uint32_t*>(ws + (size_t)cells * slabs_max * sizeof(double));
            ws += level_bytes(cells, slabs_max);
        }
    }
    if (one_launch) {
        const int rc = launch_cells(pl, p, st, fc);
        if (rc != kEncodeFailed) return rc;                        // only with nlev > 1: no tensor map, take the passes below
    }
    // several lengths without the stream kernel: one pass of the fused path per length, then the
    // excision of every flagged cell of every length (all lengths see the data before excision)
    for (uint32_t l = 0; l < nlev; ++l) {
        sk::FrameParams pl_l = p;
        pl_l.M = M << l; pl_l.B = B >> l; pl_l.nlev = 1; pl_l.excise = nullptr;
        pl_l.lev[0] = p.lev[l];
        pl_l.S1out = l == 0 ? S1o : nullptr; pl_l.S2out = l == 0 ? S2o : nullptr;
        pl_l.inputs_ready = l == 0 ? p.inputs_ready : 0u;
        Plan q = make_plan(data, E, M << l, B >> l, F, subset, first_n, pl_l.S1out != nullptr, false, 1, fc);
        q.vec = pl.vec;
        if (int rc = launch_cells(q, pl_l, st, fc)) return rc;
    }
    for (uint32_t l = 0; l < nlev && p.excise; ++l) {
        if (!mask[l]) continue;
        const uint32_t Ml = M << l;
        const dim3 grid((B >> l) * F, (Ml + sk::kExciseRows - 1) / sk::kExciseRows);
        if (pl.vec) sk::sk_excise_kernel<true><<<grid, 256, 0, st>>>(p, mask[l], Ml);
        else        sk::sk_excise_kernel<false><<<grid, 256, 0, st>>>(p, mask[l], Ml);
        ++g_launches;
        if (int rc = launch_status()) return rc;
    }
    return SK_OK;
}

}  // namespace

// ---- sk_frame_noalloc: the fused path for callers that cannot allocate ---------------------------
// The scratch sk_frame otherwise takes from the caller (per-slab partial sums and per-cell arrival
// counters) lives in this array instead.  It is part of the library's device image: every GPU on
// which the library's kernels are loaded holds these SK_NOALLOC_SCRATCH_BYTES until the process exits.
// In host code the name below is only a handle for the runtime, NOT a device address; the address is
// asked for once per device (noalloc_scratch) and that pointer is what the kernels get.
static __device__ __align__(256) unsigned char sk_noalloc_scratch[SK_NOALLOC_SCRATCH_BYTES];

namespace {

// Device address of sk_noalloc_scratch on the CURRENT device, looked up on the first call made with
// that device current and remembered afterwards (threads racing on the first call look up the same
// address twice, nothing worse).  Returns a cudaError_t (> 0) if the runtime cannot resolve the symbol.
int noalloc_scratch(void** out) {
    static std::atomic<void*> cache[kMaxDevices];
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    const bool cached = dev >= 0 && dev < kMaxDevices;
    void* ptr = cached ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (!ptr) {
        e = cudaGetSymbolAddress(&ptr, sk_noalloc_scratch);
        if (e != cudaSuccess) return (int)e;
        if (!ptr) return (int)cudaErrorInvalidSymbol;
        if (cached) cache[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return SK_OK;
}

}  // namespace

extern "C" {

int sk_power_sums(const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                  uint32_t* S1, uint32_t* S2, void* stream) {
    if (!data || !S1 || !S2) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    Plan pl = make_plan(data, E, M, T / M, F, nullptr, E, true, false, 1);
    if ((reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2)) & 15u) pl.vec = false;
    sk::FrameParams p{};
    p.data = data; p.T = T; p.F = F; p.E = E; p.M = M; p.B = T / M;
    p.first_n = E;
    p.nlev = 1;
    p.S1out = S1; p.S2out = S2;
    return launch_cells(pl, p, (cudaStream_t)stream);
}

size_t sk_frame_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M) {
    if (check_shape(T, F, E, M)) return 0;
    return workspace_bytes(T / M, F, E, 1);
}

size_t sk_frame_multi_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t nlev) {
    if (check_shape(T, F, E, M) || nlev < 1 || nlev > (uint32_t)sk::kMaxLevels) return 0;
    return workspace_bytes(T / M, F, E, nlev);
}

int sk_combine(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E, uint32_t M,
               const uint8_t* subset, uint32_t first_n, float* SK, void* stream) {
    if (!S1 || !S2 || !SK) return SK_ERR_NULL;
    if (B == 0 || (unsigned long long)B * M > 0xFFFFFFFFull) return SK_ERR_SHAPE;
    if (int rc = check_shape(B * M, F, E, M)) return rc;
    if (!subset && (first_n == 0 || first_n > E)) return SK_ERR_N;
    cudaStream_t st = (cudaStream_t)stream;
    sk::FrameParams p{};
    p.T = B * M; p.F = F; p.E = E; p.M = M; p.B = B;
    p.subset = subset; p.first_n = subset ? 0 : first_n;
    p.nlev = 1;
    p.lev[0].SK = SK; p.S1in = S1; p.S2in = S2;
    const uint32_t cells = B * F;
    const bool vec = E % 16 == 0 &&
                     ((reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2)) & 15u) == 0;
    if (vec) {
        // one CTA per cell keeps the cell's per-slab partials in shared memory: widest slabs
        int L = 16;
        while (L > 1 && (uint32_t)L > E / 16) L >>= 1;
        p.slabs = (E + 16u * L - 1) / (16u * L);
        p.nunits = cells * p.slabs;
        const size_t smem = (size_t)p.slabs * sizeof(double);      // E <= 2^20: at most 32 KiB
        const unsigned block = sk::kWarpsPerCta * 32;
        switch (L) {
            case 16: sk::sk_combine_kernel<16><<<cells, block, smem, st>>>(p); break;
            case 8:  sk::sk_combine_kernel<8><<<cells, block, smem, st>>>(p); break;
            case 4:  sk::sk_combine_kernel<4><<<cells, block, smem, st>>>(p); break;
            case 2:  sk::sk_combine_kernel<2><<<cells, block, smem, st>>>(p); break;
            default: sk::sk_combine_kernel<1><<<cells, block, smem, st>>>(p); break;
        }
    } else {
        sk::sk_cell_kernel_scalar<<<cells, sk::kScalarThreads, 0, st>>>(p);
    }
    ++g_launches;
    return launch_status();
}

int sk_flag(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N, float n_sigma,
            float sk_mean, uint8_t* mask, void* stream) {
    if (!SK || !mask) return SK_ERR_NULL;
    if (M < 2 || M > 65536) return SK_ERR_M;
    if (B == 0 || F == 0 || (unsigned long long)B * F >= (1ull << 31)) return SK_ERR_SHAPE;
    if (N == 0) return SK_ERR_N;
    if (!std::isfinite(n_sigma) || !std::isfinite(sk_mean) || n_sigma < 0) return SK_ERR_PARAM;
    const size_t cells = (size_t)B * F;
    const float thr = sk::flag_threshold(n_sigma, (double)M, (double)N);
    sk::sk_flag_kernel<<<(unsigned)((cells + 255) / 256), 256, 0, (cudaStream_t)stream>>>(SK, mask, cells,
                                                                                         sk_mean, thr);
    ++g_launches;
    return launch_status();
}

int sk_frame(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, const uint8_t* subset,
             uint32_t first_n, float n_sigma, float sk_mean, int flags, float* SK, uint8_t* mask,
             uint32_t* S1_opt, uint32_t* S2_opt, void* workspace, size_t workspace_bytes_given,
             void* stream) {
    if (!data || !SK || !mask) return SK_ERR_NULL;
    return frame_impl(data, T, F, E, M, 1, subset, first_n, n_sigma, &sk_mean, flags, &SK, &mask, S1_opt,
                      S2_opt, workspace, workspace_bytes_given, (cudaStream_t)stream);
}

int sk_frame_noalloc(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, const uint8_t* subset,
                     uint32_t first_n, float n_sigma, float sk_mean, int flags, float* SK, uint8_t* mask,
                     uint32_t* S1_opt, uint32_t* S2_opt, void* stream) {
    if (!data || !SK || !mask) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    // the size test comes before anything touches the device: a frame that does not fit is an
    // argument error like any other
    const size_t need = workspace_bytes(T / M, F, E, 1);
    if (need > (size_t)SK_NOALLOC_SCRATCH_BYTES) return SK_ERR_SCRATCH;
    // every other argument error too, so that "< 0 means nothing was enqueued" holds for the clear below
    if (int rc = check_frame_args(subset, E, first_n, n_sigma, &sk_mean, 1, true)) return rc;
    if ((S1_opt == nullptr) != (S2_opt == nullptr)) return SK_ERR_NULL;
    void* scratch = nullptr;
    if (int rc = noalloc_scratch(&scratch)) return rc;
    // The array keeps whatever the last call left in it.  A completed call leaves zeros, one that
    // failed half-way may not have, and the kernels count arrivals up from zero: clear the part this
    // shape uses, in stream order, before the kernel.
    const cudaError_t e = cudaMemsetAsync(scratch, 0, need, (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    return frame_impl(data, T, F, E, M, 1, subset, first_n, n_sigma, &sk_mean, flags, &SK, &mask, S1_opt, S2_opt,
                      scratch, (size_t)SK_NOALLOC_SCRATCH_BYTES, (cudaStream_t)stream);
}

int sk_frame_multi(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t nlev,
                   const uint8_t* subset, uint32_t first_n, float n_sigma, const float* h_sk_means, int flags,
                   float* const* h_SK, uint8_t* const* h_mask, void* workspace, size_t workspace_bytes_given,
                   void* stream) {
    if (!data || !h_sk_means || !h_SK || !h_mask) return SK_ERR_NULL;
    if (nlev < 1 || nlev > (uint32_t)sk::kMaxLevels) return SK_ERR_SHAPE;
    for (uint32_t l = 0; l < nlev; ++l)
        if (!h_SK[l] || !h_mask[l]) return SK_ERR_NULL;
    return frame_impl(data, T, F, E, M, nlev, subset, first_n, n_sigma, h_sk_means, flags, h_SK, h_mask, nullptr,
                      nullptr, workspace, workspace_bytes_given, (cudaStream_t)stream);
}

int sk_frame_host(uint8_t* h_data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, const uint8_t* subset,
                  uint32_t first_n, float n_sigma, float sk_mean, int flags, float* h_SK,
                  uint8_t* h_mask, uint8_t* d_data, float* d_SK, uint8_t* d_mask, void* workspace,
                  size_t workspace_bytes_given, void* stream) {
    if (!h_data || !h_SK || !h_mask || !d_data || !d_SK || !d_mask) return SK_ERR_NULL;
    // every argument error is reported before the upload is enqueued
    if (int rc = check_shape(T, F, E, M)) return rc;
    if (int rc = check_frame_args(subset, E, first_n, n_sigma, &sk_mean, 1, true)) return rc;
    if (vector_ok(d_data, E) && (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7u) ||
                                 workspace_bytes_given < workspace_bytes(T / M, F, E, 1)))
        return SK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)T * F * E, cells = (size_t)(T / M) * F;
    cudaError_t e = cudaMemcpyAsync(d_data, h_data, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return (int)e;
    const int keep = flags & ~SK_FRAME_INPUTS_READY;
    int rc = sk_frame(d_data, T, F, E, M, subset, first_n, n_sigma, sk_mean, keep, d_SK, d_mask, nullptr,
                      nullptr, workspace, workspace_bytes_given, stream);
    if (rc == SK_OK) {
        e = cudaMemcpyAsync(h_SK, d_SK, cells * sizeof(float), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h_mask, d_mask, cells, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && (flags & SK_FRAME_ZERO_FLAGGED))
            e = cudaMemcpyAsync(h_data, d_data, bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) rc = (int)e;
    }
    // the upload has been enqueued: wait for whatever was, also on an error
    e = cudaStreamSynchronize(st);
    if (rc == SK_OK && e != cudaSuccess) rc = (int)e;
    return rc;
}

int sk_frames_host(uint8_t* const* h_frames, uint32_t nframes, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                   const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean, int flags, float* h_SK,
                   uint8_t* h_mask, uint8_t* d_data, float* d_SK, uint8_t* d_mask, void* workspace,
                   size_t workspace_bytes_given, void* stream) {
    if (!h_frames || !h_SK || !h_mask || !d_data || !d_SK || !d_mask) return SK_ERR_NULL;
    if (nframes == 0) return SK_ERR_SHAPE;
    for (uint32_t i = 0; i < nframes; ++i)
        if (!h_frames[i]) return SK_ERR_NULL;
    // every argument error is reported before the first upload is enqueued
    if (int rc = check_shape(T, F, E, M)) return rc;
    if (int rc = check_frame_args(subset, E, first_n, n_sigma, &sk_mean, 1, true)) return rc;
    if (vector_ok(d_data, E) && (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7u) ||
                                 workspace_bytes_given < workspace_bytes(T / M, F, E, 1)))
        return SK_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)T * F * E, cells = (size_t)(T / M) * F;
    const int keep = flags & ~SK_FRAME_INPUTS_READY;
    int rc = SK_OK;
    // upload i, kernel i, read-back i, upload i+1, ...: stream order keeps the one staging frame and the one
    // set of device outputs safe, and the host is not in the loop, so the link never waits for it
    for (uint32_t i = 0; i < nframes && rc == SK_OK; ++i) {
        cudaError_t e = cudaMemcpyAsync(d_data, h_frames[i], bytes, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) { rc = (int)e; break; }
        rc = sk_frame(d_data, T, F, E, M, subset, first_n, n_sigma, sk_mean, keep, d_SK, d_mask, nullptr, nullptr,
                      workspace, workspace_bytes_given, stream);
        if (rc != SK_OK) break;
        e = cudaMemcpyAsync(h_SK + (size_t)i * cells, d_SK, cells * sizeof(float), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(h_mask + (size_t)i * cells, d_mask, cells, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && (flags & SK_FRAME_ZERO_FLAGGED))
            e = cudaMemcpyAsync(h_frames[i], d_data, bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) rc = (int)e;
    }
    const cudaError_t e = cudaStreamSynchronize(st);       // wait for whatever was enqueued, also after an error
    if (rc == SK_OK && e != cudaSuccess) rc = (int)e;
    return rc;
}

int sk_rebin_sums(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E, uint32_t M,
                  uint32_t factor, uint32_t* S1out, uint32_t* S2out, void* stream) {
    if (!S1 || !S2 || !S1out || !S2out) return SK_ERR_NULL;
    if (M < 2 || factor == 0 || (unsigned long long)M * factor > 65536ull) return SK_ERR_M;
    if (B == 0 || F == 0 || E == 0 || B % factor != 0 || B / factor > 65535u) return SK_ERR_SHAPE;
    const size_t FE = (size_t)F * E;
    const uintptr_t al = reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2) |
                         reinterpret_cast<uintptr_t>(S1out) | reinterpret_cast<uintptr_t>(S2out);
    const bool vec = FE % 4 == 0 && (al & 15u) == 0;
    const size_t per = vec ? FE / 4 : FE;
    if ((per + 255) / 256 > 0x7fffffffull) return SK_ERR_SHAPE;
    const dim3 grid((unsigned)((per + 255) / 256), B / factor);
    cudaStream_t st = (cudaStream_t)stream;
    if (vec) sk::sk_rebin_kernel<true><<<grid, 256, 0, st>>>(S1, S2, S1out, S2out, FE, factor);
    else     sk::sk_rebin_kernel<false><<<grid, 256, 0, st>>>(S1, S2, S1out, S2out, FE, factor);
    ++g_launches;
    return launch_status();
}

int sk_single(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E, uint32_t M,
              float* SKi, void* stream) {
    if (!S1 || !S2 || !SKi) return SK_ERR_NULL;
    if (M < 2 || M > 65536) return SK_ERR_M;
    if (B == 0 || F == 0 || E == 0) return SK_ERR_SHAPE;
    const size_t n = (size_t)B * F * E;
    const uintptr_t al = reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2) |
                         reinterpret_cast<uintptr_t>(SKi);
    const bool vec = n % 4 == 0 && (al & 15u) == 0;
    const size_t per = vec ? n / 4 : n;
    if ((per + 255) / 256 > 0x7fffffffull) return SK_ERR_SHAPE;
    const double Md = (double)M, a = (Md + 1.0) / (Md - 1.0);
    const unsigned grid = (unsigned)((per + 255) / 256);
    if (vec) sk::sk_single_kernel<true><<<grid, 256, 0, (cudaStream_t)stream>>>(S1, S2, SKi, n, Md, a);
    else     sk::sk_single_kernel<false><<<grid, 256, 0, (cudaStream_t)stream>>>(S1, S2, SKi, n, Md, a);
    ++g_launches;
    return launch_status();
}

int sk_significance(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N, float sk_mean, float* sig,
                    void* stream) {
    if (!SK || !sig) return SK_ERR_NULL;
    if (M < 2 || M > 65536) return SK_ERR_M;
    if (B == 0 || F == 0 || (unsigned long long)B * F >= (1ull << 31)) return SK_ERR_SHAPE;
    if (N == 0) return SK_ERR_N;
    if (!std::isfinite(sk_mean)) return SK_ERR_PARAM;
    const size_t cells = (size_t)B * F;
    const double sd = std::sqrt(4.0 / ((double)M * (double)N));
    sk::sk_significance_kernel<<<(unsigned)((cells + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        SK, sig, cells, (double)sk_mean, sd);
    ++g_launches;
    return launch_status();
}

int sk_sim_digitised(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, const uint32_t* thr, uint64_t seed,
                     uint64_t frame, void* stream) {
    if (!data || !thr) return SK_ERR_NULL;
    if (T == 0 || F == 0 || E == 0 || (unsigned long long)T * F > 0xFFFFFFFFull) return SK_ERR_SHAPE;
    const unsigned long long rows = (unsigned long long)T * F;
    unsigned long long rpt = (rows + 65534ull) / 65535ull;          // rows per thread: grid.y <= 65535
    if (rpt < (unsigned long long)sk::kSimRows) rpt = sk::kSimRows;
    const uint32_t pairs = (E + 1) / 2;
    const dim3 grid((pairs + sk::kSimThreads - 1) / sk::kSimThreads, (unsigned)((rows + rpt - 1) / rpt));
    sk::sk_sim_kernel<<<grid, sk::kSimThreads, 0, (cudaStream_t)stream>>>(
        data, rows, (uint32_t)rpt, E, thr, (uint32_t)seed, (uint32_t)(seed >> 32), (uint32_t)frame,
        (uint32_t)(frame >> 32));
    ++g_launches;
    return launch_status();
}

int sk_sim_common_mode(uint32_t D, uint32_t M, uint32_t N, double amp, uint64_t seed, float* SK, void* stream) {
    if (!SK) return SK_ERR_NULL;
    if (M < 2 || M > 2048) return SK_ERR_M;             // the common-mode samples live in shared memory
    if (D == 0 || D > 0x7fffffffu) return SK_ERR_SHAPE;
    if (N == 0) return SK_ERR_N;
    if (!std::isfinite(amp)) return SK_ERR_PARAM;
    sk::sk_sim_common_mode_kernel<<<D, sk::kCmThreads, (size_t)M * sizeof(double2), (cudaStream_t)stream>>>(
        M, N, amp, (uint32_t)seed, (uint32_t)(seed >> 32), SK);
    ++g_launches;
    return launch_status();
}

int sk_moments(const float* SK, uint32_t B, uint32_t F, double* mean, double* var, void* stream) {
    if (!SK || !mean || !var) return SK_ERR_NULL;
    if (B == 0 || F == 0) return SK_ERR_SHAPE;
    sk::sk_moments_kernel<<<F, sk::kMomThreads, 0, (cudaStream_t)stream>>>(SK, B, F, mean, var);
    ++g_launches;
    return launch_status();
}

const char* sk_strerror(int code) {
    switch (code) {
        case SK_OK: return "ok";
        case SK_ERR_NULL: return "a required pointer is NULL";
        case SK_ERR_SHAPE: return "bad shape: T, F, E must be >= 1, T % M == 0, T*F*E < 2^40";
        case SK_ERR_M: return "M must be in [2, 65536]";
        case SK_ERR_N: return "receiver count N must be in [1, E]";
        case SK_ERR_PARAM: return "n_sigma and sk_mean must be finite, n_sigma >= 0";
        case SK_ERR_WORKSPACE: return "workspace is NULL, misaligned or smaller than sk_frame_workspace_bytes()";
        case SK_ERR_SCRATCH: return "sk_frame_noalloc: this shape needs more scratch than the built-in SK_NOALLOC_SCRATCH_BYTES";
        default: return code > 0 ? cudaGetErrorString((cudaError_t)code) : "unknown error";
    }
}

int sk_version(void) { return 200; }

unsigned long long sk_launch_count(void) { return g_launches.load(); }

int sk_frame_plan(uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t first_n, int flags, uint32_t nlev,
                  uint32_t* plan4) {
    if (!plan4) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    if (nlev < 1 || nlev > (uint32_t)sk::kMaxLevels || (T / M) % (1u << (nlev - 1)) != 0) return SK_ERR_SHAPE;
    if (first_n == 0 || first_n > E) return SK_ERR_N;
    // an aligned data pointer is assumed (the vector path)
    const Force fc = force_of(flags);
    const Plan pl = make_plan(nullptr, E, M, T / M, F, nullptr, first_n, false, (flags & SK_FRAME_INPUTS_READY) != 0, nlev, fc);
    plan4[0] = (uint32_t)pl.L;
    plan4[1] = pl.slabs;
    plan4[2] = (pl.vec && stream_wanted(pl, fc)) ? (pl.ragged_tpb ? sk::kRaggedTilesPerReadout * sk::kTileBytes / (16u * pl.L) : pl.chunk) : 0u;
    plan4[3] = pl.bpu;
    return SK_OK;
}

}  // extern "C"
