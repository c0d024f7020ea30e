// sk_bench.cu — libsk_b200_bench.so: measurement kernels only (see sk_bench.h).  Built from the
// product's own headers, so the loop body, the ring and the epilogue measured here are the product's.
#include <atomic>
#include <chrono>
#include <cstdint>

#include "../../../include/sk_b200.h"
#include "sk_bench.h"
#include "sk_ceiling.cuh"

namespace {

std::atomic<unsigned long long> g_launches{0};

inline int launch_status() {
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SK_OK : (int)e;
}

int sm_count() {
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v <= 0)
        v = 148;
    (void)cudaGetLastError();
    return v;
}

template <int VAR>
int launch_ceiling(uint32_t warps_per_sm, uint32_t rounds, uint32_t* sink, unsigned long long* cycles, cudaStream_t st) {
    const size_t smem = (size_t)warps_per_sm * sk::kTileBytes;
    cudaFuncSetAttribute(sk::sk_loop_ceiling_kernel<VAR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    sk::sk_loop_ceiling_kernel<VAR><<<sm_count(), warps_per_sm * 32, smem, st>>>(sink, cycles, rounds);
    ++g_launches;
    return launch_status();
}

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled() {
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

template <int VAR>
int launch_stream_variant(const CUtensorMap& tmap, const sk::FrameParams& p, cudaStream_t st) {
    auto kernel = sk::sk_stream_kernel<16, 1, false, VAR>;
    cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sk::kStreamSmemBytes);
    cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(p.slabs, p.F, p.B);
    cfg.blockDim = dim3(32);
    cfg.dynamicSmemBytes = sk::kStreamSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, tmap, p);
    if (e == cudaSuccess) ++g_launches;
    return e == cudaSuccess ? SK_OK : (int)e;
}

bool stream_shape_ok(uint32_t T, uint32_t F, uint32_t E, uint32_t M) {
    if (M < 32 || M > 256 || M % 32 != 0 || T == 0 || T % M != 0 || F == 0 || E == 0 || E % 256 != 0) return false;
    if (T / M > 65535u || F > 65535u) return false;
    if ((unsigned long long)F * E + 256ull > (1ull << 31) || (unsigned long long)T >= (1ull << 31)) return false;
    return true;
}

}  // namespace

extern "C" {

int skb_loop_ceiling(int variant, uint32_t warps_per_sm, uint32_t rounds, uint32_t* sink, unsigned long long* cycles,
                     double* h_samples_per_lane, void* stream) {
    if (!sink || !cycles) return SK_ERR_NULL;
    if (warps_per_sm < 1 || warps_per_sm > (uint32_t)sk::kCeilingMaxWarps || rounds == 0) return SK_ERR_SHAPE;
    // samples every lane of every warp has added: rounds x 8 tiles x 256 samples per lane and tile
    if (h_samples_per_lane) *h_samples_per_lane = (double)rounds * sk::kCeilingTilesPerReadout * (sk::kTileBytes / 32);
    cudaStream_t st = (cudaStream_t)stream;
    switch (variant) {
        case SKB_VAR_PRODUCT:   return launch_ceiling<sk::kVarProduct>(warps_per_sm, rounds, sink, cycles, st);
        case SKB_VAR_NO_SUB:    return launch_ceiling<sk::kVarNoSub>(warps_per_sm, rounds, sink, cycles, st);
        case SKB_VAR_NO_PICK:   return launch_ceiling<sk::kVarNoPick>(warps_per_sm, rounds, sink, cycles, st);
        case SKB_VAR_NO_UNPACK: return launch_ceiling<sk::kVarNoUnpack>(warps_per_sm, rounds, sink, cycles, st);
        default: return SK_ERR_PARAM;
    }
}

int skb_pipe_rate(int mode, uint32_t warps_per_sm, uint32_t* io, unsigned long long* cycles,
                  double* h_instructions_per_warp, void* stream) {
    if (!io || !cycles) return SK_ERR_NULL;
    if (mode < 0 || mode >= sk::kPipeModes || warps_per_sm < 1 || warps_per_sm > (uint32_t)sk::kCeilingMaxWarps)
        return SK_ERR_SHAPE;
    const unsigned grid = (unsigned)sm_count(), block = warps_per_sm * 32;
    cudaStream_t st = (cudaStream_t)stream;
    switch (mode) {
        case 0: sk::sk_pipe_rate_kernel<0><<<grid, block, 0, st>>>(io, cycles); break;
        case 1: sk::sk_pipe_rate_kernel<1><<<grid, block, 0, st>>>(io, cycles); break;
        case 2: sk::sk_pipe_rate_kernel<2><<<grid, block, 0, st>>>(io, cycles); break;
        case 3: sk::sk_pipe_rate_kernel<3><<<grid, block, 0, st>>>(io, cycles); break;
        case 4: sk::sk_pipe_rate_kernel<4><<<grid, block, 0, st>>>(io, cycles); break;
        case 5: sk::sk_pipe_rate_kernel<5><<<grid, block, 0, st>>>(io, cycles); break;
        case 6: sk::sk_pipe_rate_kernel<6><<<grid, block, 0, st>>>(io, cycles); break;
        case 7: sk::sk_pipe_rate_kernel<7><<<grid, block, 0, st>>>(io, cycles); break;
        default: sk::sk_pipe_rate_kernel<8><<<grid, block, 0, st>>>(io, cycles); break;
    }
    ++g_launches;
    if (h_instructions_per_warp) *h_instructions_per_warp = (double)sk::kPipeIters * 8 * (mode >= 5 ? 2 : 1);
    return launch_status();
}

size_t skb_stream_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M) {
    if (!stream_shape_ok(T, F, E, M)) return 0;
    const size_t cells = (size_t)(T / M) * F;
    return cells * (E / 256u) * sizeof(double) + ((cells * sizeof(uint32_t) + 7u) & ~(size_t)7u);
}

int skb_stream(int variant, const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, float* SK,
               uint8_t* mask, void* workspace, size_t workspace_bytes, int inputs_ready, void* stream) {
    if (!data || !SK || !mask) return SK_ERR_NULL;
    if (!stream_shape_ok(T, F, E, M) || (reinterpret_cast<uintptr_t>(data) & 15u)) return SK_ERR_SHAPE;
    if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7u) ||
        workspace_bytes < skb_stream_workspace_bytes(T, F, E, M))
        return SK_ERR_WORKSPACE;
    if (!encode_tiled()) return (int)cudaErrorNotSupported;
    constexpr uint32_t W = 256, R = sk::kTileBytes / W;
    sk::FrameParams p{};
    p.data = data; p.T = T; p.F = F; p.E = E; p.M = M; p.B = T / M;
    p.first_n = E;
    p.n_sigma = 5.0f;
    p.nlev = 1;
    p.inputs_ready = inputs_ready ? 1u : 0u;
    p.chunk = M; p.bpu = 1; p.unit_tiles = M / R;
    p.slabs = E / W;
    p.nunits = p.B * F * p.slabs;
    const size_t cells = (size_t)p.B * F;
    p.lev[0].SK = SK; p.lev[0].mask = mask; p.lev[0].sk_mean = 1.0f;
    p.lev[0].partial = static_cast<double*>(workspace);
    p.lev[0].counter = reinterpret_cast<uint32_t*>(static_cast<uint8_t*>(workspace) + cells * p.slabs * sizeof(double));
    CUtensorMap tmap;
    const cuuint64_t gdim[2] = {(cuuint64_t)F * E, (cuuint64_t)T};
    const cuuint64_t gstride[1] = {(cuuint64_t)F * E};
    const cuuint32_t box[2] = {W, R};
    const cuuint32_t estr[2] = {1, 1};
    if (encode_tiled()(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t*>(data), gdim, gstride, box, estr,
                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return (int)cudaErrorInvalidValue;
    cudaStream_t st = (cudaStream_t)stream;
    switch (variant) {
        case SKB_VAR_PRODUCT: return launch_stream_variant<sk::kVarProduct>(tmap, p, st);
        case SKB_VAR_MEMONLY: return launch_stream_variant<sk::kVarMemOnly>(tmap, p, st);
        default: return SK_ERR_PARAM;
    }
}

int skb_frame_loop(void* sk_frame_fn, uint8_t* const* h_frames, uint32_t nframes, uint32_t T, uint32_t F, uint32_t E,
                   uint32_t M, float n_sigma, float sk_mean, int flags, float* SK, uint8_t* mask, void* workspace,
                   size_t workspace_bytes, uint32_t calls, double* h_host_seconds, void* stream) {
    if (!sk_frame_fn || !h_frames || nframes == 0) return SK_ERR_NULL;
    using FrameFn = int (*)(uint8_t*, uint32_t, uint32_t, uint32_t, uint32_t, const uint8_t*, uint32_t, float, float, int,
                            float*, uint8_t*, uint32_t*, uint32_t*, void*, size_t, void*);
    const FrameFn fn = reinterpret_cast<FrameFn>(sk_frame_fn);
    const auto t0 = std::chrono::steady_clock::now();
    int rc = SK_OK;
    for (uint32_t i = 0; i < calls && rc == SK_OK; ++i)
        rc = fn(h_frames[i % nframes], T, F, E, M, nullptr, E, n_sigma, sk_mean, flags, SK, mask, nullptr, nullptr,
                workspace, workspace_bytes, stream);
    const auto t1 = std::chrono::steady_clock::now();
    if (h_host_seconds) *h_host_seconds = std::chrono::duration<double>(t1 - t0).count();
    return rc;
}

unsigned long long skb_launch_count(void) { return g_launches.load(); }

}  // extern "C"
