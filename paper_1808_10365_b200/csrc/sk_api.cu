// sk_api.cu — the C ABI of include/sk_b200.h: argument checks, shape -> kernel choice, launches.
// Nothing here allocates device memory or synchronises (sk_frame_host waits for its own copies).
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>

#include "../../include/sk_b200.h"
#include "sk_kernels.cuh"
#include "sk_tma.cuh"
#include "sk_sim.cuh"

#include <cstdlib>
#include <cstring>

namespace {

std::atomic<unsigned long long> g_launches{0};

inline int launch_status() {
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SK_OK : (int)e;
}

int sm_count();

// Lanes per row for the vector path (slab width = 16*L inputs).  The sum over inputs follows a
// canonical tree over the input indices (sk_kernels.cuh), so the choice affects speed only, never
// a result: wide 256-byte slabs (fewest units, least per-unit work) when that still gives every
// SM enough warps; otherwise narrower slabs.  A lone frame needs ~16 warps per SM of its own;
// frames that overlap their neighbours on the stream (SK_FRAME_INPUTS_READY) share the SM with
// them and run best on wide slabs from 8 warps per SM up (measured on config 1: 16.3 vs 17.0 us).
inline int lanes_per_row(uint32_t E, uint32_t cells, uint32_t M, bool overlapped) {
    const uint32_t vecs = E / 16;            // 128-bit vectors per row
    int L = 16;
    while (L > 1 && (uint32_t)L > vecs) L >>= 1;
    const unsigned long long want = (unsigned long long)sm_count() * (overlapped ? 8u : 16u);
    while (L > 4 && (unsigned long long)cells * ((E + 16u * L - 1) / (16u * L)) < want) L >>= 1;
    if (const char* e = std::getenv("SK_B200_LANES")) {     // tests: force a (narrower) slab width
        const int v = std::atoi(e);
        if (v >= 1 && v <= L && (v & (v - 1)) == 0) L = v;
    }
    // long blocks: narrower slabs put more rows under one warp-wide read, so that a lane still
    // adds at most AccChain::kMaxSamples samples per unit (the stream kernel's exactness limit)
    while (L > 1 && (M + 32u / L - 1) / (32u / L) > sk::AccChain::kMaxSamples) L >>= 1;
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

struct Plan {
    bool vec;
    int L;
    uint32_t slabs;       // launched slabs per cell
    bool wide;            // AccWide usable (samples per lane <= 511)
    bool stream;          // stream kernel usable (samples per lane <= 128)
    bool grid_ok;         // F and B fit the y and z grid dimensions
};

Plan make_plan(const void* data, uint32_t E, uint32_t M, uint32_t B, uint32_t F, const uint8_t* subset,
               uint32_t first_n, bool need_all_inputs, bool overlapped) {
    Plan pl{};
    const uint32_t cells = B * F;
    // the stream kernel's grid is (slabs, F, B) and its tensor map has a row of F*E bytes
    pl.grid_ok = B <= 65535u && F <= 65535u && (unsigned long long)F * E < (1ull << 32);
    pl.vec = vector_ok(data, E);
    pl.L = lanes_per_row(E, cells, M, overlapped);
    const uint32_t W = 16u * pl.L;
    uint32_t cover = E;
    if (!subset && !need_all_inputs) cover = first_n;    // inputs beyond first_n are never read
    pl.slabs = (cover + W - 1) / W;
    const uint32_t RPW = 32u / pl.L;
    const uint32_t iters = (M + RPW - 1) / RPW;
    pl.wide = iters <= sk::AccWide::kMaxSamples;
    pl.stream = iters <= sk::AccChain::kMaxSamples;
    return pl;
}

template <class Acc>
void launch_vec_L(int L, const sk::FrameParams& p, cudaStream_t st) {
    const unsigned grid = (p.nunits + sk::kWarpsPerCta - 1) / sk::kWarpsPerCta;
    const unsigned block = sk::kWarpsPerCta * 32;
    switch (L) {
        case 16: sk::sk_frame_kernel<16, Acc><<<grid, block, 0, st>>>(p); break;
        case 8:  sk::sk_frame_kernel<8, Acc><<<grid, block, 0, st>>>(p); break;
        case 4:  sk::sk_frame_kernel<4, Acc><<<grid, block, 0, st>>>(p); break;
        case 2:  sk::sk_frame_kernel<2, Acc><<<grid, block, 0, st>>>(p); break;
        default: sk::sk_frame_kernel<1, Acc><<<grid, block, 0, st>>>(p); break;
    }
    ++g_launches;
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

int sm_count() {
    static int n = [] {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
            v = 148;
        return v > 0 ? v : 148;
    }();
    return n;
}

// SK_B200_PATH=ldg|tma forces one vector kernel (for tests and A/B timing); default: TMA when it applies
// (the stream kernel keeps its sums in AccWide fields: at most 511 samples per lane and unit).
bool tma_wanted(const Plan& pl) {
    const char* e = std::getenv("SK_B200_PATH");
    if (e && std::strcmp(e, "ldg") == 0) return false;
    return pl.stream && pl.grid_ok && encode_tiled() != nullptr;
}

template <int L>
int launch_stream_L(const CUtensorMap& tmap, const sk::FrameParams& p, cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(sk::sk_stream_kernel<L>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)sk::kStreamSmemBytes);
        cudaFuncSetAttribute(sk::sk_stream_kernel<L>, cudaFuncAttributePreferredSharedMemoryCarveout,
                             cudaSharedmemCarveoutMaxShared);
        attr_set = true;
    }
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
    const cudaError_t e = cudaLaunchKernelEx(&cfg, sk::sk_stream_kernel<L>, tmap, p);
    return e == cudaSuccess ? SK_OK : (int)e;
}

int launch_stream(int L, const sk::FrameParams& p, cudaStream_t st) {
    CUtensorMap tmap;
    const uint32_t W = 16u * L;
    const cuuint64_t gdim[2] = {(cuuint64_t)p.F * p.E, (cuuint64_t)p.T};
    const cuuint64_t gstride[1] = {(cuuint64_t)p.F * p.E};
    const cuuint32_t box[2] = {(cuuint32_t)W, (cuuint32_t)(sk::kTileBytes / W)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode_tiled()(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t*>(p.data), gdim,
                                      gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return (int)cudaErrorInvalidValue;
    int rc;
    switch (L) {
        case 16: rc = launch_stream_L<16>(tmap, p, st); break;
        case 8:  rc = launch_stream_L<8>(tmap, p, st); break;
        case 4:  rc = launch_stream_L<4>(tmap, p, st); break;
        case 2:  rc = launch_stream_L<2>(tmap, p, st); break;
        default: rc = launch_stream_L<1>(tmap, p, st); break;
    }
    if (rc == SK_OK) ++g_launches;
    return rc;
}

int launch_cells(const Plan& pl, sk::FrameParams& p, cudaStream_t st) {
    const uint32_t cells = p.B * p.F;
    if (pl.vec) {
        p.slabs = pl.slabs;
        p.nunits = cells * pl.slabs;
        if (tma_wanted(pl)) {
            const int rc = launch_stream(pl.L, p, st);
            if (rc != SK_OK) return rc;
        } else if (pl.stream) launch_vec_L<sk::AccChain>(pl.L, p, st);
        else if (pl.wide) launch_vec_L<sk::AccWide>(pl.L, p, st);
        else                launch_vec_L<sk::AccPlain>(pl.L, p, st);
    } else {
        sk::sk_cell_kernel_scalar<<<cells, sk::kScalarThreads, 0, st>>>(p);
        ++g_launches;
    }
    return launch_status();
}

size_t workspace_bytes(uint32_t cells, uint32_t slabs_max) {
    return (size_t)cells * slabs_max * sizeof(double) + (size_t)cells * sizeof(uint32_t);
}

}  // namespace

extern "C" {

int sk_power_sums(const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                  uint32_t* S1, uint32_t* S2, void* stream) {
    if (!data || !S1 || !S2) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    Plan pl = make_plan(data, E, M, T / M, F, nullptr, E, true, false);
    if ((reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2)) & 15u) pl.vec = false;
    sk::FrameParams p{};
    p.data = data; p.T = T; p.F = F; p.E = E; p.M = M; p.B = T / M;
    p.first_n = E;
    p.S1out = S1; p.S2out = S2;
    return launch_cells(pl, p, (cudaStream_t)stream);
}

size_t sk_frame_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M) {
    if (check_shape(T, F, E, M)) return 0;
    const uint32_t cells = (T / M) * F;
    return workspace_bytes(cells, (E + 15u) / 16u);     // room for the narrowest slabs any plan uses
}

static int frame_impl(const uint8_t* data, uint32_t T,
                      uint32_t F, uint32_t E, uint32_t M, const uint8_t* subset, uint32_t first_n,
                      float n_sigma, float sk_mean, int flags, float* SK, uint8_t* mask, uint32_t* S1o,
                      uint32_t* S2o, void* workspace, size_t workspace_bytes_given, cudaStream_t st) {
    if (!SK) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    if (!subset && (first_n == 0 || first_n > E)) return SK_ERR_N;
    if (mask && (!std::isfinite(n_sigma) || !std::isfinite(sk_mean) || n_sigma < 0)) return SK_ERR_PARAM;
    if ((S1o == nullptr) != (S2o == nullptr)) return SK_ERR_NULL;
    Plan pl = make_plan(data, E, M, T / M, F, subset, first_n, S1o != nullptr, (flags & SK_FRAME_INPUTS_READY) != 0);
    if (S1o && ((reinterpret_cast<uintptr_t>(S1o) | reinterpret_cast<uintptr_t>(S2o)) & 15u)) pl.vec = false;
    sk::FrameParams p{};
    p.data = data; p.T = T; p.F = F; p.E = E; p.M = M; p.B = T / M;
    p.subset = subset; p.first_n = subset ? 0 : first_n;
    p.n_sigma = n_sigma; p.sk_mean = sk_mean;
    p.inputs_ready = (flags & SK_FRAME_INPUTS_READY) ? 1u : 0u;
    p.SK = SK; p.mask = mask; p.S1out = S1o; p.S2out = S2o;
    if (pl.vec) {
        const uint32_t cells = p.B * F;
        const size_t need = workspace_bytes(cells, pl.slabs);
        if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7u) || workspace_bytes_given < need)
            return SK_ERR_WORKSPACE;
        p.partial = static_cast<double*>(workspace);
        // counters sit after the largest possible partial array, so their place does not depend
        // on first_n or on the slab width and a workspace stays clean across calls
        const uint32_t slabs_max = (E + 15u) / 16u;
        if (workspace_bytes_given < workspace_bytes(cells, slabs_max)) return SK_ERR_WORKSPACE;
        p.counter = reinterpret_cast<uint32_t*>(static_cast<double*>(workspace) + (size_t)cells * slabs_max);
    }
    return launch_cells(pl, p, st);
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
    p.SK = SK; p.S1in = S1; p.S2in = S2;
    const uint32_t cells = B * F;
    const bool vec = E % 16 == 0 &&
                     ((reinterpret_cast<uintptr_t>(S1) | reinterpret_cast<uintptr_t>(S2)) & 15u) == 0;
    if (vec) {
        const int L = lanes_per_row(E, cells, M, false);
        p.slabs = (E + 16u * L - 1) / (16u * L);
        p.nunits = cells * p.slabs;
        const size_t smem = (size_t)p.slabs * sizeof(double);
        if (smem > 48 * 1024) return SK_ERR_SHAPE;
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
    const int zero_flagged = flags & SK_FRAME_ZERO_FLAGGED;
    if (!data || !SK || !mask) return SK_ERR_NULL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = frame_impl(data, T, F, E, M, subset, first_n, n_sigma, sk_mean, flags, SK, mask,
                        S1_opt, S2_opt, workspace, workspace_bytes_given, st);
    if (rc != SK_OK || !zero_flagged) return rc;
    const uint32_t cells = (T / M) * F;
    const dim3 grid(cells, (M + sk::kExciseRows - 1) / sk::kExciseRows);
    if (vector_ok(data, E)) sk::sk_excise_kernel<true><<<grid, 256, 0, st>>>(data, mask, F, E, M);
    else                    sk::sk_excise_kernel<false><<<grid, 256, 0, st>>>(data, mask, F, E, M);
    ++g_launches;
    return launch_status();
}

int sk_frame_host(uint8_t* h_data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, const uint8_t* subset,
                  uint32_t first_n, float n_sigma, float sk_mean, int flags, float* h_SK,
                  uint8_t* h_mask, uint8_t* d_data, float* d_SK, uint8_t* d_mask, void* workspace,
                  size_t workspace_bytes_given, void* stream) {
    if (!h_data || !h_SK || !h_mask || !d_data || !d_SK || !d_mask) return SK_ERR_NULL;
    if (int rc = check_shape(T, F, E, M)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)T * F * E, cells = (size_t)(T / M) * F;
    cudaError_t e = cudaMemcpyAsync(d_data, h_data, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return (int)e;
    const int zero_flagged = flags & SK_FRAME_ZERO_FLAGGED;
    const int rc = sk_frame(d_data, T, F, E, M, subset, first_n, n_sigma, sk_mean, zero_flagged, d_SK,
                            d_mask, nullptr, nullptr, workspace, workspace_bytes_given, stream);
    if (rc != SK_OK) return rc;
    e = cudaMemcpyAsync(h_SK, d_SK, cells * sizeof(float), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_mask, d_mask, cells, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && zero_flagged)
        e = cudaMemcpyAsync(h_data, d_data, bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? SK_OK : (int)e;
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
        default: return code > 0 ? cudaGetErrorString((cudaError_t)code) : "unknown error";
    }
}

int sk_version(void) { return 101; }

unsigned long long sk_launch_count(void) { return g_launches.load(); }

}  // extern "C"
