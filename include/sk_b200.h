/* sk_b200.h — C ABI of the B200 spectral-kurtosis (SK) RFI detector.
 *
 * Implements the data-parallel hot path of arXiv 1808.10365 ("Spectral Kurtosis Based RFI
 * Mitigation for CHIME"; citations are lines of /root/reference/PAPER.md):
 *
 *   a1-a3  unpack 4+4-bit samples, |x|^2, S1 = sum |x|^2, S2 = sum |x|^4 per M-sample block
 *          (PAPER.md:45 Eq. 1, :77 Eq. 7, :278 for the 4+4-bit data)
 *   a4-a6  SK~ = (M+1)/(M-1) * (S2bar/(M N) - 1),  S2bar = sum_i M^2 (S2)_i / (S1)_i^2
 *          (PAPER.md:84-88 Eq. 9-11, :108-113 Eq. 14 — the estimator CHIME runs)
 *   a7     flag cells outside sk_mean +- n_sigma * sqrt(4/(M N))   (PAPER.md:183, :119 Eq. 16, :284)
 *   a8     optional excision of flagged cells
 *
 * Conventions common to every call
 *   - Layout: data[T][F][E] uint8, E contiguous.  byte = (re+8)<<4 | (im+8), re, im in [-8, 7]
 *     (nibble 0 decodes to -8; the encoded zero sample is 0x88).  A "cell" is one (block b,
 *     frequency f): rows t = b*M .. (b+1)*M-1, each E contiguous bytes at stride F*E.
 *     B = T/M blocks.  S1, S2: uint32 [B][F][E].  SK: float32 [B][F].  mask: uint8 [B][F].
 *   - Pointers are DEVICE pointers owned by the caller unless the name starts with h_.
 *     The library allocates no device memory, never synchronises the device (except
 *     sk_frame_host, which waits for its own copies) and enqueues all work on `stream`
 *     (a cudaStream_t cast to void*; NULL = the legacy default stream) before returning.
 *   - Return value: 0 = enqueued; < 0 = argument error (SK_ERR_*), nothing was enqueued;
 *     > 0 = a cudaError_t reported by a launch or copy.  No exceptions.  The only process-wide
 *     state is the launch counter (sk_launch_count) and per-device caches of device attributes and
 *     of the address of sk_frame_noalloc's scratch; nothing a caller can set outlives its call.
 *   - Receiver selection ("total number of receivers"): `subset` is NULL or E
 *     bytes on the device (non-zero = combine this input).  With subset == NULL the first
 *     `first_n` inputs are combined (first_n = E for the whole array).  N is the number of
 *     combined inputs; with a subset it is counted on the device.  An empty subset yields
 *     SK = NaN and mask = 1 for every cell.
 *   - A receiver whose S1 is 0 contributes the term M (its own SK^_i taken as 0), so an
 *     all-0x88 cell gives SK = 0 exactly and re-running on excised data is NaN-free.
 *   - Limits: 2 <= M <= 65536, T % M == 0, T, F, E >= 1, T*F*E < 2^40, E <= 2^20, (T/M)*F < 2^31
 *     (anything beyond returns SK_ERR_SHAPE or SK_ERR_M).
 *     Any E and any alignment is accepted; E % 16 == 0 with a 16-byte-aligned `data` takes the
 *     vector kernels, everything else a slower scalar kernel with identical results.
 *   - Floating point: per-input terms and the sum over inputs are float64 in a fixed order
 *     (deterministic run to run); SK is that value rounded to float32; the flag decision is
 *     taken in float32: fabsf(SK - sk_mean) > (float)(n_sigma * sqrt(4.0/(M*N))), strict,
 *     NaN => flagged.
 */
#ifndef SK_B200_H
#define SK_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SK_OK                 0
#define SK_ERR_NULL          -1   /* a required pointer is NULL */
#define SK_ERR_SHAPE         -2   /* T, F, E, B out of range, or T % M != 0, or too large */
#define SK_ERR_M             -3   /* M < 2 or M > 65536 */
#define SK_ERR_N             -4   /* first_n == 0 or first_n > E (subset == NULL), or N == 0 */
#define SK_ERR_PARAM         -5   /* n_sigma or sk_mean not finite, n_sigma < 0 */
#define SK_ERR_WORKSPACE     -6   /* workspace NULL, misaligned (8 bytes) or too small */
#define SK_ERR_SCRATCH       -7   /* sk_frame_noalloc: the shape needs more than SK_NOALLOC_SCRATCH_BYTES */

/* a1-a3 (Eq. 7).  Reads data[T][F][E]; writes S1, S2 [T/M][F][E] (exact integers). */
int sk_power_sums(const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                  uint32_t* S1, uint32_t* S2, void* stream);

/* a4-a6 (PAPER.md:84-88 Eq. 9-11, :108-113 Eq. 14).  Reads S1, S2 [B][F][E]; writes SK [B][F]. */
int sk_combine(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E,
               uint32_t M, const uint8_t* subset, uint32_t first_n, float* SK, void* stream);

/* a7 (variance PAPER.md:119 Eq. 16; centre sk_mean = 1 by Eq. 15 or the simulated
 * null mean of PAPER.md:284).  Reads SK [B][F]; writes mask [B][F] (0/1). */
int sk_flag(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N, float n_sigma,
            float sk_mean, uint8_t* mask, void* stream);

/* Bytes of device workspace sk_frame needs for this shape (0 on a bad shape).  The workspace
 * must be 8-byte aligned and ZERO-FILLED before its first use; every completed sk_frame call
 * leaves it zero-filled again, so it can be reused by later calls on the same stream without
 * clearing.  Do not share one workspace between calls that may run concurrently. */
size_t sk_frame_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M);

/* Bits of sk_frame's `flags`. */
#define SK_FRAME_ZERO_FLAGGED  1  /* a8: excise flagged cells in place */
#define SK_FRAME_INPUTS_READY  2  /* see below */
#define SK_FRAME_EQ13          4  /* SK = the un-rescaled estimator of PAPER.md:97-104 Eq. 13,
                                   * (MN+1)/(MN-1) * (S2bar/(MN) - 1), instead of Eq. 14; the flag
                                   * interval is applied to it unchanged (pass the matching sk_mean) */
/* Tests and A/B timing: override the library's kernel choice for THIS call (sk_frame, sk_frame_multi,
 * sk_frame_noalloc, sk_frame_host, sk_frame_plan).  Results do not depend on any of them
 * (DESIGN.md section 5.1): every kernel and slab width gives the same bits. */
#define SK_FRAME_PLAN_LDG      (1 << 8)   /* the direct-load kernel instead of the TMA stream kernel */
#define SK_FRAME_PLAN_NO_TMAP  (1 << 9)   /* plan as usual, then behave as if the driver had refused to encode
                                           * the tensor map: exercises the fall-back to the direct-load kernels */
#define SK_FRAME_PLAN_LANES(l) (((l) & 31) << 12)   /* l = 1, 2, 4, 8, 16: slab width 16*l inputs, if not wider
                                                     * than a row; 0 = automatic */

/* a1-a8 in one pass over HBM.  Writes SK and mask [T/M][F]; S1_opt / S2_opt [T/M][F][E] are
 * written when non-NULL.  With SK_FRAME_ZERO_FLAGGED every byte (all E inputs, all M rows) of
 * each flagged cell is overwritten in place with 0x88 as soon as the cell's mask is known, by
 * the same kernel (the mask and SK are those of the data before excision); otherwise `data` is
 * only read.
 * SK_FRAME_INPUTS_READY is a promise by the caller that nothing enqueued on `stream` since the
 * last stream synchronisation or the last sk_frame call made WITHOUT this flag writes this
 * call's `data` or `subset` (e.g. the frame was uploaded and synchronised earlier, and the calls
 * in between worked on, and excised, other buffers).  The kernel is launched with programmatic
 * stream serialization; with the promise it reads `data` while the previous kernel on the stream
 * is still draining and waits for it only before its first write (outputs and workspace), so
 * back-to-back frames overlap tail and ramp-up.  Without the flag the kernel waits for all
 * previous work on the stream before its first read.  Results are identical either way. */
int sk_frame(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
             const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean,
             int flags, float* SK, uint8_t* mask, uint32_t* S1_opt, uint32_t* S2_opt,
             void* workspace, size_t workspace_bytes, void* stream);

/* sk_frame for callers that cannot allocate device memory.
 *
 * Who that is: a stage plugged into a real-time correlator pipeline is usually handed its frame and
 * output buffers by the host framework, which reserved the whole GPU at start-up and gives a stage no
 * allocator of its own; a plug-in running inside somebody else's process may be forbidden to touch
 * the device heap at all; and a frame loop that has gone real-time cannot afford cudaMalloc anyway,
 * because it synchronises the device and stalls every other stage sharing the GPU.  sk_frame asks
 * such a caller for a zero-filled workspace it has no way to provide.  This call does not: its
 * workspace is an array of SK_NOALLOC_SCRATCH_BYTES built into the library's device image.  The
 * caller passes only the frame and the outputs, exactly as for sk_frame; results are identical.
 *
 * What it costs and where the limit is: every GPU on which this library's kernels are loaded holds
 * those SK_NOALLOC_SCRATCH_BYTES (4 MiB) from then until the process exits, whether or not this
 * call is ever made.  A shape whose sk_frame_workspace_bytes(T, F, E, M) is larger (it grows as
 * (T/M) * F * ceil(E/16) * 8 bytes: configs 0-2 of BASELINE.json fit, the 8 GiB frames of config 4
 * do not) is refused with SK_ERR_SCRATCH before anything is enqueued; use sk_frame with a
 * workspace from the framework's pool for those.
 *
 * The call itself never calls cudaMalloc, cudaFree or any library routine that allocates.  The
 * first call made with a given device current also looks up the array's address on that device
 * (cudaGetSymbolAddress, which may make the runtime load the library's kernels onto the device):
 * make that first call during start-up, with the right device current, and before any stream
 * capture begins; later calls on that device only enqueue work.
 *
 * Sharing: there is ONE array per device, used by every sk_frame_noalloc call of the process on
 * that device, and it keeps what the last call left in it.  Each call therefore first clears the
 * part it needs (a memset enqueued on `stream` ahead of the kernel), so a previous call of any
 * shape, even a failed one, cannot disturb the result.  But two calls whose work overlaps on the
 * GPU (different streams, or different host threads on different streams) race on the array and
 * give wrong results: keep all sk_frame_noalloc calls of one device on one stream, or order
 * them with events.  sk_frame with caller workspaces has no such restriction.
 * Because of the clear, SK_FRAME_INPUTS_READY is accepted but buys no overlap with the previous
 * kernel.  Arguments, flags, outputs and return values otherwise as for sk_frame. */
#define SK_NOALLOC_SCRATCH_BYTES (4u << 20)
int sk_frame_noalloc(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                     const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean,
                     int flags, float* SK, uint8_t* mask, uint32_t* S1_opt, uint32_t* S2_opt,
                     void* stream);

/* Several integration lengths from ONE pass over HBM ("compute real-time SK
 * estimates at a variety of integration lengths"): the fused path at M, 2M, ..., M << (nlev-1),
 * 1 <= nlev <= 4.  Eq. 7's sums over 2M samples are the sums of two adjacent M-sample blocks
 * (exact integers), so the data is streamed once and every length gets its own Eq. 14 estimate
 * and flag decision.  h_SK / h_mask / h_sk_means are HOST arrays of nlev entries: device
 * pointers SK_l float32 [T/(M<<l)][F] and mask_l uint8 [T/(M<<l)][F], and the flag centre of each
 * length.  T % (M << (nlev-1)) == 0 and M << (nlev-1) <= 65536.  Workspace: the size
 * sk_frame_multi_workspace_bytes returns, zero-filled before first use, left zero-filled.
 * With SK_FRAME_ZERO_FLAGGED a sample is excised when the cell of ANY length that contains it is
 * flagged; every estimate is that of the data before excision.  Other flags as for sk_frame. */
size_t sk_frame_multi_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t nlev);
int sk_frame_multi(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t nlev,
                   const uint8_t* subset, uint32_t first_n, float n_sigma, const float* h_sk_means,
                   int flags, float* const* h_SK, uint8_t* const* h_mask,
                   void* workspace, size_t workspace_bytes, void* stream);

/* End-to-end form with HOST buffers (pinned memory recommended): copies h_data to d_data,
 * runs sk_frame there, copies SK and mask (and, with SK_FRAME_ZERO_FLAGGED, the excised data) back, and
 * waits for the copies.  d_data (T*F*E bytes), d_SK, d_mask, workspace are caller-owned device
 * buffers; subset is a device pointer as above.  h_data is written only with SK_FRAME_ZERO_FLAGGED;
 * SK_FRAME_INPUTS_READY is ignored (the upload precedes the kernel).  Argument errors (< 0) are
 * reported before anything is enqueued; after a launch or copy error (> 0) the call still waits
 * for what it had enqueued. */
int sk_frame_host(uint8_t* h_data, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                  const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean,
                  int flags, float* h_SK, uint8_t* h_mask,
                  uint8_t* d_data, float* d_SK, uint8_t* d_mask,
                  void* workspace, size_t workspace_bytes, void* stream);

/* sk_frame_host for a QUEUE of frames: h_frames is a HOST array of nframes host pointers (T*F*E bytes each,
 * pinned memory recommended); h_SK float32 [nframes][T/M][F] and h_mask uint8 [nframes][T/M][F] receive the
 * results of frame i at index i.  Upload, kernel and read-back of all frames are enqueued back to back on
 * `stream` and the call waits ONCE at the end, so the host-to-device link is never idle while the host turns
 * a call around (sk_frame_host waits after every frame).  One staging frame d_data and one set of device
 * outputs d_SK / d_mask / workspace serve all frames (stream order keeps them safe).  With
 * SK_FRAME_ZERO_FLAGGED every h_frames[i] is overwritten with its excised frame.  Results per frame are those
 * of sk_frame_host.  Errors as for sk_frame_host; after a launch or copy error the frames not yet enqueued are
 * dropped and the call still waits for what it had enqueued. */
int sk_frames_host(uint8_t* const* h_frames, uint32_t nframes, uint32_t T, uint32_t F, uint32_t E, uint32_t M,
                   const uint8_t* subset, uint32_t first_n, float n_sigma, float sk_mean, int flags,
                   float* h_SK, uint8_t* h_mask, uint8_t* d_data, float* d_SK, uint8_t* d_mask,
                   void* workspace, size_t workspace_bytes, void* stream);

/* ---- outputs next to the hot path ---------------------------------- */

/* Several integration lengths from one pass ("a variety of integration
 * lengths"): Eq. 7's sums over factor*M samples are the sums of `factor` adjacent M-sample blocks.
 * Reads S1, S2 [B][F][E] (from sk_power_sums or sk_frame's S1_opt/S2_opt); writes S1out, S2out
 * [B/factor][F][E], exact integers, which sk_combine / sk_single then take with M*factor.
 * B % factor == 0, factor >= 1, M*factor <= 65536 (the sums must still fit 32 bits). */
int sk_rebin_sums(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E,
                  uint32_t M, uint32_t factor, uint32_t* S1out, uint32_t* S2out, void* stream);

/* Per-receiver estimates (Eq. 8; the "independent SK estimates" of PAPER.md:73):
 * SKi[b][f][e] = (M+1)/(M-1) * (M S2/S1^2 - 1), float64 inside, float32 out; 0 where S1 == 0.
 * Their mean over the combined receivers is sk_combine's SK (Eq. 14, third line). */
int sk_single(const uint32_t* S1, const uint32_t* S2, uint32_t B, uint32_t F, uint32_t E, uint32_t M,
              float* SKi, void* stream);

/* Detection significance: sig = (SK - sk_mean) / sqrt(4/(M N)) (Eq. 16), float64
 * inside, float32 out; NaN stays NaN.  sk_flag's mask is |sig| > n_sigma up to float32 rounding
 * at the boundary (the mask itself is always decided as the header's conventions state). */
int sk_significance(const float* SK, uint32_t B, uint32_t F, uint32_t M, uint32_t N, float sk_mean,
                    float* sig, void* stream);

/* Digitisation simulation (App. B: "4+4-bit complex Gaussian data (bounded
 * between -7 and 7) with an RMS of ~1.52 least-significant bits in each component").  Fills
 * data[T][F][E] with seeded samples: for row r = t*F + f and receiver pair j = e/2 the
 * counter-based generator Philox4x32-10 is called with counter (j, r, frame_lo, frame_hi) and key
 * (seed_lo, seed_hi); words 0, 1 give (re, im) of receiver 2j, words 2, 3 of receiver 2j+1; a
 * component is -7 + #{k : word >= thr[e][k]}.  thr: uint32 [E][14] on the device, ascending per
 * receiver, thr[e][k] = 2^32 * P(component <= k - 7) for the caller's sigma_e.  T*F < 2^32.
 * Run sk_frame on the result and sk_moments on its SK to get the null mean to pass as sk_mean
 * ("this offset is added directly to the value of the RFI excision threshold"). */
int sk_sim_digitised(uint8_t* data, uint32_t T, uint32_t F, uint32_t E, const uint32_t* thr,
                     uint64_t seed, uint64_t frame, void* stream);

/* Common-mode simulation (App. A, Fig. 5): D independent datasets of M time
 * samples x N receivers, x = z + amp * c with z independent unit circular complex Gaussians and c
 * one common circular Gaussian per time sample; writes SK[d] = Eq. 14 of dataset d (float64
 * inside, float32 out; the samples are never stored).  Random numbers: Philox4x32-10, key
 * (seed_lo, seed_hi), counter (e/2, t, d, 0) for the receivers (words 0,1 / 2,3 = receivers 2j /
 * 2j+1) and (0, t, d, 1) for c; a Gaussian pair is the Box-Muller transform of two words.
 * 2 <= M <= 2048.  sk_moments(SK, D, 1) then gives var(SK) and N_eff = 4 / (M var). */
int sk_sim_common_mode(uint32_t D, uint32_t M, uint32_t N, double amp, uint64_t seed, float* SK,
                       void* stream);

/* Mean and unbiased variance (NaN if B < 2) of SK [B][F] over the blocks, per frequency:
 * float64 mean[F], var[F] on the device.  Two passes, fixed summation order. */
int sk_moments(const float* SK, uint32_t B, uint32_t F, double* mean, double* var, void* stream);

/* Text for a return value of the calls above (static storage; never NULL). */
const char* sk_strerror(int code);

/* Library version: major*10000 + minor*100 + patch. */
int sk_version(void);

/* Number of kernels the library has launched in this process so far (for the bench's
 * gpu_launches count; monotonically increasing, thread-safe). */
unsigned long long sk_launch_count(void);

/* The launch plan sk_frame / sk_frame_multi would use for this shape with a 16-byte-aligned `data`
 * and no subset (a pure function of its arguments and the device's SM count; for tests and for
 * bench reporting).  flags: SK_FRAME_INPUTS_READY and the SK_FRAME_PLAN_* bits matter.  plan4 (HOST,
 * 4 words) = { lanes (slab width / 16), slabs launched per cell (only those covering first_n), rows
 * per accumulator read-out of the TMA stream kernel or 0 when the direct-load kernel would run,
 * M-row blocks per unit }. */
int sk_frame_plan(uint32_t T, uint32_t F, uint32_t E, uint32_t M, uint32_t first_n, int flags,
                  uint32_t nlev, uint32_t* plan4);

#ifdef __cplusplus
}
#endif
#endif /* SK_B200_H */
