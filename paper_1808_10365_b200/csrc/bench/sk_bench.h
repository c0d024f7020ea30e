/* sk_bench.h — C ABI of libsk_b200_bench.so: MEASUREMENT ONLY.
 *
 * Not part of the product boundary (that is include/sk_b200.h -> libsk_b200.so, which contains none of
 * this).  bench.py and one GPU test load it; it holds the kernels DESIGN.md section 6 argues from, so
 * that every number there can be re-run from the tree:
 *   - the SM-side ceiling of the hot loop (the stream kernel's loop body on a fixed shared-memory tile)
 *     and its removal variants (without the FADD2, without the PRMTs, without the unpack);
 *   - issue rates of the loop's instructions alone and in pairs;
 *   - the stream kernel with its arithmetic replaced by an XOR of the loaded words ("is memory the limit?").
 * Same conventions as sk_b200.h: device pointers unless the name starts with h_, work is enqueued on
 * `stream`, 0 = enqueued, < 0 = argument error (SK_ERR_* of sk_b200.h), > 0 = cudaError_t. */
#ifndef SK_B200_BENCH_H
#define SK_B200_BENCH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Loop-body variants (sk_device.cuh kVar*). */
#define SKB_VAR_PRODUCT   0
#define SKB_VAR_MEMONLY   1
#define SKB_VAR_NO_SUB    2
#define SKB_VAR_NO_PICK   3
#define SKB_VAR_NO_UNPACK 4

/* The stream kernel's tile loop (a1-a3 on 128-bit shared-memory reads) on a fixed shared-memory tile with
 * no global-memory traffic: one CTA per SM, warps_per_sm (1..16) warps each, `rounds` x 8 tiles of 8 KiB per
 * warp.  variant: SKB_VAR_PRODUCT, _NO_SUB, _NO_PICK or _NO_UNPACK.  sink: (SM count) * warps_per_sm * 32
 * words, written (keeps the arithmetic alive); cycles: one 64-bit word = elapsed SM clocks of CTA 0;
 * h_samples_per_lane (HOST, may be NULL) = samples every lane has added.  Sub-partition cycles per 32
 * samples = cycles / (samples_per_lane * warps_per_sm / 4), warps_per_sm a multiple of 4. */
int skb_loop_ceiling(int variant, uint32_t warps_per_sm, uint32_t rounds, uint32_t* sink, unsigned long long* cycles,
                     double* h_samples_per_lane, void* stream);

/* Issue rate of the hot loop's instructions, alone and in pairs, 8 independent chains per lane.  mode:
 * 0 FFMA, 1 FFMA2 (fma.rn.f32x2), 2 FADD2 (sub.rn.f32x2), 3 IDP.4A (dp4a), 4 PRMT, 5 IDP + FFMA2,
 * 6 IDP + FFMA, 7 PRMT + FFMA2, 8 IDP + PRMT.  io: 2048 + (SM count) * warps_per_sm * 32 words (the first
 * 2048 are read as operands, the rest written); cycles: elapsed SM clocks of CTA 0;
 * h_instructions_per_warp (HOST, may be NULL) = warp instructions every warp issued.  Sub-partition cycles
 * per instruction = cycles / (instructions * warps_per_sm / 4). */
int skb_pipe_rate(int mode, uint32_t warps_per_sm, uint32_t* io, unsigned long long* cycles,
                  double* h_instructions_per_warp, void* stream);

/* The product's TMA stream kernel (256-byte slabs, one M-row cell per unit, programmatic dependent launch)
 * with the loop body of `variant` (SKB_VAR_PRODUCT or SKB_VAR_MEMONLY) on data[T][F][E]: same loads, same
 * ring, same epilogue and finalizer, so the time difference is the arithmetic.  With SKB_VAR_MEMONLY the SK
 * and mask it writes are meaningless.  Needs E % 256 == 0, M % 32 == 0, 32 <= M <= 256, a 16-byte-aligned
 * `data`, F*E + 256 <= 2^31; workspace: (T/M)*F*(E/256)*8 + (T/M)*F*4 bytes (rounded up to 8), zero-filled
 * before first use, left zero-filled.  inputs_ready as SK_FRAME_INPUTS_READY. */
size_t skb_stream_workspace_bytes(uint32_t T, uint32_t F, uint32_t E, uint32_t M);
int skb_stream(int variant, const uint8_t* data, uint32_t T, uint32_t F, uint32_t E, uint32_t M, float* SK,
               uint8_t* mask, void* workspace, size_t workspace_bytes, int inputs_ready, void* stream);

/* What a plain C caller of the PRODUCT gets without a CUDA graph: calls sk_frame (the product library's own
 * entry point, passed in as sk_frame_fn so that this library does not link against it) `calls` times in a
 * plain loop on `stream`, call i on h_frames[i % nframes] (HOST array of device pointers), all with the same
 * outputs and workspace.  *h_host_seconds (HOST, may be NULL) = wall time the loop took on the host, i.e.
 * calls x the host cost of one sk_frame call (argument checks, plan, tensor-map encode, launch) when the
 * device keeps up, or the device time when it does not.  The caller times the device side with events around
 * this call.  Returns the first non-zero sk_frame result. */
int skb_frame_loop(void* sk_frame_fn, uint8_t* const* h_frames, uint32_t nframes, uint32_t T, uint32_t F, uint32_t E,
                   uint32_t M, float n_sigma, float sk_mean, int flags, float* SK, uint8_t* mask, void* workspace,
                   size_t workspace_bytes, uint32_t calls, double* h_host_seconds, void* stream);

/* Kernels this library has launched so far in this process. */
unsigned long long skb_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SK_B200_BENCH_H */
