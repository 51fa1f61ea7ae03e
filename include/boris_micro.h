/* boris_micro.h — two device probes behind the design arguments of DESIGN.md §5-§6 (measurement
 * tooling of libborisdemag.so, not part of the hot path).  `bench.py --micro` prints their table.
 *
 *   boris_micro_fp32_rate     lane-operations per second of one FP32 instruction kind issued from
 *                             independent register chains on every SM: the ALU roofline the FFT
 *                             butterflies ("1D FFTs") are measured against, and the
 *                             evidence that the packed f32x2 forms run at the same lane rate in half
 *                             the issue slots.
 *   boris_micro_segment_bw    HBM throughput of a stream that touches memory in contiguous pieces
 *                             of `seg_bytes` scattered over a large buffer: what the kx-tiled
 *                             spectrum layouts cost when a kernel meets them in
 *                             32-, 64- or 128-byte pieces.
 *
 * Both allocate and free their own device buffers, run on the current device, synchronise, and
 * return 0, -1 (invalid argument) or -2 (CUDA error; boris_demag_last_error() has the text).
 */
#ifndef BORIS_MICRO_H
#define BORIS_MICRO_H
#ifdef __cplusplus
extern "C" {
#endif

/* op: 0 FADD, 1 FFMA, 2 FADD2 (packed pair), 3 FFMA2 (packed pair).  *lane_ops_per_s: scalar
 * operations per second over the whole device (an FFMA counts once, a packed instruction as two). */
int boris_micro_fp32_rate(int op, double* lane_ops_per_s);

/* seg_bytes: 16, 32, 64, 128, 256 or 512.  write: 0 = read stream, 1 = write stream.
 * *gbs: useful bytes per second / 1e9 over a 1 GiB buffer (larger than L2). */
int boris_micro_segment_bw(int seg_bytes, int write, double* gbs);

#ifdef __cplusplus
}
#endif
#endif
