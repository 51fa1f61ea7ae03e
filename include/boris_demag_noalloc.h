/* boris_demag_noalloc.h — an entry point of libborisdemag.so that allocates nothing.
 *
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it): the demagnetizing energy of S8,
 *
 *     E = -(mu0/2) hx hy hz sum_cells M.H        (integrated; reading R13),
 *
 * computed by a variant of the energy kernel of boris_demag_energy whose scratch memory (the fp64 block sums of its
 * two-level reduction and the ticket counter that elects the block which adds them) lives in a file-scope
 * `static __device__` array of the library instead of a plan's cudaMalloc'd workspace.  No plan is needed.
 *
 * The array has BORIS_DEMAG_NOALLOC_SCRATCH_BYTES bytes (128 KB of block sums + 256 bytes for the ticket): every GPU
 * that loads the library holds it until the process exits.  One block sums 8192 values of M.H, so at most
 * BORIS_DEMAG_NOALLOC_MAX_VALUES = 2^27 values per field (44.7 M cells; 1024 x 1024 x 32 is 100.7 M values) are accepted.
 *
 * The call runs no cudaMalloc, cudaFree or allocating library routine: it enqueues, on `stream`, one 4-byte
 * cudaMemsetAsync (the ticket must start at zero whatever an earlier, possibly failed, call left there) and one
 * kernel.  The address of the array is looked up once per device with cudaGetSymbolAddress, the first time the
 * entry point is called with that device current.
 *
 * Sharing: EVERY call on a device uses the same array, which keeps the last call's contents.  Calls on one stream
 * are ordered and safe.  Calls that overlap on the GPU (different streams, or several host threads on streams that
 * are not ordered with respect to each other) race on the block sums and the ticket: their results are undefined.
 * Serialise them, or use boris_demag_energy, whose scratch belongs to the plan.
 */
#ifndef BORIS_DEMAG_NOALLOC_H
#define BORIS_DEMAG_NOALLOC_H

#ifdef __cplusplus
extern "C" {
#endif

#define BORIS_DEMAG_NOALLOC_MAX_VALUES (1LL << 27)
#define BORIS_DEMAG_NOALLOC_SCRATCH_BYTES (16384 * 8 + 256)

/* M, H: DEVICE pointers, 16-byte aligned, n_values floats each (n_values = 3 nx ny nz for the [3][nz][ny][nx] arrays
 * of boris_demag_apply; any layout in which M and H match element by element gives the same sum).  They are only read.
 * hx, hy, hz: cell size in metres (> 0).  E_dev: DEVICE pointer to one double, written asynchronously on `stream`
 * (a cudaStream_t, or NULL for the default stream).  The caller owns every buffer.
 * Deterministic: fixed blocks of 8192 values, block sums added in index order; bit-identical across calls.
 * Returns 0, or -1 for an invalid argument (null or misaligned pointer, n_values < 1, n_values above
 * BORIS_DEMAG_NOALLOC_MAX_VALUES, non-positive cell size), -2 for a CUDA error; boris_demag_last_error()
 * (boris_demag.h) has the message.  There is no CPU fallback. */
int boris_demag_energy_noalloc(const float* M, const float* H, long long n_values, double hx, double hy, double hz,
                               double* E_dev, void* stream);

#ifdef __cplusplus
}
#endif
#endif
