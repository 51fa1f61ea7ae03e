/* boris_demag_f64.h — the double-precision variant of the demagnetizing-field convolution
 * (the convolution runs "either with single or double floating
 * point precision").
 *
 *     H(r0) = - sum_r N(r - r0) M(r)          PAPER.md:L323, evaluated as in PAPER.md:L275 / L283
 *
 * Same method, tensor and kernel spectrum as boris_demag.h (the plan-time code is fp64 for both), with fp64
 * data and arithmetic throughout, organised as the paper's pipelined convolution: x FFTs, y FFTs, one launch for
 * "the z (inverse)FFTs and point-by-point multiplications ... simultaneously for all 3 vector components"
 * (PAPER.md:L275), inverse y and x FFTs — five kernel launches per evaluation.
 *
 * Conventions as in boris_demag.h: SI units; M, H are fp64, planar [3][nz][ny][nx], x fastest, DEVICE pointers,
 * 8-byte aligned, must not alias; 1 <= nx, ny <= 1024, 1 <= nz <= 512 (nz = 1: 2-D mode); a mesh that is not
 * a power of two is evaluated exactly as the corner of the next power-of-two mesh; periodic boundary
 * conditions by copies of the mesh as in boris_demag_plan_create_pbc.  The plan owns the fp64 kernel
 * spectrum, twiddle tables and workspace (the x spectrum X and its y-padded transform Y, about 144 bytes per cell) on the
 * device that was current at creation; one stream at a time.  Return codes and boris_demag_last_error() as in
 * boris_demag.h.  No CPU fallback.  FP64 is not this chip's fast path: the variant exists for accuracy.
 */
#ifndef BORIS_DEMAG_F64_H
#define BORIS_DEMAG_F64_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct boris_demag_f64_plan boris_demag_f64_plan;   /* opaque; owns device memory */

/* images_x / _y / _z: copies of the mesh on each side along x / y / z (0: open boundary).
 * Synchronous.  Returns NULL on failure (see boris_demag_last_error). */
boris_demag_f64_plan* boris_demag_f64_plan_create(int nx, int ny, int nz, double hx, double hy, double hz,
                                                  int images_x, int images_y, int images_z);
void boris_demag_f64_plan_destroy(boris_demag_f64_plan* plan);

/* H = -N * M in fp64.  Enqueues five kernels on `stream` (a cudaStream_t as void*) and
 * returns at once; never allocates; bit-identical across calls. */
int boris_demag_f64_apply(boris_demag_f64_plan* plan, const double* M, double* H, void* stream);

/* E = -(mu0/2) hx hy hz sum_cells M.H into a DEVICE double (reading R13): fixed-shape
 * two-level fp64 reduction in one launch, bit-identical across calls.  M and H may alias. */
int boris_demag_f64_energy(boris_demag_f64_plan* plan, const double* M, const double* H, double* E_dev, void* stream);

/* workspace_bytes = device memory owned by the plan; padded[3] = (Px, Py, Pz) of the power-of-two mesh;
 * kernel_launches = kernels enqueued by one apply (5).  Any out pointer may be NULL. */
int boris_demag_f64_plan_info(const boris_demag_f64_plan* plan, long long* workspace_bytes, int padded[3],
                              int* kernel_launches);

#ifdef __cplusplus
}
#endif
#endif
