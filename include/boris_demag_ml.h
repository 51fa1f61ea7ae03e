/* boris_demag_ml.h — multi-layered demagnetizing-field convolution
 *
 * PAPER.md:L71-L76, Eq. (4): for a collection of meshes V_k
 *
 *     H(r'_kl) = - sum_i sum_{r_ij in V_i} N(r'_kl - r_ij, h_k, h_i) M(r_ij),      r'_kl in V_k,
 *
 * evaluated as the paper says (L76): per mesh a forward transform, "summation of inter-mesh contributions moved
 * to the transform space", per mesh an inverse transform.  Ref. [23], which generalizes the tensor to arbitrary
 * pairs of meshes, is not available; this library covers the case its use in the paper reduces to, a film STACK
 * (reading R17): `nlayers` layers, each one cell thick, nx x ny cells of the same in-plane size
 * (hx, hy) on the same in-plane grid, every layer with its own thickness and centre height (arbitrary spacers,
 * no common z grid).  N between unequal cuboids is Newell's formula [50] with the z part of its stencil
 * generalized to two heights (csrc/ml_math.h).
 *
 * M, H: DEVICE pointers, planar [3][nlayers][ny][nx], x fastest — the layer index where boris_demag.h has z —
 * fp32 (plan created with fp64 = 0) or fp64 (fp64 = 1); must not alias.  1 <= nx, ny <= 1024, 1 <= nlayers <= 32;
 * in-plane sizes that are not powers of two sit in the corner of the next power-of-two mesh.  SI units.  Open
 * boundaries.  The plan owns the layer-pair kernel spectra (6 real arrays per ordered pair), twiddle tables and
 * workspace on the device that was current at creation; one stream at a time.  Return codes and
 * boris_demag_last_error() as in boris_demag.h.  No CPU fallback.  Five kernel launches per evaluation (x, y,
 * multiply over layer pairs, inverse y, inverse x); correctness-first kernels (csrc/simple_engine.cuh), not the
 * tuned single-mesh path.
 */
#ifndef BORIS_DEMAG_ML_H
#define BORIS_DEMAG_ML_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct boris_demag_ml_plan boris_demag_ml_plan;   /* opaque; owns device memory */

/* thickness[k] > 0 and z_centre[k] (metres, HOST arrays of nlayers doubles): cell height and centre height of
 * layer k.  Layers must not overlap.  Synchronous.  Returns NULL on failure. */
boris_demag_ml_plan* boris_demag_ml_plan_create(int nx, int ny, int nlayers, double hx, double hy,
                                                const double* thickness, const double* z_centre, int fp64);
void boris_demag_ml_plan_destroy(boris_demag_ml_plan* plan);

/* H_k = - sum_i N_ki * M_i for every layer k (Eq. 4).  M, H: float* (fp32 plan) or double* (fp64 plan) passed as
 * void*.  Enqueues on `stream` (a cudaStream_t as void*), returns at once, never allocates. */
int boris_demag_ml_apply(boris_demag_ml_plan* plan, const void* M, void* H, void* stream);

/* E = -(mu0/2) sum_k hx hy thickness[k] sum_cells M_k . H_k into a DEVICE double (PAPER.md:L293 integrated over
 * the stack; fp64 accumulation, fixed-shape reduction). */
int boris_demag_ml_energy(boris_demag_ml_plan* plan, const void* M, const void* H, double* E_dev, void* stream);

/* Host-only: the library's tensor between unequal cuboids on the in-plane octant, out[6][ny][nx] =
 * N_c((i hx, j hy, Z), target thickness tk, source thickness ti), c = xx,yy,zz,xy,xz,yz (CPU tests). */
int boris_demag_ml_pair_tensor_host(int nx, int ny, double hx, double hy, double tk, double ti, double Z, double* out);

#ifdef __cplusplus
}
#endif
#endif
