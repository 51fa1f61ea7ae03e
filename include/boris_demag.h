/* boris_demag.h — C ABI of libborisdemag.so
 *
 * Demagnetizing field of one rectangular mesh of equal cuboid cells on one
 * NVIDIA B200 (sm_100a):
 *
 *     H(r0) = - sum_r N(r - r0) M(r)              PAPER.md:L323 (Table 1), Eq. 4 (L73) with n = 1
 *
 * with N the Newell cell-averaged demagnetizing tensor (Ref. [50]),
 * evaluated by the convolution theorem with zero padding to twice
 * the mesh size in every non-flat dimension, organised as the
 * paper's "pipelined convolution" (the innermost forward FFT, the
 * point-by-point tensor multiplication and the innermost inverse FFT in a single
 * kernel launch, for all three vector components at once).
 *
 * Conventions
 *   - SI units: M, H in A/m; cell sides in metres; energy in joules; mu0 = 4 pi 1e-7.
 *   - M and H are fp32, planar, [3][nz][ny][nx], x fastest: element (c, k, j, i) of
 *     a component c in {x, y, z} at cell (i, j, k) is at ((c*nz + k)*ny + j)*nx + i.
 *   - Supported sizes: 1 <= nx, ny <= 1024, 1 <= nz <= 512 (nz = 1: 2-D mode, Nxz and Nyz
 *     dropped); anything else: error -1.  The kernels work on power-of-two meshes (nx >= 4,
 *     ny >= 2, nz = 1 or >= 2): any other mesh is evaluated exactly as the corner of the next
 *     power-of-two mesh whose remaining cells hold M = 0 (linear convolution only needs a
 *     padded length >= 2n - 1), staged through plan-owned buffers by two copy
 *     kernels per call; M and H then only need 4-byte alignment.
 *   - All fp32 arithmetic on the device; fp64 only at plan time and in the energy sum.
 *   - A plan owns the kernel spectrum, twiddle tables and workspace on the device
 *     that was current when it was created; every apply / energy call checks that the
 *     same device is current and fails with -1 otherwise.  It may be used from one
 *     stream at a time (the workspace is shared).  The caller owns M, H and E.
 *   - Return codes: 0 ok; -1 invalid argument; -2 CUDA error; -3 out of memory.
 *     boris_demag_last_error() returns a thread-local message for the last failure.
 *   - There is no CPU fallback: without a CUDA device plan_create fails with -2.
 */
#ifndef BORIS_DEMAG_H
#define BORIS_DEMAG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct boris_demag_plan boris_demag_plan;   /* opaque; owns device memory */

/* Build a plan (PAPER.md:L324 tensor, L275 kernel "in the transform space").
 * nx, ny, nz: cells; hx, hy, hz: cell sides in metres (> 0).
 * Synchronous; evaluates the tensor and its real, symmetry-reduced spectrum in
 * fp64 on the device, stores it as fp32.  Returns NULL on failure (see last_error). */
boris_demag_plan* boris_demag_plan_create(int nx, int ny, int nz, double hx, double hy, double hz);

/* The same with periodic boundary conditions by the multiple-images method (section 3: "we
 * extend this algorithm to use periodic boundary conditions based on the multiple images method [51]"; Ref. [51]
 * at L434).  images_x / _y / _z >= 0: copies of the mesh on EACH side along x / y / z (0: open boundary; all 0
 * is boris_demag_plan_create).  The field in the mesh is that of the finite block of (2 images + 1) copies per
 * periodic direction, all carrying the mesh's own M:
 *     H(r0) = - sum_{|n_a| <= images_a} sum_r N(r - r0 + (n_x nx hx, n_y ny hy, n_z nz hz)) M(r).
 * Only the plan-time tensor changes (the copies' tensors are summed into the kernel spectrum in fp64); apply,
 * energy and every other call work as for an open mesh and cost the same.  Plan time grows with the number
 * of copies.  Returns NULL on failure (images < 0 or > 1000: -1). */
boris_demag_plan* boris_demag_plan_create_pbc(int nx, int ny, int nz, double hx, double hy, double hz,
                                              int images_x, int images_y, int images_z);

/* Free everything the plan owns.  NULL is allowed. */
void boris_demag_plan_destroy(boris_demag_plan* plan);

/* H = -N * M.  M, H: DEVICE pointers, fp32 [3][nz][ny][nx],
 * 16-byte aligned, must not alias.  H is overwritten.  `stream` is a cudaStream_t
 * passed as void* (NULL = default stream).  Enqueues kernels and returns at once;
 * never allocates, never synchronises; bit-identical across calls. */
int boris_demag_apply(boris_demag_plan* plan, const float* M, float* H, void* stream);

/* Variants of boris_demag_apply selected by `flags` (0 = boris_demag_apply itself):
 *   BORIS_DEMAG_AOS         M and H hold one float3 per cell, [nz][ny][nx][3], the layout of a vector-field
 *                           library instead of planar components;
 *   BORIS_DEMAG_ACCUMULATE  H += -N * M instead of H = -N * M: the demag term added to an effective field
 *                           that already holds other contributions ("additive field contributions").
 * ACCUMULATE alone, on a mesh the tiled or plane kernels take as it is (power-of-two sizes), is
 * fused: the kernel that writes H reads the old value and adds (12 more bytes per cell, no extra launch, M and H
 * 16-byte aligned as for boris_demag_apply).  Every other combination (AOS, other meshes) goes
 * through plan-owned planar staging buffers and two copy kernels (M in, H out); on a power-of-two
 * mesh the buffers are allocated (both or neither) by the FIRST such call (24 bytes per cell), which is the
 * one case in which an apply allocates and synchronises — do not make that first call inside a stream capture.  M, H: DEVICE pointers, 4-byte aligned, must not alias.  Error codes as boris_demag_apply. */
#define BORIS_DEMAG_AOS 1u
#define BORIS_DEMAG_ACCUMULATE 2u
int boris_demag_apply_ex(boris_demag_plan* plan, const float* M, float* H, unsigned flags, void* stream);

/* boris_demag_apply, instrumented for the measurement harness: a CUDA event pair is
 * recorded on `stream` around every kernel launch, the stream is synchronised, and the
 * device time is returned summed per kernel kind, in the order
 *   0 XFwd (S1)  1 Y2D (S2+S4+S6, nz = 1)  2 YFwd (S2)  3 ZFused (S3+S4+S5)  4 YInv (S6)  5 XInv (S7)
 * ms_by_kind[6] (milliseconds) and launches_by_kind[6] are HOST arrays.  Synchronous;
 * computes exactly what boris_demag_apply computes (same kernels, same order). */
int boris_demag_apply_timed(boris_demag_plan* plan, const float* M, float* H, void* stream,
                            float ms_by_kind[6], int launches_by_kind[6]);

/* E = -(mu0/2) hx hy hz sum_cells M.H  (PAPER.md:L293 relation between field and
 * energy density, integrated; reading R13).  M, H: DEVICE pointers as in
 * apply.  E_dev: DEVICE pointer to one double, written asynchronously on `stream`.
 * Deterministic fixed-shape two-level reduction in one launch (warp shuffles; the last block to
 * finish adds the block sums in index order, so E is bit-identical across calls). */
int boris_demag_energy(boris_demag_plan* plan, const float* M, const float* H, double* E_dev, void* stream);

/* boris_demag_apply followed by boris_demag_energy in one enqueue: H = -N * M and
 * E = -(mu0/2) hx hy hz sum(M.H) (north_star).  On the tiled kernel paths the
 * sum is gathered by the kernel that writes H (fp64 per-block sums, added in block order by the
 * block that finishes last: bit-identical across calls), so M and H are not read again; other
 * meshes run the two calls back to back.  Arguments, layout, aliasing and error codes as for
 * boris_demag_apply and boris_demag_energy; E_dev is a DEVICE double. */
int boris_demag_apply_energy(boris_demag_plan* plan, const float* M, float* H, double* E_dev, void* stream);

/* Same computation with HOST buffers: copies M host->device, applies, computes the
 * energy, copies H (and E if E_host != NULL) device->host and synchronises `stream`.
 * M_host, H_host: host pointers, fp32 [3][nz][ny][nx] (pinned memory makes the
 * copies asynchronous; pageable works).  Uses device staging buffers owned by the
 * plan (allocated on first use: the first call may return -3). */
int boris_demag_apply_host(boris_demag_plan* plan, const float* M_host, float* H_host, double* E_host, void* stream);

/* Thread-local description of the last error in this library ("" if none). */
const char* boris_demag_last_error(void);

/* Introspection for the measurement harness (north_star: "with the number of HBM
 * passes stated").  Any out pointer may be NULL.
 *   compulsory_bytes   = 12 N (M in) + 12 N (H out) + 4 ncomp (Px/2+1)(Py/2+1)(Pz/2+1),
 *                        ncomp = 4 and Pz/2+1 -> 1 when nz = 1, else 6
 *   designed_hbm_bytes = bytes the kernels of one apply are designed to move to/from HBM
 *   workspace_bytes    = device memory owned by the plan
 *   padded[3]          = (Px, Py, Pz)
 *   kernel_launches    = kernels enqueued by one apply */
int boris_demag_plan_info(const boris_demag_plan* plan, long long* compulsory_bytes,
                          long long* designed_hbm_bytes, long long* workspace_bytes,
                          int padded[3], int* kernel_launches);

/* The caller's mesh the plan was created for: cells[3] = (nx, ny, nz), sides[3] = (hx, hy, hz) in metres
 * (one rectangular mesh of equal cuboid cells).  Either out pointer may be NULL. */
int boris_demag_plan_mesh(const boris_demag_plan* plan, int cells[3], double sides[3]);

/* Which kernel path the plan uses and how much it stores (harness bookkeeping).
 * Any out pointer may be NULL.
 *   path                 = 2: tiled 2-D (XFwdT, YFused, XInvT), 3: tiled 3-D (XZFwd, YFused, ZXInv),
 *                          4: plane path of nz = 32 slabs (XFwdT, YZFused, XInvP; csrc/plane.h),
 *                          0: chunked fallback (XFwd, [Y2D | YFwd, ZFused, YInv per chunk], XInv)
 *   spectrum_bytes       = bytes of the intermediate spectrum array in HBM (V, W or the plane path's X)
 *   kernel_storage_bytes = bytes of the stored fp32 kernel spectrum (with layout padding)
 *   cols                 = kx columns per tile of the tiled paths, ky residues (partial planes) of the
 *                          plane path (0 otherwise) */
int boris_demag_plan_layout(const boris_demag_plan* plan, int* path, long long* spectrum_bytes,
                            long long* kernel_storage_bytes, int* cols);

/* Copy the plan's kernel spectrum back to the host in natural, symmetry-reduced
 * order: out[c][kz][ky][kx], c in (xx,yy,zz,xy[,xz,yz]), kz <= Pz/2 (1 plane if nz = 1),
 * ky <= Py/2, kx <= Px/2, INCLUDING the folded factor -1/(2 Px Py Pz) (DESIGN.md
 * reading R12).  out must hold ncomp*(Pz/2+1)*(Py/2+1)*(Px/2+1) floats.  Synchronous. */
int boris_demag_plan_kernel_spectrum(const boris_demag_plan* plan, float* out_host);

/* ---- host-only entry points (no GPU needed; used by the CPU tests) -------------- */

/* The library's own real-space tensor (fp64 Newell formulas near, Gauss quadrature of
 * the point-dipole tensor over the cell-separation distribution far),
 * evaluated on the host with the same source code the device kernel compiles.
 * out[6][nz][ny][nx]: N_c at displacement (i hx, j hy, k hz), c = xx,yy,zz,xy,xz,yz. */
int boris_demag_tensor_host(int nx, int ny, int nz, double hx, double hy, double hz, double* out);

/* The tensor of boris_demag_plan_create_pbc (the image sum above), same layout.  Small meshes and few copies. */
int boris_demag_tensor_host_pbc(int nx, int ny, int nz, double hx, double hy, double hz, int images_x, int images_y,
                                int images_z, double* out);

/* The natural-order reduced kernel spectrum (as boris_demag_plan_kernel_spectrum, in
 * fp64, same folded factor) computed on the host from boris_demag_tensor_host by the
 * same cosine/sine-transform code the device kernels compile.  Small meshes only. */
int boris_demag_spectrum_host(int nx, int ny, int nz, double hx, double hy, double hz, double* out);

/* Library version string, e.g. "boris-demag-b200 0.1 (sm_100a)". */
const char* boris_demag_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BORIS_DEMAG_H */
