/* boris_llg.h — C ABI of the Landau-Lifshitz-Gilbert evaluation around the demag path
 * (SURVEY.md section 8(f), NEXT-1): what one "evaluation" of the paper's benchmark unit
 * ("time per evaluation") contains besides the demagnetizing field.
 *
 *   H_eff(m) = H_demag(Ms m)                        boris_demag_apply
 *            + 2A/(mu0 Ms) laplacian(m), dm/dn = 0  direct exchange
 *            + H_applied                            uniform Zeeman term
 *   dm/dt    = -gamma/(1 + alpha^2) [ m x H_eff + alpha m x (m x H_eff) ]    Eq. (1) solved for dm/dt
 *   RK4 with a fixed time step, 4 evaluations per step, m renormalised after each step.
 *
 * m, H_eff: DEVICE pointers, fp32, planar [3][nz][ny][nx] (the layout of boris_demag.h), m a unit vector per cell.
 * SI units (A/m, m, s, J/m); uniform Ms, A, alpha.  The Laplacian is the 6-neighbour (4 in 2-D) second-order
 * finite difference on the cell centres.  All calls enqueue on `stream` (a cudaStream_t as void*) and return at
 * once.  Return codes and boris_demag_last_error() as in boris_demag.h.  No CPU fallback.
 */
#ifndef BORIS_LLG_H
#define BORIS_LLG_H

#include "boris_demag.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct boris_llg boris_llg;   /* opaque; owns device work arrays, borrows the demag plan */

/* `plan` is the demag plan of the same nx x ny x nz mesh and cell (it must outlive the solver and is used on
 * the solver's stream).  Ms > 0 (A/m), A >= 0 (J/m), alpha >= 0, gamma > 0 (m/(A s); mu0 |gamma_e| = 2.2128e5).
 * (nx, ny, nz) and (hx, hy, hz) are checked against the plan (boris_demag_plan_mesh): a mismatch is rejected.
 * Returns NULL on failure, with the reason in boris_demag_last_error(). */
boris_llg* boris_llg_create(boris_demag_plan* plan, int nx, int ny, int nz, double hx, double hy, double hz,
                            double Ms, double A, double alpha, double gamma);
void boris_llg_destroy(boris_llg* s);

/* Uniform applied field in A/m (default 0). */
int boris_llg_set_applied_field(boris_llg* s, double Hx, double Hy, double Hz);

/* One evaluation of the effective field: Heff = H_demag(Ms m) + H_exchange(m) + H_applied.  m and Heff must not alias. */
int boris_llg_effective_field(boris_llg* s, const float* m, float* Heff, void* stream);

/* nsteps RK4 steps of length dt (seconds) in place on m: 4 effective-field evaluations per step. */
int boris_llg_rk4(boris_llg* s, float* m, double dt, int nsteps, void* stream);

#ifdef __cplusplus
}
#endif
#endif
