/*
 * cans_poisson.h -- C ABI of the B200-native FP64 pressure-projection library.
 *
 * What the library computes (citations: /root/reference/PAPER.md, "P:L<n>" = line n):
 *
 *   eq. 2b  P:L59    L Phi = D u* / (gamma_k dt)           divergence of the staggered velocity
 *   eq. 5   P:L95    7-point second-order Laplacian        the linear system
 *   eq. 6   P:L102   F^x, F^y, tridiagonal in z            eigenfunction-expansion direct solve
 *   P:L98-100        "Gauss elimination" along z           Thomas solve per (kx, ky) mode
 *   P:L104           z may be non-uniform                  dzc / dzf arrays
 *   eq. 2c  P:L62    u^{k+1} = u* - gamma_k dt G Phi       pressure-gradient correction
 *
 * Every step runs in hand-written sm_100a CUDA kernels on the device the caller made current;
 * there is no CPU fallback and no other backend.  All floating point is FP64.
 *
 * Layout: every field is a DEVICE pointer to nx*ny*nz contiguous doubles, x fastest
 * (linear index i + nx*(j + ny*k); a torch tensor of shape (nz, ny, nx)), no halo,
 * 16-byte aligned, owned by the caller; the library never frees or retains it.
 * Staggering (marker-and-cell): u[i,j,k] lives on the +x face of cell (i,j,k), v on the
 * +y face, w on the +z face.  Out-of-range neighbours are synthesised from `bc`.
 *
 * Threading: calls only enqueue work on `stream` (a cudaStream_t passed as void*) and never
 * synchronise.  A plan is immutable after creation apart from the registered lower-face planes, the cached
 * tensor maps of the last field and (Helmholtz) the pivot tables per alpha, which calls rewrite on their
 * stream: a plan may be used by ONE stream at a time -- for work that overlaps (u, v, w Helmholtz solves next to
 * a Poisson solve) create one plan per stream.  No function throws or prints.
 */
#ifndef CANS_POISSON_H
#define CANS_POISSON_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cans_poisson_plan cans_poisson_plan;   /* opaque, owned by the library */

/* Return codes of the int-valued entry points. */
#define CANS_OK                    0
#define CANS_ERR_INVALID_ARG       1   /* null pointer, n < 2, non-positive length/spacing/dt, bad bc letter, one-sided 'P' */
#define CANS_ERR_UNSUPPORTED_BC    2   /* face-located unknown along a direction the Helmholtz plan does not implement */
#define CANS_ERR_UNSUPPORTED_SIZE  3   /* nx or ny not in the instantiated transform sizes, or nz too large */
#define CANS_ERR_ALLOC             4   /* device or host allocation failed */
#define CANS_ERR_CUDA              5   /* a CUDA runtime call or kernel launch failed */
#define CANS_ERR_NEEDS_FACE        6   /* projection with a lower 'D' side needs cans_projection_set_lower_face */

/*
 * cans_poisson_plan_create -- build the plan for L Phi = f (eqs. 5-6).
 *
 *   nx, ny, nz   cells per direction (x, y uniform: "uniformly-spaced in two directions").
 *                nx and ny must be one of 16,32,48,64,96,128,192,256,384,512,768,1024,1536,2048
 *                (512, 768 and 1024 run the warp-level 2-pass kernels, the others the 3-pass kernels);
 *                2 <= nz <= 1024.
 *   lx, ly, lz   domain lengths (> 0); dx = lx/nx, dy = ly/ny.
 *   bc           bc[d][0] / bc[d][1] = PRESSURE boundary condition on the lower / upper face of
 *                direction d (0 = x, 1 = y, 2 = z), homogeneous, imposed at the boundary face:
 *                'P' periodic (both sides), 'N' dPhi/dn = 0, 'D' Phi = 0.
 *                Implemented: every pair in every direction -- x, y, z in {PP, NN, DD, ND, DN} ("all combinations of
 *                pressure boundary conditions"; mixed pairs in x, y run DCT-IV / DST-IV).  Periodic z (the triperiodic
 *                Taylor-Green case) solves cyclic tridiagonal systems; for the projection to stay exact its
 *                wrap spacing must be single-valued, dzc[0] == dzc[nz] (uniform grids satisfy this).
 *   dzc          HOST, nz+1 doubles: dzc[k] = distance between the centres of cells k-1 and k
 *                (k = 0 and k = nz reach the mirror ghost centres), or NULL.
 *   dzf          HOST, nz doubles: dzf[k] = width of cell k, or NULL.  Both NULL => uniform lz/nz.
 *                The arrays are copied; the caller keeps ownership.
 *
 * Returns NULL on failure; cans_last_error()/cans_last_status() tell why.
 * The plan owns O(nx + ny + nz + nx*ny*nz/16) doubles of device tables; the solve is in place.
 */
cans_poisson_plan* cans_poisson_plan_create(int nx, int ny, int nz,
                                            double lx, double ly, double lz,
                                            const char bc[3][2],
                                            const double* dzc, const double* dzf);

/*
 * cans_helmholtz_plan_create / cans_helmholtz_solve -- the Helmholtz solves of the implicit-diffusion step (SURVEY 8f row
 * f4): eq. 3b, u* - (gamma nu dt / 2) L u* = rhs, "solved with the same type of direct solver".  Divided by
 * -(gamma nu dt / 2) it reads (L + alpha I) Phi = f with alpha = -2/(gamma nu dt) < 0 and f = alpha * rhs: the same three
 * passes as cans_poisson_solve with every tridiagonal system shifted by alpha (never singular).
 *
 *   bc       here the ghost rule of the UNKNOWN (a velocity component), not of the pressure: 'D' = zero on the boundary face
 *            (no-slip wall for a tangential component), 'N' = zero normal derivative (free slip / outflow), 'P' periodic.
 *   stagger  -1: the unknown lives at the cell centres in every direction (cans_poisson_plan_create is this case);
 *            0, 1, 2: it lives on the +x / +y / +z faces (u, v, w of the staggered arrangement).  Along a periodic
 *            direction the operator is the one for centres.  stagger = 2 with z walls ('D','D'): faces 0..nz-2 are the
 *            unknowns, the wall nodes below face 0 and at face nz-1 are homogeneous (a moving wall is folded into f by the
 *            caller) and slot nz-1 of q is returned as it came; stagger = 2 with ('D','N'): wall below, zero normal
 *            derivative AT the upper boundary face (outflow / free-slip top), face nz-1 is an unknown with a mirrored upper
 *            neighbour; stagger = 2 with periodic z: cyclic systems.  Every other face-located case (non-periodic x or y:
 *            node-based DST-I / DCT-I; a lower 'N' in z: the lower boundary face has no slot in this layout) returns NULL
 *            with CANS_ERR_UNSUPPORTED_BC.
 *   q        DEVICE, nx*ny*nz doubles: f on entry, Phi on exit.     alpha < 0.
 * The pivots entering each z segment depend on alpha: the plan keeps up to CANS_MAX_PIVOT_TABLES tables (N/16 doubles each;
 * the first, for alpha = 0, from plan creation) and builds one -- one device allocation and one extra kernel on the caller's
 * stream -- the first time it meets a new alpha.  The three gamma_k of an RK3 loop therefore cost three builds in the whole
 * run; a further alpha, or a full board, replaces the table used longest ago.  A stagger = 2 plan serves
 * cans_helmholtz_solve only.
 */
#define CANS_MAX_PIVOT_TABLES 4
cans_poisson_plan* cans_helmholtz_plan_create(int nx, int ny, int nz, double lx, double ly, double lz,
                                              const char bc[3][2], const double* dzc, const double* dzf, int stagger);
int cans_helmholtz_solve(cans_poisson_plan* plan, double* q, double alpha, void* stream);

/* Free the plan and its device tables.  NULL is ignored.  Outstanding work must have completed. */
void cans_poisson_plan_destroy(cans_poisson_plan* plan);

/*
 * cans_poisson_solve -- in-place direct solve of eq. 5 by eq. 6.
 *   p       DEVICE, nx*ny*nz doubles.  On entry f, on exit Phi with L Phi = f.
 *           If every direction is PP or NN the operator is singular: f must satisfy
 *           sum f*dzf = 0 to rounding and the returned Phi has zero dzf-weighted mean
 *           (the kx = ky = 0 column is solved with its last row dropped, then shifted).
 *   stream  cudaStream_t as void* (NULL = default stream).
 */
int cans_poisson_solve(cans_poisson_plan* plan, double* p, void* stream);

/*
 * cans_projection -- one pressure-projection step, eqs. 2b-2c:
 *     f = D(u,v,w)/dt ;  L Phi = f ;  (u,v,w) -= dt * G Phi.
 *   u, v, w  DEVICE, corrected in place.
 *   p        DEVICE, overwritten with Phi (entry contents ignored; eq. 2d is the caller's).  u, v, w, p must be four
 *            distinct arrays (CANS_ERR_INVALID_ARG otherwise).
 *   dt       the whole factor gamma_k*Delta_t of eqs. 2b-2c (> 0).
 * The boundary-normal velocity on a lower 'P' face is the wrapped value, on a lower 'N' face 0
 * (or the plane registered with cans_projection_set_lower_face), on a lower 'D' face the registered plane
 * (required); the value on an upper 'N' face
 * (array index n-1) is read and left bit-identical.
 */
int cans_projection(cans_poisson_plan* plan, double* u, double* v, double* w, double* p,
                    double dt, void* stream);

/*
 * cans_projection_step -- cans_projection plus the two bandwidth-only steps a time loop runs after it:
 *   p_acc   DEVICE or NULL: the accumulated pressure; eq. 2d  p_acc += Phi  is done by the correction kernel itself
 *           (the same pass that applies eq. 2c: +16 B/cell instead of a separate 24 B/cell sweep).  Must not alias p, u, v, w.
 *   dti     DEVICE scalar (one double) or NULL: receives the reduction of Listing 1 (`chkdt`; eq. 4)
 *           over the CORRECTED velocities, see cans_chkdt.
 * Everything else as cans_projection (which is this call with p_acc = dti = NULL).
 */
int cans_projection_step(cans_poisson_plan* plan, double* u, double* v, double* w, double* p, double* p_acc,
                         double dt, double* dti, void* stream);

/*
 * cans_projection_step_implicit -- cans_projection_step with the pressure update of the implicit-diffusion scheme, eq. 3e
 * (SURVEY 8f row f4):
 *     p_acc += Phi - nu_dt_half * L Phi,      nu_dt_half = gamma_k nu dt / 2  (>= 0; 0 is eq. 2d and needs no p_acc),
 * L the 7-point Laplacian of eq. 5 with the ghost rule of Phi on every side.  The correction kernel forms L Phi from the Phi
 * values it already holds for the gradient plus its lower neighbours (its own carry in z, cache hits in x and y): the pass
 * still moves 72 B/cell.  p_acc is required when nu_dt_half > 0.  Everything else as cans_projection_step.
 */
int cans_projection_step_implicit(cans_poisson_plan* plan, double* u, double* v, double* w, double* p, double* p_acc,
                                  double dt, double nu_dt_half, double* dti, void* stream);

/*
 * cans_chkdt -- the max-reduction of Listing 1:
 *     dti = max over cells of max(dtix, dtiy, dtiz),
 *     dtix = |u|/dx + |v(i,j)+v(i,j-1)+v(i+1,j)+v(i+1,j-1)|/(4 dy) + |w(i,j,k)+w(i,j,k-1)+w(i+1,j,k)+w(i+1,j,k-1)|/(4 dzf[k])
 *     (P:L181-187), dtiy and dtiz the same pattern on the v and w faces, the latter with 1/dzc[k+1];
 * the stable step of eq. 4 is then min(1.65 dl^2/nu, sqrt(3)/dti) on the host.  Neighbours outside the arrays:
 * wrapped in a periodic direction; otherwise the lower boundary face (registered plane, else 0) for the component normal to
 * it and 0 for every other out-of-range value.
 *   u, v, w  DEVICE, read only.    dti  DEVICE, one double, overwritten (0 for a field at rest).
 * A lower 'D' side without a registered plane returns CANS_ERR_NEEDS_FACE, as in cans_projection.
 */
int cans_chkdt(cans_poisson_plan* plan, const double* u, const double* v, const double* w, double* dti, void* stream);

/*
 * cans_chkdt_static -- cans_chkdt for callers that cannot allocate device memory: no plan, no cudaMalloc / cudaFree and no
 * allocating library routine anywhere inside it.
 *
 * Why it exists.  A plan owns device tables, so creating one allocates and destroying one frees.  Two kinds of caller
 * cannot do that at the point where they need the time step: a solver whose own arena already fills the board's memory
 * (the driver has nothing left to give, the plan's cudaMalloc fails), and a time loop that keeps several streams busy
 * (cudaMalloc and cudaFree wait for the whole device, so every stream in flight stalls behind them).  For them the memory
 * the kernel needs besides the caller's arrays -- the reciprocal z spacings and one partial maximum per CTA -- is a fixed
 * array inside the library image: 528 KB on every GPU that loads libcans_poisson.so, held until the process exits.
 *
 *   nx, ny, nz, lx, ly, lz, bc   as cans_poisson_plan_create (bc = the pressure pairs that fix the ghost rule of cans_chkdt);
 *                nx even and (nx/2)*ny a multiple of 32 (every size a plan accepts is), and within the fixed array:
 *                nz <= CANS_STATIC_MAX_NZ  and  ceil(nx*ny/512) * ceil(nz/32) <= CANS_STATIC_MAX_CTAS
 *                (about 2^30 cells: 1024 x 768 x 512 and 1536 x 768 x 576 fit).  Anything larger returns
 *                CANS_ERR_UNSUPPORTED_SIZE with a message that names the limit; nothing is launched.
 *   dzc, dzf     DEVICE (not host, unlike the plan: a host array would have to be staged), nz+1 / nz doubles with the meaning
 *                given at cans_poisson_plan_create, or both NULL for the uniform spacing lz/nz.  Read on the stream.
 *   u, v, w      DEVICE, nx*ny*nz doubles each, 16-byte aligned, read only.
 *   face_x/y/z   DEVICE lower-face planes with the layout of cans_projection_set_lower_face, or NULL.  Required on a lower
 *                'D' side (CANS_ERR_NEEDS_FACE), optional on a lower 'N' side (prescribed inflow), must be NULL on 'P'.
 *   dti          DEVICE, one double, overwritten; the same value cans_chkdt returns, bit for bit.
 *   stream       cudaStream_t as void*.  Two kernels are enqueued; nothing synchronises.
 *
 * The fixed array is shared by every call in the process and keeps the contents of the last one.  Each call rewrites the
 * spacing tables and zeroes its arrival counter before use, so calls on one stream, or otherwise ordered on the GPU, are
 * independent of each other; calls that can overlap on the GPU (two streams, two host threads) race and return garbage.
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, once, cached): make that first
 * call with the device current and outside any stream capture.
 */
#define CANS_STATIC_MAX_NZ    1024
#define CANS_STATIC_MAX_CTAS  65536
int cans_chkdt_static(int nx, int ny, int nz, double lx, double ly, double lz, const char bc[3][2],
                      const double* dzc, const double* dzf, const double* u, const double* v, const double* w,
                      const double* face_x, const double* face_y, const double* face_z, double* dti, void* stream);

/*
 * cans_projection_set_lower_face -- register the boundary-normal velocity on the LOWER face of
 * direction dir (0,1,2): DEVICE plane of (product of the other two extents) doubles, x fastest among the
 * remaining indices (dir 0: j + ny*k; dir 1: i + nx*k; dir 2: i + nx*j), 16-byte aligned, or NULL to
 * unregister.  The library keeps the pointer (caller-owned memory, must outlive its registration).
 * On a 'D' side the plane is read by the divergence (eq. 2b) and corrected in place by eq. 2c with the
 * anti-mirrored ghost (-= dt*2*Phi_0/h, h = dx, dy or dzc[0]); without it cans_projection returns
 * CANS_ERR_NEEDS_FACE, because the projected field would not be divergence free.  On an 'N' side it is a
 * prescribed inflow, read by the divergence and not modified.  A periodic direction has no lower face:
 * CANS_ERR_INVALID_ARG.  cans_poisson_solve ignores the planes.
 */
int cans_projection_set_lower_face(cans_poisson_plan* plan, int dir, double* face_plane);

/*
 * Host-buffer convenience entry points (used for end-to-end timing): copy the HOST arrays to
 * device buffers owned by the plan (allocated on first use), run the device path on `stream`,
 * copy the results back and synchronise the stream.  Pinned host memory gives full PCIe rate.
 * Only the four fields travel: lower-face planes registered with cans_projection_set_lower_face stay DEVICE pointers
 * here too -- they are read, and on 'D' sides corrected, where they are; the caller copies them if it wants them.
 */
int cans_poisson_solve_host(cans_poisson_plan* plan, double* p_host, void* stream);
int cans_projection_host(cans_poisson_plan* plan, double* u_host, double* v_host, double* w_host,
                         double* p_host, double dt, void* stream);

/* Thread-local message / status code of the last failure on this thread ("" / CANS_OK if none). */
const char* cans_last_error(void);
int cans_last_status(void);

/* Number of kernel launches one cans_poisson_solve / cans_projection call enqueues (for bench.py). */
int cans_plan_launches_per_solve(const cans_poisson_plan* plan);
int cans_plan_launches_per_projection(const cans_poisson_plan* plan);

/*
 * Optional per-kernel timing for bench.py.  With profiling enabled every kernel launch of the next
 * cans_poisson_solve / cans_projection call is bracketed by a cudaEvent pair on the caller's stream; at most
 * CANS_MAX_KERNEL_RECORDS records per call.  cans_plan_kernel_times waits for those events and writes the duration (ms) of each record of
 * the LAST call, in launch order, into ms[0..capacity); returns the number written, or -1 on error.
 * cans_plan_kernel_name returns the name of record idx of the last call ("" if out of range).
 */
#define CANS_MAX_KERNEL_RECORDS 16
int cans_plan_set_profiling(cans_poisson_plan* plan, int enable);
int cans_plan_kernel_times(cans_poisson_plan* plan, float* ms, int capacity);
const char* cans_plan_kernel_name(const cans_poisson_plan* plan, int idx);

/* "x.y" version string of the library. */
const char* cans_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CANS_POISSON_H */
