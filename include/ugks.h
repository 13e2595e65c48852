/* ugks.h -- C ABI of libugks: the 2-D BGK Unified Gas-Kinetic Scheme time step on one B200
 * (hand-written CUDA for sm_100a, fp64).  Plain C: no C++ or torch types cross this boundary.
 *
 * The operation is the time step of arXiv:1810.08137 (cited as P:Lnn = /root/reference/PAPER.md line nn):
 *   model and Maxwellian g            P:L27-32  Eq. (1)
 *   integral solution at a cell face  P:L34-37  Eq. (2)
 *   update of f (implicit BGK)        P:L39-43  Eq. (3)
 *   update of W                       P:L45-46  Eq. (4)
 *   flux evaluation steps S1..S8
 * The paper delegates the flux construction to its refs [1,2]; the concrete formulas are the
 * readings O0..O12 / AMB-1..22 of DESIGN.md.
 *
 * Conventions
 *   - Cells (i,j), i in [0,I), j in [0,J), uniform on [x0,x1]x[y0,y1]; cell index c = j*I + i.
 *   - Velocity nodes u[k] (k<Nu), v[m] (m<Nv), 1-D weights wu, wv; point q = m*Nu + k.
 *   - f is fp64, dense row-major [J][I][Nv][Nu] (u fastest): the paper's f_{i,j,k,m}.
 *   - W is fp64 [J][I][4] = (rho, rho U, rho V, rho E); K_int = 0, gamma = 2 (AMB-2).
 *   - Every function returns UGKS_OK (0) or an error code; ugks_last_error() gives a message.
 *   - Pointers passed in stay owned by the caller and are not retained after the call returns, EXCEPT
 *     workspace_dev and cuda_stream given to ugks_init, which the caller keeps alive until ugks_destroy.
 *   - "ptrs_on_device" says whether the data pointers of that call are device (1) or host (0) pointers.
 *     Host copies are enqueued on the context's stream and the call returns after they complete.
 *   - All work is enqueued on the stream given to ugks_init.  ugks_step is asynchronous.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with UGKS_ECUDA.
 *   - The two kernels that sweep f are compiled by NVRTC at ugks_init with the context's geometry as compile-time constants
 *     (csrc/ugks_jit_*.cuh, read from the directory of libugks.so); if NVRTC or those sources are missing, ugks_init fails.
 *   - A context belongs to the device that was current at ugks_init; every call switches to it and back.
 *   - Calls on different contexts may run concurrently from different host threads; calls on one context may not.
 */
#ifndef UGKS_H
#define UGKS_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ugks_ctx ugks_ctx;                       /* opaque, owned by the library */

enum { UGKS_OK = 0, UGKS_EINVAL = 1, UGKS_ENOMEM = 2, UGKS_ECUDA = 3, UGKS_ESTATE = 4 };
enum { UGKS_BC_PERIODIC = 0, UGKS_BC_FIXED = 1, UGKS_BC_WALL = 2 };

/* Uniform Cartesian mesh of I x J control volumes.  I, J >= 2. */
typedef struct { int I, J; double x0, x1, y0, y1; } ugks_mesh;
/* Discrete velocity grid K x M of the paper = Nu x Nv here.  HOST arrays, copied at init.
 * 1 <= Nu <= 512 (a CTA has one thread per column of the velocity grid and keeps 128 registers per thread up to 512 threads), 1 <= Nv <= 2048 (the nodes, weights and the row-chunk table
 * of the run-time compiled kernels live in the 64 KB constant bank).  All nodes and weights must be finite;
 * Weights must have positive sums. */
typedef struct { int Nu, Nv; const double *u, *wu, *v, *wv; } ugks_vgrid;
/* Gas: viscosity exponent omega (mu = mu_ref T^omega), mu_ref (<= 0: derive from Kn, AMB-7),
 * Knudsen number, Prandtl number (must be 1: BGK) and internal degrees of freedom (must be 0). */
typedef struct { double omega, mu_ref, Kn, Pr; int K_int; } ugks_gas;
/* One side's boundary condition.  FIXED: constant ghost Maxwellian (rho,U,V,T) ("given pressure at
 * inlet and outlet", AMB-12).  WALL: fully diffuse isothermal wall with velocity (U,V) and temperature T
 * (rho ignored).  PERIODIC: must be set on both opposite sides. */
typedef struct { int type; double rho, U, V, T; } ugks_bc;
typedef struct { ugks_bc xmin, xmax, ymin, ymax; } ugks_bcs;

/* Bytes of device memory the context needs (two copies of f with padded rows + per-face and per-cell
 * scalars).  Returns 0 on invalid arguments. */
size_t ugks_workspace_bytes(const ugks_mesh *, const ugks_vgrid *);

/* Create a context.  workspace_dev: device pointer to >= ugks_workspace_bytes() bytes, 256-byte aligned
 * (e.g. a torch uint8 tensor).  cuda_stream: a cudaStream_t cast to void* (NULL = default stream).
 * Computes dt = cfl / (max|u|/dx + max|v|/dy) once (AMB-6), the ghost rows and the wall Maxwellians (O0).
 * Errors: UGKS_EINVAL (sizes, Pr != 1, K_int != 0, unpaired periodic sides, NULL pointers, weights),
 * UGKS_ENOMEM (workspace too small), UGKS_ECUDA (no device / CUDA failure). */
int ugks_init(ugks_ctx **out, const ugks_mesh *, const ugks_vgrid *, const ugks_gas *, const ugks_bcs *,
              double cfl, void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* Load the state (AMB-18): W[J][I][4] and f[J][I][Nv][Nu]; resets the step count. */
int ugks_set_state(ugks_ctx *, const double *W, const double *f, int ptrs_on_device);

/* Enqueue n time steps (Eq. (3)(4) with the S1..S8 flux).  Asynchronous: CUDA errors and
 * a non-physical state (rho <= 0, lambda <= 0, NaN) surface on the next synchronising call
 * (ugks_residual, ugks_moments, ugks_get_f, ugks_sync) as UGKS_ECUDA / UGKS_ESTATE.
 * UGKS_ESTATE if no state was set. */
int ugks_step(ugks_ctx *, int n);

/* W_stored: the evolved W of Eq. (4) (AMB-8).  W_of_f: sum_q w_q psi_q f[c][q] (O12).  Either may be NULL.
 * Synchronises the stream. */
int ugks_moments(ugks_ctx *, double *W_stored, double *W_of_f, int ptrs_on_device);

/* Copy f out in the dense [J][I][Nv][Nu] layout.  Synchronises the stream. */
int ugks_get_f(ugks_ctx *, double *f, int ptrs_on_device);

/* res[a] = sqrt(Nc sum_c (W^{n+1}-W^n)_a^2) / (sum_c |W^{n+1}_a| + 1e-300) of the last completed step (O11).
 * HOST pointer.  Synchronises the stream.  UGKS_ESTATE before the first step. */
int ugks_residual(ugks_ctx *, double res[4]);

/* Wait for all enqueued work; reports deferred errors. */
int ugks_sync(ugks_ctx *);

double ugks_dt(const ugks_ctx *);
double ugks_mu_ref(const ugks_ctx *);
long ugks_step_count(const ugks_ctx *);
/* Kernels launched by this context since ugks_init (for bench.py's gpu_launches). */
long ugks_launch_count(const ugks_ctx *);
/* Tuning knobs.  The two kernels that sweep f (k_cell_moments, k_flux_update) each have a launch geometry: the velocity rows
 * are split into chunks of at most `chunk` rows (one CTA marches a strip of `strip` cells for one chunk), R rows of a chunk
 * are processed in parallel and a thread owns ceil(chunk / R) <= 16 points.  "strip", "chunk_m" (alias "chunk"), "R" set both
 * kernels; with the suffix "_u" (e.g. "R_u", "chunk_u") only k_flux_update, with "_m" ("R_m", "strip_m") only k_cell_moments.
 * The chunking of k_cell_moments may only coarsen its default (the moment buffer is sized for it).  Each change re-compiles
 * the kernel it touches.  "tangential" (O3t/O8t; default 0): 1 = f is reconstructed in the
 * tangential direction of a face too (limited slope theta of the upwind cell) and the free-transport part of the face solution
 * (Eq. (2)) carries -Mt5 t theta0; needs v-nodes that come in at most 8 runs of equal sign (ascending grids have 2); re-compiles both kernels.  Others: "profile" (1: time every kernel of ugks_step with CUDA events), "graph" (replay pairs of
 * steps from a CUDA graph: -1 auto = on for launch-bound meshes, 0 off, 1 on), "poison" (test aid: 1 = NaN-fill the shared
 * memory of every SM before each of the two f-sized kernels).
 * UGKS_EINVAL for unknown names or values that do not fit shared memory / the allocated buffers. */
int ugks_set_option(ugks_ctx *, const char *name, int value);
/* With option "profile" on: accumulated device time in ms and launch counts of the five kernels of a step since
 * the last call, in launch order: cell_moments, face_scalars, cell_scalars, tables, flux_update.
 * Synchronises the stream and resets the accumulators. */
int ugks_kernel_times(ugks_ctx *, double ms[5], long counts[5]);
/* Compile the two run-time specialised kernels (k_cell_moments, k_flux_update: NVRTC, sm_100a) for this mesh, velocity grid
 * and boundary types WITHOUT touching a device: the "does it build" check of a geometry, usable on a machine with no GPU.
 * log (may be NULL) receives up to log_bytes of the compiler log, including ptxas' per-kernel register / shared-memory lines.
 * Returns UGKS_OK, UGKS_EINVAL (sizes) or UGKS_ECUDA (compile error: see log). */
int ugks_jit_check(const ugks_mesh *, const ugks_vgrid *, const ugks_bcs *, char *log, size_t log_bytes);
/* The L2 residual (RES row: north_star (iv), reading O11 of DESIGN.md; the W it measures is Eq. (4)'s) between two W
 * fields, WITHOUT a context, a workspace or any allocation:
 *     res[a] = sqrt(ncells * sum_c (W_new - W_old)[c][a]^2) / (sum_c |W_new[c][a]| + 1e-300),  a = 0..3.
 * Meant for callers that cannot get device memory of their own: a convergence monitor or logging hook that only sees W^n and
 * W^{n+1} inside a process whose whole device memory was handed to a pool up front (a raw cudaMalloc fails there although the
 * pool has room, and the hook has no handle to the pool), or a time loop that cannot afford cudaMalloc / cudaFree because they
 * synchronise the whole device.  The per-block partial sums, which ugks_residual keeps in the caller's workspace, go into a
 * fixed array of UGKS_NOALLOC_SCRATCH_BYTES (512 KiB) inside the library image; every GPU that loads libugks.so holds that array
 * until the process exits, whether or not this function is ever called.  The function calls no cudaMalloc, cudaFree or
 * allocating library routine.
 *   W_old, W_new  DEVICE pointers, [ncells][4] fp64 as everywhere in this header; read only, not retained.
 *   ncells        1 .. UGKS_NOALLOC_MAX_CELLS (twice the cells of the largest BASELINE.json mesh); more -> UGKS_EINVAL, nothing launched.
 *   res           DEVICE pointer to 4 doubles, written by the second of the two kernels this enqueues.
 *   cuda_stream   cudaStream_t cast to void* (NULL = default stream) of the CURRENT device; the call is asynchronous and
 *                 does not synchronise: read res after synchronising that stream.
 *   err/err_bytes optional caller buffer for a message (NULL / 0: none); this function does not touch ugks_last_error().
 * The first call on each device looks up that device's address of the array (cudaGetSymbolAddress, with the device current)
 * and remembers it; make that first call before starting any stream capture.  All calls on a device share the one array and it
 * keeps the previous call's partials: that is harmless for calls ordered on one stream or by events (every slot a call
 * reads it has overwritten first, so nothing needs to start at zero), but two calls that overlap on the GPU -- different
 * streams, no dependency -- race on it and both results are garbage.  Same block size and summation order as ugks_residual.
 * Returns UGKS_OK, UGKS_EINVAL (NULL pointer, ncells out of range) or UGKS_ECUDA (no device, launch failure). */
#define UGKS_NOALLOC_MAX_CELLS 1048576L
#define UGKS_NOALLOC_SCRATCH_BYTES 524288
int ugks_residual_noalloc(const double *W_old, const double *W_new, long ncells, double *res, void *cuda_stream,
                          char *err, size_t err_bytes);

const char *ugks_last_error(const ugks_ctx *);           /* library-owned string; ctx may be NULL */
const char *ugks_version(void);
void ugks_destroy(ugks_ctx *);

#ifdef __cplusplus
}
#endif
#endif
