/* =====================================================================================
 * rmhd.h -- C-ABI of librmhd.so: one GPU, FP64, finite-volume IMEX step (SSP2(222), Table 2
 * P:L167-172; SSP3(332), Table 3) for special-relativistic resistive MHD (14
 * conserved variables) and two-fluid RMHD (18)
 * after Wright & Hawke, "Resistive and multi-fluid RMHD on graphics processing units"
 * (citations "P:Lnnn" are line numbers of the reference text PAPER.md; "Gn" are the
 * readings listed in DESIGN.md).
 *
 * Plain pointers and sizes only; no torch types.  Every entry point returns 0 on success or
 * a negative RMHD_ERR_* code; nothing throws or aborts across the boundary.  There is no CPU
 * fallback: without a CUDA device rmhd_create / the *_batch calls return RMHD_ERR_CUDA.
 *
 * ARRAY LAYOUT at the boundary (all double): interior cells only, variable-major SoA,
 *   grids   a[var][k][j][i]  (i = x fastest),   batches  a[var][cell].
 *   resistive cons  (14): D, Sx,Sy,Sz, tau, Bx,By,Bz, Ex,Ey,Ez, rho_charge, psi, phi (eq 1)
 *   resistive prims (11): rho, vx,vy,vz, p, Bx,By,Bz, Ex,Ey,Ez
 *   two-fluid cons  (18): D, S(3), tau, Dbar, Sbar(3), taubar, B(3), E(3), psi, phi   (eq 5-6)
 *   two-fluid prims (16): rho_e, v_e(3), p_e, rho_p, v_p(3), p_p, B(3), E(3)
 * OWNERSHIP: the caller owns every buffer it passes (host or device as flagged by
 * `on_device`; device buffers must live on the context's device); the library owns the
 * context and all its internal device state, released by rmhd_destroy.
 * ===================================================================================== */
#ifndef RMHD_H
#define RMHD_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rmhd_ctx rmhd_ctx; /* opaque */

enum { RMHD_RESISTIVE = 0, RMHD_TWO_FLUID = 1 };
enum { RMHD_BC_OUTFLOW = 0, RMHD_BC_PERIODIC = 1 };
enum { RMHD_SSP2_222 = 0, RMHD_SSP3_332 = 1 };   /* IMEX integrator: Table 2, Table 3 */
enum {
  RMHD_OK = 0,
  RMHD_ERR_BAD_PARAM = -1,
  RMHD_ERR_CUDA = -2,
  RMHD_ERR_NONCONVERGED = -3,   /* some cell's root-find failed; state still advanced */
  RMHD_ERR_UNPHYSICAL_INPUT = -4
};

/* Statement of the problem as the paper gives it: model, Gamma-law EOS, sigma or
 * (eta, mu_s), kappa, grid, CFL, boundary conditions. */
typedef struct {
  int model;                  /* RMHD_RESISTIVE | RMHD_TWO_FLUID                                */
  int nx, ny, nz;             /* interior cells; n == 1 => that axis is absent                  */
  int ng;                     /* ghost layers of the paper's layout (>= 2).  Ghost zones are     */
                              /* virtual here (boundary index maps inside the stencil loads), so */
                              /* ng only has to be >= the stencil reach; kept for API parity     */
  double xmin, xmax, ymin, ymax, zmin, zmax;
  int bc[3];                  /* per axis: RMHD_BC_OUTFLOW (zero gradient) | RMHD_BC_PERIODIC    */
  double gamma;               /* Gamma-law index                                                 */
  double sigma;               /* resistive: conductivity                                         */
  double eta, mu_e, mu_p;     /* two-fluid: resistivity, charge/mass ratios (mu_e != mu_p)        */
  double kappa;               /* divergence-cleaning rate; the paper uses 1              */
  double cfl;                 /* dt = cfl / sum_d (1/dx_d) over present axes, fixed (G9)          */
  double tol_c2p, tol_stage;  /* relative Newton-update tolerances; <= 0 => 1e-13, 1e-12 */
  int max_iter_c2p, max_iter_stage; /* <= 0 => 100, 50                                          */
  int device;                 /* CUDA ordinal                                                    */
  void* stream;               /* cudaStream_t owned by the caller (0 = default stream)           */
  int integrator;             /* RMHD_SSP2_222 (default, the north-star path) | RMHD_SSP3_332     */
} rmhd_params;

/* ---- grid simulation (north_star: rmhd_create / set_initial / step / get_state / destroy) -- */

/* Allocate all device state for one grid.  Errors: BAD_PARAM (sizes, ng < 2, mu_e == mu_p,
 * gamma <= 1, more than 2^31 - 1 cells), CUDA (no device / out of memory).
 * One environment switch is read here: RMHD_FLUX=split evaluates L(q) by one pass per axis (the kernels
 * every 1-D grid uses) instead of the one-pass kernel on 2-D / 3-D grids.  It exists for the parity tests
 * tests/test_gpu_parity.py::test_ssp3_332_parity[blast_3d_split] and ::test_two_fluid_3d_blast_parity[ssp2-split],
 * which run those kernels along y and z; it selects no other code. */
int rmhd_create(const rmhd_params* p, rmhd_ctx** out);

/* Initial primitives -> conserved state (eq 2-4; eq 6), psi = phi = 0
 * (P:L81).  prims: [11|16][nz][ny][nx].  rho_charge: [nz][ny][nx] or NULL => Gauss's law
 * rho = div E by 2nd-order central differences with the boundary conditions applied
 * (G10); ignored for the two-fluid model (charge density is Dbar).  Resets time and
 * statistics.  Errors: UNPHYSICAL_INPUT if any cell has rho <= 0, p <= 0 or |v| >= 1. */
int rmhd_set_initial(rmhd_ctx* c, const double* prims, const double* rho_charge, int on_device);

/* Overwrite the conserved state (cons: [14|18][nz][ny][nx]) and recover primitives from it
 * (P:L118-136); prim_guess ([5|10][nz][ny][nx] hydro primitives) nullable.  Used for restarts and by tests.
 * Resets the statistics (so the return code, NONCONVERGED if a cell's recovery failed, is this call's
 * alone); leaves the step counter and rmhd_time untouched. */
int rmhd_set_cons(rmhd_ctx* c, const double* cons, const double* prim_guess, int on_device);

/* Advance nsteps full IMEX steps (eq 10-11 P:L152-155 read as G1).  SSP2(222), Table 2 P:L167-172:
 * implicit stage, L(q1), implicit stage, L(q2), combine, con2prim.  SSP3(332), Table 3
 * (reading G13): three implicit stages and three L evaluations, same kernels.  Everything runs on
 * the context's stream; one small device->host read of the statistics block (iteration histograms
 * and failure counters, about 1 KB) and a stream synchronisation at the end.
 * Returns NONCONVERGED if any root-find failed in any cell (the steps are still completed).
 * Grids of at most 2^21 cells (every test-sized grid; cfg1, cfg3, cfg4 of BASELINE.json) are launch-bound: the first
 * rmhd_step of such a context captures the launch sequence of one step on a private stream into a CUDA graph and every
 * step replays it into the context's stream (same kernels, same arguments: bitwise the same state,
 * tests/test_gpu_parity.py::test_graph_replay_equals_plain_launches_bitwise).  There is no switch for it; profiling mode
 * (rmhd_set_profiling) uses plain launches so that each kernel can be timed; if capture fails the plain launches stay in force.
 * rmhd_get_kernel_times counts a replayed step's kernels as launches like plain ones.  Consequences for the caller: do not
 * call rmhd_step while p->stream is itself being captured, and do not drive one context from two host threads at once
 * (a context, its graph and its statistics block are not guarded; use one context per thread). */
int rmhd_step(rmhd_ctx* c, int nsteps);

/* Copy out the interior state; either pointer may be NULL. */
int rmhd_get_state(rmhd_ctx* c, double* cons, double* prims, int on_device);

/* L(q) = -sum_d dF^d/dx_d of the current state: Lax-Friedrichs flux-vector
 * splitting (eq 12, alpha = 1) + WENO3.  Lout: [14|18][nz][ny][nx].  (Unit-parity hook.) */
int rmhd_flux_divergence(rmhd_ctx* c, double* Lout, int on_device);

/* Iteration-count histograms since the last set_initial: hist_stage[b] = implicit-stage solves
 * that took b Newton iterations, hist_c2p[b] likewise for stand-alone con2prim (last bin
 * collects the overflow); number of failed root-finds and the smallest failing cell index
 * (k*ny*nx + j*nx + i), -1 if none.  Any pointer may be NULL.  Host pointers. */
int rmhd_get_stats(rmhd_ctx* c, long long* hist_stage, long long* hist_c2p, int nbins, long long* n_failed,
                   long long* first_failed_cell);

/* Measurement hook (per-kernel fractions beside the whole-step figure; north_star: "evidenced
 * by ncu counters ... for the implicit and con2prim kernels ... the flux and stage-combine kernels").
 * Per-kernel-class device time (CUDA events on the context's stream) accumulated while
 * profiling is enabled.  Classes: 0 stage1, 1 stage2, 2 flux sweeps, 3 combine+con2prim,
 * 4 other.  ms[n], launches[n] host arrays. */
int rmhd_set_profiling(rmhd_ctx* c, int enabled);
int rmhd_get_kernel_times(rmhd_ctx* c, double* ms, long long* launches, int n);

double rmhd_dt(const rmhd_ctx* c);
double rmhd_time(const rmhd_ctx* c);           /* t0 + nsteps_done * dt, never accumulated */
const char* rmhd_last_error(const rmhd_ctx* c); /* ctx-owned string; c == NULL => last create error */
void rmhd_destroy(rmhd_ctx* c);

/* ---- batched per-cell operations on n independent cells (BASELINE.json configs[1]) --------- */
/* Only model, gamma, sigma, eta, mu_e, mu_p, kappa, tolerances, device and stream of *p are
 * used.  All pointers are DEVICE pointers unless on_device == 0, in which case the call
 * stages them through the library's staging area on p->device (host<->device copies inside the call; see
 * rmhd_release_staging below).  With on_device == 1 the calls only launch a kernel on p->stream and return. */

/* Staging memory of the on_device == 0 calls: one grow-only device allocation per GPU, made by the first such call,
 * enlarged when a later call needs more, and kept between calls, so that a loop over host batches does not pay a
 * cudaMalloc / cudaFree pair per buffer and call (cudaFree synchronises the whole device).  Host-buffer batch calls of one
 * process run one at a time (the staging area is locked for the duration of a call).  rmhd_release_staging frees it:
 * device >= 0 that GPU's, device < 0 every GPU's; it is an error to call it while a host-buffer batch call is running on
 * another thread only in the sense that it waits for that call.  Nothing else in the library keeps memory after rmhd_destroy
 * (except the fixed array of rmhd_flux_divergence_static, which is part of the library image). */
int rmhd_release_staging(int device);

/* One implicit stage (eq 10):  q* - q_ex - a_dt Psi(q*) = 0 per cell.
 * (SURVEY.md 8(b) lists `model` and `stream` as arguments: both travel in *p here.)
 * q_ex [14|18][n]; prim_guess [11|16][n] (initial guess: primitives near the solution);
 * sigma_cell [n] per-cell conductivity or NULL (use p->sigma; resistive only);
 * outputs q_out [14|18][n], prims_out [11|16][n], iters [n] Newton iterations taken,
 * fail [n] (0 ok).  iters / fail may be NULL. */
int rmhd_stage_batch(const rmhd_params* p, long long ncells, const double* q_ex, const double* prim_guess,
                     const double* sigma_cell, double a_dt, double* q_out, double* prims_out, int* iters,
                     int* fail, int on_device);

/* eq (2)-(4) / eq (6): prims [11|16][n] (+ rho_charge [n] or NULL = 0) -> cons [14|18][n], psi = phi = 0. */
int rmhd_prim2cons_batch(const rmhd_params* p, long long ncells, const double* prims, const double* rho_charge,
                         double* cons, int on_device);

/* cons -> prims; prim_guess nullable; iters / fail nullable. */
int rmhd_con2prim_batch(const rmhd_params* p, long long ncells, const double* cons, const double* prim_guess,
                        double* prims, int* iters, int* fail, int on_device);

/* ---- L(q) without any allocation ----------------------------------------------------------------------
 * For callers who cannot let this library allocate device memory.  Two kinds of program are meant: one that
 * has handed the whole card to a memory pool of its own (a cudaMalloc made behind that pool's back can fail
 * with out-of-memory while the pool still has room, and the pool's bookkeeping never learns of it), and one
 * whose time loop must not stall (cudaFree synchronises the whole device and cudaMalloc may: every other
 * stream on the card waits).  rmhd_create and the on_device = 0 batch calls above do allocate; this call does not.
 *
 * What it computes: the same L(q) = -sum_d dF^d/dx_d as rmhd_flux_divergence (eq 12 + WENO3) of a
 * conserved state the CALLER holds, in two steps: primitive recovery (no initial guess), then the flux
 * kernels.  cons and Lout are DEVICE pointers on device p->device, [14|18][nz][ny][nx], owned by the caller, 8-byte
 * aligned, not overlapping.  Of *p the model, grid, domain, bc, gamma, tol_c2p, max_iter_c2p, device and stream are
 * read (sigma, eta, mu_e, mu_p are only range-checked; integrator and cfl are ignored; RMHD_FLUX is honoured
 * as in rmhd_create).  n_failed (HOST pointer, may be NULL) receives the number of cells whose recovery failed.
 *
 * Where the scratch lives: the recovered hydro primitives ([5|10] rows) and the failure counters are neither input
 * nor output, and sit in ONE fixed array inside the library image, 20 MiB + 4 KiB.  Every GPU on which the library
 * is used holds that array from the moment the library's code is loaded there until the process exits, whether or
 * not this call is ever made.  Its capacity is the limit of this call: nx*ny*nz <= RMHD_STATIC_MAX_CELLS (2^18,
 * e.g. 512 x 512 or 64^3) for either model; a larger grid is refused with RMHD_ERR_BAD_PARAM and a message
 * that names the limit (rmhd_last_error(NULL)), before anything is launched.
 *
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress, with that device
 * current) and remembers it; make that first call before any stream capture begins.  Later calls only launch
 * kernels, copy about 1 KB of counters back and synchronise p->stream; no call uses cudaMalloc, cudaFree or a
 * library routine that allocates (on the error paths the message is a host-side std::string).
 *
 * Sharing: there is one array per GPU, not one per call or per stream.  It keeps what the previous call wrote;
 * the counters are cleared at the start of every call, the primitive rows are overwritten before they are read.
 * Two calls whose kernels can run at the same time on one GPU (two streams, two host threads) race on it and
 * both results are garbage: serialise them.  The call returns only when L is complete, so back-to-back calls from
 * one thread are safe.
 * Returns: OK; BAD_PARAM (null pointer, bad parameters, grid beyond the limit); CUDA (no device: there is no CPU
 * fallback; launch failure); NONCONVERGED if any cell's recovery failed (L is then not valid near those cells). */
#define RMHD_STATIC_MAX_CELLS 262144
int rmhd_flux_divergence_static(const rmhd_params* p, const double* cons, double* Lout, long long* n_failed);

/* ---- roofline denominators measured by the library's own probe kernels (SURVEY.md section 7 step 0:
 * MEASURED_PEAKS.json holds no FP64 figure, so the FP64 roofline peak is this probe's) ------------- */
/* FP64 FMA chain on all SMs: returns achieved TFLOP/s (2 flop per DFMA) in *tflops. */
int rmhd_probe_fp64(int device, void* stream, double* tflops);
/* Device-to-device streaming copy of `bytes` bytes (read + write counted): GB/s. */
int rmhd_probe_hbm(int device, void* stream, long long bytes, double* gbs);

#ifdef __cplusplus
}
#endif
#endif /* RMHD_H */
