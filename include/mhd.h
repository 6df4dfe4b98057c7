/*
 * include/mhd.h -- C ABI of libmhd.so: the fp64 Van Leer + Constrained Transport (VL+CT)
 * ideal-MHD time step of Cholla-MHD (arxiv 2402.05240) as hand-written CUDA for sm_100a.
 *
 * Citations are to /root/reference/PAPER.md (line numbers) and to the readings O0..O12 /
 * G1..G24 restated in DESIGN.md.
 *
 * Conventions
 *   - One global context per process (one GPU, no MPI: BASELINE.json north_star).
 *   - Unit box, Delta_a = 1/n_a.  Cells (i,j,k), i fastest.
 *   - State = 8 fp64 SoA fields: rho, mx, my, mz, E at cell centres,
 *     nx*ny*nz values each, index i + nx*(j + ny*k);  bx on x-faces, (nx+1)*ny*nz values,
 *     index i + (nx+1)*(j + ny*k); by nx*(ny+1)*nz; bz nx*ny*(nz+1).  Face index f is the
 *     LOWER face of cell f (position f-1/2; Eq. 20 indexing B_{x,i-1/2}).
 *   - "host" pointers are ordinary CPU memory (pageable or pinned), "device" pointers are
 *     CUDA device memory of the current device.  The caller owns every buffer it passes;
 *     the library owns its internal device arrays (or the workspace handed to
 *     mhd_init_workspace, which the caller must keep alive until mhd_finalize).
 *   - All kernels are launched on the library's stream (default: the legacy default stream;
 *     change with mhd_set_stream).  Calls are asynchronous on that stream unless stated.
 *   - Every function returns MHD_OK (0) or a negative MHD_ERR_* code; nothing throws or
 *     aborts across the ABI.  mhd_last_error() gives a static human-readable string.
 *   - No floors or fix-ups are applied to the state (the paper describes none, G18).  A
 *     non-physical state (rho <= 0, P <= 0 or non-finite) seen by the CFL kernel makes
 *     mhd_compute_dt return MHD_ERR_UNPHYSICAL.
 */
#ifndef MHD_H_
#define MHD_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MHD_OK 0
#define MHD_ERR_ARG (-1)        /* bad argument */
#define MHD_ERR_NOT_INIT (-2)   /* mhd_init has not been called */
#define MHD_ERR_NOMEM (-3)      /* device allocation failed / workspace too small */
#define MHD_ERR_CUDA (-4)       /* a CUDA call failed; see mhd_last_error() */
#define MHD_ERR_UNPHYSICAL (-5) /* rho <= 0, P <= 0 or non-finite value in the state */

#define MHD_RECON_PCM 0  /* Eq. 14, PAPER.md:139-147 (debug: first order everywhere) */
#define MHD_RECON_PLMC 1 /* Eq. 23-28 */
#define MHD_RECON_PPMC 2 /* PAPER.md:231, 431; reading O10 */
#define MHD_RECON_PLMP 3 /* PLM limited in the primitive variables */
#define MHD_RECON_PPMP 4 /* PPM limited in the primitive variables */

#define MHD_BC_PERIODIC 0
#define MHD_BC_OUTFLOW 1 /* zero-gradient copy of the nearest active cell/face (O12) */

/* Number of bytes of device memory the context for an nx*ny*nz grid with this
 * reconstruction needs (state, half-step state, face fluxes, edge fields, scratch).
 * Returns 0 on bad arguments. */
size_t mhd_workspace_bytes(int nx, int ny, int nz, int recon);

/* Create the context (the nine-step VL+CT list): nx*ny*nz cells on the unit
 * box, adiabatic index gamma > 1, recon one of MHD_RECON_*.  All axes periodic
 * until mhd_set_boundary says otherwise.  Device memory is obtained with cudaMalloc.
 * A previous context is destroyed first.
 * Developer switch: if the environment variable MHD_STAGE_TY is "0" when the context is created,
 * the predictor stage (steps 2-5 of the list) runs as three kernels through the flux arrays instead
 * of the single fused kernel (same arithmetic, results equal to rounding; slower). */
int mhd_init(int nx, int ny, int nz, double gamma, int recon);

/* Same, but all device arrays are carved out of `workspace` (a DEVICE pointer, 256-byte
 * aligned, at least mhd_workspace_bytes() long, e.g. a torch tensor's data_ptr()).  The
 * library never frees it. */
int mhd_init_workspace(int nx, int ny, int nz, double gamma, int recon, void *workspace,
                       size_t workspace_bytes);

/* axis 0/1/2 = x/y/z; kind MHD_BC_*.  Takes effect at the next boundary update (the next
 * mhd_set_state* or mhd_step). */
int mhd_set_boundary(int axis, int kind);

/* Domain lengths L_x, L_y, L_z > 0 (default 1 x 1 x 1): Delta_a = L_a / n_a.  The paper's non-cubic
 * test boxes keep cubic cells this way (3 x 1.5 x 1.5 at 2N x N x N; 1 x 1 x 2 at
 * N x N x 2N; 1 x 1.5 x 1 at 200 x 300 x 200). */
int mhd_set_domain(double lx, double ly, double lz);

/* cudaStream_t (as void*) on which all later work is launched; NULL = default stream. */
int mhd_set_stream(void *cuda_stream);

/* Copy a full state in from 8 HOST arrays (layout above) and fill the ghost layers.
 * Synchronous with respect to the host buffers (they may be reused on return). */
int mhd_set_state(const double *rho, const double *mx, const double *my, const double *mz,
                  const double *E, const double *bx, const double *by, const double *bz);

/* Same with 8 DEVICE arrays; asynchronous on the library stream. */
int mhd_set_state_device(const double *rho, const double *mx, const double *my,
                         const double *mz, const double *E, const double *bx,
                         const double *by, const double *bz);

/* Eq. 11-12: dt = cfl * min over cells and directions of
 * Delta_a / (|v_a| + c_f,a), by a warp-shuffle + block + atomic-min reduction
 * (PAPER.md:317-327).  Synchronous: *dt (HOST pointer) is valid on return. */
int mhd_compute_dt(double cfl, double *dt);

/* One full VL+CT step of size dt (steps 2-9): boundary update, PCM+HLLD
 * predictor fluxes, CT edge fields, half update, high-order reconstruction + HLLD, CT edge
 * fields, full update.  Asynchronous on the library stream. */
int mhd_step(double dt);

/* n_steps times { dt = cfl * CFL minimum on the device; full step with that dt } without
 * any host synchronisation; the dt of each step stays on the device.  If t_accum is
 * non-NULL (HOST pointer) the call synchronises and stores the sum of the dt taken. */
int mhd_advance(int n_steps, double cfl, double *t_accum);

/* Copy the state out to 8 HOST arrays (any pointer may be NULL = skip).  Synchronises. */
int mhd_get_state(double *rho, double *mx, double *my, double *mz, double *E, double *bx,
                  double *by, double *bz);

/* Same to 8 DEVICE arrays; asynchronous on the library stream. */
int mhd_get_state_device(double *rho, double *mx, double *my, double *mz, double *E,
                         double *bx, double *by, double *bz);

/* Debug/parity: the predictor's U^{n+1/2} left by the last mhd_step,
 * to HOST arrays.  Synchronises. */
int mhd_get_half_state(double *rho, double *mx, double *my, double *mz, double *E, double *bx,
                       double *by, double *bz);

/* Debug/parity: component comp (0 mass, 1 mom_n, 2 mom_t1, 3 mom_t2, 4 energy, 5 B_t1 flux,
 * 6 B_t2 flux; solver-local axes of reading O0) of the corrector HLLD flux on
 * the LOWER `axis`-face of every active cell, as left by the last mhd_step; nx*ny*nz values to a
 * HOST array.  Synchronises.  Host transfers of every get / set call are staged through a scratch
 * array of the library's own, so the flux arrays, the half-step state and the state may be read in
 * any order after a step.  The momentum and energy fluxes of the z sweep (axis 2, comp 1..4) are
 * applied inside the sweep kernel and never stored: MHD_ERR_ARG. */
int mhd_get_flux(int axis, int comp, double *out);

/* Debug layout check.  With MHD_GUARD=1 in the environment at mhd_workspace_bytes / mhd_init time every
 * array of the context sits between guard bands filled with a NaN pattern and itself starts as that pattern;
 * *n_bad receives the number of guard words that no longer hold it (0 = no kernel has written outside its
 * arrays), or -1 if the context is not guarded.  Synchronous; *n_bad is a HOST pointer. */
int mhd_debug_guard_errors(long long *n_bad);

/* max over active cells of |sum_a (B_a[upper] - B_a[lower]) / Delta_a|.
 * Synchronous; *out is a HOST pointer. */
int mhd_max_divb(double *out);

/* Instrumented variant of { CFL reduction; mhd_step(dt) }: records a CUDA event on the library
 * stream after every kernel launch and returns, for launch i, its duration ms[i] (milliseconds,
 * event to event, so it includes the launch gap) and a static name names[i].  At most
 * max_entries are written; *n_entries receives the count.  Synchronises.  Used by bench.py for
 * the per-kernel roofline; the state advances exactly as with mhd_step. */
int mhd_step_profile(double dt, int max_entries, double *ms, const char **names, int *n_entries);

/* The same for n_steps (1..4096) consecutive steps of mhd_advance (each with its own dt from the CFL
 * reduction), enqueued back to back without synchronisation in between: ms[i] is the
 * duration of launch i of a step averaged over the steps (launch 0 is the dt kernel), i.e. the
 * kernels' durations in the steady state of a long run.  Always the kernel-per-stage path (no CUDA
 * graph, no cooperative small-grid kernel).  Synchronises at the end.  Used by bench.py for the roofline. */
int mhd_advance_profile(int n_steps, double cfl, int max_entries, double *ms, const char **names, int *n_entries);

/* Roofline denominators measured on the current device (not part of the time step): the fp64
 * FMA-pipe peak in TFLOP/s from a kernel of independent DFMA chains (8 per thread, 2048 threads
 * per SM; burst = best of 5 launches if seconds <= 0.5, else the mean over the second half of 40
 * back-to-back launches = sustained clocks) and the HBM copy bandwidth in GB/s (read + write
 * bytes of a 1 GiB copy, best of 5).  Uses the default stream; synchronises. */
int mhd_measure_peaks(double *fp64_tflops, double *copy_gbs, double seconds);

/* Unit-level entry points (tests compare the device arithmetic with the oracle function by
 * function).  All pointers are HOST pointers; the calls are synchronous on the default stream and
 * need no context.  Solver-local 1-D states W = (rho, u, v, w, P, B_t1, B_t2) (reading O0).
 *
 * mhd_unit_hlld: n independent HLLD solves (reading O4): WL, WR are n*7 values,
 * bx n face-normal fields, F receives n*7 flux components (mass, mom_n, mom_t1, mom_t2, energy,
 * B_t1 flux, B_t2 flux). */
int mhd_unit_hlld(int n, double gamma, const double *WL, const double *WR, const double *bx,
                  double *F);

/* n independent reconstructions of one cell: recon = MHD_RECON_PLMC / MHD_RECON_PLMP (Eq. 23-28,
 * PAPER.md:229-263; stencil of 3 states) or MHD_RECON_PPMC / MHD_RECON_PPMP (reading O10; stencil of 5
 * states).  Ws holds n * (stencil) * 7 values (stencil cell fastest after the component), bn0 the n cell-centred
 * normal fields of the middle cell.  Wlo = W_{R,i-1/2}, Whi = W_{L,i+1/2}, n*7 values each. */
int mhd_unit_reconstruct(int n, double gamma, int recon, const double *Ws, const double *bn0,
                         double *Wlo, double *Whi);

/* n independent CT edge fields (Eq. 15-18, reading O6).  in12 holds, per edge,
 * (Ea0, Ea1, Eb0, Eb1, Ma0, Ma1, Mb0, Mb1, Er00, Er10, Er01, Er11) as named in reading O6:
 * face fields on the two a-faces and two b-faces touching the edge, the mass fluxes on those
 * faces, and the reference field of the four cells around the edge. */
int mhd_unit_ct_edge(int n, const double *in12, double *out);

/* The kernels' own fp64 reciprocal (op 0), reciprocal square root (op 1) and square root (op 2)
 * (csrc/mhd_math.cuh: hardware seed + two Newton steps, no slow path) on n HOST values x > 0
 * (op 2 also accepts 0); tests bound their error in ulps against IEEE. */
int mhd_unit_math(int n, int op, const double *x, double *y);

/* Number of kernel launches issued by this library since mhd_init (for bench.py). */
long long mhd_launch_count(void);

/* Block until all work on the library stream is done. */
int mhd_synchronize(void);

/* Free everything.  Safe to call twice. */
int mhd_finalize(void);

/* Static string describing the last error (never NULL). */
const char *mhd_last_error(void);

/* ---- An entry point that allocates nothing (csrc/mhd_noalloc.cu) --------------------------------
 * The diagnostic of mhd_max_divb for callers that cannot call cudaMalloc: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid allocation.  It needs no
 * mhd_init and no context, and calls no cudaMalloc, cudaFree or allocating library routine: the
 * reduction's scratch (one partial maximum per block of 256 cells) is a static __device__ array of
 * MHD_NOALLOC_MAX_PARTIALS doubles (512 KiB), which every GPU that loads the library holds until the
 * process exits.  Grids of more than MHD_NOALLOC_MAX_CELLS cells (256^3) are rejected with
 * MHD_ERR_ARG and a message naming the limit; nothing is launched then.
 *   nx, ny, nz      active cells;  dx, dy, dz = cell sizes (> 0)
 *   d_bx, d_by, d_bz DEVICE pointers, the dense face arrays of the ABI layout above ((nx+1)*ny*nz,
 *                   nx*(ny+1)*nz, nx*ny*(nz+1) doubles, i fastest); read only, owned by the caller
 *   d_out           DEVICE pointer to one double: max over cells of |sum_a (B_a[upper] - B_a[lower]) / Delta_a|
 *   stream          a cudaStream_t (NULL = legacy default stream); two kernels are enqueued on it and the
 *                   call returns without synchronising
 * All calls on one device share the scratch array, which keeps the last call's contents (no part of it
 * has to be zero: a call writes every slot it later reads).  Calls that overlap on the GPU -- different
 * streams with no ordering between them -- race on it; order them.  Errors: MHD_ERR_ARG (sizes,
 * null pointers, too many cells), MHD_ERR_CUDA; text from mhd_noalloc_last_error(). */
#define MHD_NOALLOC_MAX_PARTIALS 65536
#define MHD_NOALLOC_MAX_CELLS (256LL * MHD_NOALLOC_MAX_PARTIALS)
int mhd_max_divb_noalloc(int nx, int ny, int nz, double dx, double dy, double dz, const double *d_bx,
                         const double *d_by, const double *d_bz, double *d_out, void *stream);
const char *mhd_noalloc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MHD_H_ */
