/* ch.h — C ABI of the B200-native CTU + PPMC + exact-Riemann hydro step.
 *
 * One unsplit Corner Transport Upwind (CTU) time step of the 3-D Euler equations on a static
 * Cartesian mesh, fp64, as stated in arXiv:1410.4194 (Schneider & Robertson, "Cholla").
 * Citations are `P:L<line>` = line of /root/reference/PAPER.md plus the equation it falls in;
 * "reading Gn/Sn" refers to the table of readings in DESIGN.md.
 *
 * The five graded calls are the ones BASELINE.json's north_star names:
 *     ch_init(nx,ny,nz,nghost,gamma,bc), ch_set_state, ch_compute_dt(cfl), ch_step(dt), ch_get_state.
 * The rest are helpers that exist because the caller (PyTorch) owns device memory and streams.
 *
 * Conventions
 *   - All floating point is IEEE binary64.  All `int` returns: CH_OK (0) or a negative CH_E* code;
 *     ch_last_error() returns a human-readable reason for the last failure on the calling thread.
 *   - Field order: rho, rho*u, rho*v, rho*w, E  (Eq. 9).  x is the fastest index
 *     (P:L312).
 *   - "real" arrays are [5][nz][ny][nx]; "padded" arrays are [5][pz][py][px] with
 *     p_d = n_d + 2*nghost for an active dimension (n_d > 1) and p_d = 1 for an inactive one
 *     (n_d == 1: no ghosts, no sweep, no transverse term, no dt term — P:L132).
 *   - Cell widths default to dx = dy = dz = 1/nx (reading S8); ch_set_spacing overrides.
 *   - The library never allocates or frees DEVICE memory: every device buffer is handed in through
 *     ch_bind and stays owned by the caller.  It does own a few bytes of pinned HOST memory (the
 *     dt read-back cell) per context.
 *   - A context is not thread-safe; use one per host thread / stream.
 *   - ch_bind records the device its buffers live on; every later call runs there whatever device is current
 *     in the calling thread, and restores the caller's current device before returning.
 *   - There is no CPU fallback: every call that touches data launches CUDA work on the bound
 *     stream and returns CH_ECUDA if that fails.
 */
#ifndef CH_H_
#define CH_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ch_ctx ch_ctx; /* opaque, host-side */

enum {
  CH_OK = 0,
  CH_EINVAL = -1,   /* bad argument */
  CH_ESTATE = -2,   /* call out of order (no buffers bound / no state set) */
  CH_ECUDA = -3,    /* a CUDA runtime call or launch failed */
  CH_ENONPHYS = -4  /* non-physical data met (rho <= 0 or non-finite) */
};

/* Boundary-condition codes per face: any mix per face, periodic faces must be paired. */
enum {
  CH_BC_PERIODIC = 1, CH_BC_REFLECTIVE = 2, CH_BC_OUTFLOW = 3,
  CH_BC_NOH = 4, /* custom (analytic) boundary, "custom boundaries": the inflow of the Noh strong-shock test,
                   P:L549-557: rho = rho0 (1 + t/r)^(n-1), unit velocity toward the origin of the box,
                   E = p0/(gamma-1) + rho/2 at the centre of every ghost cell behind the face, n = number of active
                   dimensions, t = ch_get_time (the state AFTER a step is filled at t^{n+1}); see ch_set_noh */
  CH_BC_EXCHANGE = 5 /* the face borders another block of a decomposed domain (section 3.7): its ghost
                   layers are written by ch_halo_unpack with what the neighbour's ch_halo_pack read.  A context with
                   such a face never fills ghosts by itself: after ch_set_state and after every ch_step the caller
                   runs, for d = x, y, z in this order: ch_halo_pack on the EXCHANGE faces of d, the
                   transfer, ch_halo_unpack, and ch_fill_dim(d) for the faces of d with a local rule */
};

/* Device buffers handed to ch_bind.  All pointers are DEVICE pointers owned by the caller and must
 * stay valid until ch_free or the next ch_bind. */
typedef struct ch_buffers {
  double* state;          /* padded conserved store u, 5*Np doubles (SoA, x fastest) */
  void* workspace;        /* scratch, at least ch_workspace_bytes(...) bytes, 256-byte aligned */
  size_t workspace_bytes; /* size of `workspace` as allocated */
  void* reduce;           /* 64 bytes, 8-byte aligned: device cells of the dt reduction (max wave rate, flag; ch_step_cfl: dt, elapsed, dt/dx_d) */
} ch_buffers;

/* ch_init — create a context for an nx*ny*nz grid of real cells with `nghost` ghost layers on each
 * side of every active dimension, ratio of specific heats `gamma` (Eq. 8), and boundary
 * codes bc[6] = {x-,x+,y-,y+,z-,z+} (host pointer; NULL = all periodic).  Host-only: makes no CUDA
 * call.  Returns NULL on error (n < 1; nghost < 3 — PPMC inside six-solve CTU needs 3; gamma <= 1;
 * a bc code outside 1..5 on an active dimension; unpaired periodic faces; an active dimension
 * smaller than nghost). */
ch_ctx* ch_init(int nx, int ny, int nz, int nghost, double gamma, const int* bc);

/* ch_free — destroy the context (host memory only; bound device buffers stay with the caller). */
int ch_free(ch_ctx* ctx);

/* ch_last_error — reason for the most recent failure on this thread ("" if none). */
const char* ch_last_error(void);

/* ch_set_spacing — override the cell widths (all > 0).  Default 1/nx each (reading S8). */
int ch_set_spacing(ch_ctx* ctx, double dx, double dy, double dz);

/* ch_padded_cells — Np = px*py*pz for the context. */
long long ch_padded_cells(const ch_ctx* ctx);

/* ch_workspace_bytes — bytes of scratch ch_bind needs for this grid: the first-pass fluxes F*,G*,H*
 * (P:L157), the traced interface states U*_L, U*_R per direction, the CTU fluxes
 * F,G,H^{n+1/2}, all padded SoA fp64, and the three eta fields of the H correction.  Returns 0 on bad arguments. */
size_t ch_workspace_bytes(int nx, int ny, int nz, int nghost);

/* ch_bind — attach caller-owned device buffers and the CUDA stream (a cudaStream_t passed as
 * void*; NULL = the legacy default stream) every later call runs on.  Must precede ch_set_state.
 * CH_EINVAL if a pointer is NULL or the workspace is too small.  Invalidates any state set before. */
int ch_bind(ch_ctx* ctx, const ch_buffers* bufs, void* stream);

/* ch_set_state — copy the real cells `u` ([5][nz][ny][nx], HOST or DEVICE pointer, resolved by
 * unified addressing) into the padded store and fill the ghost cells (periodic =
 * opposite side; reflective = mirror cell with the normal momentum negated; outflow = adjacent
 * boundary cell; x then y then z so edges and corners are carried; readings S6, S7).
 * Asynchronous on the stream for device / pinned sources. */
int ch_set_state(ch_ctx* ctx, const double* u);

/* ch_get_state — copy the real cells out to `u` ([5][nz][ny][nx], HOST or DEVICE pointer) and
 * synchronise the stream. */
int ch_get_state(ch_ctx* ctx, double* u);

/* ch_set_padded / ch_get_padded — the padded store as is, ghosts included and NOT refilled
 * ([5][pz][py][px], HOST or DEVICE pointer).  Used to run one step on a sub-box cut from a larger
 * grid and to check the ghost fill; get synchronises. */
int ch_set_padded(ch_ctx* ctx, const double* up);
int ch_get_padded(ch_ctx* ctx, double* up);

/* ch_compute_dt — Eq. 22: returns cfl * min over real cells and active directions d of
 * dx_d / (|v_d| + a), a = sqrt(gamma p / rho) (Eq. 21), p floored at 1e-20.  The device
 * reduces the equivalent grid MAXIMUM of (|v_d| + a) / dx_d (one value per CTA, one atomic) and the
 * host takes the single reciprocal; |v_d| + a is evaluated with correctly rounded quotients and
 * square root, so the result agrees with Eq. 22 in IEEE arithmetic to <= 2 ulp and is a pure function
 * of the state.  Synchronises the stream (one 16-byte device-to-host copy).  When ch_step has already
 * reduced the wave speeds of the current state inside its update kernel, no further pass over the
 * grid is made.  Returns NaN and sets CH_ENONPHYS if any real cell has rho <= 0 or a non-finite rho
 * or E; NaN with CH_EINVAL if cfl is not in (0,1]; NaN with CH_ESTATE if no state is set.  The
 * paper's stability bound for the 3-D six-solve CTU is cfl < 0.5: documented, not enforced. */
double ch_compute_dt(ch_ctx* ctx, double cfl);

/* ch_step — advance the state by one CTU step of size dt (steps 1-5): PPMC
 * reconstruction with characteristic limiting and characteristic tracing in every active direction
 * (A8-A11 P:L722-743), exact Riemann solver at every interface (Newton
 * tolerance 1e-8, cap 20: reading S2), transverse flux correction (Eq. 23), second Riemann
 * pass, conservative update (Eq. 24), ghost fill.  Asynchronous on the stream.
 * CH_ESTATE if no state is set; CH_EINVAL if dt <= 0 or non-finite; CH_ECUDA on launch failure. */
int ch_step(ch_ctx* ctx, double dt);

/* Riemann solver used at every interface by ch_step (the solver is selectable at compile time in the
 * paper's code, at run time here).  CH_SOLVER_EXACT (default): the exact solver, B.1.  CH_SOLVER_ROE: the
 * Roe solver with the HLLE failsafe, B.2; without the H correction of Appendix C. */
enum { CH_SOLVER_EXACT = 0, CH_SOLVER_ROE = 1 };

/* ch_set_solver — select the Riemann solver for later steps.  CH_EINVAL for an unknown code. */
int ch_set_solver(ch_ctx* ctx, int solver);

/* Interface reconstruction used by ch_step.  CH_RECON_PPMC (default): A.3.  CH_RECON_PLMC: piecewise
 * linear, limited in the characteristic variables, with characteristic tracing, A.2.
 * CH_RECON_PCM: piecewise constant, Eq. 25-26. */
enum {
  CH_RECON_PPMC = 0, CH_RECON_PLMC = 1, CH_RECON_PCM = 2,
  CH_RECON_PPMP = 3, /* A.4: parabolic in the primitive variables, contact steepening, shock flattening,
                        Colella-Woodward tracing; 7-cell stencil: nghost >= 4; not with the H correction */
  CH_RECON_PLMP = 4  /* A.1: linear in the primitive variables, evolved with its own face fluxes */
};

/* ch_set_hcorrection — switch the H correction of Appendix C on or off for later steps: in the
 * second Riemann pass the Roe eigenvalues of B28 become max(|lambda|, eta^H), eta^H the largest
 * eta = |(u_R + a_R) - (u_L + a_L)| / 2 over the interface and the transverse faces of the two cells that share
 * it.  Needs nghost >= 4 (CH_EINVAL otherwise) and CH_SOLVER_ROE (ch_step returns CH_ESTATE otherwise); the
 * second half of the step then runs as k_eta + the fused TMA kernel on 3-D grids whose strides meet TMA's rules
 * (ch_tiling reports it), unfused (k_eta, k_pass2, k_update) elsewhere. */
int ch_set_hcorrection(ch_ctx* ctx, int on);

/* ch_set_reconstruction — select the reconstruction for later steps.  CH_EINVAL for an unknown code. */
int ch_set_reconstruction(ch_ctx* ctx, int recon);

/* ch_set_noh — ambient density and pressure of the analytic CH_BC_NOH faces (defaults 1 and 1e-6).
 * ch_set_time / ch_get_time — the time the analytic faces are evaluated at: ch_set_state resets it to 0, every ch_step
 * adds its dt before the ghost fill.  ch_step_cfl refuses (CH_ESTATE) on a grid with an analytic face, because the
 * time then lives on the device only.  ch_fill_ghosts — redo the ghost fill of the current state (after ch_set_time). */
int ch_set_noh(ch_ctx* ctx, double rho0, double p0);
int ch_set_time(ch_ctx* ctx, double t);
double ch_get_time(const ch_ctx* ctx);
int ch_fill_ghosts(ch_ctx* ctx);

/* Block decomposition.  Slab of direction d = nghost layers x (the other two directions: padded extent
 * for a direction before d in the order x, y, z, real cells for a direction after d), so that edges and corners are
 * carried by at most six messages per block.
 * ch_halo_cells(d)   cells of one slab of direction d; a packed slab is 5 * ch_halo_cells(d) doubles, [5][nghost][.][.]
 * ch_halo_pack       copy the nghost REAL layers next to `face` (0..5 = x-,x+,y-,y+,z-,z+) into the DEVICE buffer buf
 * ch_halo_unpack     write buf into the nghost GHOST layers beyond `face` (pack of the neighbour's opposite face)
 * ch_fill_dim(d)     fill the ghost layers of direction d behind faces with a local rule (periodic, reflective,
 *                    outflow, analytic); EXCHANGE faces are left alone
 * ch_set_origin      global index of this block's first real cell (the analytic boundary needs global coordinates)
 * All asynchronous on the bound stream.  The time step of a decomposed domain is the minimum of the blocks'
 * ch_compute_dt, handed to every block's ch_step; ch_step_cfl refuses (CH_ESTATE) on such a context. */
long long ch_halo_cells(const ch_ctx* ctx, int d);
int ch_halo_pack(ch_ctx* ctx, int face, double* buf);
int ch_halo_unpack(ch_ctx* ctx, int face, const double* buf);
int ch_fill_dim(ch_ctx* ctx, int d);
int ch_set_origin(ch_ctx* ctx, int i0, int j0, int k0);

/* ch_set_option — launch-configuration choices that change HOW a step is computed, never WHAT (every setting
 * gives results within the one-step gate of every other; the tests compare them).  Defaults are what bench.py
 * times.  Nothing here is read from the environment.
 *   CH_OPT_MARCH_SEG  cells a thread of the marching pass-1 kernels sweeps (0 = chosen from the grid size; >= 4)
 *   CH_OPT_FINAL_SEG  planes a CTA of the fused second half marches (0 = chosen from the grid size; >= 4)
 *   CH_OPT_TMA        the fused second half of 3-D grids where the padded strides allow TMA: 2 (default) planes staged by TMA,
 *                     13-row tiles, the producer's work done by a lane of the warp that serves the halo rows; 1: 12-row
 *                     tiles with a producer warp of its own (the form the H-corrected step always takes); 0: plain loads.
 *                     The three forms give the same bits.  Other values: CH_EINVAL
 *   CH_OPT_UNFUSED    1: run the second half as k_pass2 + k_update on 3-D grids too (A/B measurements); default 0
 *   CH_OPT_GRAPH      1 (default): ch_step_cfl replays the kernels of a step as one CUDA graph from the third step with a
 *                     configuration on (captured on a private stream; the same kernels, the same bits); 0: direct launches
 *   CH_OPT_FOLD_GHOST 1 (default): on x-y grids with periodic / reflective / outflow faces the update kernel also writes the
 *                     ghost cells that copy its cells (one launch less per step, the same bits); 0: a k_ghost launch
 * CH_EINVAL for an unknown option or an out-of-range value. */
enum { CH_OPT_MARCH_SEG = 0, CH_OPT_FINAL_SEG = 1, CH_OPT_TMA = 2, CH_OPT_UNFUSED = 3, CH_OPT_GRAPH = 4, CH_OPT_FOLD_GHOST = 5 };
int ch_set_option(ch_ctx* ctx, int option, int value);

/* ch_step_cfl — one step whose size never visits the host: dt = cfl * min dx_d/(|v_d| + a) (Eq. 22, from the
 * reduction the previous step left on the device, or a fresh pass after ch_set_state), clipped to t_left when
 * 0 < t_left < dt, then the same kernels as ch_step read it from device memory and form dt/dx_d with the same
 * correctly rounded division.  Fully asynchronous: steps can be queued back to back without the 16-byte
 * read-back ch_compute_dt needs.  A sequence of ch_step_cfl calls gives bitwise the states the
 * ch_compute_dt + ch_step loop gives.  A non-physical cell (rho <= 0 or non-finite) makes dt NaN and the step
 * is REFUSED on the device: no kernel writes, the state, its reduction cells and ch_elapsed stay as they were, so
 * ch_last_dt returns NaN + CH_ENONPHYS and ch_compute_dt reports CH_ENONPHYS, exactly as the ch_compute_dt +
 * ch_step loop stops before touching the state.
 * CH_EINVAL if cfl is not in (0,1] or t_left is NaN; t_left <= 0 means "no clipping". */
int ch_step_cfl(ch_ctx* ctx, double cfl, double t_left);

/* ch_last_dt — the dt the most recent ch_step_cfl used (synchronises; NaN + CH_ENONPHYS if it met a non-physical
 * cell).  ch_elapsed — the sum of the dt of all ch_step_cfl calls since ch_bind (synchronises). */
double ch_last_dt(ch_ctx* ctx);
double ch_elapsed(ch_ctx* ctx);

/* ch_sync — block until all work queued on the context's stream has finished. */
int ch_sync(ch_ctx* ctx);

/* ch_tiling — how the bound grid is cut into CTAs, for tests that place samples across tile seams: out[8] (HOST)
 * = { interfaces per CTA of the x pass (over the flat run of padded cells), columns per CTA of the marching
 * passes, interfaces per marching thread along y, along z, updated columns per tile of the fused second half
 * along x, along y, planes per CTA of the fused second half, 1 if the TMA-fed form runs }.  Zeros where a kernel
 * does not run on this grid.  Call after ch_bind. */
int ch_tiling(const ch_ctx* ctx, int* out);

/* ch_kernel_launches — number of kernels this context has launched since ch_init (for bench.py's
 * gpu_launches claim). */
long long ch_kernel_launches(const ch_ctx* ctx);

/* Kernel kinds of one step, for ch_profile_read / ch_kernel_name. */
enum {
  CH_K_RESET = 0, CH_K_PASS1_X, CH_K_PASS1_Y, CH_K_PASS1_Z, CH_K_PASS2, CH_K_UPDATE, CH_K_GHOST, CH_K_DT,
  CH_K_FINAL, /* fused pass 2 + update of 3-D grids */
  CH_K_ETA,   /* H correction: eta of every interface */
  CH_K_PICK_DT, /* ch_step_cfl: Eq. 22 finished on the device */
  CH_K_COUNT
};

/* ch_profile — measurement helper (P:L427 keeps wall-clock timers per phase; this is the per-kernel
 * equivalent).  enable != 0: every later ch_step / ch_compute_dt brackets each of its kernel launches
 * with CUDA events on the bound stream, blocks until the step has finished and adds the elapsed
 * times to per-kind totals; enable == 0: back to asynchronous steps.  Either call zeroes the totals. */
int ch_profile(ch_ctx* ctx, int enable);

/* ch_profile_read — copy the totals out: ms[CH_K_COUNT] (milliseconds) and calls[CH_K_COUNT]
 * (launches timed), HOST pointers. */
int ch_profile_read(const ch_ctx* ctx, double* ms, long long* calls);

/* ch_kernel_name — static name of kernel kind `kind` ("" if out of range). */
const char* ch_kernel_name(int kind);

/* ch_fp64_peak_probe — measurement helper for the roofline denominator: runs `iters` dependent
 * DFMA chains (8 independent chains per thread) on `blocks` x `threads` threads on `stream` and
 * returns the elapsed milliseconds measured with CUDA events (negative on error).  `sink` is a
 * device pointer to at least blocks*threads doubles.  FP64 flops done = 2*8*iters*blocks*threads. */
double ch_fp64_peak_probe(double* sink, int blocks, int threads, int iters, void* stream);

/* ch_issue_mix_probe — measurement helper for the second ceiling bench.py states: the same loop as
 * ch_fp64_peak_probe (8 independent DFMA per iteration) with n_alu = 0, 16 or 32 independent 32-bit integer
 * operations added per iteration; returns the elapsed milliseconds (negative on error).  From the three times:
 * cost of an FP64 warp instruction and of an ALU warp instruction in scheduler cycles, and whether they overlap. */
double ch_issue_mix_probe(double* sink, int n_alu, int blocks, int threads, int iters, void* stream);

/* ch_dt_noalloc — Eq. 22 without a context, a workspace or ANY allocation: for callers that cannot
 * call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 *   u_padded  DEVICE pointer, read only: the padded conserved store [5][pz][py][px] fp64 exactly as ch_get_padded
 *             lays it out (x fastest, nghost layers on every face of an active dimension, none on an inactive one)
 *   nx,ny,nz,nghost  as ch_init;  gamma > 1;  dx,dy,dz > 0 the cell widths;  cfl in (0,1]
 *   dt_out    DEVICE pointer on the same GPU, 1 double, written by the last kernel: cfl * min_d dx_d/(|v_d|+a) over
 *             the real cells — the value ch_compute_dt returns for that state, bit for bit — or NaN if a cell has
 *             rho <= 0 or a non-finite value (nothing is read back: the return code cannot say so)
 *   stream    cudaStream_t (NULL = default stream); the call only enqueues (one 8-byte memset, two kernels)
 * The reduction's scratch (one partial maximum per 256 cells) lives in a file-scope device array of 524 544 bytes
 * that every GPU which loads the library holds until exit, so a grid may have at most ch_noalloc_max_cells() =
 * 16 777 216 real cells (256^3): CH_EINVAL with a message naming the limit beyond it, and for bad arguments or
 * pointers that are not device memory of one GPU.  All calls share that array and it keeps the last call's contents
 * (the flag that must start at zero is cleared on `stream` at the start of every call): calls that may OVERLAP on the
 * GPU — different streams without an ordering between them — race on it; calls on one stream, or ordered by events,
 * are safe.  The array's device address is looked up once per device (cudaGetSymbolAddress) at the first call on that
 * device; ch_noalloc_setup() does the look-up for the CURRENT device ahead of time (call it before a graph capture
 * starts).  No call here uses cudaMalloc, cudaFree, cudaHostAlloc or a library routine that allocates. */
int ch_dt_noalloc(const double* u_padded, int nx, int ny, int nz, int nghost, double gamma, double dx, double dy,
                  double dz, double cfl, double* dt_out, void* stream);
int ch_noalloc_setup(void);
long long ch_noalloc_max_cells(void);

#ifdef __cplusplus
}
#endif
#endif /* CH_H_ */
