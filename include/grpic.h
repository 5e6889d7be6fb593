/* grpic.h -- C ABI of libgrpic.so: the B200-native (sm_100a) data-parallel hot path of the
 * GRPIC method of arxiv 2503.04558 (Aperture): general-relativistic particle push fused with
 * charge-conserving current deposition on a 2D axisymmetric (log r, theta) Kerr-Schild Yee
 * grid, the GR Maxwell (D,B) field update that consumes that current, and the particle
 * cell-sort / compaction passes around them.
 *
 * Citations are to the paper text (PAPER.md:<line>, section / equation).
 *
 * Conventions
 *  - Every array argument is a CALLER-OWNED DEVICE pointer (cudaMalloc / torch CUDA tensor)
 *    unless it says "host".  The library never frees them and keeps no reference after the
 *    call returns, except the workspace registered with grpic_set_workspace.  The context owns
 *    its metric/area tables and (once grpic_step_host has been used) that call's staging buffers.
 *  - All work is enqueued on the caller's CUDA stream (`void* stream` = cudaStream_t; NULL =
 *    default stream) and is asynchronous; nothing synchronises the device.
 *  - Every call returns 0 on success or a negative grpic error code for argument / state
 *    errors found synchronously on the host (nothing is launched then).  Device-side
 *    anomalies are OR-ed into a caller-provided device word `status` (see GRPIC_STATUS_*).
 *  - No CPU fallback exists: without a CUDA device grpic_create fails with GRPIC_ERR_CUDA.
 *
 * Grid (Fig.1; Appendix B :476-518): nr x nth cells, nodes i=0..nr,
 * j=0..nth, xi = ln r, xi_i = xi_in + i*dxi, theta_j = j*pi/nth.  Staggering, index (i,j) =
 *     D^r, J^r, B^th : (i+1/2, j)     D^th, J^th, B^r : (i, j+1/2)
 *     D^ph, J^ph, rho: (i, j)         B^ph            : (i+1/2, j+1/2)
 * Every grid array has the same pitched layout, r fastest: element (i,j), i in [-ng, nr+ng],
 * j in [-ng, nth+ng], lives at  (j + j0)*pitch + (i + i0)  with pitch, rows, i0, j0 from
 * grpic_grid_layout (i = 0 is 32-byte aligned, pitch is a multiple of 16 doubles).
 * Radial guard values are copies of the last physical value; theta ghost
 * rows hold the parity image about the axis (r, phi components even, theta components odd).
 */
#ifndef GRPIC_H_
#define GRPIC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct grpic_ctx grpic_ctx; /* opaque; owns only its own metric/area tables */

typedef struct {
  double a, M;           /* Kerr spin and mass (M = 1 in production; M = 0: flat space) PAPER.md:433 */
  int32_t nr, nth;       /* physical cells in ln r and theta                                        */
  int32_t ng;            /* guard nodes on each side in r and theta (>= 2)                          */
  double xi_in, xi_out;  /* ln r of the inner / outer physical boundary               */
  double dphi;           /* azimuthal extent of the axisymmetric slab (Delta phi of B8/B10), 2 pi   */
  int32_t geo_iters;     /* K: trapezoidal corrector iterations of the geodesic step  */
  int32_t field_iters;   /* N: corrector iterations of the field step                 */
  double beta_impl;      /* semi-implicit weight beta (alpha = 1 - beta)              */
  int32_t damp_cells;    /* width (radial cells) of the outer damping layer; 0 = off  */
  double damp_coef;      /* lambda_i = 1 - damp_coef * s^3, s = (i - i_start)/damp_cells in (0,1]   */
} grpic_params;

/* Particle store, structure of arrays, FP64 (contravariant x^i, covariant u_i,
 * both at integer time steps :176).  x1 = ln r, x2 = theta, x3 = phi.  w = macro-particle
 * weight.  cell = j*nr + i of the current position (0xFFFFFFFF once removed).
 * flag bit0: species sign, 1 = positron (q/m = +1), 0 = electron (q/m = -1);
 * flag bit1: removed (left through the inner or outer radial boundary);
 * flag bit2: photon species: eps = 0 in u^0, no Lorentz force, no charge
 * (pushed along null geodesics by the same calls; deposits nothing). */
typedef struct {
  double *x1, *x2, *x3, *u1, *u2, *u3, *w;
  uint32_t *cell, *flag;
  int64_t n;
} grpic_particles;

typedef struct { double *Dr, *Dth, *Dph, *Br, *Bth, *Bph; } grpic_fields; /* contravariant D^i, B^i */
typedef struct { double *Fr, *Fth, *Fph; } grpic_current;                  /* fluxes or densities   */

enum {
  GRPIC_OK = 0,
  GRPIC_ERR_ARG = -1,       /* null pointer / out-of-range parameter                 */
  GRPIC_ERR_CUDA = -2,      /* CUDA runtime error (no device, launch failure, ...)   */
  GRPIC_ERR_WORKSPACE = -3, /* workspace missing or too small for this call          */
  GRPIC_ERR_ALLOC = -4,     /* could not allocate the context's own tables           */
  GRPIC_ERR_TOO_LARGE = -5  /* size beyond the fixed capacity of a *_static entry point */
};
#define GRPIC_STATUS_FAR_MOVE 1u   /* a particle moved more than one cell in a step (still deposited exactly) */
#define GRPIC_STATUS_NONFINITE 2u  /* a particle state became NaN/Inf (particle is flagged removed)           */
#define GRPIC_STATUS_OFFGRID 4u    /* a deposit window left the guard region (contribution dropped), or an active
                                      particle was handed in outside [xi_in, xi_out) x [0, pi] (it is flagged
                                      removed, its cell is clamped for the gather, nothing is deposited)      */
#define GRPIC_STATUS_CAPACITY 8u   /* grpic_pair_production created more particles than the arrays hold       */

/* Create a context: validates params, computes on the device the area elements of Eq.(8)
 * (10-point Gauss-Legendre in xi and theta; D- and B-staggered sets) and
 * the 1-D coordinate tables.  Blocking (synchronises once).  *out is host memory. */
int grpic_create(const grpic_params* params, grpic_ctx** out);
int grpic_destroy(grpic_ctx* ctx);

/* Pitched layout shared by every grid array (host out-pointers). */
int grpic_grid_layout(const grpic_ctx* ctx, int32_t* pitch, int32_t* rows, int32_t* i0, int32_t* j0);

/* Copy the six area-element tables A^D_r, A^D_th, A^D_ph, A^B_r, A^B_th, A^B_ph (Eq.8; the
 * phi areas WITHOUT dphi, i.e. dV = dphi*A^D_ph) into six caller device arrays of the grid
 * layout.  For tests and diagnostics. */
int grpic_get_areas(const grpic_ctx* ctx, double* const out[6], void* stream);

/* Scratch memory: the caller allocates grpic_workspace_bytes(ctx, max particles) bytes of
 * device memory and registers it; push_deposit needs none, field_step / sort / compact do. */
size_t grpic_workspace_bytes(const grpic_ctx* ctx, int64_t n_particles);
int grpic_set_workspace(grpic_ctx* ctx, void* dev_ptr, size_t bytes);

/* One particle step n -> n+1 for all particles not yet removed (Fig.2 :239):
 *   gather D^n,B^n at x^n (first order, :228) -> full-dt generalised Boris (Eq.16-19, :176-200)
 *   -> geodesic predictor + K trapezoidal correctors (Eq.12,14,15, :142-174) -> axis
 *   reflection (:136) -> removal flag (:138) and new cell -> charge-conserving deposit of the
 *   move x^n -> x^{n+1} (Eq.21-23, :208-233, CIC shape).
 * Particles are updated IN PLACE.  The FLUXES  F_r = J^r A^D_r, F_th = J^th A^D_th,
 * F_ph = J^ph dV  of the step are ACCUMULATED (+=) into `flux` (zero it first; guards and
 * theta ghost rows receive the parts deposited beyond the domain).  `fields` must have
 * valid guard / ghost values (grpic_field_step and grpic_fill_guards maintain them).
 * `status` may be NULL.  The particle arrays must be 16-byte aligned (they are streamed
 * through shared memory with bulk TMA copies); otherwise GRPIC_ERR_ARG.  Particles that leave are
 * only FLAGGED (bit 1) here; see grpic_set_removed_counter for the lazy-removal scheme and
 * grpic_push_deposit_compact for compaction fused into the push.  On grids whose cells are no larger
 * than 2^-8 in ln r and theta, at a time step with 2 dt <= 2^-8 r_in, r, sin(theta), cos(theta) are
 * taken from the context's node tables plus a short in-cell series (a few ulp from exp / sincos). */
int grpic_push_deposit(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                       grpic_current* flux, double dt, uint32_t* status, void* stream);

/* Lazy removal: grpic_push_deposit only FLAGS the particles that leave; they are
 * skipped by every later call and moved behind the live particles by the next grpic_sort /
 * grpic_sort_interleaved (their key is the largest), so a caller that sorts periodically needs no
 * compaction pass.  To know the survivor count without a pass over the flags, hand the library a
 * DEVICE counter: every grpic_push_deposit / grpic_push_deposit_compact call adds to *counter the
 * number of particles it flagged removed (NULL, the default, disables it).  The counter is the
 * caller's memory; the library keeps only the pointer until it is replaced. */
int grpic_set_removed_counter(grpic_ctx* ctx, unsigned long long* device_counter);

/* The same particle step with the THIRD-ORDER (cubic B-spline) shape, the paper's configuration
 * option ("a third order spline is also available"): gather over the 4 x 4 nodes of
 * the spline's support on each component's own lattice, prefix-sum deposit (Eq.21-23) over the
 * window the spline covers during the move.  In place, fluxes accumulated (+=) as in
 * grpic_push_deposit.  The context must have been created with ng >= 3 guard nodes
 * (GRPIC_ERR_ARG otherwise).  General kernel (one thread per particle, 96 loads and up to 96 REDs per
 * particle): about 4.5 x the time of the first-order step (profiles/r02_late_experiments.md). */
int grpic_push_deposit_spline3(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                               grpic_current* flux, double dt, uint32_t* status, void* stream);

/* The particle step with the paper's method variants selected by argument (same in-place
 * semantics as grpic_push_deposit).  (1, 1) runs the tuned kernel of grpic_push_deposit with the Vay
 * update in place of Boris when the particle arrays are 16-byte aligned; everything else the general
 * kernel:
 *   shape_order = 1 (cloud-in-cell) or 3 (cubic B-spline, needs ng >= 3);
 *   pusher = 0: generalised Boris (Eq.16-19); 1: Vay update in the FIDO frame (Vay
 *   2008) with the triad e_(1) = sqrt(gamma^rr)(d_r - gamma_rphi/gamma_phiphi d_phi),
 *   e_(2) = d_theta/sqrt(gamma_thth), e_(3) = d_phi/sqrt(gamma_phiphi) and proper time alpha*dt.
 * grpic_push_deposit_spline3 is (3, 0).  Other values: GRPIC_ERR_ARG. */
int grpic_push_deposit_variant(grpic_ctx* ctx, grpic_particles* ptc, const grpic_fields* fields,
                               grpic_current* flux, double dt, int32_t shape_order, int32_t pusher,
                               uint32_t* status, void* stream);

/* Removal fused into the push (SURVEY 8(a) rows a1-a5 + a9): exactly
 * grpic_compact(in -> out) followed by grpic_push_deposit(out), in one pass over the particles.
 * `out` (must not alias `in`; in is not modified) receives, in their original order, the
 * particles of `in` that are not flagged removed, each advanced one step (a particle that leaves
 * during THIS step is stored with its removed flag set and is squeezed out by the next call);
 * the DEVICE word *n_alive = number of particles pushed (= survivors of `in`); entries
 * [*n_alive, n) of out are marked removed, so the caller may keep using n as the upper bound
 * without reading n_alive back.  out->n = in->n.  Needs workspace (one word per 32 particles). */
int grpic_push_deposit_compact(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out,
                               const grpic_fields* fields, grpic_current* flux, double dt,
                               int64_t* n_alive, uint32_t* status, void* stream);

/* Multi-GPU hook of grpic_step_host (partitioning A: particles sharded over ranks, grid
 * replicated): when set, the callback is invoked once per grpic_step_host call, after the last
 * particle chunk has been deposited and before the current is finalised, with the DEVICE pointer of
 * the context's three flux arrays (contiguous, 3 x rows x pitch doubles) and the caller's stream.  It
 * must sum them over the ranks in stream order (e.g. one ncclAllReduce on that stream) and return 0;
 * any other value aborts the step with GRPIC_ERR_CUDA.  fn = NULL removes the hook. */
typedef int (*grpic_flux_exchange_fn)(void* user, double* flux3, size_t n_doubles, void* stream);
int grpic_set_flux_exchange(grpic_ctx* ctx, grpic_flux_exchange_fn fn, void* user);

/* END-TO-END step with the particle state in HOST memory (the one call that takes host
 * pointers): host_ptc (HOST SoA; pinned memory makes the copies asynchronous), host_J (HOST,
 * grid layout, nullable) and host_status (HOST word, nullable); `fields` / `background` stay
 * DEVICE arrays.  Does, for one step: stream the particles through the GPU in chunks of
 * `chunk_particles` (0 = 4 Mi) -- host->device copy, grpic_push_deposit_compact, device->host
 * copy of the survivors, the three overlapped on separate streams -- then
 * grpic_finalize_current and grpic_field_step on the device, and copies J back.  On return
 * (the call BLOCKS until the host buffers are complete) host_ptc holds the survivors of the
 * input, pushed one step, in their original order in entries [0, host_ptc->n) -- n is updated
 * to the survivor count -- and `fields` is advanced one step.  The chunk staging buffers and the
 * device flux arrays belong to the context (allocated on first use, freed by grpic_destroy);
 * the workspace of grpic_field_step must be registered.  The step equals the device-resident
 * sequence exactly, except for the summation order of the deposit. */
int grpic_step_host(grpic_ctx* ctx, grpic_particles* host_ptc, grpic_fields* fields,
                    const grpic_fields* background, grpic_current* host_J, double dt,
                    int32_t filter_passes, int64_t chunk_particles, uint32_t* host_status, void* stream);

/* Simplified pair production of the paper's Section 4 (Eq.26), one pass over
 * particles [0, ptc->n) of arrays that have room for `capacity` particles:
 *  - a lepton whose FIDO Lorentz factor sqrt(1 + gamma^ij u_i u_j) >= gamma_thr (and whose
 *    |u| = sqrt(gamma^ij u_i u_j) > eps_ph) emits one photon (flag bit2) of FIDO energy eps_ph
 *    along its motion, u_i^ph = u_i eps_ph/|u|, and keeps u_i (1 - eps_ph/|u|);
 *  - a photon converts with probability p_convert (= 1 - exp(-tau dt), Eq.26; the caller passes
 *    the number), decided by the counter-based Philox4x32-10 uniform U(seed; index, step) <
 *    p_convert, provided half its FIDO energy exceeds 1: its slot becomes the electron and a
 *    positron is created, both with Lorentz factor E/2 along the photon's direction;
 *  - created particles inherit position, cell and weight of their parent and are appended at
 *    ptc->n, ptc->n + 1, ... in the order of their parents.
 * The DEVICE word *n_new receives the new particle count (<= capacity; children beyond capacity
 * are dropped and GRPIC_STATUS_CAPACITY is OR-ed into *status).  ptc->n is NOT changed by the
 * call (the count is only known on the device).  Needs workspace (two words per 32 particles). */
typedef struct {
  double gamma_thr;   /* threshold FIDO Lorentz factor for emission (paper: 100)       */
  double eps_ph;      /* FIDO energy of an emitted photon (paper: 4.0)                 */
  double p_convert;   /* conversion probability per step, 1 - exp(-tau dt), in [0, 1]  */
  uint64_t seed;      /* Philox key                                                    */
  uint32_t step;      /* time-step counter (third counter word)                        */
} grpic_pair_params;
int grpic_pair_production(grpic_ctx* ctx, grpic_particles* ptc, int64_t capacity,
                          const grpic_pair_params* params, int64_t* n_new, uint32_t* status, void* stream);

/* Fluxes -> current densities, in place: fold the theta ghost rows onto their mirror rows
 * (particles never cross the axis, :136), `filter_passes` passes of the (1,2,1)x(1,2,1)/16
 * binomial filter on the fluxes (BASELINE.json config 5), then J^r = F_r/A^D_r,
 * J^th = F_th/A^D_th, J^ph = F_ph/dV (:228).  Needs workspace when filter_passes > 0. */
int grpic_finalize_current(grpic_ctx* ctx, grpic_current* flux_to_J, int32_t filter_passes, void* stream);

/* One field step D^n,B^n -> D^{n+1},B^{n+1} in place: predictor Eq.(9), N correctors
 * Eq.(10) (:113-128), each sweep = auxiliary fields (B9),(B11) + circulations (B8),(B10)
 * (:478-518), axis conditions incl. Eq.(11) (:132-136), radial guards (:138), outer damping
 * layer towards `background` (NULL = towards zero).  J may be NULL (vacuum). */
int grpic_field_step(grpic_ctx* ctx, grpic_fields* fields, const grpic_current* J,
                     const grpic_fields* background, double dt, void* stream);

/* Impose axis values, radial guards and theta ghost rows on caller-initialised fields. */
int grpic_fill_guards(grpic_ctx* ctx, grpic_fields* fields, void* stream);

/* Circulations C_H (3) and C_E (3) of the given fields (B8)-(B11), for diagnostics/tests. */
int grpic_circulation(grpic_ctx* ctx, const grpic_fields* fields, double* const out[6], void* stream);

/* Stable sort by key = removed ? ncells : cell.  `out` receives the reordered SoA (must not
 * alias `in`), `perm[k]` = source index of output k (may be NULL).  out->n = in->n. */
int grpic_sort(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, uint32_t* perm, void* stream);

/* Cell sort in the contention-free order (BASELINE.json north_star: "deposition ... keyed by sorted
 * cell", "heavy atomic contention"; not in the paper).  Order = lexicographic (cell / block_cells,
 * rank, cell % block_cells), where rank is the position of the particle among the particles of
 * its cell in the stable order of grpic_sort; removed particles follow in their input order.
 * All keys are distinct, so the permutation is unique (bit-exact against the oracle).  Particles
 * that are neighbours in memory then sit in different, adjacent cells: the lanes of a warp of
 * grpic_push_deposit never add to one address in one RED instruction.  block_cells: power of two
 * in [1, 32] (1 = the order of grpic_sort; 8 is the measured best).  Same arguments, ownership and
 * errors as grpic_sort; the workspace must come from grpic_workspace_bytes. */
int grpic_sort_interleaved(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, uint32_t* perm,
                           int32_t block_cells, void* stream);

/* Order-preserving removal of flagged particles: survivors are copied to `out` (must not
 * alias `in`) in order; their count is written to the DEVICE word n_alive. */
int grpic_compact(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, int64_t* n_alive, void* stream);

/* grpic_compact for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same result bit for bit, but NO workspace -- neither
 * grpic_set_workspace nor any cudaMalloc / cudaFree / allocating library call.  The scratch (per-tile
 * survivor counts and their scan) lives in a file-scope `static __device__` array of the library,
 * 160 KiB that every GPU that loads the library holds until exit, sized for at most
 * GRPIC_COMPACT_STATIC_MAX_PARTICLES particles: in->n beyond that returns GRPIC_ERR_TOO_LARGE and
 * launches nothing.  ALL calls on one device share that array: calls that overlap on the GPU (two
 * streams, two contexts, two host threads) race and give wrong results -- serialise them.  The array
 * keeps the last call's contents; nothing in it has to start at zero (every word a call reads was
 * written by that call first).  The first call on each device resolves the array's device address
 * (cudaGetSymbolAddress, no allocation): make that first call outside stream capture, with the device
 * of the arrays current. */
#define GRPIC_COMPACT_STATIC_MAX_PARTICLES (1 << 26)
int grpic_compact_static(grpic_ctx* ctx, const grpic_particles* in, grpic_particles* out, int64_t* n_alive,
                         void* stream);

/* Charge density on vertices, rho_ij = sum q w S_ij(x) / dV_ij (theta ghosts folded);
 * divide = 0 returns rho*dV.  Overwrites `rho`. */
int grpic_deposit_rho(grpic_ctx* ctx, const grpic_particles* ptc, double* rho, int32_t divide, void* stream);

/* Diagnostics in Boyer-Lindquist coordinates and in the FIDO frame ((A6)-(A7)): for
 * every particle k < ptc->n writes  E_inf[k] = -u_t = alpha^2 u^0 - beta^r u_r  (energy at infinity),
 * gamma_fido[k] = alpha u^0,  ur_bl[k] = u_r^KS - (2 M r E_inf - a u_phi)/Delta  (covariant radial
 * momentum in BL; u_t, u_theta, u_phi are the same in both systems) and  phi_bl[k] = phi_KS -
 * a/(2 sqrt(M^2-a^2)) ln|(r-r_+)/(r-r_-)|.  Output arrays are caller-owned DEVICE arrays of length
 * >= ptc->n, each may be NULL; removed particles get NaN.  The particle arrays are not modified. */
int grpic_ks_to_bl(grpic_ctx* ctx, const grpic_particles* ptc, double* E_inf, double* gamma_fido,
                   double* ur_bl, double* phi_bl, void* stream);

/* Measurement aid: the SM clock a push ran at.  When set, every grpic_push_deposit(_compact) launch
 * writes four DEVICE words { cycle counter at start, nanosecond timer at start, cycle counter at the
 * end, nanosecond timer at the end } taken by the first thread of its persistent grid; (w[2]-w[0]) /
 * (w[3]-w[1]) is the SM clock in GHz during that launch (under the board's power cap it can be lower
 * than the clock of a register-only probe kernel).  NULL (the default) disables it. */
int grpic_set_clock_probe(grpic_ctx* ctx, unsigned long long* device_words4);

/* Roofline denominator: measured FP64 pipe throughput of this device.  Runs a register-only
 * kernel of independent DFMA chains on every SM (blocking, ~10 ms) and writes the achieved
 * FP64 instructions (lane-operations) per second to the HOST double *dfma_per_second. */
int grpic_measure_fp64_peak(grpic_ctx* ctx, double* dfma_per_second);
/* The same, also returning the SM clock (MHz, cycle counter over nanosecond timer) the probe ran at. */
int grpic_measure_fp64_peak_clocked(grpic_ctx* ctx, double* dfma_per_second, double* sm_mhz);

/* Number of CUDA kernels this library has launched in this process so far (all contexts);
 * used by bench.py to report `gpu_launches`. */
int64_t grpic_kernel_launches(void);

const char* grpic_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* GRPIC_H_ */
