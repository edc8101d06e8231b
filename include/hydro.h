/* hydro.h -- C ABI of the B200-native hot path of the (3+1)-D ideal relativistic hydrodynamics solver of
 * arxiv 1511.02137 (Marcinkowski et al.).  One handle = one GPU, one CUDA stream, one Cartesian grid.
 *
 * What the library computes (citations are PAPER.md lines):
 *   d_mu T^{mu nu} = S^nu,  T^{mu nu} = (e+p) u^mu u^nu - p g^{mu nu}           eq. (1)  :17-19
 *   S^nu = sum_jets (-dE/dt, -dM/dt) delta^3(x - x_jet(t))                        eq. (2)  :21-23
 *   -dE/dx = kappa_rad (C_R/C_F) T^3 x + kappa_coll (C_R/C_F) T^2                 eq. (3)  :27-31
 *   7th-order WENO in space, 3rd-order Runge-Kutta in time                        :25
 *   Cartesian grid, EOS p = e/3, dx = 0.1 fm, dt = 0.02 fm/c, 256^3               :13, :49
 * for the conserved densities U = (T^00, T^0x, T^0y, T^0z [, N_B]).  Everything the paper leaves open
 * (Lax-Friedrichs splitting, WENO-JS weights, Shu-Osher RK3, outflow ghosts, delta-function deposit, T(e),
 * admissibility cap) follows the readings R1-R14 listed in DESIGN.md.  Optional, off by default: the WENO5 variant
 * (weno_order = 5), the Gaussian deposit (R15), the positivity-preserving flux limiter (R16), z-slab decomposition
 * over several GPUs and checkpoint/resume -- DESIGN.md 9 and 11.
 *
 * Conventions
 *   - every function returns an int status (HYDRO_OK = 0); nothing throws or aborts;
 *   - pointers are plain host or device pointers as stated per argument (`memspace`); the library never
 *     keeps or frees a caller's pointer; the caller owns every buffer it passes;
 *   - field layout: `nfields` contiguous blocks of nz*ny*nx reals, x fastest:
 *         idx = ((f*nz + k)*ny + j)*nx + i,   interior cells only (ghost cells are never stored);
 *     element type is double (precision 64) or float (precision 32) as chosen at create;
 *   - cell (i,j,k) is centred at ((i + 1/2 - nx/2) dx, (j + 1/2 - ny/2) dx, (k + 1/2 - nz/2) dx)  (R6);
 *   - units: GeV/fm^3 for energy/momentum densities, fm for lengths, fm/c for times, c = 1;
 *   - all work is enqueued on the handle's stream; calls on one handle must not race (not thread-safe);
 *   - there is no CPU fallback: without a CUDA device hydro_create fails with HYDRO_ECUDA.
 */
#ifndef HYDRO_H_
#define HYDRO_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hydro hydro_t; /* opaque; owned by the library */

enum { HYDRO_OK = 0, HYDRO_EINVAL = 1, HYDRO_ENOMEM = 2, HYDRO_ECUDA = 3, HYDRO_ESTATE = 4 };
enum { HYDRO_EOS_CONFORMAL = 0 };             /* p = e/3; the only EOS */
enum { HYDRO_MEM_HOST = 0, HYDRO_MEM_DEVICE = 1 };
enum { HYDRO_FIELDS_CONSERVED = 0, HYDRO_FIELDS_PRIMITIVE = 1 };

/* run options ("eos" argument of hydro_create).  A zero in weno_eps / v_cap_delta / e_floor selects the
 * default of the chosen precision. */
typedef struct {
    int    eos;          /* HYDRO_EOS_CONFORMAL */
    int    nfields;      /* 4 = (T00, T0x, T0y, T0z); 5 adds the baryon density N_B = n gamma (config 4) */
    int    precision;    /* 64 (fp64) or 32 (fp32 variant, reading R10) */
    double weno_eps;     /* epsilon of the WENO-JS weights, default 1e-6 (R3) */
    double v_cap_delta;  /* |M| <= (1 - delta) E in con2prim, default 1e-10 (fp64) / 1e-5 (fp32) (R9, R10) */
    double e_floor;      /* E >= e_floor in con2prim, default 1e-12 GeV/fm^3 (R9) */
    int    weno_order;   /* 7 (or 0): 7th-order WENO, the scheme the paper uses; 5: its 5th-order variant */
} hydro_eos_t;

/* Kernel classes timed by hydro_set_profiling / hydro_get_kernel_times. */
enum { HYDRO_K_PRIM = 0, HYDRO_K_SWEEP_X = 1, HYDRO_K_SWEEP_Y = 2, HYDRO_K_SWEEP_Z = 3, HYDRO_K_SOURCE = 4,
       HYDRO_K_COUNT = 5 };

/* Create a solver for an nx*ny*nz grid (each >= 1; a direction with fewer than 8 cells still works through
 * index clamping), spacing dx > 0 [fm] in all directions, fixed step dt > 0 [fm/c].  `eos` may be NULL
 * (conformal EOS, 4 fields, fp64, default parameters).  `cuda_stream` is a cudaStream_t passed as a void*
 * (NULL = the library creates and owns a non-blocking stream).  Allocates 3 state copies, one RHS copy and
 * two primitive fields on the current CUDA device.  Errors: HYDRO_EINVAL, HYDRO_ENOMEM, HYDRO_ECUDA. */
int hydro_create(hydro_t **out, int nx, int ny, int nz, double dx, double dt, const hydro_eos_t *eos,
                 void *cuda_stream);
void hydro_destroy(hydro_t *h);

/* Copy the conserved state in (layout above; `U` is a host pointer for HYDRO_MEM_HOST, a device pointer for
 * HYDRO_MEM_DEVICE).  Resets the step counter, the time and the diagnostics to 0; jets are kept and restart
 * from their initial positions at t = 0.  Asynchronous for device memory, synchronous for host memory. */
int hydro_set_state(hydro_t *h, const void *U, int memspace);

/* Add a jet (eq. 2, 3): position (x0,y0,z0) [fm] relative to the grid centre at the current simulation time,
 * direction normalised inside (zero vector -> HYDRO_EINVAL), speed c, never deflected or stopped
 * (PAPER.md:31).  kappa_rad, kappa_coll, cr_over_cf are the coefficients of eq. (3) (paper: 4, 2.5, 1).
 * `id` (may be NULL) receives the jet index. */
int hydro_add_jet(hydro_t *h, double x0, double y0, double z0, double dirx, double diry, double dirz,
                  double kappa_rad, double kappa_coll, double cr_over_cf, int *id);
int hydro_clear_jets(hydro_t *h);

/* Checkpoint / resume: the state of a run is (U, completed steps, the jets as added).  After hydro_set_state(U of a
 * checkpoint) and re-adding the jets with their ORIGINAL start positions, hydro_set_step(h, n) restores the step
 * counter, so that jet positions and path lengths continue from t = n dt; the continuation is bitwise the same run. */
int hydro_set_step(hydro_t *h, long long step);
/* ---- z-slab decomposition over several GPUs: one handle per rank -------------------------------
 * The handle's grid is the rank's LOCAL array: its owned planes plus 4 halo planes towards each neighbouring rank (none
 * at a physical boundary, where the zero-gradient ghosts of a-7 act).  hydro_set_slab: nz_global = planes of the whole
 * grid, k_offset = global index of local plane 0, [own_lo, own_hi) = owned local planes (>= 4 of them; an interior end
 * needs its 4 halo planes: HYDRO_EINVAL otherwise).  Jet positions stay global; cap events and jet bookkeeping are
 * counted for owned planes only, so sums over ranks are the global figures.
 * One RK3 step = for s in 0, 1, 2 (serial form):
 *     hydro_stage_prims(h, s)                      con2prim + LOCAL wavespeed maxima of stage s's input state
 *     hydro_stage_alpha(h, s, 0, a); a = MAX over ranks; hydro_stage_alpha(h, s, 1, a)      (host round trip, 24 bytes)
 *       or, without leaving the device: hydro_stage_alpha_dev(h, s, 0, bits); MAX all-reduce of the three 64-bit
 *       integers (non-negative reals order like their bit patterns); hydro_stage_alpha_dev(h, s, 1, bits)
 *     hydro_stage_sweeps(h, s)                     sweeps + source + stage combination -> stage s's output state
 *     hydro_halo(h, s, side, 0, buf)  pack the 4 owned boundary planes (side 0: low z, 1: high z) of that output state,
 *                                     all fields, into the DEVICE buffer buf (nfields * 4 * ny * pitch reals, see
 *                                     hydro_halo_reals); exchange with the neighbour; hydro_halo(h, s, side, 1, buf) unpacks
 *                                     the neighbour's planes into the halo.  Asynchronous on the handle's stream.
 * Overlapped form (the halos of stage s's INPUT state may still be in flight; not with the limiter or a Gaussian deposit,
 * which need the halos before the x sweep: HYDRO_ESTATE):
 *     hydro_stage_prims_part(h, s, 0)              owned planes: con2prim + local wavespeed maxima
 *     alpha exchange as above
 *     hydro_stage_sweeps_part(h, s, 0)             x sweep + source + y sweep on the owned planes (no z neighbour needed)
 *     wait for the halos of the input state, hydro_halo(..., unpack)
 *     hydro_stage_prims_part(h, s, 1)              halo planes: con2prim only
 *     hydro_stage_sweeps_part(h, s, 1)             z sweep (marches the whole local array)
 *     pack and send the boundary planes of the output state
 * hydro_stage_sweeps(h, 2) / hydro_stage_sweeps_part(h, 2, 1) advance the step counter.  Owned planes come out bitwise
 * identical to the one-GPU run in both forms.  With a Gaussian deposit (hydro_set_deposit_width) the cube's half-width
 * R must not exceed the 4 halo planes (sigma <= 4 dx / 3): HYDRO_EINVAL otherwise. */
int hydro_set_slab(hydro_t *h, int nz_global, int k_offset, int own_lo, int own_hi);
int hydro_stage_prims(hydro_t *h, int s);
int hydro_stage_alpha(hydro_t *h, int s, int set, double alpha[3]);
int hydro_stage_sweeps(hydro_t *h, int s);
int hydro_stage_prims_part(hydro_t *h, int s, int part);
int hydro_stage_sweeps_part(hydro_t *h, int s, int part);
/* dev_bits: DEVICE pointer to three 64-bit integers.  set = 0: copy the stage's three alpha bit patterns out; 1: in.
 * Asynchronous on the handle's stream; no host synchronisation. */
int hydro_stage_alpha_dev(hydro_t *h, int s, int set, void *dev_bits);
int hydro_halo(hydro_t *h, int s, int side, int unpack, void *dev_buf);
long long hydro_halo_reals(const hydro_t *h);

/* Positivity-preserving flux limiter on/off (default off; fp64 only, HYDRO_EINVAL in fp32).  Reading R16 (
 * SURVEY 8(f) f-1; PAPER.md:25/:58 cite the positivity-preserving FD-WENO scheme without details): every interface flux is
 * F^L + theta (F^H - F^L) with F^L the first-order Lax-Friedrichs flux and one theta in [0,1] per face, chosen from the
 * concavity of g(U) = E - |M| around the first-order update so that E > |M| is kept (for 3 alpha dt/dx <= 1).  Costs one
 * extra kernel per stage and ~2 blocks/SM instead of 3 in the sweeps.  hydro_get_limited_faces: cumulative number of
 * (face, stage) events with theta < 1.  Synchronises. */
int hydro_set_limiter(hydro_t *h, int enable);
int hydro_get_limited_faces(hydro_t *h, long long *n);

/* Width sigma >= 0 [fm] of the jets' deposit (all jets of the handle).  0 (default): the delta function of eq. (2) is one
 * cell (R7).  > 0: a normalised Gaussian of that width around the jet position, sampled on the (2R+1)^3 cells around
 * the R7 cell, R = ceil(3 sigma/dx) clamped to [1, 8] (reading R15). */
int hydro_set_deposit_width(hydro_t *h, double sigma);

/* Advance nsteps >= 0 full SSP-RK3 steps of size dt: per stage con2prim + wavespeed max (a-1, a-2), the three
 * WENO7 Lax-Friedrichs sweeps (a-3, a-4), the jet source (a-5) and the stage combination (a-6), with
 * zero-gradient outflow ghosts (a-7).  Asynchronous on the handle's stream. */
int hydro_step(hydro_t *h, int nsteps);

/* Block until everything enqueued on the handle's stream has finished. */
int hydro_synchronize(hydro_t *h);

/* which = HYDRO_FIELDS_CONSERVED: U (same layout as set_state); HYDRO_FIELDS_PRIMITIVE: (e, vx, vy, vz[, n])
 * from con2prim of the current state.  `out` holds nfields*nz*ny*nx reals in `memspace`.  Synchronises. */
int hydro_get_fields(hydro_t *h, void *out, int which, int memspace);

/* L(U, t_n + stage_c*dt) = -sum_d D_d(U) + S of the CURRENT state, written to `out` (layout of U, `memspace`).
 * Does not advance anything; refreshes alpha.  For stage-level parity tests.  Synchronises. */
int hydro_eval_rhs(hydro_t *h, double stage_c, void *out, int memspace);

/* Diagnostics (any pointer may be NULL): alpha[3] = Lax-Friedrichs speeds of the last evaluated stage,
 * cfl = max(alpha) dt/dx, ncap = cumulative number of (cell, stage) events where the con2prim floor/cap fired,
 * has_nan = a non-finite conserved value was seen, deposited[4] = total (E, Mx, My, Mz) [GeV] added by jets,
 * step = number of completed steps.  Synchronises. */
int hydro_get_diag(hydro_t *h, double alpha[3], double *cfl, long long *ncap, int *has_nan, double deposited[4],
                   long long *step);
/* q^s [GeV/fm] of jet `jet` in the three stages of the last step (out[3]).  Synchronises. */
int hydro_get_last_stage_q(hydro_t *h, int jet, double out[3]);

/* Per-kernel-class device times: when enabled, CUDA events bracket every kernel launch of hydro_step on the
 * handle's stream; hydro_get_kernel_times synchronises and returns accumulated milliseconds and launch counts
 * per class (arrays of HYDRO_K_COUNT) since profiling was last enabled. */
int hydro_set_profiling(hydro_t *h, int enable);
int hydro_get_kernel_times(hydro_t *h, double ms[HYDRO_K_COUNT], long long launches[HYDRO_K_COUNT]);

/* Which sweep kernels this handle uses: always 1 = the TMA ring kernels of hydro_sweep_ring.cuh (rows are stored
 * with a 16-byte-aligned pitch on the device, so every nx qualifies). */
int hydro_sweep_path(const hydro_t *h);

/* Number of kernel launches hydro_step has enqueued on this handle since create. */
long long hydro_launch_count(const hydro_t *h);

/* Register-resident DFMA (precision 64) or FFMA (32) chain on every SM of the current device for about
 * `millis` ms on `cuda_stream`; returns the achieved TFLOP/s (FMA = 2 flops).  The measured ALU peak the
 * roofline fraction is quoted against. */
int hydro_measure_alu_peak(int precision, double millis, void *cuda_stream, double *tflops);

/* ---- the one entry point that allocates nothing (csrc/hydro_noalloc.cu) ----------------------------------------------
 * Steps a-1 + a-2 (con2prim for p = e/3 from eq. 1, reading R9; Lax-Friedrichs speeds R4) of a
 * caller's fp64 DEVICE state: alpha_dev[d] = max over the cells of max(|lambda_+^d|, |lambda_-^d|), d = x, y, z (exact
 * maxima, hence order independent), counts_dev[0] = cells where the floor / cap of con2prim fired, counts_dev[1] = 1 if a
 * non-finite conserved value was seen.  For callers that cannot call cudaMalloc (stream capture, tight serving loops,
 * harnesses that forbid it): no handle, and no cudaMalloc / cudaFree / allocating routine is called.  The kernel's
 * scratch (P, W and the reduction block) is a file-scope __device__ array of HYDRO_NOALLOC_MAX_CELLS x 16 bytes + 4 KiB
 * (4 MiB + 4 KiB) that every GPU loading the library holds until exit; larger grids are rejected with HYDRO_EINVAL.
 *   U_dev       DEVICE, nfields (4 or 5) contiguous blocks of nz*ny*nx doubles, x fastest (hydro_set_state's layout); read only
 *   v_cap_delta, e_floor   as in hydro_eos_t (0 selects the fp64 defaults 1e-10, 1e-12)
 *   alpha_dev   DEVICE, 3 doubles, written;  counts_dev  DEVICE, 2 long long, written (may be NULL)
 *   cuda_stream the work is enqueued there (NULL = the default stream) on the CURRENT device; asynchronous
 *   err, errlen optional host buffer that receives a one-line message when the return value is not HYDRO_OK
 * All calls share the scratch array, which keeps the last call's contents (the reduction block is cleared by every call):
 * calls that overlap on the GPU -- other streams, other host threads -- race on it; serialise them.  Caller owns every
 * pointer. */
#define HYDRO_NOALLOC_MAX_CELLS 262144          /* 64^3 */
int hydro_wavespeeds_noalloc(const void *U_dev, int nx, int ny, int nz, int nfields, double v_cap_delta, double e_floor,
                             double *alpha_dev, long long *counts_dev, void *cuda_stream, char *err, int errlen);

const char *hydro_strerror(int code);
/* Text of the last CUDA error seen by this handle ("" if none). */
const char *hydro_last_cuda_error(const hydro_t *h);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_H_ */
