/*
 * glisse.h — C ABI of the B200-native GLISSE hot path.
 *
 * What the library computes (all fp64): N massless test particles are advanced through a
 * star + N_p planet system with the fixed-time-step Wisdom–Holman mixed-variable symplectic
 * step of Zhang & Gladman 2020 (§2.2 Eq. 1–2 and the 5-item step list at
 * PAPER.md:91-95): kick ½ – Kepler drift 1 – kick ½ for the particles, the standard Jacobi
 * WH step for the mutually interacting planets, close-encounter / escape tests
 * that flag and freeze a particle.  DESIGN.md §2 lists every reading of the
 * paper that this header relies on (step order, Kepler-solver form, flag priorities …).
 *
 * Every step of the path runs in hand-written CUDA kernels for sm_100a; there is no CPU
 * fallback.  If no CUDA device is usable every entry point returns GLISSE_ECUDA.
 *
 * Conventions
 *  - Return value: 0 (GLISSE_OK) on success, a negative GLISSE_E* status otherwise.  The
 *    library never throws, aborts or prints.
 *  - Units: the library is unit-agnostic; G is folded into the masses (gm = G·m).  The
 *    benchmark configurations use AU, days, solar masses with G = k² (Gaussian constant).
 *  - Pointers marked "host or device" are handed to cudaMemcpyAsync with cudaMemcpyDefault: the
 *    driver's unified addressing tells host from device, the library never classifies them itself
 *    (one exception: glisse_planet_log_static, whose kernel writes the caller's buffer directly,
 *    asks cudaPointerGetAttributes whether it is device memory).
 *    Host buffers should be pinned for the copies to overlap; pageable ones work and serialise.
 *  - Ownership: inputs are copied during glisse_create (the caller keeps its buffers); outputs
 *    are caller-allocated.  The library owns its internal device state until glisse_destroy.
 *  - Threading: a glisse_sim must be used by one host thread at a time; different sims may be used
 *    from different threads.  Process-wide state is limited to three caches behind one mutex: a
 *    stream-ordered memory pool per device (a sim's arena comes from it and goes back to it), up to
 *    eight idle streams of each priority per device (a sim's streams come from them and go back,
 *    synchronised, at glisse_destroy) and one pinned page of mailbox words for survivor counts.
 *  - Measurement and test hooks (launch counter, kernel timer, FP64 probe, primitive evaluator,
 *    solver statistics) are NOT part of this interface: include/glisse_test.h.
 */
#ifndef GLISSE_H_
#define GLISSE_H_

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------------------------- */
#define GLISSE_OK       0
#define GLISSE_EINVAL  (-1)  /* null pointer, size <= 0, n_planets outside [0,32], dt == 0,
                                non-finite input, bad params                                  */
#define GLISSE_ECUDA   (-2)  /* a CUDA call failed (sticky: the sim is unusable afterwards)    */
#define GLISSE_ENOMEM  (-3)  /* host or device allocation failed                              */
#define GLISSE_EPLANET (-4)  /* a planet's Kepler drift failed (unbound / not converged): the
                                paper requires encounter-free planets           */
#define GLISSE_ELIMIT  (-5)  /* a size beyond the fixed capacity of an entry point that may not
                                allocate (glisse_planet_log_static)                           */

/* ---- per-particle flag values ("a flag that records which planet") ------------ */
#define GLISSE_FLAG_ACTIVE    0
#define GLISSE_FLAG_RMIN      1   /* |r| < r_min                     (BASELINE.json configs)  */
#define GLISSE_FLAG_RMAX      2   /* |r| > r_max                     (BASELINE.json configs)  */
#define GLISSE_FLAG_NONCONV   3   /* Kepler solve not converged           */
#define GLISSE_FLAG_UNBOUND   4   /* 2μ/r − v² <= 0 at the drift     (reading S8)   */
#define GLISSE_FLAG_PLANET0  16   /* 16 + j : |r − q_j| < rcrit_j       */

#define GLISSE_MAX_PLANETS   32

/* ---- splitting of the step (params.scheme) ------------------------------------------------- */
#define GLISSE_SCHEME_KDK 0   /* kick 1/2 - drift - kick 1/2, planets sampled at the integer steps t_s:
                                 the step list of PAPER.md:91-95 (default)                        */
#define GLISSE_SCHEME_DKD 1   /* drift 1/2 - kick - drift 1/2, planets sampled at the half steps
                                 t_{s+1/2}: BASELINE.json's wording of the same second-order
                                 splitting (reading S20).  The planets are carried by the
                                 same Wisdom-Holman step, started with one step of dt/2.  The tests
                                 run at the one force evaluation of the step; a hit freezes the state
                                 of that instant (after the first half drift).  Planet-log record k
                                 then holds the planets at t_{s+k+1/2}; glisse_advance_with_log still
                                 takes n_steps+1 records (the last one is not used).               */

typedef struct glisse_sim glisse_sim; /* opaque */

/* User-configurable quantities the paper names: Kepler iteration count (fn 5 at
 * 135), planetary chunk size, resync interval, output interval
 * (PAPER.md:121), and the iteration-count sort the paper proposes.             */
typedef struct {
  double r_min;         /* heliocentric inner removal radius; <= 0 disables the test           */
  double r_max;         /* heliocentric outer removal radius; +inf (or <= 0) disables the test */
  int    kepler_iters;  /* maximum number of Newton updates per Kepler solve, default 5        */
  double kepler_tol;    /* |residual of Kepler's equation| above which a particle is flagged
                           GLISSE_FLAG_NONCONV, default 1e-14.  With kepler_iters >= 5
                           and kepler_tol >= 4e-15 bodies with e < 0.8 are solved by a faster method
                           that reaches the same root to roundoff and leaves a residual below 2e-15;
                           otherwise every body goes through the Newton loop these two describe
                           (a slower kernel, chosen at create)                                  */
  int    chunk_steps;   /* K: steps per planet-log chunk = per particle-kernel launch,
                           default 1024, 1..16384; performance only, results do not depend on it */
  int    resync_chunks; /* R: survivor compaction every R chunks, 0 = never, default 1;
                           performance only, results do not depend on it                       */
  int    device;        /* CUDA device ordinal, default 0                                      */
  void*  stream;        /* cudaStream_t on which the particle work is enqueued, or NULL for a
                           stream owned by the library                                         */
  int    snapshot_chunks;  /* M_s: inside glisse_advance, after every M_s-th completed chunk (a
                           chunk completes when the step count reaches a multiple of K) write a
                           snapshot into the ring attached with glisse_snapshot_ring; 0 = off
                           (default).  PAPER.md:121 "copied back to the CPU after a
                           user-configurable number of planetary chunk calculations"           */
  int    resonance_chunks; /* M_r: likewise take a glisse_resonance_sample after every M_r-th
                           completed chunk once glisse_resonance_begin has been called; 0 = off */
  int    bin_iterations;   /* 1: at every resync (and once at create) survivors are ordered by the
                           number of Kepler-solver iterations their orbit can need, hardest group
                           first, particle-ID order within a group ("sort the
                           particles by the expected number of iterations ... the most eccentric
                           group would be launched first"): a few eccentric bodies then slow down
                           a few warps instead of every warp they are scattered over; 0:
                           particle-ID order; 2 (default): 1 if at create at least
                           one body in a thousand has an orbit the solver finds hard, else 0.
                           Performance only: results are bit-identical, and glisse_read returns
                           the caller's order either way.                                       */
  int    scheme;           /* GLISSE_SCHEME_KDK (default) or GLISSE_SCHEME_DKD                          */
  int    guess_order;      /* starting point of the Kepler solve ("a judicious initial guess",
                           PAPER.md:123): 1 = dE = dM a/r for every body; 3 = the series reversion
                           of Kepler's equation to third order for bodies with e dE^2 above ~6e-5
                           (eccentric orbits at small a: saves them a solver iteration, costs
                           quiet workloads 4 %); 0 (default) = chosen once, at create, from the
                           initial conditions: 3 if more than 5 % of the particles would take it.
                           The root is the same; results differ at roundoff between 1 and 3      */
  int    segment_steps;    /* a chunk is issued as back-to-back launches of this many steps whose
                           warps hand particles on through per-group completion flags, so the
                           tail of one launch is filled by the next; default 128,
                           0 = one launch per chunk.  Performance only, results do not depend
                           on it                                                               */
} glisse_params;

/* Fill *p with the defaults listed above.  p == NULL is ignored. */
void glisse_default_params(glisse_params* p);

/*
 * Create a simulation at step 0.
 *   gm_star        G·m0.
 *   n_planets      N_p in [0, 32]; planets are given in Jacobi order = order of increasing
 *                  distance from the star.
 *   gm_planet      [n_planets] host; G·m_j > 0.
 *   planet_pos/vel [n_planets][3] host, row-major (x,y,z per planet), heliocentric.
 *   planet_rcrit   [n_planets] host; absolute encounter radius of planet j in length units
 *                  (e.g. k Hill radii); 0 disables the test for that planet.
 *                  May be NULL (all tests off).
 *   n_particles    N >= 1 (N < 2^31).
 *   pos, vel       three pointers each (x,y,z / vx,vy,vz), every one an array of N doubles,
 *                  struct-of-arrays, heliocentric, host or device (all six of the same kind).
 *   dt             time step, non-zero; negative integrates backwards (time reversal).
 *   params         NULL = defaults.
 * On success *out holds the handle.  Work is enqueued on params->stream; create synchronises.
 */
int glisse_create(glisse_sim** out,
                  double gm_star,
                  int n_planets, const double* gm_planet,
                  const double* planet_pos, const double* planet_vel,
                  const double* planet_rcrit,
                  long long n_particles,
                  const double* const pos[3], const double* const vel[3],
                  double dt, const glisse_params* params);

/*
 * Advance planets and particles by n_steps >= 0 steps of size dt.  Asynchronous: kernels are
 * enqueued on the sim's stream (planet-history kernels on an internal second stream) and the
 * call returns without waiting.  The sequence per chunk of <= K steps is: planet-history kernel
 * (a1) -> particle kernel (a2–a7) -> every R chunks the compaction kernels (a8).
 * A planet failure is reported by the next synchronising call as GLISSE_EPLANET.
 */
int glisse_advance(glisse_sim* sim, long long n_steps);

/*
 * External planet history ("these planetary positions could be supplied using any
 * method, such as interpolation from a history file"): advance the PARTICLES by n_steps using a
 * caller-supplied planet log instead of the planet-history kernel.  log holds n_steps+1 records
 * (times t_s ... t_{s+n}), each glisse_log_stride(n_planets) doubles:
 *   [ q_0x q_0y q_0z  q_1x ... q_{Np-1}z   h0x h0y h0z   (zero padding to an even count) ]
 * with h0 = -sum_j gm_j q_j/|q_j|^3, host (pinned, for the upload to overlap) or
 * device.  ASYNCHRONOUS like glisse_advance: the log is streamed chunk by chunk through the
 * library's two log buffers on the planet stream while the particle kernel works on the previous
 * chunk — the paper's own double-buffered upload ("always two sets of planetary
 * data at a time on the GPU") — with no allocation and no host synchronisation; the caller's log
 * must stay valid until the next synchronising call (glisse_sync, glisse_read ...).
 * The internal planet state is NOT advanced: afterwards glisse_advance, glisse_read_planets,
 * glisse_planet_log and glisse_resonance_sample return GLISSE_EINVAL until glisse_set_planets
 * re-seeds the planets (glisse_advance_with_log itself can be called again at once).
 */
int glisse_advance_with_log(glisse_sim* sim, long long n_steps, const double* log);

/* Re-seed the internal planet integration at the CURRENT step: heliocentric positions and
 * velocities [n_planets][3] each, HOST.  The next glisse_advance continues from them. */
int glisse_set_planets(glisse_sim* sim, const double* planet_pos, const double* planet_vel);

/* Doubles per planet-log record: 3·(n_planets+1) rounded up to a multiple of 2 (16-byte rows
 * for bulk copies).  Returns 0 if n_planets is out of range. */
int glisse_log_stride(int n_planets);

/*
 * A planet log from a SPARSE history by interpolation ("these planetary positions could
 * be supplied using any method, such as interpolation from a history file"; reading S24).
 * The history holds n_samples >= 2 instants sample_time[m] (strictly increasing, in the unit of dt) with
 * the heliocentric positions sample_pos and velocities sample_vel of the sim's planets at them,
 * [n_samples][n_planets][3] each, in the planet order of glisse_create; host or device.  Record
 * r = 0 .. n_records-1 is taken at t_first + r dt_record by cubic Hermite interpolation of positions and
 * velocities on the interval that holds that instant, h0 from the interpolated positions, and written to
 * log (host or device, n_records x glisse_log_stride(n_planets) doubles, layout above) — ready for
 * glisse_advance_with_log (kick-drift-kick: n_steps+1 records from the current time with dt_record = dt;
 * drift-kick-drift: the same count from half a step later, the last one unused).  The simulation is not
 * changed.
 * GLISSE_EINVAL if the instants are not increasing or a record falls outside them.  Synchronises.
 */
int glisse_interpolate_log(glisse_sim* sim, long long n_samples, const double* sample_time,
                           const double* sample_pos, const double* sample_vel, double t_first,
                           double dt_record, long long n_records, double* log);

/*
 * Write the planet log the library itself would generate for the next n_steps steps
 * (n_steps+1 records, layout above) into log (host or device) WITHOUT changing the simulation.
 * Used to check the planet-history kernel (a1) against the oracle.  Synchronises.
 */
int glisse_planet_log(glisse_sim* sim, long long n_steps, double* log);

/*
 * glisse_planet_log for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same planet-history kernel, the same records, but NO
 * cudaMalloc / cudaFree / allocating routine anywhere in the call.  glisse_planet_log allocates two
 * buffers per call (a staging copy of the log, and the kernel's scratch: the Jacobi state it writes at
 * every record); here the kernel writes the log straight into the caller's buffer and its scratch is a
 * fixed array in device memory that the library holds on every GPU that loads it (2 MiB, until the
 * process exits).
 *   log: DEVICE memory of this sim's device, 16-byte aligned, (n_steps+1) x glisse_log_stride(n_planets)
 *        doubles (GLISSE_EINVAL for a host pointer: the kernel writes it directly).
 *   Limit: (n_steps + 1) x 6 n_planets doubles of scratch must fit 2^18 doubles, i.e. n_steps <=
 *        glisse_planet_log_static_limit(n_planets) (10 921 steps at 4 planets, 5 460 at 8, 1 364 at 32);
 *        beyond it GLISSE_ELIMIT, nothing launched, nothing changed.
 *   Sharing: every call on a device uses the same scratch array, which keeps the last call's contents.
 *        Nothing in it has to start at zero (the kernel writes each record before anything reads it), but
 *        two calls that OVERLAP on the GPU — different sims on different streams, or different host
 *        threads — race on it; this call synchronises before it returns, so calls made one after the other
 *        from one thread never overlap.
 * The simulation is not changed.  Synchronises.  Statuses otherwise as glisse_planet_log.
 */
int glisse_planet_log_static(glisse_sim* sim, long long n_steps, double* log);

/* Largest n_steps glisse_planet_log_static accepts for n_planets planets; < 0 if n_planets is out of range. */
long long glisse_planet_log_static_limit(int n_planets);

/*
 * Read the particle state in ORIGINAL particle order (compaction is invisible).
 * Any of pos, vel, flag, removal_step may be NULL (skipped); pos/vel are three pointers to
 * arrays of N doubles; flag is int[N]; removal_step is long long[N] (number of completed steps
 * when the particle was flagged, −1 while active).  Buffers host or device.  Synchronises.
 * A removed particle reports the state frozen at its removal.
 */
int glisse_read(glisse_sim* sim, double* const pos[3], double* const vel[3],
                int* flag, long long* removal_step);

/*
 * Snapshot: the periodic output of the particle arrays ("copied back to the CPU after
 * a user-configurable number of planetary chunk calculations"; "logged orbital
 * elements").  ASYNCHRONOUS: the call queues a device-side copy of the state
 * at the current step, in original particle order, and returns; a third stream then copies it to
 * the caller's buffers while later glisse_advance calls keep the device busy.  The buffers must stay
 * valid, and must not be read, until glisse_snapshot_wait returns.  One snapshot is in flight at a
 * time: a second call first waits (on the device) for the first one's copies.
 *   kind   GLISSE_SNAPSHOT_CARTESIAN  out[0..5] = x, y, z, vx, vy, vz
 *          GLISSE_SNAPSHOT_ELEMENTS   out[0..5] = a, e, i, Omega, omega, M: osculating heliocentric
 *          elements about gm_star (Murray & Dermott §2.8: h = r x v, vis-viva, eccentricity vector;
 *          tan i = |h_xy|/h_z; i = 0: Omega = 0 and omega from x; e = 0: omega = 0, M = angle of r;
 *          unbound: a < 0, M = NaN; angles in [0, 2 pi))
 *   out    six pointers to arrays of N doubles (any may be NULL: skipped); flag int[N] and
 *          removal_step long long[N] as in glisse_read (may be NULL).  Host (pinned, for the copy
 *          to overlap) or device.
 * A removed particle reports the state (or elements of the state) frozen at its removal.
 */
#define GLISSE_SNAPSHOT_CARTESIAN 0
#define GLISSE_SNAPSHOT_ELEMENTS  1
int glisse_snapshot(glisse_sim* sim, int kind, double* const out[6], int* flag, long long* removal_step);

/* Wait until the buffers of the last glisse_snapshot — and every ring slot written so far — are
 * filled.  Does not wait for the particles. */
int glisse_snapshot_wait(glisse_sim* sim);

/*
 * Output ring for the periodic snapshots a long glisse_advance emits on its own (params
 * snapshot_chunks): the k-th emitted snapshot (k = 0, 1, ...) goes to slot
 * k mod n_slots,
 *   data         [n_slots][6][N] doubles (kind as in glisse_snapshot), may not be NULL
 *   flag         [n_slots][N] ints, or NULL
 *   removal_step [n_slots][N] long longs, or NULL
 *   slot_step    [n_slots] long longs, or NULL: the step count at which the slot's snapshot was
 *                taken, written AFTER the slot's data (same stream), so a host that polls a
 *                pinned slot_step[] sees complete slots without synchronising the sim
 * all host (pinned) or device.  No host round trip: glisse_advance only enqueues.  The library
 * never waits for the caller to consume a slot: size the ring for the snapshots of one
 * glisse_advance call, or consume between calls.  n_slots = 0 detaches the ring.
 * glisse_snapshots_emitted returns k (host counter).
 */
int glisse_snapshot_ring(glisse_sim* sim, int kind, int n_slots, double* data, int* flag, long long* removal_step,
                         long long* slot_step);
long long glisse_snapshots_emitted(glisse_sim* sim);

/*
 * Resonant-argument reduction on the device.  For the p:q
 * mean-motion resonance with planet `planet` the argument is
 *     phi = p lambda − q lambda_planet − (p − q) varpi,   lambda = Omega + omega + M,  varpi = Omega + omega
 * (phi_31 = 3 lambda − lambda_N − 2 varpi, phi_52 = 5 lambda − 2 lambda_N − 3 varpi in the paper), from
 * the osculating heliocentric elements of glisse_snapshot; the planet's about gm_star + gm_planet.
 * "Librating particles [are] those with a resonant argument that never comes within 10 deg of 0 deg or
 * never within 10 deg of 180 deg": the library keeps, per particle, whether phi has been within
 * `window` (radians) of 0 and of pi at any sample.
 *   glisse_resonance_begin   choose the resonance and clear the record.  p > q >= 1.
 *   glisse_resonance_sample  evaluate phi at the current step for every ACTIVE particle and update the
 *                            record; asynchronous on the particle stream (call it between advances,
 *                            at the cadence of the paper's element log).
 *   glisse_resonance_read    seen0[N], seen180[N] (bytes, 0/1), phi_last[N] (the last sample's phi in
 *                            [0, 2 pi); NaN-free only for particles sampled at least once), original
 *                            particle order, host or device, any may be NULL; *n_samples = samples
 *                            taken since begin.  Synchronises.
 * With params.resonance_chunks = M_r > 0 the samples are taken inside glisse_advance after every
 * M_r-th chunk, fused with the snapshot of the same chunk boundary if there is one (the elements
 * are computed once for both).
 * GLISSE_EINVAL without a preceding begin, for planet outside [0, n_planets), or p <= q or q < 1.
 *
 * Libration amplitude ("a running window that diagnosed successive maxima and minima of
 * the resonant angle and measured the difference between them"): with phi taken in [0, 2 pi) — i.e.
 * unwrapped about pi, where the symmetric librators sit and which the asymmetric ones never leave —
 * every sample updates, per particle, the running minimum and maximum of phi and a turning-point
 * detector: sample k-1 is a maximum (minimum) if phi rose (fell) into it and falls (rises) out of it,
 * equal neighbours continuing the trend; each turning point after the first yields one amplitude
 * sample |phi_ext - phi_previous_ext| / 2.
 *   glisse_libration_read    phi_min[N], phi_max[N] (running extrema over all samples; +inf / -inf if
 *                            never sampled), amp_mean[N] (mean of the amplitude samples, NaN if
 *                            none), amp_max[N] (largest, 0 if none), n_amp[N] (their number), original
 *                            order, host or device, any may be NULL.  Synchronises.
 */
int glisse_resonance_begin(glisse_sim* sim, int planet, int p, int q, double window);
int glisse_resonance_sample(glisse_sim* sim);
int glisse_resonance_read(glisse_sim* sim, unsigned char* seen0, unsigned char* seen180, double* phi_last,
                          long long* n_samples);
int glisse_libration_read(glisse_sim* sim, double* phi_min, double* phi_max, double* amp_mean, double* amp_max,
                          int* n_amp);

/* Heliocentric planet positions and velocities at the current step, [n_planets][3] each, host
 * or device, either may be NULL.  Synchronises. */
int glisse_read_planets(glisse_sim* sim, double* pos, double* vel);

/* Number of particles with flag == 0 at the current step (synchronises); < 0 on error. */
long long glisse_active_count(glisse_sim* sim);

/* Number of steps completed since create (host counter, no synchronisation); < 0 on error. */
long long glisse_step(glisse_sim* sim);

/* Particle-steps actually integrated so far = Σ over steps of the number of particles that were
 * still active when the step began (the "useful work" of BASELINE.json's metric). Synchronises. */
long long glisse_particle_steps(glisse_sim* sim);

/* Block until all enqueued work of this sim has finished; returns its sticky status. */
int glisse_sync(glisse_sim* sim);

void glisse_destroy(glisse_sim* sim);

/*
 * One-shot run: glisse_create + glisse_advance(n_steps) + glisse_read + glisse_destroy over caller arrays
 * (host or device; pinned host arrays for the copies to overlap), PIPELINED over n_parts contiguous slices
 * of the particles.  Test particles never interact and the paper's own scaling strategy is
 * particles partitioned, planets replicated; here the partition is over time slots of one
 * GPU: each part is a simulation of its own (own planet-history kernel, same planets), part i+1 is
 * uploaded and part i read back while the kernels of the other parts run, so all but about one part's
 * share of the host<->device copies hides behind the integration.
 *   n_parts: 1 .. 64, or 0 = automatic (parts of about 2^17 particles, at most 8; one part below 2^18).
 *            Cuts fall on multiples of 256 particles.
 *   out_pos / out_vel / flag / removal_step: as glisse_read (each may be NULL), original particle order.
 *   particle_steps: if not NULL, receives the particle-steps integrated (sum over the parts).
 * The result of every particle is what a single simulation over all of them returns, bit for bit, when
 * params fixes guess_order (1 or 3); with guess_order = 0 each part chooses its Kepler starting point from
 * its own particles, as every rank of a multi-GPU run does (a roundoff-level difference).  Arguments and
 * statuses otherwise as glisse_create (a caller's params->stream is then shared by all parts, whose particle
 * kernels no longer overlap: leave it NULL here).  Synchronous.
 */
int glisse_run(double gm_star, int n_planets, const double* gm_planet, const double* planet_pos,
               const double* planet_vel, const double* planet_rcrit, long long n_particles,
               const double* const pos[3], const double* const vel[3], double dt, const glisse_params* params,
               long long n_steps, int n_parts, double* const out_pos[3], double* const out_vel[3], int* flag,
               long long* removal_step, long long* particle_steps);

/* Static string for a status code. */
const char* glisse_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* GLISSE_H_ */
