// glisse_internal.cuh — declarations shared by the translation units of libglisse (CUDA path only).
// Nothing here is used by, or derived from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/glisse.h"

namespace glisse {

constexpr int kMaxPlanets = GLISSE_MAX_PLANETS;
#ifndef GL_BLOCK
#define GL_BLOCK 32
#endif
#ifndef GL_PPT
#define GL_PPT 1
#endif
constexpr int kParticleBlock = GL_BLOCK;     // threads per particle-kernel block
constexpr int kParticlesPerThread = GL_PPT;  // particles per thread: the kernel as built supports 1 only
constexpr int kParticleWarps = kParticleBlock / 32;
constexpr int kRingSlots = 2;        // planet-log stages resident in shared memory per WARP
#ifndef GL_MIN_BLOCKS
#define GL_MIN_BLOCKS 20
#endif

// Doubles per planet-log record (include/glisse.h: glisse_log_stride).
__host__ __device__ inline int log_stride(int np) { return (3 * (np + 1) + 1) & ~1; }

// Records per shared-memory ring stage (one cp.async.bulk each): about 1 KB per stage.
inline int stage_records(int np) {
  int s = 1024 / (log_stride(np) * 8);
  if (s > 16) s = 16;
  if (s < 2) s = 2;
  return s;
}

// ---- arguments of the particle kernel (a2–a7), passed by value as a __grid_constant__ ----------
struct ParticleArgs {
  // Read by every step of the kernel, so laid out for 16-byte constant-bank loads: the scalars of the
  // drift first, then the kick's per-planet constants, each group on a 16-byte boundary.
  alignas(16) double mu;
  double inv_mu;
  double inv_mu_dt;
  double two_mu;                       // 2 mu
  double inv_mu_hdt;                   // (dt / 2) / mu: the half drifts of the drift-kick-drift scheme
  double hdt;
  alignas(16) double gm[kMaxPlanets];
  // high words of rc2[], rmin2, rmax2: the hot path's integer superset of the distance tests
  alignas(16) int rc2_hi[kMaxPlanets];
  alignas(16) int rmin2_hi;
  int rmax2_hi;
  // ---- the rest is read once per launch or in the removal blocks only
  double rmin2, rmax2, tol;
  double rc2[kMaxPlanets];
  double* st[6];                       // x, y, z, vx, vy, vz  (struct of arrays, working order)
  int* flag;                           // 0 = active
  long long* rstep;                    // removal step
  const int* n_slots;                  // device: length of the working prefix in use
  const double* log;                   // (nsteps + 1) records of `stride` doubles, 16-byte aligned
  unsigned long long* pstep_counter;   // device: += number of drifts started
  long long step0;                     // completed steps at record 0
  int nsteps;
  int stride;
  int stage_recs;
  int np;
  int iters;
  // Launch chaining: a chunk is issued as back-to-back launches of a few hundred steps
  // each, the later ones with programmatic stream serialisation, so that they become resident while
  // the earlier one drains.  A warp of launch j+1 takes the k-th group of 32 particles that launch j
  // COMPLETED (not a fixed one), so it never waits on a particular slow warp.
  int* wait_list;          // previous launch's completion list: entry k = group + 1, 0 = not yet; null = first
  int* done_list;          // this launch's completion list (zero on entry)
  unsigned* done_ticket;   // this launch's completion counter
  unsigned ticket_base;    // value of *done_ticket when this launch starts
  int* error;              // device word: != 0 once a chained warp gave up waiting (never expected)
  unsigned long long* solver_stats;  // [3] warp drift calls, fast-solver iterations, slow-path entries (STATS only)
};

// ---- planet system constants, resident in device memory -----------------------------------------
struct PlanetSystem {
  int np;
  double gm0;
  double gm[kMaxPlanets];
  double eta[kMaxPlanets];       // eta_k = gm0 + sum_{i<=k} gm_i
  double eta_prev[kMaxPlanets];  // eta_{k-1}
};
// A planet failure (drift unbound / not converged, GLISSE_EPLANET) is recorded as the absolute index
// of the first step whose drift failed, in a device word that starts at kNoPlanetFailure: records up
// to and including that step are valid, so the failure concerns the caller only once the particles
// have gone past it — a look-ahead chunk that fails does not poison the state already computed.
constexpr long long kNoPlanetFailure = 0x7fffffffffffffffLL;

// Jacobi state record: [r'_0 .. r'_{Np-1} | v'_0 .. v'_{Np-1}], 6·Np doubles.
inline int jstate_stride(int np) { return 6 * np; }

// launchers (each returns the cudaError_t of the launch); *launches += kernels launched
// chained: launch with programmatic stream serialisation behind the previous particle-kernel launch
// stats: the instrumented instantiation (glisse_test.h: glisse_solver_stats)
// dkd: the drift-kick-drift instantiation (include/glisse.h: GLISSE_SCHEME_DKD)
// refine: the instantiation with the third-order starting point of the Kepler solve (guess_order 3)
// definition_only: the instantiation without the fast solver (see fast_solver_allowed)
cudaError_t launch_particle_kernel(const ParticleArgs& a, int n_groups, bool chained, bool stats, bool dkd, bool refine,
                                   bool definition_only, cudaStream_t s);
// the one pass over the particles at create: identity order, cleared flags and removal steps (working and
// original order); counts[0] += non-finite bodies, counts[1] += bodies that would take the third-order
// starting point at this instant
cudaError_t launch_create_pass(const double* const st[6], long long n, double mu, double dt, unsigned long long* counts,
                               int* id, int* flag, long long* rstep, int* fin_flag, long long* fin_rstep,
                               cudaStream_t s);
cudaError_t configure_particle_kernels();
// whether kepler_iters / kepler_tol admit the fast solver (kepler.cuh: kFastMinIters, kFastMinTol); if not,
// the simulation uses the particle-kernel instantiation that carries the definition's solver alone
bool fast_solver_allowed(int kepler_iters, double kepler_tol);
int particles_per_group();

// Planet-history kernel (a1): from the Jacobi state `jin` write nsteps+1 log records and nsteps+1
// Jacobi state records (record 0 = the input state).  exclusive_sm_bytes > 0: dynamic
// shared memory to request (unused) so that no other block fits on its SM.
// fail_step: see kNoPlanetFailure; step0 = absolute step index of record 0.
cudaError_t launch_planet_kernel(const PlanetSystem* sys, int np, const double* jin, double* log, double* jlog,
                                 int nsteps, double dt, long long step0, long long* fail_step, int exclusive_sm_bytes,
                                 cudaStream_t s);
// allows the planet-history kernel the whole shared memory of an SM; returns that size in bytes
cudaError_t configure_planet_kernels(int* exclusive_sm_bytes);
// heliocentric (q, qd) [np][3] -> Jacobi state record
cudaError_t launch_planet_init(const PlanetSystem* sys, const double* q, const double* qd, double* jstate,
                               cudaStream_t s);
// Jacobi state record -> heliocentric q, qd [np][3] (either may be null)
cudaError_t launch_planet_read(const PlanetSystem* sys, const double* jstate, double* q, double* qd,
                               cudaStream_t s);

// The same kernel with its Jacobi-state scratch in a file-scope static __device__ array (planets.cu) instead of
// caller memory: kStaticJlogDoubles doubles per device, shared by every call on that device.
constexpr size_t kStaticJlogDoubles = size_t(1) << 18;   // 2 MiB
// largest nsteps the static scratch holds for np planets (-1: np out of range)
long long static_planet_log_limit(int np);
cudaError_t launch_planet_kernel_static(const PlanetSystem* sys, int np, const double* jin, double* log, int nsteps,
                                        double dt, long long step0, long long* fail_step, cudaStream_t s);

// planet log records by cubic Hermite interpolation of a sparse history (all pointers device)
cudaError_t launch_interpolate_log(const PlanetSystem* sys, long long n_samples, const double* sample_time,
                                   const double* sample_pos, const double* sample_vel, double t_first, double dt_record,
                                   long long n_records, double* log, cudaStream_t s);

struct CompactArgs {
  const double* src[6];
  double* dst[6];
  double* fin[6];          // original order: frozen state of compacted-away particles
  const int* src_id;  int* dst_id;
  const int* src_flag; const long long* src_rstep;
  int* dst_flag; long long* dst_rstep;
  int* fin_flag; long long* fin_rstep;
  const int* n_in;         // prefix length of src
  int* n_out;              // number of survivors = prefix length of dst
  int* n_out_host;         // mapped pinned word that receives the same count (or null)
  int* block_counts;       // scratch [kCompactBins * ceil(n_upper/256) + 1]
  // iteration-count binning (include/glisse.h bin_iterations): bins > 1 orders the
  // survivors by bin (hardest first), particle order within a bin
  unsigned char* bin;      // scratch [n_upper]: bin of every slot (written by the count pass)
  int bins;                // 1 = plain stable partition, kCompactBins = binned
  double mu, dt;           // for the hardness key
  int refine;              // the run uses the third-order Kepler starting point (kepler.cuh)
};
constexpr int kCompactBins = 3;
cudaError_t launch_compaction(const CompactArgs& a, int n_slots_upper, cudaStream_t s, long long* launches);

struct ScatterArgs {
  const double* st[6];
  const int* id; const int* flag; const long long* rstep;
  const int* n_slots;
  double* fin[6];          // original order
  int* fin_flag; long long* fin_rstep;
};
cudaError_t launch_scatter_to_original(const ScatterArgs& a, int n_slots_upper, cudaStream_t s);
cudaError_t launch_count_active(const int* flag, const int* n_slots, int n_slots_upper,
                                unsigned long long* out, cudaStream_t s);

// snapshot.cu: ONE pass over the original-order arrays that serves the snapshot (staging copy,
// Cartesian or osculating elements) and the resonant-argument reduction of the same instant: the
// elements are computed once for both.
struct LibrationRecord {     // per particle, original order (include/glisse.h: glisse_libration_read)
  double* phi;              // last value of the argument, [0, 2 pi)
  unsigned char* seen0;     // phi has been within `window` of 0
  unsigned char* seen180;   // phi has been within `window` of pi
  double* phi_min;          // running extrema of phi
  double* phi_max;
  double* ext_last;         // value of the latest turning point
  double* amp_sum;          // sum and maximum of the amplitude samples |ext - previous ext| / 2
  double* amp_max;
  int* n_amp;               // number of amplitude samples
  int* n_seen;              // samples this particle has taken
  signed char* trend;       // +1 rising, -1 falling, 0 unknown
  signed char* ext_kind;    // +1 the latest turning point was a maximum, -1 a minimum, 0 none yet
};
struct SampleArgs {
  const double* fin[6];
  const int* fin_flag; const long long* fin_rstep;
  long long n;
  double mu;
  // snapshot part (do_snapshot)
  int do_snapshot, kind;
  long long step;           // written to *step_out (if not null) by the pass: the snapshot's step count
  long long* step_out;
  double* out[6];
  int* out_flag; long long* out_rstep;
  // resonance part (do_resonance)
  int do_resonance, p, q;
  const double* planet_q;   // [3] heliocentric position of the planet at the current step (device)
  const double* planet_qd;  // [3] velocity
  double mu_planet, window;
  LibrationRecord lib;
};
cudaError_t launch_sample(const SampleArgs& a, cudaStream_t s);
cudaError_t launch_libration_reset(const LibrationRecord& lib, long long n, cudaStream_t s);
// amp_mean[n] = amp_sum / n_amp (NaN where n_amp = 0)
cudaError_t launch_libration_mean(const LibrationRecord& lib, double* amp_mean, long long n, cudaStream_t s);

cudaError_t run_fp64_probe(cudaStream_t s, double millis, double* flops);
cudaError_t run_primitive(int which, long long n, const double* in, double* out, cudaStream_t s);

}  // namespace glisse
