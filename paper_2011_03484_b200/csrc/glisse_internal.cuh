// glisse_internal.cuh — declarations shared by the translation units of libglisse (CUDA path only).
// Nothing here is used by, or derived from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/glisse.h"

namespace glisse {

constexpr int kMaxPlanets = GLISSE_MAX_PLANETS;
constexpr int kParticleBlock = 128;  // threads per particle-kernel block (one particle per thread)
constexpr int kRingStages = 3;       // planet-log ring buffers in shared memory per block

// Doubles per planet-log record (include/glisse.h: glisse_log_stride).
__host__ __device__ inline int log_stride(int np) { return (3 * (np + 1) + 1) & ~1; }

// Records per shared-memory ring stage: about 4 KB per stage.
inline int stage_records(int np) {
  int s = 4096 / (log_stride(np) * 8);
  if (s > 32) s = 32;
  if (s < 4) s = 4;
  return s;
}

// ---- arguments of the particle kernel (a2–a7), passed by value as a __grid_constant__ ----------
struct ParticleArgs {
  double* st[6];                       // x, y, z, vx, vy, vz  (struct of arrays, working order)
  int* flag;                           // 0 = active
  long long* rstep;                    // removal step
  const int* n_slots;                  // device: length of the working prefix in use
  const double* log;                   // (nsteps + 1) records of `stride` doubles
  unsigned long long* pstep_counter;   // device: += number of drifts started
  long long step0;                     // completed steps at record 0
  int nsteps;
  int stride;
  int stage_recs;
  int np;
  int iters;
  double dt, hdt, mu, inv_mu, rmin2, rmax2, tol;
  double gm[kMaxPlanets];
  double rc2[kMaxPlanets];
};

// ---- planet system constants + state, resident in device memory --------------------------------
struct PlanetSystem {
  int np;
  double gm0;
  double gm[kMaxPlanets];
  double eta[kMaxPlanets];       // eta_k = gm0 + sum_{i<=k} gm_i
  double eta_prev[kMaxPlanets];  // eta_{k-1}
  double rj[3 * kMaxPlanets];    // Jacobi positions   (persisted between chunks)
  double vj[3 * kMaxPlanets];    // Jacobi velocities
  int status;                    // 0, or 1-based index of the first planet whose drift failed
};

// launchers (each returns the cudaError_t of the launch)
cudaError_t launch_particle_kernel(const ParticleArgs& a, int n_slots_upper, cudaStream_t s);
cudaError_t launch_planet_kernel(PlanetSystem* sys, double* log, int nsteps, double dt, bool save_state,
                                 cudaStream_t s);
cudaError_t launch_planet_init(PlanetSystem* sys, const double* q, const double* qd, cudaStream_t s);
cudaError_t launch_planet_read(const PlanetSystem* sys, double* q, double* qd, cudaStream_t s);

struct CompactArgs {
  double* src[6];
  double* dst[6];
  double* fin[6];          // original order: frozen state of compacted-away particles
  int* src_id;  int* dst_id;
  int* src_flag; long long* src_rstep;
  int* fin_flag; long long* fin_rstep;
  int* n_slots;            // in: prefix length; out: number of survivors
  int* block_counts;       // scratch [ceil(n/256)]
};
cudaError_t launch_compaction(const CompactArgs& a, int n_slots_upper, cudaStream_t s, int* launches);

struct GatherArgs {
  const double* st[6];
  const int* id; const int* flag; const long long* rstep;
  const int* n_slots;
  double* out[6];          // original order, may be null individually
  int* out_flag; long long* out_rstep;
};
cudaError_t launch_scatter_to_original(const GatherArgs& a, int n_slots_upper, cudaStream_t s);
cudaError_t launch_count_active(const int* flag, const int* n_slots, int n_slots_upper, int* out, cudaStream_t s);
cudaError_t launch_init_ids(int* id, int* flag, long long* rstep, int n, cudaStream_t s);

cudaError_t run_fp64_probe(cudaStream_t s, double millis, double* flops);

}  // namespace glisse
