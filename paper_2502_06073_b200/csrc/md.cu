// md.cu — row a-6: velocity-Verlet NVE (kick-drift-kick) with skin-triggered neighbour-list rebuilds, all on
// the device.  PAPER.md:89 ("explicit reversible integrator"), PAPER.md:116 (0.5 fs step); readings A20-A22.
// Units: a[A/fs^2] = 9.648533212e-3 * F[eV/A] / m[amu].  The rebuild decision is a device flag: the rebuild
// kernels are enqueued every step and return at once when the flag is clear, so the step loop has no host sync.
#include <algorithm>

#include "model.h"

namespace allegro {
namespace {

constexpr double ACC_CONV = 9.648533212e-3;

__global__ void k_kick_drift(double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ F,
                             const double* __restrict__ mass, int64_t N, double dt, int drift, const int* flags) {
  if (flags[FLAG_HALT]) return;   // a rebuild ran out of capacity earlier in this call: the host finishes the step (md_step)
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 3 * N) return;
  const int64_t i = idx / 3;
  double v = vel[idx] + 0.5 * dt * ACC_CONV * F[idx] / mass[i];
  vel[idx] = v;
  if (drift) pos[idx] += dt * v;
}

// A22: rebuild when max_i |r_i - r_i^build| > skin/2 (skin = 0: always)
__global__ void k_skin_test(const double* __restrict__ pos, const double* __restrict__ r_build, int64_t N, double half_skin2,
                            int always, int* flags) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || flags[FLAG_HALT]) return;
  if (always) { if (i == 0) flags[FLAG_REBUILD] = 1; return; }
  // same rounding as the oracle's test (no FMA contraction), so that the rebuild decisions agree
  const double dx = __dsub_rn(pos[3 * i], r_build[3 * i]), dy = __dsub_rn(pos[3 * i + 1], r_build[3 * i + 1]), dz = __dsub_rn(pos[3 * i + 2], r_build[3 * i + 2]);
  if (__dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)) > half_skin2) flags[FLAG_REBUILD] = 1;
}

// end of a step: count it unless the integrator is halted
__global__ void k_step_done(int* flags) { if (!flags[FLAG_HALT]) flags[FLAG_STEPS] += 1; }

// Berendsen weak coupling after the second half-kick of step k (reading A25; PAPER.md:49, :116 NVT, :75 heating ramp):
// T_inst = 2 E_kin / ((3N - 3) kB), T_target = T0 + (T1 - T0) min(1, k / n_ramp), v <- v sqrt(1 + (dt / tau)(T_target / T_inst - 1)).
// par = {T0, T1, n_ramp, tau}; k = completed steps of this call + 1.
__global__ void k_berendsen(double* __restrict__ vel, int64_t N, const double* __restrict__ ekin, const double* __restrict__ par, double dt,
                            const int* flags) {
  if (flags[FLAG_HALT]) return;
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 3 * N) return;
  const double kB = 8.617333262e-5;
  const double T_inst = 2.0 * ekin[0] / ((double)(3 * N - 3) * kB);
  const double k = (double)(flags[FLAG_STEPS] + 1);
  const double frac = par[2] > 0.0 ? fmin(1.0, k / par[2]) : 1.0;
  const double T_tgt = par[0] + (par[1] - par[0]) * frac;
  vel[idx] *= sqrt(1.0 + (dt / par[3]) * (T_tgt / T_inst - 1.0));
}

__global__ void k_scale_pos(double* __restrict__ pos, int64_t N, double sx, double sy, double sz) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 3 * N) return;
  const int d = (int)(idx % 3);
  pos[idx] *= (d == 0 ? sx : (d == 1 ? sy : sz));
}

// general cell: x' = x A with A = H^-1 H' (fractional coordinates kept), (x_0 A_0b + x_1 A_1b) + x_2 A_2b
struct Affine { double A[9]; };
__global__ void k_affine_pos(double* __restrict__ pos, int64_t N, Affine af) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
#pragma unroll
  for (int b = 0; b < 3; ++b) pos[3 * i + b] = __dadd_rn(__dadd_rn(__dmul_rn(x, af.A[b]), __dmul_rn(y, af.A[3 + b])), __dmul_rn(z, af.A[6 + b]));
}

__global__ void k_clear_flag(int* flags, int which) { flags[which] = 0; }

__global__ void k_kinetic_partial(const double* __restrict__ vel, const double* __restrict__ mass, int64_t N, double* __restrict__ partial) {
  __shared__ double sh[256];
  double s = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x)
    s += mass[i] * (vel[3 * i] * vel[3 * i] + vel[3 * i + 1] * vel[3 * i + 1] + vel[3 * i + 2] * vel[3 * i + 2]);
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int d = 128; d > 0; d >>= 1) {
    if (threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void k_kinetic_final(const double* __restrict__ partial, int nb, double* __restrict__ out) {
  __shared__ double sh[256];
  double s = 0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) s += partial[i];
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int d = 128; d > 0; d >>= 1) {
    if (threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = 0.5 * sh[0] / ACC_CONV;
}

}  // namespace

void md_graph_reset(Model* m);

int md_init(Model* m, const double* pos, const double* vel, const double* mass, const int32_t* species, int64_t N,
            const double* cell, double cutoff, double skin, cudaStream_t st) {
  int rc = 0;
  rc |= ensure(m, &m->md_pos, sizeof(double) * 3 * N + 8);
  rc |= ensure(m, &m->md_vel, sizeof(double) * 3 * N + 8);
  rc |= ensure(m, &m->md_F, sizeof(double) * 3 * N + 8);
  rc |= ensure(m, &m->md_mass, sizeof(double) * N + 8);
  rc |= ensure(m, &m->md_species, sizeof(int32_t) * N + 8);
  rc |= ensure(m, &m->md_E, sizeof(double) * 16);
  if (rc) return ALLEGRO_ERR_ALLOC;
  cudaMemcpyAsync(m->md_pos.p, pos, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(m->md_vel.p, vel, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(m->md_mass.p, mass, sizeof(double) * N, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(m->md_species.p, species, sizeof(int32_t) * N, cudaMemcpyDeviceToDevice, st);
  for (int k = 0; k < 9; ++k) m->md_cell[k] = cell[k];
  md_graph_reset(m);   // buffers may move: the captured step is rebuilt on the next allegro_md_step
  if ((rc = nl_build(m, m->md_pos.as<double>(), N, cell, cutoff, skin, false, st))) return rc;
  m->nl.n_rebuilds = 0;
  if ((rc = network_energy_forces(m, m->md_pos.as<double>(), m->md_species.as<int32_t>(), N, m->md_E.as<double>(),
                                  m->md_F.as<double>(), nullptr, st)))
    return rc;
  m->md_ready = true;
  return 0;
}

// One velocity-Verlet step enqueued on st (no host synchronisation: the rebuild decision is a device flag).
// second_half_only finishes a step whose kick + drift already happened (capacity recovery, see md_step).
static int md_one_step(Model* m, double dt, bool nvt, cudaStream_t st, bool second_half_only = false) {
  NeighborList& nl = m->nl;
  const int64_t N = nl.N;
  int* flags = m->flags.as<int>();
  double* pos = m->md_pos.as<double>();
  double* vel = m->md_vel.as<double>();
  double* F = m->md_F.as<double>();
  const int T = 256;
  const unsigned g3 = (unsigned)((3 * N + T - 1) / T), g1 = (unsigned)((N + T - 1) / T);
  const double hs = 0.5 * nl.skin;
  if (!second_half_only) {
    prof_begin(m, st, KC_MD, 0);
    k_kick_drift<<<g3, T, 0, st>>>(pos, vel, F, m->md_mass.as<double>(), N, dt, 1, flags);
    k_skin_test<<<g1, T, 0, st>>>(pos, nl.r_build.as<double>(), N, hs * hs, nl.skin == 0.0 ? 1 : 0, flags);
    prof_end(m, st);
    m->launches += 2;
    prof_begin(m, st, KC_NEIGHBOR, 0);
    if (int rc = nl_build(m, pos, N, m->md_cell, nl.cutoff, nl.skin, true, st)) return rc;
    k_clear_flag<<<1, 1, 0, st>>>(flags, FLAG_REBUILD);
    prof_end(m, st);
  }
  if (int rc = network_energy_forces(m, pos, m->md_species.as<int32_t>(), N, m->md_E.as<double>(), F, nullptr, st)) return rc;
  prof_begin(m, st, KC_MD, 0);
  k_kick_drift<<<g3, T, 0, st>>>(pos, vel, F, m->md_mass.as<double>(), N, dt, 0, flags);
  m->launches += 2;
  if (nvt && N > 1) {
    if (int rc = md_kinetic(m, m->md_E.as<double>() + 1, st)) return rc;
    k_berendsen<<<g3, T, 0, st>>>(vel, N, m->md_E.as<double>() + 1, m->nvt_par.as<double>(), dt, flags);
    m->launches += 3;
  }
  k_step_done<<<1, 1, 0, st>>>(flags);
  prof_end(m, st);
  m->launches += 1;
  return 0;
}

void md_graph_reset(Model* m) {
  if (m->md_graph) { cudaGraphExecDestroy(m->md_graph); m->md_graph = nullptr; }
  m->md_warm = false;
}

// Enqueue n_steps steps.  The step is a fixed sequence of launches (conditional rebuild included), so after one plain step
// (which performs every allocation and weight packing) it is captured once into a CUDA graph and replayed: the host cost
// per step drops from ~50 launches to one cudaGraphLaunch.  Profiling runs (allegro_profile) use the plain path.  The
// legacy default stream cannot be captured: an internal blocking stream, which the legacy stream orders itself with
// implicitly, carries the work instead.
static int md_enqueue(Model* m, double dt, int64_t n_steps, bool nvt, cudaStream_t* stp) {
  cudaStream_t st = *stp;
  if (n_steps > 0 && m->use_graph && !m->prof.on && n_steps >= 2) {
    if (st == nullptr) {
      if (!m->own_stream && cudaStreamCreate(&m->own_stream) != cudaSuccess) { cudaGetLastError(); m->own_stream = nullptr; }
      if (m->own_stream) st = m->own_stream;
    }
    *stp = st;
    if (st != nullptr) {
      if (!m->md_warm) {
        if (int rc = md_one_step(m, dt, nvt, st)) return rc;
        m->md_warm = true;
        --n_steps;
      }
      if (!m->md_graph || m->graph_dt != dt || m->graph_stream != st || m->graph_nvt != (int)nvt) {
        if (m->md_graph) { cudaGraphExecDestroy(m->md_graph); m->md_graph = nullptr; }
        const int64_t l0 = m->launches;
        cudaGraph_t g = nullptr;
        int rc = 0;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
          rc = md_one_step(m, dt, nvt, st);
          cudaError_t ce = cudaStreamEndCapture(st, &g);
          if (rc == 0 && ce == cudaSuccess && g && cudaGraphInstantiate(&m->md_graph, g, 0) == cudaSuccess) {
            m->graph_dt = dt; m->graph_stream = st; m->graph_nvt = (int)nvt; m->graph_launches = m->launches - l0;
          } else {
            m->md_graph = nullptr;
          }
          if (g) cudaGraphDestroy(g);
        }
        cudaGetLastError();
        m->launches = l0;
        if (rc) return rc;
      }
      if (m->md_graph) {
        for (int64_t s = 0; s < n_steps; ++s) {
          if (cudaGraphLaunch(m->md_graph, st) != cudaSuccess) return cuda_fail(m, cudaGetLastError(), "cudaGraphLaunch");
          m->launches += m->graph_launches;
        }
        return 0;
      }
    }
  }
  for (int64_t s = 0; s < n_steps; ++s)
    if (int rc = md_one_step(m, dt, nvt, st)) return rc;
  return 0;
}

// n_steps steps of NVE (nvt == NULL) or Berendsen NVT.  When a device-side rebuild (or the activation workspace of a chunk)
// runs out of capacity, the integrator kernels of the remaining steps do nothing (FLAG_HALT) and FLAG_STEPS holds the number
// of completed steps; the halted step has had its kick + drift.  The host then rebuilds the list with fresh capacity at the
// current positions, finishes that step (forces, second half-kick, thermostat) and enqueues the rest: the trajectory is the
// one an unbounded list would have given.
int md_step(Model* m, double dt, int64_t n_steps, const double* nvt, cudaStream_t st) {
  int* flags = m->flags.as<int>();
  if (nvt) {
    if (int rc = ensure(m, &m->nvt_par, sizeof(double) * 4)) return rc;
    cudaMemcpyAsync(m->nvt_par.p, nvt, sizeof(double) * 4, cudaMemcpyHostToDevice, st);
    cudaStreamSynchronize(st);   // nvt is a caller buffer
  }
  cudaMemsetAsync(flags + FLAG_STEPS, 0, sizeof(int), st);
  int64_t left = n_steps;
  m->stats[4] = 0;
  for (int attempt = 0; attempt < 8 && left > 0; ++attempt) {
    if (attempt > 0 && st == nullptr && m->own_stream) cudaStreamSynchronize(m->own_stream);
    cudaStream_t run = st;
    if (int rc = md_enqueue(m, dt, left, nvt != nullptr, &run)) return rc;
    int h[FLAG_COUNT];
    cudaError_t e = cudaMemcpyAsync(h, flags, sizeof(h), cudaMemcpyDeviceToHost, run);
    if (e == cudaSuccess) e = cudaStreamSynchronize(run);
    if (e != cudaSuccess) return cuda_fail(m, e, "allegro_md_step");
    m->stats[4] = h[FLAG_STEPS];
    if (!h[FLAG_HALT]) return 0;
    // ---- capacity recovery
    const int64_t done = h[FLAG_STEPS];
    if (h[FLAG_ERR_CAP] == 2) m->ws.slack *= 1.5;            // a chunk held more active edges than its share of the list
    else { m->nl.slack_frac = std::max(0.125, 2.0 * m->nl.slack_frac); m->nl.slack_extra = std::max<int64_t>(4096, m->nl.slack_extra); }
    m->ws.for_N = -1;                                        // re-size the workspace for the new capacities
    int zero3[2] = {0, 0};
    cudaMemcpyAsync(flags + FLAG_ERR_CAP, zero3, sizeof(int), cudaMemcpyHostToDevice, run);
    cudaMemcpyAsync(flags + FLAG_HALT, zero3, sizeof(int), cudaMemcpyHostToDevice, run);
    cudaMemcpyAsync(flags + FLAG_STALE, zero3, sizeof(int), cudaMemcpyHostToDevice, run);
    cudaMemcpyAsync(flags + FLAG_NONFINITE, zero3, sizeof(int), cudaMemcpyHostToDevice, run);
    md_graph_reset(m);                                        // buffers move
    if (int rc = nl_build(m, m->md_pos.as<double>(), m->nl.N, m->md_cell, m->nl.cutoff, m->nl.skin, false, run)) return rc;
    if (int rc = md_one_step(m, dt, nvt != nullptr, run, true)) return rc;
    m->md_warm = true;
    left = n_steps - done - 1;
    m->stats[6] += 1;                                         // capacity recoveries
  }
  if (left > 0) {
    int h[FLAG_COUNT];
    cudaMemcpy(h, flags, sizeof(h), cudaMemcpyDeviceToHost);
    if (h[FLAG_HALT]) { m->err = "neighbour list capacity could not be recovered"; return ALLEGRO_ERR_ALLOC; }
    m->stats[4] = h[FLAG_STEPS];
  }
  return 0;
}

// A26: affine remap of the MD state to a new cell (x' = x L'/L; x' = x H^-1 H' when either cell is not orthorhombic), full list
// rebuild, forces re-evaluated.
int md_deform(Model* m, const double* cell_new, cudaStream_t st) {
  const int64_t N = m->nl.N;
  bool diag = true;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      if (a != b && (cell_new[3 * a + b] != 0.0 || m->md_cell[3 * a + b] != 0.0)) diag = false;
  if (diag) {
    double sc[3];
    for (int d = 0; d < 3; ++d) {
      if (!(cell_new[4 * d] > 0.0)) { m->err = "cell lengths must be positive"; return ALLEGRO_ERR_INVALID; }
      sc[d] = cell_new[4 * d] / m->md_cell[4 * d];
    }
    if (N > 0) k_scale_pos<<<(unsigned)((3 * N + 255) / 256), 256, 0, st>>>(m->md_pos.as<double>(), N, sc[0], sc[1], sc[2]);
  } else {
    const double* Hi = m->nl.Hinv;                      // inverse of the current cell (the list was built with it)
    Affine af;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) af.A[3 * a + b] = (Hi[3 * a] * cell_new[b] + Hi[3 * a + 1] * cell_new[3 + b]) + Hi[3 * a + 2] * cell_new[6 + b];
    if (N > 0) k_affine_pos<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(m->md_pos.as<double>(), N, af);
  }
  for (int k = 0; k < 9; ++k) m->md_cell[k] = cell_new[k];
  md_graph_reset(m);
  if (int rc = nl_build(m, m->md_pos.as<double>(), N, m->md_cell, m->nl.cutoff, m->nl.skin, false, st)) return rc;
  return network_energy_forces(m, m->md_pos.as<double>(), m->md_species.as<int32_t>(), N, m->md_E.as<double>(), m->md_F.as<double>(), nullptr, st);
}

// checkpoint / resume: new positions and velocities for the masses, species and cell of allegro_md_init
int md_set_state(Model* m, const double* pos, const double* vel, cudaStream_t st) {
  const int64_t N = m->nl.N;
  cudaMemcpyAsync(m->md_pos.p, pos, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(m->md_vel.p, vel, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  md_graph_reset(m);
  if (int rc = nl_build(m, m->md_pos.as<double>(), N, m->md_cell, m->nl.cutoff, m->nl.skin, false, st)) return rc;
  return network_energy_forces(m, m->md_pos.as<double>(), m->md_species.as<int32_t>(), N, m->md_E.as<double>(), m->md_F.as<double>(), nullptr, st);
}

int md_kinetic(Model* m, double* Ekin_dev, cudaStream_t st) {
  const int64_t N = m->nl.N;
  if (int rc = ensure(m, &m->e_partial, sizeof(double) * 1024)) return rc;
  const int nb = (int)std::max<int64_t>(1, std::min<int64_t>(1024, (N + 255) / 256));
  k_kinetic_partial<<<nb, 256, 0, st>>>(m->md_vel.as<double>(), m->md_mass.as<double>(), N, m->e_partial.as<double>());
  k_kinetic_final<<<1, 256, 0, st>>>(m->e_partial.as<double>(), nb, Ekin_dev);
  return 0;
}

}  // namespace allegro
