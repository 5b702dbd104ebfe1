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
                             const double* __restrict__ mass, int64_t N, double dt, int drift) {
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
  if (i >= N) return;
  if (always) { if (i == 0) flags[FLAG_REBUILD] = 1; return; }
  const double dx = pos[3 * i] - r_build[3 * i], dy = pos[3 * i + 1] - r_build[3 * i + 1], dz = pos[3 * i + 2] - r_build[3 * i + 2];
  if (dx * dx + dy * dy + dz * dz > half_skin2) flags[FLAG_REBUILD] = 1;
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
  rc |= ensure(m, &m->md_E, sizeof(double) * 4);
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
static int md_one_step(Model* m, double dt, cudaStream_t st) {
  NeighborList& nl = m->nl;
  const int64_t N = nl.N;
  int* flags = m->flags.as<int>();
  double* pos = m->md_pos.as<double>();
  double* vel = m->md_vel.as<double>();
  double* F = m->md_F.as<double>();
  const int T = 256;
  const unsigned g3 = (unsigned)((3 * N + T - 1) / T), g1 = (unsigned)((N + T - 1) / T);
  const double hs = 0.5 * nl.skin;
  prof_begin(m, st, KC_MD, 0);
  k_kick_drift<<<g3, T, 0, st>>>(pos, vel, F, m->md_mass.as<double>(), N, dt, 1);
  k_skin_test<<<g1, T, 0, st>>>(pos, nl.r_build.as<double>(), N, hs * hs, nl.skin == 0.0 ? 1 : 0, flags);
  prof_end(m, st);
  m->launches += 2;
  prof_begin(m, st, KC_NEIGHBOR, 0);
  if (int rc = nl_build(m, pos, N, m->md_cell, nl.cutoff, nl.skin, true, st)) return rc;
  k_clear_flag<<<1, 1, 0, st>>>(flags, FLAG_REBUILD);
  prof_end(m, st);
  if (int rc = network_energy_forces(m, pos, m->md_species.as<int32_t>(), N, m->md_E.as<double>(), F, nullptr, st)) return rc;
  prof_begin(m, st, KC_MD, 0);
  k_kick_drift<<<g3, T, 0, st>>>(pos, vel, F, m->md_mass.as<double>(), N, dt, 0);
  prof_end(m, st);
  m->launches += 2;
  return 0;
}

void md_graph_reset(Model* m) {
  if (m->md_graph) { cudaGraphExecDestroy(m->md_graph); m->md_graph = nullptr; }
  m->md_warm = false;
}

// n_steps steps.  The step is a fixed sequence of launches (conditional rebuild included), so after one plain step
// (which performs every allocation and weight packing) it is captured once into a CUDA graph and replayed: the host
// cost per step drops from ~50 launches to one cudaGraphLaunch.  Profiling runs (allegro_profile) and
// ALLEGRO_GRAPH=0 use the plain path.  The legacy default stream cannot be captured: an internal blocking stream,
// which the legacy stream orders itself with implicitly, carries the work instead.
int md_step(Model* m, double dt, int64_t n_steps, cudaStream_t st) {
  if (n_steps > 0 && m->use_graph && !m->prof.on && n_steps >= 2) {
    if (st == nullptr) {
      if (!m->own_stream && cudaStreamCreate(&m->own_stream) != cudaSuccess) { cudaGetLastError(); m->own_stream = nullptr; }
      if (m->own_stream) st = m->own_stream;
    }
    if (st != nullptr) {
      if (!m->md_warm) {
        if (int rc = md_one_step(m, dt, st)) return rc;
        m->md_warm = true;
        --n_steps;
      }
      if (!m->md_graph || m->graph_dt != dt || m->graph_stream != st) {
        if (m->md_graph) { cudaGraphExecDestroy(m->md_graph); m->md_graph = nullptr; }
        const int64_t l0 = m->launches;
        cudaGraph_t g = nullptr;
        int rc = 0;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed) == cudaSuccess) {
          rc = md_one_step(m, dt, st);
          cudaError_t ce = cudaStreamEndCapture(st, &g);
          if (rc == 0 && ce == cudaSuccess && g && cudaGraphInstantiate(&m->md_graph, g, 0) == cudaSuccess) {
            m->graph_dt = dt; m->graph_stream = st; m->graph_launches = m->launches - l0;
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
        m->stats[4] += n_steps;
        return 0;
      }
    }
  }
  for (int64_t s = 0; s < n_steps; ++s)
    if (int rc = md_one_step(m, dt, st)) return rc;
  m->stats[4] += n_steps;
  return 0;
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
