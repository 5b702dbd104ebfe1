// api.cu — the C-ABI entry points declared in include/allegro.h (argument checking, ownership, error codes).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "gemm.cuh"
#include "model.h"
#include "tp_gen.cuh"

namespace allegro {

static thread_local std::string g_create_err;

int ensure(Model* m, DevBuf* b, size_t bytes) {
  if (bytes <= b->bytes && b->p) return 0;
  if (b->p) { cudaFree(b->p); b->p = nullptr; b->bytes = 0; }
  md_graph_reset(m);   // a captured MD step holds the old pointer
  bytes = (bytes + 255) / 256 * 256;
  cudaError_t e = cudaMalloc(&b->p, bytes);
  if (e != cudaSuccess) {
    cudaGetLastError();
    m->err = std::string("device allocation of ") + std::to_string(bytes) + " bytes failed: " + cudaGetErrorString(e);
    b->p = nullptr;
    return ALLEGRO_ERR_ALLOC;
  }
  b->bytes = bytes;
  return 0;
}

int cuda_fail(Model* m, cudaError_t e, const char* what) {
  m->err = std::string(what) + ": " + cudaGetErrorString(e);
  return ALLEGRO_ERR_CUDA;
}

void prof_begin(Model* m, cudaStream_t st, int cls, double work) {
  Prof& p = m->prof;
  if (!p.on) return;
  if (2 * p.used + 2 > p.ev.size()) {
    for (int k = 0; k < 2; ++k) { cudaEvent_t e; cudaEventCreate(&e); p.ev.push_back(e); }
    p.cls.push_back(cls);
  }
  p.cls[p.used] = cls;
  p.work[cls] += work;
  p.launches[cls] += 1;
  cudaEventRecord(p.ev[2 * p.used], st);
}
void prof_end(Model* m, cudaStream_t st) {
  Prof& p = m->prof;
  if (!p.on) return;
  cudaEventRecord(p.ev[2 * p.used + 1], st);
  p.used += 1;
}
static void prof_collect(Model* m) {
  Prof& p = m->prof;
  for (size_t k = 0; k < p.used; ++k) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, p.ev[2 * k], p.ev[2 * k + 1]) == cudaSuccess) p.ms[p.cls[k]] += ms;
  }
  p.used = 0;
}

static void free_buf(DevBuf& b) { if (b.p) cudaFree(b.p); b.p = nullptr; b.bytes = 0; }

static int check_flags(Model* m, cudaStream_t st, const char* what) {
  int h[FLAG_COUNT];
  cudaError_t e = cudaMemcpyAsync(h, m->flags.p, sizeof(h), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(m, e, what);
  m->nl.n_rebuilds = h[FLAG_NREBUILD];
  int rc = 0;
  if (h[FLAG_ERR_SHIFT]) { m->err = "neighbour list: periodic image shift outside int8 range or asymmetric list"; rc = ALLEGRO_ERR_UNSUPPORTED; }
  else if (h[FLAG_ERR_CAP]) { m->err = "neighbour list / workspace capacity exceeded during a device-side rebuild"; rc = ALLEGRO_ERR_ALLOC; }
  else if (h[FLAG_SPECIES]) { m->err = "species index outside [0, n_species)"; rc = ALLEGRO_ERR_SPECIES; }
  else if (h[FLAG_STALE]) { m->err = "stale neighbour list: an atom moved more than skin/2 since allegro_build_neighbors"; rc = ALLEGRO_ERR_STALE_LIST; }
  else if (h[FLAG_NONFINITE]) { m->err = "NaN/Inf detected in energy or forces"; rc = ALLEGRO_ERR_NONFINITE; }
  if (rc) {   // clear the sticky error flags (keep the rebuild counter)
    int keep = h[FLAG_NREBUILD];
    cudaMemsetAsync(m->flags.p, 0, sizeof(int) * FLAG_COUNT, st);
    cudaMemcpyAsync(m->flags.as<int>() + FLAG_NREBUILD, &keep, sizeof(int), cudaMemcpyHostToDevice, st);
    cudaStreamSynchronize(st);
  }
  return rc;
}

}  // namespace allegro

using namespace allegro;

extern "C" {

int allegro_weight_layout(const allegro_hparams* hp, int32_t* kind, int64_t* rows, int64_t* cols, int max_tensors) {
  if (!hp) return ALLEGRO_ERR_INVALID;
  Plan P;
  std::string e = build_plan(*hp, &P);
  if (!e.empty()) { g_create_err = e; return ALLEGRO_ERR_INVALID; }
  const int nt = (int)P.lay_kind.size();
  for (int t = 0; t < nt && t < max_tensors; ++t) {
    if (kind) kind[t] = P.lay_kind[t];
    if (rows) rows[t] = P.lay_rows[t];
    if (cols) cols[t] = P.lay_cols[t];
  }
  return nt;
}

int allegro_debug_coupling(int l1, int l2, int l3, double* out) {
  if (!out || l1 < 0 || l2 < 0 || l3 < 0 || l1 > 3 || l2 > 3 || l3 > 3) return ALLEGRO_ERR_INVALID;
  std::vector<double> C = coupling_tensor(l1, l2, l3);
  std::memcpy(out, C.data(), sizeof(double) * C.size());
  return (int)C.size();
}

int allegro_debug_num_paths(const allegro_hparams* hp, int layer) {
  if (!hp) return ALLEGRO_ERR_INVALID;
  Plan P;
  std::string e = build_plan(*hp, &P);
  if (!e.empty()) { g_create_err = e; return ALLEGRO_ERR_INVALID; }
  if (layer < 1 || layer > hp->n_layers) return ALLEGRO_ERR_INVALID;
  return (int)P.layers[layer - 1].paths.size();
}

int allegro_create(const float* weights_host, size_t n_weights, const allegro_hparams* hp, void** handle_out) {
  if (!weights_host || !hp || !handle_out) { g_create_err = "null argument"; return ALLEGRO_ERR_INVALID; }
  *handle_out = nullptr;
  Model* m = new (std::nothrow) Model();
  if (!m) { g_create_err = "out of host memory"; return ALLEGRO_ERR_ALLOC; }
  std::string e = build_plan(*hp, &m->plan);
  if (!e.empty()) { g_create_err = "bad hyper-parameters: " + e; delete m; return ALLEGRO_ERR_INVALID; }
  const Plan& P = m->plan;
  if ((int64_t)n_weights != P.n_weights) {
    g_create_err = "weight blob has " + std::to_string(n_weights) + " floats, plan needs " + std::to_string(P.n_weights);
    delete m; return ALLEGRO_ERR_INVALID;
  }
  if (hp->n_channels % 4 != 0) { g_create_err = "n_channels must be a multiple of 4"; delete m; return ALLEGRO_ERR_UNSUPPORTED; }
  if (hp->n_channels > 256) { g_create_err = "n_channels must be <= 256"; delete m; return ALLEGRO_ERR_UNSUPPORTED; }
  if (hp->n_channels * P.d_sh > 4096) { g_create_err = "n_channels * (lmax+1)^2 must be <= 4096"; delete m; return ALLEGRO_ERR_UNSUPPORTED; }
  if (hp->two_body_nl < 2 || hp->latent_nl < 2) { g_create_err = "two-body and latent MLPs need >= 2 linear layers"; delete m; return ALLEGRO_ERR_UNSUPPORTED; }
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    g_create_err = std::string("no CUDA device (there is no CPU fallback): ") + cudaGetErrorString(ce);
    delete m; return ALLEGRO_ERR_CUDA;
  }
  cudaGetDevice(&m->device);
  m->use_big = m->use_tc && m->use_tp3 && (hp->n_channels == 64 || hp->n_channels == 128 || hp->n_channels == 256);
  cudaDeviceGetAttribute(&m->num_sms, cudaDevAttrMultiProcessorCount, m->device);
  virial_noalloc_setup(m);   // address lookup only; a failure is reported by allegro_virial_noalloc itself
  auto fail = [&](int rc, const std::string& msg) { g_create_err = msg; allegro_destroy(m); return rc; };
  if (cudaMalloc(&m->d_w, sizeof(float) * std::max<size_t>(n_weights, 1)) != cudaSuccess) return fail(ALLEGRO_ERR_ALLOC, "weights allocation failed");
  {
    // device copy of the blob with the rows of W_init / W_env^L reordered from (c, l) to (l, c): the kernels keep
    // the channel index fastest in every per-edge tensor (tp.cuh)
    std::vector<float> wd(weights_host, weights_host + n_weights);
    const int nl1 = hp->lmax + 1, nch = hp->n_channels;
    auto permute = [&](int64_t off) {
      for (int c = 0; c < nch; ++c)
        for (int l = 0; l < nl1; ++l)
          std::memcpy(&wd[off + (int64_t)(l * nch + c) * P.D], &weights_host[off + (int64_t)(c * nl1 + l) * P.D], sizeof(float) * P.D);
    };
    permute(P.w_init);
    for (const Layer& ly : P.layers) permute(ly.w_env);
    cudaMemcpy(m->d_w, wd.data(), sizeof(float) * n_weights, cudaMemcpyHostToDevice);
  }
  for (const Layer& ly : P.layers) {
    const std::string sig = layer_signature(ly, hp->lmax);
    int id = -1;
    for (int k = 0; k < tpgen::N_SIGS; ++k) if (sig == tpgen::SIG_STR[k]) id = k;
    if (id < 0) return fail(ALLEGRO_ERR_UNSUPPORTED, "no generated tensor-product code for layer signature " + sig);
    m->tp_sig.push_back(id);
  }
  // collapsed edge-energy chain (no non-linearity): w_eff = W_1^T ... W_last^T, in fp64 on the host
  {
    std::vector<double> v(1, 1.0);   // row vector [1 x width]
    int width = 1;
    for (int k = (int)P.w_edge.size() - 1; k >= 0; --k) {
      const int rows = width;                                    // W_k is [rows, cols]
      const int cols = (k == 0) ? P.D : hp->edge_dims[k - 1];
      std::vector<double> nv(cols, 0.0);
      for (int r = 0; r < rows; ++r)
        for (int c = 0; c < cols; ++c) nv[c] += v[r] * (double)weights_host[P.w_edge[k] + (int64_t)r * cols + c];
      v.swap(nv); width = cols;
    }
    std::vector<float> wf(P.D);
    for (int d = 0; d < P.D; ++d) wf[d] = (float)v[d];
    if (cudaMalloc(&m->d_weff, sizeof(float) * P.D) != cudaSuccess) return fail(ALLEGRO_ERR_ALLOC, "w_eff allocation failed");
    cudaMemcpy(m->d_weff, wf.data(), sizeof(float) * P.D, cudaMemcpyHostToDevice);
  }
  for (int L = 1; L <= hp->n_layers; ++L) {
    const Layer& ly = P.layers[L - 1];
    m->c_old.push_back(weights_host[ly.w_res]);
    m->c_new.push_back(weights_host[ly.w_res + 1]);
    CgDev cg;
    cg.n_paths = (int)ly.paths.size();
    std::vector<int> tab(cg.n_paths * 8);
    for (int p = 0; p < cg.n_paths; ++p) {
      const Path& pa = ly.paths[p];
      int* t = &tab[p * 8];
      t[0] = ly.in_off[pa.ir1]; t[1] = 2 * ly.in_irreps[pa.ir1].l + 1; t[2] = pa.l2 * pa.l2; t[3] = 2 * pa.l2 + 1;
      t[4] = pa.iro; t[5] = pa.pidx; t[6] = pa.cg_begin; t[7] = pa.cg_end;
    }
    std::vector<int> idx(ly.cg.size()); std::vector<float> val(ly.cg.size());
    for (size_t q = 0; q < ly.cg.size(); ++q) { idx[q] = ly.cg[q].m1 | (ly.cg[q].m2 << 8) | (ly.cg[q].m3 << 16); val[q] = ly.cg[q].coef; }
    if (cudaMalloc(&cg.path_tab, sizeof(int) * std::max<size_t>(tab.size(), 1)) != cudaSuccess ||
        cudaMalloc(&cg.cg_idx, sizeof(int) * std::max<size_t>(idx.size(), 1)) != cudaSuccess ||
        cudaMalloc(&cg.cg_val, sizeof(float) * std::max<size_t>(val.size(), 1)) != cudaSuccess) {
      m->cg.push_back(cg);
      return fail(ALLEGRO_ERR_ALLOC, "coupling table allocation failed");
    }
    cudaMemcpy(cg.path_tab, tab.data(), sizeof(int) * tab.size(), cudaMemcpyHostToDevice);
    cudaMemcpy(cg.cg_idx, idx.data(), sizeof(int) * idx.size(), cudaMemcpyHostToDevice);
    cudaMemcpy(cg.cg_val, val.data(), sizeof(float) * val.size(), cudaMemcpyHostToDevice);
    m->cg.push_back(cg);
    if ((int)ly.out_irreps.size() > 8) return fail(ALLEGRO_ERR_UNSUPPORTED, "more than 8 output irreps in a layer");
  }
  if (ensure(m, &m->flags, sizeof(int) * FLAG_COUNT)) return fail(ALLEGRO_ERR_ALLOC, m->err);
  cudaMemset(m->flags.p, 0, sizeof(int) * FLAG_COUNT);
  ce = cudaDeviceSynchronize();
  if (ce != cudaSuccess) return fail(ALLEGRO_ERR_CUDA, std::string("allegro_create: ") + cudaGetErrorString(ce));
  *handle_out = m;
  return ALLEGRO_OK;
}

int allegro_destroy(void* h) {
  if (!h) return ALLEGRO_OK;
  Model* m = static_cast<Model*>(h);
  md_graph_reset(m);
  if (m->own_stream) cudaStreamDestroy(m->own_stream);
  if (m->d_w) cudaFree(m->d_w);
  if (m->d_weff) cudaFree(m->d_weff);
  for (cudaEvent_t e : m->prof.ev) cudaEventDestroy(e);
  for (auto& kv : m->packed_w) if (kv.second) cudaFree(kv.second);
  for (CgDev& c : m->cg) { if (c.path_tab) cudaFree(c.path_tab); if (c.cg_idx) cudaFree(c.cg_idx); if (c.cg_val) cudaFree(c.cg_val); }
  NeighborList& nl = m->nl;
  for (DevBuf* b : {&nl.r_build, &nl.img, &nl.cell_of, &nl.cell_cnt, &nl.cell_start, &nl.cell_fill, &nl.sorted, &nl.row_cnt, &nl.rowptr,
                    &nl.keys_tmp, &nl.keys, &nl.revpos, &nl.scan_tmp, &m->ws.arena, &m->ws.scan_tmp, &m->g_list, &m->e_atom, &m->e_partial, &m->act_total,
                    &m->flags, &m->md_pos, &m->md_vel, &m->md_mass, &m->md_species, &m->md_F, &m->md_E, &m->vir_partial, &m->nvt_par, &nl.rowptr_new, &m->decomp_tmp})
    free_buf(*b);
  delete m;
  return ALLEGRO_OK;
}

int allegro_build_neighbors(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, double cutoff,
                            double skin, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  (void)species;
  if ((!pos && N > 0) || !cell || N < 0 || skin < 0.0) { m->err = "allegro_build_neighbors: bad argument"; return ALLEGRO_ERR_INVALID; }
  if (cutoff != m->plan.hp.r_cut) { m->err = "cutoff must equal hp.r_cut"; return ALLEGRO_ERR_INVALID; }
  if (N >= (int64_t)1 << 31) { m->err = "N must be < 2^31"; return ALLEGRO_ERR_UNSUPPORTED; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  m->md_ready = false;
  int rc = nl_build(m, pos, N, cell, cutoff, skin, false, st);
  if (rc) return rc;
  rc = check_flags(m, st, "allegro_build_neighbors");
  m->stats[1] = m->nl.E_list; m->stats[2] = m->launches;
  return rc;
}

int allegro_energy_forces(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, double* E_out,
                          double* F_out, float* E_atom_out, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!pos || !species || !cell || !E_out || !F_out) { m->err = "allegro_energy_forces: null argument"; return ALLEGRO_ERR_INVALID; }
  if (!m->nl.valid) { m->err = "allegro_energy_forces called before allegro_build_neighbors"; return ALLEGRO_ERR_NO_LIST; }
  if (N != m->nl.N) { m->err = "N differs from the neighbour list"; return ALLEGRO_ERR_INVALID; }
  for (int d = 0; d < 3; ++d)
    if (cell[3 * d] != m->nl.H[3 * d] || cell[3 * d + 1] != m->nl.H[3 * d + 1] || cell[3 * d + 2] != m->nl.H[3 * d + 2]) { m->err = "cell differs from the one the neighbour list was built with"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  int rc = network_energy_forces(m, pos, species, N, E_out, F_out, E_atom_out, st);
  if (rc) return rc;
  int64_t act = 0;
  if (N > 0 && m->act_total.p) cudaMemcpyAsync(&act, m->act_total.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
  rc = check_flags(m, st, "allegro_energy_forces");
  if (rc == ALLEGRO_ERR_ALLOC) { m->ws.slack *= 1.5; m->ws.for_N = -1; }   // a chunk overflowed its workspace share: a retry gets more
  m->stats[0] = act; m->stats[2] = m->launches; m->stats[3] = 0; m->stats[4] = 1;
  return rc;
}

int allegro_energy_forces_owned(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, int64_t n_owned,
                                double* E_out, double* F_out, float* E_atom_out, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!pos || !species || !cell || !E_out || !F_out || n_owned < 0 || n_owned > N) { m->err = "allegro_energy_forces_owned: bad argument"; return ALLEGRO_ERR_INVALID; }
  if (!m->nl.valid) { m->err = "allegro_energy_forces_owned called before allegro_build_neighbors"; return ALLEGRO_ERR_NO_LIST; }
  if (N != m->nl.N) { m->err = "N differs from the neighbour list"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  int rc = network_energy_forces(m, pos, species, N, E_out, F_out, E_atom_out, st, n_owned);
  if (rc) return rc;
  int64_t act = 0;
  if (N > 0 && m->act_total.p) cudaMemcpyAsync(&act, m->act_total.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
  rc = check_flags(m, st, "allegro_energy_forces_owned");
  if (rc == ALLEGRO_ERR_ALLOC) { m->ws.slack *= 1.5; m->ws.for_N = -1; }
  m->stats[0] = act; m->stats[2] = m->launches; m->stats[3] = 0; m->stats[4] = 1;
  return rc;
}

int allegro_decomp_select(void* h, const double* pos, const int32_t* species, int64_t N, const double* cell, const int32_t* grid,
                          const int32_t* coord, double r_halo, int64_t cap, double* local_pos, int32_t* local_species, int64_t* local_src,
                          int64_t* counts, double* local_cell, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if ((!pos && N > 0) || !cell || !grid || !coord || !local_pos || !local_src || !counts || !local_cell || N < 0 || cap < 0 || !(r_halo > 0.0)) {
    m->err = "allegro_decomp_select: bad argument"; return ALLEGRO_ERR_INVALID;
  }
  return decomp_select(m, pos, species, N, cell, grid, coord, r_halo, cap, local_pos, local_species, local_src, counts, local_cell,
                       static_cast<cudaStream_t>(stream));
}

int allegro_decomp_scatter(const double* F_local, const int64_t* local_src, int64_t n_local, double* F_global, int64_t N, void* stream) {
  if ((!F_local || !local_src) && n_local > 0) return ALLEGRO_ERR_INVALID;
  if (!F_global && N > 0) return ALLEGRO_ERR_INVALID;
  return decomp_scatter(F_local, local_src, n_local, F_global, N, static_cast<cudaStream_t>(stream));
}

int allegro_kick_drift(double* pos, double* vel, const double* F, const double* mass, int64_t N, double dt_fs, int drift, void* stream) {
  if ((!pos || !vel || !F || !mass) && N > 0) return ALLEGRO_ERR_INVALID;
  return ext_kick_drift(pos, vel, F, mass, N, dt_fs, drift, static_cast<cudaStream_t>(stream));
}

int allegro_md_init(void* h, const double* pos, const double* vel, const double* mass, const int32_t* species, int64_t N,
                    const double* cell, double cutoff, double skin, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!pos || !vel || !mass || !species || !cell || N < 0 || skin < 0.0) { m->err = "allegro_md_init: bad argument"; return ALLEGRO_ERR_INVALID; }
  if (cutoff != m->plan.hp.r_cut) { m->err = "cutoff must equal hp.r_cut"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  int rc = md_init(m, pos, vel, mass, species, N, cell, cutoff, skin, st);
  if (rc) return rc;
  int zero = 0;
  cudaMemcpyAsync(m->flags.as<int>() + FLAG_NREBUILD, &zero, sizeof(int), cudaMemcpyHostToDevice, st);
  rc = check_flags(m, st, "allegro_md_init");
  m->stats[2] = m->launches;
  return rc;
}

static int md_step_api(void* h, double dt_fs, int64_t n_steps, const double* nvt, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!m->md_ready) { m->err = "allegro_md_step called before allegro_md_init"; return ALLEGRO_ERR_INVALID; }
  if (n_steps < 0 || !(dt_fs > 0.0)) { m->err = "allegro_md_step: bad argument"; return ALLEGRO_ERR_INVALID; }
  if (nvt && (!(nvt[0] > 0.0) || !(nvt[1] > 0.0) || nvt[2] < 0.0 || !(nvt[3] >= dt_fs))) {
    m->err = "allegro_md_step_nvt: temperatures must be > 0, n_ramp >= 0, tau >= dt"; return ALLEGRO_ERR_INVALID;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  const int64_t reb0 = m->nl.n_rebuilds;
  m->stats[4] = 0; m->stats[6] = 0;
  int rc = md_step(m, dt_fs, n_steps, nvt, st);
  if (rc) return rc;
  int64_t act = 0, elist = 0;
  if (m->nl.N > 0) {
    if (m->act_total.p) cudaMemcpyAsync(&act, m->act_total.p, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
    cudaMemcpyAsync(&elist, m->nl.rowptr.as<int64_t>() + m->nl.N, sizeof(int64_t), cudaMemcpyDeviceToHost, st);
  }
  rc = check_flags(m, st, "allegro_md_step");
  if (m->nl.N > 0) m->nl.E_list = elist;
  m->stats[0] = act; m->stats[1] = m->nl.E_list; m->stats[2] = m->launches; m->stats[3] = m->nl.n_rebuilds - reb0;
  return rc;
}

int allegro_md_step(void* h, double dt_fs, int64_t n_steps, void* stream) { return md_step_api(h, dt_fs, n_steps, nullptr, stream); }

int allegro_md_step_nvt(void* h, double dt_fs, int64_t n_steps, double T0, double T1, int64_t n_ramp, double tau_fs, void* stream) {
  const double par[4] = {T0, T1, (double)n_ramp, tau_fs};
  return md_step_api(h, dt_fs, n_steps, par, stream);
}

int allegro_md_deform(void* h, const double* cell_new, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!m->md_ready || !cell_new) { m->err = "allegro_md_deform: no MD state or null cell"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  int rc = md_deform(m, cell_new, st);
  if (rc) return rc;
  rc = check_flags(m, st, "allegro_md_deform");
  m->stats[2] = m->launches;
  return rc;
}

int allegro_set_state(void* h, const double* pos, const double* vel, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!m->md_ready || !pos || !vel) { m->err = "allegro_set_state: no MD state (call allegro_md_init first) or null argument"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  m->launches = 0;
  int rc = md_set_state(m, pos, vel, st);
  if (rc) return rc;
  rc = check_flags(m, st, "allegro_set_state");
  m->stats[2] = m->launches;
  return rc;
}

int allegro_virial(void* h, const double* pos, double* W_out, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!W_out) { m->err = "allegro_virial: null output"; return ALLEGRO_ERR_INVALID; }
  if (!m->nl.valid) { m->err = "allegro_virial called before a force evaluation"; return ALLEGRO_ERR_NO_LIST; }
  if (!pos && !m->md_ready) { m->err = "allegro_virial: pos == NULL needs an MD state"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  int rc = network_virial(m, pos ? pos : m->md_pos.as<double>(), W_out, st);
  if (rc) return rc;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_virial");
  return ALLEGRO_OK;
}

int allegro_debug_set_fusion(void* h, int on) {
  if (!h) return ALLEGRO_ERR_INVALID;
  static_cast<Model*>(h)->use_tpmix = on != 0;
  return ALLEGRO_OK;
}

int allegro_debug_set_list_slack(void* h, double frac, int64_t extra) {
  if (!h || frac < 0.0 || extra < 0) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  m->nl.slack_frac = frac; m->nl.slack_extra = extra;
  return ALLEGRO_OK;
}

int allegro_get_state(void* h, double* pos, double* vel, double* F, double* E_pot, double* E_kin, int64_t* n_rebuilds, void* stream) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!m->md_ready) { m->err = "allegro_get_state called before allegro_md_init"; return ALLEGRO_ERR_INVALID; }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int64_t N = m->nl.N;
  if (pos) cudaMemcpyAsync(pos, m->md_pos.p, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  if (vel) cudaMemcpyAsync(vel, m->md_vel.p, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  if (F) cudaMemcpyAsync(F, m->md_F.p, sizeof(double) * 3 * N, cudaMemcpyDeviceToDevice, st);
  if (E_pot) cudaMemcpyAsync(E_pot, m->md_E.p, sizeof(double), cudaMemcpyDeviceToDevice, st);
  if (E_kin) { if (int rc = md_kinetic(m, E_kin, st)) return rc; }
  if (n_rebuilds) *n_rebuilds = m->nl.n_rebuilds;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_get_state");
  return ALLEGRO_OK;
}

int allegro_get_neighbors(void* h, int64_t* rowptr, int32_t* col, int8_t* shift, int64_t* E_list) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  if (!m->nl.valid) { m->err = "allegro_get_neighbors called before allegro_build_neighbors"; return ALLEGRO_ERR_NO_LIST; }
  if (E_list) *E_list = m->nl.E_list;
  int rc = nl_export(m, rowptr, col, shift, 0);
  if (rc) return rc;
  cudaError_t e = cudaStreamSynchronize(0);
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_get_neighbors");
  return ALLEGRO_OK;
}

int allegro_get_stats(void* h, int64_t* stats) {
  if (!h || !stats) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  for (int k = 0; k < 8; ++k) stats[k] = m->stats[k];
  return ALLEGRO_OK;
}

int allegro_profile(void* h, int enable) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  cudaDeviceSynchronize();
  prof_collect(m);
  m->prof.on = enable != 0;
  if (enable) for (int k = 0; k < KC_COUNT; ++k) { m->prof.ms[k] = 0; m->prof.launches[k] = 0; m->prof.work[k] = 0; }
  return ALLEGRO_OK;
}

int allegro_get_profile(void* h, double* ms, int64_t* launches, double* work, int max_classes) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  cudaDeviceSynchronize();
  prof_collect(m);
  for (int k = 0; k < KC_COUNT && k < max_classes; ++k) {
    if (ms) ms[k] = m->prof.ms[k];
    if (launches) launches[k] = m->prof.launches[k];
    if (work) work[k] = m->prof.work[k];
  }
  return KC_COUNT;
}

int allegro_debug_set_precision(void* h, int passes) {
  if (!h || passes < 1 || passes > 3) return ALLEGRO_ERR_INVALID;
  static_cast<Model*>(h)->f16_passes = passes;
  return ALLEGRO_OK;
}

int allegro_debug_gemm(void* h, int64_t M, int64_t rows_cap, const float* A0, int lda0, int K0, const float* A1, int lda1, int K1,
                       const float* W, int ldw, int wtrans, int N, int pro, int epi, const float* aux, int ldaux, const float* geo,
                       float* C, int ldc, float* C2, int ldc2, int split, float c_old, float c_new, void* stream) {
  if (!h || !A0 || !W || !C || M < 0 || rows_cap < M) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (int rc = ensure(m, &m->act_total, sizeof(int64_t))) return rc;
  cudaMemcpyAsync(m->act_total.p, &M, sizeof(int64_t), cudaMemcpyHostToDevice, st);
  GemmArgs g;
  g.Mptr = m->act_total.as<int64_t>(); g.geo = geo;
  g.A0 = A0; g.lda0 = lda0; g.K0 = K0; g.A1 = A1; g.lda1 = lda1; g.K1 = K1;
  g.W = W; g.ldw = ldw; g.wtrans = wtrans; g.N = N; g.pro = pro; g.epi = epi;
  g.aux = aux; g.ldaux = ldaux; g.C = C; g.ldc = ldc; g.C2 = C2; g.ldc2 = ldc2; g.split = split; g.c_old = c_old; g.c_new = c_new;
  const int64_t keep = m->f16_rows_cap;
  m->f16_rows_cap = rows_cap;
  const bool ok = launch_gemm_f16s(m, g, M, st);
  m->f16_rows_cap = keep;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_debug_gemm");
  if (!ok) { m->err = "allegro_debug_gemm: shape or alignment outside the split-fp16 kernel"; return ALLEGRO_ERR_UNSUPPORTED; }
  return ALLEGRO_OK;
}

int allegro_debug_forget_weights(void* h) {
  if (!h) return ALLEGRO_ERR_INVALID;
  Model* m = static_cast<Model*>(h);
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return cuda_fail(m, e, "allegro_debug_forget_weights");
  for (auto& kv : m->packed_w) if (kv.second) cudaFree(kv.second);
  m->packed_w.clear();
  m->tmaps.clear();
  md_graph_reset(m);   // a captured MD step holds the old pointers
  return ALLEGRO_OK;
}

const char* allegro_last_error(void* h) {
  if (!h) return g_create_err.c_str();
  return static_cast<Model*>(h)->err.c_str();
}

}  // extern "C"
