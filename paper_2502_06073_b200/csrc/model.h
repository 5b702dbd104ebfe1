// model.h — device-side state of one allegro handle and the launchers shared by the .cu files.
#pragma once
#include <cuda_runtime.h>

#include <array>
#include <cstdint>
#include <map>
#include <string>
#include <vector>

#include "plan.h"

namespace allegro {

// geometry record per active edge: 8 floats = two float4 (SoA of records keeps 128-bit loads)
//   [0..2] unit vector rhat, [3] r, [4] u(r/rc), [5] du/dr, [6] bit-cast int zi, [7] bit-cast int zj
constexpr int GEO_W = 8;

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

struct alignas(64) TMapStore { uint64_t w[16]; };   // storage of one CUtensorMap (gemm_f16s.cu)

struct CgDev {           // one tensor-product layer's tables on the device
  int n_paths = 0;
  int* path_tab = nullptr;   // [n_paths][8]: in_off, d1, l2off, d2, out_irrep, pidx, cg_begin, cg_end
  int* cg_idx = nullptr;     // [nnz] packed m1 | m2<<8 | m3<<16
  float* cg_val = nullptr;   // [nnz]
};

struct NeighborList {
  bool valid = false;
  int64_t N = 0;
  double H[9] = {0};         // cell, rows = lattice vectors a_1, a_2, a_3 (reading A27); diagonal for an orthorhombic box
  double Hinv[9] = {0};      // fractional coordinates f = x Hinv
  bool ortho = true;
  double cutoff = 0, skin = 0;
  int nc[3] = {1, 1, 1};
  int64_t E_list = 0, cap = 0;
  int64_t n_rebuilds = 0;
  DevBuf r_build, img, cell_of, cell_cnt, cell_start, cell_fill, sorted, row_cnt, rowptr, keys_tmp, keys, revpos;
  DevBuf scan_tmp, rowptr_new;
  double slack_frac = 0.125; int64_t slack_extra = 4096;   // list capacity beyond the count of the sizing build
};

struct Workspace {       // per-chunk activations, sized for cap_edges active edges and cap_atoms atoms
  int64_t cap_edges = 0, cap_atoms = 0;
  int64_t for_N = -1, for_cap = -1, atoms_per = 0;   // chunking decided for this (N, list capacity); kept while it fits
  double slack = 1.25;                                  // active edges of a chunk allowed over the average list row
  DevBuf arena;          // one allocation, carved below
  // chunk-local CSR of active edges
  int* act_cnt = nullptr; int64_t* rowptr_c = nullptr; DevBuf scan_tmp;
  int* e_center = nullptr; int* e_j = nullptr; int64_t* e_lidx = nullptr;
  float* geo = nullptr; float* bes = nullptr;
  std::vector<float*> z2b;           // two-body hidden pre-activations
  float* y0 = nullptr;
  std::vector<float*> x;             // x^0..x^NL
  std::vector<float*> wenv;          // wenv[L-1]: [E, n_sc] (layer 1: second half of winit_w1)
  float* winit_w1 = nullptr;         // [E, 2 n_sc] = W_init x0 | W_env^1 x0
  std::vector<float*> s;             // scalars per layer
  std::vector<std::vector<float*>> zlat;  // latent hidden pre-activations per layer
  std::vector<float*> ylat;          // latent MLP outputs per layer
  std::vector<float*> V;             // V^1..V^{NL-1}  ([E, n, out_dim])
  std::vector<float*> gamma;         // per layer [atoms, n, d_sh]
  // backward
  float* xb[2] = {nullptr, nullptr}; float* zb[2] = {nullptr, nullptr};
  float* sb = nullptr; float* vb[2] = {nullptr, nullptr}; float* ge = nullptr; float* wb = nullptr;
  float* yb = nullptr; float* ub = nullptr; float* eps = nullptr; float* Tbig = nullptr; float* bb = nullptr; float* gammab = nullptr;
};

// optional per-kernel-class timing with CUDA events on the launching stream (allegro_profile)
enum { KC_GEMM = 0, KC_TP_FWD, KC_TP_BWD, KC_GAMMA, KC_GAMMABAR, KC_ACTIVE, KC_EDGE_MISC, KC_NEIGHBOR, KC_MD, KC_GATHER, KC_GEMM16, KC_TP_MIX, KC_TP_MIX16, KC_COUNT };
struct Prof {
  bool on = false;
  std::vector<cudaEvent_t> ev;      // pairs
  std::vector<int> cls;             // class of each pair
  size_t used = 0;                  // pairs in flight
  double ms[KC_COUNT] = {0};
  int64_t launches[KC_COUNT] = {0};
  double work[KC_COUNT] = {0};      // class-specific work units: GEMM/TP = flops per active edge, summed over launches
};

struct Model {
  Plan plan;
  Prof prof;
  std::string err;
  int device = 0;
  int num_sms = 148;
  bool use_tc = true;              // dense linears on tcgen05
  bool use_chain = true;           // MLP chains in one kernel (gemm_tc.cu k_gemm_chain) where the widths fit
  bool use_tpmix = true;           // n = 64: forward tensor product + channel mixing in one kernel (tp_mix.cu)
  bool use_big = false;            // many-channel tensor product: T buffers + tcgen05 channel mixing (tp_big.cuh)
  bool use_tp3 = true;             // few-channel tensor-product kernels (tp3.cuh) where the channel count is 8, 16 or 32, else tp.cuh
  float* d_w = nullptr;            // weight blob
  float* d_weff = nullptr;         // collapsed edge-energy chain W_last...W_1 -> [D]
  std::vector<CgDev> cg;           // per layer
  std::vector<int> tp_sig;         // per layer: index of the generated coupling code (tp_gen.cuh)
  std::map<std::array<int64_t, 5>, float*> packed_w;   // tcgen05 B operands: hi/lo split, canonical UMMA layout (gemm_tc.cu)
  std::map<std::array<int64_t, 6>, TMapStore> tmaps;   // TMA tensor maps of the A operands, by (pointer, K, ld, rows) (gemm_f16s.cu)
  int f16_passes = 3;              // tensor-core passes per product in every GEMM kernel: 3 (default); 2 or 1 only for the precision study (R4)
  int64_t f16_rows_cap = 0;        // rows every edge-sized workspace array holds (bounds the tensor maps)
  std::vector<float> c_old, c_new; // host copies
  NeighborList nl;
  Workspace ws;
  // global per-list-edge gradient and per-atom outputs
  DevBuf g_list, e_atom, e_partial, act_total, flags, md_pos, md_vel, md_mass, md_species, md_F, md_E, vir_partial, nvt_par, decomp_tmp;
  bool md_ready = false;
  // CUDA-graph replay of one MD step (md.cu)
  bool use_graph = true, md_warm = false;
  cudaStream_t own_stream = nullptr, graph_stream = nullptr;
  cudaGraphExec_t md_graph = nullptr;
  double graph_dt = 0;
  int graph_nvt = 0;
  int64_t graph_launches = 0;
  double md_cell[9] = {0};
  int64_t stats[8] = {0};
  int64_t launches = 0;
};

// device flag slots (int32 array in Model::flags)
enum { FLAG_REBUILD = 0, FLAG_ERR_SHIFT = 1, FLAG_ERR_CAP = 2, FLAG_STALE = 3, FLAG_NONFINITE = 4, FLAG_SPECIES = 5,
       FLAG_NREBUILD = 6, FLAG_HALT = 7, FLAG_STEPS = 8, FLAG_COUNT = 16 };
// FLAG_HALT: a device-side rebuild (or the activation workspace) ran out of capacity: the integrator kernels of the remaining
// steps of the call do nothing, FLAG_STEPS counts the completed steps, the host regrows and finishes the call (md.cu).

// ---- profiling brackets (api.cu)
void prof_begin(Model* m, cudaStream_t st, int cls, double work);
void prof_end(Model* m, cudaStream_t st);

// ---- helpers (api.cu)
int ensure(Model* m, DevBuf* b, size_t bytes);            // grow-only cudaMalloc; 0 or ALLEGRO_ERR_ALLOC
int cuda_fail(Model* m, cudaError_t e, const char* what);  // records message, returns ALLEGRO_ERR_CUDA

// ---- virial_noalloc.cu: looks up the device address of the fixed scratch array (once per device, that device current)
int virial_noalloc_setup(Model* m);

// ---- scan.cu: exclusive scan of n int32 counts into n+1 int64 offsets (device), optionally conditional on *flag != 0
int scan_counts(Model* m, const int* cnt, int64_t* out, int64_t n, DevBuf* tmp, const int* flag, cudaStream_t st);

// ---- neighbor.cu
int nl_build(Model* m, const double* pos, int64_t N, const double* cell, double cutoff, double skin,
             bool conditional, cudaStream_t st);
int nl_export(Model* m, int64_t* rowptr, int32_t* col, int8_t* shift, cudaStream_t st);

// ---- network.cu
int ws_prepare(Model* m, int64_t cap_edges, int64_t cap_atoms);
int network_energy_forces(Model* m, const double* pos, const int32_t* species, int64_t N,
                          double* E_out, double* F_out, float* E_atom_out, cudaStream_t st, int64_t n_owned = -1);

// ---- decomp.cu
int decomp_select(Model* m, const double* pos, const int32_t* species, int64_t N, const double* cell, const int32_t* grid, const int32_t* coord,
                  double r_halo, int64_t cap, double* lpos, int32_t* lspecies, int64_t* lsrc, int64_t* counts_host, double* local_cell_host,
                  cudaStream_t st);
int decomp_scatter(const double* F_local, const int64_t* lsrc, int64_t n_local, double* F_global, int64_t N, cudaStream_t st);
int ext_kick_drift(double* pos, double* vel, const double* F, const double* mass, int64_t N, double dt, int drift, cudaStream_t st);

// ---- md.cu
int md_init(Model* m, const double* pos, const double* vel, const double* mass, const int32_t* species, int64_t N,
            const double* cell, double cutoff, double skin, cudaStream_t st);
int md_step(Model* m, double dt, int64_t n_steps, const double* nvt /*[4] T0, T1, n_ramp, tau or NULL*/, cudaStream_t st);
int md_deform(Model* m, const double* cell_new, cudaStream_t st);
int md_set_state(Model* m, const double* pos, const double* vel, cudaStream_t st);
int network_virial(Model* m, const double* pos, double* W_out, cudaStream_t st);
int md_kinetic(Model* m, double* Ekin_dev, cudaStream_t st);
void md_graph_reset(Model* m);

}  // namespace allegro
