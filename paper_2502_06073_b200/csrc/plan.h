// plan.h — host-side plan of the Allegro network: irreps, tensor-product paths, real coupling tables
// and the offsets of every tensor inside the flat weight blob.
//
// Follows PAPER.md:93 ("two layers of 64 tensor features with l=2 in full O(3) symmetry") under the
// readings A8 (path set), A9 (coupling normalisation/sign) and the blob order of SURVEY.md 8b.
// Independent of oracle/ (no shared code or tables): the library derives its own plan and its own
// coupling tables in C++; tests compare them with the oracle's through allegro_debug_coupling.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/allegro.h"

namespace allegro {

struct Irrep {
  int l, p;  // p = +1 (even) / -1 (odd)
  bool operator==(const Irrep& o) const { return l == o.l && p == o.p; }
};

struct CgEntry {  // T[m3] += coef * V[m1] * G[m2]   (indices 0..2l)
  int16_t m1, m2, m3;
  float coef;
};

struct Path {
  int ir1;      // index into Layer::in_irreps   (irrep of V^{L-1})
  int l2;       // env irrep (l2, (-1)^l2)
  int iro;      // index into Layer::out_irreps  (0 = the scalar 0e)
  int pidx;     // index among the paths into out irrep iro (column block of W_lin)
  int cg_begin, cg_end;  // range in Layer::cg
};

struct Layer {
  std::vector<Irrep> in_irreps;    // K^{L-1}, sorted (l asc, natural parity first)
  std::vector<int> in_off;         // component offset of each in irrep inside V^{L-1} (per channel)
  int in_dim = 0;                  // sum (2l+1)
  std::vector<Irrep> out_irreps;   // [0] = 0e, then K^L (if L < NL) without duplicates of 0e
  std::vector<int> out_off;        // component offset inside V^L per out irrep (-1 if not kept)
  std::vector<int> out_npaths;     // number of paths into each out irrep
  int out_dim = 0;                 // dim of V^L per channel (0 for the last layer)
  std::vector<Path> paths;         // enumeration order: l1 asc (natural first), l2 asc, lo asc
  std::vector<CgEntry> cg;
  // weight blob offsets (in floats)
  int64_t w_env = 0;
  std::vector<int64_t> w_latent;   // one per latent linear
  int64_t w_res = 0;               // c_old, c_new
  std::vector<int64_t> w_lin;      // per out irrep (index like out_irreps; -1 when none)
};

struct Plan {
  allegro_hparams hp;
  int D = 0;        // latent width
  int n_sc = 0;     // n_channels * (lmax+1): scalars fed to each latent MLP / width of W_env, W_init
  int d_sh = 0;     // (lmax+1)^2
  std::vector<Layer> layers;
  std::vector<int64_t> w_two_body;
  int64_t w_init = 0;
  std::vector<int64_t> w_edge;     // edge_nl + 1 matrices
  int64_t w_sigma = 0, w_mu = 0;
  int64_t n_weights = 0;
  // layout as reported by allegro_weight_layout
  std::vector<int32_t> lay_kind;
  std::vector<int64_t> lay_rows, lay_cols;
};

// Returns "" on success, else an error message.  Does not touch CUDA.
std::string build_plan(const allegro_hparams& hp, Plan* out);

// Text key of one layer's tensor-product structure (irreps in/out, paths in order): two layers with the same key
// run the same generated coupling code (gen_tp.cpp -> tp_gen.cuh).
std::string layer_signature(const Layer& ly, int lmax);

// Real coupling tensor for (l1,l2,l3) in the F3 basis, dense [2l1+1][2l2+1][2l3+1] (double).
std::vector<double> coupling_tensor(int l1, int l2, int l3);

}  // namespace allegro
