// gen_tp.cpp — build-time generator (host C++17, linked with plan.cpp) that writes tp_gen.cuh: the
// Clebsch-Gordan tensor product of every layer signature the plan builder can produce for lmax <= 3, with the
// sparse real coupling tensors (reading A9, plan.cpp) unrolled into straight-line FMA code so that V, Gamma and T
// stay in registers (F8 / B5 of SURVEY.md 8c; "tensor features with l=2 in full O(3) symmetry").
//
// Per signature S it emits
//   tp_path_fwd_S(p, V, G, T):            T(m3, sum C V(in_off+m1) G(l2^2+m2))              for path p
//   tp_path_bwd_S(p, V, G, Tb, Vb, Gb):   Vb(in_off+m1, sum C Tb(m3) G) ; Gb(l2^2+m2, sum C Tb(m3) V)
// with V/G/T/Tb/Vb/Gb accessor functors supplied by the kernels of tp.cuh, plus the signature strings that the
// library matches against layer_signature() at create time.
#include <cstdio>
#include <map>
#include <string>
#include <vector>

#include "plan.h"

using namespace allegro;

static std::string fl(double v) {
  char b[64];
  snprintf(b, sizeof b, "%.9gf", v);
  std::string s(b);
  if (s.find('.') == std::string::npos && s.find('e') == std::string::npos) s.insert(s.size() - 1, ".0");
  return s;
}

struct Nz { int m1, m2, m3; double c; };

static void emit_layer(FILE* f, int id, const Layer& ly) {
  const int np = (int)ly.paths.size();
  std::vector<std::vector<Nz>> nz(np);
  std::vector<int> in_off(np), l2off(np), d1(np), d2(np), d3(np);
  for (int p = 0; p < np; ++p) {
    const Path& pa = ly.paths[p];
    in_off[p] = ly.in_off[pa.ir1]; d1[p] = 2 * ly.in_irreps[pa.ir1].l + 1; l2off[p] = pa.l2 * pa.l2; d2[p] = 2 * pa.l2 + 1;
    d3[p] = 2 * ly.out_irreps[pa.iro].l + 1;
    for (int q = pa.cg_begin; q < pa.cg_end; ++q) nz[p].push_back(Nz{ly.cg[q].m1, ly.cg[q].m2, ly.cg[q].m3, (double)ly.cg[q].coef});
  }
  auto loads = [&](int p, bool tb) {
    std::vector<bool> u1(d1[p], false), u2(d2[p], false), u3(d3[p], false);
    for (const Nz& z : nz[p]) { u1[z.m1] = u2[z.m2] = u3[z.m3] = true; }
    for (int a = 0; a < d1[p]; ++a) if (u1[a]) fprintf(f, "      const float v%d = V(%d);\n", a, in_off[p] + a);
    for (int b = 0; b < d2[p]; ++b) if (u2[b]) fprintf(f, "      const float g%d = G(%d);\n", b, l2off[p] + b);
    if (tb) for (int c = 0; c < d3[p]; ++c) if (u3[c]) fprintf(f, "      const float t%d = Tb(%d);\n", c, c);
  };
  // ---- forward
  fprintf(f, "template <class VA, class GA, class TA>\n__device__ __forceinline__ void tp_path_fwd_%d(int p, VA V, GA G, TA T) {\n  switch (p) {\n", id);
  for (int p = 0; p < np; ++p) {
    fprintf(f, "    case %d: {\n", p);
    loads(p, false);
    std::map<std::pair<int, int>, bool> prod;
    for (const Nz& z : nz[p]) prod[{z.m1, z.m2}] = true;
    for (auto& kv : prod) fprintf(f, "      const float p%d_%d = v%d * g%d;\n", kv.first.first, kv.first.second, kv.first.first, kv.first.second);
    for (int c = 0; c < d3[p]; ++c) {
      std::string e;
      for (const Nz& z : nz[p]) if (z.m3 == c) {
        if (!e.empty()) e += " + ";
        e += fl(z.c) + " * p" + std::to_string(z.m1) + "_" + std::to_string(z.m2);
      }
      if (e.empty()) e = "0.0f";
      fprintf(f, "      T(%d, %s);\n", c, e.c_str());
    }
    fprintf(f, "    } break;\n");
  }
  fprintf(f, "    default: break;\n  }\n}\n\n");
  // ---- backward
  fprintf(f, "template <class VA, class GA, class TBA, class VBA, class GBA>\n__device__ __forceinline__ void tp_path_bwd_%d(int p, VA V, GA G, TBA Tb, VBA Vb, GBA Gb) {\n  switch (p) {\n", id);
  for (int p = 0; p < np; ++p) {
    fprintf(f, "    case %d: {\n", p);
    loads(p, true);
    std::map<std::pair<int, int>, std::string> q;
    for (const Nz& z : nz[p]) {
      std::string& e = q[{z.m1, z.m2}];
      if (!e.empty()) e += " + ";
      e += fl(z.c) + " * t" + std::to_string(z.m3);
    }
    for (auto& kv : q) fprintf(f, "      const float q%d_%d = %s;\n", kv.first.first, kv.first.second, kv.second.c_str());
    for (int a = 0; a < d1[p]; ++a) {
      std::string e;
      for (auto& kv : q) if (kv.first.first == a) {
        if (!e.empty()) e += " + ";
        e += "q" + std::to_string(a) + "_" + std::to_string(kv.first.second) + " * g" + std::to_string(kv.first.second);
      }
      if (!e.empty()) fprintf(f, "      Vb(%d, %s);\n", in_off[p] + a, e.c_str());
    }
    for (int b = 0; b < d2[p]; ++b) {
      std::string e;
      for (auto& kv : q) if (kv.first.second == b) {
        if (!e.empty()) e += " + ";
        e += "q" + std::to_string(kv.first.first) + "_" + std::to_string(b) + " * v" + std::to_string(kv.first.first);
      }
      if (!e.empty()) fprintf(f, "      Gb(%d, %s);\n", l2off[p] + b, e.c_str());
    }
    fprintf(f, "    } break;\n");
  }
  fprintf(f, "    default: break;\n  }\n}\n\n");
}

int main(int argc, char** argv) {
  if (argc < 2) { fprintf(stderr, "usage: gen_tp <out.cuh>\n"); return 2; }
  FILE* f = fopen(argv[1], "w");
  if (!f) { perror("fopen"); return 1; }
  std::vector<std::string> sigs;
  std::vector<Layer> layers;
  for (int lmax = 0; lmax <= 3; ++lmax)
    for (int NL = 1; NL <= 5; ++NL)
      for (int o3 = 0; o3 <= 1; ++o3) {
        allegro_hparams hp{};
        hp.n_species = 1; hp.n_bessel = 8; hp.poly_p = 6; hp.lmax = lmax; hp.n_layers = NL; hp.n_channels = 4; hp.full_o3 = o3;
        hp.two_body_nl = 2; hp.two_body_dims[0] = hp.two_body_dims[1] = 8;
        hp.latent_nl = 2; hp.latent_dims[0] = hp.latent_dims[1] = 8;
        hp.edge_nl = 1; hp.edge_dims[0] = 8; hp.r_cut = 4.0; hp.avg_num_neighbors = 10.0;
        Plan P;
        std::string e = build_plan(hp, &P);
        if (!e.empty()) { fprintf(stderr, "gen_tp: plan failed: %s\n", e.c_str()); return 1; }
        for (const Layer& ly : P.layers) {
          std::string s = layer_signature(ly, lmax);
          bool have = false;
          for (const std::string& t : sigs) if (t == s) have = true;
          if (!have) { sigs.push_back(s); layers.push_back(ly); }
        }
      }
  fprintf(f, "// GENERATED by gen_tp.cpp at build time — do not edit.  %zu layer signatures.\n#pragma once\nnamespace allegro {\nnamespace tpgen {\n\n", sigs.size());
  fprintf(f, "constexpr int N_SIGS = %zu;\n", sigs.size());
  fprintf(f, "static const char* const SIG_STR[N_SIGS] = {\n");
  for (const std::string& s : sigs) fprintf(f, "  \"%s\",\n", s.c_str());
  fprintf(f, "};\n");
  fprintf(f, "template <int SIG> struct SigDims;\n");
  for (size_t i = 0; i < sigs.size(); ++i) {
    const Layer& ly = layers[i];
    int lmax = sigs[i][1] - '0';
    auto arr = [&](const char* name, const std::vector<int>& v) {
      fprintf(f, "  static constexpr __host__ __device__ int %s(int i) { constexpr int t[] = {", name);
      for (size_t k = 0; k < v.size(); ++k) fprintf(f, "%s%d", k ? ", " : "", v[k]);
      fprintf(f, "}; return t[i]; }\n");
    };
    std::vector<int> piro, ppidx, od3, onp, ooff;
    for (const Path& pa : ly.paths) { piro.push_back(pa.iro); ppidx.push_back(pa.pidx); }
    for (size_t o = 0; o < ly.out_irreps.size(); ++o) { od3.push_back(2 * ly.out_irreps[o].l + 1); onp.push_back(ly.out_npaths[o]); ooff.push_back(ly.out_off[o]); }
    fprintf(f, "template <> struct SigDims<%zu> {\n  static constexpr int IN_DIM = %d, DSH = %d, LMAX = %d, NPATH = %zu, NOUT = %zu, OUT_DIM = %d;\n", i,
            ly.in_dim, (lmax + 1) * (lmax + 1), lmax, ly.paths.size(), ly.out_irreps.size(), ly.out_dim);
    arr("p_iro", piro); arr("p_pidx", ppidx); arr("o_d3", od3); arr("o_np", onp); arr("o_off", ooff);
    fprintf(f, "};\n");
  }
  fprintf(f, "\n#ifdef __CUDACC__\n");
  for (size_t i = 0; i < sigs.size(); ++i) emit_layer(f, (int)i, layers[i]);
  fprintf(f, "template <int SIG, class VA, class GA, class TA>\n__device__ __forceinline__ void tp_path_fwd(int p, VA V, GA G, TA T) {\n");
  for (size_t i = 0; i < sigs.size(); ++i) fprintf(f, "  if constexpr (SIG == %zu) tp_path_fwd_%zu(p, V, G, T);\n", i, i);
  fprintf(f, "}\ntemplate <int SIG, class VA, class GA, class TBA, class VBA, class GBA>\n__device__ __forceinline__ void tp_path_bwd(int p, VA V, GA G, TBA Tb, VBA Vb, GBA Gb) {\n");
  for (size_t i = 0; i < sigs.size(); ++i) fprintf(f, "  if constexpr (SIG == %zu) tp_path_bwd_%zu(p, V, G, Tb, Vb, Gb);\n", i, i);
  fprintf(f, "}\n#endif  // __CUDACC__\n\n#define TPGEN_FOR_EACH_SIG(X)");
  for (size_t i = 0; i < sigs.size(); ++i) fprintf(f, " X(%zu)", i);
  fprintf(f, "\n\n}  // namespace tpgen\n}  // namespace allegro\n");
  fclose(f);
  fprintf(stderr, "gen_tp: %zu signatures -> %s\n", sigs.size(), argv[1]);
  return 0;
}
