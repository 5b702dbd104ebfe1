// plan.cpp — see plan.h.  Host-only C++17.
#include "plan.h"

#include <algorithm>
#include <cmath>
#include <complex>

namespace allegro {
namespace {

double fact(int n) {
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= i;
  return f;
}

// <j1 m1 j2 m2 | j3 m3>, integer angular momenta, Racah's closed form.
double cg_complex(int j1, int m1, int j2, int m2, int j3, int m3) {
  if (m1 + m2 != m3 || j3 < std::abs(j1 - j2) || j3 > j1 + j2) return 0.0;
  if (std::abs(m1) > j1 || std::abs(m2) > j2 || std::abs(m3) > j3) return 0.0;
  double pre = std::sqrt((2.0 * j3 + 1.0) * fact(j3 + j1 - j2) * fact(j3 - j1 + j2) * fact(j1 + j2 - j3) /
                         fact(j1 + j2 + j3 + 1));
  pre *= std::sqrt(fact(j3 + m3) * fact(j3 - m3) * fact(j1 - m1) * fact(j1 + m1) * fact(j2 - m2) * fact(j2 + m2));
  double sum = 0.0;
  for (int k = 0; k <= j1 + j2 - j3; ++k) {
    int d[6] = {k, j1 + j2 - j3 - k, j1 - m1 - k, j2 + m2 - k, j3 - j2 + m1 + k, j3 - j1 - m2 + k};
    bool ok = true;
    double den = 1.0;
    for (int v : d) {
      if (v < 0) { ok = false; break; }
      den *= fact(v);
    }
    if (ok) sum += ((k & 1) ? -1.0 : 1.0) / den;
  }
  return pre * sum;
}

using cd = std::complex<double>;

// Real-from-complex unitary for degree l: Yreal_m = sum_mu U(m,mu) Ycomplex_mu  (A9 recipe).
std::vector<cd> real_basis(int l) {
  int d = 2 * l + 1;
  std::vector<cd> U(d * d, cd(0, 0));
  const double r2 = 1.0 / std::sqrt(2.0);
  for (int m = -l; m <= l; ++m) {
    if (m > 0) {
      U[(m + l) * d + (m + l)] = cd(((m & 1) ? -1.0 : 1.0) * r2, 0);
      U[(m + l) * d + (-m + l)] = cd(r2, 0);
    } else if (m == 0) {
      U[l * d + l] = cd(1, 0);
    } else {
      int mu = -m;
      U[(m + l) * d + (-mu + l)] = cd(0, r2);
      U[(m + l) * d + (mu + l)] = cd(0, -((mu & 1) ? -1.0 : 1.0) * r2);
    }
  }
  return U;
}

bool triangle(int a, int b, int c) { return c >= std::abs(a - b) && c <= a + b; }

bool irrep_less(const Irrep& a, const Irrep& b) {
  if (a.l != b.l) return a.l < b.l;
  int na = (a.p == ((a.l & 1) ? -1 : 1)) ? 0 : 1;
  int nb = (b.p == ((b.l & 1) ? -1 : 1)) ? 0 : 1;
  return na < nb;
}

bool contains(const std::vector<Irrep>& v, const Irrep& x) { return std::find(v.begin(), v.end(), x) != v.end(); }

}  // namespace

std::vector<double> coupling_tensor(int l1, int l2, int l3) {
  const int d1 = 2 * l1 + 1, d2 = 2 * l2 + 1, d3 = 2 * l3 + 1;
  std::vector<double> C(d1 * d2 * d3, 0.0);
  if (!triangle(l1, l2, l3)) return C;
  auto U1 = real_basis(l1), U2 = real_basis(l2), U3 = real_basis(l3);
  const bool even = ((l1 + l2 + l3) % 2) == 0;
  double nrm = 0.0;
  for (int a = 0; a < d1; ++a)
    for (int b = 0; b < d2; ++b)
      for (int c = 0; c < d3; ++c) {
        cd acc(0, 0);
        for (int i = 0; i < d1; ++i)
          for (int j = 0; j < d2; ++j) {
            int mu3 = (i - l1) + (j - l2);
            if (std::abs(mu3) > l3) continue;
            double g = cg_complex(l1, i - l1, l2, j - l2, l3, mu3);
            if (g == 0.0) continue;
            acc += U1[a * d1 + i] * U2[b * d2 + j] * std::conj(U3[c * d3 + (mu3 + l3)]) * g;
          }
        double v = even ? acc.real() : acc.imag();
        C[(a * d2 + b) * d3 + c] = v;
        nrm += v * v;
      }
  const double scale = std::sqrt((double)d3) / std::sqrt(nrm);
  double first = 0.0;
  for (double& v : C) {
    v *= scale;
    if (std::fabs(v) < 1e-12) v = 0.0;
    if (first == 0.0 && v != 0.0) first = v;
  }
  if (first < 0.0)
    for (double& v : C) v = -v;
  return C;
}

std::string layer_signature(const Layer& ly, int lmax) {
  std::string s = "L" + std::to_string(lmax) + "|in";
  for (const Irrep& a : ly.in_irreps) s += ":" + std::to_string(a.l) + (a.p > 0 ? "e" : "o");
  s += "|out";
  for (size_t o = 0; o < ly.out_irreps.size(); ++o)
    s += ":" + std::to_string(ly.out_irreps[o].l) + (ly.out_irreps[o].p > 0 ? "e" : "o") + "@" + std::to_string(ly.out_off[o]);
  s += "|p";
  for (const Path& p : ly.paths)
    s += ":" + std::to_string(p.ir1) + "," + std::to_string(p.l2) + "," + std::to_string(p.iro) + "," + std::to_string(p.pidx);
  return s;
}

std::string build_plan(const allegro_hparams& hp, Plan* out) {
  Plan P;
  P.hp = hp;
  if (hp.lmax < 0 || hp.lmax > 3) return "lmax must be in [0,3]";
  if (hp.n_layers < 1 || hp.n_layers > 8) return "n_layers must be in [1,8]";
  if (hp.n_species < 1 || hp.n_bessel < 1 || hp.n_bessel > 16 || hp.n_channels < 1) return "bad n_species/n_bessel/n_channels";
  if (hp.poly_p < 2) return "poly_p must be >= 2";
  if (hp.two_body_nl < 1 || hp.two_body_nl > 8 || hp.latent_nl < 1 || hp.latent_nl > 8 || hp.edge_nl < 0 || hp.edge_nl > 8)
    return "MLP depth out of range";
  for (int i = 0; i < hp.two_body_nl; ++i) if (hp.two_body_dims[i] <= 0) return "two_body_dims must be > 0";
  for (int i = 0; i < hp.latent_nl; ++i) if (hp.latent_dims[i] <= 0) return "latent_dims must be > 0";
  for (int i = 0; i < hp.edge_nl; ++i) if (hp.edge_dims[i] <= 0) return "edge_dims must be > 0";
  if (!(hp.r_cut > 0.0) || !(hp.avg_num_neighbors > 0.0)) return "r_cut and avg_num_neighbors must be > 0";
  P.D = hp.two_body_dims[hp.two_body_nl - 1];
  if (hp.latent_dims[hp.latent_nl - 1] != P.D) return "last latent width must equal last two-body width (A10)";
  const int lmax = hp.lmax, NL = hp.n_layers, n = hp.n_channels;
  P.n_sc = n * (lmax + 1);
  P.d_sh = (lmax + 1) * (lmax + 1);

  std::vector<Irrep> G;
  for (int l = 0; l <= lmax; ++l) G.push_back({l, (l & 1) ? -1 : 1});
  auto allowed = [&](const Irrep& a, const Irrep& b, int lo) {
    if (!triangle(a.l, b.l, lo) || lo > lmax) return false;
    if (!hp.full_o3 && ((a.l + b.l + lo) & 1)) return false;
    return true;
  };
  // reachable irreps forward
  std::vector<std::vector<Irrep>> R(NL + 1);
  R[0] = G;
  for (int L = 1; L <= NL; ++L) {
    for (const Irrep& a : R[L - 1])
      for (const Irrep& b : G)
        for (int lo = 0; lo <= lmax; ++lo)
          if (allowed(a, b, lo)) {
            Irrep o{lo, a.p * b.p};
            if (!contains(R[L], o)) R[L].push_back(o);
          }
    std::sort(R[L].begin(), R[L].end(), irrep_less);
  }
  // kept irreps backward
  std::vector<std::vector<Irrep>> K(NL), targets(NL + 1);
  targets[NL] = {Irrep{0, 1}};
  for (int L = NL - 1; L >= 0; --L) {
    for (const Irrep& a : R[L]) {
      bool hit = false;
      for (const Irrep& b : G)
        for (int lo = 0; lo <= lmax && !hit; ++lo)
          if (allowed(a, b, lo) && contains(targets[L + 1], Irrep{lo, a.p * b.p})) hit = true;
      if (hit) K[L].push_back(a);
    }
    std::sort(K[L].begin(), K[L].end(), irrep_less);
    targets[L] = K[L];
    if (!contains(targets[L], Irrep{0, 1})) targets[L].push_back(Irrep{0, 1});
    std::sort(targets[L].begin(), targets[L].end(), irrep_less);
  }
  if (K[0].size() != G.size()) return "internal: V^0 irreps != natural-parity irreps";

  // ---- weight blob offsets, in the order of SURVEY.md 8b
  int64_t off = 0;
  auto add = [&](int kind, int64_t r, int64_t c) {
    P.lay_kind.push_back(kind); P.lay_rows.push_back(r); P.lay_cols.push_back(c);
    int64_t o = off; off += r * c; return o;
  };
  int fan = 2 * hp.n_species + hp.n_bessel;
  for (int i = 0; i < hp.two_body_nl; ++i) { P.w_two_body.push_back(add(ALLEGRO_WK_MATRIX, hp.two_body_dims[i], fan)); fan = hp.two_body_dims[i]; }
  P.w_init = add(ALLEGRO_WK_MATRIX, P.n_sc, P.D);

  P.layers.resize(NL);
  for (int L = 1; L <= NL; ++L) {
    Layer& ly = P.layers[L - 1];
    ly.in_irreps = K[L - 1];
    for (const Irrep& a : ly.in_irreps) { ly.in_off.push_back(ly.in_dim); ly.in_dim += 2 * a.l + 1; }
    // out irreps: 0e first, then K^L in order (0e, if kept, is the same entry)
    ly.out_irreps.push_back(Irrep{0, 1});
    if (L < NL)
      for (const Irrep& o : K[L]) if (!(o == Irrep{0, 1})) ly.out_irreps.push_back(o);
    ly.out_off.assign(ly.out_irreps.size(), -1);
    ly.out_npaths.assign(ly.out_irreps.size(), 0);
    if (L < NL) {
      // V^L component layout follows K^L order
      for (const Irrep& o : K[L]) {
        int idx = (int)(std::find(ly.out_irreps.begin(), ly.out_irreps.end(), o) - ly.out_irreps.begin());
        ly.out_off[idx] = ly.out_dim;
        ly.out_dim += 2 * o.l + 1;
      }
    }
    for (int i1 = 0; i1 < (int)ly.in_irreps.size(); ++i1)
      for (const Irrep& b : G)
        for (int lo = 0; lo <= lmax; ++lo) {
          const Irrep& a = ly.in_irreps[i1];
          Irrep o{lo, a.p * b.p};
          if (!allowed(a, b, lo) || !contains(targets[L], o)) continue;
          int io = (int)(std::find(ly.out_irreps.begin(), ly.out_irreps.end(), o) - ly.out_irreps.begin());
          Path p;
          p.ir1 = i1; p.l2 = b.l; p.iro = io; p.pidx = ly.out_npaths[io]++;
          p.cg_begin = (int)ly.cg.size();
          std::vector<double> C = coupling_tensor(a.l, b.l, lo);
          const int d2 = 2 * b.l + 1, d3 = 2 * lo + 1;
          // entries grouped by output component m3 (then m1, m2)
          for (int m3 = 0; m3 < d3; ++m3)
            for (int m1 = 0; m1 < 2 * a.l + 1; ++m1)
              for (int m2 = 0; m2 < d2; ++m2) {
                double v = C[(m1 * d2 + m2) * d3 + m3];
                if (v != 0.0) ly.cg.push_back(CgEntry{(int16_t)m1, (int16_t)m2, (int16_t)m3, (float)v});
              }
          p.cg_end = (int)ly.cg.size();
          ly.paths.push_back(p);
        }
    if (ly.out_npaths[0] != lmax + 1) return "internal: number of scalar paths != lmax+1";
    ly.w_env = add(ALLEGRO_WK_MATRIX, P.n_sc, P.D);
    fan = P.D + P.n_sc;
    for (int i = 0; i < hp.latent_nl; ++i) { ly.w_latent.push_back(add(ALLEGRO_WK_MATRIX, hp.latent_dims[i], fan)); fan = hp.latent_dims[i]; }
    ly.w_res = add(ALLEGRO_WK_RESIDUAL, 1, 2);
    ly.w_lin.assign(ly.out_irreps.size(), -1);
    if (L < NL)
      for (const Irrep& o : K[L]) {  // blob order = K^L order
        int idx = (int)(std::find(ly.out_irreps.begin(), ly.out_irreps.end(), o) - ly.out_irreps.begin());
        ly.w_lin[idx] = add(ALLEGRO_WK_MATRIX, n, (int64_t)ly.out_npaths[idx] * n);
      }
  }
  fan = P.D;
  for (int i = 0; i < hp.edge_nl; ++i) { P.w_edge.push_back(add(ALLEGRO_WK_MATRIX, hp.edge_dims[i], fan)); fan = hp.edge_dims[i]; }
  P.w_edge.push_back(add(ALLEGRO_WK_MATRIX, 1, fan));
  P.w_sigma = add(ALLEGRO_WK_SIGMA, 1, hp.n_species);
  P.w_mu = add(ALLEGRO_WK_MU, 1, hp.n_species);
  P.n_weights = off;
  *out = std::move(P);
  return "";
}

}  // namespace allegro
