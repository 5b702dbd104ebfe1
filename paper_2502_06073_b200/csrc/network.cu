// network.cu — rows a-2..a-5: orchestration of one energy+force evaluation (forward F1-F12, analytic backward
// B1-B12 of SURVEY.md 8c) over the active edges of the current neighbour list, in chunks of centre atoms
// (exact: the model is strictly local).
#include <algorithm>
#include <cmath>

#include "edge_kernels.cuh"
#include "gemm.cuh"
#include "model.h"
#include "tp_big.cuh"

namespace allegro {

static ListView list_view(const NeighborList& nl) {
  ListView lv{nl.rowptr.as<int64_t>(), nl.keys.as<uint64_t>(), nl.revpos.as<int>(), {}};
  for (int k = 0; k < 9; ++k) lv.H[k] = nl.H[k];
  return lv;
}

namespace {
size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
}

// bytes of workspace per active edge / per atom of a chunk
// floats per edge of the per-irrep tensor-product buffers of the many-channel path (tp_big.cuh), max over layers
static size_t tbig_per_edge(const Plan& P) {
  size_t best = 0;
  for (int L = 1; L < P.hp.n_layers; ++L) {
    const Layer& ly = P.layers[L - 1];
    size_t f = 0;
    for (size_t o = 0; o < ly.out_irreps.size(); ++o)
      if (ly.out_off[o] >= 0) f += (size_t)(2 * ly.out_irreps[o].l + 1) * ly.out_npaths[o] * P.hp.n_channels;
    best = std::max(best, f);
  }
  return best;
}

static void ws_sizes(const Plan& P, bool big, size_t* per_edge, size_t* per_atom) {
  const allegro_hparams& hp = P.hp;
  const int n = hp.n_channels, NL = hp.n_layers;
  size_t f = GEO_W + hp.n_bessel;
  for (int i = 0; i + 1 < hp.two_body_nl; ++i) f += hp.two_body_dims[i];
  f += P.D;                         // y0
  f += (size_t)(NL + 1) * P.D;      // x^0..x^NL
  f += 2 * P.n_sc;                  // winit | w1
  int maxh = 4, maxv = 4;
  for (int L = 1; L <= NL; ++L) {
    const Layer& ly = P.layers[L - 1];
    if (L >= 2) f += P.n_sc;        // w^L
    f += P.n_sc;                    // s^L
    for (int i = 0; i + 1 < hp.latent_nl; ++i) { f += hp.latent_dims[i]; maxh = std::max(maxh, hp.latent_dims[i]); }
    f += P.D;                       // y^L
    if (L < NL) f += (size_t)n * ly.out_dim;
    maxv = std::max(maxv, std::max(ly.in_dim, ly.out_dim));
  }
  for (int i = 0; i + 1 < hp.two_body_nl; ++i) maxh = std::max(maxh, hp.two_body_dims[i]);
  f += 2 * P.D + 2 * maxh + P.n_sc + 2 * (size_t)n * maxv + (size_t)n * P.d_sh + 2 * P.n_sc + P.d_sh + 2 + hp.n_bessel;
  if (big) f += tbig_per_edge(P);
  *per_edge = f * sizeof(float) + 2 * sizeof(int) + sizeof(int64_t) + 64;
  *per_atom = ((size_t)NL + 1) * n * P.d_sh * sizeof(float) + sizeof(int) + sizeof(int64_t) + 64;
}

int ws_prepare(Model* m, int64_t cap_edges, int64_t cap_atoms) {
  Workspace& ws = m->ws;
  if (cap_edges <= ws.cap_edges && cap_atoms <= ws.cap_atoms && ws.arena.p) return 0;
  cap_edges = std::max<int64_t>(cap_edges, 256);
  cap_atoms = std::max<int64_t>(cap_atoms, 32);
  const Plan& P = m->plan;
  const allegro_hparams& hp = P.hp;
  const int n = hp.n_channels, NL = hp.n_layers;
  size_t pe, pa;
  ws_sizes(P, m->use_big, &pe, &pa);
  const size_t total = pe * cap_edges + pa * (cap_atoms + 1) + (1 << 16);
  if (int rc = ensure(m, &ws.arena, total)) return rc;
  char* base = ws.arena.as<char>();
  size_t off = 0;
  auto carve = [&](size_t bytes) { void* p = base + off; off = align_up(off + bytes, 256); return p; };
  auto cf = [&](size_t count) { return (float*)carve(count * sizeof(float)); };
  const size_t E = (size_t)cap_edges, A = (size_t)cap_atoms;
  ws.act_cnt = (int*)carve((A + 1) * sizeof(int));
  ws.rowptr_c = (int64_t*)carve((A + 2) * sizeof(int64_t));
  ws.e_center = (int*)carve(E * sizeof(int));
  ws.e_j = (int*)carve(E * sizeof(int));
  ws.e_lidx = (int64_t*)carve(E * sizeof(int64_t));
  ws.geo = cf(E * GEO_W);
  ws.bes = cf(E * hp.n_bessel);
  ws.z2b.clear();
  for (int i = 0; i + 1 < hp.two_body_nl; ++i) ws.z2b.push_back(cf(E * hp.two_body_dims[i]));
  ws.y0 = cf(E * P.D);
  ws.x.clear();
  for (int L = 0; L <= NL; ++L) ws.x.push_back(cf(E * P.D));
  ws.winit_w1 = cf(E * 2 * P.n_sc);
  ws.wenv.assign(NL, nullptr); ws.s.clear(); ws.zlat.assign(NL, {}); ws.ylat.clear(); ws.V.assign(NL, nullptr); ws.gamma.clear();
  int maxh = 4, maxv = 4;
  for (int i = 0; i + 1 < hp.two_body_nl; ++i) maxh = std::max(maxh, hp.two_body_dims[i]);
  for (int L = 1; L <= NL; ++L) {
    const Layer& ly = P.layers[L - 1];
    ws.wenv[L - 1] = (L == 1) ? ws.winit_w1 + P.n_sc : cf(E * P.n_sc);
    ws.s.push_back(cf(E * P.n_sc));
    for (int i = 0; i + 1 < hp.latent_nl; ++i) { ws.zlat[L - 1].push_back(cf(E * hp.latent_dims[i])); maxh = std::max(maxh, hp.latent_dims[i]); }
    ws.ylat.push_back(cf(E * P.D));
    if (L < NL) ws.V[L - 1] = cf(E * n * ly.out_dim);
    ws.gamma.push_back(cf(A * n * P.d_sh));
    maxv = std::max(maxv, std::max(ly.in_dim, ly.out_dim));
  }
  ws.xb[0] = cf(E * P.D); ws.xb[1] = cf(E * P.D);
  ws.zb[0] = cf(E * maxh); ws.zb[1] = cf(E * maxh);
  ws.sb = cf(E * P.n_sc);
  ws.vb[0] = cf(E * n * maxv); ws.vb[1] = cf(E * n * maxv);
  ws.ge = cf(E * n * P.d_sh);
  ws.wb = cf(E * 2 * P.n_sc);
  ws.yb = cf(E * P.d_sh);
  ws.ub = cf(E);
  ws.eps = cf(E);
  ws.bb = cf(E * hp.n_bessel);
  ws.gammab = cf(A * n * P.d_sh);
  ws.Tbig = m->use_big ? cf(E * tbig_per_edge(P)) : nullptr;
  if (off > total) { m->err = "internal: workspace carve overflow"; return ALLEGRO_ERR_ALLOC; }
  ws.cap_edges = cap_edges; ws.cap_atoms = cap_atoms;
  m->f16_rows_cap = cap_edges;
  return 0;
}

// algorithmic flop per active edge of one layer's tensor product on the FP32 pipe: 3 flop per coupling nonzero and channel
// (the backward has two coupling products); mix = the channel-mixing flop 2 n^2 (2l+1) per path through W_lin, which run on
// the tensor cores (mma.sync inside k_tp_*3, or the GEMM kernels for many channels, where the GEMM class counts them).
static double tp_work(const Plan& P, int L, bool backward, double* mix) {
  const Layer& ly = P.layers[L - 1];
  const double n = P.hp.n_channels;
  double f = 0;
  *mix = 0;
  for (const Path& p : ly.paths) {
    f += (backward ? 6.0 : 3.0) * n * (p.cg_end - p.cg_begin);
    if (L < P.hp.n_layers) *mix += 2.0 * n * n * (2 * ly.out_irreps[p.iro].l + 1);
  }
  return f;
}

static TpLayerDev make_tp(const Model* m, int L) {
  const Plan& P = m->plan;
  const Layer& ly = P.layers[L - 1];
  TpLayerDev t{};
  t.n = P.hp.n_channels; t.lmax = P.hp.lmax; t.dsh = P.d_sh; t.in_dim = ly.in_dim; t.out_dim = ly.out_dim;
  t.n_paths = (int)ly.paths.size(); t.n_out = (int)ly.out_irreps.size(); t.layer1 = (L == 1); t.has_lin = (L < P.hp.n_layers);
  t.path_tab = m->cg[L - 1].path_tab;
  for (int o = 0; o < t.n_out; ++o) {
    t.out_d3[o] = 2 * ly.out_irreps[o].l + 1; t.out_off[o] = ly.out_off[o]; t.out_np[o] = ly.out_npaths[o];
    t.wlin[o] = ly.w_lin[o];
  }
  return t;
}

// forward + backward for the centre atoms [a0, a1); m_cap bounds the number of active edges (list edges of the chunk)
static int run_chunk(Model* m, const double* pos, const int32_t* species, int64_t a0, int64_t a1, int64_t m_cap, cudaStream_t st) {
  const Plan& P = m->plan;
  const allegro_hparams& hp = P.hp;
  Workspace& ws = m->ws;
  NeighborList& nl = m->nl;
  int* flags = m->flags.as<int>();
  const int n = hp.n_channels, NL = hp.n_layers, D = P.D, nsc = P.n_sc, dsh = P.d_sh, S = hp.n_species, Nb = hp.n_bessel;
  const int64_t na = a1 - a0;
  const float inv_sqrt_navg = (float)(1.0 / std::sqrt(hp.avg_num_neighbors));
  const ListView lv = list_view(nl);
  const int T = 256;
  const unsigned gridWA = (unsigned)((na * 32 + T - 1) / T);
  // ---- active edges of the chunk
  prof_begin(m, st, KC_ACTIVE, 0);
  k_active<0><<<gridWA, T, 0, st>>>(pos, species, lv, a0, a1, hp.r_cut, hp.poly_p, Nb, ws.act_cnt, nullptr, nullptr, nullptr, nullptr,
                                    nullptr, nullptr, nullptr, 0, flags);
  if (int rc = scan_counts(m, ws.act_cnt, ws.rowptr_c, na, &ws.scan_tmp, nullptr, st)) return rc;
  k_ws_check<<<1, 1, 0, st>>>(ws.rowptr_c, na, ws.cap_edges, flags);
  k_ws_clamp<<<(unsigned)((na + 1 + T - 1) / T), T, 0, st>>>(ws.rowptr_c, na, flags);
  k_active<1><<<gridWA, T, 0, st>>>(pos, species, lv, a0, a1, hp.r_cut, hp.poly_p, Nb, nullptr, ws.rowptr_c, ws.e_center, ws.e_j,
                                    ws.e_lidx, ws.geo, ws.bes, m->g_list.as<float>(), ws.cap_edges, flags);
  k_add_count<<<1, 1, 0, st>>>(ws.rowptr_c + na, m->act_total.as<int64_t>());
  prof_end(m, st);
  m->launches += 5;
  const int64_t* Mptr = ws.rowptr_c + na;
  const float* w = m->d_w;
  const unsigned gridE = (unsigned)((m_cap + T - 1) / T), gridWE = (unsigned)((m_cap * 32 + T - 1) / T);
  if (m_cap <= 0) return 0;

  // Dependent linears are collected and launched as one chained kernel where the shapes allow (gemm_tc.cu)
  std::vector<GemmArgs> ch;
  // Returns true when every stage that carries a fused row dot went through the chained kernel (which computes it); false when
  // such a stage fell back to a single-linear launch, which does not — the caller then runs the dot as its own kernel.  (Groups
  // are decided one by one: a fallback of a group WITHOUT a dot must not make the caller add the dot a second time.)
  auto flush = [&]() {
    bool dots_fused = true;
    size_t i = 0;
    while (i < ch.size()) {
      const size_t cnt = std::min<size_t>(4, ch.size() - i);
      if (!launch_gemm_chain(m, ch.data() + i, (int)cnt, m_cap, st)) {
        for (size_t k = i; k < i + cnt; ++k) {
          if (ch[k].dot_out) dots_fused = false;
          launch_gemm(m, ch[k], m_cap, st);
        }
      }
      i += cnt;
    }
    ch.clear();
    return dots_fused;
  };
  // ---- F4: two-body MLP.  First layer = gather of the two one-hot columns + N_b-wide mat-vec.
  GemmArgs g;
  const int fan0 = 2 * S + Nb;
  {
    g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo;
    g.A0 = ws.bes; g.lda0 = Nb; g.K0 = Nb;
    g.W = w + P.w_two_body[0] + 2 * S; g.ldw = fan0; g.wtrans = 0; g.N = hp.two_body_dims[0];
    g.Wg = w + P.w_two_body[0]; g.ldwg = fan0; g.S = S; g.epi = EPI_GATHER2;
    if (hp.two_body_nl == 1) { m->err = "two_body MLP needs at least 2 linear layers"; return ALLEGRO_ERR_UNSUPPORTED; }
    g.C = ws.z2b[0]; g.ldc = hp.two_body_dims[0];
    ch.push_back(g);
    for (int i = 1; i < hp.two_body_nl; ++i) {
      g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo;
      g.A0 = ws.z2b[i - 1]; g.lda0 = g.K0 = hp.two_body_dims[i - 1]; g.pro = PRO_SILU;
      g.W = w + P.w_two_body[i]; g.ldw = hp.two_body_dims[i - 1]; g.N = hp.two_body_dims[i];
      if (i + 1 < hp.two_body_nl) { g.C = ws.z2b[i]; g.ldc = g.N; g.epi = EPI_STORE; }
      else { g.C = ws.y0; g.ldc = D; g.C2 = ws.x[0]; g.ldc2 = D; g.epi = EPI_Y_X; }   // x0 = u * y0
      ch.push_back(g);
    }
  }
  // ---- F5/F6 (layer 1): [W_init; W_env^1] x0 in one GEMM (adjacent in the blob)
  g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo;
  g.A0 = ws.x[0]; g.lda0 = g.K0 = D; g.W = w + P.w_init; g.ldw = D; g.N = 2 * nsc; g.C = ws.winit_w1; g.ldc = 2 * nsc;
  ch.push_back(g);
  flush();

  std::vector<TpLayerDev> tps;
  std::vector<int> te_f(NL), te_b(NL), d3m(NL);
  for (int L = 1; L <= NL; ++L) {
    const Layer& ly = P.layers[L - 1];
    tps.push_back(make_tp(m, L));
    const TpLayerDev& tp = tps.back();
    const int ldw_env = (L == 1) ? 2 * nsc : nsc;
    if (L >= 2) {   // F6
      g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo;
      g.A0 = ws.x[L - 1]; g.lda0 = g.K0 = D; g.W = w + ly.w_env; g.ldw = D; g.N = nsc; g.C = ws.wenv[L - 1]; g.ldc = nsc;
      ch.push_back(g);
      flush();   // latent MLP of layer L-1 + this projection of its output
    }
    // F7
    prof_begin(m, st, KC_GAMMA, 0);
    launch_gamma(ws.rowptr_c, ws.geo, ws.wenv[L - 1], ldw_env, n, hp.lmax, inv_sqrt_navg, ws.gamma[L - 1], na, st);
    prof_end(m, st);
    // F8, F9, F11
    int d3max = 1;
    for (int o = 0; o < tp.n_out; ++o) if (tp.has_lin || o == 0) d3max = std::max(d3max, tp.out_d3[o]);
    d3m[L - 1] = d3max;
    int npmax = 1;
    for (int o = 0; o < tp.n_out; ++o) if (tp.has_lin || o == 0) npmax = std::max(npmax, tp.out_np[o]);
    const size_t budget = (n <= 32 ? 56 : 100) * 1024;
    int TE = 32;
    while (TE > 4 && TE * d3max * n > 16 * TP_T * TP_MAXMT) TE >>= 1;
    auto smem_f = [&](int te, int pc) { return (size_t)(pc * n * (tp_ldr(te * d3max) + n) + te * 16) * sizeof(float); };
    int PC = npmax;
    while (PC > 1 && smem_f(TE, PC) > budget) --PC;
    while (TE > 4 && smem_f(TE, PC) > 200 * 1024) TE >>= 1;
    te_f[L - 1] = TE;
    TpIo io{}; io.Mptr = Mptr; io.e_center = ws.e_center; io.geo = ws.geo; io.gamma = ws.gamma[L - 1];
    io.vprev = (L >= 2) ? ws.V[L - 2] : nullptr; io.winit = ws.winit_w1; io.ldwi = 2 * nsc; io.w = w;
    io.s = ws.s[L - 1]; io.vout = (L < NL) ? ws.V[L - 1] : nullptr;
    {
      dim3 grid((unsigned)((m_cap + TE - 1) / TE), (unsigned)(tp.has_lin ? tp.n_out : 1));
      double mixf = 0;
      prof_begin(m, st, KC_TP_FWD, tp_work(P, L, false, &mixf));
      if (m->prof.on && !(m->use_big && tpbig_supported(tp))) m->prof.work[KC_TP_MIX] += mixf;
      if (m->use_big && tpbig_supported(tp)) {
        // many channels, n = 64: tensor product and channel mixing in one kernel (tp_mix.cu), T stays on chip
        if (m->use_tpmix && launch_tpmix_fwd(m, m->tp_sig[L - 1], st, tp, io)) {
          if (m->prof.on) m->prof.work[KC_TP_MIX16] += mixf;
          prof_end(m, st);
          prof_begin(m, st, KC_TP_FWD, 0);
        } else {
        // many channels: tensor product to per-irrep T buffers, channel mixing as tcgen05 GEMMs written straight into V^L
        TpBig big{};
        size_t off = 0;
        for (int o = 0; o < tp.n_out; ++o)
          if (tp.has_lin && tp.out_off[o] >= 0) { big.T[o] = ws.Tbig + off; off += (size_t)ws.cap_edges * tp.out_d3[o] * tp.out_np[o] * n; }
        launch_tpo(m->tp_sig[L - 1], false, m_cap, st, tp, io, big);
        prof_end(m, st);
        for (int o = 0; o < tp.n_out && tp.has_lin; ++o) {
          if (tp.out_off[o] < 0) continue;
          GemmArgs gm; gm.Mptr = Mptr; gm.geo = ws.geo; gm.m_mul = tp.out_d3[o];
          gm.A0 = big.T[o]; gm.lda0 = gm.K0 = tp.out_np[o] * n;
          gm.W = w + tp.wlin[o]; gm.ldw = tp.out_np[o] * n; gm.wtrans = 0; gm.N = n;
          gm.C = ws.V[L - 1]; gm.ldc = n; gm.cmap_d3 = tp.out_d3[o]; gm.cmap_od = tp.out_dim; gm.cmap_off = tp.out_off[o];
          launch_gemm(m, gm, m_cap * tp.out_d3[o], st);
        }
        prof_begin(m, st, KC_TP_FWD, 0);
        }
      } else if (tp3_supported(tp) && m->use_tp3) {
        const size_t sm3 = tp3_smem_bytes(tp, false);
        const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(3, (227 * 1024) / (sm3 + 2048)));
        const int64_t nsub = (m_cap + 256 / n - 1) / (256 / n);
        launch_tp3(m->tp_sig[L - 1], false, (int)std::min<int64_t>(nsub, (int64_t)m->num_sms * per_sm), st, tp, io);
      } else {
        launch_tp_fwd(m->tp_sig[L - 1], grid, smem_f(TE, PC), st, tp, io, TE, PC);
      }
      prof_end(m, st);
    }
    m->launches += 2;
    // F10: latent MLP on (x | s), residual update
    for (int i = 0; i < hp.latent_nl; ++i) {
      g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo;
      if (i == 0) { g.A0 = ws.x[L - 1]; g.lda0 = g.K0 = D; g.A1 = ws.s[L - 1]; g.lda1 = g.K1 = nsc; g.ldw = D + nsc; }
      else { g.A0 = ws.zlat[L - 1][i - 1]; g.lda0 = g.K0 = hp.latent_dims[i - 1]; g.pro = PRO_SILU; g.ldw = hp.latent_dims[i - 1]; }
      g.W = w + ly.w_latent[i]; g.N = hp.latent_dims[i];
      if (i + 1 < hp.latent_nl) { g.C = ws.zlat[L - 1][i]; g.ldc = g.N; }
      else {
        g.C = ws.ylat[L - 1]; g.ldc = D; g.C2 = ws.x[L]; g.ldc2 = D; g.aux = ws.x[L - 1]; g.ldaux = D;
        g.c_old = m->c_old[L - 1]; g.c_new = m->c_new[L - 1]; g.epi = EPI_RESIDUAL;
        if (L == NL) { g.dot_out = ws.eps; g.dotv = m->d_weff; }   // F12: eps_e = w_eff . x^NL_e in the epilogue
        if (hp.latent_nl == 1) { m->err = "latent MLP needs at least 2 linear layers"; return ALLEGRO_ERR_UNSUPPORTED; }
      }
      ch.push_back(g);
    }
  }
  const bool eps_fused = flush();
  // ---- F12
  prof_begin(m, st, KC_EDGE_MISC, 0);
  if (eps_fused) k_readout_eps<<<gridWA, T, 0, st>>>(ws.rowptr_c, ws.eps, species, a0, na, w + P.w_sigma, w + P.w_mu, m->e_atom.as<float>());
  else k_readout<<<gridWA, T, 0, st>>>(ws.rowptr_c, ws.x[NL], D, m->d_weff, species, a0, na, w + P.w_sigma, w + P.w_mu, m->e_atom.as<float>());
  prof_end(m, st);
  m->launches += 1;

  // ================= backward =================
  cudaMemsetAsync(ws.yb, 0, sizeof(float) * (size_t)m_cap * dsh, st);
  prof_begin(m, st, KC_EDGE_MISC, 0);
  // B1 + the first B3 dot: xbar^NL = sigma w_eff;  ubar = c_new (xbar^NL . y^NL)
  if (D % 4 == 0 && D / 4 <= 32 && ((D / 4) & (D / 4 - 1)) == 0)
    k_xbar_init_dot4<<<(unsigned)((m_cap * (D / 4) + T - 1) / T), T, 0, st>>>(Mptr, ws.geo, w + P.w_sigma, m->d_weff, D, ws.ylat[NL - 1],
                                                                               m->c_new[NL - 1], ws.xb[0], ws.ub);
  else
    k_xbar_init_dot<<<gridWE, T, 0, st>>>(Mptr, ws.geo, w + P.w_sigma, m->d_weff, D, ws.ylat[NL - 1], m->c_new[NL - 1], ws.xb[0], ws.ub);
  m->launches += 1;
  prof_end(m, st);
  int xcur = 0, vcur = 0;
  bool dot_done = true;   // the B3 dot of the layer about to be processed is already in ubar
  for (int L = NL; L >= 1; --L) {
    const Layer& ly = P.layers[L - 1];
    const TpLayerDev& tp = tps[L - 1];
    const float c_old = m->c_old[L - 1], c_new = m->c_new[L - 1];
    // B3: ubar += c_new (xbar . y) rides on the epilogue that finalised xbar^L (xbar_init for L = NL, else the W_env^T
    // accumulation still waiting in `ch`); the plain kernel below is the fallback when that stage could not be chained
    const bool dot_pending = !dot_done;
    // B3/B4: latent MLP backward.  ybar = c_new u xbar is applied as the prologue of the first transposed GEMM.
    {
      const float* cur = ws.xb[xcur];
      int zc = 0;
      for (int i = hp.latent_nl - 1; i >= 0; --i) {
        const int in_w = (i == 0) ? D + nsc : hp.latent_dims[i - 1];
        g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo; g.wtrans = 1;
        g.W = w + ly.w_latent[i]; g.ldw = in_w; g.N = in_w;
        g.A0 = cur; g.lda0 = g.K0 = hp.latent_dims[i];
        if (i == hp.latent_nl - 1) { g.pro = PRO_SCALE_U; g.c_new = c_new; }
        if (i > 0) {   // zbar = hbar * silu'(z)
          g.C = ws.zb[zc]; g.ldc = in_w; g.aux = ws.zlat[L - 1][i - 1]; g.ldaux = in_w; g.epi = EPI_DSILU;
          cur = ws.zb[zc]; zc ^= 1;
        } else {       // (xbar_in | sbar): xbar^{L-1} = c_old xbar^L + xbar_in
          g.C = ws.xb[xcur ^ 1]; g.ldc = D; g.aux = ws.xb[xcur]; g.ldaux = D; g.c_old = c_old; g.split = D;
          g.C2 = ws.sb; g.ldc2 = nsc; g.epi = EPI_SPLIT_RES;
        }
        ch.push_back(g);
      }
    }
    {
      const bool chained = flush();
      if (dot_pending && !chained) {
        prof_begin(m, st, KC_EDGE_MISC, 0);
        k_rowdot<<<gridWE, T, 0, st>>>(Mptr, ws.xb[xcur], ws.ylat[L - 1], D, c_new, 1, ws.ub);
        prof_end(m, st);
        m->launches += 1;
      }
    }
    xcur ^= 1;
    // B2 + B5: tensor-product backward -> Vbar^{L-1}, GE
    {
      const int d3max = d3m[L - 1];
      const size_t per_edge = (size_t)n * (ly.in_dim + dsh) + 16;
      int npmax = 1;
      for (int o = 0; o < tp.n_out; ++o) if (tp.has_lin || o == 0) npmax = std::max(npmax, tp.out_np[o]);
      const size_t budget = (n <= 32 ? 56 : 110) * 1024;
      auto smem_of = [&](int te, int pc) {
        return (per_edge * te + (size_t)(1 + pc) * n * (tp_ldr(te * d3max) + 4) + (size_t)pc * n * n) * sizeof(float);
      };
      int TE = 32;
      while (TE > 4 && smem_of(TE, 1) > budget / 2) TE >>= 1;
      int PC = npmax;
      while (PC > 1 && smem_of(TE, PC) > budget) --PC;
      if (smem_of(TE, PC) > 220 * 1024) { m->err = "tensor-product backward tile does not fit in shared memory"; return ALLEGRO_ERR_UNSUPPORTED; }
      TpIo io{}; io.Mptr = Mptr; io.e_center = ws.e_center; io.geo = ws.geo; io.gamma = ws.gamma[L - 1];
      io.vprev = (L >= 2) ? ws.V[L - 2] : nullptr; io.winit = ws.winit_w1; io.ldwi = 2 * nsc; io.w = w;
      io.sbar = ws.sb; io.vbar = (L < NL) ? ws.vb[vcur] : nullptr; io.vbar_prev = ws.vb[vcur ^ 1]; io.ge = ws.ge;
      io.wbar_init = ws.wb; io.ldwb = 2 * nsc; io.ybar = ws.yb;   // layer 1: B8 applied inside the kernel
      size_t smem = smem_of(TE, PC);
      double mixb = 0;
      prof_begin(m, st, KC_TP_BWD, tp_work(P, L, true, &mixb));
      if (m->prof.on && !(m->use_big && tpbig_supported(tp))) m->prof.work[KC_TP_MIX] += mixb;
      if (m->use_big && tpbig_supported(tp)) {
        TpBig big{};
        size_t off = 0;
        for (int o = 0; o < tp.n_out; ++o)
          if (tp.has_lin && tp.out_off[o] >= 0) { big.T[o] = ws.Tbig + off; off += (size_t)ws.cap_edges * tp.out_d3[o] * tp.out_np[o] * n; }
        prof_end(m, st);
        for (int o = 0; o < tp.n_out && tp.has_lin; ++o) {   // B2: Tbar_o = Vbar^L[., o, ., :] W_o
          if (tp.out_off[o] < 0) continue;
          GemmArgs gm; gm.Mptr = Mptr; gm.geo = ws.geo; gm.m_mul = tp.out_d3[o]; gm.wtrans = 1;
          gm.A0 = io.vbar; gm.lda0 = n; gm.K0 = n; gm.amap_d3 = tp.out_d3[o]; gm.amap_od = tp.out_dim; gm.amap_off = tp.out_off[o];
          gm.W = w + tp.wlin[o]; gm.ldw = tp.out_np[o] * n; gm.N = tp.out_np[o] * n;
          gm.C = big.T[o]; gm.ldc = tp.out_np[o] * n;
          launch_gemm(m, gm, m_cap * tp.out_d3[o], st);
        }
        prof_begin(m, st, KC_TP_BWD, 0);
        launch_tpo(m->tp_sig[L - 1], true, m_cap, st, tp, io, big);
      } else if (tp3_supported(tp) && m->use_tp3) {
        const size_t sm3 = tp3_smem_bytes(tp, true);
        const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(3, (227 * 1024) / (sm3 + 2048)));
        const int64_t nsub = (m_cap + 256 / n - 1) / (256 / n);
        launch_tp3(m->tp_sig[L - 1], true, (int)std::min<int64_t>(nsub, (int64_t)m->num_sms * per_sm), st, tp, io);
      } else {
        launch_tp_bwd(m->tp_sig[L - 1], dim3((unsigned)((m_cap + TE - 1) / TE)), smem, st, tp, io, TE, d3max, PC);
      }
      prof_end(m, st);
      vcur ^= 1;
      m->launches += 1;
    }
    // B5 (row reduction) + B6
    const int ldw_env = (L == 1) ? 2 * nsc : nsc;
    float* wbar = (L == 1) ? ws.wb + nsc : ws.wb;
    const int ldwb = (L == 1) ? 2 * nsc : nsc;
    prof_begin(m, st, KC_GAMMABAR, 0);
    launch_gammabar(ws.rowptr_c, ws.geo, ws.ge, ws.wenv[L - 1], ldw_env, n, hp.lmax, inv_sqrt_navg, wbar, ldwb, ws.yb, na, st);
    prof_end(m, st);
    m->launches += 1;
    if (L >= 2) {   // B7: xbar^{L-1} += W_env^T wbar
      g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo; g.wtrans = 1;
      g.A0 = ws.wb; g.lda0 = g.K0 = nsc; g.W = w + ly.w_env; g.ldw = D; g.N = D; g.C = ws.xb[xcur]; g.ldc = D; g.epi = EPI_ACCUM;
      // xbar^{L-1} is final here: the B3 dot of layer L-1 rides on this epilogue
      g.dot_out = ws.ub; g.dotB = ws.ylat[L - 2]; g.lddot = D; g.dot_scale = m->c_new[L - 2]; g.dot_accum = 1;
      ch.push_back(g);   // not flushed: the latent-MLP backward of layer L-1 chains behind it
      dot_done = false;
    }
  }
  // [W_init; W_env^1]^T [wbar_init; wbar^1] in one GEMM (B7 of layer 1 + B8; wbar_init comes from k_tp_bwd of layer 1)
  g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo; g.wtrans = 1;
  g.A0 = ws.wb; g.lda0 = g.K0 = 2 * nsc; g.W = w + P.w_init; g.ldw = D; g.N = D; g.C = ws.xb[xcur]; g.ldc = D; g.epi = EPI_ACCUM;
  g.dot_out = ws.ub; g.dotB = ws.y0; g.lddot = D; g.dot_scale = 1.0f; g.dot_accum = 1;   // B9: ubar += xbar0 . y0
  ch.push_back(g);
  // two-body MLP backward with ybar0 = u xbar0, chained behind the accumulation above
  {
    const float* cur = ws.xb[xcur];
    int zc = 0;
    for (int i = hp.two_body_nl - 1; i >= 1; --i) {
      g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo; g.wtrans = 1;
      g.W = w + P.w_two_body[i]; g.ldw = hp.two_body_dims[i - 1]; g.N = hp.two_body_dims[i - 1];
      g.A0 = cur; g.lda0 = g.K0 = hp.two_body_dims[i];
      if (i == hp.two_body_nl - 1) { g.pro = PRO_SCALE_U; g.c_new = 1.0f; }
      g.C = ws.zb[zc]; g.ldc = g.N; g.aux = ws.z2b[i - 1]; g.ldaux = g.N; g.epi = EPI_DSILU;
      cur = ws.zb[zc]; zc ^= 1;
      ch.push_back(g);
    }
    // bbar = W_1[:, 2S:]^T zbar_1
    g = GemmArgs(); g.Mptr = Mptr; g.geo = ws.geo; g.wtrans = 1;
    g.A0 = cur; g.lda0 = g.K0 = hp.two_body_dims[0]; g.W = w + P.w_two_body[0] + 2 * S; g.ldw = fan0; g.N = Nb;
    g.C = ws.bb; g.ldc = Nb;
    ch.push_back(g);
  }
  if (!flush()) {
    prof_begin(m, st, KC_EDGE_MISC, 0);
    k_rowdot<<<gridWE, T, 0, st>>>(Mptr, ws.xb[xcur], ws.y0, D, 1.0f, 1, ws.ub);
    prof_end(m, st);
    m->launches += 1;
  }
  // B10, B11
  prof_begin(m, st, KC_EDGE_MISC, 0);
  k_edge_grad<<<gridE, T, 0, st>>>(Mptr, ws.geo, ws.bes, ws.bb, ws.ub, ws.yb, ws.e_lidx, Nb, hp.lmax, (float)hp.r_cut, m->g_list.as<float>());
  prof_end(m, st);
  m->launches += 1;
  return 0;
}

int network_energy_forces(Model* m, const double* pos, const int32_t* species, int64_t N, double* E_out, double* F_out,
                          float* E_atom_out, cudaStream_t st, int64_t n_owned) {
  NeighborList& nl = m->nl;
  if (n_owned < 0 || n_owned > N) n_owned = N;                 // centre atoms [0, n_owned); the rest are ghosts (neighbours only)
  int* flags = m->flags.as<int>();
  if (int rc = ensure(m, &m->e_atom, sizeof(float) * (N + 1))) return rc;
  if (int rc = ensure(m, &m->e_partial, sizeof(double) * 1024)) return rc;
  if (int rc = ensure(m, &m->act_total, sizeof(int64_t))) return rc;
  cudaMemsetAsync(m->act_total.p, 0, sizeof(int64_t), st);
  const int T = 256;
  if (N > 0) {
    const double hs = 0.5 * nl.skin;
    k_check_inputs<<<(unsigned)((N + T - 1) / T), T, 0, st>>>(pos, nl.r_build.as<double>(), species, N, hs * hs, m->plan.hp.n_species, flags);
    m->launches += 1;
  }
  // single chunk when the workspace fits; otherwise atom chunks bounded by list edges (sized with the average row).  The
  // decision is taken once per (N, list capacity) and kept, so that a captured MD step never sees its buffers move.
  Workspace& ws = m->ws;
  const int64_t Ecap = std::max<int64_t>(nl.cap, 1);
  if (ws.for_N != N || ws.for_cap != Ecap || !ws.arena.p) {
    size_t pe, pa;
    ws_sizes(m->plan, m->use_big, &pe, &pa);
    size_t free_b = 0, total_b = 0;
    cudaMemGetInfo(&free_b, &total_b);
    const size_t budget = (size_t)(0.80 * (double)(free_b + ws.arena.bytes));
    int64_t n_chunks = 1;
    while ((pe * (size_t)(Ecap / n_chunks + 1) * ws.slack + pa * (size_t)(N / n_chunks + 1)) > budget && n_chunks < N) n_chunks *= 2;
    const int64_t atoms_per = (N + n_chunks - 1) / std::max<int64_t>(n_chunks, 1);
    const int64_t edges_per = (n_chunks == 1) ? Ecap : (int64_t)((double)Ecap / n_chunks * ws.slack) + 4096;
    if (int rc = ws_prepare(m, edges_per, atoms_per)) return rc;
    ws.for_N = N; ws.for_cap = Ecap; ws.atoms_per = std::max<int64_t>(atoms_per, 1);
  }
  const int64_t atoms_per = ws.atoms_per;
  if (n_owned < N) {
    // rows of the ghost atoms are not evaluated: their per-edge gradients and energies must read as zero
    cudaMemsetAsync(m->g_list.p, 0, sizeof(float) * 3 * (size_t)std::max<int64_t>(nl.cap, 1), st);
    cudaMemsetAsync(m->e_atom.p, 0, sizeof(float) * (N + 1), st);
  }
  for (int64_t a0 = 0; a0 < n_owned; a0 += atoms_per) {
    const int64_t a1 = std::min(n_owned, a0 + atoms_per);
    if (int rc = run_chunk(m, pos, species, a0, a1, m->ws.cap_edges, st)) return rc;
  }
  const ListView lv = list_view(nl);
  if (N > 0) {
    prof_begin(m, st, KC_GATHER, 0);
    k_force_gather<<<(unsigned)((N * 32 + T - 1) / T), T, 0, st>>>(lv, N, m->g_list.as<float>(), F_out, flags);
    const int nb = (int)std::min<int64_t>(1024, (N + 255) / 256);
    k_energy_partial<<<nb, 256, 0, st>>>(m->e_atom.as<float>(), n_owned, m->e_partial.as<double>());
    k_energy_final<<<1, 256, 0, st>>>(m->e_partial.as<double>(), nb, E_out, flags);
    prof_end(m, st);
    m->launches += 3;
  } else {
    cudaMemsetAsync(E_out, 0, sizeof(double), st);
  }
  if (E_atom_out && N > 0) cudaMemcpyAsync(E_atom_out, m->e_atom.p, sizeof(float) * N, cudaMemcpyDeviceToDevice, st);
  m->stats[1] = nl.E_list;
  m->stats[5] = (N + atoms_per - 1) / std::max<int64_t>(atoms_per, 1);   // atom chunks of this force call
  return 0;
}

// W = -sum_e rvec_e (x) g_e from the per-edge gradients of the last force evaluation
int network_virial(Model* m, const double* pos, double* W_out, cudaStream_t st) {
  NeighborList& nl = m->nl;
  const int64_t N = nl.N;
  const int nb = (int)std::max<int64_t>(1, std::min<int64_t>(1024, (N + 7) / 8));
  if (int rc = ensure(m, &m->vir_partial, sizeof(double) * 9 * 1024)) return rc;
  const ListView lv = list_view(nl);
  if (N == 0) { cudaMemsetAsync(W_out, 0, sizeof(double) * 9, st); return 0; }
  k_virial_partial<<<nb, 256, 0, st>>>(lv, pos, N, m->g_list.as<float>(), m->vir_partial.as<double>());
  k_virial_final<<<1, 32, 0, st>>>(m->vir_partial.as<double>(), nb, W_out);
  m->launches += 2;
  return 0;
}

}  // namespace allegro
