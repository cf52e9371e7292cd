// fenc_conv.cu -- fragment layout (Algorithm 1), Conv-aware planner, the HConv
// operation graph and its batched execution (R2.9), and AAC compress.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <functional>
#include <map>
#include <set>
#include <tuple>

#include "fenc_ctx.h"

static u32 next_pow2(u32 x) {
  u32 p = 1;
  while (p < x) p <<= 1;
  return p;
}

struct Term {
  int src;  // input ciphertext within a batch group: (g_in * S + u') * S + v'
  int amt;  // inner rotation amount (0 = the input itself)
  int w;    // weight plaintext index (fenc_wts_keys order)
};
struct OutCt {
  std::vector<int> diags;                // existing diagonals d, ascending
  std::vector<int> rots;                 // outer rotation amount of each existing diagonal (0 for d = 0)
  std::vector<std::vector<Term>> terms;  // per existing diagonal
};
// what the batched executor needs from a linear layer's operation graph (conv or fc)
struct LinGraph {
  size_t nin_bg = 0, BG = 1, n_w = 0;
  std::vector<OutCt> outs;                   // per output ciphertext of one batch group
  std::vector<std::pair<int, int>> inner;    // distinct (src, amt != 0), sorted
  std::map<std::pair<int, int>, int> inner_index;
  std::vector<int> rot_steps;                // distinct rotation amounts (inner and outer), ascending
  size_t n_outer = 0, n_pmult = 0;
};
struct ConvGraph : LinGraph {              // outs index: (g_out * S_out + u_o) * S_out + v_o
  fenc_conv_desc d;
  int n, M, S, S_out, m, B, ch, cs, G_in, G_out, H_out, W_out;
  int chp = 0, seg = 1;  // physical channel positions of a ciphertext = seg segments of ch positions (R2.11b; seg = 1: plain)
  int g = 1;             // baby steps over the channel diagonals (R2.9d); OutCt.diags then hold the giant steps
  std::vector<std::array<u32, 7>> wkeys;      // (u_o, v_o, g_out, g_in, dkey, i, j) per weight plaintext
  // diagonal keys: d in [0, ch); in a segmented layout also chp + d (d >= 1), the part of diagonal d that wraps inside
  // its segment (input positions pl < d, outer rotation (d - ch) cs instead of d cs)
  std::vector<int> dkeys() const {
    std::vector<int> k;
    for (int dd = 0; dd < ch; dd++) k.push_back(dd);
    if (seg > 1)
      for (int dd = 1; dd < ch; dd++) k.push_back(chp + dd);
    return k;
  }
  int diag_rot(int dkey) const {
    const int part = seg > 1 ? dkey / chp : 0, dl = seg > 1 ? dkey % chp : dkey;
    const long r = part ? (long)(dl - ch) * cs : (long)dl * cs;
    return (int)(((r % n) + n) % n);
  }
  // factored form (R2.9c), built on first use: a weight plaintext with ONE valid channel position is value x mask
  struct Mask { int cpos; std::vector<int> rows, cols; };
  bool factors_built = false, factorable = false;
  std::vector<int> mask_of;                   // weight index -> mask id (first-appearance order)
  std::vector<Mask> masks;
  void build_factors() {
    if (factors_built) return;
    factors_built = true, factorable = true;
    std::map<std::tuple<int, std::vector<int>, std::vector<int>>, int> seen;
    mask_of.assign(wkeys.size(), -1);
    for (size_t w = 0; w < wkeys.size(); w++) {
      const auto &wk = wkeys[w];
      auto cp = valid_cpos(wk[2], wk[3], wk[4]);
      if (cp.size() != 1) { factorable = false; mask_of.clear(); masks.clear(); return; }
      auto key = std::make_tuple(cp[0][0], valid_blocks(wk[0], wk[5], d.H, H_out), valid_blocks(wk[1], wk[6], d.W, W_out));
      auto it = seen.find(key);
      if (it == seen.end()) {
        it = seen.emplace(key, (int)masks.size()).first;
        masks.push_back(Mask{std::get<0>(key), std::get<1>(key), std::get<2>(key)});
      }
      mask_of[w] = it->second;
    }
  }
  double weight_value(const std::array<u32, 7> &wk, const double *w) const {  // the single valid channel position's K[o][c][i][j]
    auto cp = valid_cpos(wk[2], wk[3], wk[4]);
    const int K = d.K, Cw = d.depthwise ? 1 : (int)d.C_in;
    return w[(((size_t)cp[0][1] * Cw + (d.depthwise ? 0 : cp[0][2])) * K + wk[5]) * K + wk[6]];
  }
  void mask_slots(const Mask &mk, std::vector<double> &vec) const {
    vec.assign(n, 0.0);
    for (int bi : mk.rows)
      for (int bj : mk.cols) {
        size_t base = (size_t)mk.cpos * cs + (size_t)(bi * m + bj) * B;
        for (int b = 0; b < B; b++) vec[base + b] = 1.0;
      }
  }
  // R2.9 step 2: the validity conditions factorise into channel positions, block rows and block columns
  std::vector<std::array<int, 3>> valid_cpos(int go, int gi, int dkey) const {  // (physical position, o, c)
    std::vector<std::array<int, 3>> v;
    const int part = seg > 1 ? dkey / chp : 0, dl = seg > 1 ? dkey % chp : dkey;
    for (int sg = 0; sg < seg; sg++)
      for (int pl = 0; pl < ch; pl++) {
        if (seg > 1 && (pl >= dl) != (part == 0)) continue;  // part 0 stays inside its segment under a shift by dl, part 1 wraps
        int c = gi * ch + pl, o = go * ch + (((pl - dl) % ch + ch) % ch);
        if (c < (int)d.C_in && o < (int)d.C_out && (!d.depthwise || o == c)) v.push_back({sg * ch + pl, o, c});
      }
    return v;
  }
  std::vector<int> valid_blocks(int frag_o, int tap, int size_in, int size_out) const {
    std::vector<int> v;
    for (int bi = 0; bi < m; bi++) {
      int ho = bi * S_out + frag_o, hi = (int)d.stride * ho + tap - (int)d.pad;
      if (ho < size_out && hi >= 0 && hi < size_in) v.push_back(bi);
    }
    return v;
  }
  // slot vector of weight plaintext wk for kernel tensor w[C_out][C_in or 1][K][K]
  void weight_slots(const std::array<u32, 7> &wk, const double *w, std::vector<double> &vec) const {
    vec.assign(n, 0.0);
    const int uo = wk[0], vo = wk[1], go = wk[2], gi = wk[3], dd = wk[4], i = wk[5], j = wk[6];
    const int K = d.K, Cw = d.depthwise ? 1 : (int)d.C_in;
    auto cp = valid_cpos(go, gi, dd);
    auto rows = valid_blocks(uo, i, d.H, H_out), cols = valid_blocks(vo, j, d.W, W_out);
    for (auto &t : cp) {
      const double val = w[(((size_t)t[1] * Cw + (d.depthwise ? 0 : t[2])) * K + i) * K + j];
      for (int bi : rows)
        for (int bj : cols) {
          size_t base = (size_t)t[0] * cs + (size_t)(bi * m + bj) * B;
          for (int b = 0; b < B; b++) vec[base + b] = val;
        }
    }
    if (g > 1) {  // W' = Rot(W, j cs), j = d mod g: the baby step of this plaintext's diagonal (R2.9d)
      const size_t sh = (size_t)(dd % g) * cs % n;
      if (sh) std::rotate(vec.begin(), vec.begin() + sh, vec.end());
    }
  }
};

static fenc_status build_graph(fenc_ctx *ctx, const fenc_conv_desc *cd, int S, std::shared_ptr<ConvGraph> &out) {
  char keybuf[256];
  snprintf(keybuf, sizeof keybuf, "%u,%u,%u,%u,%u,%u,%u,%u,%d,%d,%u,%u,%u,%u", cd->BS, cd->C_in, cd->H, cd->W, cd->C_out, cd->K,
           cd->stride, cd->pad, cd->depthwise, S, cd->M, cd->seg_v, cd->B_cap, cd->bsgs);
  auto it = ctx->graphs.find(keybuf);
  if (it != ctx->graphs.end()) {
    out = std::static_pointer_cast<ConvGraph>(it->second);
    return FENC_OK;
  }
  if (cd->BS < 1 || cd->C_in < 1 || cd->C_out < 1 || cd->K < 1 || cd->stride < 1 || cd->H + 2 * cd->pad < cd->K || cd->W + 2 * cd->pad < cd->K)
    return fail(ctx, FENC_ERR_INVALID_ARG, "bad convolution shape");
  if (cd->depthwise && cd->C_in != cd->C_out) return fail(ctx, FENC_ERR_INVALID_ARG, "depthwise needs C_in == C_out");
  auto g = std::make_shared<ConvGraph>();
  g->d = *cd;
  g->n = ctx->n;
  g->M = cd->M ? cd->M : next_pow2(std::max(cd->H, cd->W));
  g->S = S;
  if (S < 1 || g->M % S || S % (int)cd->stride || (u32)g->M < std::max(cd->H, cd->W))
    return fail(ctx, FENC_ERR_LAYOUT, "S=%d must divide M=%d and be a multiple of the stride", S, g->M);
  g->m = g->M / S;
  const long m2 = (long)g->m * g->m;
  if (m2 > g->n || g->n % m2) return fail(ctx, FENC_ERR_LAYOUT, "m^2=%ld does not fit %d slots", m2, g->n);
  g->B = (int)std::min<long>(next_pow2(cd->BS), g->n / m2);
  if (cd->B_cap) g->B = (int)std::min<long>(g->B, cd->B_cap);
  if (g->B & (g->B - 1)) return fail(ctx, FENC_ERR_LAYOUT, "B_cap=%u must be a power of two", cd->B_cap);
  g->chp = (int)(g->n / (g->B * m2));
  g->ch = cd->seg_v ? (int)cd->seg_v : g->chp;
  if (g->ch < 1 || g->chp % g->ch) return fail(ctx, FENC_ERR_LAYOUT, "segment size %d must divide the %d channel positions", g->ch, g->chp);
  g->seg = g->chp / g->ch;
  g->cs = (int)(g->B * m2);
  g->G_in = (cd->C_in + g->ch - 1) / g->ch;
  g->G_out = (cd->C_out + g->ch - 1) / g->ch;
  g->BG = ((cd->BS + g->B - 1) / g->B + g->seg - 1) / g->seg;
  g->S_out = S / cd->stride;
  g->H_out = (cd->H + 2 * cd->pad - cd->K) / cd->stride + 1;
  g->W_out = (cd->W + 2 * cd->pad - cd->K) / cd->stride + 1;
  const int K = cd->K, So = g->S_out;
  const std::vector<int> dkeys = g->dkeys();
  std::set<std::pair<int, int>> inner;
  std::set<int> steps;
  g->outs.resize((size_t)g->G_out * So * So);
  for (int uo = 0; uo < So; uo++)
    for (int vo = 0; vo < So; vo++)
      for (int go = 0; go < g->G_out; go++) {
        OutCt &oc = g->outs[((size_t)go * So + uo) * So + vo];
        for (int dd : dkeys) {
          std::vector<Term> lst;
          for (int gi = 0; gi < g->G_in; gi++) {
            if (g->valid_cpos(go, gi, dd).empty()) continue;
            for (int i = 0; i < K; i++) {
              if (g->valid_blocks(uo, i, cd->H, g->H_out).empty()) continue;
              for (int j = 0; j < K; j++) {
                if (g->valid_blocks(vo, j, cd->W, g->W_out).empty()) continue;
                const int ti = (int)cd->stride * uo + i - (int)cd->pad, tj = (int)cd->stride * vo + j - (int)cd->pad;
                const int up = ((ti % S) + S) % S, di = (ti - up) / S;  // floor division
                const int vp = ((tj % S) + S) % S, dj = (tj - vp) / S;
                const long a = ((long)(di * g->m + dj) * g->B) % g->n;
                const int amt = (int)((a + g->n) % g->n);
                const int src = (gi * S + up) * S + vp;
                lst.push_back(Term{src, amt, (int)g->wkeys.size()});
                g->wkeys.push_back({(u32)uo, (u32)vo, (u32)go, (u32)gi, (u32)dd, (u32)i, (u32)j});
                if (amt) inner.insert({src, amt}), steps.insert(amt);
              }
            }
          }
          if (!lst.empty()) {
            oc.diags.push_back(dd);
            oc.rots.push_back(g->diag_rot(dd));
            oc.terms.push_back(std::move(lst));
            g->n_pmult += oc.terms.back().size();
            if (g->diag_rot(dd)) g->n_outer++, steps.insert(g->diag_rot(dd));
          }
        }
      }
  // ---- baby-step giant-step over the channel diagonals (R2.9d): regroup the plain graph's diagonals d = i gs + j by giant
  // step i; the baby step joins the inner amount, the outer rotation becomes i gs cs
  if (cd->bsgs > 1 && g->ch > 1) {
    auto regroup = [&](int gs, std::vector<OutCt> &outs, std::set<std::pair<int, int>> &inn, std::set<int> &stp, size_t &n_outer) {
      outs.assign(g->outs.size(), OutCt{});
      n_outer = 0;
      for (size_t o = 0; o < g->outs.size(); o++) {
        const OutCt &src = g->outs[o];
        std::map<int, std::vector<Term>> giants;
        for (size_t k = 0; k < src.diags.size(); k++) {
          // segmented layouts (R2.11b): dd = d + part*chp; both parts of diagonal d share its baby step, the giant key
          // keeps the part and its outer rotation is (i gs - part ch) cs
          const int dd = src.diags[k], part = g->seg > 1 ? dd / g->chp : 0, dl = g->seg > 1 ? dd % g->chp : dd;
          const int gi = dl / gs + part * g->chp, j = dl % gs;
          for (Term t : src.terms[k]) {
            t.amt = (int)(((long)t.amt + (long)j * g->cs) % g->n);
            giants[gi].push_back(t);
            if (t.amt) inn.insert({t.src, t.amt}), stp.insert(t.amt);
          }
        }
        for (auto &kv : giants) {
          const int kpart = g->seg > 1 ? kv.first / g->chp : 0, ki = g->seg > 1 ? kv.first % g->chp : kv.first;
          const long r0 = ((long)ki * gs - (long)kpart * g->ch) * g->cs;
          const int rot = (int)(((r0 % g->n) + g->n) % g->n);
          outs[o].diags.push_back(kv.first), outs[o].rots.push_back(rot), outs[o].terms.push_back(std::move(kv.second));
          if (rot) n_outer++, stp.insert(rot);
        }
      }
    };
    std::vector<int> cands;
    if (cd->bsgs == FENC_CONV_BSGS_AUTO) {
      for (int c = 1; c <= g->ch; c *= 2)
        if (g->ch % c == 0) cands.push_back(c);
    } else {
      const int c = (int)cd->bsgs;
      if (c > g->ch || g->ch % c || (c & (c - 1))) return fail(ctx, FENC_ERR_LAYOUT, "bsgs=%d must be a power of two dividing ch=%d", c, g->ch);
      cands.push_back(c);
    }
    size_t best = ~(size_t)0;
    int best_g = 1;
    for (int c : cands) {  // fewest rotations (inner + outer), ties to the smaller g
      std::vector<OutCt> o2;
      std::set<std::pair<int, int>> i2;
      std::set<int> s2;
      size_t no = 0;
      regroup(c, o2, i2, s2, no);
      if (i2.size() + no < best) best = i2.size() + no, best_g = c;
    }
    if (best_g > 1) {
      std::vector<OutCt> o2;
      size_t no = 0;
      inner.clear(), steps.clear();
      regroup(best_g, o2, inner, steps, no);
      g->outs = std::move(o2), g->n_outer = no, g->g = best_g;
    }
  }
  g->inner.assign(inner.begin(), inner.end());
  for (size_t i = 0; i < g->inner.size(); i++) g->inner_index[g->inner[i]] = (int)i;
  g->rot_steps.assign(steps.begin(), steps.end());
  g->nin_bg = (size_t)g->S * g->S * g->G_in, g->n_w = g->wkeys.size();
  ctx->graphs[keybuf] = g;
  out = g;
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ planner (R2.10)
static double paper_rot_count(const fenc_conv_desc *cd, int n, int M, int S) {
  // Table IX: n_in I(S,K) + n_out (ch - 1), I = ceil(K/S)^2 - 1 for K > S else 0 (A6, A18)
  const double alpha = (double)n / ((double)M * M);
  const double n_in = cd->C_in * cd->BS / alpha, n_out = cd->C_out * cd->BS / alpha, ch = alpha * S * S / cd->BS;
  const int c = (cd->K + S - 1) / S;
  const double inner = (S >= M || (int)cd->K <= S) ? 0.0 : (double)(c * c - 1);
  return n_in * inner + n_out * (ch - 1.0);
}

extern "C" fenc_status fenc_layout_plan(fenc_ctx *ctx, const fenc_conv_desc *cd, fenc_layout *out) {
  if (!ctx || !cd || !out) return FENC_ERR_INVALID_ARG;
  const int M = cd->M ? cd->M : next_pow2(std::max(cd->H, cd->W));
  const double alpha = (double)ctx->n / ((double)M * M);
  int S = cd->S;
  std::shared_ptr<ConvGraph> g;
  if (S == 0) {
    // Conv-aware selection: feasible powers of two under Eq. 7, arg-min of the exact rotation count
    std::vector<int> feas, ok;
    for (int s = 1; s <= M; s <<= 1)
      if (M % s == 0 && s % (int)cd->stride == 0 && (long)(M / s) * (M / s) <= ctx->n) feas.push_back(s);
    if (feas.empty()) return fail(ctx, FENC_ERR_LAYOUT, "no feasible block size");
    const double bound = std::sqrt(cd->BS * cd->C_in / alpha);
    for (int s : feas)
      if (s <= bound) ok.push_back(s);
    if (ok.empty()) ok.push_back(feas[0]);
    size_t best = ~(size_t)0;
    for (int s : ok) {
      std::shared_ptr<ConvGraph> gs;
      fenc_status st = build_graph(ctx, cd, s, gs);
      if (st != FENC_OK) return st;
      size_t tot = (gs->inner.size() + gs->n_outer) * gs->BG;
      if (tot < best) best = tot, S = s, g = gs;
    }
  } else {
    fenc_status st = build_graph(ctx, cd, S, g);
    if (st != FENC_OK) return st;
  }
  memset(out, 0, sizeof *out);
  out->S = g->S, out->S_out = g->S_out, out->M = g->M, out->M_out = g->M / cd->stride, out->m = g->m, out->B = g->B;
  out->ch = g->ch, out->cs = g->cs, out->G_in = g->G_in, out->G_out = g->G_out, out->BG = g->BG;
  out->ch_phys = g->chp, out->seg = g->seg;
  out->H_out = g->H_out, out->W_out = g->W_out;
  out->n_in_ct = g->S * g->S * g->G_in * g->BG;
  out->n_out_ct = g->S_out * g->S_out * g->G_out * g->BG;
  out->n_inner_rot = (u32)(g->inner.size() * g->BG);
  out->n_outer_rot = (u32)(g->n_outer * g->BG);
  out->n_pmult = (u32)(g->n_pmult * g->BG);
  out->n_distinct_pt = (u32)g->wkeys.size();
  out->n_rot_keys = (u32)g->rot_steps.size();
  if (g->rot_steps.size() > 512) return fail(ctx, FENC_ERR_LAYOUT, "more than 512 rotation amounts");
  for (size_t i = 0; i < g->rot_steps.size(); i++) out->rot_steps[i] = g->rot_steps[i];
  out->S_star_real = std::pow((double)cd->K * cd->K * cd->C_in * cd->BS / (alpha * cd->C_out), 0.25);
  out->paper_rot_count = paper_rot_count(cd, ctx->n, M, g->S);
  return FENC_OK;
}

static fenc_status graph_for(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, std::shared_ptr<ConvGraph> &g) {
  if (!lay || lay->S == 0) return fail(ctx, FENC_ERR_INVALID_ARG, "layout not planned");
  return build_graph(ctx, cd, (int)lay->S, g);
}

// ------------------------------------------------------------------------------------------------ Algorithm 1
// ciphertext (u, v, g, bg) holds at slot cpos*cs + (bi*m+bj)*B + b the value X[bg*B+b][g*ch+cpos][bi*S+u][bj*S+v]
extern "C" fenc_status fenc_encode_fragment(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, const double *x,
                                            uint32_t u, uint32_t v, uint32_t group, uint32_t bgi, uint32_t n_limbs, double scale,
                                            fenc_pt **out) {
  if (!ctx || !cd || !lay || !x || !out) return FENC_ERR_INVALID_ARG;
  if (u >= lay->S || v >= lay->S || group >= lay->G_in || bgi >= lay->BG) return fail(ctx, FENC_ERR_LAYOUT, "fragment index out of range");
  std::vector<double> vec(ctx->n, 0.0);
  const int m = lay->m, B = lay->B, S = lay->S;
  const u32 seg = lay->seg ? lay->seg : 1;
  for (u32 sg = 0; sg < seg; sg++)
    for (u32 pl = 0; pl < lay->ch; pl++) {
      u32 c = group * lay->ch + pl;
      if (c >= cd->C_in) continue;
      for (int b = 0; b < B; b++) {
        u32 bb = (bgi * seg + sg) * B + b;
        if (bb >= cd->BS) continue;
        for (int bi = 0; bi < m; bi++) {
          u32 h = bi * S + u;
          if (h >= cd->H) continue;
          for (int bj = 0; bj < m; bj++) {
            u32 w = bj * S + v;
            if (w < cd->W) vec[(size_t)(sg * lay->ch + pl) * lay->cs + (size_t)(bi * m + bj) * B + b] = x[(((size_t)bb * cd->C_in + c) * cd->H + h) * cd->W + w];
          }
        }
      }
    }
  return fenc_encode_slots(ctx, vec.data(), nullptr, n_limbs, scale, out);
}

extern "C" fenc_status fenc_decrypt_decode(fenc_ctx *ctx, const fenc_keys *K, const fenc_ct *ct, const fenc_conv_desc *cd,
                                           const fenc_layout *lay, int which, uint32_t u, uint32_t v, uint32_t group, uint32_t bgi,
                                           double *y) {
  if (!ctx || !K || !ct || !cd || !lay || !y) return FENC_ERR_INVALID_ARG;
  const u32 S = which ? lay->S_out : lay->S, C = which ? cd->C_out : cd->C_in, H = which ? lay->H_out : cd->H,
            W = which ? lay->W_out : cd->W, G = which ? lay->G_out : lay->G_in;
  if (u >= S || v >= S || group >= G || bgi >= lay->BG) return fail(ctx, FENC_ERR_LAYOUT, "fragment index out of range");
  std::vector<double> vec(ctx->n);
  fenc_status st = fenc_decrypt_slots(ctx, K, ct, vec.data(), nullptr);
  if (st != FENC_OK) return st;
  const int m = lay->m, B = lay->B;
  const u32 seg = lay->seg ? lay->seg : 1;
  for (u32 sg = 0; sg < seg; sg++)
    for (u32 pl = 0; pl < lay->ch; pl++) {
      u32 c = group * lay->ch + pl;
      if (c >= C) continue;
      for (int b = 0; b < B; b++) {
        u32 bb = (bgi * seg + sg) * B + b;
        if (bb >= cd->BS) continue;
        for (int bi = 0; bi < m; bi++) {
          u32 h = bi * S + u;
          if (h >= H) continue;
          for (int bj = 0; bj < m; bj++) {
            u32 w = bj * S + v;
            if (w < W) y[(((size_t)bb * C + c) * H + h) * W + w] = vec[(size_t)(sg * lay->ch + pl) * lay->cs + (size_t)(bi * m + bj) * B + b];
          }
        }
      }
    }
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ weights
extern "C" fenc_status fenc_wts_keys(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, uint32_t *keys7,
                                     size_t capacity, size_t *n) {
  if (!ctx || !cd || !n) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  *n = g->wkeys.size();
  if (keys7) {
    if (capacity < g->wkeys.size()) return fail(ctx, FENC_ERR_INVALID_ARG, "capacity %zu < %zu weight plaintexts", capacity, g->wkeys.size());
    for (size_t i = 0; i < g->wkeys.size(); i++) memcpy(keys7 + 7 * i, g->wkeys[i].data(), 7 * sizeof(u32));
  }
  return FENC_OK;
}

static u64 fnv64(const void *data, size_t n, u64 h) {
  const unsigned char *p = (const unsigned char *)data;
  for (size_t i = 0; i < n; i++) h = (h ^ p[i]) * 0x100000001B3ull;
  return h;
}
// Encodes (or takes pre-encoded) every weight plaintext; plaintexts with identical coefficients are stored once
// (content deduplication: in the large-batch layouts the same masked constant serves several fragments).
static fenc_status make_wts(fenc_ctx *ctx, size_t n, const std::function<void(size_t, std::vector<double> &)> &slots,
                            const int64_t *coeffs, uint32_t n_limbs, double scale, fenc_wts **out) {
  if (n_limbs < 1 || (int)n_limbs > ctx->nq) return FENC_ERR_INVALID_ARG;
  const int L = n_limbs;
  const size_t N = ctx->N;
  std::unique_ptr<fenc_wts, void (*)(fenc_wts *)> W(new fenc_wts{ctx, L, scale > 0 ? scale : (double)ctx->mod[L - 1], n},
                                                     fenc_wts_free);  // A14: s_w = q_{L-1}
  W->slot.resize(n);
  std::vector<std::vector<int64_t>> uniq;
  std::map<std::pair<u64, u64>, int> seen;
  std::vector<double> vec;
  std::vector<int64_t> c(N);
  for (size_t i = 0; i < n; i++) {
    const int64_t *src = coeffs ? coeffs + i * N : c.data();
    if (!coeffs) {
      slots(i, vec);
      fh::encode_slots(ctx->logN, vec.data(), nullptr, W->scale, c.data());
    }
    std::pair<u64, u64> key{fnv64(src, N * 8, 0xcbf29ce484222325ull), fnv64(src, N * 8, 0x9E3779B97F4A7C15ull)};
    auto it = seen.find(key);
    if (it != seen.end() && memcmp(uniq[it->second].data(), src, N * 8) == 0) {
      W->slot[i] = it->second;
    } else {
      W->slot[i] = (int)uniq.size();
      if (it == seen.end()) seen[key] = (int)uniq.size();
      uniq.emplace_back(src, src + N);
    }
  }
  W->n_unique = uniq.size();
  W->d_all = dalloc_t<u64>(ctx, W->n_unique * L * N);
  if (!W->d_all) return fail(ctx, FENC_ERR_OOM, "weight plaintexts (%zu x %d limbs)", W->n_unique, L);
  for (size_t i = 0; i < uniq.size(); i++) {
    fenc_status st = coeffs_to_mont(ctx, uniq[i].data(), L, W->d_all + i * L * N);
    if (st != FENC_OK) return st;
  }
  if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return FENC_ERR_CUDA;
  *out = W.release();
  return FENC_OK;
}
extern "C" fenc_status fenc_conv_weights(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, const double *w,
                                         uint32_t n_limbs, double scale, fenc_wts **out) {
  if (!ctx || !cd || !w || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  const ConvGraph *gp = g.get();
  return make_wts(ctx, gp->wkeys.size(), [gp, w](size_t i, std::vector<double> &v) { gp->weight_slots(gp->wkeys[i], w, v); }, nullptr,
                  n_limbs, scale, out);
}
extern "C" fenc_status fenc_conv_weights_from_coeffs(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay,
                                                     const int64_t *coeffs, size_t n, uint32_t n_limbs, double scale,
                                                     fenc_wts **out) {
  if (!ctx || !cd || !coeffs || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  if (n != g->wkeys.size()) return fail(ctx, FENC_ERR_MISMATCH, "expected %zu weight plaintexts, got %zu", g->wkeys.size(), n);
  return make_wts(ctx, n, nullptr, coeffs, n_limbs, scale, out);
}
extern "C" void fenc_wts_free(fenc_wts *W) {
  if (!W) return;
  cudaStreamSynchronize(W->ctx->stream);
  dfree(W->ctx, W->d_all);
  dfree(W->ctx, W->d_k);
  delete W;
}

// ------------------------------------------------------------------------------------------------ factored weights (R2.9c)
extern "C" fenc_status fenc_wts_factors(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, uint32_t *mask_of, size_t capacity,
                                        size_t *n, size_t *n_masks) {
  if (!ctx || !cd || !n || !n_masks) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  g->build_factors();
  if (!g->factorable) return fail(ctx, FENC_ERR_LAYOUT, "a weight plaintext has several valid channel positions (ch = %d): not value x mask", g->ch);
  *n = g->wkeys.size(), *n_masks = g->masks.size();
  if (mask_of) {
    if (capacity < g->wkeys.size()) return fail(ctx, FENC_ERR_INVALID_ARG, "capacity %zu < %zu weights", capacity, g->wkeys.size());
    for (size_t i = 0; i < g->wkeys.size(); i++) mask_of[i] = (uint32_t)g->mask_of[i];
  }
  return FENC_OK;
}
extern "C" fenc_status fenc_wts_mask_slots(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, uint32_t mask_id, double *slots) {
  if (!ctx || !cd || !slots) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  g->build_factors();
  if (!g->factorable || mask_id >= g->masks.size()) return fail(ctx, FENC_ERR_LAYOUT, "no such mask");
  std::vector<double> v;
  g->mask_slots(g->masks[mask_id], v);
  memcpy(slots, v.data(), v.size() * sizeof(double));
  return FENC_OK;
}
// k[n]: integer multipliers; mask coefficient vectors either given (parity path) or encoded here at E2
static fenc_status make_factored(fenc_ctx *ctx, ConvGraph &g, const int64_t *k, const int64_t *mask_coeffs, uint32_t n_limbs, double E1,
                                 double E2, fenc_wts **out) {
  if (n_limbs < 1 || (int)n_limbs > ctx->nq) return FENC_ERR_INVALID_ARG;
  const int L = n_limbs;
  const size_t N = ctx->N, n = g.wkeys.size(), nm = g.masks.size();
  std::unique_ptr<fenc_wts, void (*)(fenc_wts *)> W(new fenc_wts{ctx, L, E1 * E2, n}, fenc_wts_free);
  W->factored = true, W->n_unique = nm, W->slot = g.mask_of;
  W->k_fp64 = true;
  for (int t = 0; t < L; t++) W->k_fp64 = W->k_fp64 && fh::f64_modulus(ctx->mod[t], ctx->logN);
  // Mode of the scalar MAC (fenc_elem.cu): with every modulus below 2^50 and small multipliers the ciphertext word is
  // split in 2 x 25 (or 3 x 17) bits and the SIGNED k multiplies the pieces; `lazy` products plus a reduced remainder
  // (< 2^49) must sum exactly in a double: 2^49 + lazy 2^B kmax <= 2^53.  FENC_SMAC_MODE=1|2|3 forces a mode that is valid
  // (diagnostics and tests: all modes give identical limbs).
  {
    u64 kmax = 1, qmax = 0;
    for (size_t i = 0; i < n; i++) kmax = std::max<u64>(kmax, (u64)(k[i] < 0 ? -k[i] : k[i]));
    for (int t = 0; t < L; t++) qmax = std::max(qmax, ctx->mod[t]);
    const long double room = 9007199254740992.0L - 562949953421312.0L;  // 2^53 - 2^49
    const u64 lazy2 = (u64)(room / (33554432.0L * (long double)kmax)), lazy3 = (u64)(room / (131072.0L * (long double)kmax));
    const u64 lazy1 = (((u64)1 << 53) / qmax) - 1;
    const char *force = getenv("FENC_SMAC_MODE");
    const int want = force ? atoi(force) : 0;
    int mode = !W->k_fp64 ? 0 : (lazy2 >= 8 ? 2 : (lazy3 >= 8 ? 3 : 1));
    if (W->k_fp64 && want == 1) mode = 1;
    if (W->k_fp64 && want == 2 && lazy2 >= 1) mode = 2;
    if (W->k_fp64 && want == 3 && lazy3 >= 1) mode = 3;
    W->k_mode = mode;
    const u64 lz = mode == 2 ? lazy2 : (mode == 3 ? lazy3 : (mode == 1 ? lazy1 : (u64)std::max(1, ctx->max_lazy - 1)));
    W->k_lazy = (int)std::min<u64>(lz, 1u << 20);
  }
  W->d_all = dalloc_t<u64>(ctx, nm * L * N);
  W->d_k = dalloc_t<ShoupC>(ctx, n * L);
  if (!W->d_all || !W->d_k) return fail(ctx, FENC_ERR_OOM, "factored weights (%zu masks, %zu scalars)", nm, n);
  std::vector<double> vec;
  std::vector<int64_t> c(N);
  for (size_t i = 0; i < nm; i++) {
    const int64_t *src = mask_coeffs ? mask_coeffs + i * N : c.data();
    if (!mask_coeffs) {
      g.mask_slots(g.masks[i], vec);
      fh::encode_slots(ctx->logN, vec.data(), nullptr, E2, c.data());
    }
    fenc_status st = coeffs_to_mont(ctx, src, L, W->d_all + i * L * N);
    if (st != FENC_OK) return st;
    if (cudaStreamSynchronize(ctx->stream) != cudaSuccess) return FENC_ERR_CUDA;  // c is reused
  }
  std::vector<ShoupC> kp(n * L);
  for (size_t i = 0; i < n; i++)
    for (int t = 0; t < L; t++) {
      const u64 q = ctx->mod[t];
      const u64 mag = (u64)(k[i] < 0 ? -k[i] : k[i]) % q;
      const u64 r = (k[i] < 0 && mag) ? q - mag : mag;
      kp[i * L + t] = W->k_mode >= 2 ? ShoupC{fh::double_bits((double)k[i]), 0}
                      : W->k_mode == 1 ? ShoupC{fh::double_bits((double)r), fh::double_bits((double)((long double)r / (long double)q))}
                                       : ShoupC{fh::to_mont(r, q), 0};
    }
  if (cudaMemcpyAsync(W->d_k, kp.data(), kp.size() * sizeof(ShoupC), cudaMemcpyHostToDevice, ctx->stream) != cudaSuccess ||
      cudaStreamSynchronize(ctx->stream) != cudaSuccess)
    return FENC_ERR_CUDA;
  *out = W.release();
  return FENC_OK;
}
// (E1, E2) with E1 E2 = s_w, E1 = 2^ceil(log2(s_w)/2)
static void factor_scales(double sw, double *E1, double *E2) {
  int bits = 0;
  while (std::ldexp(1.0, bits) < sw) bits++;
  *E1 = std::ldexp(1.0, (bits + 1) / 2);
  *E2 = sw / *E1;  // exact: a division by a power of two
}
extern "C" fenc_status fenc_conv_weights_factored(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay, const double *w,
                                                  uint32_t n_limbs, double scale, fenc_wts **out) {
  if (!ctx || !cd || !w || !out || n_limbs < 1 || (int)n_limbs > ctx->nq) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  g->build_factors();
  if (!g->factorable) return fail(ctx, FENC_ERR_LAYOUT, "a weight plaintext has several valid channel positions (ch = %d): not value x mask", g->ch);
  double E1, E2;
  factor_scales(scale > 0 ? scale : (double)ctx->mod[n_limbs - 1], &E1, &E2);
  std::vector<int64_t> k(g->wkeys.size());
  for (size_t i = 0; i < k.size(); i++) {
    // round_half_up(v E1): v E1 is exact (E1 a power of two), its floor and fractional part are exact doubles
    const double a = g->weight_value(g->wkeys[i], w) * E1, f = std::floor(a);
    k[i] = (int64_t)f + ((a - f) >= 0.5 ? 1 : 0);
  }
  return make_factored(ctx, *g, k.data(), nullptr, n_limbs, E1, E2, out);
}
extern "C" fenc_status fenc_conv_weights_factored_from_ints(fenc_ctx *ctx, const fenc_conv_desc *cd, const fenc_layout *lay,
                                                            const int64_t *k, size_t n, const int64_t *mask_coeffs, size_t n_masks,
                                                            uint32_t n_limbs, double E1, double E2, fenc_wts **out) {
  if (!ctx || !cd || !k || !mask_coeffs || !out || !(E1 > 0) || !(E2 > 0)) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> g;
  fenc_status st = graph_for(ctx, cd, lay, g);
  if (st != FENC_OK) return st;
  g->build_factors();
  if (!g->factorable) return fail(ctx, FENC_ERR_LAYOUT, "a weight plaintext has several valid channel positions (ch = %d): not value x mask", g->ch);
  if (n != g->wkeys.size() || n_masks != g->masks.size())
    return fail(ctx, FENC_ERR_MISMATCH, "expected %zu multipliers and %zu masks, got %zu and %zu", g->wkeys.size(), g->masks.size(), n, n_masks);
  return make_factored(ctx, *g, k, mask_coeffs, n_limbs, E1, E2, out);
}

// ------------------------------------------------------------------------------------------------ HConv (R2.9)
// 1. inner rotations: every distinct (input ciphertext, amount) once, always from the original input, ONE batch
// 2. MAC: P_d = sum over (g_in, taps) of R (*) W per existing channel diagonal d, one launch for all (bg, output, d)
// 3. outer rotations: Rot(P_d, d cs) for d != 0, ONE batch;  4. Y = P_0 + sum of those;  5. one rescale per output (A13)
static fenc_status run_linear(fenc_ctx *ctx, const fenc_keys *K, const LinGraph &g, const fenc_wts *W, fenc_ct *const *in,
                              size_t n_in, int do_rescale, fenc_ct **out, size_t cap, size_t *n_out) {
  Scope sc(ctx);
  fenc_status st;
  const size_t nin_bg = g.nin_bg, nout_bg = g.outs.size(), BG = g.BG;
  if (n_in != nin_bg * BG) return fail(ctx, FENC_ERR_MISMATCH, "expected %zu input ciphertexts, got %zu", nin_bg * BG, n_in);
  if (cap < nout_bg * BG) return fail(ctx, FENC_ERR_INVALID_ARG, "output capacity %zu < %zu", cap, nout_bg * BG);
  if (W->n != g.n_w) return fail(ctx, FENC_ERR_MISMATCH, "weights belong to another layer");
  const int L = in[0]->L;
  const double s_in = in[0]->scale;
  for (size_t i = 0; i < n_in; i++)
    if (in[i]->L != L || std::fabs(in[i]->scale - s_in) > 1e-9 * s_in) return fail(ctx, FENC_ERR_MISMATCH, "inputs differ in level or scale");
  if (W->L != L) return fail(ctx, FENC_ERR_MISMATCH, "weights at %d limbs, inputs at %d", W->L, L);
  if (do_rescale && L < 2) return fail(ctx, FENC_ERR_LEVEL, "no level left to rescale");
  for (auto &oc : g.outs)
    if (oc.diags.empty()) return fail(ctx, FENC_ERR_LAYOUT, "an output ciphertext receives no term");
  const size_t N = ctx->N, CT = (size_t)2 * L * N;
  const size_t n_inner = g.inner.size();
  // ---- 1. inner rotations
  u64 *Rbuf = n_inner ? sc.alloc<u64>(n_inner * BG * CT) : nullptr;
  if (n_inner && !Rbuf) return fail(ctx, FENC_ERR_OOM, "inner-rotation results (%zu ciphertexts)", n_inner * BG);
  {
    std::vector<const u64 *> vin;
    std::vector<u64 *> vout;
    std::vector<int> vs, src_of;
    std::vector<const u64 *> srcs;  // hoisted form: the distinct inputs that are rotated at all
    std::map<const u64 *, int> src_index;
    for (size_t bg = 0; bg < BG; bg++)
      for (size_t r = 0; r < n_inner; r++) {
        const u64 *x = in[bg * nin_bg + g.inner[r].first]->d;
        vin.push_back(x);
        vs.push_back(g.inner[r].second);
        vout.push_back(Rbuf + (bg * n_inner + r) * CT);
        auto ins = src_index.insert({x, (int)srcs.size()});
        if (ins.second) srcs.push_back(x);
        src_of.push_back(ins.first->second);
      }
    st = ctx->hoist_inner ? rotate_hoisted_raw(ctx, K, L, srcs, src_of, vs, vout) : rotate_raw(ctx, K, L, vin, vs, vout);
    if (st != FENC_OK) return st;
  }
  // ---- 2. MAC over every (bg, output, diagonal)
  size_t n_P = 0, n_rot_out = 0;
  for (auto &oc : g.outs) {
    if (!(oc.diags.size() == 1 && oc.rots[0] == 0)) n_P += oc.diags.size();  // a lone unrotated diagonal is summed in place
    for (int r : oc.rots) n_rot_out += r != 0;
  }
  std::vector<fenc_ct *> res(nout_bg * BG, nullptr);
  const double s_acc = s_in * W->scale;
  u64 *Ybuf = do_rescale ? sc.alloc<u64>(nout_bg * BG * CT) : nullptr;  // pre-rescale sums
  u64 *Pbuf = n_P ? sc.alloc<u64>(n_P * BG * CT) : nullptr;               // diagonal partial sums
  u64 *Obuf = n_rot_out ? sc.alloc<u64>(n_rot_out * BG * CT) : nullptr;   // outer-rotation results
  if ((do_rescale && !Ybuf) || (n_P && !Pbuf) || (n_rot_out && !Obuf)) return fail(ctx, FENC_ERR_OOM, "hconv partial sums");
  for (size_t i = 0; i < res.size(); i++) {
    res[i] = sc.ct(do_rescale ? L - 1 : L, do_rescale ? s_acc / (double)ctx->mod[L - 1] : s_acc);
    if (!res[i]) return fail(ctx, FENC_ERR_OOM, "hconv outputs");
  }
  MacJob job;
  SmacJob sjob;  // factored weights (R2.9c): scalar multiply-accumulates, one plaintext product per mask
  std::vector<const u64 *> rot_in, sum_terms;
  std::vector<u64 *> rot_out, sum_out;
  std::vector<int> rot_step, sum_start{0};
  size_t pi = 0, oi = 0;
  for (size_t bg = 0; bg < BG; bg++)
    for (size_t o = 0; o < nout_bg; o++) {
      const OutCt &oc = g.outs[o];
      u64 *Y = do_rescale ? Ybuf + (bg * nout_bg + o) * CT : res[bg * nout_bg + o]->d;
      const bool single = oc.diags.size() == 1 && oc.rots[0] == 0;
      for (size_t k = 0; k < oc.diags.size(); k++) {
        u64 *P = single ? Y : Pbuf + (pi++) * CT;
        auto ct_of = [&](const Term &t) { return t.amt ? Rbuf + (bg * n_inner + g.inner_index.at({t.src, t.amt})) * CT : in[bg * nin_bg + t.src]->d; };
        if (W->factored) {
          sjob.terms.emplace_back();
          for (const Term &t : oc.terms[k]) sjob.terms.back().push_back({ct_of(t), t.w, W->d_all + (size_t)W->slot[t.w] * L * N});
          std::stable_sort(sjob.terms.back().begin(), sjob.terms.back().end(), [](const SmacTerm &a, const SmacTerm &b) { return a.mask < b.mask; });
          sjob.outs.push_back(P);
        } else {
          job.terms.emplace_back();
          for (const Term &t : oc.terms[k]) job.terms.back().push_back({ct_of(t), W->d_all + (size_t)W->slot[t.w] * L * N});
          job.outs.push_back(P);
        }
        if (single) continue;
        if (oc.rots[k] == 0) sum_terms.push_back(P);
        else {
          u64 *R = Obuf + (oi++) * CT;
          rot_in.push_back(P), rot_out.push_back(R), rot_step.push_back(oc.rots[k]);
          sum_terms.push_back(R);
        }
      }
      if (!single) sum_start.push_back((int)sum_terms.size()), sum_out.push_back(Y);
    }
  st = W->factored ? run_smac(ctx, sjob, W, L) : run_mac(ctx, job, L);
  if (st != FENC_OK) return st;
  // ---- 3. outer rotations, 4. sums
  st = rotate_raw(ctx, K, L, rot_in, rot_step, rot_out);
  if (st != FENC_OK) return st;
  if (!sum_out.empty()) {
    DescStage ds(ctx);
    size_t o0 = ds.add(sum_terms), o1 = ds.add(sum_start), o2 = ds.add(sum_out);
    char *base = ds.commit();
    if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    CUDA_OK(ctx, k_add_many(ctx->k, (const u64 *const *)(base + o0), (const int *)(base + o1), (u64 *const *)(base + o2), (int)sum_out.size(), L, (int)sum_terms.size()));
  }
  // ---- 5. rescale
  if (do_rescale) {
    std::vector<BatchItem> items(res.size());
    for (size_t i = 0; i < res.size(); i++) {
      items[i] = BatchItem{};
      items[i].sub_in = Ybuf + i * CT, items[i].out = res[i]->d;
    }
    st = rescale_batch(ctx, L, items);
    if (st != FENC_OK) return st;
  }
  sc.ok = true;
  for (size_t i = 0; i < res.size(); i++) out[i] = res[i];
  *n_out = res.size();
  return FENC_OK;
}

extern "C" fenc_status fenc_hconv(fenc_ctx *ctx, const fenc_keys *K, const fenc_conv_desc *cd, const fenc_layout *lay,
                                  const fenc_wts *W, fenc_ct *const *in, size_t n_in, int do_rescale, fenc_ct **out,
                                  size_t cap, size_t *n_out) {
  if (!ctx || !K || !cd || !lay || !W || !in || !out || !n_out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<ConvGraph> gp;
  fenc_status st = graph_for(ctx, cd, lay, gp);
  if (st != FENC_OK) return st;
  return run_linear(ctx, K, *gp, W, in, n_in, do_rescale, out, cap, n_out);
}

// ------------------------------------------------------------------------------------------------ AAC compress (R2.11)
extern "C" fenc_status fenc_compress(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n_in, const fenc_pt *mask_c,
                                     const uint32_t *term_out, const uint32_t *term_src, const int32_t *term_rot, size_t n_terms,
                                     int do_rescale, fenc_ct **out, size_t n_out) {
  Scope sc(ctx);
  if (!ctx || !K || !in || !term_out || !term_src || !term_rot || !out || n_in == 0 || n_out == 0) return FENC_ERR_INVALID_ARG;
  fenc_pt *mask = const_cast<fenc_pt *>(mask_c);
  const int L = in[0]->L;
  const double s_in = in[0]->scale;
  for (size_t i = 0; i < n_in; i++)
    if (in[i]->L != L || std::fabs(in[i]->scale - s_in) > 1e-9 * s_in) return fail(ctx, FENC_ERR_MISMATCH, "sources differ in level or scale");
  if (mask && mask->L != L) return fail(ctx, FENC_ERR_MISMATCH, "mask level");
  if (do_rescale && L < 2) return fail(ctx, FENC_ERR_LEVEL, "no level left to rescale");
  const size_t N = ctx->N, CT = (size_t)2 * L * N;
  std::vector<int> cnt(n_out, 0);
  for (size_t i = 0; i < n_terms; i++) {
    if (term_out[i] >= n_out || term_src[i] >= n_in) return fail(ctx, FENC_ERR_INVALID_ARG, "compress term out of range");
    cnt[term_out[i]]++;
  }
  for (size_t t = 0; t < n_out; t++)
    if (!cnt[t]) return fail(ctx, FENC_ERR_INVALID_ARG, "compress output %zu has no term", t);
  double s_mid = s_in;
  u64 *Mbuf = nullptr;
  if (mask) {  // masked sources: one PMult each (split-scale mode)

    fenc_status st = pt_device(ctx, mask);
    if (st != FENC_OK) return st;
    s_mid = s_in * mask->scale;
    Mbuf = sc.alloc<u64>(n_in * CT);
    if (!Mbuf) return fail(ctx, FENC_ERR_OOM, "compress masked sources");
    MacJob job;
    for (size_t i = 0; i < n_in; i++) {
      job.terms.push_back({{in[i]->d, mask->d_mont}});
      job.outs.push_back(Mbuf + i * CT);
    }
    st = run_mac(ctx, job, L);
    if (st != FENC_OK) return st;
  }
  u64 *Rbuf = sc.alloc<u64>(n_terms * CT);
  u64 *Ybuf = do_rescale ? sc.alloc<u64>(n_out * CT) : nullptr;
  if (!Rbuf || (do_rescale && !Ybuf)) return fail(ctx, FENC_ERR_OOM, "compress workspace");
  std::vector<fenc_ct *> res(n_out);
  for (size_t t = 0; t < n_out; t++) {
    res[t] = sc.ct(do_rescale ? L - 1 : L, do_rescale ? s_mid / (double)ctx->mod[L - 1] : s_mid);
    if (!res[t]) return fail(ctx, FENC_ERR_OOM, "compress outputs");
  }
  std::vector<const u64 *> vin(n_terms);
  std::vector<u64 *> vout(n_terms);
  std::vector<int> vs(n_terms);
  for (size_t i = 0; i < n_terms; i++) {
    vin[i] = mask ? Mbuf + term_src[i] * CT : in[term_src[i]]->d;
    vout[i] = Rbuf + i * CT, vs[i] = term_rot[i];
  }
  fenc_status st = rotate_raw(ctx, K, L, vin, vs, vout);
  if (st != FENC_OK) return st;
  std::vector<const u64 *> sum_terms;
  std::vector<int> sum_start{0};
  std::vector<u64 *> sum_out;
  for (size_t t = 0; t < n_out; t++) {
    for (size_t i = 0; i < n_terms; i++)
      if (term_out[i] == t) sum_terms.push_back(vout[i]);
    sum_start.push_back((int)sum_terms.size());
    sum_out.push_back(do_rescale ? Ybuf + t * CT : res[t]->d);
  }
  {
    DescStage ds(ctx);
    size_t o0 = ds.add(sum_terms), o1 = ds.add(sum_start), o2 = ds.add(sum_out);
    char *base = ds.commit();
    if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    CUDA_OK(ctx, k_add_many(ctx->k, (const u64 *const *)(base + o0), (const int *)(base + o1), (u64 *const *)(base + o2), (int)n_out, L, (int)sum_terms.size()));
  }
  if (do_rescale) {
    std::vector<BatchItem> items(n_out);
    for (size_t t = 0; t < n_out; t++) {
      items[t] = BatchItem{};
      items[t].sub_in = Ybuf + t * CT, items[t].out = res[t]->d;
    }
    st = rescale_batch(ctx, L, items);
    if (st != FENC_OK) return st;
  }
  sc.ok = true;
  for (size_t t = 0; t < n_out; t++) out[t] = res[t];
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ repack (R2.11c)
// out[t] = Rescale( sum_i Rot(mask_i (*) in[src_i], r_i) ): one MAC launch for all (output, amount) groups, one batch of
// rotations, one sum kernel, one rescale batch.
extern "C" fenc_status fenc_repack(fenc_ctx *ctx, const fenc_keys *K, fenc_ct *const *in, size_t n_in, fenc_pt *const *masks,
                                   const uint32_t *term_out, const uint32_t *term_src, const int32_t *term_rot, size_t n_terms,
                                   int do_rescale, fenc_ct **out, size_t n_out) {
  Scope sc(ctx);
  if (!ctx || !K || !in || !masks || !term_out || !term_src || !term_rot || !out || n_in == 0 || n_out == 0 || n_terms == 0)
    return FENC_ERR_INVALID_ARG;
  const int L = in[0]->L;
  const double s_in = in[0]->scale;
  for (size_t i = 0; i < n_in; i++)
    if (in[i]->L != L || std::fabs(in[i]->scale - s_in) > 1e-9 * s_in) return fail(ctx, FENC_ERR_MISMATCH, "sources differ in level or scale");
  if (do_rescale && L < 2) return fail(ctx, FENC_ERR_LEVEL, "no level left to rescale");
  const double s_m = masks[0] ? masks[0]->scale : 0;
  std::map<std::pair<u32, int>, std::vector<size_t>> groups;  // (output, amount) -> terms
  for (size_t i = 0; i < n_terms; i++) {
    if (term_out[i] >= n_out || term_src[i] >= n_in || !masks[i]) return fail(ctx, FENC_ERR_INVALID_ARG, "repack term %zu out of range", i);
    if (masks[i]->L != L || std::fabs(masks[i]->scale - s_m) > 1e-9 * s_m) return fail(ctx, FENC_ERR_MISMATCH, "masks differ in level or scale");
    fenc_status st = pt_device(ctx, masks[i]);
    if (st != FENC_OK) return st;
    groups[{term_out[i], ((term_rot[i] % ctx->n) + ctx->n) % ctx->n}].push_back(i);
  }
  std::vector<int> cnt(n_out, 0);
  for (auto &kv : groups) cnt[kv.first.first]++;
  for (size_t t = 0; t < n_out; t++)
    if (!cnt[t]) return fail(ctx, FENC_ERR_INVALID_ARG, "repack output %zu has no term", t);
  const size_t N = ctx->N, CT = (size_t)2 * L * N, ng = groups.size();
  const double s_acc = s_in * s_m;
  u64 *Gbuf = sc.alloc<u64>(ng * CT), *Rbuf = sc.alloc<u64>(ng * CT);
  u64 *Ybuf = do_rescale ? sc.alloc<u64>(n_out * CT) : nullptr;
  if (!Gbuf || !Rbuf || (do_rescale && !Ybuf)) return fail(ctx, FENC_ERR_OOM, "repack workspace");
  std::vector<fenc_ct *> res(n_out);
  for (size_t t = 0; t < n_out; t++) {
    res[t] = sc.ct(do_rescale ? L - 1 : L, do_rescale ? s_acc / (double)ctx->mod[L - 1] : s_acc);
    if (!res[t]) return fail(ctx, FENC_ERR_OOM, "repack outputs");
  }
  MacJob job;
  std::vector<const u64 *> rin, sum_terms;
  std::vector<u64 *> rout, sum_out;
  std::vector<int> rstep, sum_start{0};
  size_t gi = 0;
  u32 cur = groups.begin()->first.first;
  for (auto &kv : groups) {  // ordered by output, then amount
    if (kv.first.first != cur) sum_start.push_back((int)sum_terms.size()), sum_out.push_back(do_rescale ? Ybuf + cur * CT : res[cur]->d), cur = kv.first.first;
    u64 *G = Gbuf + gi * CT;
    job.terms.emplace_back();
    for (size_t i : kv.second) job.terms.back().push_back({in[term_src[i]]->d, masks[i]->d_mont});
    job.outs.push_back(G);
    if (kv.first.second) {
      rin.push_back(G), rout.push_back(Rbuf + gi * CT), rstep.push_back(kv.first.second);
      sum_terms.push_back(Rbuf + gi * CT);
    } else {
      sum_terms.push_back(G);
    }
    gi++;
  }
  sum_start.push_back((int)sum_terms.size()), sum_out.push_back(do_rescale ? Ybuf + cur * CT : res[cur]->d);
  fenc_status st = run_mac(ctx, job, L);
  if (st != FENC_OK) return st;
  st = rotate_raw(ctx, K, L, rin, rstep, rout);
  if (st != FENC_OK) return st;
  {
    DescStage ds(ctx);
    size_t o0 = ds.add(sum_terms), o1 = ds.add(sum_start), o2 = ds.add(sum_out);
    char *base = ds.commit();
    if (!base) return fail(ctx, FENC_ERR_OOM, "descriptor staging");
    CUDA_OK(ctx, k_add_many(ctx->k, (const u64 *const *)(base + o0), (const int *)(base + o1), (u64 *const *)(base + o2), (int)sum_out.size(), L, (int)sum_terms.size()));
  }
  if (do_rescale) {
    std::vector<BatchItem> items(n_out);
    for (size_t t = 0; t < n_out; t++) {
      items[t] = BatchItem{};
      items[t].sub_in = Ybuf + t * CT, items[t].out = res[t]->d;
    }
    st = rescale_batch(ctx, L, items);
    if (st != FENC_OK) return st;
  }
  sc.ok = true;
  for (size_t t = 0; t < n_out; t++) out[t] = res[t];
  return FENC_OK;
}

// ------------------------------------------------------------------------------------------------ FC by diagonals (R2.12, R2.12b)
// With g baby steps (d = i g + j):  out_{c'} = sum_i Rot( sum_j sum_c Rot(x_c, j B) (*) Rot(Wd(c',c,d), j B), i g B ):
// the baby rotations are the executor's inner rotations (once per input ciphertext), the giant ones its outer rotations.
struct FcGraph : LinGraph {
  fenc_fc_desc d;
  int n, B, P, m, ch, n_in_ct, n_out_ct, g = 1;
  std::vector<std::array<u32, 3>> wkeys;  // (c_out_ct, c_in_ct, d)
  // feature index of (input ct c, position p) or -1
  long feat(int c, int p) const {
    if (d.frag_in) {  // fragment-encoded embeddings (R2.13): coordinate p S + c of every token
      const long f = (long)p * d.frag_in + c;
      return f < (long)d.n_in ? f : -1;
    }
    if (d.in_C) {
      const int m2 = m * m, cpos = p / m2, k = p % m2, chan = c * ch + cpos, h = k / m, w = k % m;
      if (chan >= (int)d.in_C || h >= (int)d.in_H || w >= (int)d.in_W) return -1;
      return ((long)chan * d.in_H + h) * d.in_W + w;
    }
    const long f = (long)c * P + p;
    return f < (long)d.n_in ? f : -1;
  }
  long neuron(int c, int p) const {
    const long v = d.frag_out ? (long)p * d.frag_out + c : (long)c * P + p;
    return v < (long)d.n_out ? v : -1;
  }
  bool nonzero(int co, int ci, int dd) const {
    for (int p = 0; p < P; p++)
      if (feat(ci, p) >= 0 && neuron(co, ((p - dd) % P + P) % P) >= 0) return true;
    return false;
  }
  void weight_slots(const std::array<u32, 3> &wk, const double *w, std::vector<double> &vec) const {
    vec.assign(n, 0.0);
    const int co = wk[0], ci = wk[1], dd = wk[2], j = dd % g;  // the diagonal, rotated left by its baby step
    for (int p = 0; p < P; p++) {
      const long f = feat(ci, (p + j) % P), v = neuron(co, ((p + j - dd) % P + P) % P);
      if (f < 0 || v < 0) continue;
      const double val = w[(size_t)v * d.n_in + f];
      for (int b = 0; b < B; b++) vec[(size_t)p * B + b] = val;
    }
  }
};

static fenc_status fc_graph(fenc_ctx *ctx, const fenc_fc_desc *fd, std::shared_ptr<FcGraph> &out) {
  char keybuf[256];
  snprintf(keybuf, sizeof keybuf, "fc,%u,%u,%u,%u,%u,%u,%u,%u,%u,%u", fd->BS, fd->n_in, fd->n_out, fd->in_C, fd->in_H, fd->in_W, fd->in_M, fd->bsgs,
           fd->frag_in, fd->frag_out);
  auto it = ctx->graphs.find(keybuf);
  if (it != ctx->graphs.end()) {
    out = std::static_pointer_cast<FcGraph>(it->second);
    return FENC_OK;
  }
  if (fd->BS < 1 || fd->n_in < 1 || fd->n_out < 1 || fd->in_M < 1) return fail(ctx, FENC_ERR_INVALID_ARG, "bad fc shape");
  auto g = std::make_shared<FcGraph>();
  g->d = *fd, g->n = ctx->n, g->m = fd->in_M;
  const long m2 = (long)g->m * g->m;
  if (m2 > g->n || g->n % m2) return fail(ctx, FENC_ERR_LAYOUT, "frame %u^2 does not fit %d slots", fd->in_M, g->n);
  g->B = (int)std::min<long>(next_pow2(fd->BS), g->n / m2);
  g->P = g->n / g->B;
  g->ch = (int)(g->n / (g->B * m2));
  g->BG = (fd->BS + g->B - 1) / g->B;
  if (fd->frag_in) {
    if (fd->in_C || (fd->n_in + fd->frag_in - 1) / fd->frag_in > (u32)g->P)
      return fail(ctx, FENC_ERR_LAYOUT, "frag_in=%u: the %u sub-blocks of an embedding must fit the %d positions (and in_C = 0)", fd->frag_in,
                  (fd->n_in + fd->frag_in - 1) / fd->frag_in, g->P);
    g->n_in_ct = fd->frag_in;
  } else if (fd->in_C) {
    if (fd->in_H > fd->in_M || fd->in_W > fd->in_M || (size_t)fd->in_C * fd->in_H * fd->in_W != fd->n_in)
      return fail(ctx, FENC_ERR_LAYOUT, "fc input tensor does not match n_in");
    g->n_in_ct = (fd->in_C + g->ch - 1) / g->ch;
  } else {
    g->n_in_ct = (fd->n_in + g->P - 1) / g->P;
  }
  if (fd->frag_out) {
    if ((fd->n_out + fd->frag_out - 1) / fd->frag_out > (u32)g->P) return fail(ctx, FENC_ERR_LAYOUT, "frag_out=%u: sub-blocks do not fit the %d positions", fd->frag_out, g->P);
    g->n_out_ct = fd->frag_out;
  } else {
    g->n_out_ct = (fd->n_out + g->P - 1) / g->P;
  }
  g->nin_bg = g->n_in_ct;
  // baby-step count: 1 (or 0) = plain diagonals; FENC_FC_BSGS_AUTO = the power of two g | P with the fewest rotations
  // n_in_ct (g-1) + n_out_ct (P/g - 1) of a dense layer, ties to the smaller g; else a power of two dividing P
  int gs = fd->bsgs <= 1 ? 1 : (int)fd->bsgs;
  if (fd->bsgs == FENC_FC_BSGS_AUTO) {
    long best = -1;
    for (int c = 1; c <= g->P; c *= 2) {
      const long cost = (long)g->n_in_ct * (c - 1) + (long)g->n_out_ct * (g->P / c - 1);
      if (best < 0 || cost < best) best = cost, gs = c;
    }
  }
  if (gs < 1 || gs > g->P || g->P % gs || (gs & (gs - 1))) return fail(ctx, FENC_ERR_LAYOUT, "bsgs=%d must be a power of two dividing P=%d", gs, g->P);
  g->g = gs;
  std::set<int> steps;
  std::set<std::pair<int, int>> inner;
  g->outs.resize(g->n_out_ct);
  for (int co = 0; co < g->n_out_ct; co++) {
    OutCt &oc = g->outs[co];
    for (int i = 0; i < g->P / gs; i++) {
      std::vector<Term> lst;
      for (int j = 0; j < gs; j++)
        for (int ci = 0; ci < g->n_in_ct; ci++) {
          const int dd = i * gs + j;
          if (!g->nonzero(co, ci, dd)) continue;
          const int amt = (int)(((long)j * g->B) % g->n);
          lst.push_back(Term{ci, amt, (int)g->wkeys.size()});
          g->wkeys.push_back({(u32)co, (u32)ci, (u32)dd});
          if (amt) inner.insert({ci, amt}), steps.insert(amt);
        }
      if (lst.empty()) continue;
      const int rot = (int)(((long)i * gs * g->B) % g->n);
      oc.diags.push_back(i), oc.rots.push_back(rot);
      g->n_pmult += lst.size();
      oc.terms.push_back(std::move(lst));
      if (i) g->n_outer++, steps.insert(rot);
    }
  }
  g->inner.assign(inner.begin(), inner.end());
  for (size_t k = 0; k < g->inner.size(); k++) g->inner_index[g->inner[k]] = (int)k;
  g->rot_steps.assign(steps.begin(), steps.end());
  g->n_w = g->wkeys.size();
  ctx->graphs[keybuf] = g;
  out = g;
  return FENC_OK;
}

extern "C" fenc_status fenc_fc_plan(fenc_ctx *ctx, const fenc_fc_desc *fd, fenc_fc_info *out) {
  if (!ctx || !fd || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  if (g->rot_steps.size() > 512) return fail(ctx, FENC_ERR_LAYOUT, "more than 512 rotation amounts (use more baby steps or a larger B)");
  memset(out, 0, sizeof *out);
  out->B = g->B, out->P = g->P, out->BG = (u32)g->BG, out->n_in_ct = g->n_in_ct * (u32)g->BG, out->n_out_ct = g->n_out_ct * (u32)g->BG;
  out->n_rot = (u32)((g->n_outer + g->inner.size()) * g->BG), out->bsgs = (u32)g->g, out->n_pmult = (u32)(g->n_pmult * g->BG), out->n_distinct_pt = (u32)g->wkeys.size();
  out->n_rot_keys = (u32)g->rot_steps.size();
  for (size_t i = 0; i < g->rot_steps.size(); i++) out->rot_steps[i] = g->rot_steps[i];
  return FENC_OK;
}
extern "C" fenc_status fenc_fc_encode_input(fenc_ctx *ctx, const fenc_fc_desc *fd, const double *x, uint32_t c, uint32_t bgi, uint32_t n_limbs,
                                            double scale, fenc_pt **out) {
  if (!ctx || !fd || !x || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  if ((int)c >= g->n_in_ct || (int)bgi >= g->BG) return fail(ctx, FENC_ERR_LAYOUT, "fc input ciphertext index out of range");
  std::vector<double> vec(ctx->n, 0.0);
  for (int p = 0; p < g->P; p++) {
    const long f = g->feat((int)c, p);
    if (f < 0) continue;
    for (int b = 0; b < g->B; b++) {
      const size_t bb = (size_t)bgi * g->B + b;
      if (bb < fd->BS) vec[(size_t)p * g->B + b] = x[bb * fd->n_in + f];
    }
  }
  return fenc_encode_slots(ctx, vec.data(), nullptr, n_limbs, scale, out);
}
extern "C" fenc_status fenc_fc_decrypt_decode(fenc_ctx *ctx, const fenc_keys *K, const fenc_ct *ct, const fenc_fc_desc *fd, int side, uint32_t c,
                                              uint32_t bgi, double *y) {
  if (!ctx || !K || !ct || !fd || !y) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  if ((int)c >= (side ? g->n_out_ct : g->n_in_ct) || (int)bgi >= g->BG) return fail(ctx, FENC_ERR_LAYOUT, "fc ciphertext index out of range");
  std::vector<double> vec(ctx->n);
  if ((st = fenc_decrypt_slots(ctx, K, ct, vec.data(), nullptr)) != FENC_OK) return st;
  const size_t width = side ? fd->n_out : fd->n_in;
  for (int p = 0; p < g->P; p++) {
    const long v = side ? g->neuron((int)c, p) : g->feat((int)c, p);
    if (v < 0) continue;
    for (int b = 0; b < g->B; b++) {
      const size_t bb = (size_t)bgi * g->B + b;
      if (bb < fd->BS) y[bb * width + v] = vec[(size_t)p * g->B + b];
    }
  }
  return FENC_OK;
}
extern "C" fenc_status fenc_fc_wts_keys(fenc_ctx *ctx, const fenc_fc_desc *fd, uint32_t *keys3, size_t capacity, size_t *n) {
  if (!ctx || !fd || !n) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  *n = g->wkeys.size();
  if (keys3) {
    if (capacity < g->wkeys.size()) return fail(ctx, FENC_ERR_INVALID_ARG, "capacity too small");
    for (size_t i = 0; i < g->wkeys.size(); i++) memcpy(keys3 + 3 * i, g->wkeys[i].data(), 3 * sizeof(u32));
  }
  return FENC_OK;
}
extern "C" fenc_status fenc_fc_weights(fenc_ctx *ctx, const fenc_fc_desc *fd, const double *w, uint32_t n_limbs, double scale,
                                       fenc_wts **out) {
  if (!ctx || !fd || !w || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  const FcGraph *gp = g.get();
  return make_wts(ctx, gp->wkeys.size(), [gp, w](size_t i, std::vector<double> &v) { gp->weight_slots(gp->wkeys[i], w, v); }, nullptr,
                  n_limbs, scale, out);
}
extern "C" fenc_status fenc_fc_weights_from_coeffs(fenc_ctx *ctx, const fenc_fc_desc *fd, const int64_t *coeffs, size_t n,
                                                   uint32_t n_limbs, double scale, fenc_wts **out) {
  if (!ctx || !fd || !coeffs || !out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  if (n != g->wkeys.size()) return fail(ctx, FENC_ERR_MISMATCH, "expected %zu weight plaintexts, got %zu", g->wkeys.size(), n);
  return make_wts(ctx, n, nullptr, coeffs, n_limbs, scale, out);
}
extern "C" fenc_status fenc_fc(fenc_ctx *ctx, const fenc_keys *K, const fenc_fc_desc *fd, const fenc_wts *W, fenc_ct *const *in,
                               size_t n_in, int do_rescale, fenc_ct **out, size_t cap, size_t *n_out) {
  if (!ctx || !K || !fd || !W || !in || !out || !n_out) return FENC_ERR_INVALID_ARG;
  std::shared_ptr<FcGraph> g;
  fenc_status st = fc_graph(ctx, fd, g);
  if (st != FENC_OK) return st;
  return run_linear(ctx, K, *g, W, in, n_in, do_rescale, out, cap, n_out);
}
