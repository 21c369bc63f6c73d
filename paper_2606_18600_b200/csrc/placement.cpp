// placement.cpp — libshuntplace.so: the paper's serving performance estimator (Eq. 1-5, Table 2), batch-size rule
// (Eq. 6), objective (Eq. 7) and partitioned model placement optimizer (Algorithm 1: DP over (layers placed, stages
// used) with beam k).  Host-only C++; see include/shuntplace.h for the ABI and the readings.
#include "../../include/shuntplace.h"

#include <math.h>
#include <string.h>

#include <algorithm>
#include <cmath>
#include <vector>

namespace {

inline double op_latency(double flops, double mem_elems, const sp_model *m, const sp_instance *g) {
  const double lc = flops / g->flops;                        // L_compute
  const double lm = mem_elems * m->elem_bytes / g->mem_bw;   // L_memory  (reading A5)
  return lc > lm ? lc : lm;                                  // Eq. 1
}

bool model_ok(const sp_model *m) {
  return m && m->hidden > 0 && m->hq > 0 && m->hkv > 0 && m->ffn > 0 && m->vocab >= 0 && m->n_layers > 0 &&
         m->elem_bytes > 0;
}
bool inst_ok(const sp_instance *g) {
  return g && g->flops > 0 && g->mem_bw > 0 && g->mem_bytes > 0 && g->n_gpus >= 1 && g->cost > 0 &&
         (g->n_gpus == 1 || g->beta_intra > 0);
}
bool opts_ok(const sp_opts *o) {
  return o && o->s_in > 0 && o->s_out > 0 && o->beta_inter > 0 && o->beam >= 1 && o->max_stages >= 1 &&
         o->max_stages <= SP_MAX_STAGES && o->gamma >= 0;
}

double params_per_layer(const sp_model *m) {
  const double H = m->hidden, Hq = m->hq, Hkv = m->hkv, F = m->ffn;
  return H * Hq + 2 * H * Hkv + Hq * H + 3 * H * F;
}

}  // namespace

extern "C" {

double sp_stage_latency(const sp_model *m, const sp_instance *g, const sp_opts *o, int layers, int B, int phase,
                        int is_last, int has_next) {
  if (!model_ok(m) || !inst_ok(g) || !opts_ok(o) || layers < 1 || B < 1 || (phase != 0 && phase != 1)) return -1.0;
  const double H = m->hidden, Hq = m->hq, Hkv = m->hkv, F = m->ffn, V = m->vocab, D = g->n_gpus;
  const double Si = o->s_in, So = o->s_out, b = B;
  double per_layer, logits, tokens_per_msg, n_msgs;
  if (phase == 0) {  // Table 2, "Prefill" rows
    const double qkv = op_latency(b * (2 * Si * H * Hq + 4 * Si * H * Hkv) / D, b * Si * H + (H * Hq + 2 * H * Hkv) / D, m, g);
    const double att = op_latency(4 * b * Si * Si * Hq / D, (b * Si * Hq + 2 * b * Si * Hkv) / D, m, g);
    const double out = op_latency(2 * b * Si * Hq * H / D, (b * Si * Hq + Hq * H) / D, m, g);
    const double ug = op_latency(4 * b * Si * H * F / D, b * Si * H + 2 * H * F / D, m, g);
    const double dn = op_latency(2 * b * Si * H * F / D, (b * Si * F + H * F) / D, m, g);
    per_layer = qkv + att + out + ug + dn;
    logits = op_latency(2 * b * Si * H * V / D, b * Si * H + H * V / D, m, g);
    tokens_per_msg = Si;
    n_msgs = 1;
  } else {  // Table 2, "Decode" rows: all S_out iterations; the attention rows are sums over t = 1..S_out
    const double sum_ctx = So * Si + So * (So + 1) / 2;  // sum_t (S_in + t)
    const double qkv = op_latency(b * So * (2 * H * Hq + 4 * H * Hkv) / D, So * (b * H + (H * Hq + 2 * H * Hkv) / D), m, g);
    const double att = op_latency(4 * b * sum_ctx * Hq / D, (So * b * Hq + 2 * b * sum_ctx * Hkv) / D, m, g);  // A3
    const double out = op_latency(2 * b * So * Hq * H / D, So * (b * Hq + Hq * H) / D, m, g);
    const double ug = op_latency(4 * b * So * H * F / D, So * (b * H + 2 * H * F / D), m, g);
    const double dn = op_latency(2 * b * So * H * F / D, So * (b * F + H * F) / D, m, g);
    per_layer = qkv + att + out + ug + dn;
    logits = op_latency(2 * b * So * H * V / D, So * (b * H + H * V / D), m, g);
    tokens_per_msg = 1;
    n_msgs = So;
  }
  double lat = layers * per_layer;
  if (is_last && m->vocab > 0) lat += logits;
  const double msg_bytes = b * tokens_per_msg * H * m->elem_bytes;  // B S H E
  if (g->n_gpus > 1)  // Eq. 3: two ring all-reduces per layer
    lat += n_msgs * 4.0 * (g->alpha_intra + msg_bytes / (D * g->beta_intra)) * (D - 1) * layers;
  if (has_next) lat += n_msgs * (o->alpha_inter + msg_bytes / o->beta_inter);  // Eq. 2
  return lat;
}

static int max_batch(const sp_model *m, const sp_instance *types, const sp_opts *o, int n_stages,
                     const int32_t *inst, const int32_t *layers, bool complete) {
  if (!model_ok(m) || !types || !opts_ok(o) || n_stages < 1 || !inst || !layers) return -1;
  const double E = m->elem_bytes;
  const double kv_per_req_layer = (o->s_in + o->s_out) * 2.0 * m->hkv * E;  // reading A18
  double best = 1e300;
  for (int i = 0; i < n_stages; ++i) {
    const sp_instance *g = &types[inst[i]];
    double w = layers[i] * params_per_layer(m) * E;
    if (i == 0) w += (double)m->vocab * m->hidden * E;             // embedding
    if (i == n_stages - 1 && complete) w += (double)m->vocab * m->hidden * E;  // lm_head
    const double free_b = g->n_gpus * g->mem_bytes - w - o->act_bytes;
    if (free_b <= 0) return 0;
    const double bi = floor(free_b / (layers[i] * kv_per_req_layer));
    if (bi < best) best = bi;
  }
  if (best < 1) return 0;
  if (o->max_batch > 0 && best > o->max_batch) best = o->max_batch;
  if (best > 1e9) best = 1e9;
  return (int)best;
}

int sp_max_batch(const sp_model *m, const sp_instance *types, const sp_opts *o, int n_stages, const int32_t *inst,
                 const int32_t *layers) {
  return max_batch(m, types, o, n_stages, inst, layers, true);
}

int sp_evaluate(const sp_model *m, const sp_instance *types, int n_types, const sp_opts *o, sp_placement *p) {
  if (!model_ok(m) || !types || n_types < 1 || !opts_ok(o) || !p || p->n_stages < 1 || p->n_stages > SP_MAX_STAGES)
    return -1;
  int placed = 0;
  for (int i = 0; i < p->n_stages; ++i) {
    if (p->inst[i] < 0 || p->inst[i] >= n_types || p->layers[i] < 1 || !inst_ok(&types[p->inst[i]])) return -1;
    placed += p->layers[i];
  }
  if (placed > m->n_layers) return -1;
  const bool complete = placed == m->n_layers;
  p->cost = 0;
  for (int i = 0; i < p->n_stages; ++i) p->cost += types[p->inst[i]].cost;
  p->batch = max_batch(m, types, o, p->n_stages, p->inst, p->layers, complete);
  p->prefill_s = p->decode_s = p->rps = p->score = 0;
  if (p->batch <= 0) {
    p->batch = 0;
    return 0;
  }
  for (int i = 0; i < p->n_stages; ++i) {
    const int last = (i == p->n_stages - 1);
    const int is_last = last && complete;          // only the model's last stage computes logits
    const int has_next = !(last && complete);      // a partial placement's last stage still feeds a later one
    const sp_instance *g = &types[p->inst[i]];
    p->prefill_s = std::max(p->prefill_s, sp_stage_latency(m, g, o, p->layers[i], p->batch, 0, is_last, has_next));
    p->decode_s = std::max(p->decode_s, sp_stage_latency(m, g, o, p->layers[i], p->batch, 1, is_last, has_next));
  }
  const double lat = p->prefill_s + p->decode_s;  // Eq. 5
  p->rps = p->batch / lat;                        // Eq. 4
  double pen = 1.0;
  if (o->gamma > 0 && o->slo > 0) pen = 1.0 - o->gamma * std::max(0.0, lat / o->slo - 1.0);
  p->score = p->rps / p->cost * pen;              // Eq. 7
  return 0;
}

int sp_optimize(const sp_model *m, const sp_instance *types, int n_types, const int32_t *avail, const sp_opts *o,
                sp_placement *out) {
  if (!model_ok(m) || !types || n_types < 1 || !opts_ok(o) || !out) return -1;
  for (int t = 0; t < n_types; ++t)
    if (!inst_ok(&types[t])) return -1;
  const int NL = m->n_layers;
  const int S = std::min<int>(o->max_stages, NL);
  const size_t k = (size_t)o->beam;
  // DP[l][s]: the top-k placements of the first l layers on s stages (Algorithm 1, line 1)
  std::vector<std::vector<std::vector<sp_placement>>> dp(NL + 1, std::vector<std::vector<sp_placement>>(S + 1));
  sp_placement empty;
  memset(&empty, 0, sizeof(empty));
  dp[0][0].push_back(empty);
  auto better = [](const sp_placement &a, const sp_placement &b) { return a.score > b.score; };
  for (int l = 1; l <= NL; ++l) {                    // line 2
    for (int lp = 0; lp < l; ++lp) {                 // line 2: l' = 0 .. l-1
      const int l_new = l - lp;                      // line 3
      for (int s = 0; s <= std::min(lp, S - 1); ++s) {  // line 4
        for (const sp_placement &c : dp[lp][s]) {    // line 6: the top-k combinations of DP[l'][s]
          for (int t = 0; t < n_types; ++t) {        // line 7
            if (avail) {
              int used = 0;
              for (int i = 0; i < c.n_stages; ++i) used += (c.inst[i] == t);
              if (used >= avail[t]) continue;
            }
            sp_placement cn = c;                     // line 8: c.add_stage(i, l_new)
            cn.inst[cn.n_stages] = t;
            cn.layers[cn.n_stages] = l_new;
            cn.n_stages += 1;
            if (sp_evaluate(m, types, n_types, o, &cn) != 0 || cn.batch <= 0) continue;  // lines 9-10
            std::vector<sp_placement> &cell = dp[l][s + 1];                              // line 11
            cell.push_back(cn);
            std::stable_sort(cell.begin(), cell.end(), better);
            if (cell.size() > k) cell.resize(k);
          }
        }
      }
    }
  }
  bool found = false;
  for (int s = 1; s <= S; ++s)
    for (const sp_placement &c : dp[NL][s])
      if (!found || c.score > out->score) {
        *out = c;
        found = true;
      }
  return found ? 0 : 1;
}

// ---- request dispatch: smooth weighted round-robin over pipelines (reading in shuntplace.h) ----------
struct sp_wrr {
  std::vector<double> weight, credit;
};

int sp_wrr_create(sp_wrr **out, int n, const double *weights) {
  if (!out || !weights || n <= 0) return -1;
  for (int i = 0; i < n; ++i)
    if (!(weights[i] >= 0.0) || !std::isfinite(weights[i])) return -1;
  sp_wrr *w = new sp_wrr();
  w->weight.assign(weights, weights + n);
  w->credit.assign(n, 0.0);
  *out = w;
  return 0;
}

int sp_wrr_destroy(sp_wrr *w) {
  if (!w) return -1;
  delete w;
  return 0;
}

int sp_wrr_next(sp_wrr *w) {
  if (!w) return -1;
  double total = 0.0;
  int best = -1;
  for (size_t i = 0; i < w->weight.size(); ++i) {
    if (w->weight[i] <= 0.0) continue;
    w->credit[i] += w->weight[i];
    total += w->weight[i];
    if (best < 0 || w->credit[i] > w->credit[best]) best = (int)i;
  }
  if (best < 0) return -1;
  w->credit[best] -= total;
  return best;
}

int sp_wrr_set_weight(sp_wrr *w, int i, double weight) {
  if (!w || i < 0 || i >= (int)w->weight.size() || !(weight >= 0.0) || !std::isfinite(weight)) return -1;
  w->weight[i] = weight;
  w->credit[i] = 0.0;
  return 0;
}

}  // extern "C"
