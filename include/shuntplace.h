/* shuntplace.h — C ABI of libshuntplace.so: ShuntServe's serving performance estimator and partitioned model placement
 * optimizer (arxiv/paper_2606_18600 section 4).  Host-only C++, no device code, no allocation
 * the caller does not own.  Everything here is the paper's own method restated:
 *   - Eq. 1 + Table 2: latency of an operation = max(FLOPs / FLOPS, MemScanCost * E / BW);
 *   - Eq. 2, 3: pipeline point-to-point and ring all-reduce communication (alpha-beta model);
 *   - Eq. 4, 5: RPS = B / (max_i L_prefill^i(B) + max_i L_decode^i(B));
 *   - Eq. 6: the largest batch the stages' memory admits;
 *   - Eq. 7: objective = throughput / cost * (1 - gamma * max(0, latency / SLO - 1));
 *   - Algorithm 1: DP over (layers placed, stages used) with beam size k.
 * Readings of garbled / silent points are those of DESIGN.md (A2: H_kv = n_kv * d; A4: H^2 -> H * Hq when
 * n_q * d != H; A5; A18: Eq. 6 lacks the KV bytes per token, restored here).  Units: seconds, bytes, FLOP/s, B/s. */
#ifndef SHUNTPLACE_H
#define SHUNTPLACE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define SP_MAX_STAGES 64

typedef struct {       /* transformer dimensions (Table 3) */
  int32_t hidden;      /* H */
  int32_t hq;          /* n_q * d (= H for Llama-3.1-70B; 8192 vs H = 5120 for Qwen3-32B: reading A4) */
  int32_t hkv;         /* H_kv = n_kv * d (reading A2) */
  int32_t ffn;         /* H_ffn */
  int32_t vocab;       /* V; 0 = no logits row */
  int32_t n_layers;    /* N_L */
  int32_t elem_bytes;  /* E (2 for BF16) */
} sp_model;

typedef struct {       /* one instance type of the cluster (Table 1 rows, calibrated values: PAPER.md:199) */
  double flops;        /* effective FLOP/s of ONE GPU */
  double mem_bw;       /* effective memory bandwidth of ONE GPU, B/s */
  double mem_bytes;    /* memory capacity of ONE GPU */
  int32_t n_gpus;      /* GPUs of the instance = D_TP of a stage placed on it (TP is intra-node only) */
  double alpha_intra;  /* intra-node network latency, s   (Eq. 3) */
  double beta_intra;   /* intra-node network bandwidth, B/s */
  double cost;         /* price per unit time (any unit; Eq. 7 uses ratios) */
} sp_instance;

typedef struct {
  double s_in, s_out;  /* S_in, S_out: mean input / output lengths of the workload */
  double alpha_inter;  /* inter-stage network latency, s (Eq. 2) */
  double beta_inter;   /* inter-stage bandwidth, B/s */
  double act_bytes;    /* M_activation of Eq. 6 */
  double gamma, slo;   /* Eq. 7; gamma = 0 (the paper's default) ignores the SLO */
  int32_t beam;        /* k of Algorithm 1 (>= 1) */
  int32_t max_stages;  /* upper bound on D_PP (<= SP_MAX_STAGES, <= n_layers) */
  int32_t max_batch;   /* cap on B (0 = none) */
} sp_opts;

typedef struct {       /* a (possibly partial) placement and its evaluation */
  int32_t n_stages;
  int32_t inst[SP_MAX_STAGES];    /* instance type of each stage */
  int32_t layers[SP_MAX_STAGES];  /* layers of each stage */
  int32_t batch;                  /* B of Eq. 6 (0: the placement does not fit) */
  double prefill_s, decode_s;     /* max over stages of the prefill / decode latency at that B (Eq. 5) */
  double rps;                     /* Eq. 4 */
  double cost;                    /* sum of the instances' cost */
  double score;                   /* Eq. 7 */
} sp_placement;

/* Latency in seconds of ONE stage of `layers` layers on instance `inst` for a batch of B requests, following Table 2
 * row by row: phase 0 = prefill of S_in tokens per request, phase 1 = all S_out decode iterations.  `is_last` adds the
 * logits row; `has_next` adds the point-to-point transfer of Eq. 2; D_TP > 1 adds Eq. 3.  Returns < 0 on bad input. */
double sp_stage_latency(const sp_model *m, const sp_instance *inst, const sp_opts *o, int layers, int B, int phase,
                        int is_last, int has_next);

/* Largest batch the placement's memory admits (Eq. 6 with reading A18): min over stages of
 * floor((n_gpus * mem - weights_of_the_stage - act) / (layers * (S_in + S_out) * 2 * H_kv * E)); 0 if a stage's
 * weights do not fit.  The first stage also holds the embedding and the last the lm_head (V * H * E each). */
int sp_max_batch(const sp_model *m, const sp_instance *types, const sp_opts *o, int n_stages, const int32_t *inst,
                 const int32_t *layers);

/* Fill batch, latencies, rps, cost and score of `p` (n_stages, inst[], layers[] given; the layers need not sum to
 * n_layers: Algorithm 1 scores partial placements the same way).  Returns 0, or -1 on bad input. */
int sp_evaluate(const sp_model *m, const sp_instance *types, int n_types, const sp_opts *o, sp_placement *p);

/* Algorithm 1.  `avail[t]` = instances of type t that may be used (NULL: unlimited).  On success returns 0 and the
 * best complete placement (all n_layers placed) in *out; returns 1 if no placement fits; -1 on bad input. */
int sp_optimize(const sp_model *m, const sp_instance *types, int n_types, const int32_t *avail, const sp_opts *o,
                sp_placement *out);

/* Request dispatch over the pipelines a placement produced (the global server routes requests to
 * pipelines; "load balancing via a weighted round-robin policy based on the throughput of each
 * pipeline").  The paper names the policy, not the variant; reading: SMOOTH weighted round-robin — every
 * pick adds each pipeline's weight to its running credit, takes the pipeline with the largest credit (lowest index on
 * ties) and charges it the sum of the weights — which spreads a heavy pipeline's turns instead of bursting them and is
 * deterministic.  Weights are the pipelines' throughputs (rps of sp_placement, or measured); weight 0 = no traffic (a
 * pipeline being drained for replacement, section 5.2: the server "stops routing requests to the old pipeline ... and
 * shunts the request path to the new pipeline").  Changing a weight keeps the credits of the others and clears that
 * pipeline's own.  Returns: create 0 / -1 (n <= 0, null, negative or non-finite weight); next = pipeline index, or -1
 * if every weight is 0; set_weight 0 / -1. */
typedef struct sp_wrr sp_wrr;
int sp_wrr_create(sp_wrr **out, int n, const double *weights);
int sp_wrr_destroy(sp_wrr *w);
int sp_wrr_next(sp_wrr *w);
int sp_wrr_set_weight(sp_wrr *w, int i, double weight);

#ifdef __cplusplus
}
#endif
#endif
