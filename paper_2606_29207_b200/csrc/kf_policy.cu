// kf_policy.cu -- Algorithm 1 of the paper ("A-node scaling policy") as a host-side controller.
// Pure host arithmetic in double precision: no kernel, no device state.  The caller feeds it the occupancy that
// kf_partition_state() reports and acts on its decisions with kf_set_active_partitions() (the route install).
#include <math.h>

#include "../../include/kflume.h"

namespace {

bool valid(const kf_policy_config *c) {
    return c && c->beta_mem > 0 && c->beta_mem <= 1 && c->beta_slo > 0 && c->beta_slo <= 1 && c->gamma > 0 &&
           c->gamma <= 1 && c->t_a_max_s > 0 && c->bw_hbm > 0 && c->c_kv_cap > 0 && c->t_step_s > 0 &&
           c->t_prewarm_s >= 0 && c->n_kv_heads > 0 && c->head_dim > 0 && c->n_layers > 0;
}

}  // namespace

extern "C" {

// per-token KV bytes 2 * H_kv * d_h * L * 2B ("2B" = two bytes per fp16 element)
double kf_policy_bytes_per_token(const kf_policy_config *c) {
    if (!valid(c)) return 0.0;
    return 2.0 * c->n_kv_heads * c->head_dim * c->n_layers * 2.0;
}

// Eq. (1) / Alg. 1 line 1: C_thresh = min(beta_mem * C_kv_cap, beta_slo * T_A^max * BW_HBM)
double kf_policy_threshold(const kf_policy_config *c) {
    if (!valid(c)) return 0.0;
    const double c_mem = c->beta_mem * c->c_kv_cap;
    const double c_slo = c->beta_slo * c->t_a_max_s * c->bw_hbm;
    return c_mem < c_slo ? c_mem : c_slo;
}

// Alg. 1 lines 2-3: C_total = sum_i s_i * bytes_per_token ; N_A = ceil(C_total / C_thresh)
int64_t kf_policy_initial_nodes(const kf_policy_config *c, const int64_t *s, int32_t n_requests) {
    if (!valid(c) || !s || n_requests < 0) return -1;
    double total = 0.0;
    for (int32_t i = 0; i < n_requests; ++i) {
        if (s[i] < 0) return -1;
        total += (double)s[i] * kf_policy_bytes_per_token(c);
    }
    return (int64_t)ceil(total / kf_policy_threshold(c));
}

// Alg. 1 lines 6-19, one pass of the per-step monitor over the P nodes
int kf_policy_step(const kf_policy_config *c, int32_t n_partitions, const int64_t *tokens, const int32_t *tails,
                   const uint8_t *prewarm_pending, const uint8_t *prewarm_ready, kf_policy_decision *out) {
    if (!valid(c) || n_partitions < 1 || !tokens || !tails || !prewarm_pending || !prewarm_ready || !out) return KF_EINVAL;
    const double per_tok = kf_policy_bytes_per_token(c);
    const double thresh = kf_policy_threshold(c);
    for (int32_t i = 0; i < n_partitions; ++i) {
        kf_policy_decision d;
        d.tau_fill = INFINITY;
        d.want_prewarm = 0;
        d.want_publish = 0;
        const double n_i = (double)tails[i];            // l.7  active requests whose tail is on node i
        const double g_i = n_i * per_tok;               // l.8  growth in bytes per step
        const double b_i = (double)tokens[i] * per_tok; // l.9  KVBytes(A_i)
        if (tails[i] > 0) {                             //      "foreach tail-holding A-node"
            if (g_i > 0) {                              // l.10
                d.tau_fill = (thresh - b_i) / g_i;      // l.11 Eq. (2)
                if (d.tau_fill * c->t_step_s < c->t_prewarm_s && !prewarm_pending[i] && !prewarm_ready[i])
                    d.want_prewarm = 1;                 // l.12-13
            }
            if (b_i >= c->gamma * thresh && prewarm_ready[i]) d.want_publish = 1;  // l.16-17
        }
        out[i] = d;
    }
    return KF_OK;
}

}  // extern "C"
