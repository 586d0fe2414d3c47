// kstep_pipeline.cu — host side of SURVEY.md §8(f).4: the k-step-off pipeline schedule (Algorithm 1,
// PAPER.md L130-176) and the latency model that sizes the summary (eq. 5-7).
// Pure host code behind the C ABI (no device work, no allocation): the plan tells a serving loop, per agent
// step, whether a finished memory job is adopted (KV cache invalidated), whether the prefill is cached or
// full, and whether a memory job is launched; bench.py --pipeline drives the two decode-attention streams
// from it and checks eq. 5 against the measured step times.
#include "../../include/comem_decode_attn.h"

#include <cmath>

extern "C" {

int comem_kstep_plan(int num_steps, int k, int mem_delay, comem_kstep_event *events)
{
    if (num_steps < 0 || k < 1 || (num_steps > 0 && !events)) return COMEM_ERR_INVALID_ARG;
    const int d = mem_delay <= 0 ? k : mem_delay;  // "available at the start of the next cycle" (L122)
    if (d > k) return COMEM_ERR_INVALID_ARG;       // Alg. 1 line 20 must never overwrite a job in flight
    int summary_upto = 0;   // line 1: s <- {}
    int job_launched = 0;   // line 1: P_mem <- None (0); else the step after which it was launched
    bool kv_valid = false;
    for (int t = 1; t <= num_steps; ++t) {  // line 2
        comem_kstep_event &e = events[t - 1];
        e.step = t;
        e.adopt_summary = 0;
        if (job_launched != 0 && t >= job_launched + d) {  // lines 4-7
            summary_upto = job_launched;  // the job compressed tau_{<= job_launched}
            kv_valid = false;
            job_launched = 0;
            e.adopt_summary = 1;
        }
        e.summary_upto = summary_upto;
        e.prefill_uncached = kv_valid ? 0 : 1;  // lines 9-13
        kv_valid = true;
        e.launch_memory = (t % k == 0) ? 1 : 0;  // lines 19-21
        if (e.launch_memory) job_launched = t;
    }
    return COMEM_OK;
}

int comem_kstep_context_lengths(const comem_kstep_event *events, int num_steps, int turn_tokens,
                                int summary_tokens, int32_t *comem_ctx, int32_t *full_ctx, int32_t *memory_input)
{
    if (num_steps < 0 || turn_tokens < 0 || summary_tokens < 0) return COMEM_ERR_INVALID_ARG;
    if (num_steps > 0 && (!events || !comem_ctx || !full_ctx || !memory_input)) return COMEM_ERR_INVALID_ARG;
    for (int i = 0; i < num_steps; ++i) {
        const comem_kstep_event &e = events[i];
        const int64_t c = (e.summary_upto > 0 ? (int64_t)summary_tokens : 0) +
                          (int64_t)(e.step - e.summary_upto) * turn_tokens;
        const int64_t f = (int64_t)e.step * turn_tokens;
        if (c > 0x7fffffff || f > 0x7fffffff) return COMEM_ERR_INVALID_ARG;
        comem_ctx[i] = (int32_t)c;
        full_ctx[i] = (int32_t)f;
        memory_input[i] = e.launch_memory ? (int32_t)f : 0;
    }
    return COMEM_OK;
}

double comem_decode_saving_seconds(double l_full, double l_sum, double s_gb_per_token, double w_gb_per_s)
{
    return (l_full - l_sum) * s_gb_per_token / w_gb_per_s;  // eq. 5
}

int comem_net_speedup(double y_tokens, double l_full, double l_sum, double s_gb_per_token, double w_gb_per_s,
                      double p_tokens_per_s)
{
    return y_tokens * comem_decode_saving_seconds(l_full, l_sum, s_gb_per_token, w_gb_per_s) >
                   l_sum / p_tokens_per_s ? 1 : 0;  // eq. 6
}

double comem_max_compression_ratio(double w_gb_per_s, double y_tokens, double s_gb_per_token, double p_tokens_per_s)
{
    return 1.0 / (1.0 + w_gb_per_s / (y_tokens * s_gb_per_token * p_tokens_per_s));  // eq. 7
}

}  // extern "C"
