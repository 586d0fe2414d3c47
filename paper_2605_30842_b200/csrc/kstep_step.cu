// kstep_step.cu — comem_kstep_step_async: one agent step of Algorithm 1 as a host scheduler
// over the library's own attention calls.  Host logic + one tiny kernel that sets the
// per-sequence lengths and the ragged query offsets of a step; everything else is enqueued through the C ABI
// (comem_prefill_attn_async, comem_kv_append_async, comem_decode_attn_async, comem_sm_partition), so the scheduler
// can hold no arithmetic of the method.
#include "../../include/comem_decode_attn.h"

#include <cuda_runtime.h>

#include "ptx.cuh"

namespace comem {
namespace {

// seq_lens[b] <- ctx; q_start[b] <- b * n_new (b = 0 .. batch): every sequence of the batch sits at the same step of
// the trajectory (fixed-length turns, constant concurrency)
__global__ void kstep_set_lens_kernel(int32_t *seq_lens, int32_t *q_start, int batch, int ctx, int n_new)
{
    pdl_wait_prior_grid();
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b <= batch; b += gridDim.x * blockDim.x) {
        if (b < batch) seq_lens[b] = ctx;
        q_start[b] = b * n_new;
    }
}

bool model_ok(const comem_kstep_model *m)
{
    return m && m->q_decode && m->out_decode && m->q_prefill && m->out_prefill && m->new_k && m->new_v && m->k_pages &&
           m->v_pages && m->block_table && m->seq_lens && m->q_start && m->workspace && m->batch > 0 &&
           m->num_q_heads > 0 && m->num_kv_heads > 0 && m->max_pages_per_seq > 0 && m->num_pages > 0 && m->prefill_cap > 0;
}

double step_bytes(const comem_kstep_model *m, int ctx)
{
    return (double)ctx * m->batch * m->num_kv_heads * m->head_dim * 4.0;
}

int set_lens(const comem_kstep_model *m, int ctx, int n_new, cudaStream_t s)
{
    kstep_set_lens_kernel<<<(m->batch + 256) / 256, 256, 0, s>>>(m->seq_lens, m->q_start, m->batch, ctx, n_new);
    if (cudaGetLastError() != cudaSuccess) return COMEM_ERR_CUDA;
    return COMEM_OK;
}

int prefill(const comem_kstep_model *m, int n_new, void *stream, const comem_launch_opts *o)
{
    if (n_new <= 0) return COMEM_OK;
    return comem_prefill_attn_async(m->q_prefill, m->k_pages, m->v_pages, m->block_table, m->seq_lens, m->q_start,
                                    m->num_q_heads, m->num_kv_heads, m->head_dim, m->page_size, m->softmax_scale,
                                    m->out_prefill, m->batch, m->batch * n_new, m->max_pages_per_seq, m->num_pages,
                                    nullptr, stream, o);
}

int decode_token(const comem_kstep_model *m, void *stream, const comem_launch_opts *o)
{
    int st = comem_kv_append_async(m->k_pages, m->v_pages, m->block_table, m->seq_lens, m->new_k, m->new_v,
                                   m->num_kv_heads, m->head_dim, m->page_size, m->batch, m->max_pages_per_seq, stream);
    if (st != COMEM_OK) return st;
    return comem_decode_attn_async(m->q_decode, m->k_pages, m->v_pages, m->block_table, m->seq_lens, m->num_q_heads,
                                   m->num_kv_heads, m->head_dim, m->page_size, m->softmax_scale, m->out_decode, m->batch,
                                   m->max_pages_per_seq, m->num_pages, nullptr, m->workspace, m->workspace_bytes, stream,
                                   o);
}

}  // namespace
}  // namespace comem

using namespace comem;

extern "C" int comem_kstep_step_async(const comem_kstep_event *e, int turn_tokens, int summary_tokens,
                                      int decode_tokens, int memory_decode_tokens, const comem_kstep_model *agent,
                                      const comem_kstep_model *memory, void *agent_stream, void *memory_stream,
                                      void *memory_done_event, void *agent_step_event, comem_kstep_step_stats *stats)
{
    if (!e || !model_ok(agent) || (memory && !model_ok(memory))) return COMEM_ERR_INVALID_ARG;
    if (turn_tokens <= 0 || summary_tokens < 0 || decode_tokens < 0 || memory_decode_tokens < 0) return COMEM_ERR_INVALID_ARG;
    if (e->step < 1 || e->summary_upto < 0 || e->summary_upto > e->step) return COMEM_ERR_INVALID_ARG;
    if (memory && e->launch_memory && (!memory_stream || !agent_step_event || !memory_done_event)) return COMEM_ERR_INVALID_ARG;
    // eq. 4: the summary of tau_{<= u} (none while u = 0) followed by the raw turns tau_{u+1 : t}
    const int64_t ctx64 = (e->summary_upto > 0 ? (int64_t)summary_tokens : 0) + (int64_t)(e->step - e->summary_upto) * turn_tokens;
    const int64_t cap_a = (int64_t)agent->max_pages_per_seq * agent->page_size;
    if (ctx64 + decode_tokens > cap_a) return COMEM_ERR_INVALID_ARG;
    const int ctx = (int)ctx64;
    // lines 9-13: the whole context when the cache is invalid, else only the turn that arrived
    const int n_new = e->prefill_uncached ? ctx : (turn_tokens < ctx ? turn_tokens : ctx);
    if ((int64_t)agent->batch * n_new > agent->prefill_cap) return COMEM_ERR_INVALID_ARG;
    const int64_t mem_ctx64 = (memory && e->launch_memory) ? (int64_t)e->step * turn_tokens : 0;
    if (memory && e->launch_memory) {
        if (mem_ctx64 + memory_decode_tokens > (int64_t)memory->max_pages_per_seq * memory->page_size ||
            (int64_t)memory->batch * mem_ctx64 > memory->prefill_cap)
            return COMEM_ERR_INVALID_ARG;
    }
    cudaStream_t sa = static_cast<cudaStream_t>(agent_stream);
    cudaStream_t sm = static_cast<cudaStream_t>(memory_stream);

    // Is an earlier memory job still running?  (A query, never a wait.  An event that was never recorded reads complete.)
    bool in_flight = false;
    if (memory && memory_done_event) {
        const cudaError_t q = cudaEventQuery(static_cast<cudaEvent_t>(memory_done_event));
        if (q == cudaErrorNotReady) in_flight = true;
        else if (q != cudaSuccess) { cudaGetLastError(); return COMEM_ERR_CUDA; }
    }
    const int sms = comem_grid_ctas(agent->head_dim);
    if (sms <= 0) return sms < 0 ? -sms : COMEM_ERR_CUDA;
    comem_kstep_step_stats st_ = {};
    st_.agent_ctx = ctx;
    st_.agent_prefill_tokens = n_new;
    st_.memory_ctx = (int)mem_ctx64;
    st_.memory_in_flight = in_flight ? 1 : 0;

    // the agent's share of the SMs while a memory job runs beside it: proportional to the bytes each streams per step
    // (decode grids and the persistent prefill grid alike)
    comem_launch_opts oa = {0, -1, 0};
    if (in_flight) {
        int ga = 0, gm = 0;
        // (the memory job's own context is not known here: its decode steps stream at least the agent's trajectory so far)
        const double bytes_m = step_bytes(memory, (e->step - 1) * turn_tokens > 0 ? (e->step - 1) * turn_tokens : turn_tokens);
        if (comem_sm_partition(step_bytes(agent, ctx), bytes_m, sms, 8, &ga, &gm) != COMEM_OK) return COMEM_ERR_INVALID_ARG;
        oa.grid_ctas = ga;
        oa.programmatic_launch = 0;  // a stream's next kernel must not park on the other model's SMs
        st_.agent_grid = ga;
    }

    int rc = set_lens(agent, ctx, n_new, sa);
    if (rc != COMEM_OK) return rc;
    ++st_.launches;
    if ((rc = prefill(agent, n_new, agent_stream, &oa)) != COMEM_OK) return rc;
    st_.launches += n_new > 0 ? 1 : 0;
    for (int y = 0; y < decode_tokens; ++y) {
        if ((rc = decode_token(agent, agent_stream, &oa)) != COMEM_OK) return rc;
        st_.launches += 2;
    }
    if (memory && e->launch_memory) {  // lines 19-21: P_mem <- f(tau_{<= t}), asynchronously
        if (cudaEventRecord(static_cast<cudaEvent_t>(agent_step_event), sa) != cudaSuccess ||
            cudaStreamWaitEvent(sm, static_cast<cudaEvent_t>(agent_step_event), 0) != cudaSuccess) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
        const int mem_ctx = (int)mem_ctx64;
        int ga = 0, gm = 0;
        // the agent's next steps run beside this job: their context is the one of this step plus a turn
        if (comem_sm_partition(step_bytes(agent, ctx + turn_tokens), step_bytes(memory, mem_ctx), sms, 8, &ga, &gm) != COMEM_OK)
            return COMEM_ERR_INVALID_ARG;
        comem_launch_opts om = {gm, 0, 0};
        st_.memory_grid = gm;
        if ((rc = set_lens(memory, mem_ctx, mem_ctx, sm)) != COMEM_OK) return rc;
        ++st_.launches;
        if ((rc = prefill(memory, mem_ctx, memory_stream, &om)) != COMEM_OK) return rc;
        ++st_.launches;
        for (int y = 0; y < memory_decode_tokens; ++y) {
            if ((rc = decode_token(memory, memory_stream, &om)) != COMEM_OK) return rc;
            st_.launches += 2;
        }
        if (cudaEventRecord(static_cast<cudaEvent_t>(memory_done_event), sm) != cudaSuccess) {
            cudaGetLastError();
            return COMEM_ERR_CUDA;
        }
    }
    if (stats) *stats = st_;
    return COMEM_OK;
}
