// dfssm_sched_*: a continuous-batching greedy generator on top of the public entry points (second half: "a
// multi-replica batch scheduler ... turns the step into a usable generator; no new math from the paper"; the generation loop of
// PAPER.md P:126).  Host logic only: it calls dfssm_reset_state / dfssm_prefill / dfssm_step / dfssm_next_tokens of ONE context
// (one replica = one GPU; N replicas are N schedulers fed by the caller's dispatcher) and owns no kernel.
//
// Requests (prompt, number of new tokens) wait in a FIFO.  Each iteration admits waiting requests into the free sequence slots of
// the context (lowest slot first: reset the slot's state, prefill its prompt - the prefill leaves the request's first generated
// token in the context's token buffer), then runs ONE dfssm_step for slots 0 .. highest active slot with the context's own
// token buffer as input (greedy tokens never leave the device), reads the new tokens back, appends them to their requests and
// retires the finished ones.  Sequences are independent in every kernel of the step (batch invariance), so a
// request's tokens are exactly those of running it alone, whatever the schedule: that is the test (tests/test_gpu_sched.py).
// Idle slots below the highest active one are stepped too (their state is reset at the next admission).
//
// Sampling (dfssm_sched_set_sampling): one temperature / top-k for the scheduler; token k of request id draws the uniform
// dfssm_sched_uniform(seed + id, k), a counter-based generator (splitmix64 finaliser of seed' + (k + 1) * 0x9E3779B97F4A7C15, top
// 24 bits / 2^24) - so a request's random numbers do not depend on the schedule either.  dfssm_sample (R23) is a
// pure function of (logits, u): slots that already drew their token are re-sampled with the same u and get the same token.
#include "../../include/dfssm.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <deque>
#include <new>
#include <vector>

struct dfssm_sched {
    dfssm_ctx* ctx;
    int max_batch;
    cudaStream_t stream;
    int32_t* dev_prompt;          // caller's device scratch: one prompt at a time
    size_t max_prompt;
    int32_t* host_next;           // pinned, [max_batch]
    struct Request {
        std::vector<int32_t> prompt;
        int max_new;
        std::vector<int32_t> out;
        int slot;                 // -1: waiting or done
        bool done;
    };
    std::vector<Request> req;
    std::deque<int> waiting;
    std::vector<int> slot_req;    // request id per slot, -1 = free
    long long steps, slot_steps_used, slot_steps_run;
    float temperature;            // <= 0: greedy
    int top_k;
    unsigned long long seed;
    float* dev_u;                 // [max_batch] uniforms, the tail of the caller's scratch
    float* host_u;                // pinned, [max_batch]: the uniform each slot drew last
    char err[256];
};

namespace {

int sfail(dfssm_sched* s, int code, const char* msg)
{
    if (s) snprintf(s->err, sizeof s->err, "%s", msg);
    return code;
}

int from_ctx(dfssm_sched* s, int rc)
{
    if (rc != DFSSM_OK) snprintf(s->err, sizeof s->err, "%s", dfssm_last_error(s->ctx));
    return rc;
}

// sample the next token of slots 0 .. hi (no-op when greedy): `draw` lists the slots that draw a NEW uniform (token index = the
// number of tokens their request has so far); every other slot keeps its last one
int sample_slots(dfssm_sched* s, int hi, const std::vector<int>& draw)
{
    if (!(s->temperature > 0.0f) || s->top_k <= 1 || hi < 0) return DFSSM_OK;
    for (int slot : draw) {
        const int id = s->slot_req[slot];
        s->host_u[slot] = dfssm_sched_uniform(s->seed + (unsigned long long)id, (int)s->req[id].out.size());
    }
    if (cudaMemcpyAsync(s->dev_u, s->host_u, sizeof(float) * (size_t)(hi + 1), cudaMemcpyHostToDevice, s->stream) != cudaSuccess)
        return sfail(s, DFSSM_E_CUDA, "uniform copy failed");
    return from_ctx(s, dfssm_sample(s->ctx, hi + 1, s->temperature, s->top_k, s->dev_u));
}

}  // namespace

extern "C" {

float dfssm_sched_uniform(unsigned long long seed, int k)
{
    unsigned long long x = seed + (unsigned long long)(k + 1) * 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    x ^= x >> 31;
    return (float)(x >> 40) * (1.0f / 16777216.0f);       // 24 bits: exact in binary32, in [0, 1)
}

int dfssm_sched_create(dfssm_ctx* ctx, int max_batch, void* dev_scratch, size_t scratch_bytes, void* cuda_stream, dfssm_sched** out)
{
    if (!ctx || !out || max_batch < 1 || !dev_scratch || scratch_bytes < 4 * ((size_t)max_batch + 1)) return DFSSM_E_ARG;
    dfssm_sched* s = new (std::nothrow) dfssm_sched();
    if (!s) return DFSSM_E_ARG;
    s->ctx = ctx;
    s->max_batch = max_batch;
    s->stream = (cudaStream_t)cuda_stream;
    s->dev_prompt = (int32_t*)dev_scratch;
    s->max_prompt = scratch_bytes / 4 - (size_t)max_batch;          // the last max_batch words hold the uniforms of dfssm_sample
    s->dev_u = (float*)dev_scratch + s->max_prompt;
    s->host_next = nullptr;
    s->host_u = nullptr;
    s->temperature = 0.0f;
    s->top_k = 1;
    s->seed = 0;
    s->slot_req.assign((size_t)max_batch, -1);
    s->steps = s->slot_steps_used = s->slot_steps_run = 0;
    s->err[0] = 0;
    *out = s;
    if (cudaMallocHost((void**)&s->host_next, sizeof(int32_t) * (size_t)max_batch) != cudaSuccess ||
        cudaMallocHost((void**)&s->host_u, sizeof(float) * (size_t)max_batch) != cudaSuccess)
        return sfail(s, DFSSM_E_CUDA, "cudaMallocHost failed");
    memset(s->host_u, 0, sizeof(float) * (size_t)max_batch);
    return DFSSM_OK;
}

int dfssm_sched_set_sampling(dfssm_sched* s, float temperature, int top_k, unsigned long long seed)
{
    if (!s) return DFSSM_E_ARG;
    if (top_k < 1 || top_k > 64) return sfail(s, DFSSM_E_ARG, "top_k outside [1, 64]");
    for (int id : s->slot_req)
        if (id >= 0) return sfail(s, DFSSM_E_STATE, "sampling parameters cannot change while requests are generating");
    s->temperature = temperature;
    s->top_k = top_k;
    s->seed = seed;
    return DFSSM_OK;
}

int dfssm_sched_submit(dfssm_sched* s, const int32_t* prompt_host, int n_prompt, int max_new_tokens, int* request_id)
{
    if (!s || !prompt_host || !request_id) return DFSSM_E_ARG;
    if (n_prompt < 1 || (size_t)n_prompt > s->max_prompt) return sfail(s, DFSSM_E_SIZE, "prompt length outside [1, scratch_bytes / 4]");
    if (max_new_tokens < 1) return sfail(s, DFSSM_E_ARG, "max_new_tokens < 1");
    dfssm_sched::Request r;
    r.prompt.assign(prompt_host, prompt_host + n_prompt);
    r.max_new = max_new_tokens;
    r.slot = -1;
    r.done = false;
    s->req.push_back(std::move(r));
    *request_id = (int)s->req.size() - 1;
    s->waiting.push_back(*request_id);
    return DFSSM_OK;
}

// one iteration: admissions, one step, retirements.  *n_active = requests still generating afterwards (+ waiting ones)
int dfssm_sched_iterate(dfssm_sched* s, int* n_active)
{
    if (!s) return DFSSM_E_ARG;
    const int32_t* next_dev = nullptr;
    int rc = from_ctx(s, dfssm_next_tokens(s->ctx, &next_dev));
    if (rc != DFSSM_OK) return rc;
    // ---- admit: lowest free slot first ----
    std::vector<int> fresh;
    for (int slot = 0; slot < s->max_batch && !s->waiting.empty(); ++slot) {
        if (s->slot_req[slot] >= 0) continue;
        const int id = s->waiting.front();
        s->waiting.pop_front();
        dfssm_sched::Request& r = s->req[id];
        if ((rc = from_ctx(s, dfssm_reset_state(s->ctx, slot))) != DFSSM_OK) return rc;
        if (cudaMemcpyAsync(s->dev_prompt, r.prompt.data(), sizeof(int32_t) * r.prompt.size(), cudaMemcpyHostToDevice, s->stream) != cudaSuccess)
            return sfail(s, DFSSM_E_CUDA, "prompt copy failed");
        if ((rc = from_ctx(s, dfssm_prefill(s->ctx, s->dev_prompt, (int)r.prompt.size(), slot))) != DFSSM_OK) return rc;
        // the scratch holds one prompt: the copy of the next one must not overtake this prefill (same stream: it cannot), but the
        // host vector must stay alive until the copy ran -- it does, requests are never erased
        r.slot = slot;
        s->slot_req[slot] = id;
        fresh.push_back(slot);
    }
    int hi = -1;
    for (int slot = 0; slot < s->max_batch; ++slot)
        if (s->slot_req[slot] >= 0) hi = slot;
    if (hi < 0) { if (n_active) *n_active = 0; return DFSSM_OK; }
    // ---- the first generated token of the fresh requests is already in the token buffer (prefill); read it ----
    if (!fresh.empty()) {
        if ((rc = sample_slots(s, hi, fresh)) != DFSSM_OK) return rc;
        if (cudaMemcpyAsync(s->host_next, next_dev, sizeof(int32_t) * (size_t)(hi + 1), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
            cudaStreamSynchronize(s->stream) != cudaSuccess)
            return sfail(s, DFSSM_E_CUDA, "token read-back failed");
        for (int slot : fresh) {
            dfssm_sched::Request& r = s->req[s->slot_req[slot]];
            r.out.push_back(s->host_next[slot]);
            if ((int)r.out.size() >= r.max_new) { r.done = true; r.slot = -1; s->slot_req[slot] = -1; }
        }
        hi = -1;
        for (int slot = 0; slot < s->max_batch; ++slot)
            if (s->slot_req[slot] >= 0) hi = slot;
    }
    // ---- one decode step for slots 0 .. hi, input = the device's own greedy tokens ----
    if (hi >= 0) {
        if ((rc = from_ctx(s, dfssm_step(s->ctx, next_dev, hi + 1))) != DFSSM_OK) return rc;
        {
            std::vector<int> live;
            for (int slot = 0; slot <= hi; ++slot)
                if (s->slot_req[slot] >= 0) live.push_back(slot);
            if ((rc = sample_slots(s, hi, live)) != DFSSM_OK) return rc;
        }
        if (cudaMemcpyAsync(s->host_next, next_dev, sizeof(int32_t) * (size_t)(hi + 1), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
            cudaStreamSynchronize(s->stream) != cudaSuccess)
            return sfail(s, DFSSM_E_CUDA, "token read-back failed");
        ++s->steps;
        s->slot_steps_run += hi + 1;
        for (int slot = 0; slot <= hi; ++slot) {
            const int id = s->slot_req[slot];
            if (id < 0) continue;
            ++s->slot_steps_used;
            dfssm_sched::Request& r = s->req[id];
            r.out.push_back(s->host_next[slot]);
            if ((int)r.out.size() >= r.max_new) { r.done = true; r.slot = -1; s->slot_req[slot] = -1; }
        }
    }
    int act = (int)s->waiting.size();
    for (int slot = 0; slot < s->max_batch; ++slot) act += s->slot_req[slot] >= 0;
    if (n_active) *n_active = act;
    return DFSSM_OK;
}

int dfssm_sched_run(dfssm_sched* s)
{
    if (!s) return DFSSM_E_ARG;
    int act = 1;
    while (act > 0) {
        const int rc = dfssm_sched_iterate(s, &act);
        if (rc != DFSSM_OK) return rc;
    }
    return from_ctx(s, dfssm_sync(s->ctx));
}

int dfssm_sched_result(dfssm_sched* s, int request_id, int32_t* tokens_host, int capacity, int* n_tokens, int* done)
{
    if (!s || request_id < 0 || request_id >= (int)s->req.size() || !n_tokens) return DFSSM_E_ARG;
    const dfssm_sched::Request& r = s->req[request_id];
    *n_tokens = (int)r.out.size();
    if (done) *done = r.done ? 1 : 0;
    if (tokens_host) {
        if (capacity < (int)r.out.size()) return sfail(s, DFSSM_E_SIZE, "result buffer too small");
        memcpy(tokens_host, r.out.data(), sizeof(int32_t) * r.out.size());
    }
    return DFSSM_OK;
}

int dfssm_sched_stats(dfssm_sched* s, long long* steps, long long* slot_steps_used, long long* slot_steps_run)
{
    if (!s) return DFSSM_E_ARG;
    if (steps) *steps = s->steps;
    if (slot_steps_used) *slot_steps_used = s->slot_steps_used;
    if (slot_steps_run) *slot_steps_run = s->slot_steps_run;
    return DFSSM_OK;
}

const char* dfssm_sched_last_error(const dfssm_sched* s) { return s ? s->err : ""; }

void dfssm_sched_destroy(dfssm_sched* s)
{
    if (!s) return;
    if (s->host_next) cudaFreeHost(s->host_next);
    if (s->host_u) cudaFreeHost(s->host_u);
    delete s;
}

}  // extern "C"
