// awg_ring.cu -- streaming ring (hot-path step a7): the stand-in for the paper's RDMA -> DAC FIFO.
//
// The paper's Streaming pathway computes chunk c+1 "in the time interval between the current and upcoming
// RDMA transfers" (Fig. 2b, Fig. 7) and under/overflows the FIFO when the compute rate does
// not match the DAC rate.  No DAC is present, so the ring is: n_slots device buffers filled
// by a synthesis stream, optionally mirrored into pinned host memory by a copy stream (the D2H transfer
// stands in for the RDMA), a virtual DAC clock that starts at the first acquire and consumes one chunk
// every chunk_len/fs seconds, and an underrun counter for chunks that were not complete when due.
#include <chrono>
#include <new>
#include <vector>

#include "awg_internal.h"
#include "awg_plan.h"

using namespace awg;
using Clock = std::chrono::steady_clock;

struct RingSlot {
    int16_t *dev = nullptr;
    int16_t *host = nullptr;
    cudaEvent_t start = nullptr, synth_done = nullptr, copy_done = nullptr;
    int64_t chunk = -1;
    Clock::time_point submitted;
};

struct awg_ring {
    awg_plan *plan = nullptr;
    int n_slots = 0;
    bool mirror = false;
    std::vector<RingSlot> slots;
    cudaStream_t s_syn = nullptr, s_cpy = nullptr;
    int64_t n_submitted = 0, n_acquired = 0, n_released = 0;  // sequence numbers; slot = seq % n_slots
    int64_t last_chunk = -1;
    int64_t underruns = 0;
    double max_ms = 0.0;
    bool started = false;
    Clock::time_point t0;
};

extern "C" {

awg_status awg_ring_destroy(awg_ring *r)
{
    if (!r) return AWG_OK;
    if (r->s_syn) cudaStreamSynchronize(r->s_syn);
    if (r->s_cpy) cudaStreamSynchronize(r->s_cpy);
    for (RingSlot &s : r->slots) {
        if (s.dev) cudaFree(s.dev);
        if (s.host) cudaFreeHost(s.host);
        if (s.start) cudaEventDestroy(s.start);
        if (s.synth_done) cudaEventDestroy(s.synth_done);
        if (s.copy_done) cudaEventDestroy(s.copy_done);
    }
    if (r->s_syn) cudaStreamDestroy(r->s_syn);
    if (r->s_cpy) cudaStreamDestroy(r->s_cpy);
    if (r->plan) r->plan->n_rings--;
    delete r;
    return AWG_OK;
}

awg_status awg_ring_create(awg_ring **out, awg_plan *p, int32_t n_slots, int32_t host_mirror)
{
    if (!out) return fail(AWG_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!p) return fail(AWG_ERR_INVALID_ARG, "plan is NULL");
    if (n_slots < 2 || n_slots > 64) return fail(AWG_ERR_INVALID_ARG, "n_slots must be in [2, 64]");
    awg_ring *r = new (std::nothrow) awg_ring();
    if (!r) return fail(AWG_ERR_ALLOC, "out of host memory");
    r->plan = p;
    p->n_rings++;
    r->n_slots = n_slots;
    r->mirror = host_mirror != 0;
    r->slots.resize(n_slots);
    const size_t bytes = static_cast<size_t>(p->chunk_len) * sizeof(int16_t);
    cudaError_t e = cudaStreamCreateWithFlags(&r->s_syn, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&r->s_cpy, cudaStreamNonBlocking);
    for (int i = 0; e == cudaSuccess && i < n_slots; ++i) {
        RingSlot &s = r->slots[i];
        e = cudaMalloc(reinterpret_cast<void **>(&s.dev), bytes);
        if (e == cudaSuccess && r->mirror) e = cudaMallocHost(reinterpret_cast<void **>(&s.host), bytes);
        if (e == cudaSuccess) e = cudaEventCreate(&s.start);
        if (e == cudaSuccess) e = cudaEventCreate(&s.synth_done);
        if (e == cudaSuccess) e = cudaEventCreate(&s.copy_done);
    }
    if (e != cudaSuccess) {
        awg_status st = (e == cudaErrorMemoryAllocation) ? fail(AWG_ERR_ALLOC, "ring allocation failed: %s", cudaGetErrorString(e))
                                                         : fail_cuda(e, "ring creation");
        awg_ring_destroy(r);
        return st;
    }
    *out = r;
    return AWG_OK;
}

awg_status awg_ring_submit(awg_ring *r, int64_t chunk_idx, int32_t n_upd, const int32_t *tone_idx, const double *f1,
                           const double *t_dur, const int32_t *profile)
{
    if (!r) return fail(AWG_ERR_INVALID_ARG, "ring is NULL");
    if (r->n_submitted - r->n_released >= r->n_slots) return fail(AWG_ERR_STATE, "ring full: acquire and release a chunk first");
    if (chunk_idx <= r->last_chunk) return fail(AWG_ERR_STATE, "chunks must be submitted in increasing order");
    awg_plan *p = r->plan;
    awg_status st;
    RingSlot &s = r->slots[r->n_submitted % r->n_slots];
    // the chunk is validated first: a rejected submit leaves the trajectory table as it was
    if ((st = check_chunk_call(p, chunk_idx, 1, s.dev, 16)) != AWG_OK) return st;
    if (n_upd > 0 && (st = apply_update(p, chunk_idx, n_upd, tone_idx, f1, t_dur, profile)) != AWG_OK) return st;
    cudaError_t e;
    // table upload (if an update is pending) goes first so that the chunk's device time measures synthesis + mirror
    if ((st = ensure_table(p, r->s_syn)) != AWG_OK) return st;
    if ((e = cudaEventRecord(s.start, r->s_syn)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
    if ((st = synthesize_samples(p, chunk_idx * p->chunk_len, p->chunk_len, s.dev, false, r->s_syn)) != AWG_OK) return st;
    if ((e = cudaEventRecord(s.synth_done, r->s_syn)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
    if (r->mirror) {
        if ((e = cudaStreamWaitEvent(r->s_cpy, s.synth_done, 0)) != cudaSuccess) return fail_cuda(e, "cudaStreamWaitEvent");
        if ((e = cudaMemcpyAsync(s.host, s.dev, static_cast<size_t>(p->chunk_len) * sizeof(int16_t), cudaMemcpyDeviceToHost, r->s_cpy)) != cudaSuccess)
            return fail_cuda(e, "cudaMemcpyAsync(D2H)");
        if ((e = cudaEventRecord(s.copy_done, r->s_cpy)) != cudaSuccess) return fail_cuda(e, "cudaEventRecord");
        p->d2h_bytes += p->chunk_len * static_cast<int64_t>(sizeof(int16_t));
    }
    s.chunk = chunk_idx;
    s.submitted = Clock::now();
    r->last_chunk = chunk_idx;
    r->n_submitted++;
    return AWG_OK;
}

awg_status awg_ring_acquire(awg_ring *r, int64_t *chunk_idx, const int16_t **dev_ptr, const int16_t **host_ptr)
{
    if (!r) return fail(AWG_ERR_INVALID_ARG, "ring is NULL");
    if (r->n_acquired >= r->n_submitted) return fail(AWG_ERR_STATE, "no submitted chunk to acquire");
    RingSlot &s = r->slots[r->n_acquired % r->n_slots];
    cudaEvent_t fin = r->mirror ? s.copy_done : s.synth_done;
    const double period = static_cast<double>(r->plan->chunk_len) / static_cast<double>(r->plan->fs);
    bool late = false;
    cudaError_t e;
    if (r->started) {
        // virtual DAC: acquired chunk j is due j periods after the first acquire returned
        const auto due = r->t0 + std::chrono::duration_cast<Clock::duration>(std::chrono::duration<double>(period * static_cast<double>(r->n_acquired)));
        if (s.submitted > due) late = true;  // enqueued after its deadline: cannot have been ready in time
        if (Clock::now() >= due) {
            e = cudaEventQuery(fin);
            if (e == cudaErrorNotReady) late = true;
            else if (e != cudaSuccess) return fail_cuda(e, "cudaEventQuery");
            if ((e = cudaEventSynchronize(fin)) != cudaSuccess) return fail_cuda(e, "cudaEventSynchronize");
        } else {
            if ((e = cudaEventSynchronize(fin)) != cudaSuccess) return fail_cuda(e, "cudaEventSynchronize");
            late = late || Clock::now() > due;
        }
    } else {
        if ((e = cudaEventSynchronize(fin)) != cudaSuccess) return fail_cuda(e, "cudaEventSynchronize");
        r->started = true;
        r->t0 = Clock::now();
    }
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s.start, fin) == cudaSuccess && ms > r->max_ms) r->max_ms = ms;
    if (chunk_idx) *chunk_idx = s.chunk;
    if (dev_ptr) *dev_ptr = s.dev;
    if (host_ptr) *host_ptr = s.host;
    r->n_acquired++;
    if (late) {
        r->underruns++;
        return fail(AWG_ERR_UNDERRUN, "chunk %lld missed its deadline", static_cast<long long>(s.chunk));
    }
    return AWG_OK;
}

awg_status awg_ring_release(awg_ring *r, int64_t chunk_idx)
{
    if (!r) return fail(AWG_ERR_INVALID_ARG, "ring is NULL");
    if (r->n_released >= r->n_acquired) return fail(AWG_ERR_STATE, "no acquired chunk to release");
    RingSlot &s = r->slots[r->n_released % r->n_slots];
    if (s.chunk != chunk_idx) return fail(AWG_ERR_STATE, "chunks are released in acquire order (expected %lld)", static_cast<long long>(s.chunk));
    r->n_released++;
    return AWG_OK;
}

awg_status awg_ring_stats(awg_ring *r, int64_t *produced, int64_t *underruns, double *max_chunk_ms)
{
    if (!r) return fail(AWG_ERR_INVALID_ARG, "ring is NULL");
    if (produced) *produced = r->n_acquired;
    if (underruns) *underruns = r->underruns;
    if (max_chunk_ms) *max_chunk_ms = r->max_ms;
    return AWG_OK;
}

}  // extern "C"
