// fdas_batch.cu -- fdas_search_batch: many independent DM trials streamed through one plan
// (BASELINE.json configs[3] "streamed through one GPU with double-buffered planes" and configs[4];
// PAPER.md:35 "5925 DM trials").  Three plan-owned streams and two slots of every per-trial buffer:
//   copy stream   H2D of series i (host input only)                        slot i % 2
//   stream A      cuFFT R2C + K1 whitening + K2 convolve of trial i          slot i % 2
//   stream B      K3 harmonic sum of trial i, D2H of its count and candidates
// so that the copy of trial i+1 and the harmonic sum of trial i-1 run beside the convolution of
// trial i.  Ordering is by events only; the host blocks just once per trial, on the count of the
// PREVIOUS trial (to size its candidate copy), while the next convolution is already queued.
#include <algorithm>
#include <new>

#include "fdas_plan_priv.h"

namespace fdas {

struct BatchState {
    cudaStream_t copy = nullptr, a = nullptr, b = nullptr;
    cudaEvent_t in_ready[2] = {}, spec_done[2] = {}, k2_done[2] = {}, k3_done[2] = {}, entry = nullptr;
    cudaEvent_t leave[3] = {};
    float* series[2] = {};
    void* spec[2] = {};
    void* plane[2] = {};
    unsigned short* maxplane[2] = {};
    fdas_cand_t* cands[2] = {};
    unsigned long long* count[2] = {};
    unsigned long long* h_count = nullptr;   // pinned, 2 entries
    int64_t cap = 0;
};

void free_batch_state(BatchState* s) {
    if (!s) return;
    for (int i = 0; i < 2; ++i) {
        cudaFree(s->series[i]); cudaFree(s->spec[i]); cudaFree(s->plane[i]); cudaFree(s->maxplane[i]);
        cudaFree(s->cands[i]); cudaFree(s->count[i]);
        if (s->in_ready[i]) cudaEventDestroy(s->in_ready[i]);
        if (s->spec_done[i]) cudaEventDestroy(s->spec_done[i]);
        if (s->k2_done[i]) cudaEventDestroy(s->k2_done[i]);
        if (s->k3_done[i]) cudaEventDestroy(s->k3_done[i]);
    }
    if (s->entry) cudaEventDestroy(s->entry);
    for (int i = 0; i < 3; ++i)
        if (s->leave[i]) cudaEventDestroy(s->leave[i]);
    if (s->h_count) cudaFreeHost(s->h_count);
    if (s->copy) cudaStreamDestroy(s->copy);
    if (s->a) cudaStreamDestroy(s->a);
    if (s->b) cudaStreamDestroy(s->b);
    delete s;
}

static int make_batch_state(fdas_plan_s* plan, bool need_series, int64_t capacity) {
    const fdas_info_t& in = plan->info;
    if (!plan->batch) {
        BatchState* s = new (std::nothrow) BatchState();
        if (!s) return FDAS_EALLOC;
        plan->batch = s;
        CU(cudaStreamCreateWithFlags(&s->copy, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&s->a, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&s->b, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&s->entry, cudaEventDisableTiming));
        for (int i = 0; i < 3; ++i) CU(cudaEventCreateWithFlags(&s->leave[i], cudaEventDisableTiming));
        for (int i = 0; i < 2; ++i) {
            CU(cudaEventCreateWithFlags(&s->in_ready[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&s->spec_done[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&s->k2_done[i], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&s->k3_done[i], cudaEventDisableTiming));
            CU(cudaMalloc(&s->spec[i], (size_t)in.nbins * in.spec_elem_bytes));
            CU(cudaMalloc(&s->plane[i], (size_t)in.nz * in.plane_pitch * in.plane_elem_bytes));
            CU(cudaMalloc(&s->maxplane[i], (size_t)in.nz * (size_t)(in.nbins / 8) * sizeof(unsigned short)));
            CU(cudaMalloc(&s->count[i], sizeof(unsigned long long)));
        }
        CU(cudaMallocHost(&s->h_count, 2 * sizeof(unsigned long long)));
    }
    BatchState* s = plan->batch;
    if (need_series && !s->series[0])
        for (int i = 0; i < 2; ++i) CU(cudaMalloc(&s->series[i], (size_t)in.n_in * sizeof(float)));
    if (s->cap < capacity || !s->cands[0]) {
        for (int i = 0; i < 2; ++i) {
            cudaFree(s->cands[i]);
            s->cands[i] = nullptr;
        }
        s->cap = 0;
        const int64_t c = std::max<int64_t>(capacity, 1);
        for (int i = 0; i < 2; ++i) CU(cudaMalloc(&s->cands[i], (size_t)c * sizeof(fdas_cand_t)));
        s->cap = c;
    }
    return FDAS_OK;
}

// Count of trial t is in h_count[t & 1] once k3_done[t & 1] has fired: queue its candidate copy.
static int collect(fdas_plan_s* plan, int t, fdas_cand_t* h_cands, int64_t capacity, int64_t* h_counts,
                   bool* overflow) {
    BatchState* s = plan->batch;
    const int sl = t & 1;
    CU(cudaEventSynchronize(s->k3_done[sl]));
    const int64_t found = (int64_t)s->h_count[sl];
    h_counts[t] = found;
    if (found > capacity) *overflow = true;
    const int64_t ncopy = std::min(found, capacity);
    if (ncopy > 0)
        CU(cudaMemcpyAsync(h_cands + (size_t)t * capacity, s->cands[sl], (size_t)ncopy * sizeof(fdas_cand_t),
                           cudaMemcpyDeviceToHost, s->b));
    return FDAS_OK;
}

}  // namespace fdas

using namespace fdas;

// Queues the whole batch; on an error it returns at once (fdas_search_batch then drains the streams).
static int run_batch(fdas_plan_s* plan, const float* const* series, int series_on_host, int ntrials, int H,
                     const float* h_thresholds, int64_t r_lo, fdas_cand_t* h_cands, int64_t capacity,
                     int64_t* h_counts, cudaStream_t user) {
    const fdas_info_t& in = plan->info;
    BatchState* s = plan->batch;
    int rc = FDAS_OK;

    // everything queued on the caller's stream so far (e.g. the upload of the series) comes first
    CU(cudaEventRecord(s->entry, user));
    CU(cudaStreamWaitEvent(s->copy, s->entry, 0));
    CU(cudaStreamWaitEvent(s->a, s->entry, 0));
    CU(cudaStreamWaitEvent(s->b, s->entry, 0));

    bool overflow = false;
    // host series: the copies run two trials ahead of the kernels (both slots are filled up front;
    // slot sl is refilled with trial t+2 as soon as the spectrum of trial t exists), so that a copy
    // never waits for the host to come back from collecting an earlier trial's candidates
    auto queue_copy = [&](int t) -> int {
        const int sl = t & 1;
        CU(cudaMemcpyAsync(s->series[sl], series[t], (size_t)in.nfft * sizeof(float),   // reading A1: nfft samples used
                           cudaMemcpyHostToDevice, s->copy));
        CU(cudaEventRecord(s->in_ready[sl], s->copy));
        return FDAS_OK;
    };
    if (series_on_host)
        for (int t = 0; t < std::min(2, ntrials); ++t)
            if ((rc = queue_copy(t)) != FDAS_OK) return rc;
    for (int t = 0; t < ntrials; ++t) {
        const int sl = t & 1;
        const float* d_series = series[t];
        if (series_on_host) {
            CU(cudaStreamWaitEvent(s->a, s->in_ready[sl], 0));
            d_series = s->series[sl];
        }
        // spec[sl] was last read by K2 of trial t-2: same stream A, already ordered
        rc = fdas_enqueue_prepare(plan, d_series, s->spec[sl], s->a);
        if (rc != FDAS_OK) return rc;
        CU(cudaEventRecord(s->spec_done[sl], s->a));
        if (series_on_host && t + 2 < ntrials) {
            CU(cudaStreamWaitEvent(s->copy, s->spec_done[sl], 0));   // the slot's series has been consumed
            if ((rc = queue_copy(t + 2)) != FDAS_OK) return rc;
        }
        // plane[sl] / maxplane[sl] are free once K3 (and its flag pass) of trial t-2 is done
        if (t >= 2) CU(cudaStreamWaitEvent(s->a, s->k3_done[sl], 0));
        rc = fdas_enqueue_convolve(plan, s->spec[sl], s->plane[sl], s->maxplane[sl], s->a);
        if (rc != FDAS_OK) return rc;
        CU(cudaEventRecord(s->k2_done[sl], s->a));

        CU(cudaStreamWaitEvent(s->b, s->k2_done[sl], 0));
        rc = fdas_enqueue_harmonic(plan, s->plane[sl], s->maxplane[sl], false, H, h_thresholds, r_lo,
                                   s->cands[sl], capacity, s->count[sl], s->b);
        if (rc != FDAS_OK) return rc;
        CU(cudaMemcpyAsync(s->h_count + sl, s->count[sl], sizeof(unsigned long long), cudaMemcpyDeviceToHost, s->b));
        CU(cudaEventRecord(s->k3_done[sl], s->b));

        // candidates of the previous trial: its K3 ran beside this trial's prepare/K2 being queued.
        // cands[(t-1)&1] is next written by K3 of trial t+1, queued on stream B after this copy.
        if (t >= 1) {
            rc = collect(plan, t - 1, h_cands, capacity, h_counts, &overflow);
            if (rc != FDAS_OK) return rc;
        }
    }
    rc = collect(plan, ntrials - 1, h_cands, capacity, h_counts, &overflow);
    if (rc != FDAS_OK) return rc;
    // the caller's stream is ordered after everything the batch queued (an event recorded on it
    // after this call times the batch on the device), then wait for the last copies
    cudaStream_t all[3] = {s->copy, s->a, s->b};
    for (int i = 0; i < 3; ++i) {
        CU(cudaEventRecord(s->leave[i], all[i]));
        CU(cudaStreamWaitEvent(user, s->leave[i], 0));
    }
    for (int i = 0; i < 3; ++i) CU(cudaStreamSynchronize(all[i]));
    return overflow ? FDAS_EOVERFLOW : FDAS_OK;
}

extern "C" int fdas_search_batch(fdas_plan_t plan, const float* const* series, int series_on_host,
                                 int ntrials, int H, const float* h_thresholds, int64_t r_lo,
                                 fdas_cand_t* h_cands, int64_t capacity, int64_t* h_counts,
                                 void* cuda_stream) {
    if (!plan || !series || ntrials < 0 || !h_thresholds || !h_counts || capacity < 0 ||
        (capacity > 0 && !h_cands) || H < 1 || H > 32 || r_lo < 0)
        return FDAS_EARG;
    for (int t = 0; t < ntrials; ++t)
        if (!series[t]) return FDAS_EARG;
    for (int i = 0; i < H; ++i)
        if (h_thresholds[i] != h_thresholds[i]) return FDAS_EARG;   // NaN
    if (ntrials == 0) return FDAS_OK;
    int rc = make_batch_state(plan, series_on_host != 0, capacity);
    if (rc != FDAS_OK) return rc;
    cudaStream_t user = (cudaStream_t)cuda_stream;
    if (plan->have_last) {   // work of earlier per-trial calls on other streams comes first
        if (cudaStreamWaitEvent(user, plan->ev_last, 0) != cudaSuccess) return FDAS_ECUDA;
    }
    rc = run_batch(plan, series, series_on_host, ntrials, H, h_thresholds, r_lo, h_cands, capacity, h_counts,
                   user);
    if (rc != FDAS_OK && rc != FDAS_EOVERFLOW) {
        // an enqueue failed mid-pipeline: work already queued still writes into h_cands and the pinned
        // counters, so wait for it (best effort) before the caller may free or reuse them
        BatchState* s = plan->batch;
        cudaStreamSynchronize(s->copy);
        cudaStreamSynchronize(s->a);
        cudaStreamSynchronize(s->b);
        // the failed call left its code in the runtime's last-error slot: clear it, or the next kernel launch
        // of this thread would report it (the launch checks read cudaGetLastError)
        cudaGetLastError();
    }
    // every stream of the batch has been waited for: nothing of this plan is in flight
    plan->have_last = false;
    plan->max_valid_for = nullptr;
    return rc;
}
