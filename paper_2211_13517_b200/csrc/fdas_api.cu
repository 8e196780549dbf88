// fdas_api.cu -- the C ABI of libfdas.so (include/fdas.h): plan construction, the three per-trial
// calls, the host end-to-end entry point.  No exceptions cross the boundary.
#include <cuda_runtime.h>
#include <cufft.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/fdas.h"
#include "fdas_fft_core.cuh"
#include "fdas_host.h"
#include "fdas_kernels.h"
#include "fdas_plan_priv.h"

using namespace fdas;

thread_local std::string g_detail;

// K3 prefilter survivors (fundamentals) listed per call: half of the plane's points, between 2^16 and 2^22
// records of 8 bytes (a list that overflows falls back to the exact full scan, so the size is a speed matter)
static int64_t maybe_capacity_for(const fdas_info_t& in) {
    const int64_t half = (int64_t)in.nz * in.nbins / 2;
    return std::min<int64_t>((int64_t)1 << 22, std::max<int64_t>((int64_t)1 << 16, half));
}

static void free_plan(fdas_plan_s* p) {
    if (!p) return;
    free_batch_state(p->batch);
    cudaFree(p->d_maxplane); cudaFree(p->d_maxplane_nbr); cudaFree(p->d_maybe); cudaFree(p->d_maybe_count);
    cudaFree(p->d_max2);
    cudaFree(p->d_bank); cudaFree(p->d_tw1); cudaFree(p->d_tw2); cudaFree(p->d_fft_work);
    cudaFree(p->d_X); cudaFree(p->d_blk_start); cudaFree(p->d_blk_len); cudaFree(p->d_blk_med);
    cudaFree(p->ws_series); cudaFree(p->ws_spec); cudaFree(p->ws_plane); cudaFree(p->ws_cands);
    cudaFree(p->ws_count);
    if (p->h_count) cudaFreeHost(p->h_count);
    if (p->ev_last) cudaEventDestroy(p->ev_last);
    if (p->fft_made) cufftDestroy(p->fft);
    delete p;
}

static int derive_info(int64_t N, double tsamp, double zmax, double zstep, int seg_len, int precision,
                       fdas_info_t* o) {
    if (N < 2 || !(tsamp > 0.0) || !(zmax >= 0.0) || !(zstep > 0.0) || seg_len < 2) return FDAS_EARG;
    if (precision < FDAS_FP32 || precision > FDAS_BF16_TC_PLANE16) return FDAS_EARG;
    if ((seg_len & (seg_len - 1)) != 0) return FDAS_EARG;
    if (N < 2 * (int64_t)seg_len) return FDAS_EARG;
    const double cnt = 2.0 * zmax / zstep;
    const double rc = std::floor(cnt + 0.5);
    if (std::fabs(cnt - rc) > 1e-9 * (1.0 + cnt) || rc + 1 > 32767.0) return FDAS_EARG;
    std::memset(o, 0, sizeof(*o));
    o->n_in = N;
    int64_t nfft = 1;
    while (nfft * 2 <= N) nfft *= 2;
    if (nfft > ((int64_t)1 << 30)) return FDAS_EUNSUPPORTED;  // cuFFT plan size and 32-bit bin indices
    o->nfft = nfft;
    o->nbins = nfft / 2;
    o->nz = (int)rc + 1;
    o->seg_len = seg_len;
    o->halfwidth = template_halfwidth(zmax);
    o->valid = seg_len - 2 * o->halfwidth;
    if (o->valid <= 0) return FDAS_EARG;
    o->nseg = (o->nbins + o->valid - 1) / o->valid;
    o->plane_pitch = o->nbins;
    o->spec_elem_bytes = (precision == FDAS_FP32) ? 8 : 4;
    o->plane_elem_bytes = fdas_plane16(precision) ? 2 : 4;
    o->precision = precision;
    o->zmax = zmax; o->zstep = zstep; o->tsamp = tsamp; o->tobs = (double)nfft * tsamp;
    if (!seg_len_supported(seg_len)) return FDAS_EUNSUPPORTED;
    return FDAS_OK;
}

static int build_plan(fdas_plan_s* p) {
    const fdas_info_t& in = p->info;
    Bank bank;
    build_bank(in.zmax, in.zstep, in.nz, in.halfwidth, in.seg_len, &bank);
    p->bank_time = bank.time;
    if (fdas_is_tc(in.precision)) {
        bool fits = tc_geometry(in.nz, in.halfwidth, &p->tc) && in.nbins % 128 == 0;
        if (fits) {   // window stages + epilogue tiles within the CTA's shared memory
            int dev0 = 0, optin = 0;
            CU(cudaGetDevice(&dev0));
            CU(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev0));
            fits = convolve_tc_smem_bytes(p->tc.kp, p->tc.chunk, fdas_plane16(in.precision)) <= optin;
        }
        if (!fits) {
            g_detail = "FDAS_BF16_TC: template bank does not fit the tensor-core kernel (at least one conjugate pair, <= 255 taps, nbins % 128 == 0)";
            return FDAS_EUNSUPPORTED;
        }
        std::vector<uint32_t> img;
        double asym = 0.0;
        pack_bank_tc(bank, p->tc, &img, &asym);
        if (asym > 1e-12) {
            g_detail = "FDAS_BF16_TC: bank is not conjugate-symmetric in z";
            return FDAS_EUNSUPPORTED;
        }
        CU(cudaMalloc(&p->d_bank, img.size() * sizeof(uint32_t)));
        CU(cudaMemcpy(p->d_bank, img.data(), img.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    } else if (in.precision == FDAS_FP32) {
        std::vector<float> packed;
        pack_bank_fp32(bank, &packed);
        CU(cudaMalloc(&p->d_bank, packed.size() * sizeof(float)));
        CU(cudaMemcpy(p->d_bank, packed.data(), packed.size() * sizeof(float), cudaMemcpyHostToDevice));
    } else {
        std::vector<uint32_t> packed;
        pack_bank_bf16(bank, &packed);
        CU(cudaMalloc(&p->d_bank, packed.size() * sizeof(uint32_t)));
        CU(cudaMemcpy(p->d_bank, packed.data(), packed.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    }
    if (!fdas_is_tc(in.precision)) {   // twiddle tables of the segment FFT: the tensor-core path has no use for them
        std::vector<float> t1, t2;
        build_twiddles(in.seg_len, &t1, &t2);
        CU(cudaMalloc(&p->d_tw1, t1.size() * sizeof(float)));
        CU(cudaMalloc(&p->d_tw2, t2.size() * sizeof(float)));
        CU(cudaMemcpy(p->d_tw1, t1.data(), t1.size() * sizeof(float), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(p->d_tw2, t2.data(), t2.size() * sizeof(float), cudaMemcpyHostToDevice));
    }

    std::vector<int32_t> bs, bl;
    whitening_blocks(in.nbins, &bs, &bl);
    p->nblk = (int)bs.size();
    CU(cudaMalloc(&p->d_blk_start, bs.size() * sizeof(int32_t)));
    CU(cudaMalloc(&p->d_blk_len, bl.size() * sizeof(int32_t)));
    CU(cudaMalloc(&p->d_blk_med, bs.size() * sizeof(float)));
    CU(cudaMemcpy(p->d_blk_start, bs.data(), bs.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    CU(cudaMemcpy(p->d_blk_len, bl.data(), bl.size() * sizeof(int32_t), cudaMemcpyHostToDevice));

    CU(cudaMalloc(&p->d_maxplane, (size_t)in.nz * (size_t)(in.nbins / 8) * sizeof(unsigned short)));
    p->maybe_capacity = maybe_capacity_for(in);
    CU(cudaMalloc(&p->d_maybe, (size_t)p->maybe_capacity * sizeof(uint2)));
    CU(cudaMalloc(&p->d_maybe_count, 2 * sizeof(unsigned long long)));
    if (in.nbins % 64 == 0) {
        CU(cudaMalloc(&p->d_max2, (size_t)(in.nbins / 64) * (size_t)in.nz * sizeof(unsigned short)));
    }
    CU(cudaMalloc(&p->d_X, (size_t)(in.nfft / 2 + 1) * sizeof(float2)));
    size_t ws = 0;
    CF(cufftCreate(&p->fft));
    p->fft_made = true;
    CF(cufftSetAutoAllocation(p->fft, 0));
    CF(cufftMakePlan1d(p->fft, (int)in.nfft, CUFFT_R2C, 1, &ws));
    if (ws > 0) CU(cudaMalloc(&p->d_fft_work, ws));
    CF(cufftSetWorkArea(p->fft, p->d_fft_work));

    int dev = 0, nsm = 148;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    p->nsm = nsm;
    const int64_t slots = (int64_t)convolve_ctas_per_sm(in.seg_len) * nsm;
    int nsplit = 1;
    if (in.nseg < 4 * slots) nsplit = (int)std::min<int64_t>(in.nz, (4 * slots + in.nseg - 1) / in.nseg);
    p->nsplit = nsplit;
    CU(cudaEventCreateWithFlags(&p->ev_last, cudaEventDisableTiming));
    return FDAS_OK;
}

int fdas_enqueue_prepare(fdas_plan_s* plan, const float* d_series, void* d_spec, cudaStream_t st) {
    if (plan->fail_prepare_in >= 0 && plan->fail_prepare_in-- == 0) {   // test hook, off (-1) unless armed
        cudaMemcpyAsync(nullptr, nullptr, 1, cudaMemcpyDeviceToDevice, st);   // a real refused call: leaves its code in the last-error slot
        g_detail = "injected failure (fdas_plan_debug_fail_prepare)";
        return FDAS_ECUDA;
    }
    CF(cufftSetStream(plan->fft, st));
    CF(cufftExecR2C(plan->fft, const_cast<float*>(d_series), reinterpret_cast<cufftComplex*>(plan->d_X)));
    WhitenParams w;
    w.X = plan->d_X; w.spec = d_spec;
    w.blk_start = plan->d_blk_start; w.blk_len = plan->d_blk_len; w.blk_med = plan->d_blk_med;
    w.nblk = plan->nblk; w.nbins = plan->info.nbins;
    CU(launch_whiten(plan->info.precision == FDAS_FP32 ? FDAS_FP32 : FDAS_BF16, w, st));
    plan->launches += 2;
    return FDAS_OK;
}

int fdas_enqueue_convolve(fdas_plan_s* plan, const void* d_spec, void* d_plane,
                          unsigned short* d_maxplane, cudaStream_t st) {
    if (fdas_is_tc(plan->info.precision)) {
        ConvTcParams t;
        t.spec = reinterpret_cast<const unsigned*>(d_spec); t.plane = d_plane;
        t.nbins = plan->info.nbins; t.pitch = plan->info.plane_pitch;
        t.nz = plan->info.nz; t.h = plan->info.halfwidth; t.kp = plan->tc.kp; t.npair_total = plan->tc.npair;
        t.maxplane = d_maxplane; t.mpitch = plan->info.nbins / 8;
        // a bank of more than 128 conjugate pairs takes one launch per chunk of pairs (each reads the
        // spectrum again, 17 MB, and writes its own rows of the plane)
        for (int c = 0; c < plan->tc.nchunk; ++c) {
            t.pair0 = c * plan->tc.chunk;
            t.npair = std::min(plan->tc.chunk, plan->tc.npair - t.pair0);
            t.bimg = reinterpret_cast<const uint32_t*>(plan->d_bank) + (size_t)c * 2 * 128 * (plan->tc.kp / 2);
            CU(launch_convolve_tc(fdas_plane16(plan->info.precision), t, &plan->tc_maps, plan->nsm, st));
            plan->launches += 1;
        }
        return FDAS_OK;
    }
    ConvParams c;
    c.spec = d_spec; c.plane = d_plane; c.bank = plan->d_bank; c.tw1 = plan->d_tw1; c.tw2 = plan->d_tw2;
    c.nbins = plan->info.nbins; c.pitch = plan->info.plane_pitch;
    c.nz = plan->info.nz; c.h = plan->info.halfwidth; c.V = plan->info.valid;
    c.maxplane = d_maxplane; c.mpitch = plan->info.nbins / 8;
    CU(launch_convolve(plan->info.precision, plan->info.seg_len, c, plan->info.nseg, plan->nsplit, st));
    plan->launches += 1;
    return FDAS_OK;
}

int fdas_enqueue_harmonic(fdas_plan_s* plan, const void* d_plane, unsigned short* d_maxplane,
                          bool build_max, int H, const float* h_thresholds, int64_t r_lo,
                          fdas_cand_t* d_cands, int64_t capacity, unsigned long long* d_count,
                          cudaStream_t st) {
    HarmParams hp;
    hp.plane = d_plane; hp.nbins = plan->info.nbins; hp.pitch = plan->info.plane_pitch;
    hp.nz = plan->info.nz; hp.H = H; hp.r_lo = r_lo;
    for (int i = 0; i < 32; ++i) hp.thr[i] = (i < H) ? h_thresholds[i] : INFINITY;
    hp.cands = d_cands; hp.capacity = capacity; hp.count = d_count;
    hp.maxplane = d_maxplane; hp.mpitch = plan->info.nbins / 8;
    hp.maybe = plan->d_maybe; hp.maybe_capacity = plan->maybe_capacity; hp.maybe_count = plan->d_maybe_count;
    hp.overflow = reinterpret_cast<unsigned*>(plan->d_maybe_count + 1);
    hp.max2 = plan->d_max2;
    hp.nbr = plan->hsum_mode == FDAS_HSUM_NEIGHBOUR_MAX ? 1 : 0;
    hp.maxplane_nbr = plan->d_maxplane_nbr;
    int nl = 0;
    CU(launch_harmonic(fdas_plane16(plan->info.precision), build_max, hp, st, &nl));
    plan->launches += nl;
    return FDAS_OK;
}

// The plan's scratch (cuFFT work area, median table, block-max plane, prefilter list) is shared by
// every call, so calls on different streams are ordered in issue order: a call on a stream other than
// the previous call's first waits (on the device) for that call's work.
static int order_before(fdas_plan_s* p, cudaStream_t st) {
    if (p->have_last && p->last_stream != st) CU(cudaStreamWaitEvent(st, p->ev_last, 0));
    return FDAS_OK;
}
static int order_after(fdas_plan_s* p, cudaStream_t st) {
    CU(cudaEventRecord(p->ev_last, st));
    p->last_stream = st;
    p->have_last = true;
    return FDAS_OK;
}

extern "C" {

int fdas_plan(fdas_plan_t* out, int64_t N, double tsamp, double zmax, double zstep, int seg_len,
              int precision) {
    if (!out) return FDAS_EARG;
    *out = nullptr;
    fdas_info_t info;
    const int rc = derive_info(N, tsamp, zmax, zstep, seg_len, precision, &info);
    if (rc != FDAS_OK) return rc;
    fdas_plan_s* p = new (std::nothrow) fdas_plan_s();
    if (!p) return FDAS_EALLOC;
    p->info = info;
    int st;
    try {
        st = build_plan(p);
    } catch (const std::bad_alloc&) {
        st = FDAS_EALLOC;
    } catch (...) {
        st = FDAS_ECUDA;
    }
    if (st != FDAS_OK) {
        free_plan(p);
        return st;
    }
    *out = p;
    return FDAS_OK;
}

int fdas_plan_info(fdas_plan_t plan, fdas_info_t* out) {
    if (!plan || !out) return FDAS_EARG;
    *out = plan->info;
    return FDAS_OK;
}

int fdas_prepare_spectrum(fdas_plan_t plan, const float* d_series, void* d_spec, void* cuda_stream) {
    if (!plan || !d_series || !d_spec) return FDAS_EARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = order_before(plan, st);
    if (rc == FDAS_OK) rc = fdas_enqueue_prepare(plan, d_series, d_spec, st);
    if (rc == FDAS_OK) rc = order_after(plan, st);
    return rc;
}

int fdas_convolve_plane(fdas_plan_t plan, const void* d_spec, void* d_plane, void* cuda_stream) {
    if (!plan || !d_spec || !d_plane) return FDAS_EARG;
    if ((reinterpret_cast<uintptr_t>(d_plane) & 15u) != 0) return FDAS_EARG;
    plan->max_valid_for = nullptr;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = order_before(plan, st);
    if (rc == FDAS_OK) rc = fdas_enqueue_convolve(plan, d_spec, d_plane, plan->d_maxplane, st);
    if (rc == FDAS_OK) rc = order_after(plan, st);
    if (rc == FDAS_OK) plan->max_valid_for = d_plane;
    return rc;
}

int fdas_plan_set_harmonic_mode(fdas_plan_t plan, int mode) {
    if (!plan || (mode != FDAS_HSUM_PLAIN && mode != FDAS_HSUM_NEIGHBOUR_MAX)) return FDAS_EARG;
    if (mode == FDAS_HSUM_NEIGHBOUR_MAX && !plan->d_maxplane_nbr)
        CU(cudaMalloc(&plan->d_maxplane_nbr,
                      (size_t)plan->info.nz * (size_t)(plan->info.nbins / 8) * sizeof(unsigned short)));
    plan->hsum_mode = mode;
    return FDAS_OK;
}

int fdas_plan_invalidate_plane(fdas_plan_t plan) {
    if (!plan) return FDAS_EARG;
    plan->max_valid_for = nullptr;
    return FDAS_OK;
}

int fdas_harmonic_sum_peaks(fdas_plan_t plan, const void* d_plane, int H, const float* h_thresholds,
                            int64_t r_lo, fdas_cand_t* d_cands, int64_t capacity,
                            unsigned long long* d_count, void* cuda_stream) {
    if (!plan || !d_plane || !h_thresholds || !d_count) return FDAS_EARG;
    if (H < 1 || H > 32 || r_lo < 0 || capacity < 0 || (capacity > 0 && !d_cands)) return FDAS_EARG;
    for (int i = 0; i < H; ++i)
        if (std::isnan(h_thresholds[i])) return FDAS_EARG;
    // M describes the plane fdas_convolve_plane last wrote (until fdas_plan_invalidate_plane); any
    // other plane gets its own M first, on every call: its contents may have changed since the last one
    const bool build_max = (plan->max_valid_for != d_plane);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = order_before(plan, st);
    if (rc == FDAS_OK)
        rc = fdas_enqueue_harmonic(plan, d_plane, plan->d_maxplane, build_max, H, h_thresholds, r_lo, d_cands,
                                   capacity, d_count, st);
    if (rc == FDAS_OK) rc = order_after(plan, st);
    if (build_max) plan->max_valid_for = nullptr;   // M now belongs to a plane this plan did not write
    return rc;
}

int fdas_search_host(fdas_plan_t plan, const float* h_series, int H, const float* h_thresholds,
                     int64_t r_lo, fdas_cand_t* h_cands, int64_t capacity, int64_t* h_count,
                     void* cuda_stream) {
    if (!plan || !h_series || !h_thresholds || !h_count || capacity < 0 || (capacity > 0 && !h_cands))
        return FDAS_EARG;
    // everything fdas_harmonic_sum_peaks would refuse is refused here, before any work is queued
    if (H < 1 || H > 32 || r_lo < 0) return FDAS_EARG;
    for (int i = 0; i < H; ++i)
        if (std::isnan(h_thresholds[i])) return FDAS_EARG;
    const fdas_info_t& in = plan->info;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the workspace is the plan's: wait for the previous call's work (possibly on another stream) before
    // the copy below overwrites its series
    {
        const int rc0 = order_before(plan, st);
        if (rc0 != FDAS_OK) return rc0;
    }
    if (!plan->ws_series) {
        CU(cudaMalloc(&plan->ws_series, (size_t)in.n_in * sizeof(float)));
        CU(cudaMalloc(&plan->ws_spec, (size_t)in.nbins * in.spec_elem_bytes));
        CU(cudaMalloc(&plan->ws_plane, (size_t)in.nz * in.plane_pitch * in.plane_elem_bytes));
        CU(cudaMalloc(&plan->ws_count, sizeof(unsigned long long)));
        CU(cudaMallocHost(&plan->h_count, sizeof(unsigned long long)));
    }
    if (plan->ws_cap < capacity) {
        cudaFree(plan->ws_cands);
        plan->ws_cands = nullptr;
        plan->ws_cap = 0;
        CU(cudaMalloc(&plan->ws_cands, (size_t)capacity * sizeof(fdas_cand_t)));
        plan->ws_cap = capacity;
    }
    // only the first nfft samples enter the transform (reading A1): the tail is not copied
    CU(cudaMemcpyAsync(plan->ws_series, h_series, (size_t)in.nfft * sizeof(float), cudaMemcpyHostToDevice, st));
    int rc = fdas_prepare_spectrum(plan, plan->ws_series, plan->ws_spec, cuda_stream);
    if (rc != FDAS_OK) return rc;
    rc = fdas_convolve_plane(plan, plan->ws_spec, plan->ws_plane, cuda_stream);
    if (rc != FDAS_OK) return rc;
    rc = fdas_harmonic_sum_peaks(plan, plan->ws_plane, H, h_thresholds, r_lo, plan->ws_cands, capacity,
                                 plan->ws_count, cuda_stream);
    if (rc != FDAS_OK) return rc;
    CU(cudaMemcpyAsync(plan->h_count, plan->ws_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    const int64_t found = (int64_t)*plan->h_count;
    *h_count = found;
    const int64_t ncopy = found < capacity ? found : capacity;
    if (ncopy > 0) {
        CU(cudaMemcpyAsync(h_cands, plan->ws_cands, (size_t)ncopy * sizeof(fdas_cand_t), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
    }
    return found > capacity ? FDAS_EOVERFLOW : FDAS_OK;
}

int fdas_thresholds_from_sigma(int H, double nsigma, float* h_thresholds_out) {
    if (H < 1 || H > 32 || !h_thresholds_out || !(nsigma > 0.0)) return FDAS_EARG;
    return thresholds_from_sigma(H, nsigma, h_thresholds_out) == 0 ? FDAS_OK : FDAS_EARG;
}

int fdas_plan_templates_host(fdas_plan_t plan, double* h_out) {
    if (!plan || !h_out) return FDAS_EARG;
    std::memcpy(h_out, plan->bank_time.data(), plan->bank_time.size() * sizeof(cd));
    return FDAS_OK;
}

int fdas_plan_debug_maxplane(fdas_plan_t plan, const uint16_t** d_out, int64_t* pitch_out) {
    if (!plan || !d_out || !pitch_out) return FDAS_EARG;
    *d_out = plan->d_maxplane;
    *pitch_out = plan->info.nbins / 8;
    return FDAS_OK;
}

int fdas_plan_debug_rawspectrum(fdas_plan_t plan, const float** d_out, int64_t* ncomplex_out) {
    if (!plan || !d_out || !ncomplex_out) return FDAS_EARG;
    *d_out = reinterpret_cast<const float*>(plan->d_X);
    *ncomplex_out = plan->info.nfft / 2 + 1;
    return FDAS_OK;
}

int fdas_plan_debug_fail_prepare(fdas_plan_t plan, int nth) {
    if (!plan) return FDAS_EARG;
    plan->fail_prepare_in = nth;
    return FDAS_OK;
}

int64_t fdas_plan_launch_count(fdas_plan_t plan) { return plan ? plan->launches : -1; }

int fdas_destroy(fdas_plan_t plan) {
    if (!plan) return FDAS_EARG;
    free_plan(plan);
    return FDAS_OK;
}

const char* fdas_strerror(int status) {
    switch (status) {
        case FDAS_OK: return "ok";
        case FDAS_EARG: return "invalid argument";
        case FDAS_EALLOC: return "allocation failed";
        case FDAS_ECUDA: return "CUDA error";
        case FDAS_ECUFFT: return "cuFFT error";
        case FDAS_EOVERFLOW: return "more candidates than capacity";
        case FDAS_EUNSUPPORTED: return "unsupported configuration (this build: seg_len = 1024, 2048 or 4096; nfft <= 2^30)";
        default: return "unknown status";
    }
}

const char* fdas_last_error_detail(void) { return g_detail.c_str(); }

}  // extern "C"
