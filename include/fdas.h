/*
 * fdas.h -- C ABI of libfdas.so: the data-parallel hot path of the Fourier Domain Acceleration
 * Search (FDAS), hand-written for NVIDIA B200 (sm_100a).
 *
 * Method: arxiv 2211.13517 (White, Adamek, Armour), /root/reference/PAPER.md.  The paper states
 * the method in words only -- "a matched filtering approach" whose cost "scales linearly with the
 * number of acceleration values" (section 2.1) that "relies on the Fast Fourier
 * Transform (FFT) to perform convolutions in the frequency domain", with "the most
 * computationally demanding section (the convolution stage)" optionally in bfloat16 (PAPER.md:23,
 * section 2.2), run on an SKA-like workload of "193 acceleration trials" per DM trial
 * (section 3).  The concrete definitions (FFT length, whitening, template response,
 * overlap-save bookkeeping, harmonic sums, thresholds) are the readings A1..A19 of DESIGN.md,
 * which the CPU oracle (oracle/fdas_oracle.c) implements independently.
 *
 * Conventions for every call
 *   - returns an int status (FDAS_OK = 0); nothing throws or aborts across this boundary;
 *   - pointers named d_* are DEVICE pointers owned by the caller (allocate them with the sizes
 *     fdas_plan_info reports); pointers named h_* are HOST pointers; the plan owns its templates,
 *     twiddle tables, cuFFT plan + workspace, whitening scratch and the harmonic-sum scratch
 *     (block-maximum plane of nz x nbins/8 16-bit codes, prefilter list);
 *   - the three per-trial calls only ENQUEUE work on `cuda_stream` (a cudaStream_t passed as
 *     void*, NULL = legacy default stream) and return; they never synchronise, allocate or free;
 *   - the plan's scratch is not duplicated, so the per-trial calls of one plan are ordered on the
 *     device in the order they are issued: a call on a stream other than the previous call's first
 *     waits (cudaStreamWaitEvent) for that call's work.  Independent trials overlap through
 *     fdas_search_batch or through one plan per stream; one plan is for one host thread at a time.
 */
#ifndef FDAS_H
#define FDAS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdas_plan_s* fdas_plan_t; /* opaque, library-owned */

/* Storage precision of the convolution stage (reading A10).  Arithmetic is
 * always fp32.  FP32: spectrum, templates and plane in fp32.  BF16: whitened spectrum and templates
 * stored as bfloat16 (round-to-nearest-even), plane fp32.  BF16_PLANE16: plane stored bf16 too.
 * BF16_TC / BF16_TC_PLANE16 (a separate labelled path): the same bf16 storage
 * contract, but the matched filter is evaluated as the direct tap-domain contraction
 * y_j(r) = sum_m w[r+m] conj(T_j[m]) on the tensor cores (bf16 spectrum x bf16 tap-domain templates,
 * exact products, fp32 accumulation) instead of through segment FFTs on the fp32 ALUs.  seg_len is
 * accepted and reported but does not enter this path (no overlap-save segmentation). */
enum { FDAS_FP32 = 0, FDAS_BF16 = 1, FDAS_BF16_PLANE16 = 2, FDAS_BF16_TC = 3, FDAS_BF16_TC_PLANE16 = 4 };

enum {
    FDAS_OK = 0,
    FDAS_EARG = 1,         /* invalid argument (see each call) */
    FDAS_EALLOC = 2,       /* host or device allocation failed */
    FDAS_ECUDA = 3,        /* a CUDA runtime call or kernel launch failed */
    FDAS_ECUFFT = 4,       /* a cuFFT call failed */
    FDAS_EOVERFLOW = 5,    /* more candidates than capacity (host-side helper only) */
    FDAS_EUNSUPPORTED = 6  /* valid request this build does not implement (e.g. seg_len not in {1024, 2048, 4096}, nfft > 2^30) */
};

typedef struct {
    int64_t n_in;        /* samples in the caller's series (N given to fdas_plan)            */
    int64_t nfft;        /* FFT length: largest power of two <= n_in (reading A1)            */
    int64_t nbins;       /* Nb = nfft/2 Fourier bins kept, k = 0..Nb-1 (reading A2)          */
    int32_t nz;          /* number of templates, z_j = -zmax + j*zstep (reading A6)          */
    int32_t seg_len;     /* L, overlap-save segment length in complex bins                   */
    int32_t halfwidth;   /* h: templates have 2h+1 taps (reading A5)                         */
    int32_t valid;       /* V = L - 2h valid outputs per segment                             */
    int64_t nseg;        /* S = ceil(Nb / V)                                                 */
    int64_t plane_pitch; /* elements between consecutive rows of the plane (= Nb)            */
    int32_t spec_elem_bytes;  /* bytes per COMPLEX spectrum element: 8 (fp32) or 4 (bf16)    */
    int32_t plane_elem_bytes; /* bytes per plane element: 4 or 2                             */
    int32_t precision;
    int32_t reserved;
    double zmax, zstep, tsamp, tobs; /* tobs = nfft * tsamp; f = r/tobs, fdot = z/tobs^2     */
} fdas_info_t;

/* One candidate (16 bytes).  zidx is the row j (z = -zmax + zidx*zstep); power is S_h(r, z);
 * flags bit 0 = local maximum of S_h over the 8 neighbours (r+-1, j+-1) (reading A14). */
typedef struct {
    uint32_t r;
    int16_t zidx;
    uint16_t h;
    float power;
    uint32_t flags;
} fdas_cand_t;

/*
 * fdas_plan -- build everything that does not depend on the data (readings A1, A5,
 * A6): derives nfft, Nb, nz, h, V, S; generates the template bank on the host in double precision
 * (closed-form Fresnel response of a constant-fdot signal, Ransom et al. 2002 cited at PAPER.md:75,
 * truncated to 2h+1 taps, unit L2 norm, shifted by h, FFT_L, conjugated, scaled by 1/L), casts it
 * once to fp32 or bf16 and uploads it in the kernel's register order; creates the cuFFT R2C plan
 * and the whitening block table.
 *   N        samples per time series (>= 2*seg_len); tsamp  sampling time in seconds (> 0; units only)
 *   zmax     largest |z| searched, in Fourier bins of drift over the observation (>= 0)
 *   zstep    template spacing in z (> 0); 2*zmax/zstep must be an integer (nz = that + 1 <= 32767)
 *   seg_len  L, the overlap-save segment length in complex bins: 1024, 2048 or 4096 (another power of two:
 *            FDAS_EUNSUPPORTED; FDAS_EARG if not a power of two or if V = L - 2h <= 0).  SURVEY.md 8(f) #3:
 *            the flop count per plane point, 5 L log2(L) / (L - 2h), has its minimum near 1024-2048 for the
 *            129 taps of the zmax = 96 bank.
 *   precision  FDAS_FP32 | FDAS_BF16 | FDAS_BF16_PLANE16 | FDAS_BF16_TC | FDAS_BF16_TC_PLANE16
 * On success *out receives the handle (release with fdas_destroy).
 */
int fdas_plan(fdas_plan_t* out, int64_t N, double tsamp, double zmax, double zstep, int seg_len,
              int precision);

/* Sizes and derived constants of a plan.  FDAS_EARG on NULL. */
int fdas_plan_info(fdas_plan_t plan, fdas_info_t* out);

/*
 * fdas_prepare_spectrum -- real FFT + running-median power whitening (BASELINE.json north_star;
 * readings A1, A2, A3).  X = cuFFT R2C of the first nfft samples (the one library call on the
 * path); block medians of |X|^2 over the A3 block schedule; w[k] = X[k]*sqrt(ln2/m(k)), w[0] = 0,
 * stored as complex fp32 (FDAS_FP32) or complex bf16 (RNE).
 *   d_series  device, n_in float32 samples (only the first nfft are read)
 *   d_spec    device, nbins complex elements of spec_elem_bytes each (output)
 */
int fdas_prepare_spectrum(fdas_plan_t plan, const float* d_series, void* d_spec, void* cuda_stream);

/*
 * fdas_convolve_plane -- the convolution stage (readings A7, A8, A9): for every
 * overlap-save segment s and template j, P[j][sV+t] = |IFFT_L(FFT_L(g_s) . K_j)[t]|^2, t < V,
 * g_s[i] = w[sV-h+i] (zero outside [0,Nb)), which equals |sum_m w[r+m] conj(T_j[m])|^2.
 *   d_spec   device, as written by fdas_prepare_spectrum
 *   d_plane  device, nz rows of plane_pitch elements of plane_elem_bytes (output, every element
 *            with r < nbins is written; 16-byte aligned)
 */
int fdas_convolve_plane(fdas_plan_t plan, const void* d_spec, void* d_plane, void* cuda_stream);

/*
 * fdas_harmonic_sum_peaks -- harmonic summing, thresholding, candidate compaction (BASELINE.json
 * north_star; readings A12, A13, A14): S_h(r,j) = sum_{k=1..h} P[row(k z_j)][k r] while k r <= Nb-1
 * and |k z_j| <= zmax; emits (r, j, h, S_h, flags) for every S_h > h_thresholds[h-1] (strict),
 * r in [r_lo, Nb).
 *   H             1..32;  h_thresholds  host, H floats (copied at call time)
 *   d_cands       device, capacity records, filled in unspecified order
 *   d_count       device; set to 0 by this call, then receives the TRUE number of candidates found
 *                 (it may exceed capacity; only the first `capacity` claimed slots are stored)
 * The search is exact (identical to evaluating every fundamental) but proceeds branch-and-bound on
 * a plan-owned block-maximum plane M that fdas_convolve_plane writes beside d_plane.  Contract: M is
 * trusted only when d_plane is the buffer this plan's fdas_convolve_plane wrote last and
 * fdas_plan_invalidate_plane has not been called since; a caller that changes that buffer in place
 * calls fdas_plan_invalidate_plane first.  For every other d_plane M is rebuilt from the plane on
 * EVERY call (one extra pass over it), so a caller-made plane may be refilled freely between calls.
 * Plane values must be >= 0 (they are powers).
 * FDAS_EARG: NULL pointers, H out of range, r_lo < 0, capacity < 0, a NaN threshold.
 */
int fdas_harmonic_sum_peaks(fdas_plan_t plan, const void* d_plane, int H, const float* h_thresholds,
                            int64_t r_lo, fdas_cand_t* d_cands, int64_t capacity,
                            unsigned long long* d_count, void* cuda_stream);

/*
 * fdas_plan_set_harmonic_mode -- which harmonic sum fdas_harmonic_sum_peaks (and the search calls)
 * evaluate from now on (reading A24; serves PAPER.md:9 "less than 3 % in
 * numerical sensitivity"):
 *   FDAS_HSUM_PLAIN          S_h(r,j)  = sum_{k<=h} P[row(k z_j)][k r]                       (default)
 *   FDAS_HSUM_NEIGHBOUR_MAX  S'_h(r,j) = sum_{k<=h} max_{|d| <= floor(k/2)} P[row(k z_j)][k r + d]
 * (bins clipped to [0, Nb); defined where S_h is).  A fundamental at r + delta, |delta| <= 1/2, has
 * harmonic k at k r + k delta: the plain sum misses it as soon as |k delta| > 1/2, the second form does
 * not.  S'_1 = S_1 and S'_h >= S_h, so thresholds for a given false-alarm rate are higher for S'; they
 * are the caller's.  The first switch to FDAS_HSUM_NEIGHBOUR_MAX allocates a second side plane
 * (nz x nbins/8 x 2 bytes).  FDAS_EARG: NULL plan, unknown mode.
 */
enum { FDAS_HSUM_PLAIN = 0, FDAS_HSUM_NEIGHBOUR_MAX = 1 };
int fdas_plan_set_harmonic_mode(fdas_plan_t plan, int mode);

/* Tells the plan that the plane fdas_convolve_plane wrote last has been modified (or its buffer reused)
 * by the caller: the next fdas_harmonic_sum_peaks rebuilds the block maxima from the plane it is given. */
int fdas_plan_invalidate_plane(fdas_plan_t plan);

/*
 * fdas_search_host -- the same three steps for a HOST time series (the end-to-end entry point):
 * copies the first nfft of h_series' n_in floats (the samples the transform uses, reading A1) to the
 * device, runs prepare -> convolve -> harmonic_sum_peaks on
 * `cuda_stream`, copies the count and the first min(count, capacity) candidates back and waits for
 * them.  Device workspace (series, spectrum, plane, candidates) is allocated on first use and owned
 * by the plan.  Returns FDAS_EOVERFLOW (after copying `capacity` records) if count > capacity.
 * FDAS_EARG (NULL pointers, capacity < 0, H outside 1..32, r_lo < 0, a NaN threshold) is returned before any
 * work is queued; the call first orders itself after the plan's previous call, whatever stream that used.
 */
int fdas_search_host(fdas_plan_t plan, const float* h_series, int H, const float* h_thresholds,
                     int64_t r_lo, fdas_cand_t* h_cands, int64_t capacity, int64_t* h_count,
                     void* cuda_stream);

/*
 * fdas_search_batch -- many independent DM trials through one plan ("5925 DM trials";
 * BASELINE.json configs[3] "streamed through one GPU with double-buffered planes", configs[4]).
 * Trial t is series[t]: n_in float32 samples, all DEVICE pointers (series_on_host = 0) or all HOST
 * pointers (series_on_host = 1, pinned memory for full-speed copies); `series` itself is a host array
 * of ntrials pointers.  The trials run through three plan-owned streams with two slots of every
 * per-trial buffer (series, spectrum, plane, block-max plane, candidates): the host-to-device copy of
 * trial t+1 and the harmonic sum of trial t-1 overlap the convolution of trial t.  Results are those
 * of calling prepare -> convolve -> harmonic_sum_peaks per trial:
 *   h_counts  host, ntrials: TRUE number of candidates of each trial
 *   h_cands   host, ntrials x capacity records; trial t's first min(h_counts[t], capacity) candidates
 *             start at h_cands + t*capacity (unspecified order)
 * Work already queued on `cuda_stream` is waited for first, and `cuda_stream` is ordered after all of
 * the batch's work (so events recorded on it before and after the call time the batch on the device);
 * the call returns after the last copy has landed.  The device workspace (2 planes etc.) is allocated on first use and owned by the plan.
 * FDAS_EOVERFLOW if some h_counts[t] > capacity (everything else is still valid); FDAS_EARG for NULL
 * pointers, ntrials < 0, H outside 1..32, r_lo < 0, capacity < 0.
 */
int fdas_search_batch(fdas_plan_t plan, const float* const* series, int series_on_host, int ntrials,
                      int H, const float* h_thresholds, int64_t r_lo, fdas_cand_t* h_cands,
                      int64_t capacity, int64_t* h_counts, void* cuda_stream);

/*
 * fdas_whiten_static -- the whitening half of fdas_prepare_spectrum (K1: block medians of |X|^2 over the A3
 * schedule, interpolation, w[k] = X[k] sqrt(ln2 / m(k)), w[0] = 0; readings A2, A3) as a stand-alone call
 * that needs no plan and allocates no device memory.
 *
 * Who it is for: code that is not allowed to call cudaMalloc.  Two cases we know of: a stage of a real-time
 * telescope backend that handed all of its HBM to its own pool when it started (a later cudaMalloc may fail
 * there, and even when it succeeds it synchronises the whole device and stalls the ingest streams), and a
 * plug-in inside someone else's framework that may only touch the buffers it is handed.  Such a caller
 * brings its own raw spectrum (its own FFT) and its own output buffer; the medians and the block table, which
 * fdas_plan would otherwise cudaMalloc, live in a fixed 51 KB array inside libfdas.so.  Every GPU on which the
 * library is loaded carries those 51 KB until the process exits.
 *
 *   d_X        device, at least nbins complex float32 (re, im interleaved), e.g. the output of an R2C FFT
 *   nbins      number of bins to whiten, 1024 <= nbins <= 2^24 (16 777 216).  LIMIT: the fixed array holds the
 *              tables of at most 2^24 bins; a longer spectrum is refused with FDAS_EUNSUPPORTED and a text in
 *              fdas_last_error_detail() -- use a plan for those.
 *   d_spec     device, nbins complex outputs: float32 pairs (spec_bf16 = 0) or bfloat16 pairs (spec_bf16 = 1)
 *   The three kernels are only enqueued on cuda_stream; the call does not wait for them.
 *
 * The call never calls cudaMalloc, cudaFree, cuFFT or anything else that allocates.  The first call on each
 * device looks up the device address of the array (cudaGetSymbolAddress, with that device current; the CUDA
 * runtime may load the library's kernels at that moment): make that first call during start-up, before any
 * stream capture begins on that device.
 * All calls on one device share the one array, and it keeps what the previous call left in it.  Nothing in it
 * has to be zero at the start (each call rewrites every entry it later reads), but two calls whose kernels
 * can run at the same time on the GPU -- different streams with no dependency between them, or two host
 * threads -- overwrite each other's tables: order them (one stream, or an event between the streams).
 * Results are bit-identical to fdas_prepare_spectrum's for the same X.
 * FDAS_EARG: NULL pointers, spec_bf16 not 0/1, nbins < 1024.  FDAS_ECUDA: the lookup or a launch failed.
 */
int fdas_whiten_static(const float* d_X, int64_t nbins, void* d_spec, int spec_bf16, void* cuda_stream);

/*
 * fdas_thresholds_from_sigma -- host helper (reading A13): h_thresholds_out[h-1] = T_h with
 * Q(h, T_h) = erfc(nsigma/sqrt2)/2, Q the survival function of a sum of h unit exponentials.
 */
int fdas_thresholds_from_sigma(int H, double nsigma, float* h_thresholds_out);

int fdas_destroy(fdas_plan_t plan);
const char* fdas_strerror(int status);
const char* fdas_last_error_detail(void); /* thread-local text of the last CUDA/cuFFT failure */

/* ---------------------------------------------------------------------------------------------
 * FDAS_DIAGNOSTICS -- test and measurement hooks.  NOT part of the stable ABI: they expose plan
 * internals (template bank, side plane, launch counter) and may change with the kernels.
 * ------------------------------------------------------------------------------------------- */

/*
 * fdas_plan_templates_host -- diagnostic: copies the plan's time-domain template bank
 * (nz x (2h+1) complex doubles, interleaved re/im, unit L2 norm) to h_out.  Host only.
 */
int fdas_plan_templates_host(fdas_plan_t plan, double* h_out);

/*
 * fdas_plan_debug_maxplane -- diagnostic: device pointer and row pitch (elements) of the plan-owned
 * block-maximum plane that fdas_convolve_plane writes for the harmonic-sum prefilter:
 * M[j][b] = min(1023, ceil(8 * max(P[j][8b..8b+7]))) as a 16-bit code: code/8 is an upper bound of the 8
 * stored values (the prefilter only needs M >= P), 1023 means "no bound".  The buffer stays owned by the plan.
 */
int fdas_plan_debug_maxplane(fdas_plan_t plan, const uint16_t** d_out, int64_t* pitch_out);

/*
 * fdas_plan_debug_rawspectrum -- diagnostic: device pointer to the plan-owned raw spectrum X (nfft/2 + 1
 * complex float32, the cuFFT R2C output the last fdas_prepare_spectrum whitened) and its length in complex
 * elements.  The buffer stays owned by the plan and is overwritten by the next prepare call.
 */
int fdas_plan_debug_rawspectrum(fdas_plan_t plan, const float** d_out, int64_t* ncomplex_out);

/*
 * fdas_plan_debug_fail_prepare -- diagnostic, fault injection for the error paths: the (nth + 1)-th prepare step
 * this plan enqueues from now on (through fdas_prepare_spectrum, fdas_search_host or fdas_search_batch) issues a
 * CUDA call the runtime refuses and returns FDAS_ECUDA; the counter then disarms.  nth < 0 disarms at once.
 */
int fdas_plan_debug_fail_prepare(fdas_plan_t plan, int nth);

/* Number of kernels the library launched on behalf of this plan since it was created. */
int64_t fdas_plan_launch_count(fdas_plan_t plan);

#ifdef __cplusplus
}
#endif
#endif /* FDAS_H */
