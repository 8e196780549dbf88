// fdas_convolve_tc.cu -- K2-TC: the convolution stage as a dense contraction on the 5th-generation
// tensor cores (tcgen05.mma, accumulators in TMEM); precision modes FDAS_BF16_TC[_PLANE16].
//
// The matched filter ("a matched filtering approach") is, written out (O4),
//     y_j(r) = sum_{m=-h..h} w[r+m] conj(T_j[m]),   P[j][r] = |y_j(r)|^2 :
// a Toeplitz contraction over the 2h+1 taps.  The FFT is the fast algorithm for the
// fp32 ALUs; on B200 the tensor cores have ~30x the fp32-FMA rate, so the plain contraction
// (1032 flop/point, halved below) beats the FFT's 68 flop/point that bound K2 to the ALUs
// (profiles/r01c).  Operands are exactly the bf16 storage of reading A10 (bf16 spectrum, bf16
// templates -- here rounded in the tap domain), products are exact in fp32, accumulation is fp32.
//
//   D[r][n] = sum_k A[r][k] B[n][k],  A[r][k] = w[r - h + k]  (sliding window),  B = bank
//
// * A is never materialised: with H[rho][e] = s[rho + e] (rows of 8 bf16 = 16 bytes, s = the tile's
//   spectrum slice), the 8x16-byte core matrix (row block i, tap block a) of A is rows
//   8(i+a)..8(i+a)+7 of H, so one UMMA shared-memory descriptor with LBO = SBO = 128 bytes walks the
//   window: 4.2 KB of shared memory per part (Re w, Im w) feed a 128 x 144 operand.
// * T_{-z} = conj(T_z): with A~ = w (*) Re T_z and B~ = w (*) Im T_z (complex), y_{+z} = A~ - i B~ and
//   y_{-z} = A~ + i B~, so one pair of rows costs 4 real correlations instead of 8:
//   D1 = H_re x B, D2 = H_im x B with B's columns (Re T_z, Im T_z) interleaved, and
//   P_{+-z} = (Ar^2 + Ai^2 + Br^2 + Bi^2) +- 2 (Ar Bi - Ai Br).   The z = 0 row is |w|^2 exactly.
// * TMEM lane = r (128 per tile), column = operand column: a warp's store of one plane row is
//   128 contiguous bytes; the thread that owns r has all four values of a pair in its own lane.
//
// Warp roles of the persistent CTA (one per SM, 448 threads): warp 0 builds H for tile i+1.. (3
// stages), warp 1 allocates TMEM and issues the MMAs (one lane), warps 2..13 drain the two
// accumulator stages (TMEM -> registers -> power -> plane + block-max side plane).
#include <cuda_bf16.h>

#include <cstdint>

#include "fdas_kernels.h"
#include "fdas_tc_common.h"

namespace fdas {
namespace tc {

// Timing experiments only (never set in the product build): 1 = epilogue skips its arithmetic and
// stores, 2 = the MMA issuer skips the MMAs.
#ifndef FDAS_TC_DIAG
#define FDAS_TC_DIAG 0
#endif
#ifndef FDAS_TC_SLEEP_PROD
#define FDAS_TC_SLEEP_PROD 2000
#endif
#ifndef FDAS_TC_SLEEP_MMA
#define FDAS_TC_SLEEP_MMA 100
#endif

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// Same, for the two single-warp roles that wait most of the time (producer, MMA issuer): back off
// between polls so that the spinning warp does not take issue slots from the epilogue warps of its
// scheduler.
__device__ __forceinline__ void mbar_wait_backoff(uint32_t bar, uint32_t parity, unsigned ns) {
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        __nanosleep(ns);
    }
}
__device__ __forceinline__ void fence_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_after() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar)
                 : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 operands, fp32 accumulate, issued by one thread.
__device__ __forceinline__ void tc_mma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                       uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// TMEM -> registers: this warp's 32 lanes x 16 consecutive columns (thread = lane, v[c] = column c).
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, "
        "%13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]),
          "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
// Wait for the loads above; the registers pass through the asm so that no use is scheduled before it.
__device__ __forceinline__ void tmem_wait16(uint32_t (&a)[16], uint32_t (&b)[16]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]),
                   "+r"(a[7]), "+r"(a[8]), "+r"(a[9]), "+r"(a[10]), "+r"(a[11]), "+r"(a[12]), "+r"(a[13]),
                   "+r"(a[14]), "+r"(a[15])
                 :
                 : "memory");
    asm volatile(""
                 : "+r"(b[0]), "+r"(b[1]), "+r"(b[2]), "+r"(b[3]), "+r"(b[4]), "+r"(b[5]), "+r"(b[6]),
                   "+r"(b[7]), "+r"(b[8]), "+r"(b[9]), "+r"(b[10]), "+r"(b[11]), "+r"(b[12]), "+r"(b[13]),
                   "+r"(b[14]), "+r"(b[15])
                 :
                 : "memory");
}

// bf16 bit pattern that bounds a non-negative power from above (as fdas_convolve.cu's block max).
__device__ __forceinline__ unsigned bf16_up_pair(float a, float b) {
    return __byte_perm(__float_as_uint(a) + 0xffffu, __float_as_uint(b) + 0xffffu, 0x7632);
}

// Block maxima are reduced one chunk late so that the shared-memory round trip and the dependent
// max chain of chunk i-1 overlap the arithmetic of chunk i: this is what is still owed.
struct PendingMax {
    unsigned short* mup;
    unsigned short* mdn;
    int buf;     // scratch buffer (0/1) holding the packed powers
    int nval;    // real pairs in that chunk (0: nothing pending)
};

// Lane (pp, blk) reduces pair pp over lanes 8 blk..+7 (two 128-bit rows of the scratch buffer).
__device__ __forceinline__ void pending_load(const uint32_t* scratch, const PendingMax& pm, const int lane,
                                             uint4* v0, uint4* v1) {
    const uint32_t* row = scratch + pm.buf * 256 + (lane >> 2) * 32 + (lane & 3) * 8;
    *v0 = *reinterpret_cast<const uint4*>(row);
    *v1 = *reinterpret_cast<const uint4*>(row + 4);
}
template <int TAIL>
__device__ __forceinline__ void pending_store(const PendingMax& pm, const int lane, const uint4& v0,
                                              const uint4& v1) {
    unsigned m = __vmaxu2(__vmaxu2(v0.x, v0.y), __vmaxu2(v0.z, v0.w));
    m = __vmaxu2(m, __vmaxu2(__vmaxu2(v1.x, v1.y), __vmaxu2(v1.z, v1.w)));
    if (!TAIL || (lane >> 2) < pm.nval) {
        *pm.mup = (unsigned short)m;
        *pm.mdn = (unsigned short)(m >> 16);
    }
}

// One chunk = 8 template pairs = 16 columns of D1 (Ar, Br interleaved) and D2 (Ai, Bi): powers of
// the 16 plane rows at this thread's bin, coalesced row stores through two running row pointers
// (`up`: row mid+1+p0 ascending, `dn`: row mid-1-p0 descending; `step` = row pitch in bytes); the
// packed bf16 upper bounds go to the warp's scratch for the block maxima over aligned groups of 8
// bins, which the NEXT call reduces and stores (`pm`).  nval = real pairs in the chunk (8 unless
// TAIL, the bank's padded last chunk).
template <int PLANE16, int TAIL>
__device__ __forceinline__ void chunk_out(const uint32_t (&a)[16], const uint32_t (&b)[16], char* up,
                                          char* dn, const int64_t step, unsigned short* mup,
                                          unsigned short* mdn, const int nval, uint32_t* scratch,
                                          const int lane, PendingMax& pm) {
    uint4 v0 = make_uint4(0, 0, 0, 0), v1 = v0;
    const bool owed = pm.nval > 0;
    if (owed) pending_load(scratch, pm, lane, &v0, &v1);
    const int buf = pm.buf ^ 1;
    uint32_t* mine = scratch + buf * 256 + lane;
#pragma unroll
    for (int pp = 0; pp < 8; ++pp) {
        const float Ar = __uint_as_float(a[2 * pp]), Br = __uint_as_float(a[2 * pp + 1]);
        const float Ai = __uint_as_float(b[2 * pp]), Bi = __uint_as_float(b[2 * pp + 1]);
        float Pp, Pm;
        pair_powers(Ar, Br, Ai, Bi, &Pp, &Pm);
        unsigned packed;
        if (PLANE16) {
            const __nv_bfloat162 pk = __floats2bfloat162_rn(Pp, Pm);
            packed = *reinterpret_cast<const unsigned*>(&pk);
            if (!TAIL || pp < nval) {
                __stcs(reinterpret_cast<unsigned short*>(up), (unsigned short)packed);
                __stcs(reinterpret_cast<unsigned short*>(dn), (unsigned short)(packed >> 16));
            }
        } else {
            packed = bf16_up_pair(Pp, Pm);
            if (!TAIL || pp < nval) {
                __stcs(reinterpret_cast<float*>(up), Pp);
                __stcs(reinterpret_cast<float*>(dn), Pm);
            }
        }
        up += step;
        dn -= step;
        mine[pp * 32] = packed;
    }
    if (owed) pending_store<TAIL>(pm, lane, v0, v1);
    __syncwarp();
    pm.mup = mup;
    pm.mdn = mdn;
    pm.buf = buf;
    pm.nval = nval;
}

// z = 0: T_0 = delta, so the row is |w[r]|^2 of the stored (bf16) spectrum.
template <int PLANE16>
__device__ __forceinline__ void zero_row_out(const int mid, const int64_t r, const ConvTcParams& p,
                                             const int lane) {
    const unsigned v = __ldg(p.spec + r);
    const float re = __uint_as_float(v << 16), im = __uint_as_float(v & 0xffff0000u);
    float P = fmaf(re, re, im * im);
    unsigned w;
    if (PLANE16) {
        const __nv_bfloat16 hb = __float2bfloat16_rn(P);
        const unsigned short bits = *reinterpret_cast<const unsigned short*>(&hb);
        __stcs(reinterpret_cast<unsigned short*>(p.plane) + (int64_t)mid * p.pitch + r, bits);
        w = bits;
    } else {
        __stcs(reinterpret_cast<float*>(p.plane) + (int64_t)mid * p.pitch + r, P);
        w = (__float_as_uint(P) + 0xffffu) >> 16;
    }
    w = max(w, __shfl_xor_sync(0xffffffffu, w, 1));
    w = max(w, __shfl_xor_sync(0xffffffffu, w, 2));
    w = max(w, __shfl_xor_sync(0xffffffffu, w, 4));
    if ((lane & 7) == 0) p.maxplane[(int64_t)mid * p.mpitch + (r >> 3)] = (unsigned short)w;
}

// MAXC = ceil(gch / 3): chunks one epilogue warp drains per accumulator stage; TAIL: the bank's
// last chunk has fewer than 8 real pairs.
template <int PLANE16, int MAXC, int TAIL>
__global__ void __launch_bounds__(kThreads, 1) convolve_tc_kernel(const ConvTcParams p) {
    extern __shared__ __align__(128) unsigned char smem[];
    const Layout L = make_layout(p.bimg_bytes, p.kp);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t bar0 = smem_u32(smem + L.bar_off);
    // barriers: hfull[3] | hempty[3] | tfull[2] | tempty[2]; then the TMEM base address slot
    auto hfull = [&](int s) { return bar0 + 8u * s; };
    auto hempty = [&](int s) { return bar0 + 8u * (kHStages + s); };
    auto tfull = [&](int s) { return bar0 + 8u * (2 * kHStages + s); };
    auto tempty = [&](int s) { return bar0 + 8u * (2 * kHStages + 2 + s); };
    volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + L.bar_off + 8 * (2 * kHStages + 4));

    // ---- one-time setup: B image to shared memory, barriers, TMEM
    {
        const uint4* src = reinterpret_cast<const uint4*>(p.bimg);
        uint4* dst = reinterpret_cast<uint4*>(smem + L.b_off);
        for (int i = tid; i < p.bimg_bytes / 16; i += kThreads) dst[i] = __ldg(src + i);
        fence_async_smem();
    }
    if (warp == 0 && lane == 0) {
        for (int s = 0; s < kHStages; ++s) {
            mbar_init(hfull(s), 1);
            mbar_init(hempty(s), 1);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(tfull(s), 1);
            mbar_init(tempty(s), kEpiWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32(const_cast<uint32_t*>(tmem_slot))),
                     "r"(512u)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int64_t ntiles = p.nbins / kTileR;
    const int npair = (p.nz - 1) / 2, mid = npair;
    const int ksteps = p.kp / 16;

    if (warp == 0) {
        // ===== producer: the tile's spectrum slice -> sliding-window rows H_re, H_im
        unsigned short* sre = reinterpret_cast<unsigned short*>(smem + L.st_off);
        unsigned short* sim = reinterpret_cast<unsigned short*>(smem + L.st_off + L.st_part);
        const int nrows = p.kp + 120, nsrc = p.kp + 130;
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            const int hs = it % kHStages;
            mbar_wait_backoff(hempty(hs), ((it / kHStages) & 1) ^ 1, FDAS_TC_SLEEP_PROD);
            const int64_t base = tile * kTileR - p.h;
            for (int i = lane; i < nsrc; i += 32) {
                const int64_t idx = base + i;
                const unsigned v = (idx >= 0 && idx < p.nbins) ? __ldg(p.spec + idx) : 0u;
                sre[i] = (unsigned short)v;
                sim[i] = (unsigned short)(v >> 16);
            }
            __syncwarp();
            unsigned char* hst = smem + L.h_off + hs * L.h_stage;
            for (int rho = lane; rho < nrows; rho += 32) {
#pragma unroll
                for (int part = 0; part < 2; ++part) {
                    const uint32_t* w32 = reinterpret_cast<const uint32_t*>(part ? sim : sre) + (rho >> 1);
                    const uint4 o = window_row(w32, rho);
                    *reinterpret_cast<uint4*>(hst + part * L.h_part + rho * 16) = o;
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(hfull(hs));
        }
    } else if (warp == 1) {
        // ===== MMA issuer (one lane)
        if (lane == 0) {
            const uint32_t idesc = instr_desc(p.ng_cols());
            const uint32_t lbo = (uint32_t)(p.ngroups * p.gch * 2) * 128u;   // (ntot / 8) * 128
            int it = 0;
            uint32_t item = 0;
            for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
                const int hs = it % kHStages;
                mbar_wait_backoff(hfull(hs), (it / kHStages) & 1, FDAS_TC_SLEEP_MMA);
                tc_fence_after();
                const uint32_t a_re = smem_u32(smem + L.h_off + hs * L.h_stage);
                const uint32_t a_im = a_re + L.h_part;
                for (int g = 0; g < p.ngroups; ++g, ++item) {
                    const uint32_t st = item & 1u;
                    mbar_wait_backoff(tempty(st), ((item >> 1) & 1u) ^ 1u, FDAS_TC_SLEEP_MMA);
                    tc_fence_after();
                    const uint32_t d1 = tmem_base + st * 256u, d2 = d1 + 128u;
                    const uint32_t bbase = smem_u32(smem + L.b_off) + (uint32_t)(g * p.gch * 2) * 128u;
                    for (int ks = 0; ks < ksteps; ++ks) {
                        const uint64_t bd = smem_desc(bbase + (uint32_t)ks * 2u * lbo, lbo, 128u);
                        if (FDAS_TC_DIAG == 2) continue;
                        tc_mma(d1, smem_desc(a_re + ks * 256u, 128u, 128u), bd, idesc, ks > 0);
                        tc_mma(d2, smem_desc(a_im + ks * 256u, 128u, 128u), bd, idesc, ks > 0);
                    }
                    tc_commit(tfull(st));
                }
                tc_commit(hempty(hs));
            }
        }
    } else {
        // ===== epilogue warps: TMEM lane quarter = warp % 4, chunks c = hf, hf + 2, ...
        const int q = warp & 3, t3 = (warp - 2) >> 2;      // chunks c = t3, t3 + 3, ...
        uint32_t* scratch = reinterpret_cast<uint32_t*>(smem + L.sc_off) + (warp - 2) * 512;
        const int gch = p.gch, ngroups = p.ngroups;
        const int nmine = (gch - t3 + 2) / 3;
        constexpr int kElem = PLANE16 ? 2 : 4;
        const int64_t step = p.pitch * kElem, mpitch = p.mpitch;
        char* const plane = reinterpret_cast<char*>(p.plane);
        unsigned short* const maxplane = p.maxplane;
        const int rpp = lane >> 2;                     // the pair this lane reduces in every chunk
        PendingMax pm = {nullptr, nullptr, 0, 0};
        uint32_t item = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const int64_t r = tile * kTileR + 32 * q + lane;
            char* const col = plane + r * kElem;                                    // this bin, row 0
            unsigned short* const mcol = maxplane + ((r - lane) >> 3) + (lane & 3);    // its block
            for (int g = 0; g < ngroups; ++g, ++item) {
                const uint32_t st = item & 1u;
                if (g == 0 && t3 == 2) zero_row_out<PLANE16>(mid, r, p, lane);
                mbar_wait(tfull(st), (item >> 1) & 1u);
                tc_fence_after();
                const uint32_t tb = tmem_base + ((uint32_t)(32 * q) << 16) + st * 256u;
                uint32_t a[2][16], b[2][16];
                if (nmine > 0) {
                    tmem_ld16(tb + 16u * t3, a[0]);
                    tmem_ld16(tb + 128u + 16u * t3, b[0]);
                }
#pragma unroll
                for (int i = 0; i < MAXC; ++i) {
                    if (i < nmine) {
                        tmem_wait16(a[i & 1], b[i & 1]);
                        if (i + 1 < nmine) {
                            const uint32_t c = (uint32_t)(t3 + 3 * (i + 1));
                            tmem_ld16(tb + 16u * c, a[(i + 1) & 1]);
                            tmem_ld16(tb + 128u + 16u * c, b[(i + 1) & 1]);
                        } else {
                            // every load of this stage has landed in registers: hand it back
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) mbar_arrive(tempty(st));
                        }
                        const int p0 = (g * gch + t3 + 3 * i) * 8;
                        const int nval = TAIL ? min(8, npair - p0) : 8;
                        if ((!TAIL || nval > 0) && FDAS_TC_DIAG != 1)
                            chunk_out<PLANE16, TAIL>(a[i & 1], b[i & 1], col + (int64_t)(mid + 1 + p0) * step,
                                                     col + (int64_t)(mid - 1 - p0) * step, step,
                                                     mcol + (int64_t)(mid + 1 + p0 + rpp) * mpitch,
                                                     mcol + (int64_t)(mid - 1 - p0 - rpp) * mpitch, nval,
                                                     scratch, lane, pm);
                    }
                }
                if (nmine == 0) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty(st));
                }
            }
        }
        if (pm.nval > 0) {
            uint4 v0, v1;
            pending_load(scratch, pm, lane, &v0, &v1);
            pending_store<TAIL>(pm, lane, v0, v1);
        }
    }

    // ---- teardown
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (warp == 1) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u)
                     : "memory");
    }
}

}  // namespace tc

int convolve_tc_smem_bytes(const ConvTcParams& p) {
    const int need = tc::make_layout(p.bimg_bytes, p.kp).total;
    // at least half of the SM's shared memory, so that two CTAs (2 x 512 TMEM columns) never share an SM
    return need < 120 * 1024 ? 120 * 1024 : need;
}

template <int PLANE16>
static cudaError_t launch_tc_maxc(const ConvTcParams& p, int nsm, cudaStream_t st) {
    const int smem = convolve_tc_smem_bytes(p);
    const int maxc = (p.gch + 2) / 3;
    const bool tail = ((p.nz - 1) / 2) % 8 != 0;
    auto go = [&](auto kern) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        const int64_t ntiles = p.nbins / tc::kTileR;
        const unsigned grid = (unsigned)(ntiles < nsm ? ntiles : nsm);
        kern<<<grid, tc::kThreads, smem, st>>>(p);
        return cudaGetLastError();
    };
    if (tail) return maxc == 1 ? go(tc::convolve_tc_kernel<PLANE16, 1, 1>) : go(tc::convolve_tc_kernel<PLANE16, 2, 1>);
    return maxc == 1 ? go(tc::convolve_tc_kernel<PLANE16, 1, 0>) : go(tc::convolve_tc_kernel<PLANE16, 2, 0>);
}

cudaError_t launch_convolve_tc(int plane16, const ConvTcParams& p, int nsm, cudaStream_t st) {
    if (p.nbins % tc::kTileR != 0 || p.kp % 16 != 0 || p.gch < 1 || p.gch > 6 || (p.bimg_bytes & 15))
        return cudaErrorInvalidValue;
    return plane16 ? launch_tc_maxc<1>(p, nsm, st) : launch_tc_maxc<0>(p, nsm, st);
}

}  // namespace fdas
