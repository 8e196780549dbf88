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
//   P_{+z} = (Ar + Bi)^2 + (Ai - Br)^2,  P_{-z} = (Ar - Bi)^2 + (Ai + Br)^2.   The z = 0 row is |w|^2 exactly.
// * TMEM lane = r (128 per tile), column = operand column: the thread that owns r has all four values
//   of a pair in its own lane, and a plane row segment of the tile is 512 contiguous bytes, staged in
//   shared memory and written with TMA tensor stores.
//
// Warp roles of the persistent CTA (one per SM, 448 threads): warp 0 builds H for tile i+1.. (3
// stages), warp 1 allocates TMEM and issues the MMAs (one lane), warps 2..13 (three warpgroups) drain
// the two accumulator stages (TMEM -> registers -> power -> plane + block-max side plane).  Two
// warpgroups are 14 % slower (too few warps to hide the drain's latencies), four do not fit the
// register file (profiles/r01e).
#include <cuda.h>
#include <cuda_bf16.h>

#include <cstdint>

#include "fdas_kernels.h"
#include "fdas_tc_common.h"

namespace fdas {
namespace tc {

// Timing experiments only (never set in the product build): 1 = epilogue skips its arithmetic and
// stores, 2 = the MMA issuer skips the MMAs, 3 = no block maxima, 4 = no TMA stores,
// 7 = every TMA store of a CTA goes to the same column block (no DRAM write stream).
#ifndef FDAS_TC_DIAG
#define FDAS_TC_DIAG 0
#endif
#ifndef FDAS_TC_WAIT_HINT
#define FDAS_TC_WAIT_HINT 20000
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
// Same for the two single-warp roles that wait most of the time (producer, MMA issuer): the thread
// is suspended in hardware until the phase completes or the time hint (ns) runs out, so the waiting
// warp does not take issue slots from the epilogue warps of its scheduler.
__device__ __forceinline__ void mbar_wait_suspend(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAITH_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
        "@p bra DONEH_%=;\n\t"
        "bra WAITH_%=;\n\t"
        "DONEH_%=:\n\t"
        "}" ::"r"(bar), "r"(parity), "r"((unsigned)FDAS_TC_WAIT_HINT) : "memory");
}
// One poll (the hardware may block for a short system-dependent time): true if the phase completed.
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t"
        "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
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

// ---- epilogue staging: a warpgroup (4 warps = the 128 bins of the tile) turns one chunk of 8
// template pairs into a [16 rows][128 bins] tile of powers in shared memory -- local rows 0..7 are
// plane rows mid+1+p0 .. +7, local rows 8..15 are plane rows mid-1-p0-7 .. mid-1-p0 (ascending) --
// which two TMA tensor stores (8 rows x 128 bins each) write to the plane; the block maxima over
// aligned groups of 8 bins are then read back from the same tile.
__device__ __forceinline__ void bar_sync_wg(int id) {
    asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory");
}
__device__ __forceinline__ void tma_store_2d(const void* tmap, uint32_t smem_src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(tmap),
                 "r"(smem_src), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// Returns once all but the newest kStageBufs - 2 committed store groups have finished READING shared
// memory (their buffers may be overwritten).
__device__ __forceinline__ void tma_wait_read_older() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kStageBufs - 2) : "memory");
}
__device__ __forceinline__ void tma_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Powers of one chunk from the accumulators of this thread's bin (column `col` of the tile) into the
// staging tile.
template <int PLANE16>
__device__ __forceinline__ void chunk_to_smem(const uint32_t (&a)[16], const uint32_t (&b)[16], void* sbuf,
                                              const int col) {
#pragma unroll
    for (int pp = 0; pp < 8; ++pp) {
        const float Ar = __uint_as_float(a[2 * pp]), Br = __uint_as_float(a[2 * pp + 1]);
        const float Ai = __uint_as_float(b[2 * pp]), Bi = __uint_as_float(b[2 * pp + 1]);
        float Pp, Pm;
        pair_powers(Ar, Br, Ai, Bi, &Pp, &Pm);
        if (PLANE16) {
            const __nv_bfloat162 pk = __floats2bfloat162_rn(Pp, Pm);
            const unsigned packed = *reinterpret_cast<const unsigned*>(&pk);
            unsigned short* t = reinterpret_cast<unsigned short*>(sbuf) + col;
            t[pp * 128] = (unsigned short)packed;
            t[(15 - pp) * 128] = (unsigned short)(packed >> 16);
        } else {
            float* t = reinterpret_cast<float*>(sbuf) + col;
            t[pp * 128] = Pp;
            t[(15 - pp) * 128] = Pm;
        }
    }
}

// Block maxima of a staged tile, one chunk late (the loads overlap the next chunk's arithmetic):
// thread tw of the warpgroup reduces block (tw & 15) of local rows tw >> 4 and 8 + (tw >> 4) and
// writes the bf16 upper bound into the [16][16] side tile, which goes out with the next TMA group.
// The two 16-byte halves of a block are read in lane-dependent order so that the 8 lanes of a
// shared-memory phase touch 8 different 16-byte bank groups.
struct MaxRegs {
    unsigned x[2];   // per task: the block's largest bit pattern (fp32) / packed bf16 pair maximum
};
template <int PLANE16>
__device__ __forceinline__ void block_max_load(const void* sbuf, const int tw, MaxRegs* m) {
    const int lr0 = tw >> 4, blk = tw & 15;
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const int lr = lr0 + 8 * t;
        if (PLANE16) {
            const uint4 u = *reinterpret_cast<const uint4*>(reinterpret_cast<const unsigned short*>(sbuf) + lr * 128 + blk * 8);
            m->x[t] = __vmaxu2(__vmaxu2(u.x, u.y), __vmaxu2(u.z, u.w));
        } else {
            // powers are >= 0: the order of the bit patterns is the order of the values
            const float* row = reinterpret_cast<const float*>(sbuf) + lr * 128 + blk * 8;
            const int sw = (blk >> 2) & 1;
            const uint4 u = *reinterpret_cast<const uint4*>(row + 4 * sw);
            const uint4 v = *reinterpret_cast<const uint4*>(row + 4 * (sw ^ 1));
            m->x[t] = max(max(max(u.x, u.y), max(u.z, u.w)), max(max(v.x, v.y), max(v.z, v.w)));
        }
    }
}
template <int PLANE16>
__device__ __forceinline__ void block_max_finish(const MaxRegs& m, unsigned short* mtile, const int tw) {
    const int lr0 = tw >> 4, blk = tw & 15;
#pragma unroll
    for (int t = 0; t < 2; ++t) {
        const unsigned bits = PLANE16 ? max(m.x[t] & 0xffffu, m.x[t] >> 16) : (m.x[t] + 0xffffu) >> 16;
        mtile[(lr0 + 8 * t) * 16 + blk] = (unsigned short)bits;
    }
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

// TAIL: the bank's pair count is not a multiple of 8 (its last chunk holds padded pairs).
template <int PLANE16, int TAIL>
__global__ void __launch_bounds__(kThreads, 1)
convolve_tc_kernel(const ConvTcParams p, const __grid_constant__ CUtensorMap tmap,
                   const __grid_constant__ CUtensorMap mmap, const __grid_constant__ CUtensorMap tmap1) {
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
            mbar_wait_suspend(hempty(hs), ((it / kHStages) & 1) ^ 1);
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
                mbar_wait_suspend(hfull(hs), (it / kHStages) & 1);
                tc_fence_after();
                const uint32_t a_re = smem_u32(smem + L.h_off + hs * L.h_stage);
                const uint32_t a_im = a_re + L.h_part;
                for (int g = 0; g < p.ngroups; ++g, ++item) {
                    const uint32_t st = item & 1u;
                    mbar_wait_suspend(tempty(st), ((item >> 1) & 1u) ^ 1u);
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
    } else if (warp < 2 + kEpiWarps) {
        // ===== epilogue warps: TMEM lane quarter = warp % 4, chunks c = hf, hf + 2, ...
        const int q = warp & 3, wg = (warp - 2) >> 2;      // warpgroup wg drains chunks wg, wg + kWarpGroups, ..
        const int tw = ((warp - 2) & 3) * 32 + lane;        // thread index inside the warpgroup
        const bool elected = (tw == 0);      // issues the warpgroup's TMA stores
        const int gch = p.gch, ngroups = p.ngroups;
        const int nmine = (gch - wg + kWarpGroups - 1) / kWarpGroups;
        unsigned char* const stage0 = smem + L.sc_off + wg * (kStageBufs * kStageBufBytes);
        const int col = 32 * q + lane;
        const uint32_t lane_base = tmem_base + ((uint32_t)(32 * q) << 16);
        const int64_t tstep = gridDim.x;
        if (nmine == 0) {
            // nothing to drain (small banks): hand every stage straight back, keep the z = 0 duty
            uint32_t item = 0;
            for (int64_t tile = blockIdx.x; tile < ntiles; tile += tstep)
                for (int g = 0; g < ngroups; ++g, ++item) {
                    if (g == 0 && wg == kWarpGroups - 1) zero_row_out<PLANE16>(mid, tile * kTileR + col, p, lane);
                    mbar_wait(tfull(item & 1u), (item >> 1) & 1u);
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty(item & 1u));
                }
        } else {
            // flat software pipeline over this warp's chunks (tile, group g, i-th own chunk): the
            // TMEM loads of chunk n+1 are issued before the arithmetic of chunk n, across stages too;
            // chunk n's powers leave through TMA group n together with the block maxima of chunk n-1
            int64_t tile = blockIdx.x;
            int g = 0, i = 0;
            uint32_t item = 0, n = 0;
            int prev_c0 = 0, prev_p0 = 0;
            uint32_t ra[16], rb[16], sa[16], sb[16];
            auto issue_ld = [&](uint32_t it_, int i_, uint32_t (&x)[16], uint32_t (&y)[16]) {
                const uint32_t tb = lane_base + (it_ & 1u) * 256u + 16u * (uint32_t)(wg + kWarpGroups * i_);
                tmem_ld16(tb, x);
                tmem_ld16(tb + 128u, y);
            };
            auto buf_of = [&](uint32_t k) { return stage0 + (k % kStageBufs) * kStageBufBytes; };
            // elected thread: the staged rows of the chunk of pairs p0.. go out as two boxes of 8 rows;
            // the bank's last chunk may hold fewer than 8 real pairs -- its rows go one by one (the
            // other local rows belong to padded pairs, whose plane rows do not exist)
            constexpr int kRowBytes = 128 * (PLANE16 ? 2 : 4);
            auto store_tile = [&](uint32_t src, int c0, int p0) {
                const int nval = npair - p0;
                if (!TAIL || nval >= 8) {
                    tma_store_2d(&tmap, src, c0, mid + 1 + p0);
                    tma_store_2d(&tmap, src + 8 * kRowBytes, c0, mid - 1 - p0 - 7);
                } else {
                    for (int pp = 0; pp < nval; ++pp) {
                        tma_store_2d(&tmap1, src + pp * kRowBytes, c0, mid + 1 + p0 + pp);
                        tma_store_2d(&tmap1, src + (15 - pp) * kRowBytes, c0, mid - 1 - p0 - pp);
                    }
                }
            };
            auto store_maxes = [&](uint32_t k, int c0, int p0) {      // side tile of chunk k
                const uint32_t src = smem_u32(buf_of(k) + kStageTileBytes);
                const int nval = npair - p0;
                if (!TAIL || nval >= 8) {
                    tma_store_2d(&mmap, src, c0 >> 3, mid + 1 + p0);
                    tma_store_2d(&mmap, src + 8 * 16 * 2, c0 >> 3, mid - 1 - p0 - 7);
                } else {
                    // 32-byte rows are below the TMA's shared-memory alignment: plain 16-byte stores
                    const uint4* t = reinterpret_cast<const uint4*>(buf_of(k) + kStageTileBytes);
                    for (int pp = 0; pp < nval; ++pp) {
                        uint4* up = reinterpret_cast<uint4*>(p.maxplane + (int64_t)(mid + 1 + p0 + pp) * p.mpitch + (c0 >> 3));
                        uint4* dn = reinterpret_cast<uint4*>(p.maxplane + (int64_t)(mid - 1 - p0 - pp) * p.mpitch + (c0 >> 3));
                        up[0] = t[2 * pp]; up[1] = t[2 * pp + 1];
                        dn[0] = t[2 * (15 - pp)]; dn[1] = t[2 * (15 - pp) + 1];
                    }
                }
            };
            // one pipeline step: consume (x, y) = chunk (tile, g, i), prefetch the next into (nx, ny)
            auto step = [&](uint32_t (&x)[16], uint32_t (&y)[16], uint32_t (&nx)[16], uint32_t (&ny)[16]) {
                int64_t ntile = tile;
                int ng = g, ni = i + 1;
                uint32_t nitem = item;
                if (ni == nmine) {
                    ni = 0;
                    ++nitem;
                    if (++ng == ngroups) {
                        ng = 0;
                        ntile += tstep;
                    }
                }
                const bool have_next = ntile < ntiles;
                tmem_wait16(x, y);
                bool fetched = false;
                if (have_next && (nitem == item || mbar_test(tfull(nitem & 1u), (nitem >> 1) & 1u))) {
                    if (nitem != item) tc_fence_after();
                    issue_ld(nitem, ni, nx, ny);
                    fetched = true;
                }
                if (nitem != item) {
                    // every load of this stage has landed in registers: hand it back to the MMA warp
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty(item & 1u));
                }
                if (g == 0 && i == 0 && wg == kWarpGroups - 1) zero_row_out<PLANE16>(mid, tile * kTileR + col, p, lane);
                const int p0 = (g * gch + wg + kWarpGroups * i) * 8;
                const int c0 = FDAS_TC_DIAG == 7 ? (int)(blockIdx.x * kTileR) : (int)(tile * kTileR);
                if (FDAS_TC_DIAG != 1) {
                    MaxRegs mr;
                    if (n > 0 && FDAS_TC_DIAG != 3) block_max_load<PLANE16>(buf_of(n - 1), tw, &mr);
                    unsigned char* sbuf = buf_of(n);
                    chunk_to_smem<PLANE16>(x, y, sbuf, col);
                    if (n > 0 && FDAS_TC_DIAG != 3)
                        block_max_finish<PLANE16>(mr, reinterpret_cast<unsigned short*>(buf_of(n - 1) + kStageTileBytes), tw);
                    if (elected) tma_wait_read_older();      // buffer n+1 (chunk n+1-kStageBufs) is free
                    fence_async_smem();
                    bar_sync_wg(1 + wg);
                    if (elected && FDAS_TC_DIAG != 4) {
                        if (p0 < npair) store_tile(smem_u32(sbuf), c0, p0);
                        if (n > 0 && prev_p0 < npair) store_maxes(n - 1, prev_c0, prev_p0);
                        tma_commit();
                    }
                }
                if (have_next && !fetched) {
                    mbar_wait(tfull(nitem & 1u), (nitem >> 1) & 1u);
                    tc_fence_after();
                    issue_ld(nitem, ni, nx, ny);
                }
                prev_c0 = c0;
                prev_p0 = p0;
                tile = ntile;
                g = ng;
                i = ni;
                item = nitem;
                ++n;
            };
            if (tile < ntiles) {
                mbar_wait(tfull(0), 0);
                tc_fence_after();
                issue_ld(0, 0, ra, rb);
            }
            while (tile < ntiles) {
                step(ra, rb, sa, sb);
                if (tile >= ntiles) break;
                step(sa, sb, ra, rb);
            }
            if (n > 0 && FDAS_TC_DIAG != 1) {
                // the last chunk's block maxima
                MaxRegs mr;
                block_max_load<PLANE16>(buf_of(n - 1), tw, &mr);
                block_max_finish<PLANE16>(mr, reinterpret_cast<unsigned short*>(buf_of(n - 1) + kStageTileBytes), tw);
                fence_async_smem();
                bar_sync_wg(1 + wg);
                if (elected) {
                    if (prev_p0 < npair) store_maxes(n - 1, prev_c0, prev_p0);
                    tma_commit();
                }
            }
            if (elected) tma_wait_all();
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

// cuTensorMapEncodeTiled through the runtime's driver entry point (libfdas.so does not link libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = [] {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qr) != cudaSuccess ||
            qr != cudaDriverEntryPointSuccess)
            f = nullptr;
        return reinterpret_cast<EncodeTiledFn>(f);
    }();
    return fn;
}

// A row-major [rows][cols] array (row pitch `pitch` elements) as a 2-D tensor stored in boxes of
// `box_rows` rows x `box_cols`.
static cudaError_t make_map(void* base, int elem_bytes, bool is_float, int64_t cols, int64_t rows,
                            int64_t pitch, int box_cols, int box_rows, CUtensorMap* map) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return cudaErrorNotSupported;
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)pitch * elem_bytes};
    const cuuint32_t box[2] = {(cuuint32_t)box_cols, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1u, 1u};
    const CUresult r = enc(map, is_float ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_UINT16, 2,
                           base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int PLANE16>
static cudaError_t launch_tc(const ConvTcParams& p, int nsm, cudaStream_t st) {
    const int smem = convolve_tc_smem_bytes(p);
    CUtensorMap pmap, mmap, pmap1;   // boxes of 8 rows; single plane rows for the bank's ragged last chunk
    cudaError_t e = make_map(p.plane, PLANE16 ? 2 : 4, !PLANE16, p.nbins, p.nz, p.pitch, tc::kTileR, 8, &pmap);
    if (e == cudaSuccess)
        e = make_map(p.plane, PLANE16 ? 2 : 4, !PLANE16, p.nbins, p.nz, p.pitch, tc::kTileR, 1, &pmap1);
    if (e == cudaSuccess)
        e = make_map(p.maxplane, 2, false, p.nbins / 8, p.nz, p.mpitch, tc::kTileR / 8, 8, &mmap);
    if (e != cudaSuccess) return e;
    const bool tail = ((p.nz - 1) / 2) % 8 != 0;
    auto kern = tail ? tc::convolve_tc_kernel<PLANE16, 1> : tc::convolve_tc_kernel<PLANE16, 0>;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    const int64_t ntiles = p.nbins / tc::kTileR;
    const unsigned grid = (unsigned)(ntiles < nsm ? ntiles : nsm);
    kern<<<grid, tc::kThreads, smem, st>>>(p, pmap, mmap, pmap1);
    return cudaGetLastError();
}

cudaError_t launch_convolve_tc(int plane16, const ConvTcParams& p, int nsm, cudaStream_t st) {
    if (p.nbins % tc::kTileR != 0 || p.kp % 16 != 0 || p.gch < 1 || p.gch > 6 || (p.bimg_bytes & 15) ||
        (reinterpret_cast<uintptr_t>(p.plane) & 15u) || ((p.pitch * (plane16 ? 2 : 4)) & 15))
        return cudaErrorInvalidValue;
    return plane16 ? launch_tc<1>(p, nsm, st) : launch_tc<0>(p, nsm, st);
}

}  // namespace fdas
