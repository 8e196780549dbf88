// fdas_convolve_tc.cu -- K2-TC: the convolution stage as a dense contraction on the 5th-generation
// tensor cores (tcgen05.mma, accumulators in TMEM); precision modes FDAS_BF16_TC[_PLANE16].
//
// The matched filter ("a matched filtering approach") is, written out (O4),
//     y_j(r) = sum_{m=-h..h} w[r+m] conj(T_j[m]),   P[j][r] = |y_j(r)|^2 :
// a Toeplitz contraction over the 2h+1 taps.  The FFT is the fast algorithm for the
// fp32 ALUs; on B200 the tensor cores have ~30x the fp32-FMA rate, so the plain contraction beats the
// FFT's 68 flop/point that bound K2 to the ALUs (profiles/r01c).  Operands are exactly the bf16
// storage of reading A10/A22 (bf16 spectrum, bf16 tap-domain templates), products are exact in fp32,
// accumulation is fp32.
//
//   D[p][n] = sum_k A[p][k] B[n][k]      A = the BANK (M = 128 template pairs, in TMEM),
//                                        B = the sliding window of the spectrum (N, shared memory)
//
// * T_{-z} = conj(T_z): with A~ = w (*) Re T_z and B~ = w (*) Im T_z (complex), y_{+z} = A~ - i B~ and
//   y_{-z} = A~ + i B~, so one PAIR of rows costs 4 real correlations instead of 8.  Lane p of TMEM
//   belongs to pair p (rows j+ = nz - npair + p and j- = npair - 1 - p); D_R = (Re T) x window and
//   D_I = (Im T) x window are two accumulators over the same B operand.  A z = 0 row (odd nz) is
//   |w|^2 exactly (T_0 = delta) and is written by the producer warp.
// * The bank never leaves TMEM: both images (Re T, Im T; 128 lanes x kp/2 columns of packed bf16
//   pairs) are written once per CTA with tcgen05.st and read by every MMA as the A operand
//   (tcgen05.mma with A in tensor memory), so the only shared-memory operand traffic is the window.
// * The window is never materialised as a matrix: row rho of a part is the 16 bytes s[rho..rho+7] of
//   the tile's spectrum slice, groups of 8 rows of Re w and Im w alternate, and ONE K-major no-swizzle
//   descriptor (SBO = 128 B, LBO = 256 B) reads the N = 64 operand rows (32 bins x {re, im}) of a
//   sub-tile: columns 16 g .. 16 g + 7 of D_R are Ar of bins 8 g .. 8 g + 7, columns 16 g + 8 .. + 15 Ai.
// * Epilogue: the thread that owns lane p reads 16 + 16 consecutive columns (tcgen05.ld 32x32b.x16)
//   = everything for 8 consecutive bins of rows j+ and j-: powers, the 8-bin block maximum (a register
//   reduction), two 16-byte shared-memory stores per row into a swizzled [32 rows][32 bins] tile, and
//   one TMA tensor store per tile.  A warp works alone (no block-level barrier in the epilogue); the only
//   exchange between warps is the 16 bytes of block maxima per row that set 0 hands to set 1 (fp32 plane), so
//   that they reach memory as whole 32-byte sectors.
//
// Warp roles of the persistent CTA (one per SM, 320 threads): warps 0..3 drain sub-tiles 0, 1 of
// every 128-bin tile and warps 4..7 sub-tiles 2, 3 (warp % 4 = the TMEM lane quarter = 32 template
// pairs); warp 8 builds the window for tile i+1.. and writes the z = 0 row; warp 9 allocates TMEM and
// issues the MMAs (one lane).
#include <cuda.h>
#include <cuda_bf16.h>

#include <cstdint>

#include "fdas_kernels.h"
#include "fdas_maxcode.h"
#include "fdas_tc_common.h"

namespace fdas {
namespace tc {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// The waiting thread is suspended in hardware until the phase completes or a system-dependent time
// limit runs out, so a waiting warp takes no issue slots from the working warps of its scheduler.
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
// One lane of the (converged) warp: the issuer of the warp's tcgen05.mma / tcgen05.commit instructions.
// The same lane is elected every time, so the commits track the MMAs of the same thread.
__device__ __forceinline__ bool elect_one() {
    uint32_t pred = 0;
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "@p mov.u32 %0, 1;\n\t"
        "}" : "+r"(pred));
    return pred != 0;
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
// D[tmem] (+)= A[tmem] * B[smem]^T, bf16 operands, fp32 accumulate, issued by one thread.
__device__ __forceinline__ void tc_mma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc,
                                          uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t"
        "}" ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// TMEM <-> registers: this warp's 32 lanes x consecutive columns (thread = lane, v[c] = column c).
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
// Wait for the loads above; every register passes through an asm so that no use is scheduled before it.
__device__ __forceinline__ void tmem_wait64(uint32_t (&a)[64], uint32_t (&b)[64]) {
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 64; i += 8) {
        asm volatile("" : "+r"(a[i]), "+r"(a[i + 1]), "+r"(a[i + 2]), "+r"(a[i + 3]), "+r"(a[i + 4]), "+r"(a[i + 5]),
                          "+r"(a[i + 6]), "+r"(a[i + 7]) :: "memory");
        asm volatile("" : "+r"(b[i]), "+r"(b[i + 1]), "+r"(b[i + 2]), "+r"(b[i + 3]), "+r"(b[i + 4]), "+r"(b[i + 5]),
                          "+r"(b[i + 6]), "+r"(b[i + 7]) :: "memory");
    }
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
                 "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
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
__device__ __forceinline__ void tma_store_2d(const void* tmap, uint32_t smem_src, int c0, int c1) {
    asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];" ::"l"(tmap),
                 "r"(smem_src), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void tma_store_3d(const void* tmap, uint32_t smem_src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(tmap),
                 "r"(smem_src), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// Returns once all but the newest N committed store groups have finished READING shared memory.
template <int N>
__device__ __forceinline__ void tma_wait_read() {
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void tma_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// Packed fp32x2 arithmetic (two IEEE fp32 results per instruction, sm_100).
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2u(uint32_t lo, uint32_t hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "r"(lo), "r"(hi));
    return r;
}
__device__ __forceinline__ void up2f(u64 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 add2(u64 x, u64 y) {
    u64 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(x), "l"(y));
    return r;
}
__device__ __forceinline__ u64 sub2(u64 x, u64 y) {
    u64 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(x), "l"(y));
    return r;
}
__device__ __forceinline__ u64 mul2(u64 x, u64 y) {
    u64 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(x), "l"(y));
    return r;
}
__device__ __forceinline__ u64 fma2(u64 x, u64 y, u64 z) {
    u64 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(x), "l"(y), "l"(z));
    return r;
}

// One 32-byte sector of the side plane, marked evict-last in L2: K3 reads the side plane right after this kernel,
// whose 3.2 GB of plane stores would otherwise push it out (K2-TC -7 us, K3 -3 us per SKA trial).
__device__ __forceinline__ void st_global_256(void* ptr, const uint4 a, const uint4 b) {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    asm volatile("st.global.L2::cache_hint.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8}, %9;" ::"l"(ptr), "r"(a.x),
                 "r"(a.y), "r"(a.z), "r"(a.w), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w), "l"(pol)
                 : "memory");
}

// Powers of 8 consecutive bins of the rows +z and -z of this thread's pair from one group of
// accumulator columns (a = 16 columns of D_R: Ar[0..7] | Ai[0..7]; b = 16 columns of D_I: Br | Bi),
// into this thread's rows (rowp, rowm) of the two staging tiles, 16-byte unit `2 * bg` (fp32) / `bg`
// (bf16) of half `half` of the row; returns the block maxima as the codes of fdas_maxcode.h (upper bounds of
// the values AS STORED).
template <int PLANE16>
__device__ __forceinline__ unsigned group_to_smem(const uint32_t* __restrict__ a, const uint32_t* __restrict__ b,
                                                  unsigned char* tile_p, unsigned char* tile_m, const int rowp,
                                                  const int rowm, const int half, const int bg) {
    // pair_powers (fdas_tc_common.h) for two bins per instruction: the packed fp32x2 forms (FADD2 / FMUL2 /
    // FFMA2) round each half exactly like the scalar ones, at half the issue slots of the drain
    float Pp[8], Pm[8];
#pragma unroll
    for (int e = 0; e < 8; e += 2) {
        const u64 Ar = pk2u(a[e], a[e + 1]), Ai = pk2u(a[8 + e], a[9 + e]);
        const u64 Br = pk2u(b[e], b[e + 1]), Bi = pk2u(b[8 + e], b[9 + e]);
        const u64 rp = add2(Ar, Bi), ip = sub2(Ai, Br), rm = sub2(Ar, Bi), im = add2(Ai, Br);
        const u64 pp = fma2(rp, rp, mul2(ip, ip)), pm = fma2(rm, rm, mul2(im, im));
        up2f(pp, Pp[e], Pp[e + 1]);
        up2f(pm, Pm[e], Pm[e + 1]);
    }
    unsigned mp, mm;
    if (PLANE16) {
        auto pack = [](float lo, float hi) {
            return (unsigned)__bfloat16_as_ushort(__float2bfloat16_rn(lo)) |
                   ((unsigned)__bfloat16_as_ushort(__float2bfloat16_rn(hi)) << 16);
        };
        const uint4 up = make_uint4(pack(Pp[0], Pp[1]), pack(Pp[2], Pp[3]), pack(Pp[4], Pp[5]), pack(Pp[6], Pp[7]));
        const uint4 um = make_uint4(pack(Pm[0], Pm[1]), pack(Pm[2], Pm[3]), pack(Pm[4], Pm[5]), pack(Pm[6], Pm[7]));
        *reinterpret_cast<uint4*>(tile_p + stage_unit_offset(rowp, half, bg, 1)) = up;
        *reinterpret_cast<uint4*>(tile_m + stage_unit_offset(rowm, half, bg, 1)) = um;
        // powers are >= 0: the order of the bf16 bit patterns is the order of the values
        const unsigned xp = __vmaxu2(__vmaxu2(up.x, up.y), __vmaxu2(up.z, up.w));
        const unsigned xm = __vmaxu2(__vmaxu2(um.x, um.y), __vmaxu2(um.z, um.w));
        mp = max_code(__uint_as_float(max(xp & 0xffffu, xp >> 16) << 16));
        mm = max_code(__uint_as_float(max(xm & 0xffffu, xm >> 16) << 16));
    } else {
        // The swizzle phase of a row's chunk, (2 row + half) & 7, takes only 4 values over the 8 rows of a
        // shared-memory store phase, so the lanes with bit 2 set write their two 16-byte units in the
        // opposite order: every store instruction then touches 8 different 16-byte bank groups.
        const bool flip = (threadIdx.x & 4) != 0;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const int u = 2 * bg + (flip ? 1 - c : c);
            const float4 vp = (c == 0) == !flip ? make_float4(Pp[0], Pp[1], Pp[2], Pp[3]) : make_float4(Pp[4], Pp[5], Pp[6], Pp[7]);
            const float4 vm = (c == 0) == !flip ? make_float4(Pm[0], Pm[1], Pm[2], Pm[3]) : make_float4(Pm[4], Pm[5], Pm[6], Pm[7]);
            *reinterpret_cast<float4*>(tile_p + stage_unit_offset(rowp, half, u, 0)) = vp;
            *reinterpret_cast<float4*>(tile_m + stage_unit_offset(rowm, half, u, 0)) = vm;
        }
        const float fp = fmaxf(fmaxf(fmaxf(Pp[0], Pp[1]), fmaxf(Pp[2], Pp[3])), fmaxf(fmaxf(Pp[4], Pp[5]), fmaxf(Pp[6], Pp[7])));
        const float fm = fmaxf(fmaxf(fmaxf(Pm[0], Pm[1]), fmaxf(Pm[2], Pm[3])), fmaxf(fmaxf(Pm[4], Pm[5]), fmaxf(Pm[6], Pm[7])));
        return max_code2(fp, fm);
    }
    return mp | (mm << 16);
}

template <int PLANE16, int NBUF>
__global__ void __launch_bounds__(kThreads, 1)
convolve_tc_kernel(const ConvTcParams p, const __grid_constant__ CUtensorMap pmap,
                   const __grid_constant__ CUtensorMap pmap_tail) {
    extern __shared__ __align__(1024) unsigned char smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nq = (p.npair + 31) >> 5;                   // TMEM lane quarters that hold template pairs
    const Layout L = make_layout(p.kp, 2 * nq, NBUF, PLANE16);
    const uint32_t bar0 = smem_u32(smem + L.bar_off);
    // barriers: hfull[3] | hempty[3] | tfull[4] | tempty[4]; then the TMEM base address slot; at +128 the
    // mailbox barriers mfull[4] | mempty[4] (one pair per lane quarter).
    // tfull / tempty are indexed by the SUB-TILE (one phase per tile: a waiter must see every phase of
    // its barrier); the accumulator stage of sub-tile s is s >> 1 (one stage per epilogue set), so the
    // MMA of sub-tile s waits for the drain of sub-tile s ^ 1.
    auto hfull = [&](int s) { return bar0 + 8u * s; };
    auto hempty = [&](int s) { return bar0 + 8u * (kHStages + s); };
    auto tfull = [&](int s) { return bar0 + 8u * (2 * kHStages + s); };
    auto tempty = [&](int s) { return bar0 + 8u * (2 * kHStages + kSubTiles + s); };
    auto mfull = [&](int q) { return bar0 + 128u + 8u * q; };
    auto mempty = [&](int q) { return bar0 + 160u + 8u * q; };
    volatile uint32_t* tmem_slot =
        reinterpret_cast<volatile uint32_t*>(smem + L.bar_off + 8 * (2 * kHStages + 2 * kSubTiles));

    // ---- one-time setup: barriers, TMEM, the bank images
    if (warp == kMmaWarp) {
        if (lane == 0) {
            for (int s = 0; s < kHStages; ++s) {
                mbar_init(hfull(s), 1);
                mbar_init(hempty(s), 1);
            }
            for (int s = 0; s < kSubTiles; ++s) {
                mbar_init(tfull(s), 1);
                mbar_init(tempty(s), 4);          // the four warps of the set that drains the sub-tile
            }
            for (int q = 0; q < 4; ++q) {
                mbar_init(mfull(q), 1);
                mbar_init(mempty(q), 1);
            }
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncwarp();
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
    const int kw = p.kp >> 1;                             // TMEM columns of one bank image
    if (warp < 4) {
        // lane (32 warp + lane) <- row (pair) of both images: kp/2 words of two bf16 taps each
        const uint32_t lane_addr = tmem_base + ((uint32_t)(32 * warp) << 16) + kBankCol0;
        for (int part = 0; part < 2; ++part) {
            const uint4* src = reinterpret_cast<const uint4*>(p.bimg + ((size_t)part * 128 + tid) * kw);
            for (int c8 = 0; c8 < kw / 8; ++c8) {
                const uint4 lo = __ldg(src + 2 * c8), hi = __ldg(src + 2 * c8 + 1);
                const uint32_t v[8] = {lo.x, lo.y, lo.z, lo.w, hi.x, hi.y, hi.z, hi.w};
                tmem_st8(lane_addr + part * kw + c8 * 8, v);
            }
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    const int64_t ntiles = p.nbins / kTileR;
    const int ksteps = p.kp >> 4;
    const int npair = p.npair;                            // pairs of this launch: lanes 0 .. npair - 1
    const int jplus0 = p.nz - p.npair_total + p.pair0;    // row of lane 0's +z member
    const int jminus0 = p.npair_total - 1 - p.pair0;      // row of lane 0's -z member

    if (warp == kProducerWarp) {
        // ===== producer: the tile's spectrum slice -> interleaved sliding-window rows; z = 0 row
        unsigned short* sre = reinterpret_cast<unsigned short*>(smem + L.st_off);
        unsigned short* sim = reinterpret_cast<unsigned short*>(smem + L.st_off + L.st_part);
        const int nrows = window_rows(p.kp), nsrc = nrows + 24;
        const bool zero_row = (p.nz & 1) != 0 && p.pair0 == 0;
        const int mid = p.npair_total;                    // the z = 0 row of an odd bank
        // the slice s[i] = w[128 tile - h + i], i < nsrc (<= 384), as 16-byte loads of 4 bins per lane; the
        // next tile's loads are issued before this tile's window is built, so their latency is hidden
        uint4 v[3];
        auto load_slice = [&](int64_t tile) {
            const int64_t base = tile * kTileR - p.h;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int e = 4 * (lane + 32 * k);
                const int64_t idx = base + e;     // a multiple of 4, like nbins: 4 bins inside or 4 outside
                v[k] = (e < nsrc && idx >= 0 && idx < p.nbins) ? __ldg(reinterpret_cast<const uint4*>(p.spec + idx))
                                                               : make_uint4(0u, 0u, 0u, 0u);
            }
        };
        if ((int64_t)blockIdx.x < ntiles) load_slice(blockIdx.x);
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            const int hs = it % kHStages;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int e = 4 * (lane + 32 * k);
                if (e < nsrc) {
                    *reinterpret_cast<uint2*>(sre + e) =
                        make_uint2(__byte_perm(v[k].x, v[k].y, 0x5410), __byte_perm(v[k].z, v[k].w, 0x5410));
                    *reinterpret_cast<uint2*>(sim + e) =
                        make_uint2(__byte_perm(v[k].x, v[k].y, 0x7632), __byte_perm(v[k].z, v[k].w, 0x7632));
                }
            }
            __syncwarp();
            if (tile + gridDim.x < ntiles) load_slice(tile + gridDim.x);
            mbar_wait(hempty(hs), ((it / kHStages) & 1) ^ 1);
            unsigned char* hst = smem + L.h_off + hs * L.h_stage;
            for (int rho = lane; rho < nrows; rho += 32) {
#pragma unroll
                for (int part = 0; part < 2; ++part) {
                    const uint32_t* w32 = reinterpret_cast<const uint32_t*>(part ? sim : sre) + (rho >> 1);
                    *reinterpret_cast<uint4*>(hst + window_row_offset(rho, part)) = window_row(w32, rho);
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(hfull(hs));
            if (zero_row) {
                // T_0 = delta: the row is |w[r]|^2 of the stored (bf16) spectrum; 4 bins per lane
                float P[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float re = __uint_as_float((unsigned)sre[p.h + 4 * lane + e] << 16);
                    const float im = __uint_as_float((unsigned)sim[p.h + 4 * lane + e] << 16);
                    P[e] = fmaf(re, re, im * im);
                }
                const int64_t r = tile * kTileR + 4 * lane;
                unsigned m;
                if (PLANE16) {
                    unsigned short b[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) b[e] = __bfloat16_as_ushort(__float2bfloat16_rn(P[e]));
                    __stcs(reinterpret_cast<uint2*>(reinterpret_cast<unsigned short*>(p.plane) + (int64_t)mid * p.pitch + r),
                           make_uint2((unsigned)b[0] | ((unsigned)b[1] << 16), (unsigned)b[2] | ((unsigned)b[3] << 16)));
                    m = max_code(__uint_as_float(max(max((unsigned)b[0], (unsigned)b[1]), max((unsigned)b[2], (unsigned)b[3])) << 16));
                } else {
                    __stcs(reinterpret_cast<float4*>(reinterpret_cast<float*>(p.plane) + (int64_t)mid * p.pitch + r),
                           make_float4(P[0], P[1], P[2], P[3]));
                    m = max_code(fmaxf(fmaxf(P[0], P[1]), fmaxf(P[2], P[3])));
                }
                m = max(m, __shfl_xor_sync(0xffffffffu, m, 1));
                if ((lane & 1) == 0) p.maxplane[(int64_t)mid * p.mpitch + (r >> 3)] = (unsigned short)m;
            }
            __syncwarp();      // the slice staging is rewritten by the next iteration
        }
    } else if (warp == kMmaWarp) {
        // ===== MMA issuer: the warp stays converged (every lane waits on the barriers and forms the
        // descriptors in uniform registers); one elected lane issues the tensor-core instructions
        const uint32_t idesc = instr_desc(2 * kSubR);
        const uint32_t a_re = tmem_base + kBankCol0, a_im = a_re + (uint32_t)kw;
        int it = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            const int hs = it % kHStages;
            mbar_wait(hfull(hs), (it / kHStages) & 1);
            tc_fence_after();
            const uint32_t hbase = smem_u32(smem + L.h_off + hs * L.h_stage);
#pragma unroll
            for (int pos = 0; pos < kSubTiles; ++pos) {
                // issue order s = 0, 2, 1, 3: the two epilogue sets (sub-tiles {0, 1} and {2, 3}) take turns,
                // each with its own accumulator stage, so one set computes while the other one loads
                const int s = 2 * (pos & 1) + (pos >> 1);
                const uint32_t st = pos & 1u;
                // the stage was last filled for this set's previous sub-tile: s - 1 of this tile or s + 1 of
                // the previous one
                if ((s & 1) || it > 0) {
                    mbar_wait(tempty(s ^ 1), (uint32_t)((s & 1) ? it : it - 1) & 1u);
                    tc_fence_after();
                }
                const uint32_t d_r = tmem_base + st * kAccCols, d_i = d_r + 2 * kSubR;
                const uint64_t bd0 = smem_desc(hbase + window_desc_offset(s, 0), kWinLbo, kWinSbo);
                if (elect_one()) {
#pragma unroll 3
                    for (int ks = 0; ks < ksteps; ++ks) {
                        const uint64_t bd = bd0 + (uint64_t)(ks * (512 >> 4));   // one K step = 512 bytes further
                        tc_mma_ts(d_r, a_re + 8u * ks, bd, idesc, ks > 0);
                        tc_mma_ts(d_i, a_im + 8u * ks, bd, idesc, ks > 0);
                    }
                    tc_commit(tfull(s));
                }
                __syncwarp();
            }
            if (elect_one()) tc_commit(hempty(hs));
            __syncwarp();
        }
    } else {
        // ===== epilogue warps: lane quarter q = 32 template pairs; set 0 drains sub-tiles 0, 1 and
        // set 1 sub-tiles 2, 3 of every tile, each set through its own accumulator stage
        const int q = warp & 3, set = warp >> 2;
        const bool active = q < nq;
        const int slot = set * nq + q;                    // staging buffers of the active warps
        unsigned char* const stage0 = smem + L.ep_off + slot * L.ep_warp;
        const uint32_t lane_base = tmem_base + ((uint32_t)(32 * q) << 16);
        // this quarter's nreal pairs: rows row_p .. row_p + nreal - 1 of the plane (+z, ascending with the
        // lane) and row_m .. row_m + nreal - 1 (-z, descending with the lane: the tile is stored reversed).
        // A ragged last quarter (nreal < 32) goes out through a tensor map whose boxes have nreal rows (a
        // box that starts at a negative row is an illegal instruction); its unused lanes write to tile rows
        // >= nreal, which no box reads.
        const int nreal = min(32, npair - 32 * q);
        const int row_p = jplus0 + 32 * q;
        const int row_m = jminus0 - 32 * q - nreal + 1;
        const int rowm = lane < nreal ? nreal - 1 - lane : lane;
        const CUtensorMap* const pm = nreal == 32 ? &pmap : &pmap_tail;
        constexpr int kTileBytes = 32 * 2 * kSubR * (PLANE16 ? 2 : 4);   // 32 rows x this warp's 64 bins
        unsigned short* const mrow_p = p.maxplane + (int64_t)(row_p + lane) * p.mpitch + 8 * set;
        unsigned short* const mrow_m = p.maxplane + (int64_t)(row_m + rowm) * p.mpitch + 8 * set;
        int tile_iter = 0;
        for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++tile_iter) {
            unsigned mxp[4], mxm[4];                      // block maxima of 8 blocks: rows +z, -z
            unsigned char* const buf = stage0 + (tile_iter % NBUF) * (2 * kTileBytes);
#pragma unroll
            for (int ss = 0; ss < 2; ++ss) {
                const int s = 2 * set + ss;
                const uint32_t st = (uint32_t)set;
                mbar_wait(tfull(s), (uint32_t)tile_iter & 1u);
                if (!active) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty(s));
                    continue;
                }
                tc_fence_after();
                const uint32_t tb = lane_base + st * kAccCols;
                // the whole stage (2 x 64 columns of this lane) goes to registers at once and the stage is
                // handed back to the MMA warp before any arithmetic (eight 16-column loads in flight, then
                // one wait: the .x16 shape streams fastest, profiles/r02)
                uint32_t ra[64], rb[64];
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                    tmem_ld16(tb + 16 * g, *reinterpret_cast<uint32_t(*)[16]>(ra + 16 * g));
                    tmem_ld16(tb + 2 * kSubR + 16 * g, *reinterpret_cast<uint32_t(*)[16]>(rb + 16 * g));
                }
                if (ss == 0) {
                    if (lane == 0) tma_wait_read<NBUF - 1>();   // the group that read this buffer is done
                    __syncwarp();
                }
                tmem_wait64(ra, rb);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty(s));
#pragma unroll
                for (int bg = 0; bg < kSubR / 8; bg += 2) {
                    const unsigned m0 = group_to_smem<PLANE16>(ra + 16 * bg, rb + 16 * bg, buf, buf + kTileBytes, lane, rowm, ss, bg);
                    const unsigned m1 = group_to_smem<PLANE16>(ra + 16 * bg + 16, rb + 16 * bg + 16, buf, buf + kTileBytes, lane, rowm, ss, bg + 1);
                    mxp[2 * ss + (bg >> 1)] = (m0 & 0xffffu) | (m1 << 16);
                    mxm[2 * ss + (bg >> 1)] = (m0 >> 16) | (m1 & 0xffff0000u);
                }
            }
            if (!active) continue;
            // this warp's 64 bins x 32 rows x {+z, -z}: one tensor store each (256-byte rows: a store of
            // 128-byte rows runs at 3/4 of the rate, profiles/r02), and the 8 block maxima of the thread's
            // two rows as one 16-byte store each (the other half of the 32-byte sector comes from the warp
            // that drains the other half of the tile)
            fence_async_smem();
            __syncwarp();
            if (lane == 0) {
                const int c0 = (int)(tile * kTileR) + 2 * kSubR * set;
                if (PLANE16) {
                    tma_store_2d(pm, smem_u32(buf), c0, row_p);
                    tma_store_2d(pm, smem_u32(buf + kTileBytes), c0, row_m);
                } else {
                    tma_store_3d(pm, smem_u32(buf), 0, c0 / kSubR, row_p);
                    tma_store_3d(pm, smem_u32(buf + kTileBytes), 0, c0 / kSubR, row_m);
                }
                tma_commit();
            }
            if constexpr (PLANE16) {
                // (with a bf16 plane the two sets store their halves themselves: measured faster, profiles/r02b)
                if (lane < nreal) {
                    *reinterpret_cast<uint4*>(mrow_p + tile * (kTileR / 8)) = make_uint4(mxp[0], mxp[1], mxp[2], mxp[3]);
                    *reinterpret_cast<uint4*>(mrow_m + tile * (kTileR / 8)) = make_uint4(mxm[0], mxm[1], mxm[2], mxm[3]);
                }
            } else {
                // the block maxima of a row and tile leave as ONE 32-byte store (a whole sector): set 0 hands its half
                // (blocks 0..7) to the warp of set 1 with the same lane quarter through a 1 KB mailbox.  Written as
                // two 16-byte halves by the two sets, the half-written sectors wait in L2 for their other half, and
                // the kernel's time depends on how far the sets drift apart (0.650 -> 0.632 ms per SKA launch)
                uint4* const mbox = reinterpret_cast<uint4*>(smem + L.mb_off) + (q * 32 + lane) * 2;
                if (set == 0) {
                    mbar_wait(mempty(q), ((uint32_t)tile_iter & 1u) ^ 1u);
                    mbox[0] = make_uint4(mxp[0], mxp[1], mxp[2], mxp[3]);
                    mbox[1] = make_uint4(mxm[0], mxm[1], mxm[2], mxm[3]);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(mfull(q));
                } else {
                    mbar_wait(mfull(q), (uint32_t)tile_iter & 1u);
                    const uint4 ap = mbox[0], am = mbox[1];
                    __syncwarp();
                    if (lane == 0) mbar_arrive(mempty(q));
                    if (lane < nreal) {
                        st_global_256(mrow_p - 8 + tile * (kTileR / 8), ap, make_uint4(mxp[0], mxp[1], mxp[2], mxp[3]));
                        st_global_256(mrow_m - 8 + tile * (kTileR / 8), am, make_uint4(mxm[0], mxm[1], mxm[2], mxm[3]));
                    }
                }
            }
        }
        if (lane == 0) tma_wait_all();
    }

    // ---- teardown
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (warp == kMmaWarp) {
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u)
                     : "memory");
    }
}

}  // namespace tc

// Staging buffers per epilogue warp: two (a tile's stores drain while the next tile is computed) when
// the CTA's shared memory holds them -- up to 96 pairs with templates of up to 145 taps -- else one.
static int tc_nbuf(int kp, int npair, int plane16) {
    const int nq = (npair + 31) >> 5;
    return tc::make_layout(kp, 2 * nq, 2, plane16).total <= 227 * 1024 ? 2 : 1;
}

int convolve_tc_smem_bytes(int kp, int npair, int plane16) {
    const int nq = (npair + 31) >> 5;
    return tc::make_layout(kp, 2 * nq, tc_nbuf(kp, npair, plane16), plane16).total;
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

// The plane as the tensor a warp's stores address.  bf16 plane: 2-D [rows][cols], boxes of 64 bins
// (128 bytes, SWIZZLE_128B) x box_rows.  fp32 plane: 3-D [rows][cols / 32][32] so that the innermost
// box dimension stays within the 128-byte swizzle span while a box still covers 256 contiguous bytes of
// every row (two chunks of 32 bins, adjacent in shared and in global memory, which the TMA unit merges).
static cudaError_t make_plane_map(void* base, int plane16, int64_t cols, int64_t rows, int64_t pitch, int box_rows,
                                  CUtensorMap* map) {
    EncodeTiledFn enc = encode_tiled_fn();
    if (!enc) return cudaErrorNotSupported;
    CUresult r;
    if (plane16) {
        const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
        const cuuint64_t strides[1] = {(cuuint64_t)pitch * 2};
        const cuuint32_t box[2] = {(cuuint32_t)(2 * tc::kSubR), (cuuint32_t)box_rows};
        const cuuint32_t estr[2] = {1u, 1u};
        r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
        const cuuint64_t dims[3] = {(cuuint64_t)tc::kSubR, (cuuint64_t)(cols / tc::kSubR), (cuuint64_t)rows};
        const cuuint64_t strides[2] = {(cuuint64_t)tc::kSubR * 4, (cuuint64_t)pitch * 4};
        const cuuint32_t box[3] = {(cuuint32_t)tc::kSubR, 2u, (cuuint32_t)box_rows};
        const cuuint32_t estr[3] = {1u, 1u, 1u};
        r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// The tensor maps depend only on the output pointer and the plane geometry: they are encoded once per
// plane buffer and kept in the plan's cache.  Keying an entry by the pointer alone is safe because the
// cache belongs to ONE plan and everything else a map encodes (element type, nbins, nz, pitch, box rows) is
// a constant of that plan: a buffer that is freed and handed out again at the same address gets the same
// map, and a map holds no reference to the memory behind it.
static cudaError_t get_maps(TcMapCache* cache, int plane16, const ConvTcParams& p, const TcMapCache::Entry** out) {
    for (int i = 0; i < TcMapCache::kEntries; ++i) {
        const TcMapCache::Entry& e = cache->e[i];
        if (e.valid && e.plane == p.plane) {
            *out = &e;
            return cudaSuccess;
        }
    }
    TcMapCache::Entry& e = cache->e[cache->next];
    cache->next = (cache->next + 1) % TcMapCache::kEntries;
    e.valid = false;
    // rows of the boxes of a ragged last lane quarter (launches of a split bank are multiples of 32 pairs
    // except the last, so one tail size serves them all)
    const int tail = (p.npair_total & 31) ? (p.npair_total & 31) : 32;
    cudaError_t err = make_plane_map(p.plane, plane16, p.nbins, p.nz, p.pitch, 32, reinterpret_cast<CUtensorMap*>(e.pmap));
    if (err == cudaSuccess)
        err = make_plane_map(p.plane, plane16, p.nbins, p.nz, p.pitch, tail, reinterpret_cast<CUtensorMap*>(e.pmap_tail));
    if (err != cudaSuccess) return err;
    e.plane = p.plane;
    e.valid = true;
    *out = &e;
    return cudaSuccess;
}

template <int PLANE16, int NBUF>
static cudaError_t launch_tc(const ConvTcParams& p, const TcMapCache::Entry& m, int nsm, cudaStream_t st) {
    const int smem = convolve_tc_smem_bytes(p.kp, p.npair, PLANE16);
    auto kern = tc::convolve_tc_kernel<PLANE16, NBUF>;
    static PerDeviceOnce attr;          // per template instance, per device
    const cudaError_t ea = attr.run([&] {
        return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    });
    if (ea != cudaSuccess) return ea;
    const int64_t ntiles = p.nbins / tc::kTileR;
    const unsigned grid = (unsigned)(ntiles < nsm ? ntiles : nsm);
    // at least half of the SM's shared memory, so that two CTAs (2 x 512 TMEM columns) never share an SM
    kern<<<grid, tc::kThreads, smem < 120 * 1024 ? 120 * 1024 : smem, st>>>(
        p, *reinterpret_cast<const CUtensorMap*>(m.pmap), *reinterpret_cast<const CUtensorMap*>(m.pmap_tail));
    return cudaGetLastError();
}

cudaError_t launch_convolve_tc(int plane16, const ConvTcParams& p, TcMapCache* cache, int nsm, cudaStream_t st) {
    if (p.nbins % tc::kTileR != 0 || p.kp % 16 != 0 || p.npair < 1 || p.npair > 128 || p.pair0 < 0 ||
        p.pair0 + p.npair > p.npair_total || 2 * p.npair_total > p.nz ||
        tc::kBankCol0 + p.kp > 512 || (reinterpret_cast<uintptr_t>(p.plane) & 15u) ||
        (reinterpret_cast<uintptr_t>(p.spec) & 15u) ||
        ((p.pitch * (plane16 ? 2 : 4)) & 15) || ((p.mpitch * 2) & 31) ||          // 32-byte block-max stores
        (reinterpret_cast<uintptr_t>(p.maxplane) & 31u))
        return cudaErrorInvalidValue;
    const TcMapCache::Entry* m = nullptr;
    const cudaError_t e = get_maps(cache, plane16, p, &m);
    if (e != cudaSuccess) return e;
    if (tc_nbuf(p.kp, p.npair, plane16) == 2) return plane16 ? launch_tc<1, 2>(p, *m, nsm, st) : launch_tc<0, 2>(p, *m, nsm, st);
    return plane16 ? launch_tc<1, 1>(p, *m, nsm, st) : launch_tc<0, 1>(p, *m, nsm, st);
}

}  // namespace fdas
