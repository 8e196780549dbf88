// fdas_tc_common.h -- index arithmetic of K2-TC shared by the kernel (fdas_convolve_tc.cu) and the
// test-only host emulator (fdas_emu.cu): shared-memory carve-up, UMMA descriptor encoding, the
// sliding-window row builder and the pair-power formula.  Pure arithmetic, __host__ __device__.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace fdas {
namespace tc {

#ifndef FDAS_TC_WGS
#define FDAS_TC_WGS 3
#endif
constexpr int kWarpGroups = FDAS_TC_WGS;               // epilogue warpgroups (4 warps = the tile's 128 bins)
constexpr int kThreads = 64 + 128 * kWarpGroups;      // warp 0 producer, warp 1 MMA issuer, then the epilogue warps
constexpr int kHStages = 3;     // sliding-window (A operand) stages
constexpr int kTileR = 128;     // Fourier bins per tile = MMA M = TMEM lanes
constexpr int kEpiWarps = 4 * kWarpGroups;
constexpr int kStageTileBytes = 16 * 128 * 4;   // one staged chunk: 16 plane rows x 128 bins (fp32)
constexpr int kStageBufBytes = kStageTileBytes + 16 * 16 * 2;   // + its [16][16] bf16 block-max tile
constexpr int kStageBufs = 4;                   // staged chunks in flight per warpgroup

// K-major, no-swizzle shared-memory matrix descriptor: start address, LBO (between the two 8-element
// K halves of one MMA), SBO (between 8-row groups), all in 16-byte units; version 1 (sm_100).
// Element (row i, k) of the operand is read from start + (i%8)*16 + (i/8)*SBO + (k/8)*LBO + (k%8)*2.
__host__ __device__ inline uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46);
}
// Instruction descriptor: D fp32, A/B bf16, both K-major, M = 128, N = n.
__host__ __device__ constexpr uint32_t instr_desc(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}

// Shared-memory carve-up (dynamic, 128-byte aligned): B image | H stages (re, im) | slice staging |
// epilogue tiles | barriers.
struct Layout {
    int b_off, h_off, h_part, h_stage, st_off, st_part, sc_off, bar_off, total;
};
__host__ __device__ inline Layout make_layout(int bimg_bytes, int kp) {
    Layout l;
    l.b_off = 0;
    l.h_off = (bimg_bytes + 127) & ~127;
    l.h_part = ((kp + 120) * 16 + 127) & ~127;      // kp + 120 window rows of 16 bytes
    l.h_stage = 2 * l.h_part;
    l.st_off = l.h_off + kHStages * l.h_stage;
    l.st_part = ((kp + 136) * 2 + 127) & ~127;      // kp + 130 bf16 of the slice (incl. read slack)
    l.sc_off = l.st_off + 2 * l.st_part;
    l.bar_off = l.sc_off + (kEpiWarps / 4) * kStageBufs * kStageBufBytes;
    l.total = l.bar_off + 128;
    return l;
}

// Row rho of the sliding-window matrix: the 8 bf16 s[rho..rho+7], from the 32-bit view of s at
// word rho/2 (five words; the odd rows are shifted down by 16 bits).
__host__ __device__ inline uint4 window_row(const uint32_t* w32, int rho) {
    const uint32_t w0 = w32[0], w1 = w32[1], w2 = w32[2], w3 = w32[3], w4 = w32[4];
    if (rho & 1)
        return make_uint4((w0 >> 16) | (w1 << 16), (w1 >> 16) | (w2 << 16), (w2 >> 16) | (w3 << 16),
                          (w3 >> 16) | (w4 << 16));
    return make_uint4(w0, w1, w2, w3);
}

// Powers of the rows +z and -z from A~ = w (*) Re T_z = Ar + i Ai and B~ = w (*) Im T_z = Br + i Bi:
// y_{+z} = A~ - i B~ = (Ar + Bi) + i (Ai - Br),  y_{-z} = A~ + i B~ = (Ar - Bi) + i (Ai + Br).
__host__ __device__ inline void pair_powers(float Ar, float Br, float Ai, float Bi, float* Pp, float* Pm) {
    const float rp = Ar + Bi, ip = Ai - Br, rm = Ar - Bi, im = Ai + Br;
    *Pp = fmaf(rp, rp, ip * ip);
    *Pm = fmaf(rm, rm, im * im);
}

}  // namespace tc
}  // namespace fdas
