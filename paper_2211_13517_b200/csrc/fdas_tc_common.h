// fdas_tc_common.h -- index arithmetic of K2-TC shared by the kernel (fdas_convolve_tc.cu) and the
// test-only host emulator (tests/emu/fdas_emu.cu): shared-memory carve-up, UMMA descriptor encodings,
// the sliding-window row builder, the swizzled staging addresses and the pair-power formula.
// Pure arithmetic, __host__ __device__.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace fdas {
namespace tc {

constexpr int kTileR = 128;     // Fourier bins per tile (one sliding-window stage)
constexpr int kSubR = 32;       // bins per accumulator stage (MMA N = 2 * kSubR: re | im window rows)
constexpr int kSubTiles = kTileR / kSubR;
constexpr int kHStages = 3;     // sliding-window (B operand) stages
constexpr int kAccStages = 2;   // TMEM accumulator stages
constexpr int kAccCols = 4 * kSubR;          // TMEM columns of one stage: D_R (2 kSubR) | D_I (2 kSubR)
constexpr int kBankCol0 = kAccStages * kAccCols;   // first TMEM column of the bank images
constexpr int kEpiWarps = 8;    // warps 0..3: sub-tiles 0,1 of every tile; warps 4..7: sub-tiles 2,3
constexpr int kProducerWarp = 8, kMmaWarp = 9;
constexpr int kThreads = 32 * (kEpiWarps + 2);

// K-major, no-swizzle shared-memory matrix descriptor: start address, LBO (between the two 8-element
// K halves of one MMA), SBO (between 8-row groups), all in 16-byte units; version 1 (sm_100).
// Element (row n, k) of the operand is read from start + (n%8)*16 + (n/8)*SBO + (k/8)*LBO + (k%8)*2.
__host__ __device__ inline uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    return (uint64_t)((addr & 0x3ffffu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46);
}
// Instruction descriptor: D fp32, A/B bf16, both K-major, M = 128, N = n.
__host__ __device__ constexpr uint32_t instr_desc(int n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}

// ---- the sliding-window operand.  Row rho of a part (Re w or Im w) is the 16 bytes
// s[rho .. rho+7] of the tile's spectrum slice s[i] = w[128 tile - h + i].  Groups of 8 rows of the
// two parts alternate in shared memory: group G of part p sits at ((2 G + p) * 128) bytes, so that a
// descriptor with SBO = 128 B walks (re, im, re, im, ...) row groups along N and LBO = 256 B steps one
// group (= 8 taps) along K:  operand row n = 16 gb + 8 p + e  <->  bin 8 gb + e of part p, and
// B[n][k] = s_p[8 gb + e + k].
__host__ __device__ inline int window_rows(int kp) { return kTileR + kp - 8; }        // rho = 0 .. this - 1
__host__ __device__ inline int window_row_offset(int rho, int part) {
    return ((2 * (rho >> 3) + part) << 7) + ((rho & 7) << 4);
}
constexpr uint32_t kWinSbo = 128, kWinLbo = 256;
__host__ __device__ inline uint32_t window_desc_offset(int sub, int kstep) {   // start of (sub-tile, K step)
    return (uint32_t)sub * (kSubR / 8) * 256u + (uint32_t)kstep * 512u;
}
// Row rho of the window: the 8 bf16 s[rho..rho+7], from the 32-bit view of s at word rho/2 (five
// words; the odd rows are shifted down by 16 bits).
__host__ __device__ inline uint4 window_row(const uint32_t* w32, int rho) {
    const uint32_t w0 = w32[0], w1 = w32[1], w2 = w32[2], w3 = w32[3], w4 = w32[4];
    if (rho & 1)
        return make_uint4((w0 >> 16) | (w1 << 16), (w1 >> 16) | (w2 << 16), (w2 >> 16) | (w3 << 16),
                          (w3 >> 16) | (w4 << 16));
    return make_uint4(w0, w1, w2, w3);
}

// ---- epilogue staging tiles: an epilogue warp owns 32 plane rows x 64 bins (two sub-tiles) of a tile.
// fp32 plane: row r is two 128-byte chunks (sub-tile `half`), chunk index rho = 2 r + half, and the
// 16-byte unit u of a chunk sits at u ^ (rho & 7) -- the image a 3-D TMA tensor store with
// CU_TENSOR_MAP_SWIZZLE_128B and a box of (32 bins, 2 chunks, 32 rows) reads.  bf16 plane: row r is one
// 128-byte chunk (8 units: 4 per sub-tile), unit (4 half + u) ^ (r & 7): a 2-D box of 64 bins x 32 rows.
__host__ __device__ inline int stage_unit_offset(int row, int half, int unit, int plane16) {
    if (plane16) return row * 128 + (((4 * half + unit) ^ (row & 7)) << 4);
    const int rho = 2 * row + half;
    return rho * 128 + ((unit ^ (rho & 7)) << 4);
}
// one staging buffer of an epilogue warp: the +z tile, the -z tile (32 rows x 64 bins each)
__host__ __device__ inline int stage_buf_bytes(int plane16) { return 2 * 32 * 2 * kSubR * (plane16 ? 2 : 4); }

// Shared-memory carve-up (dynamic, 1024-byte aligned): window stages | spectrum-slice staging |
// per-warp epilogue buffers (nbuf staging buffers) | barriers (256 B) | block-max mailbox (1 KB per lane quarter).
struct Layout {
    int h_off, h_stage, st_off, st_part, ep_off, ep_warp, bar_off, mb_off, total;
};
__host__ __device__ inline Layout make_layout(int kp, int nactive_warps, int nbuf, int plane16) {
    Layout l;
    l.h_off = 0;
    l.h_stage = (((window_rows(kp) + 7) / 8) * 256 + 1023) & ~1023;
    l.st_off = l.h_off + kHStages * l.h_stage;
    l.st_part = ((window_rows(kp) + 24) * 2 + 127) & ~127;      // slice of kp + 127 bf16 (+ read slack)
    l.ep_off = (l.st_off + 2 * l.st_part + 1023) & ~1023;
    l.ep_warp = nbuf * stage_buf_bytes(plane16);
    l.bar_off = l.ep_off + nactive_warps * l.ep_warp;
    l.mb_off = l.bar_off + 256;                                  // mailbox: 1 KB per active lane quarter
    l.total = l.mb_off + (nactive_warps / 2) * 1024;
    return l;
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
