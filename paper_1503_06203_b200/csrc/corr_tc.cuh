// corr_tc.cuh -- steps S1-S5 of the hot path for large N: TMA fetch, nibble unpack to int8
// operand planes in shared memory, triangular persistent tile schedule, tcgen05 int8 MMA with
// int32 accumulators in TMEM, triangle-scatter epilogue.
//
// What is computed (Eq. 1, summed over time PAPER.md:48, upper triangle
// PAPER.md:50): for one channel f, one 128x128 tile (x-block bx <= y-block by) and one T-slice,
//      Re A[x][y] = sum_t  Xr[x]Xr[y] + Xi[x]Xi[y]
//      Im A[x][y] = sum_t  Xi[x]Xr[y] - Xr[x]Xi[y]
// as a real int8 contraction with K = 2T (the [Re,Im] stack of x against the stack of y):
// with operand planes  Ar = 16*Xr[x-block], Ai = 16*Xi[x-block], Br = 16*Xr[y-block],
// Bi = 16*Xi[y-block]  (int8, exact: 16*v for v in [-8,7] is in [-128,112]) two MMAs per 32
// time samples accumulate into three 128-column int32 accumulators held in TMEM:
//      D[  0..255] += Ai * [Br;Bi]^T     -> cols   0..127: IR = sum Xi[x]Xr[y],  128..255: II
//      D[128..383] += Ar * [Br;Bi]^T     -> cols 128..255: += RR,               256..383: RI
// so cols 128..255 hold 256*Re and (cols 0..127) - (cols 256..383) = 256*Im.  The epilogue shifts
// right by 8 (exact: every product is a multiple of 256).  No negated operand plane is needed,
// which matters because -16*(-8) = +128 does not fit int8.
//
// Why x16: the packed byte is ((Re+8)<<4)|(Im+8).  Flipping the top bit of a
// stored nibble turns excess-8 into two's complement, so
//      16*Re as int8 = (w ^ 0x80) & 0xF0            (1 LOP3 per 4 samples)
//      16*Im as int8 = ((w << 4) ^ 0x80) & 0xF0     (1 shift + 1 LOP3 per 4 samples)
// Headroom: |sum| <= 2*128*128*T_slice < 2^31 needs T_slice <= 65535; slices are <= 32768.
//
// Layout: the stream is [T][F][N] with the N inputs contiguous, i.e. the operands arrive
// "MN-major" (K = time is the strided axis).  kind::i8 supports MN-major operands, so the TMA box
// [ST t][128 n] lands 128-B swizzled and the unpacked planes keep the SAME physical offsets:
// the unpack is a 16-byte load, 3 logic ops per word and two 16-byte stores at the same offset,
// with no transpose and no bank conflicts.
//
// Warp roles (448 threads, 1 CTA per SM, persistent over work units):
//   warp 0       TMA producer (packed bytes -> pk ring)
//   warp 1       TMEM owner + MMA issuer (one elected thread)
//   warps 2-9    unpack (pk ring -> operand-plane ring)
//   warps 10-13  epilogue (TMEM -> registers -> smem transpose -> vis)
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode, baseline_index
#include "corr_ptx.cuh"

namespace corr {

constexpr int TC_BLK = 128;            // tile edge (inputs)
constexpr int TC_ST = 64;              // time samples per pipeline stage
constexpr int TC_PK_STAGES = 6;        // packed-byte ring depth (covers TMA latency)
constexpr int TC_PL_STAGES = 3;        // operand-plane ring depth
constexpr int TC_UNPACK_WARPS = 8;
constexpr int TC_UNPACK_THREADS = 32 * TC_UNPACK_WARPS;
constexpr int TC_EPI_WARP0 = 2 + TC_UNPACK_WARPS;  // first epilogue warp
constexpr int TC_THREADS = 32 * (TC_EPI_WARP0 + 4);
constexpr int TC_PLANE = TC_ST * TC_BLK;            // bytes of one operand plane per stage
constexpr int TC_PK_BYTES = 2 * TC_PLANE;           // X and Y packed blocks
constexpr int TC_PL_BYTES = 4 * TC_PLANE;           // Ar, Ai, Br, Bi
constexpr int TC_EPI_PITCH = 16 * 8 + 8;            // bytes per staged row (16 baselines + pad)
constexpr int TC_EPI_BYTES = 4 * 32 * TC_EPI_PITCH; // 4 warps x 32 rows
constexpr int TC_SMEM_BYTES = 1024 /*align slack*/ + TC_PK_STAGES * TC_PK_BYTES +
                              TC_PL_STAGES * TC_PL_BYTES + TC_EPI_BYTES + 256 /*barriers*/;
constexpr int TC_MAX_SLICE = 32768;

struct TcParams {
    int N, F, T;
    int tiles_per_f;   // tiles on or above the diagonal, per channel
    int slices;        // T-slices per tile
    int t_per_slice;   // multiple of TC_ST
    int num_units;     // F * tiles_per_f * slices
    int out_mode;      // OutMode
    int sub;           // 128, or 64: the tile holds two whole channels of 64 inputs (N = 128, F = channels / 2); only the
                       // two diagonal 64-blocks are written, as channels 2f and 2f + 1
    int n_out;         // inputs per channel in the layout of vis
    int win_n;         // corr_tcd_kernel<false>, > 0: the unpadded stream of win_n inputs per channel (win_n % 16 != 0) read through
                       // windows of 128 bytes that start on 16-byte boundaries; channel f is rows / columns o .. o + win_n - 1 of
                       // its tile, o = (f * win_n) % 16
    int win_c;         // ... whole channels per window ((128 - 15) / win_n): tile g holds channels g win_c .. g win_c + win_c - 1
    int f_out;         // corr_tcd_kernel, sub == 64 or windows: channels in vis (the last tile holds one channel when this is odd)
    int groups_per_f;  // corr_tcd_kernel, slices == 0: groups of 256 samples per channel, dealt to the CTAs in equal shares
    const ushort2 *tiles;
    int32_t *vis;
};

__global__ void __launch_bounds__(TC_THREADS, 1)
corr_tc_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    extern __shared__ uint8_t smem_raw[];
    // 128-B swizzle patterns are functions of the address: align every buffer to 1024 B.
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;
    const uint32_t pl0 = pk0 + TC_PK_STAGES * TC_PK_BYTES;
    const uint32_t epi0 = pl0 + TC_PL_STAGES * TC_PL_BYTES;
    const uint32_t bar0 = epi0 + TC_EPI_BYTES;
    uint8_t *epi_g = gbase + (epi0 - base);
    // barriers (8 B each)
    auto pk_full = [&](int s) { return bar0 + 8u * s; };
    auto pk_empty = [&](int s) { return bar0 + 8u * (TC_PK_STAGES + s); };
    auto pl_full = [&](int s) { return bar0 + 8u * (2 * TC_PK_STAGES + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (2 * TC_PK_STAGES + TC_PL_STAGES + s); };
    const uint32_t acc_full = bar0 + 8u * (2 * TC_PK_STAGES + 2 * TC_PL_STAGES);
    const uint32_t acc_empty = acc_full + 8u;
    const uint32_t tmem_slot = acc_empty + 8u;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap);
        for (int s = 0; s < TC_PK_STAGES; ++s) {
            ptx::mbar_init(pk_full(s), 1);
            ptx::mbar_init(pk_empty(s), TC_UNPACK_WARPS);
        }
        for (int s = 0; s < TC_PL_STAGES; ++s) {
            ptx::mbar_init(pl_full(s), TC_UNPACK_WARPS);
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, 4);
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<1>(tmem_slot, 512);
        ptx::tmem_relinquish<1>();
    }
    ptx::tc_fence_before_sync();
    __syncthreads();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot_g;

    const int units_per_f = p.tiles_per_f * p.slices;

    if (warp == 0) {
        // ===================== S1: TMA producer =====================
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            for (int u = blockIdx.x; u < p.num_units; u += gridDim.x) {
                const int f = u / units_per_f, rem = u % units_per_f;
                const ushort2 tile = p.tiles[rem / p.slices];
                const int slice = rem % p.slices;
                const int t_begin = slice * p.t_per_slice;
                const int t_end = min(p.T, t_begin + p.t_per_slice);
                const bool diag = tile.x == tile.y;
                for (int t = t_begin; t < t_end; t += TC_ST) {
                    ptx::mbar_wait(pk_empty(st), ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(pk_full(st), diag ? TC_PLANE : 2 * TC_PLANE);
                    const uint32_t dst = pk0 + st * TC_PK_BYTES;
                    ptx::tma_load_3d(dst, &tmap, pk_full(st), tile.x * TC_BLK, f, t);
                    if (!diag) ptx::tma_load_3d(dst + TC_PLANE, &tmap, pk_full(st), tile.y * TC_BLK, f, t);
                    if (++st == TC_PK_STAGES) { st = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issuer =====================
        if (lane == 0) {
            constexpr uint32_t idesc256 = make_idesc_i8(128, 256, true, true, true, true);
            constexpr uint32_t idesc128 = make_idesc_i8(128, 128, true, true, true, true);
            int st = 0;
            uint32_t ph = 0, acc_ph = 0;
            for (int u = blockIdx.x; u < p.num_units; u += gridDim.x) {
                const int rem = u % units_per_f;
                const ushort2 tile = p.tiles[rem / p.slices];
                const int slice = rem % p.slices;
                const int t_begin = slice * p.t_per_slice;
                const int t_end = min(p.T, t_begin + p.t_per_slice);
                const bool diag = tile.x == tile.y;
                ptx::mbar_wait(acc_empty, acc_ph ^ 1u);  // epilogue has drained the accumulators
                ptx::tc_fence_after_sync();
                bool first = true;
                for (int t = t_begin; t < t_end; t += TC_ST) {
                    ptx::mbar_wait(pl_full(st), ph);
                    ptx::tc_fence_after_sync();
                    const uint32_t pl = pl0 + st * TC_PL_BYTES;
                    const uint32_t a_r = pl, a_i = pl + TC_PLANE;
                    const uint32_t b_r = diag ? a_r : pl + 2 * TC_PLANE;
#pragma unroll
                    for (int ks = 0; ks < TC_ST / 32; ++ks) {
                        const uint32_t ko = ks * 32 * TC_BLK;  // 32 K-rows of 128 B
                        const uint64_t dAr = make_smem_desc(a_r + ko, TC_PLANE, 1024, 2);
                        const uint64_t dAi = make_smem_desc(a_i + ko, TC_PLANE, 1024, 2);
                        const uint64_t dB = make_smem_desc(b_r + ko, TC_PLANE, 1024, 2);  // [Br;Bi] via LBO
                        if (first) {
                            const uint64_t dBi = make_smem_desc(b_r + TC_PLANE + ko, TC_PLANE, 1024, 2);
                            ptx::mma_i8_ss<1>(tmem + 0, dAi, dB, idesc256, 0);     // IR | II   (overwrite)
                            ptx::mma_i8_ss<1>(tmem + 128, dAr, dB, idesc128, 1);   // += RR (B = Br only)
                            ptx::mma_i8_ss<1>(tmem + 256, dAr, dBi, idesc128, 0);  // RI        (overwrite)
                            first = false;
                        } else {
                            ptx::mma_i8_ss<1>(tmem + 0, dAi, dB, idesc256, 1);
                            ptx::mma_i8_ss<1>(tmem + 128, dAr, dB, idesc256, 1);
                        }
                    }
                    ptx::mma_commit<1>(pl_empty(st));  // planes free once these MMAs have read them
                    if (++st == TC_PL_STAGES) { st = 0; ph ^= 1u; }
                }
                ptx::mma_commit<1>(acc_full);
                acc_ph ^= 1u;
            }
        }
    } else if (warp < TC_EPI_WARP0) {
        // ===================== S2: unpack =====================
        const int ut = threadIdx.x - 64;  // 0..TC_UNPACK_THREADS-1
        int pst = 0, qst = 0;
        uint32_t pph = 0, qph = 0;
        for (int u = blockIdx.x; u < p.num_units; u += gridDim.x) {
            const int rem = u % units_per_f;
            const ushort2 tile = p.tiles[rem / p.slices];
            const int slice = rem % p.slices;
            const int t_begin = slice * p.t_per_slice;
            const int t_end = min(p.T, t_begin + p.t_per_slice);
            const bool diag = tile.x == tile.y;
            for (int t = t_begin; t < t_end; t += TC_ST) {
                const int rows_valid = t_end - t;  // rows >= rows_valid are beyond the slice: zero them
                ptx::mbar_wait(pk_full(pst), pph);
                ptx::mbar_wait(pl_empty(qst), qph ^ 1u);
                const uint32_t src = pk0 + pst * TC_PK_BYTES;
                const uint32_t dst = pl0 + qst * TC_PL_BYTES;
                const int nblk = diag ? 1 : 2;
                constexpr int CH = TC_PLANE / 16 / TC_UNPACK_THREADS;  // 16-byte chunks per thread per block
                const uint8_t *srcg = gbase + (src - base);
                uint8_t *dstg = gbase + (dst - base);
                uint4 w[2][CH];
                // all loads of the stage first (independent, several in flight), then logic + stores
                for (int b = 0; b < nblk; ++b)
#pragma unroll
                    for (int k = 0; k < CH; ++k)
                        w[b][k] = *reinterpret_cast<const uint4 *>(srcg + b * TC_PLANE +
                                                                   (k * TC_UNPACK_THREADS + ut) * 16);
                for (int b = 0; b < nblk; ++b) {
#pragma unroll
                    for (int k = 0; k < CH; ++k) {
                        const uint32_t off = (uint32_t)(k * TC_UNPACK_THREADS + ut) * 16u;
                        const bool ok = (int)(off >> 7) < rows_valid;
                        const uint32_t m = ok ? 0xF0F0F0F0u : 0u;
                        const uint4 v = w[b][k];
                        uint4 r, i;
                        r.x = (v.x ^ 0x80808080u) & m; r.y = (v.y ^ 0x80808080u) & m;
                        r.z = (v.z ^ 0x80808080u) & m; r.w = (v.w ^ 0x80808080u) & m;
                        i.x = ((v.x << 4) ^ 0x80808080u) & m; i.y = ((v.y << 4) ^ 0x80808080u) & m;
                        i.z = ((v.z << 4) ^ 0x80808080u) & m; i.w = ((v.w << 4) ^ 0x80808080u) & m;
                        *reinterpret_cast<uint4 *>(dstg + b * 2 * TC_PLANE + off) = r;
                        *reinterpret_cast<uint4 *>(dstg + b * 2 * TC_PLANE + TC_PLANE + off) = i;
                    }
                }
                ptx::fence_proxy_async_smem();  // planes were written by the generic proxy; MMA reads via async proxy
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive(pl_full(qst));
                    ptx::mbar_arrive(pk_empty(pst));
                }
                if (++pst == TC_PK_STAGES) { pst = 0; pph ^= 1u; }
                if (++qst == TC_PL_STAGES) { qst = 0; qph ^= 1u; }
            }
        }
    } else {
        // ===================== S5: epilogue =====================
        const int q = warp & 3;  // TMEM lane quarter this warp may read
        uint8_t *stage = epi_g + (warp - TC_EPI_WARP0) * 32 * TC_EPI_PITCH;
        const size_t Bn = (size_t)p.n_out * ((size_t)p.n_out + 1) / 2;
        const int cpt = TC_BLK / p.sub;   // channels per tile (1, or 2 when packed)
        const int ssh = (p.sub == 64) ? 6 : 7;   // log2(sub)
        uint32_t acc_ph = 0;
        for (int u = blockIdx.x; u < p.num_units; u += gridDim.x) {
            const int f = u / units_per_f, rem = u % units_per_f;
            const ushort2 tile = p.tiles[rem / p.slices];
            const int x0 = tile.x * TC_BLK, y0 = tile.y * TC_BLK;
            const int xw = x0 + q * 32;  // first row of this warp
            ptx::mbar_wait(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
            const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
#pragma unroll 1
            for (int c = 0; c < 8; ++c) {
                const int yc = y0 + c * 16;
                // whole 32x16 block below the diagonal or outside the matrix: nothing to write
                const bool skip = (yc + 15 < xw) || (yc >= p.N) || (xw >= p.N) || (((yc - y0) >> ssh) != ((xw - x0) >> ssh));   // packed: the other channel's columns
                if (!skip) {
                    uint32_t s1[16], rr[16], s2[16];
                    ptx::tmem_ld16(trow + c * 16, s1);
                    ptx::tmem_ld16(trow + 128 + c * 16, rr);
                    ptx::tmem_ld16(trow + 256 + c * 16, s2);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int re = (int)rr[j] >> 8;
                        const int im = (int)(s1[j] - s2[j]) >> 8;
                        *reinterpret_cast<int2 *>(stage + lane * TC_EPI_PITCH + j * 8) = make_int2(re, im);
                    }
                    __syncwarp();
                    const int col = lane & 15;
                    const int y = yc + col;
#pragma unroll 4
                    for (int rr2 = 0; rr2 < 16; ++rr2) {
                        const int rl = rr2 * 2 + (lane >> 4);
                        const int x = xw + rl;
                        if (x < p.N && y < p.N && x <= y) {
                            const int2 v = *reinterpret_cast<const int2 *>(stage + rl * TC_EPI_PITCH + col * 8);
                            const int cx = (x - x0) >> ssh;   // packed: channel of the tile (same for x and y, see skip)
                            int32_t *o = p.vis + ((size_t)(f * cpt + cx) * Bn + baseline_index(p.n_out, x - cx * p.sub, y - cx * p.sub)) * 2;
                            if (p.out_mode == OUT_STORE) {
                                *reinterpret_cast<int2 *>(o) = v;
                            } else if (p.out_mode == OUT_RMW) {
                                int2 old = *reinterpret_cast<int2 *>(o);
                                old.x += v.x;
                                old.y += v.y;
                                *reinterpret_cast<int2 *>(o) = old;
                            } else {
                                atomicAdd(o, v.x);
                                atomicAdd(o + 1, v.y);
                            }
                        }
                    }
                    __syncwarp();
                }
            }
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(acc_empty);
        }
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc<1>(tmem, 512);
}

}  // namespace corr
