// corr_tc2.cuh -- the CTA-pair (cta_group::2) version of the large-N path (steps S1-S5).
//
// Same mathematics as corr_tc.cuh (Eq. 1; x16 int8 operand planes; results
// shifted right by 8 in the epilogue), different mapping: two CTAs on the two SMs of one TPC
// form a cluster and compute one 256 (x) by 128 (y) tile together with M=256, N=256, K=32
// tcgen05.mma.cta_group::2 instructions.
//
// Why pairs: ncu on the single-CTA kernel shows the shared-memory data pipe at 95 % (LSU
// wavefronts 56 % + tensor-core operand wavefronts 39 %) with the tensor pipe starved.  In a pair
// each CTA feeds the tensor cores only its own 128 A rows and HALF of the B rows, and unpacks
// only its own x-block plus half of the y-block.  Per 64 time samples and per CTA the traffic
// drops from 112 KB to 80 KB (TMA 12, unpack reads 12, unpack writes 24, MMA reads 32).
//
// Per CTA r (= rank in the pair) and per stage of ST time samples:
//   packed X_r  [ST][128] bytes, 128-B swizzle   x in [256*bx2 + 128 r, +128)
//   packed Yh_r [ST][ 64] bytes,  64-B swizzle   y in [128*by + 64 r, +64)
//   planes Ar, Ai   [ST][128] MN-major SW128     (16*Re, 16*Im of the CTA's x-block)
//   planes Bhr, Bhi [ST][ 64] MN-major SW64      (16*Re, 16*Im of the CTA's y-half); the MMA sees
//          them as ONE 128-row B operand through the descriptor's leading-dimension offset.
// Accumulators (TMEM, all 512 columns, per CTA for its 128 x rows):
//   cols   0..255  D1 += Ai * B^T    B rows n: [0,64) Br(y0-63) [64,128) Bi(y0-63) [128,192) Br(y64-127) [192,256) Bi(y64-127)
//   cols 256..511  D2 += Ar * B^T
// so for y = 64 h + yl:  IR = D1[128h+yl], II = D1[128h+64+yl], RR = D2[128h+yl], RI = D2[128h+64+yl],
//   Re = (RR + II) >> 8,  Im = (IR - RI) >> 8.
//
// Synchronisation across the pair: the packed ring (TMA -> unpack) is CTA-local.  The plane ring
// is shared: unpack warps of BOTH CTAs arrive on the leader's pl_full barrier; the leader's MMA
// thread commits with multicast so pl_empty / acc_full fire in both CTAs; epilogue warps of both
// CTAs arrive on the leader's acc_empty.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode, baseline_index
#include "corr_ptx.cuh"

namespace corr {

constexpr int T2_BLK = 128;            // per-CTA tile edge in x, pair tile edge in y
constexpr int T2_ST = 64;              // time samples per stage
constexpr int T2_PK_STAGES = 6;
constexpr int T2_PL_STAGES = 4;
constexpr int T2_UNPACK_WARPS = 8;
constexpr int T2_UNPACK_THREADS = 32 * T2_UNPACK_WARPS;
constexpr int T2_EPI_WARP0 = 2 + T2_UNPACK_WARPS;
constexpr int T2_EPI_WARPS = 4;
constexpr int T2_THREADS = 32 * (T2_EPI_WARP0 + T2_EPI_WARPS);
constexpr int T2_XPLANE = T2_ST * 128;             // bytes: one x plane / packed X per stage
constexpr int T2_YPLANE = T2_ST * 64;              // bytes: one y-half plane / packed Yh per stage
constexpr int T2_PK_BYTES = T2_XPLANE + T2_YPLANE;
constexpr int T2_PL_BYTES = 2 * T2_XPLANE + 2 * T2_YPLANE;
constexpr int T2_EPI_PITCH = 16 * 8 + 8;
constexpr int T2_EPI_BYTES = T2_EPI_WARPS * 32 * T2_EPI_PITCH;
constexpr int T2_SMEM_BYTES = 1024 + T2_PK_STAGES * T2_PK_BYTES + T2_PL_STAGES * T2_PL_BYTES + T2_EPI_BYTES + 256;

struct Tc2Params {
    int N, F, T;
    int tiles_per_f;   // pair tiles (256 x 128) touching the upper triangle, per channel
    int slices;
    int t_per_slice;   // multiple of T2_ST
    int num_units;     // F * tiles_per_f * slices
    int out_mode;
    const ushort2 *tiles;  // (bx2, by): x-block of 256, y-block of 128
    int32_t *vis;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T2_THREADS, 1)
corr_tc2_kernel(const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_y,
                const Tc2Params p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;
    const uint32_t pl0 = pk0 + T2_PK_STAGES * T2_PK_BYTES;
    const uint32_t epi0 = pl0 + T2_PL_STAGES * T2_PL_BYTES;
    const uint32_t bar0 = epi0 + T2_EPI_BYTES;
    uint8_t *epi_g = gbase + (epi0 - base);
    auto pk_full = [&](int s) { return bar0 + 8u * s; };
    auto pk_empty = [&](int s) { return bar0 + 8u * (T2_PK_STAGES + s); };
    auto pl_full = [&](int s) { return bar0 + 8u * (2 * T2_PK_STAGES + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (2 * T2_PK_STAGES + T2_PL_STAGES + s); };
    const uint32_t acc_full = bar0 + 8u * (2 * T2_PK_STAGES + 2 * T2_PL_STAGES);
    const uint32_t acc_empty = acc_full + 8u;
    const uint32_t tmem_slot = acc_empty + 8u;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();  // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap_x);
        ptx::prefetch_tmap(&tmap_y);
        for (int s = 0; s < T2_PK_STAGES; ++s) {
            ptx::mbar_init(pk_full(s), 1);
            ptx::mbar_init(pk_empty(s), T2_UNPACK_WARPS);
        }
        for (int s = 0; s < T2_PL_STAGES; ++s) {
            ptx::mbar_init(pl_full(s), 2 * T2_UNPACK_WARPS);  // both CTAs' unpack warps (leader's copy is used)
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, 2 * T2_EPI_WARPS);
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<2>(tmem_slot, 512);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot_g;

    const int units_per_f = p.tiles_per_f * p.slices;

    if (warp == 0) {
        // ===================== S1: TMA producer (each CTA loads its own blocks) =====================
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            for (int u = pair; u < p.num_units; u += npairs) {
                const int f = u / units_per_f, rem = u % units_per_f;
                const ushort2 tile = p.tiles[rem / p.slices];
                const int slice = rem % p.slices;
                const int t_begin = slice * p.t_per_slice;
                const int t_end = min(p.T, t_begin + p.t_per_slice);
                const int xc = tile.x * 256 + (int)rank * 128;
                const int yc = tile.y * 128 + (int)rank * 64;
                for (int t = t_begin; t < t_end; t += T2_ST) {
                    ptx::mbar_wait(pk_empty(st), ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(pk_full(st), T2_PK_BYTES);
                    const uint32_t dst = pk0 + st * T2_PK_BYTES;
                    ptx::tma_load_3d(dst, &tmap_x, pk_full(st), xc, f, t);
                    ptx::tma_load_3d(dst + T2_XPLANE, &tmap_y, pk_full(st), yc, f, t);
                    if (++st == T2_PK_STAGES) { st = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issuer (leader CTA only) =====================
        if (lane == 0 && rank == 0) {
            constexpr uint32_t idesc = make_idesc_i8(256, 256, true, true, true, true);
            int st = 0;
            uint32_t ph = 0, acc_ph = 0;
            for (int u = pair; u < p.num_units; u += npairs) {
                const int rem = u % units_per_f;
                const int slice = rem % p.slices;
                const int t_begin = slice * p.t_per_slice;
                const int t_end = min(p.T, t_begin + p.t_per_slice);
                ptx::mbar_wait_cluster(acc_empty, acc_ph ^ 1u);
                ptx::tc_fence_after_sync();
                uint32_t acc = 0;
                for (int t = t_begin; t < t_end; t += T2_ST) {
                    ptx::mbar_wait_cluster(pl_full(st), ph);
                    ptx::tc_fence_after_sync();
                    const uint32_t pl = pl0 + st * T2_PL_BYTES;
                    const uint32_t a_r = pl, a_i = pl + T2_XPLANE, b_h = pl + 2 * T2_XPLANE;
#pragma unroll
                    for (int ks = 0; ks < T2_ST / 32; ++ks) {
                        // A: MN-major SW128, 8-row K groups 1024 B apart; K-step of 32 rows = 4096 B
                        const uint64_t dAr = make_smem_desc(a_r + ks * 4096, T2_XPLANE, 1024, 2);
                        const uint64_t dAi = make_smem_desc(a_i + ks * 4096, T2_XPLANE, 1024, 2);
                        // B half: MN-major SW64: two 64-wide MN blocks (Re plane, Im plane) T2_YPLANE apart,
                        // 8-row K groups 512 B apart; K-step of 32 rows = 2048 B
                        const uint64_t dB = make_smem_desc(b_h + ks * 2048, T2_YPLANE, 512, 4);
                        ptx::mma_i8_ss<2>(tmem + 0, dAi, dB, idesc, acc);
                        ptx::mma_i8_ss<2>(tmem + 256, dAr, dB, idesc, acc);
                        acc = 1;
                    }
                    ptx::mma_commit_mcast2(pl_empty(st), 0x3);  // planes of BOTH CTAs are free
                    if (++st == T2_PL_STAGES) { st = 0; ph ^= 1u; }
                }
                ptx::mma_commit_mcast2(acc_full, 0x3);
                acc_ph ^= 1u;
            }
        }
    } else if (warp < T2_EPI_WARP0) {
        // ===================== S2: unpack =====================
        const int ut = threadIdx.x - 64;
        int pst = 0, qst = 0;
        uint32_t pph = 0, qph = 0;
        for (int u = pair; u < p.num_units; u += npairs) {
            const int rem = u % units_per_f;
            const int slice = rem % p.slices;
            const int t_begin = slice * p.t_per_slice;
            const int t_end = min(p.T, t_begin + p.t_per_slice);
            for (int t = t_begin; t < t_end; t += T2_ST) {
                const int rows_valid = t_end - t;
                ptx::mbar_wait(pk_full(pst), pph);
                ptx::mbar_wait_cluster(pl_empty(qst), qph ^ 1u);
                const uint8_t *src = gbase + (pk0 - base) + pst * T2_PK_BYTES;
                uint8_t *dst = gbase + (pl0 - base) + qst * T2_PL_BYTES;
                constexpr int CX = T2_XPLANE / 16 / T2_UNPACK_THREADS;  // 2
                constexpr int CY = T2_YPLANE / 16 / T2_UNPACK_THREADS;  // 1
                uint4 wx[CX], wy[CY];
#pragma unroll
                for (int k = 0; k < CX; ++k)
                    wx[k] = *reinterpret_cast<const uint4 *>(src + (k * T2_UNPACK_THREADS + ut) * 16);
#pragma unroll
                for (int k = 0; k < CY; ++k)
                    wy[k] = *reinterpret_cast<const uint4 *>(src + T2_XPLANE + (k * T2_UNPACK_THREADS + ut) * 16);
                auto split = [&](const uint4 v, bool ok, uint4 &r, uint4 &i) {
                    const uint32_t m = ok ? 0xF0F0F0F0u : 0u;
                    r.x = (v.x ^ 0x80808080u) & m; r.y = (v.y ^ 0x80808080u) & m;
                    r.z = (v.z ^ 0x80808080u) & m; r.w = (v.w ^ 0x80808080u) & m;
                    i.x = ((v.x << 4) ^ 0x80808080u) & m; i.y = ((v.y << 4) ^ 0x80808080u) & m;
                    i.z = ((v.z << 4) ^ 0x80808080u) & m; i.w = ((v.w << 4) ^ 0x80808080u) & m;
                };
#pragma unroll
                for (int k = 0; k < CX; ++k) {
                    const uint32_t off = (uint32_t)(k * T2_UNPACK_THREADS + ut) * 16u;
                    uint4 r, i;
                    split(wx[k], (int)(off >> 7) < rows_valid, r, i);  // 128-B rows
                    *reinterpret_cast<uint4 *>(dst + off) = r;
                    *reinterpret_cast<uint4 *>(dst + T2_XPLANE + off) = i;
                }
#pragma unroll
                for (int k = 0; k < CY; ++k) {
                    const uint32_t off = (uint32_t)(k * T2_UNPACK_THREADS + ut) * 16u;
                    uint4 r, i;
                    split(wy[k], (int)(off >> 6) < rows_valid, r, i);  // 64-B rows
                    *reinterpret_cast<uint4 *>(dst + 2 * T2_XPLANE + off) = r;
                    *reinterpret_cast<uint4 *>(dst + 2 * T2_XPLANE + T2_YPLANE + off) = i;
                }
                ptx::fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive_cluster(pl_full(qst), 0);  // the leader's barrier
                    ptx::mbar_arrive(pk_empty(pst));
                }
                if (++pst == T2_PK_STAGES) { pst = 0; pph ^= 1u; }
                if (++qst == T2_PL_STAGES) { qst = 0; qph ^= 1u; }
            }
        }
    } else {
        // ===================== S5: epilogue =====================
        const int q = warp & 3;
        uint8_t *stage = epi_g + (warp - T2_EPI_WARP0) * 32 * T2_EPI_PITCH;
        const size_t Bn = (size_t)p.N * ((size_t)p.N + 1) / 2;
        uint32_t acc_ph = 0;
        for (int u = pair; u < p.num_units; u += npairs) {
            const int f = u / units_per_f, rem = u % units_per_f;
            const ushort2 tile = p.tiles[rem / p.slices];
            const int x0 = tile.x * 256 + (int)rank * 128, y0 = tile.y * 128;
            const int xw = x0 + q * 32;
            ptx::mbar_wait_cluster(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
            const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
#pragma unroll 1
            for (int c = 0; c < 8; ++c) {
                const int yc = y0 + c * 16;
                const bool skip = (yc + 15 < xw) || (yc >= p.N) || (xw >= p.N);
                if (!skip) {
                    const uint32_t col = (uint32_t)((c >> 2) * 128 + (c & 3) * 16);  // 128h + yl
                    uint32_t ir[16], ii[16], rr[16], ri[16];
                    ptx::tmem_ld16(trow + col, ir);
                    ptx::tmem_ld16(trow + col + 64, ii);
                    ptx::tmem_ld16(trow + 256 + col, rr);
                    ptx::tmem_ld16(trow + 256 + col + 64, ri);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int re = (int)(rr[j] + ii[j]) >> 8;
                        const int im = (int)(ir[j] - ri[j]) >> 8;
                        *reinterpret_cast<int2 *>(stage + lane * T2_EPI_PITCH + j * 8) = make_int2(re, im);
                    }
                    __syncwarp();
                    const int cl = lane & 15;
                    const int y = yc + cl;
#pragma unroll 4
                    for (int r2 = 0; r2 < 16; ++r2) {
                        const int rl = r2 * 2 + (lane >> 4);
                        const int x = xw + rl;
                        if (x < p.N && y < p.N && x <= y) {
                            const int2 v = *reinterpret_cast<const int2 *>(stage + rl * T2_EPI_PITCH + cl * 8);
                            int32_t *o = p.vis + ((size_t)f * Bn + baseline_index(p.N, x, y)) * 2;
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
            if (lane == 0) ptx::mbar_arrive_cluster(acc_empty, 0);
        }
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();  // no CTA of the pair may exit while its peer still reads its smem / barriers
    if (warp == 1) ptx::tmem_dealloc<2>(tmem, 512);
}

}  // namespace corr
