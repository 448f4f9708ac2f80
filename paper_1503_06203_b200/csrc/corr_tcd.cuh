// corr_tcd.cuh -- steps S1-S5 for N <= 256: 128 x 128 tiles, one CTA each, with the A operand in tensor memory.
// corr_tcd_kernel<false>: one tile per channel, the DIAGONAL block (N <= 128, and two channels of 64 inputs per tile);
// corr_tcd_kernel<true>: every block of the triangle (128 < N <= 256 by default), see the template's comment.
//
// Same mathematics as the other tcgen05 kernels (Eq. 1, summed over time PAPER.md:48, upper triangle
// PAPER.md:50; x16 int8 operand planes, results shifted right by 8 in the epilogue).  corr_tc.cuh serves these sizes
// with both operands' planes in shared memory and moves 768 wavefronts through the shared-memory pipe per 64-sample
// stage against 512 tensor cycles.  Here, as in corr_tc3.cuh:
//   * the rows' planes never enter shared memory: ldmatrix.m16n16.x2.trans.b8 transposes the packed block, the
//     planes 16 Re, 16 Im are formed in registers and written to TMEM with tcgen05.st (A operand of the MMAs);
//   * rows and columns are the same 128 inputs, so ONE packed block per stage is loaded (8 KB) and the columns'
//     planes Br, Bi are made from it at the same physical offsets (MN-major, 128-B swizzle as TMA wrote it);
//   * the epilogue stages the rows of the upper triangle in shared memory and sends them as bulk copies / bulk
//     reduce-adds; rows 64..127 only hold columns 64..127, which is what lets the image fit beside the rings.
// Per stage: 64 (ldmatrix) + 64 (loads) + 128 (plane stores) + 256 (tensor-core reads) = 512 wavefronts.
//
// TMEM columns:   0..127  IR += Ai Br^T     128..255  Re += Ai Bi^T + Ar Br^T     256..383  RI += Ar Bi^T
//               384..511  A planes, 4 stages x (Ar 16 columns | Ai 16 columns); lane = input
//   Re = D[128 + j] >> 8,   Im = (D[j] - D[256 + j]) >> 8.
// Two whole channels of 64 inputs per tile (TcParams::sub = 64, see corr_tc.cuh): only the two diagonal 64-blocks are
// written, as channels 2f and 2f + 1.
//
// Warps (576 threads, one CTA per SM, persistent over units = (channel, T-slice)):
//   0 TMA producer | 1 TMEM owner + MMA issue | 2-9 unpack | 10-17 epilogue (lane quarter warp % 4, column half)
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode
#include "corr_ptx.cuh"
#include "corr_tc.cuh"    // TcParams

namespace corr {

constexpr int TD_ST = 64;               // time samples per stage
#ifndef TD_PK_N
#define TD_PK_N 6
#endif
#ifndef TD_PL_N
#define TD_PL_N 4
#endif
constexpr int TD_PK_STAGES = TD_PK_N;   // packed-byte ring when every tile is a diagonal block (N <= 128): one block per stage
constexpr int TD_PK_STAGES_G = 6;       // ... when the triangle has off-diagonal blocks: rows' block + columns' block per stage
constexpr int TD_PL_STAGES = TD_PL_N;   // operand ring: TMEM A stage + smem B stage
constexpr int TD_GROUP = TD_ST * TD_PL_STAGES;   // a unit runs whole groups of stages (static ring positions in the MMA loop)
constexpr int TD_UNPACK_WARPS = 8;
constexpr int TD_EPI_WARP0 = 2 + TD_UNPACK_WARPS;
constexpr int TD_EPI_WARPS = 8;
constexpr int TD_THREADS = 32 * (TD_EPI_WARP0 + TD_EPI_WARPS);
constexpr int TD_PK_BYTES = TD_ST * 128;          // the packed block of a stage
constexpr int TD_PLANE = TD_ST * 128;             // one plane of the columns per stage
constexpr int TD_PL_BYTES = 2 * TD_PLANE;         // Br, Bi
constexpr int TD_PITCH_LO = 128 * 8 + 16;         // image of a row 0..63: 128 baselines + parity slot
constexpr int TD_PITCH_HI = 64 * 8 + 16;          // image of a row 64..127: columns 64..127 + parity slot
constexpr int TD_EPI_BYTES = 64 * (TD_PITCH_LO + TD_PITCH_HI);
constexpr int TD_SMEM_BYTES = 1024 + TD_PK_STAGES * TD_PK_BYTES + TD_PL_STAGES * TD_PL_BYTES + TD_EPI_BYTES + 384;
// with off-diagonal blocks: a ring of double stages, and an image of 64 rows that the two halves of the block use in turn
constexpr int TD_EPI_BYTES_G = 64 * TD_PITCH_LO;
constexpr int TD_SMEM_BYTES_G = 1024 + TD_PK_STAGES_G * 2 * TD_PK_BYTES + TD_PL_STAGES * TD_PL_BYTES + TD_EPI_BYTES_G + 384;
static_assert(TD_SMEM_BYTES <= 232448 && TD_SMEM_BYTES_G <= 232448, "227 KB of shared memory per CTA");
constexpr uint32_t TD_ACOL0 = 384, TD_ACOLS = 32;
constexpr int TD_MAX_SLICE = 32768;               // |sum| <= 2 * 128 * 128 * slice < 2^31

// GENERAL = false: every tile is the diagonal block (0, 0) of its channel (N <= 128, or two channels of 64 per tile).
// GENERAL = true: tiles (bx <= by) of p.tiles; off-diagonal tiles load two packed blocks per stage (rows', columns') into a
// ring of TD_PK_STAGES_G double stages and write all 128 x 128 baselines.
template <bool GENERAL>
__global__ void __launch_bounds__(TD_THREADS, 1)
corr_tcd_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int PK_STAGES = GENERAL ? TD_PK_STAGES_G : TD_PK_STAGES;
    constexpr int PK_BYTES = GENERAL ? 2 * TD_PK_BYTES : TD_PK_BYTES;
    // a (ring position, unpack group) pair of barriers is used once every PK_PERIOD stages (stage j: position j % PK_STAGES,
    // group j & 1; with an odd ring a group comes back to a position only every second time round)
    constexpr int PK_PERIOD = (PK_STAGES % 2 == 0) ? PK_STAGES : 2 * PK_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;
    const uint32_t pl0 = pk0 + PK_STAGES * PK_BYTES;
    const uint32_t epi0 = pl0 + TD_PL_STAGES * TD_PL_BYTES;
    const uint32_t bar0 = epi0 + (GENERAL ? TD_EPI_BYTES_G : TD_EPI_BYTES);
    auto pk_full = [&](int s, int g) { return bar0 + 8u * (2 * s + g); };
    auto pk_empty = [&](int s, int g) { return bar0 + 8u * (2 * PK_STAGES + 2 * s + g); };
    auto pl_full = [&](int s) { return bar0 + 8u * (4 * PK_STAGES + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (4 * PK_STAGES + TD_PL_STAGES + s); };
    const uint32_t acc_full = bar0 + 8u * (4 * PK_STAGES + 2 * TD_PL_STAGES);
    const uint32_t acc_empty = acc_full + 8u;
    const uint32_t tmem_slot = acc_empty + 8u;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap);
        for (int s = 0; s < PK_STAGES; ++s)
            for (int g = 0; g < 2; ++g) {
                ptx::mbar_init(pk_full(s, g), 1);
                ptx::mbar_init(pk_empty(s, g), TD_UNPACK_WARPS / 2);   // the group of unpack warps that takes the stage
            }
        for (int s = 0; s < TD_PL_STAGES; ++s) {
            ptx::mbar_init(pl_full(s), TD_UNPACK_WARPS / 2);
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, TD_EPI_WARPS);
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
    if (tmem != 0) __trap();  // all 512 columns were requested: the allocation starts at lane 0, column 0

    // The work of a call is cut into SEGMENTS (channel f, samples [t_begin, t_end)), each run as whole groups of TD_GROUP
    // samples (the stages beyond t_end are loaded -- TMA fills rows beyond T with zeros -- and masked to zero operands
    // by the unpack).  Two schedules, chosen by the host:
    //   slices > 0   unit u = (channel, T-slice), units dealt round-robin: every channel's sum has one owner (or a few
    //                when T is split for int32 headroom or to fill the SMs);
    //   slices == 0  all groups of all channels in one row, cut into gridDim.x EQUAL shares: a CTA's share covers
    //                parts of up to a few channels, every segment is added into vis (which the host has cleared).
    //                This is what fills 148 SMs when the channels are few and long (64 channels: 128 units otherwise).
    long long it, it_end;
    const int tiles_per_f = GENERAL ? p.tiles_per_f : 1;
    if (p.slices > 0) {
        it = blockIdx.x;
        it_end = p.num_units;
    } else {
        const long long G = (long long)p.F * tiles_per_f * p.groups_per_f;
        it = G * blockIdx.x / gridDim.x;
        it_end = G * (blockIdx.x + 1) / gridDim.x;
    }
    struct Seg { int f, bx, by, t_begin, t_end, ngroups; };
    auto next_segment = [&](Seg &sg) -> bool {
        if (it >= it_end) return false;
        int ft;   // (channel, tile)
        if (p.slices > 0) {
            const int u = (int)it;
            ft = u / p.slices;
            const int slice = u - ft * p.slices;
            sg.t_begin = slice * p.t_per_slice;
            sg.t_end = min(p.T, sg.t_begin + p.t_per_slice);
            sg.ngroups = (sg.t_end - sg.t_begin + TD_GROUP - 1) / TD_GROUP;
            it += gridDim.x;
        } else {
            ft = (int)(it / p.groups_per_f);
            const int first = (int)(it - (long long)ft * p.groups_per_f);
            sg.ngroups = (int)min((long long)min(p.groups_per_f - first, TD_MAX_SLICE / TD_GROUP), it_end - it);
            sg.t_begin = first * TD_GROUP;
            sg.t_end = min(p.T, sg.t_begin + sg.ngroups * TD_GROUP);
            it += sg.ngroups;
        }
        sg.f = ft / tiles_per_f;
        sg.bx = sg.by = 0;
        if (GENERAL) {
            const ushort2 tile = p.tiles[ft - sg.f * tiles_per_f];
            sg.bx = tile.x;
            sg.by = tile.y;
        }
        return true;
    };
    Seg sg;

    if (warp == 0) {
        // ===================== S1: TMA producer =====================
        if (lane == 0) {
            int st = 0;
            uint32_t j = 0;   // stages loaded so far: stage j goes to ring position j % PK_STAGES and to unpack group j & 1
            while (next_segment(sg)) {
                const bool diag = sg.bx == sg.by;
                for (int t = sg.t_begin; t < sg.t_begin + sg.ngroups * TD_GROUP; t += TD_ST) {
                    const int g = (int)(j & 1u);
                    if (j >= (uint32_t)PK_STAGES) {   // the position's last stage, j - PK_STAGES, has been unpacked
                        const uint32_t jp = j - PK_STAGES;
                        ptx::mbar_wait(pk_empty(st, (int)(jp & 1u)), (jp / PK_PERIOD) & 1u);
                    }
                    ptx::mbar_arrive_expect_tx(pk_full(st, g), (!GENERAL || diag) ? TD_PK_BYTES : 2 * TD_PK_BYTES);
                    if (!GENERAL && p.win_n > 0)   // unpadded stream: the window of channel f starts at column f * N rounded down to 16
                        ptx::tma_load_2d(pk0 + st * PK_BYTES, &tmap, pk_full(st, g), (sg.f * p.win_c * p.win_n) & ~15, t);
                    else if (!GENERAL && p.sub == 64)   // two channels per tile: the stream as a byte matrix, tile f at column 128 f
                        ptx::tma_load_2d(pk0 + st * PK_BYTES, &tmap, pk_full(st, g), 128 * sg.f, t);
                    else
                        ptx::tma_load_3d(pk0 + st * PK_BYTES, &tmap, pk_full(st, g), sg.bx * 128, sg.f, t);
                    if (GENERAL && !diag) ptx::tma_load_3d(pk0 + st * PK_BYTES + TD_PK_BYTES, &tmap, pk_full(st, g), sg.by * 128, sg.f, t);
                    ++j;
                    if (++st == PK_STAGES) st = 0;
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issue =====================
        // the whole warp runs the loop (warp-uniform operands, compile-time ring positions), one elected lane issues
        constexpr uint32_t idesc = make_idesc_i8(128, 128, true, true, /*A K-major (TMEM)*/ false, /*B MN-major*/ true);
        uint32_t ph = 0, acc_ph = 0;
        const bool issuer = ptx::elect_one();
        while (next_segment(sg)) {
            ptx::mbar_wait(acc_empty, acc_ph ^ 1u);
            ptx::tc_fence_after_sync();
            uint32_t acc = 0;
            for (int g = 0; g < sg.ngroups; ++g) {
#pragma unroll
                for (int st = 0; st < TD_PL_STAGES; ++st) {
                    ptx::mbar_wait(pl_full(st), ph);
                    ptx::tc_fence_after_sync();
                    if (issuer) {
                        const uint32_t pl = pl0 + st * TD_PL_BYTES;
                        const uint32_t a0 = TD_ACOL0 + (uint32_t)st * TD_ACOLS;
#pragma unroll
                        for (int ks = 0; ks < TD_ST / 32; ++ks) {
                            // one 128-wide MN block, 128-B swizzle, 8-row K groups 1024 B apart; K-step = 32 rows = 4096 B
                            const uint64_t dBr = make_smem_desc(pl + ks * 4096, TD_PLANE, 1024, 2);
                            const uint64_t dBi = make_smem_desc(pl + TD_PLANE + ks * 4096, TD_PLANE, 1024, 2);
                            const uint32_t a_r = a0 + 8u * ks, a_i = a0 + 16u + 8u * ks;
                            ptx::mma_i8_ts<1>(0, a_i, dBr, idesc, acc);    // IR
                            ptx::mma_i8_ts<1>(128, a_i, dBi, idesc, acc);  // II  -> Re
                            ptx::mma_i8_ts<1>(256, a_r, dBi, idesc, acc);  // RI
                            ptx::mma_i8_ts<1>(128, a_r, dBr, idesc, 1);    // RR  -> Re
                            acc = 1;
                        }
                        ptx::mma_commit<1>(pl_empty(st));
                    }
                    __syncwarp();
                }
                ph ^= 1u;
            }
            if (issuer) ptx::mma_commit<1>(acc_full);
            __syncwarp();
            acc_ph ^= 1u;
        }
    } else if (warp < TD_EPI_WARP0) {
        // ===================== S2: unpack =====================
        // Two groups of four warps take the stages alternately: what a stage costs a warp is a chain of waits and
        // latencies (barrier, ldmatrix, tcgen05.st, plane stores, fences, arrive) of more than the 512 cycles its MMAs
        // take, so each group gets two stage times for it.  Both rings have an even number of stages and a unit an even
        // number of stages: a ring position always belongs to the same group.  Warp <-> TMEM lane quarter q (hardware
        // rule); it transposes both 32-sample halves of the stage for its 32 inputs.
        static_assert(TD_PL_STAGES % 2 == 0, "operand ring positions must keep their group");
        const int q = warp & 3;
        const int grp = (warp - 2) >> 2;        // parity of the stages this warp works on
        const int gt = 32 * q + lane;           // thread of the group: 16-byte chunks gt + 128 c, c = 0..3
        // ldmatrix row address of this lane, per half kh: matrix m = lane/16, row r = lane%16 -> sample 32 kh + 16 m + r
        const int lrow = 16 * (lane >> 4) + (lane & 15);
        const uint32_t lds0 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 0) ^ (lrow & 7)) << 4);
        const uint32_t lds1 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 1) ^ (lrow & 7)) << 4);
        const int tbase = 4 * (lane & 3);       // first sample of this thread's r0/r1 inside a half (r2/r3: + 16)
        const uint32_t tdst = tmem + ((uint32_t)(32 * q) << 16) + TD_ACOL0;
        int pst = grp % PK_STAGES, qst = grp;   // ring positions of this group's next stage
        uint32_t uj = (uint32_t)grp, qph = 0;   // its number: use uj / PK_PERIOD of the (position, group) barriers
        while (next_segment(sg)) {
            const int t_begin = sg.t_begin, t_end = sg.t_end;
            const uint32_t yoff = (GENERAL && sg.bx != sg.by) ? (uint32_t)TD_PK_BYTES : 0u;   // the columns' block
            for (int t = t_begin + grp * TD_ST; t < t_begin + sg.ngroups * TD_GROUP; t += 2 * TD_ST) {
                const int rows_valid = t_end - t;  // <= 0 in a padding stage: all-zero operands
                ptx::mbar_wait(pk_full(pst, grp), (uj / PK_PERIOD) & 1u);
                const uint32_t src = pk0 + pst * PK_BYTES;
                // ---- loads first: four transposing loads (rows' planes), four 16-byte chunks (columns' planes)
                uint32_t xa[2][4], xb[2][4];
#pragma unroll
                for (int kh = 0; kh < 2; ++kh) {
                    ptx::ldsm_t_b8_x2(src + 4096u * kh + lds0, xa[kh][0], xa[kh][1], xa[kh][2], xa[kh][3]);   // inputs 32q + 0..15
                    ptx::ldsm_t_b8_x2(src + 4096u * kh + lds1, xb[kh][0], xb[kh][1], xb[kh][2], xb[kh][3]);   // inputs 32q + 16..31
                }
                uint4 wy[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) wy[c] = *reinterpret_cast<const uint4 *>(gbase + (src + yoff - base) + 2048 * c + gt * 16);
                ptx::mbar_wait(pl_empty(qst), qph ^ 1u);
                // ---- A planes -> TMEM
#pragma unroll
                for (int kh = 0; kh < 2; ++kh) {
                    // byte masks of this thread's four samples (zero beyond the slice)
                    uint32_t m0 = 0xF0F0F0F0u, m1 = 0xF0F0F0F0u;
                    if (rows_valid < TD_ST) {
                        const int v0 = min(4, max(0, rows_valid - 32 * kh - tbase)), v1 = min(4, max(0, rows_valid - 32 * kh - tbase - 16));
                        m0 = v0 ? (0xF0F0F0F0u >> (32 - 8 * v0)) : 0u;
                        m1 = v1 ? (0xF0F0F0F0u >> (32 - 8 * v1)) : 0u;
                    }
                    const uint32_t ta = tdst + (uint32_t)qst * TD_ACOLS + 8u * kh;
                    ptx::tmem_st_16x128b_x2(ta, (xa[kh][0] ^ 0x80808080u) & m0, (xa[kh][1] ^ 0x80808080u) & m0,
                                            (xa[kh][2] ^ 0x80808080u) & m1, (xa[kh][3] ^ 0x80808080u) & m1);
                    ptx::tmem_st_16x128b_x2(ta + (16u << 16), (xb[kh][0] ^ 0x80808080u) & m0, (xb[kh][1] ^ 0x80808080u) & m0,
                                            (xb[kh][2] ^ 0x80808080u) & m1, (xb[kh][3] ^ 0x80808080u) & m1);
                    ptx::tmem_st_16x128b_x2(ta + 16u, ((xa[kh][0] << 4) ^ 0x80808080u) & m0, ((xa[kh][1] << 4) ^ 0x80808080u) & m0,
                                            ((xa[kh][2] << 4) ^ 0x80808080u) & m1, ((xa[kh][3] << 4) ^ 0x80808080u) & m1);
                    ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 16u, ((xb[kh][0] << 4) ^ 0x80808080u) & m0,
                                            ((xb[kh][1] << 4) ^ 0x80808080u) & m0, ((xb[kh][2] << 4) ^ 0x80808080u) & m1,
                                            ((xb[kh][3] << 4) ^ 0x80808080u) & m1);
                }
                // ---- B planes -> shared memory, same physical offsets as the packed block (128-byte rows)
                {
                    uint8_t *dst = gbase + (pl0 - base) + qst * TD_PL_BYTES;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const uint32_t off = (uint32_t)gt * 16u + 2048u * c;
                        const uint32_t m = ((int)(off >> 7) < rows_valid) ? 0xF0F0F0F0u : 0u;
                        uint4 r, i;
                        r.x = (wy[c].x ^ 0x80808080u) & m; r.y = (wy[c].y ^ 0x80808080u) & m;
                        r.z = (wy[c].z ^ 0x80808080u) & m; r.w = (wy[c].w ^ 0x80808080u) & m;
                        i.x = ((wy[c].x << 4) ^ 0x80808080u) & m; i.y = ((wy[c].y << 4) ^ 0x80808080u) & m;
                        i.z = ((wy[c].z << 4) ^ 0x80808080u) & m; i.w = ((wy[c].w << 4) ^ 0x80808080u) & m;
                        *reinterpret_cast<uint4 *>(dst + off) = r;
                        *reinterpret_cast<uint4 *>(dst + TD_PLANE + off) = i;
                    }
                }
                ptx::fence_proxy_async_smem();   // B planes: generic-proxy writes, read by the MMA's async proxy
                ptx::tmem_st_wait();             // A planes are in TMEM
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive(pl_full(qst));
                    ptx::mbar_arrive(pk_empty(pst, grp));
                }
                uj += 2;
                pst += 2;
                if (pst >= PK_STAGES) pst -= PK_STAGES;
                qst += 2;
                if (qst >= TD_PL_STAGES) { qst -= TD_PL_STAGES; qph ^= 1u; }
            }
        }
    } else {
        // ===================== S5: epilogue =====================
        // Eight warps: warp % 4 = TMEM lane quarter q (hardware rule), h = column half.  Thread <-> row r = 32 q + lane of
        // the tile, columns 64 h .. 64 h + 63.  The accumulators are drained into a shared-memory image of the row (8
        // bytes per baseline, the layout of vis), TMEM is handed back as soon as the last tcgen05.ld has completed, and
        // the row segment leaves as ONE bulk copy (cp.async.bulk, or cp.reduce.async.bulk.add.s32 when the call adds)
        // that overlaps the next unit's main loop.  Rows of the packed triangle start on 8-byte boundaries and bulk
        // copies need 16: the image is shifted by one slot when the global address is odd in 8-byte units, and at most
        // one leading and one trailing baseline are written with ordinary stores.
        const int q = warp & 3;
        const int h = (warp - TD_EPI_WARP0) >> 2;
        const int r = 32 * q + lane;                       // row of the tile
        const int sub = p.sub;                             // 128, or 64: two channels per tile
        const int cs = (sub == 64) ? (r >> 6) : 0;         // channel of the tile this row belongs to
        const int xl0 = r - cs * sub;                      // input index inside its channel (block 0)
        const int cpt = 128 / sub;
        // image of this row.  One block per channel (!GENERAL): rows 0..63 hold 128 columns, rows 64..127 columns 64..127,
        // all at once.  GENERAL: the image has 64 rows of 128 columns; rows 0..63 of the block use it first, rows 64..127
        // once those have left (named barrier 2), and the next block's rows 0..63 once these have (named barrier 3)
        const uint32_t srow_own = GENERAL ? epi0 + (uint32_t)(r & 63) * TD_PITCH_LO
                                          : epi0 + (r < 64 ? (uint32_t)r * TD_PITCH_LO : 64u * TD_PITCH_LO + (uint32_t)(r - 64) * TD_PITCH_HI);
        const long long Bn = (long long)p.n_out * ((long long)p.n_out + 1) / 2;
        const bool add = (p.out_mode != OUT_STORE);
        const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
        uint32_t acc_ph = 0;
        bool first_segment = true;
        while (next_segment(sg)) {
            const bool diag = !GENERAL || sg.bx == sg.by;
            const int x0 = sg.bx * 128, y0 = sg.by * 128;   // first input of the rows / columns (0 unless GENERAL)
            // window mode: the channel's inputs are rows / columns wo .. wo + N - 1 of the tile (the bytes before belong to
            // the previous channel, the bytes after to the next: computed and dropped)
            // ... and with several whole channels per window (win_c > 1, small N) the row's channel is the k-th of the tile
            int xl = xl0 + x0, chan = sg.f * cpt + cs, coff = cs * sub, cend = p.n_out;
            bool win_valid = true;
            if (!GENERAL && p.win_n > 0) {
                const int wo = (sg.f * p.win_c * p.win_n) & 15;
                const int rel = r - wo;
                const int wk = rel >= 0 ? rel / p.win_n : 0;
                xl = rel - wk * p.win_n;
                chan = sg.f * p.win_c + wk;
                coff = wo + wk * p.win_n;          // tile column of the channel's input 0
                cend = wo + p.win_c * p.win_n;     // end of the tile's last channel
                win_valid = rel >= 0 && wk < p.win_c && chan < p.f_out;
            }
            const int img0 = (!GENERAL && r >= 64) ? 64 : 0;   // tile column held by slot `par` of this row's image
            // GENERAL, the CTA's last segment: nothing is loaded any more, so rows 64..127 take the packed ring as their
            // image instead of waiting for rows 0..63 to leave theirs
            const bool last = GENERAL && it >= it_end;
            static_assert(TD_EPI_BYTES_G <= TD_PK_STAGES_G * 2 * TD_PK_BYTES, "the packed ring holds an image");
            const uint32_t srow = (last && q >= 2) ? pk0 + (uint32_t)(r & 63) * TD_PITCH_LO : srow_own;
            uint8_t *srow_g = gbase + (srow - base);
            // 8-byte index in vis of (this row, tile column img0) -- formal when that column is left of the diagonal:
            // only its parity and offsets from it are used
            const long long gi0 = (long long)chan * Bn + (long long)xl * p.n_out - (long long)xl * (xl - 1) / 2 - xl + (y0 + img0 - coff);
            int2 *gimg = reinterpret_cast<int2 *>(p.vis) + gi0;
            const uint32_t par = (uint32_t)(reinterpret_cast<uintptr_t>(gimg) >> 3) & 1u;
            ptx::bulk_wait_read0();  // this thread's previous row segment has left shared memory
            if (GENERAL) {
                // rows 64..127 of the previous block have left the image (every thread has waited for its own copies)
                if (!first_segment) ptx::named_bar_sync(3, 32 * TD_EPI_WARPS);
                first_segment = false;
            }
            ptx::mbar_wait(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
            // columns this thread sends: [jlo, jhi) of the tile
            int jlo, jhi;
            if (diag) {
                jlo = max(64 * h, r);
                jhi = min(64 * h + 64, coff + p.n_out - x0);
                if (sub == 64 && h != cs) jhi = jlo;
            } else {
                jlo = 64 * h;
                jhi = min(64 * h + 64, p.n_out - y0);
            }
            const bool row_ok = win_valid && xl >= 0 && xl < p.n_out && (sub != 64 || chan < p.f_out);
            if (GENERAL && !last && q >= 2) ptx::named_bar_sync(2, 32 * TD_EPI_WARPS);   // rows 0..63 have left the image
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int col = 64 * h + 16 * c;
                // warp-uniform: the chunk is left of the diagonal for every row of the warp, outside the matrix, or
                // (two channels per tile) in the other channel's columns
                bool skip;
                if (diag) skip = (col + 15 < 32 * q) || (sub == 128 ? (x0 + col >= cend || x0 + 32 * q >= cend) : ((col >> 6) != (q >> 1)));
                else skip = (y0 + col >= p.n_out) || (x0 + 32 * q >= p.n_out);
                if (!skip) {
                    uint32_t ir[16], rr[16], ri[16];
                    ptx::tmem_ld16(trow + col, ir);
                    ptx::tmem_ld16(trow + 128 + col, rr);
                    ptx::tmem_ld16(trow + 256 + col, ri);
                    ptx::tmem_ld_wait();
                    uint8_t *dst = srow_g + 8 * ((int)par + col - img0);
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int re = (int)rr[j] >> 8;
                        const int im = (int)(ir[j] - ri[j]) >> 8;
                        *reinterpret_cast<int2 *>(dst + j * 8) = make_int2(re, im);
                    }
                }
            }
            // TMEM is free for the next unit
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(acc_empty);
            if (row_ok && jlo < jhi) {
                ptx::fence_proxy_async_smem();  // this thread's st.shared -> visible to the bulk-copy engine
                int a = jlo - img0, b = jhi - img0;   // as offsets from the image's first column
                if ((par + a) & 1) {             // leading baseline on an odd 8-byte slot
                    const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * ((int)par + a));
                    if (add) { atomicAdd(&gimg[a].x, v.x); atomicAdd(&gimg[a].y, v.y); }
                    else gimg[a] = v;
                    ++a;
                }
                if ((b - a) & 1) {               // trailing baseline
                    --b;
                    const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * ((int)par + b));
                    if (add) { atomicAdd(&gimg[b].x, v.x); atomicAdd(&gimg[b].y, v.y); }
                    else gimg[b] = v;
                }
                if (a < b) {
                    if (add) ptx::bulk_reduce_add_s32(gimg + a, srow + 8u * (par + a), 8u * (b - a));
                    else ptx::bulk_store(gimg + a, srow + 8u * (par + a), 8u * (b - a));
                }
            }
            ptx::bulk_commit();
            if (GENERAL && !last && q < 2) {     // rows 64..127 may have the image once these rows have been read
                ptx::bulk_wait_read0();
                ptx::named_bar_sync(2, 32 * TD_EPI_WARPS);
            }
        }
        ptx::bulk_wait0();  // every row segment has been written before the CTA retires
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc<1>(tmem, 512);
}

}  // namespace corr
