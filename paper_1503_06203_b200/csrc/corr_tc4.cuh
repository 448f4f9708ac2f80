// corr_tc4.cuh -- the large-N path (steps S1-S5) with THREE tensor-core products per complex
// multiply-accumulate instead of four (the paper's closing remark that a
// faster correlator needs "packed operations of some kind").
//
// Same result as every other path (Eq. 1, summed over time PAPER.md:48, upper
// triangle PAPER.md:50) and the same CTA-pair structure as corr_tc3.cuh (256 x 128 tiles,
// tcgen05.mma.cta_group::2.kind::i8, A operand in tensor memory).  What changes is the algebra.
//
// Write the stored byte of input x as w = 16 r' + i' with r' = Re + 8, i' = Im + 8 (excess-8 nibbles,
// PAPER.md:76), and (r, i) = (Re, Im) of x, (p, s) = (Re, Im) of y.  X * conj(Y) is the polynomial
// product (r + i z)(p - s z) = r p + (i p - r s) z - i s z^2: three coefficients, so three evaluations
// suffice.  Evaluating at z = 1/16, z = -1/16 and z = infinity makes every operand ONE logic
// operation (or none) away from the stored byte, read as an UNSIGNED int8 (kind::i8 takes the
// signedness of A and B from the instruction descriptor):
//     W = w          = 16 Re + Im + 136        V = w ^ 0x0F = 16 Re - Im + 135        L = w & 0x0F = Im + 8
//     P1 = sum_t W[x] V[y]        P2 = sum_t V[x] W[y]        P3 = sum_t L[x] L[y]
// The offsets are removed the paper's way (Eq. 3: operate on the stored values,
// correct with per-element sums).  With SW[n] = sum_t w[n], SL[n] = sum_t (w[n] & 15), Tv samples:
//     K[n] = SW[n] - 272 SL[n]                     R[n] = 32768 Tv - 271 SW[n] - 3840 SL[n]
//     32 Im  = P1 - P2 + K[x] - K[y]
//     512 Re = P1 + P2 + 514 P3 + R[x] + R[y]
// (derivation in DESIGN.md section 6.2), exact in int32 for slices of <= 16384 samples
// (|512 Re| <= 65536 Tv <= 2^30; P1, P2 <= 255^2 Tv < 2^31).  SW and SL come from corr_sums_kernel
// (below), one pass over the input per call (the paper's "offset accumulate" kernel).
//
// Per CTA r (= rank in the pair), packed stages of 64 time samples, operand slots of 32:
//   packed X_r  [64][128] bytes, 128-B swizzle   x in [256*bx2 + 128 r, +128)      (TMA)
//   packed Yh_r [64][ 64] bytes,  64-B swizzle   y in [128*by + 64 r, +64)          (TMA)
//   operand slot (ring of 5), 32 samples:
//     shared memory: B1 = V, B2 = W, B3 = L   [32][64] MN-major SW64 each (y-half)
//     TMEM: A1 = W | A2 = V | A3 = L           8 columns each (x-block, lane = x - x0)
// TMEM columns (per CTA, for its 128 x rows):
//     0..127  P1      128..255  P2      256..383  P3      384..503  A planes, 5 slots x 24 columns
// Only the A side is zeroed beyond the end of a slice (a zero A byte kills the product whatever B holds).
// Unpack warp group kh (4 warps) owns samples [32 kh, 32 kh + 32) of every packed stage.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode, baseline_index
#include "corr_ptx.cuh"

namespace corr {

constexpr int T4_ST = 64;              // time samples per packed (TMA) stage
constexpr int T4_KS = 32;              // time samples per operand slot = one MMA K-step
constexpr int T4_PK_STAGES = 5;        // packed-byte ring (covers TMA latency)
constexpr int T4_PL_STAGES = 5;        // operand ring: TMEM A slot + smem B slot (5 x 24 = 120 TMEM columns)
constexpr int T4_GROUP = T4_ST;        // every unit runs whole packed stages (two operand slots)
static_assert(T4_PL_STAGES == 5, "the MMA issue switch in corr_tc4_kernel is written for a ring of 5");
#ifndef T4_GROUPS_N
#define T4_GROUPS_N 4
#endif
constexpr int T4_GROUPS = T4_GROUPS_N;      // unpack warp groups of 4 warps; operand slot o belongs to group o % T4_GROUPS
constexpr int T4_UNPACK_WARPS = 4 * T4_GROUPS;
constexpr int T4_EPI_WARP0 = 2 + T4_UNPACK_WARPS;
constexpr int T4_EPI_WARPS = 8;             // two per TMEM lane quarter: column halves
constexpr int T4_THREADS = 32 * (T4_EPI_WARP0 + T4_EPI_WARPS);
constexpr int T4_XBYTES = T4_ST * 128;             // packed x-block per packed stage
constexpr int T4_YBYTES = T4_ST * 64;              // packed y-half per packed stage
constexpr int T4_PK_BYTES = T4_XBYTES + T4_YBYTES;
constexpr int T4_BPLANE = T4_KS * 64;              // one B plane of one operand slot (y-half)
constexpr int T4_PL_BYTES = 3 * T4_BPLANE;         // B1, B2, B3
constexpr int T4_EPI_PITCH = 128 * 8 + 16;        // one staged output row: 128 (Re,Im) pairs + parity slot
constexpr int T4_EPI_BYTES = 128 * T4_EPI_PITCH;  // the CTA's whole 128 x 128 output block
constexpr int T4_SMEM_BYTES = 1024 + T4_PK_STAGES * T4_PK_BYTES + T4_PL_STAGES * T4_PL_BYTES + T4_EPI_BYTES + 256;
constexpr uint32_t T4_ACOL0 = 384;                 // first TMEM column of the A slots
constexpr uint32_t T4_ACOLS = 24;                  // columns per A slot: A1 8 | A2 8 | A3 8
constexpr int T4_MAX_SLICE = 16384;                // |512 Re| <= 65536 * 16384 = 2^30

struct Tc4Params {
    int N, F, T;
    int tiles_per_f;   // pair tiles (256 x 128) touching the upper triangle, per channel
    int slices;
    int t_per_slice;   // multiple of T4_GROUP
    int num_units;     // F * tiles_per_f * slices
    int out_mode;
    const ushort2 *tiles;  // (bx2, by): x-block of 256, y-block of 128
    const int32_t *sum_w;   // [slices][F][N]  sum_t w          (corr_sums_kernel)
    const int32_t *sum_lo;  // [slices][F][N]  sum_t (w & 15)
    int32_t *vis;
};

// ---------------------------------------------------------------------------------------------
// Per-element sums of the stored bytes over every T-slice (the paper's offset-accumulate kernel,
// PAPER.md:84-91, restated for this path's operands): sum_w[s][f][n] = sum_t w, sum_lo = sum_t (w & 15).
// One thread owns 16 consecutive inputs (one 16-byte load per time sample) and SUMS_ROWS samples,
// summed in 16-bit lanes (255 * 64 < 65536); the threads of a block that share inputs are combined
// with shared-memory atomics and the block adds its totals atomically to the zeroed output.
constexpr int SUMS_THREADS = 512;
constexpr int SUMS_COLS = 256;   // 16-byte vectors a block covers at a time
constexpr int SUMS_ROWS = 64;    // samples per thread

__host__ __device__ inline int sums_rows_per_block(int N)
{
    const int nv = N >> 4, cw = nv < SUMS_COLS ? nv : SUMS_COLS;
    return SUMS_ROWS * (SUMS_THREADS / cw);
}

__global__ void __launch_bounds__(SUMS_THREADS)
corr_sums_kernel(const uint8_t *__restrict__ packed, int32_t *__restrict__ sum_w, int32_t *__restrict__ sum_lo,
                 int N, int F, int T, int t_per_slice)
{
    __shared__ int acc_w[16 * SUMS_COLS], acc_l[16 * SUMS_COLS];
    const int nv = N >> 4;                              // 16-byte vectors per (t, f) row
    const int cw = min(nv, SUMS_COLS);                  // threads along n
    const int rstep = SUMS_THREADS / cw;                // threads along t
    const bool active = (int)threadIdx.x < cw * rstep;
    const int f = blockIdx.y, slice = blockIdx.z;
    const int t_begin = slice * t_per_slice, t_end = min(T, t_begin + t_per_slice);
    const int r0 = t_begin + blockIdx.x * (SUMS_ROWS * rstep) + (int)threadIdx.x / cw;
    const int c = (int)threadIdx.x % cw;
    for (int v0 = 0; v0 < nv; v0 += cw) {
        for (int i = threadIdx.x; i < 16 * cw; i += SUMS_THREADS) { acc_w[i] = 0; acc_l[i] = 0; }
        __syncthreads();
        const int v = v0 + c;
        if (active && v < nv) {
            uint32_t we[4] = {0, 0, 0, 0}, wo[4] = {0, 0, 0, 0}, le[4] = {0, 0, 0, 0}, lo[4] = {0, 0, 0, 0};
            const uint8_t *src = packed + ((size_t)r0 * F + f) * (size_t)N + 16 * (size_t)v;
            const size_t stride = (size_t)rstep * F * N;
#pragma unroll 8
            for (int k = 0; k < SUMS_ROWS; ++k) {
                if (r0 + k * rstep < t_end) {
                    const uint4 q = __ldg(reinterpret_cast<const uint4 *>(src + k * stride));
                    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        we[j] += w[j] & 0x00FF00FFu;
                        wo[j] += (w[j] >> 8) & 0x00FF00FFu;
                        le[j] += w[j] & 0x000F000Fu;
                        lo[j] += (w[j] >> 8) & 0x000F000Fu;
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                atomicAdd(&acc_w[16 * c + 4 * j + 0], (int)(we[j] & 0xFFFFu));
                atomicAdd(&acc_w[16 * c + 4 * j + 1], (int)(wo[j] & 0xFFFFu));
                atomicAdd(&acc_w[16 * c + 4 * j + 2], (int)(we[j] >> 16));
                atomicAdd(&acc_w[16 * c + 4 * j + 3], (int)(wo[j] >> 16));
                atomicAdd(&acc_l[16 * c + 4 * j + 0], (int)(le[j] & 0xFFFFu));
                atomicAdd(&acc_l[16 * c + 4 * j + 1], (int)(lo[j] & 0xFFFFu));
                atomicAdd(&acc_l[16 * c + 4 * j + 2], (int)(le[j] >> 16));
                atomicAdd(&acc_l[16 * c + 4 * j + 3], (int)(lo[j] >> 16));
            }
        }
        __syncthreads();
        int32_t *ow = sum_w + ((size_t)slice * F + f) * N + 16 * (size_t)v0;
        int32_t *ol = sum_lo + ((size_t)slice * F + f) * N + 16 * (size_t)v0;
        const int ncol = min(16 * cw, N - 16 * v0);
        for (int i = threadIdx.x; i < ncol; i += SUMS_THREADS) {
            atomicAdd(ow + i, acc_w[i]);
            atomicAdd(ol + i, acc_l[i]);
        }
        __syncthreads();
    }
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T4_THREADS, 1)
corr_tc4_kernel(const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_y,
                const Tc4Params p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;
    const uint32_t pl0 = pk0 + T4_PK_STAGES * T4_PK_BYTES;
    const uint32_t epi0 = pl0 + T4_PL_STAGES * T4_PL_BYTES;
    const uint32_t bar0 = epi0 + T4_EPI_BYTES;
    uint8_t *epi_g = gbase + (epi0 - base);
    auto pk_full = [&](int s) { return bar0 + 8u * s; };
    auto pk_empty = [&](int s) { return bar0 + 8u * (T4_PK_STAGES + s); };
    auto pl_full = [&](int s) { return bar0 + 8u * (2 * T4_PK_STAGES + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (2 * T4_PK_STAGES + T4_PL_STAGES + s); };
    const uint32_t acc_full = bar0 + 8u * (2 * T4_PK_STAGES + 2 * T4_PL_STAGES);
    const uint32_t acc_empty = acc_full + 8u;
    const uint32_t tmem_slot = acc_empty + 8u;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();  // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap_x);
        ptx::prefetch_tmap(&tmap_y);
        for (int s = 0; s < T4_PK_STAGES; ++s) {
            ptx::mbar_init(pk_full(s), 1);
            ptx::mbar_init(pk_empty(s), 8);   // the two groups (4 warps each) that own the two halves of the stage
        }
        for (int s = 0; s < T4_PL_STAGES; ++s) {
            ptx::mbar_init(pl_full(s), 8);  // one warp group (4 warps) of BOTH CTAs; the leader's copy is used
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, 2 * T4_EPI_WARPS);
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
    if (tmem != 0) __trap();  // all 512 columns were requested: the allocation starts at lane 0, column 0

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
                const int t_pad = t_begin + (t_end - t_begin + T4_GROUP - 1) / T4_GROUP * T4_GROUP;
                for (int t = t_begin; t < t_pad; t += T4_ST) {
                    ptx::mbar_wait(pk_empty(st), ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(pk_full(st), T4_PK_BYTES);
                    const uint32_t dst = pk0 + st * T4_PK_BYTES;
                    ptx::tma_load_3d(dst, &tmap_x, pk_full(st), xc, f, t);
                    ptx::tma_load_3d(dst + T4_XBYTES, &tmap_y, pk_full(st), yc, f, t);
                    if (++st == T4_PK_STAGES) { st = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issuer (leader CTA only) =====================
        // The whole warp runs the loop (warp-uniform operands), one elected lane issues.
        if (rank == 0) {
            constexpr uint32_t idesc_uu = make_idesc_i8(256, 128, /*unsigned*/ false, false, /*A K-major (TMEM)*/ false, /*B MN-major*/ true);
            uint32_t ph = 0, acc_ph = 0;
            int st = 0;
            const bool issuer = ptx::elect_one();
            for (int u = pair; u < p.num_units; u += npairs) {
                const int rem = u % units_per_f;
                const int slice = rem % p.slices;
                const int t_begin = slice * p.t_per_slice;
                const int t_end = min(p.T, t_begin + p.t_per_slice);
                const int ngroups = (t_end - t_begin + T4_GROUP - 1) / T4_GROUP;
                ptx::mbar_wait_cluster(acc_empty, acc_ph ^ 1u);
                ptx::tc_fence_after_sync();
                uint32_t acc = 0;
                // One operand slot: wait until both CTAs have filled it, issue the three products, release it.
                // The slot index is a template constant so that every descriptor is "uniform base + constant".
                auto issue = [&](auto slot_c) {
                    constexpr int sl = decltype(slot_c)::value;
                    ptx::mbar_wait_cluster(pl_full(sl), ph);
                    ptx::tc_fence_after_sync();
                    if (issuer) {
                        const uint32_t pl = pl0 + sl * T4_PL_BYTES;
                        constexpr uint32_t a0 = T4_ACOL0 + (uint32_t)sl * T4_ACOLS;  // TMEM base is 0 (checked at start)
                        // B half per CTA: one 64-wide MN block, SW64, 8-row K groups 512 B apart
                        const uint64_t dB1 = make_smem_desc(pl, T4_BPLANE, 512, 4);
                        const uint64_t dB2 = make_smem_desc(pl + T4_BPLANE, T4_BPLANE, 512, 4);
                        const uint64_t dB3 = make_smem_desc(pl + 2 * T4_BPLANE, T4_BPLANE, 512, 4);
                        ptx::mma_i8_ts<2>(0, a0, dB1, idesc_uu, acc);         // P1 = W[x] V[y]
                        ptx::mma_i8_ts<2>(128, a0 + 8, dB2, idesc_uu, acc);   // P2 = V[x] W[y]
                        ptx::mma_i8_ts<2>(256, a0 + 16, dB3, idesc_uu, acc);  // P3 = L[x] L[y]
                        ptx::mma_commit_mcast2(pl_empty(sl), 0x3);  // operand slot of BOTH CTAs is free
                    }
                    acc = 1;
                    __syncwarp();
                };
                int n = 2 * ngroups;   // operand slots of this unit; the ring position st carries over between units
                while (n > 0) {
                    switch (st) {
                    case 0: issue(std::integral_constant<int, 0>{}); if (--n == 0) { st = 1; break; }  // fall through
                    case 1: issue(std::integral_constant<int, 1>{}); if (--n == 0) { st = 2; break; }
                    case 2: issue(std::integral_constant<int, 2>{}); if (--n == 0) { st = 3; break; }
                    case 3: issue(std::integral_constant<int, 3>{}); if (--n == 0) { st = 4; break; }
                    default: issue(std::integral_constant<int, 4>{}); --n; st = 0; ph ^= 1u;
                    }
                }
                if (issuer) ptx::mma_commit_mcast2(acc_full, 0x3);
                __syncwarp();
                acc_ph ^= 1u;
            }
        }
    } else if (warp < T4_EPI_WARP0) {
        // ===================== S2: unpack =====================
        const int q = warp & 3;                 // TMEM lane quarter this warp may write: inputs 32q..32q+31
        const int grp = (warp - 2) >> 2;        // warp group: owns operand slots o with o % T4_GROUPS == grp
        const int gt = threadIdx.x - 64 - 128 * grp;  // thread index inside the group, 0..127
        // ldmatrix row address of this lane inside a 32-sample half: matrix m = lane/16, row r = lane%16
        const int lrow = 16 * (lane >> 4) + (lane & 15);
        const uint32_t lds0 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 0) ^ (lrow & 7)) << 4);
        const uint32_t lds1 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 1) ^ (lrow & 7)) << 4);
        const uint32_t tdst = tmem + ((uint32_t)(32 * q) << 16) + T4_ACOL0;
        uint32_t ob = 0;   // operand slots of all previous units of this pair (even)
        for (int u = pair; u < p.num_units; u += npairs) {
            const int rem = u % units_per_f;
            const int slice = rem % p.slices;
            const int t_begin = slice * p.t_per_slice;
            const int t_end = min(p.T, t_begin + p.t_per_slice);
            const uint32_t nslots = 2u * (uint32_t)((t_end - t_begin + T4_GROUP - 1) / T4_GROUP);
            // first slot of this unit that belongs to this group
            uint32_t o = ob + ((uint32_t)grp + T4_GROUPS - ob % T4_GROUPS) % T4_GROUPS;
            for (; o < ob + nslots; o += T4_GROUPS) {
                const uint32_t kh = o & 1u;                  // which 32-sample half of the packed stage
                const uint32_t stg = o >> 1;                 // packed stage sequence number (all units)
                const int pst = (int)(stg % T4_PK_STAGES);
                const uint32_t pph = (stg / T4_PK_STAGES) & 1u;
                const int tbase = 32 * (int)kh + 4 * (lane & 3);  // first sample of this thread's r0/r1 (r2/r3: + 16)
                const int rows_valid = t_end - (t_begin + T4_ST * (int)((o - ob) >> 1));  // <= 0: padding stage
                const int qst = (int)(o % T4_PL_STAGES);
                const uint32_t qph = (o / T4_PL_STAGES) & 1u;
                ptx::mbar_wait(pk_full(pst), pph);
                const uint32_t src = pk0 + pst * T4_PK_BYTES;
                // ---- loads first: two transposing loads of the x-block, one 16-byte chunk of the y-half
                uint32_t xa[4], xb[4];
                ptx::ldsm_t_b8_x2(src + kh * 4096u + lds0, xa[0], xa[1], xa[2], xa[3]);   // inputs 32q + 0..15
                ptx::ldsm_t_b8_x2(src + kh * 4096u + lds1, xb[0], xb[1], xb[2], xb[3]);   // inputs 32q + 16..31
                const uint4 wy = *reinterpret_cast<const uint4 *>(gbase + (src - base) + T4_XBYTES + kh * T4_BPLANE + gt * 16);
                // ---- all three planes of both sides in registers (W is the stored byte itself)
                uint32_t av[8], al[8];   // V = w ^ 0x0F, L = w & 0x0F of xa[0..3], xb[0..3]
                if (rows_valid < T4_ST) {
                    // tail (rare): zero this thread's samples beyond the slice in all three A planes
                    const int v0 = min(4, max(0, rows_valid - tbase)), v1 = min(4, max(0, rows_valid - tbase - 16));
                    const uint32_t f0 = v0 ? (0xFFFFFFFFu >> (32 - 8 * v0)) : 0u;
                    const uint32_t f1 = v1 ? (0xFFFFFFFFu >> (32 - 8 * v1)) : 0u;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const uint32_t f = (j < 2) ? f0 : f1;
                        av[j] = (xa[j] ^ 0x0F0F0F0Fu) & f;      av[4 + j] = (xb[j] ^ 0x0F0F0F0Fu) & f;
                        al[j] = xa[j] & f & 0x0F0F0F0Fu;        al[4 + j] = xb[j] & f & 0x0F0F0F0Fu;
                        xa[j] &= f;                             xb[j] &= f;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        av[j] = xa[j] ^ 0x0F0F0F0Fu;            av[4 + j] = xb[j] ^ 0x0F0F0F0Fu;
                        al[j] = xa[j] & 0x0F0F0F0Fu;            al[4 + j] = xb[j] & 0x0F0F0F0Fu;
                    }
                }
                uint4 bv, bl;
                bv.x = wy.x ^ 0x0F0F0F0Fu; bv.y = wy.y ^ 0x0F0F0F0Fu; bv.z = wy.z ^ 0x0F0F0F0Fu; bv.w = wy.w ^ 0x0F0F0F0Fu;
                bl.x = wy.x & 0x0F0F0F0Fu; bl.y = wy.y & 0x0F0F0F0Fu; bl.z = wy.z & 0x0F0F0F0Fu; bl.w = wy.w & 0x0F0F0F0Fu;
                // every byte of the packed stage this warp needs is in registers (the logic ops above
                // consumed the loads): hand the stage back to the TMA producer before the slow part
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(pk_empty(pst));
                ptx::mbar_wait_cluster(pl_empty(qst), qph ^ 1u);
                // ---- A planes -> TMEM
                const uint32_t ta = tdst + (uint32_t)qst * T4_ACOLS;
                ptx::tmem_st_16x128b_x2(ta, xa[0], xa[1], xa[2], xa[3]);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16), xb[0], xb[1], xb[2], xb[3]);
                ptx::tmem_st_16x128b_x2(ta + 8u, av[0], av[1], av[2], av[3]);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 8u, av[4], av[5], av[6], av[7]);
                ptx::tmem_st_16x128b_x2(ta + 16u, al[0], al[1], al[2], al[3]);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 16u, al[4], al[5], al[6], al[7]);
                // ---- B planes -> shared memory, same physical offsets as the packed y-half (unmasked:
                //      the A side is zero wherever the slice has no sample)
                {
                    uint8_t *dst = gbase + (pl0 - base) + qst * T4_PL_BYTES + gt * 16;
                    *reinterpret_cast<uint4 *>(dst) = bv;                    // B1 = V
                    *reinterpret_cast<uint4 *>(dst + T4_BPLANE) = wy;        // B2 = W
                    *reinterpret_cast<uint4 *>(dst + 2 * T4_BPLANE) = bl;    // B3 = L
                }
                ptx::fence_proxy_async_smem();   // B planes: generic-proxy writes, read by the MMA's async proxy
                ptx::tmem_st_wait();             // A planes are in TMEM
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(pl_full(qst), 0);  // the leader's barrier
            }
            ob += nslots;
        }
    } else {
        // ===================== S5: epilogue =====================
        // Eight warps: warp%4 = TMEM lane quarter q (hardware rule), h = column half.  Thread <-> output
        // row x = x0 + 32 q + lane, columns y0 + 64 h .. + 63.  The accumulators are drained into a
        // shared-memory image of the row (8 bytes per baseline, the layout of vis), TMEM is handed
        // back to the MMA warp as soon as the last tcgen05.ld has completed, and the row segment
        // leaves as ONE bulk copy (cp.async.bulk, or cp.reduce.async.bulk.add.s32 when the call
        // accumulates) that overlaps the next unit's main loop.  Rows of the packed triangle start
        // on 8-byte boundaries and bulk copies need 16: the row image is shifted by one slot when the
        // global address is odd in 8-byte units, and at most one leading and one trailing baseline
        // are written with ordinary stores.
        const int q = warp & 3;
        const int h = (warp - T4_EPI_WARP0) >> 2;
        const int row = 32 * q + lane;
        const uint32_t srow = epi0 + (uint32_t)row * T4_EPI_PITCH;
        uint8_t *srow_g = epi_g + row * T4_EPI_PITCH;
        const long long Bn = (long long)p.N * ((long long)p.N + 1) / 2;
        const bool add = (p.out_mode != OUT_STORE);
        uint32_t acc_ph = 0;
        for (int u = pair; u < p.num_units; u += npairs) {
            const int f = u / units_per_f, rem = u % units_per_f;
            const ushort2 tile = p.tiles[rem / p.slices];
            const int slice = rem % p.slices;
            const int tv = min(p.T, (slice + 1) * p.t_per_slice) - slice * p.t_per_slice;  // samples in the slice
            const int x0 = tile.x * 256 + (int)rank * 128, y0 = tile.y * 128;
            const int xw = x0 + q * 32;
            const int x = x0 + row;
            // 8-byte index of (x, y0) in vis (formal when y0 < x: only its parity and offsets from it are used)
            const long long g0 = (long long)f * Bn + (long long)x * p.N - (long long)x * (x - 1) / 2 - x + y0;
            int2 *grow = reinterpret_cast<int2 *>(p.vis) + g0;
            const uint32_t par = (uint32_t)(reinterpret_cast<uintptr_t>(grow) >> 3) & 1u;
            // offset terms (header): kx = K[x], rx = R[x]; the column terms are formed per chunk below
            const size_t srow_off = ((size_t)slice * p.F + f) * (size_t)p.N;
            int kx = 0, rx = 0;
            if (x < p.N) {
                const int sw = __ldg(p.sum_w + srow_off + x), sl = __ldg(p.sum_lo + srow_off + x);
                kx = sw - 272 * sl;
                rx = 32768 * tv - 271 * sw - 3840 * sl;
            }
            ptx::bulk_wait_read0();  // this thread's previous row segment has left shared memory
            ptx::mbar_wait_cluster(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
            const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int col = 64 * h + 16 * c;
                const int yc = y0 + col;
                const bool skip = (yc + 15 < xw) || (yc >= p.N) || (xw >= p.N);  // warp-uniform
                if (!skip) {
                    uint32_t g1[16], g2[16], g3[16];
                    ptx::tmem_ld16(trow + col, g1);
                    ptx::tmem_ld16(trow + 128 + col, g2);
                    ptx::tmem_ld16(trow + 256 + col, g3);
                    // N % 16 == 0 on this path, so a 16-column chunk is entirely inside or outside [0, N)
                    const int4 *pw = reinterpret_cast<const int4 *>(p.sum_w + srow_off + yc);
                    const int4 *pl = reinterpret_cast<const int4 *>(p.sum_lo + srow_off + yc);
                    int sw[16], sl[16];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int4 a = __ldg(pw + j), b = __ldg(pl + j);
                        sw[4 * j + 0] = a.x; sw[4 * j + 1] = a.y; sw[4 * j + 2] = a.z; sw[4 * j + 3] = a.w;
                        sl[4 * j + 0] = b.x; sl[4 * j + 1] = b.y; sl[4 * j + 2] = b.z; sl[4 * j + 3] = b.w;
                    }
                    ptx::tmem_ld_wait();
                    uint8_t *dst = srow_g + 8 * (par + col);
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int ky = sw[j] - 272 * sl[j];
                        const int ry = 32768 * tv - 271 * sw[j] - 3840 * sl[j];
                        const int re = (int)(g1[j] + g2[j] + 514u * g3[j] + (uint32_t)rx + (uint32_t)ry) >> 9;
                        const int im = (int)(g1[j] - g2[j] + (uint32_t)kx - (uint32_t)ky) >> 5;
                        *reinterpret_cast<int2 *>(dst + j * 8) = make_int2(re, im);
                    }
                }
            }
            // TMEM is free for the next unit
            ptx::tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_cluster(acc_empty, 0);
            // ---- write the row segment [jlo, jhi) of this thread
            int jlo = max(64 * h, x - y0), jhi = min(64 * h + 64, p.N - y0);
            if (x < p.N && jlo < jhi) {
                ptx::fence_proxy_async_smem();  // this thread's st.shared -> visible to the bulk-copy engine
                if ((par + jlo) & 1) {           // leading baseline on an odd 8-byte slot
                    const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (par + jlo));
                    if (add) { atomicAdd(&grow[jlo].x, v.x); atomicAdd(&grow[jlo].y, v.y); }
                    else grow[jlo] = v;
                    ++jlo;
                }
                if ((jhi - jlo) & 1) {           // trailing baseline
                    --jhi;
                    const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (par + jhi));
                    if (add) { atomicAdd(&grow[jhi].x, v.x); atomicAdd(&grow[jhi].y, v.y); }
                    else grow[jhi] = v;
                }
                if (jlo < jhi) {
                    if (add) ptx::bulk_reduce_add_s32(grow + jlo, srow + 8u * (par + jlo), 8u * (jhi - jlo));
                    else ptx::bulk_store(grow + jlo, srow + 8u * (par + jlo), 8u * (jhi - jlo));
                }
            }
            ptx::bulk_commit();
        }
        ptx::bulk_wait0();  // every row segment has been written before the CTA retires
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();  // no CTA of the pair may exit while its peer still reads its smem / barriers
    if (warp == 1) ptx::tmem_dealloc<2>(tmem, 512);
}

}  // namespace corr
