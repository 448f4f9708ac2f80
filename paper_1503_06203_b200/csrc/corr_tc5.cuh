// corr_tc5.cuh -- the large-N path (steps S1-S5) with THREE tensor-core products per complex
// multiply-accumulate and NO separate pass over the input (SURVEY section 8(f) ranks 1 + 2; the paper's
// closing remark that a faster correlator needs "packed operations of some kind", and its
// device of working on the stored values and correcting with per-element sums, Eq. 3).
//
// Same result as every other path (Eq. 1, summed over time PAPER.md:48, upper triangle
// PAPER.md:50), same CTA-pair tiles, tile table and schedule as corr_tc3.cuh (256 x 128 pair tiles incl.
// transposed left-over tiles, whole waves + stream-K tail, tc3_next_segment / tc3_claim_store are reused).
//
// Algebra.  Stored byte w = 16 r' + i', r' = Re + 8, i' = Im + 8, read as
// UNSIGNED int8:     W = w        V = w ^ 0x0F        L = w & 0x0F
//     P1 = sum_t W[x] V[y]        P2 = sum_t V[x] W[y]        P3 = sum_t L[x] L[y]
// With SW[n] = sum_t w[n], SL[n] = sum_t (w[n] & 15) over the Tv samples of a segment,
//     K[n] = SW[n] - 272 SL[n]                     R[n] = -271 SW[n] - 3840 SL[n]
//     32 Im  = P1 - P2 + K[x] - K[y]
//     512 Re = P1 + P2 + 514 P3 + R[x] + R[y] + 65536 Tv
// exact in int32 for segments of <= 16384 samples.
//
// How it is built, and why (profiles/r02_tc5_ncu_summary.md has the counters behind every sentence):
//   * The y-half is read with the same transposing ldmatrix as the x-block, so every unpack register holds four
//     TIME-consecutive bytes of one input on BOTH sides: the per-element sums SW, SL are one __dp4a(w, 0x01010101)
//     and one on (w & 0x0F0F0F0F) per register, accumulated in registers over a segment and handed to the epilogue
//     through shared memory (the y-half sums also to the peer CTA, red.shared::cluster + release / acquire at
//     cluster scope).  There is no sums kernel and no second pass over the input (round 1's corr_tc4 had one: 50 us);
//     cut (stream-K) units get the sums of exactly their own samples for free.
//   * V, W and L of the y-half are stored K-major (no swizzle, core matrices of 8 inputs x 16 samples): the
//     transposed registers go out as 4-byte stores, 128 contiguous bytes per warp instruction, and the three MMAs
//     of a slot share one instruction descriptor.
//   * Operand slots of 32 samples (one K-step, 192 tensor cycles), a ring of 4 slots, four groups of four unpack
//     warps, group g owning ring entry g.  A group of 256 samples is exactly two turns of the ring, so every ring
//     position in the MMA issue loop is a compile-time constant and every descriptor a loop-invariant uniform
//     register: with run-time ring indices the issuing warp needed ~430 cycles per slot, with compile-time indices
//     but ten unrolled phases ~390 (the descriptors then live in ordinary registers and are moved to uniform
//     registers one by one).
//   * Four epilogue warps (a thread owns a whole row of the block): 22 warps leave 88 registers per thread, which
//     the unpack loop needs to keep its loop invariants out of the loop (at 72 it recomputed them from the thread
//     index every iteration: 176 instructions per slot and sub-partition against the 192 cycles of the MMAs).
//   * The epilogue's row image has a pitch of 129 (Re,Im) slots (conflict-free 8-byte stores).
// Where it stands: bit-exact, 0.95 - 0.97 of corr_tc3_kernel on cfg 3.  The three-product scheme moves the same
// bytes through shared memory per 32 samples as the four-product one (TMA 48 + ldmatrix 48 + plane stores 48 +
// tensor-core reads 48 wavefronts per CTA) in 192 instead of 256 tensor cycles: the shared-memory data pipe is at
// 81 % of its cycles with the tensor pipe at 65 %, and a run with the TMA loads switched off (no writes into shared
// memory) is 23 % faster.  Reading W of the y-half straight from the TMA ring (B2 = the stored byte, MN-major) saves
// 16 of the 192 wavefronts but ties that ring to the MMAs' completion (its own 8-stage ring, a two-phase issue loop,
// two instruction descriptors per slot): built on this same kernel and measured, 333 against 306 us.  So W is stored
// like V and L, and corr_tc3_kernel stays the default.
//
// Rings (per CTA r of the pair):
//   packed ring  T5_PK stages of 64 samples: X_r [64 t][128 x] 128-B swizzle | Yh_r [64 t][64 y] 64-B swizzle (TMA),
//                freed by the unpack warps as soon as the bytes are in registers
//   V|W|L ring   4 slots of 32 samples: three planes [64 y][32 t] K-major, 2 KB each, freed by tcgen05.commit
//   TMEM         0..127 P1   128..255 P2   256..383 P3   384..479 A slots, 4 x (W 8 | V 8 | L 8 columns)
// Unpack warp group g (4 warps: TMEM lane quarters) fills the operand slots o with o % 4 == g.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode
#include "corr_ptx.cuh"
#include "corr_tc3.cuh"   // Tc3Params, tc3_next_segment, tc3_claim_store, tile flags

namespace corr {

constexpr int T5_ST = 64;              // time samples per TMA stage
constexpr int T5_KS = 32;              // time samples per operand slot = one MMA K-step
#ifndef T5_PK_N
#define T5_PK_N 5
#endif
constexpr int T5_PK = T5_PK_N;         // packed-byte ring depth (TMA stages)
constexpr int T5_SLOTS = 4;            // operand ring: TMEM A slot + smem V|W|L slot; slot o lives in entry o % 4
constexpr int T5_GROUPS = 4;           // unpack warp groups: group g fills the slots o with o % 4 == g, i.e. ring entry g
constexpr int T5_UNPACK_WARPS = 4 * T5_GROUPS;
constexpr int T5_EPI_WARP0 = 2 + T5_UNPACK_WARPS;
constexpr int T5_EPI_WARPS = 4;              // one per TMEM lane quarter: a thread owns a whole row of the block
constexpr int T5_THREADS = 32 * (T5_EPI_WARP0 + T5_EPI_WARPS);
constexpr int T5_XBYTES = T5_ST * 128;
constexpr int T5_YBYTES = T5_ST * 64;
constexpr int T5_PK_BYTES = T5_XBYTES + T5_YBYTES;
constexpr int T5_BPLANE = T5_KS * 64;              // one B plane of one slot (y-half): 2 KB
constexpr int T5_VWL_BYTES = 3 * T5_BPLANE;        // V | W | L
constexpr int T5_EPI_PITCH = 129 * 8;              // 128 (Re,Im) pairs + one alignment slot; 258 words: conflict-free
constexpr int T5_EPI_BYTES = 128 * T5_EPI_PITCH;
constexpr int T5_SUMS_BYTES = 2 * 256 * 8;         // [2 buffers][128 rows + 128 columns] (K, R)
constexpr int T5_SMEM_BYTES =
    1024 + T5_PK * T5_PK_BYTES + T5_SLOTS * T5_VWL_BYTES + T5_EPI_BYTES + T5_SUMS_BYTES + 512;
static_assert(T5_SMEM_BYTES <= 232448, "corr_tc5_kernel: shared memory budget");
constexpr uint32_t T5_ACOL0 = 384;
constexpr uint32_t T5_ACOLS = 24;
constexpr int T5_MAX_SLICE = 16384;                // |512 Re| <= 65536 * 16384 = 2^30
static_assert(T3_GROUP == 8 * T5_KS && T5_SLOTS == 4, "a group of stages is 8 operand slots = two turns of the slot ring");

namespace ptx {
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
}
// Arrive with release at cluster scope on the barrier at this offset in CTA `cta`: orders this warp's earlier
// (local and remote) shared-memory updates before the arrival.  Used once per segment, not in the inner loop.
__device__ __forceinline__ void mbar_arrive_release_cluster(uint32_t bar, uint32_t cta)
{
    asm volatile(
        "{\n\t"
        ".reg .b32 ra;\n\t"
        "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
        "mbarrier.arrive.release.cluster.shared::cluster.b64 _, [ra];\n\t"
        "}\n" ::"r"(bar), "r"(cta)
        : "memory");
}
__device__ __forceinline__ void mbar_wait_acquire_cluster(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.b32 %0, 1, 0, p;\n\t"
            "}\n"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
// Integer add into the shared memory of CTA `cta` of the cluster (same offset as `addr` here).
__device__ __forceinline__ void red_add_cluster(uint32_t addr, uint32_t cta, int v)
{
    asm volatile(
        "{\n\t"
        ".reg .b32 ra;\n\t"
        "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
        "red.relaxed.cluster.shared::cluster.add.s32 [ra], %2;\n\t"
        "}\n" ::"r"(addr), "r"(cta), "r"(v)
        : "memory");
}
__device__ __forceinline__ void sts32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
}  // namespace ptx

__device__ __forceinline__ uint64_t t5_desc(uint32_t lo, uint32_t hi) { return ((uint64_t)hi << 32) | lo; }

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T5_THREADS, 1)
corr_tc5_kernel(const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_y,
                const Tc3Params p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;                                   // packed ring: X block | Y half per stage
    const uint32_t vl0 = pk0 + T5_PK * T5_PK_BYTES;              // V|W|L ring
    const uint32_t epi0 = vl0 + T5_SLOTS * T5_VWL_BYTES;
    const uint32_t sum0 = epi0 + T5_EPI_BYTES;
    const uint32_t bar0 = sum0 + T5_SUMS_BYTES;
    uint8_t *epi_g = gbase + (epi0 - base);
    int2 *sums_g = reinterpret_cast<int2 *>(gbase + (sum0 - base));   // [2][256] (K, R)
    // packed ring: one pair of barriers per (position, parity of the stage).  The stages go alternately to the unpack groups
    // {0, 1} and {2, 3}; with an odd number of positions a pair of groups comes back to a position only every second time
    // round and, on a barrier per position, would always wait for the same parity: when TMA loads complete out of order
    // it could take the other pair's not-yet-landed stage for its own (the hazard found in corr_imma_kernel,
    // profiles/r02_secondary_kernels.md).  A (position, parity) pair is used once every T5_PK_PERIOD stages.
    constexpr int T5_PK_PERIOD = (T5_PK % 2 == 0) ? T5_PK : 2 * T5_PK;
    auto pk_full = [&](int s, int par) { return bar0 + 8u * (2 * s + par); };
    auto pk_empty = [&](int s, int par) { return bar0 + 8u * (2 * T5_PK + 2 * s + par); };
    auto pl_full = [&](int s) { return bar0 + 8u * (4 * T5_PK + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (4 * T5_PK + T5_SLOTS + s); };
    const uint32_t acc_full = bar0 + 8u * (4 * T5_PK + 2 * T5_SLOTS);
    const uint32_t acc_empty = acc_full + 8u;
    auto sums_full = [&](int b) { return acc_empty + 8u + 8u * b; };
    const uint32_t tmem_slot = acc_empty + 24u;
    static_assert(8 * (4 * T5_PK + 2 * T5_SLOTS) + 48 <= 512, "barrier area");
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));
    volatile int *claim_g = reinterpret_cast<volatile int *>(gbase + (tmem_slot + 8u - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();  // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap_x);
        ptx::prefetch_tmap(&tmap_y);
        for (int s = 0; s < T5_PK; ++s) {
            for (int par = 0; par < 2; ++par) {
                ptx::mbar_init(pk_full(s, par), 1);
                ptx::mbar_init(pk_empty(s, par), 8);   // the two warp groups that own the two halves of the stage
            }
        }
        for (int s = 0; s < T5_SLOTS; ++s) {
            ptx::mbar_init(pl_full(s), 8);        // one warp group of BOTH CTAs; the leader's copy is used
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, 2 * T5_EPI_WARPS);
        ptx::mbar_init(sums_full(0), 2 * T5_UNPACK_WARPS);   // every unpack warp of both CTAs
        ptx::mbar_init(sums_full(1), 2 * T5_UNPACK_WARPS);
        ptx::fence_mbar_init();
    }
    for (int i = threadIdx.x; i < 2 * 256; i += T5_THREADS) sums_g[i] = make_int2(0, 0);
    if (warp == 1) {
        ptx::tmem_alloc<2>(tmem_slot, 512);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();
    ptx::tc_fence_after_sync();
    const uint32_t tmem = *tmem_slot_g;
    if (tmem != 0) __trap();  // all 512 columns were requested: the allocation starts at lane 0, column 0

    Tc3Iter sit = tc3_iter(p, pair, npairs);   // every role walks the same list of segments
    Tc3Seg sg;

    if (warp == 0) {
        // ===================== S1: TMA producer (each CTA loads its own blocks) =====================
        if (lane == 0) {
            int st = 0;
            uint32_t pj = 0;   // stages loaded so far: stage pj goes to position pj % T5_PK and to the groups of parity pj & 1
            while (tc3_next_segment(p, sit, sg)) {
                const int f = sg.f;
                const ushort4 tile = sg.tile;
                const int t_begin = sg.t_begin;
                const int xc = (int)(rank ? tile.y : tile.x) * 128;   // TC3_NO_BLOCK: out of bounds, TMA fills zeros
                const int yc = tile.z * 128 + (int)rank * 64;
                const int t_pad = t_begin + sg.cnt * T3_GROUP;
                for (int t = t_begin; t < t_pad; t += T5_ST) {
                    if (pj >= (uint32_t)T5_PK) {   // the position's last stage, pj - T5_PK, has been read by its groups
                        const uint32_t jp = pj - T5_PK;
                        ptx::mbar_wait(pk_empty(st, (int)(jp & 1u)), (jp / T5_PK_PERIOD) & 1u);
                    }
                    const uint32_t dst = pk0 + st * T5_PK_BYTES;
                    const int par = (int)(pj & 1u);
                    ptx::mbar_arrive_expect_tx(pk_full(st, par), T5_PK_BYTES);
                    ptx::tma_load_3d(dst, &tmap_x, pk_full(st, par), xc, f, t);
                    ptx::tma_load_3d(dst + T5_XBYTES, &tmap_y, pk_full(st, par), yc, f, t);
                    ++pj;
                    if (++st == T5_PK) st = 0;
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issuer (leader CTA only) =====================
        // One warp issues three MMAs (192 tensor cycles) per operand slot, so the issue loop itself must stay well
        // below that (a version with run-time ring indices took ~430 cycles per slot, one with compile-time indices
        // but ten unrolled phases ~390: ptxas kept the descriptors in ordinary registers and moved them to uniform
        // registers one by one).  Here a group of 256 samples = 8 slots = exactly two turns of the slot ring, so the
        // body below is the same for every group: every descriptor is a loop-invariant uniform register, as in
        // corr_tc3.cuh.  All three B planes are K-major, so the MMAs of a slot share one instruction descriptor.
        if (rank == 0) {
            constexpr uint32_t idesc_k = make_idesc_i8(256, 128, false, false, false, false);   // unsigned x unsigned
            // K-major, no swizzle: core matrices (8 inputs x 16 samples) 128 B apart along K (LBO), 256 B along N (SBO)
            constexpr uint32_t k_lo = (128u >> 4) << 16, k_hi = (256u >> 4) | (1u << 14);
            uint32_t acc_ph = 0;
            const bool issuer = ptx::elect_one();
            const uint32_t vlo = (vl0 >> 4) + k_lo;
            while (tc3_next_segment(p, sit, sg)) {
                ptx::mbar_wait_cluster(acc_empty, acc_ph ^ 1u);
                ptx::tc_fence_after_sync();
                uint32_t acc = 0;
                for (int g = 0; g < sg.cnt; ++g) {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int slot = j & 3;
                        ptx::mbar_wait_cluster(pl_full(slot), (uint32_t)(j >> 2));
                        ptx::tc_fence_after_sync();
                        if (issuer) {
                            const uint32_t a0 = T5_ACOL0 + (uint32_t)slot * T5_ACOLS;  // TMEM base is 0 (checked at start)
                            const uint32_t v = vlo + (uint32_t)(slot * (T5_VWL_BYTES >> 4));
                            ptx::mma_i8_ts<2>(0, a0, t5_desc(v, k_hi), idesc_k, acc);                                 // P1 = W[x] V[y]
                            ptx::mma_i8_ts<2>(128, a0 + 8, t5_desc(v + (T5_BPLANE >> 4), k_hi), idesc_k, acc);       // P2 = V[x] W[y]
                            ptx::mma_i8_ts<2>(256, a0 + 16, t5_desc(v + 2 * (T5_BPLANE >> 4), k_hi), idesc_k, acc);  // P3 = L[x] L[y]
                            ptx::mma_commit_mcast2(pl_empty(slot), 0x3);   // operand slot of BOTH CTAs is free
                        }
                        acc = 1;
                        __syncwarp();
                    }
                }
                if (issuer) ptx::mma_commit_mcast2(acc_full, 0x3);
                __syncwarp();
                acc_ph ^= 1u;
            }
        }
    } else if (warp < T5_EPI_WARP0) {
        // ===================== S2: unpack =====================
        // The loop below is issue-bound (one warp-iteration per operand slot and SM sub-partition), so everything that
        // does not depend on the iteration is kept in registers and the ring positions are stepped, not recomputed.
        const int q = warp & 3;                 // TMEM lane quarter this warp may write: inputs 32q..32q+31
        const int grp = (warp - 2) >> 2;        // warp group: operand slots o with o % 4 == grp
        const uint32_t kh = (uint32_t)grp & 1u; // which half of a TMA stage this group's slots are (o % 2 == grp % 2)
        // ldmatrix row address of this lane inside a 32-sample half: matrix m = lane/16, row r = lane%16
        const int lrow = 16 * (lane >> 4) + (lane & 15);
        // x-block: rows of 128 B, chunks 2q (inputs 32q..+15) and 2q+1 (= address ^ 16), 128-B swizzle
        const uint32_t xinv = pk0 + kh * 4096u + (uint32_t)lrow * 128u + ((uint32_t)((2 * q) ^ (lrow & 7)) << 4);
        // y-half: rows of 64 B, 16-byte chunk q, 64-B swizzle (chunk ^= (row / 2) % 4; a 32-row half keeps the pattern)
        const uint32_t yinv = pk0 + T5_XBYTES + kh * 2048u + (uint32_t)lrow * 64u + ((uint32_t)(q ^ ((lrow >> 1) & 3)) << 4);
        // this group's ring entry (TMEM A slot + V|W|L slot) is always entry grp
        const uint32_t ta = tmem + ((uint32_t)(32 * q) << 16) + T5_ACOL0 + (uint32_t)grp * T5_ACOLS;
        // K-major store offsets of this thread's four y-half registers: y = 16 q + lane / 4 (+ 8), k = 4 (lane % 4) (+ 16)
        const uint32_t vdst = vl0 + (uint32_t)grp * T5_VWL_BYTES + 512u * (uint32_t)q + 4u * (uint32_t)lane;
        const uint32_t my_full = pl_full(grp), my_empty = pl_empty(grp);
        const int tb = 4 * (lane & 3);          // first sample of r0 / r1 inside the slot (r2 / r3: + 16)
        // ring positions of this group's next slot o = grp, grp + 4, ... (segments hold multiples of 8 slots)
        int st = (grp >> 1) % T5_PK;
        const int spar = grp >> 1;              // parity of the stages this group reads
        const int st0 = st;                     // the walk st, st + 2, ... (mod T5_PK) is back here after T5_PK_PERIOD stages:
        uint32_t sph = 0, pph = 0;              // that is when the phase of this group's (position, parity) barriers flips
        const uint32_t pkb = bar0 + 8u * (uint32_t)spar;   // pk_full(s, spar) = pkb + 16 s,  pk_empty(s, spar) = pkb + 16 (T5_PK + s)
        static_assert(T5_PK % 2 == 1, "an even ring: the walk returns after T5_PK / 2 steps and st0 marks that as well");
        int seg_no = 0;
        while (tc3_next_segment(p, sit, sg)) {
            const int nslots = sg.cnt * (T3_GROUP / T5_KS);
            int valid = sg.t_end - sg.t_begin - T5_KS * grp;   // samples of the next slot inside the slice (<= 0: padding)
            uint32_t sxw[4] = {0, 0, 0, 0}, sxl[4] = {0, 0, 0, 0};   // x inputs 32 q + lane / 4 + 8 j
            uint32_t syw[2] = {0, 0}, syl[2] = {0, 0};            // y inputs 16 q + lane / 4 + 8 j of this CTA's half
            for (int j = grp; j < nslots; j += T5_GROUPS, valid -= T5_KS * T5_GROUPS) {
                ptx::mbar_wait(pkb + 16u * (uint32_t)st, pph);
                uint32_t xa[4], xb[4], ya[4];
                const uint32_t xsrc = xinv + (uint32_t)st * T5_PK_BYTES;
                ptx::ldsm_t_b8_x2(xsrc, xa[0], xa[1], xa[2], xa[3]);         // inputs 32q + 0..15
                ptx::ldsm_t_b8_x2(xsrc ^ 16u, xb[0], xb[1], xb[2], xb[3]);   // inputs 32q + 16..31
                ptx::ldsm_t_b8_x2(yinv + (uint32_t)st * T5_PK_BYTES, ya[0], ya[1], ya[2], ya[3]);
                uint32_t f0 = 0xFFFFFFFFu, f1 = 0xFFFFFFFFu;
                if (valid < T5_KS) {
                    // tail (rare): zero this thread's samples beyond the slice.  W and L of the x side and the y-half
                    // registers are masked here; V of the x side below (V = 0 ^ 0x0F is not zero)
                    const int v0 = min(4, max(0, valid - tb)), v1 = min(4, max(0, valid - tb - 16));
                    f0 = v0 ? (0xFFFFFFFFu >> (32 - 8 * v0)) : 0u;
                    f1 = v1 ? (0xFFFFFFFFu >> (32 - 8 * v1)) : 0u;
                    xa[0] &= f0; xa[1] &= f0; xa[2] &= f1; xa[3] &= f1;
                    xb[0] &= f0; xb[1] &= f0; xb[2] &= f1; xb[3] &= f1;
                    ya[0] &= f0; ya[1] &= f0; ya[2] &= f1; ya[3] &= f1;
                }
                uint32_t al[8], yl[4];
#pragma unroll
                for (int k = 0; k < 4; ++k) { al[k] = xa[k] & 0x0F0F0F0Fu; al[4 + k] = xb[k] & 0x0F0F0F0Fu; yl[k] = ya[k] & 0x0F0F0F0Fu; }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(pkb + 16u * (uint32_t)(T5_PK + st));   // every byte this warp needs is in registers
                ptx::mbar_wait_cluster(my_empty, sph ^ 1u);
                ptx::tmem_st_16x128b_x2(ta, xa[0], xa[1], xa[2], xa[3]);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16), xb[0], xb[1], xb[2], xb[3]);
                ptx::tmem_st_16x128b_x2(ta + 8u, (xa[0] ^ 0x0F0F0F0Fu) & f0, (xa[1] ^ 0x0F0F0F0Fu) & f0,
                                        (xa[2] ^ 0x0F0F0F0Fu) & f1, (xa[3] ^ 0x0F0F0F0Fu) & f1);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 8u, (xb[0] ^ 0x0F0F0F0Fu) & f0, (xb[1] ^ 0x0F0F0F0Fu) & f0,
                                        (xb[2] ^ 0x0F0F0F0Fu) & f1, (xb[3] ^ 0x0F0F0F0Fu) & f1);
                ptx::tmem_st_16x128b_x2(ta + 16u, al[0], al[1], al[2], al[3]);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 16u, al[4], al[5], al[6], al[7]);
                // ---- y-half: V, W and L planes K-major into the slot
                {
                    // r0: (y, k) -> +0;  r1: y + 8 -> next 8-input group (+256);  r2, r3: k + 16 -> next core matrix (+128)
                    ptx::sts32(vdst, ya[0] ^ 0x0F0F0F0Fu);
                    ptx::sts32(vdst + 256u, ya[1] ^ 0x0F0F0F0Fu);
                    ptx::sts32(vdst + 128u, ya[2] ^ 0x0F0F0F0Fu);
                    ptx::sts32(vdst + 384u, ya[3] ^ 0x0F0F0F0Fu);
                    ptx::sts32(vdst + T5_BPLANE, ya[0]);
                    ptx::sts32(vdst + T5_BPLANE + 256u, ya[1]);
                    ptx::sts32(vdst + T5_BPLANE + 128u, ya[2]);
                    ptx::sts32(vdst + T5_BPLANE + 384u, ya[3]);
                    ptx::sts32(vdst + 2 * T5_BPLANE, yl[0]);
                    ptx::sts32(vdst + 2 * T5_BPLANE + 256u, yl[1]);
                    ptx::sts32(vdst + 2 * T5_BPLANE + 128u, yl[2]);
                    ptx::sts32(vdst + 2 * T5_BPLANE + 384u, yl[3]);
                    ptx::fence_proxy_async_smem();   // V, W, L: generic-proxy writes, read by the MMA's async proxy
                    // ---- sums (while the stores drain)
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        syw[k & 1] = __dp4a(ya[k], 0x01010101u, syw[k & 1]);
                        syl[k & 1] = __dp4a(yl[k], 0x01010101u, syl[k & 1]);
                        sxw[k & 1] = __dp4a(xa[k], 0x01010101u, sxw[k & 1]);
                        sxw[2 + (k & 1)] = __dp4a(xb[k], 0x01010101u, sxw[2 + (k & 1)]);
                        sxl[k & 1] = __dp4a(al[k], 0x01010101u, sxl[k & 1]);
                        sxl[2 + (k & 1)] = __dp4a(al[4 + k], 0x01010101u, sxl[2 + (k & 1)]);
                    }
                }
                ptx::tmem_st_wait();             // A planes are in TMEM
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(my_full, 0);  // the leader's barrier
                // next slot of this group: o += 4 (two stages on, the same ring entry)
                sph ^= 1u;
                st += 2; if (st >= T5_PK) st -= T5_PK;
                if (st == st0) pph ^= 1u;
            }
            // ---- the sums of this segment: reduce over the four lanes that share an input, then into the segment's
            //      buffer (x rows: own CTA; y columns: both CTAs of the pair)
            {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    sxw[k] += __shfl_xor_sync(0xFFFFFFFFu, sxw[k], 1); sxw[k] += __shfl_xor_sync(0xFFFFFFFFu, sxw[k], 2);
                    sxl[k] += __shfl_xor_sync(0xFFFFFFFFu, sxl[k], 1); sxl[k] += __shfl_xor_sync(0xFFFFFFFFu, sxl[k], 2);
                }
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    syw[k] += __shfl_xor_sync(0xFFFFFFFFu, syw[k], 1); syw[k] += __shfl_xor_sync(0xFFFFFFFFu, syw[k], 2);
                    syl[k] += __shfl_xor_sync(0xFFFFFFFFu, syl[k], 1); syl[k] += __shfl_xor_sync(0xFFFFFFFFu, syl[k], 2);
                }
                const int buf = seg_no & 1;
                const int sel = lane & 3;           // lane sel of a quad sends input sel of the quad's four x inputs
                const int sw = (int)(sel == 0 ? sxw[0] : sel == 1 ? sxw[1] : sel == 2 ? sxw[2] : sxw[3]);
                const int sl = (int)(sel == 0 ? sxl[0] : sel == 1 ? sxl[1] : sel == 2 ? sxl[2] : sxl[3]);
                int *dx = reinterpret_cast<int *>(sums_g + buf * 256 + 32 * q + (lane >> 2) + 8 * sel);
                atomicAdd(dx, sw - 272 * sl);
                atomicAdd(dx + 1, -271 * sw - 3840 * sl);
                if (sel < 2) {                      // lanes 0, 1 of a quad: the two y inputs
                    const int yw = (int)(sel ? syw[1] : syw[0]), yl = (int)(sel ? syl[1] : syl[0]);
                    const int col = 128 + 64 * (int)rank + 16 * q + (lane >> 2) + 8 * sel;
                    const int kv = yw - 272 * yl, rv = -271 * yw - 3840 * yl;
                    atomicAdd(reinterpret_cast<int *>(sums_g + buf * 256 + col), kv);
                    atomicAdd(reinterpret_cast<int *>(sums_g + buf * 256 + col) + 1, rv);
                    const uint32_t ra = sum0 + 8u * (uint32_t)(buf * 256 + col);
                    ptx::red_add_cluster(ra, rank ^ 1u, kv);
                    ptx::red_add_cluster(ra + 4u, rank ^ 1u, rv);
                }
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive_release_cluster(sums_full(buf), 0);
                    ptx::mbar_arrive_release_cluster(sums_full(buf), 1);
                }
            }
            ++seg_no;
        }
    } else {
        // ===================== S5: epilogue =====================
        // Four warps: warp % 4 = TMEM lane quarter q.  Thread <-> MMA row 32 q + lane, all 128 columns (the register
        // budget of the unpack warps, 88 per thread, is what limits the CTA to 22 warps).  Normal tiles: the row segment is staged in shared memory in the layout of vis and leaves
        // as one bulk copy (see corr_tc3.cuh); transposed tiles write conjugated values straight from registers.
        const int q = warp & 3;
        const int row = 32 * q + lane;
        const uint32_t srow = epi0 + (uint32_t)row * T5_EPI_PITCH;
        uint8_t *srow_g = epi_g + row * T5_EPI_PITCH;
        const long long Bn = (long long)p.N * ((long long)p.N + 1) / 2;
        const bool base_add = (p.out_mode != OUT_STORE);
        uint32_t acc_ph = 0;
        int seg_no = 0;
        while (tc3_next_segment(p, sit, sg)) {
            const bool claim = !base_add && (sg.cnt != sg.len);   // a piece of a cut unit in a call that overwrites
            bool add = base_add, raise_flag = false;
            int *flag = p.flags + 2 * sg.u + (int)rank;
            const int f = sg.f;
            const ushort4 tile = sg.tile;
            const int x0 = (int)(rank ? tile.y : tile.x) * 128, y0 = tile.z * 128;   // rows and columns of the MMA
            const int xw = x0 + q * 32;
            const int x = x0 + row;
            const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
            const int tv = min(sg.t_end, sg.t_begin + sg.cnt * T3_GROUP) - sg.t_begin;   // samples of this segment
            const int buf = seg_no & 1;
            const int2 *sums_b = sums_g + buf * 256;
            const bool transposed = (tile.w & TC3_TILE_TRANSPOSED) != 0;
            // 8-byte index of (x, y0) in vis (formal when y0 < x: only its parity and offsets from it are used)
            const long long g0 = (long long)f * Bn + (long long)x * p.N - (long long)x * (x - 1) / 2 - x + y0;
            int2 *grow = reinterpret_cast<int2 *>(p.vis) + g0;
            // alignment slot: global (g0 + j) and shared (row * 129 + sh + j) 8-byte indices must have the same parity
            const uint32_t sh = ((uint32_t)(reinterpret_cast<uintptr_t>(grow) >> 3) ^ (uint32_t)row) & 1u;
            if (!transposed) ptx::bulk_wait_read0();  // this thread's previous row segment has left shared memory
            ptx::mbar_wait_cluster(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
            ptx::mbar_wait_acquire_cluster(sums_full(buf), (uint32_t)(seg_no >> 1) & 1u);
            const int2 sx = sums_b[row];
            const int kx = sx.x, rx = sx.y + 65536 * tv;
            if (transposed) {
                // ---- this thread's MMA row is the baseline's y, the MMA columns are its x: vis(x', y') = conj(D[y'][x'])
                if (claim) add = !tc3_claim_store(flag, claim_g, 32 * T5_EPI_WARP0, 32 * T5_EPI_WARPS), raise_flag = !add;
                const int yt = x;
#pragma unroll 1
                for (int c = 0; c < 16; ++c) {
                    const int col = 8 * c;
                    const int xt0 = y0 + col;
                    const bool skip = (xt0 > xw + 31) || (xt0 >= p.N) || (xw >= p.N);  // warp-uniform
                    if (!skip) {
                        uint32_t g1[8], g2[8], g3[8];
                        ptx::tmem_ld8(trow + col, g1);
                        ptx::tmem_ld8(trow + 128 + col, g2);
                        ptx::tmem_ld8(trow + 256 + col, g3);
                        const int4 *ps = reinterpret_cast<const int4 *>(sums_b + 128 + col);
                        int4 s4[4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) s4[j] = ps[j];
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ky = (j & 1) ? s4[j >> 1].z : s4[j >> 1].x;
                            const int ry = (j & 1) ? s4[j >> 1].w : s4[j >> 1].y;
                            const int xt = xt0 + j;
                            if (yt < p.N && xt <= yt) {
                                const int re = (int)(g1[j] + g2[j] + 514u * g3[j] + (uint32_t)rx + (uint32_t)ry) >> 9;
                                const int im = -((int)(g1[j] - g2[j] + (uint32_t)kx - (uint32_t)ky) >> 5);
                                int2 *o = reinterpret_cast<int2 *>(p.vis) + (long long)f * Bn + (long long)xt * p.N -
                                          (long long)xt * (xt - 1) / 2 + (yt - xt);
                                if (add) { atomicAdd(&o->x, re); atomicAdd(&o->y, im); }
                                else *o = make_int2(re, im);
                            }
                        }
                    }
                }
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(acc_empty, 0);
            } else {
#pragma unroll 1
                for (int c = 0; c < 16; ++c) {
                    const int col = 8 * c;
                    const int yc = y0 + col;
                    const bool skip = (yc + 7 < xw) || (yc >= p.N) || (xw >= p.N);  // warp-uniform
                    if (!skip) {
                        uint32_t g1[8], g2[8], g3[8];
                        ptx::tmem_ld8(trow + col, g1);
                        ptx::tmem_ld8(trow + 128 + col, g2);
                        ptx::tmem_ld8(trow + 256 + col, g3);
                        const int4 *ps = reinterpret_cast<const int4 *>(sums_b + 128 + col);
                        int4 s4[4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) s4[j] = ps[j];
                        ptx::tmem_ld_wait();
                        uint8_t *dst = srow_g + 8 * (sh + col);
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ky = (j & 1) ? s4[j >> 1].z : s4[j >> 1].x;
                            const int ry = (j & 1) ? s4[j >> 1].w : s4[j >> 1].y;
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
                int jlo = max(0, x - y0), jhi = min(128, p.N - y0);
                if (claim) add = !tc3_claim_store(flag, claim_g, 32 * T5_EPI_WARP0, 32 * T5_EPI_WARPS), raise_flag = !add;
                if (x < p.N && jlo < jhi) {
                    ptx::fence_proxy_async_smem();  // this thread's st.shared -> visible to the bulk-copy engine
                    if ((sh + jlo + row) & 1) {      // leading baseline on an odd 8-byte slot of vis
                        const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (sh + jlo));
                        if (add) { atomicAdd(&grow[jlo].x, v.x); atomicAdd(&grow[jlo].y, v.y); }
                        else grow[jlo] = v;
                        ++jlo;
                    }
                    if ((jhi - jlo) & 1) {           // trailing baseline
                        --jhi;
                        const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (sh + jhi));
                        if (add) { atomicAdd(&grow[jhi].x, v.x); atomicAdd(&grow[jhi].y, v.y); }
                        else grow[jhi] = v;
                    }
                    if (jlo < jhi) {
                        if (add) ptx::bulk_reduce_add_s32(grow + jlo, srow + 8u * (sh + jlo), 8u * (jhi - jlo));
                        else ptx::bulk_store(grow + jlo, srow + 8u * (sh + jlo), 8u * (jhi - jlo));
                    }
                }
            }
            ptx::bulk_commit();
            // the sums buffer of this segment is read: clear it for the segment after the next
            ptx::named_bar_sync(2, 32 * T5_EPI_WARPS);
            {
                const int e = (int)threadIdx.x - 32 * T5_EPI_WARP0;
                sums_g[buf * 256 + e] = make_int2(0, 0);
                sums_g[buf * 256 + 128 + e] = make_int2(0, 0);
            }
            if (raise_flag) {
                ptx::bulk_wait0();                 // this thread's part of the tile is in memory ...
                __threadfence();
                ptx::named_bar_sync(1, 32 * T5_EPI_WARPS);   // ... and so is every other epilogue thread's
                if (threadIdx.x == 32 * T5_EPI_WARP0) ptx::st_release_gpu(flag, TC3_FLAG_STORED);
            }
            ++seg_no;
        }
        ptx::bulk_wait0();  // every row segment has been written before the CTA retires
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();  // no CTA of the pair may exit while its peer still reads its smem / barriers
    if (warp == 1) ptx::tmem_dealloc<2>(tmem, 512);
    // The last CTA to get here clears the flags (see corr_tc3.cuh)
    if (threadIdx.x == 0) {
        __threadfence();
        int *done = p.flags + 2 * p.num_units;
        if (atomicAdd(done, 1) == (int)gridDim.x - 1) {
            for (int i = 0; i < 2 * p.num_units; ++i) p.flags[i] = 0;
            __threadfence();
            *done = 0;
        }
    }
}

}  // namespace corr
