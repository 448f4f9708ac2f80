// corr_tc3.cuh -- the large-N path (steps S1-S5) with the A operand in tensor memory.
//
// Same mathematics as corr_tc.cuh / corr_tc2.cuh (Eq. 1, summed over time
// PAPER.md:48, upper triangle PAPER.md:50; x16 int8 operand planes, results shifted right by 8 in
// the epilogue).  Same mapping as corr_tc2.cuh: two CTAs on the two SMs of one TPC form a cluster
// and compute one 256 (x) by 128 (y) tile with tcgen05.mma.cta_group::2.
//
// What changed and why: ncu on corr_tc2_kernel (profiles/r01_tc2_ncu_summary.md) shows the
// shared-memory data pipe at 93 % (LSU 60 % + tensor-core operand reads 33 %) with the tensor pipe at
// 66 %: per 64-sample stage a CTA moved 256 + 96 + 192 wavefronts (plus replays) through a pipe
// that carries 512 in the time the MMAs need.  Here the x-block planes never enter shared memory:
//   * the unpack warps read the packed x-block with ldmatrix.m16n16.x2.trans.b8, which hands every
//     thread four TIME-consecutive bytes of one input per register -- the transpose from the
//     stream's element-contiguous order to the K-major order a TMEM operand needs, done by the
//     load itself;
//   * the planes 16*Re, 16*Im are formed in registers (3 logic ops per word) and written straight
//     into TMEM with tcgen05.st.16x128b.x2, whose fragment is exactly the ldmatrix fragment;
//   * the MMAs take A from TMEM ([a_tmem] form) and only B from shared memory.
// Per stage and CTA: 128 (TC) + 96 (loads) + 64 (stores) wavefronts.
//
// Tried in round 2 and not kept (profiles/r02_tc3_ncu_summary.md): the same arithmetic on a finer pipeline (operand
// slots of 32 samples filled by four groups of unpack warps, 8-slot ring): same speed, this kernel is bound by the
// MMAs and the accumulator drain, not by the unpack; a row-image pitch of 129 slots (conflict-free stores) with
// pipelined 8-column TMEM loads: slower (spills at 96 registers); negating an operand through bits 13 / 14 of the
// instruction descriptor (one accumulator for Im): illegal instruction for kind::i8.
//
// Per CTA r (= rank in the pair) and per stage of 64 time samples:
//   packed X_r  [64][128] bytes, 128-B swizzle   x in [256*bx2 + 128 r, +128)      (TMA)
//   packed Yh_r [64][ 64] bytes,  64-B swizzle   y in [128*by + 64 r, +64)          (TMA)
//   planes Bhr, Bhi [64][64] MN-major SW64 in shared memory (16*Re, 16*Im of the y-half)
//   planes Ar, Ai in TMEM: lane = x - x0, 16 columns each = 64 K-bytes (2 K-steps of 32)
// TMEM columns (per CTA, for its 128 x rows):
//     0..127  IR += Ai * Br^T       128..255  Re += Ai * Bi^T + Ar * Br^T       256..383  RI += Ar * Bi^T
//   384..511  A planes, 4 stages x (Ar 16 cols | Ai 16 cols)
// column j of an accumulator <-> y = 128*by + j (j < 64 from CTA 0's y-half, j >= 64 from CTA 1's).
//   Re = D[128 + j] >> 8,   Im = (D[j] - D[256 + j]) >> 8.
//
// Synchronisation across the pair: the packed ring (TMA -> unpack) is CTA-local.  The operand
// ring (TMEM A stage + smem B stage, same index) is shared: unpack warps of BOTH CTAs arrive on the
// leader's pl_full; the leader's MMA thread commits with multicast so pl_empty / acc_full fire in
// both CTAs; epilogue warps of both CTAs arrive on the leader's acc_empty.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode, baseline_index
#include "corr_ptx.cuh"

namespace corr {

constexpr int T3_ST = 64;              // time samples per stage
constexpr int T3_PK_STAGES = 5;        // packed-byte ring (covers TMA latency)
constexpr int T3_PL_STAGES = 4;        // operand ring: TMEM A stage + smem B stage
constexpr int T3_UNPACK_WARPS = 8;
constexpr int T3_UNPACK_THREADS = 32 * T3_UNPACK_WARPS;
constexpr int T3_EPI_WARP0 = 2 + T3_UNPACK_WARPS;
constexpr int T3_EPI_WARPS = 8;             // two per TMEM lane quarter: column halves
constexpr int T3_THREADS = 32 * (T3_EPI_WARP0 + T3_EPI_WARPS);
constexpr int T3_XBYTES = T3_ST * 128;             // packed x-block per stage
constexpr int T3_YPLANE = T3_ST * 64;              // packed y-half / one y-half plane per stage
constexpr int T3_PK_BYTES = T3_XBYTES + T3_YPLANE;
constexpr int T3_PL_BYTES = 2 * T3_YPLANE;         // Bhr, Bhi
constexpr int T3_EPI_PITCH = 128 * 8 + 16;        // one staged output row: 128 (Re,Im) pairs + parity slot
constexpr int T3_EPI_BYTES = 128 * T3_EPI_PITCH;  // the CTA's whole 128 x 128 output block
constexpr int T3_SMEM_BYTES = 1024 + T3_PK_STAGES * T3_PK_BYTES + T3_PL_STAGES * T3_PL_BYTES + T3_EPI_BYTES + 256;
constexpr uint32_t T3_ACOL0 = 384;                 // first TMEM column of the A stages
constexpr uint32_t T3_ACOLS = 32;                  // columns per A stage: Ar 16 | Ai 16

constexpr int T3_GROUP = T3_ST * T3_PL_STAGES;   // samples per group of stages: the scheduling quantum

struct Tc3Params {
    int N, F, T;
    int tiles_per_f;   // pair tiles (256 x 128) touching the upper triangle, per channel
    int slices;
    int t_per_slice;   // multiple of T3_GROUP
    int num_units;     // F * tiles_per_f * slices
    int out_mode;
    int groups_full;   // groups of T3_GROUP samples in a full slice
    int groups_last;   // ... in the last slice of a tile
    long long total_groups;  // over all units
    int *flags;        // [num_units][2]: claim / stored state of (unit, CTA rank), see tc3_claim_store;
                       // [2 * num_units]: CTAs that have finished (the last one clears the array for the next launch)
    const int4 *pieces;    // [pairs][TC3_MAX_PIECES]: the tail pieces of every pair, see Tc3Iter
    const ushort4 *tiles;  // (xa, xb, by, flags): 128-blocks of the rows of CTA 0 and CTA 1, of the columns; see Tc3Tile
    int32_t *vis;
};

// S3, second half: the work of a call is the list of units (channel, tile, T-slice), each a run of groups
// of T3_GROUP samples.  Whole waves of units are dealt round-robin (unit = pair + k * npairs: the pairs then
// work on neighbouring tiles of one channel at the same time, which is what keeps the re-read input in L2).
// The units left over after the last whole wave are cut into pieces, one or two per CTA pair ("stream-K"), by a
// cost model on the host (tc3_build_pieces in corr_api.cu: groups + a fixed cost per piece), so the tail costs
// every pair the same time whatever the number of tiles.  A segment is the part of one unit that one pair
// computes: a whole unit, or a piece of a tail unit.  The first piece of a cut unit runs BEFORE its pair's whole
// units (see Tc3Iter), the others after: a cut unit is summed in memory, and this way the piece that stores
// has long finished when the others add.
// A pair tile: CTA r computes the 128 x 128 block (rows = inputs of block r ? xb : xa, columns = inputs of
// block by).  Normal tiles hold blocks of the upper triangle as they are (row block <= column block).  A
// TRANSPOSED tile holds blocks (x = by, y = xa) and (x = by, y = xb) of the triangle computed the other way round
// (rows = the y inputs): this is how the blocks left over when a block column has an odd number of row blocks
// are paired up -- as rows they differ, but transposed they all share the column block 0 -- instead of being
// computed next to an idle CTA.  The epilogue conjugates them and stages them transposed (shared-memory row =
// output row), so that they leave as bulk copies like the others.  xb = 0xFFFF: no block.
constexpr unsigned short TC3_TILE_TRANSPOSED = 1, TC3_NO_BLOCK = 0xFFFF;

struct Tc3Seg {
    int u, f, slice;
    ushort4 tile;
    int first, cnt, len;   // groups [first, first + cnt) of the unit's len groups
    int t_begin, t_end;    // first sample of the segment; end of the unit's slice (<= T)
};

// The pieces of the tail units that a pair computes (host: tc3_build_pieces in corr_api.cu): (unit, first group,
// number of groups, early).  An EARLY piece is the first piece of a cut unit and is computed BEFORE the pair's whole
// units: it stores its partial sums hundreds of microseconds before the other pieces of that unit (computed after
// the whole units) add theirs, so nobody waits for anybody at the end of the kernel.
constexpr int TC3_MAX_PIECES = 4;

struct Tc3Iter {
    int k, waves, pair, npairs;
    int phase, pi;         // 0: early pieces, 1: whole units, 2: late pieces; next piece entry
};

__device__ __forceinline__ Tc3Iter tc3_iter(const Tc3Params &p, int pair, int npairs)
{
    Tc3Iter it;
    it.k = 0;
    it.waves = p.num_units / npairs;
    it.pair = pair;
    it.npairs = npairs;
    it.phase = 0;
    it.pi = 0;
    return it;
}

__device__ __forceinline__ bool tc3_next_segment(const Tc3Params &p, Tc3Iter &it, Tc3Seg &s)
{
    int u;
    for (;;) {
        if (it.phase == 1) {                 // a whole unit of a whole wave
            if (it.k < it.waves) {
                u = it.pair + it.k * it.npairs;
                ++it.k;
                s.first = 0;
                s.cnt = -1;
                break;
            }
            it.phase = 2;
            it.pi = 0;
        } else {                             // this pair's pieces of the tail units
            bool found = false;
            while (it.pi < TC3_MAX_PIECES) {
                const int4 e = p.pieces[it.pair * TC3_MAX_PIECES + it.pi++];
                if (e.z > 0 && (e.w != 0) == (it.phase == 0)) {
                    u = e.x;
                    s.first = e.y;
                    s.cnt = e.z;
                    found = true;
                    break;
                }
            }
            if (found) break;
            if (it.phase == 2) return false;
            it.phase = 1;
        }
    }
    const int ft = u / p.slices;
    s.slice = u - ft * p.slices;
    s.len = (s.slice == p.slices - 1) ? p.groups_last : p.groups_full;
    if (s.cnt < 0) s.cnt = s.len;
    s.f = ft / p.tiles_per_f;
    s.tile = p.tiles[ft - s.f * p.tiles_per_f];
    s.u = u;
    s.t_begin = s.slice * p.t_per_slice + s.first * T3_GROUP;
    s.t_end = min(p.T, (s.slice + 1) * p.t_per_slice);
    return true;
}

// Flag of (unit, CTA rank): 0 = untouched, CLAIMED = one piece is storing, STORED = its store is in memory.
constexpr int TC3_FLAG_CLAIMED = 1, TC3_FLAG_STORED = 2;

// Called by all epilogue threads of a CTA (warp-uniform control flow).  Returns true in the CTA whose piece
// stores (the first to arrive); in every other CTA it returns, false, once the store is visible.
__device__ __forceinline__ bool tc3_claim_store(int *flag, volatile int *claim_smem, int epi_thread0 = 32 * T3_EPI_WARP0,
                                                int epi_threads = 32 * T3_EPI_WARPS)
{
    if ((int)threadIdx.x == epi_thread0) *claim_smem = atomicCAS(flag, 0, TC3_FLAG_CLAIMED);
    ptx::named_bar_sync(1, epi_threads);
    const int before = *claim_smem;
    ptx::named_bar_sync(1, epi_threads);   // everyone has read the slot before its next use
    if (before == 0) return true;
    while (ptx::ld_acquire_gpu(flag) != TC3_FLAG_STORED) {
    }
    return false;
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T3_THREADS, 1)
corr_tc3_kernel(const __grid_constant__ CUtensorMap tmap_x, const __grid_constant__ CUtensorMap tmap_y,
                const Tc3Params p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t pk0 = base;
    const uint32_t pl0 = pk0 + T3_PK_STAGES * T3_PK_BYTES;
    const uint32_t epi0 = pl0 + T3_PL_STAGES * T3_PL_BYTES;
    const uint32_t bar0 = epi0 + T3_EPI_BYTES;
    uint8_t *epi_g = gbase + (epi0 - base);
    auto pk_full = [&](int s) { return bar0 + 8u * s; };
    auto pk_empty = [&](int s) { return bar0 + 8u * (T3_PK_STAGES + s); };
    auto pl_full = [&](int s) { return bar0 + 8u * (2 * T3_PK_STAGES + s); };
    auto pl_empty = [&](int s) { return bar0 + 8u * (2 * T3_PK_STAGES + T3_PL_STAGES + s); };
    const uint32_t acc_full = bar0 + 8u * (2 * T3_PK_STAGES + 2 * T3_PL_STAGES);
    const uint32_t acc_empty = acc_full + 8u;
    const uint32_t tmem_slot = acc_empty + 8u;
    volatile uint32_t *tmem_slot_g = reinterpret_cast<volatile uint32_t *>(gbase + (tmem_slot - base));
    volatile int *claim_g = reinterpret_cast<volatile int *>(gbase + (tmem_slot + 8u - base));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = ptx::cluster_ctarank();  // 0 = leader (issues the MMAs)
    const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmap_x);
        ptx::prefetch_tmap(&tmap_y);
        for (int s = 0; s < T3_PK_STAGES; ++s) {
            ptx::mbar_init(pk_full(s), 1);
            ptx::mbar_init(pk_empty(s), T3_UNPACK_WARPS);
        }
        for (int s = 0; s < T3_PL_STAGES; ++s) {
            ptx::mbar_init(pl_full(s), 2 * T3_UNPACK_WARPS);  // both CTAs' unpack warps (the leader's copy is used)
            ptx::mbar_init(pl_empty(s), 1);
        }
        ptx::mbar_init(acc_full, 1);
        ptx::mbar_init(acc_empty, 2 * T3_EPI_WARPS);
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
    ptx::grid_dependency_wait();   // the previous kernel of the stream has completed: its output (our input, vis, the flags) is visible

    Tc3Iter sit = tc3_iter(p, pair, npairs);   // every role walks the same list of segments
    Tc3Seg sg;

    if (warp == 0) {
        // ===================== S1: TMA producer (each CTA loads its own blocks) =====================
        if (lane == 0) {
            int st = 0;
            uint32_t ph = 0;
            while (tc3_next_segment(p, sit, sg)) {
                const int f = sg.f;
                const ushort4 tile = sg.tile;
                const int t_begin = sg.t_begin;
                const int xc = (int)(rank ? tile.y : tile.x) * 128;   // TC3_NO_BLOCK: out of bounds, TMA fills zeros
                const int yc = tile.z * 128 + (int)rank * 64;
                const int t_pad = t_begin + sg.cnt * T3_GROUP;   // whole groups of stages
                for (int t = t_begin; t < t_pad; t += T3_ST) {
                    ptx::mbar_wait(pk_empty(st), ph ^ 1u);
                    ptx::mbar_arrive_expect_tx(pk_full(st), T3_PK_BYTES);
                    const uint32_t dst = pk0 + st * T3_PK_BYTES;
                    ptx::tma_load_3d(dst, &tmap_x, pk_full(st), xc, f, t);
                    ptx::tma_load_3d(dst + T3_XBYTES, &tmap_y, pk_full(st), yc, f, t);
                    if (++st == T3_PK_STAGES) { st = 0; ph ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== S4: MMA issuer (leader CTA only) =====================
        // The whole warp runs this loop so that every operand is computed in warp-uniform code
        // (uniform registers, no per-instruction ELECT / R2UR chains); one elected lane issues.
        // Every unit runs a multiple of T3_PL_STAGES stages, so the stage index is a compile-time
        // constant in the unrolled body and all descriptors are "uniform base + constant".
        if (rank == 0) {
            constexpr uint32_t idesc = make_idesc_i8(256, 128, true, true, /*A K-major (TMEM)*/ false, /*B MN-major*/ true);
            uint32_t ph = 0, acc_ph = 0;
            const bool issuer = ptx::elect_one();
            while (tc3_next_segment(p, sit, sg)) {
                const int ngroups = sg.cnt;
                ptx::mbar_wait_cluster(acc_empty, acc_ph ^ 1u);
                ptx::tc_fence_after_sync();
                uint32_t acc = 0;
                for (int g = 0; g < ngroups; ++g) {
#pragma unroll
                    for (int st = 0; st < T3_PL_STAGES; ++st) {
                        ptx::mbar_wait_cluster(pl_full(st), ph);
                        ptx::tc_fence_after_sync();
                        if (issuer) {
                            const uint32_t pl = pl0 + st * T3_PL_BYTES;
                            const uint32_t a0 = T3_ACOL0 + (uint32_t)st * T3_ACOLS;  // TMEM base is 0 (checked at start)
#pragma unroll
                            for (int ks = 0; ks < T3_ST / 32; ++ks) {
                                // B half per CTA: one 64-wide MN block, SW64, 8-row K groups 512 B apart; K-step = 2048 B
                                const uint64_t dBr = make_smem_desc(pl + ks * 2048, T3_YPLANE, 512, 4);
                                const uint64_t dBi = make_smem_desc(pl + T3_YPLANE + ks * 2048, T3_YPLANE, 512, 4);
                                const uint32_t a_r = a0 + 8u * ks, a_i = a0 + 16u + 8u * ks;
                                ptx::mma_i8_ts<2>(0, a_i, dBr, idesc, acc);    // IR
                                ptx::mma_i8_ts<2>(128, a_i, dBi, idesc, acc);  // II  -> Re
                                ptx::mma_i8_ts<2>(256, a_r, dBi, idesc, acc);  // RI
                                ptx::mma_i8_ts<2>(128, a_r, dBr, idesc, 1);    // RR  -> Re
                                acc = 1;
                            }
                            ptx::mma_commit_mcast2(pl_empty(st), 0x3);  // operand stage of BOTH CTAs is free
                        }
                        __syncwarp();
                    }
                    ph ^= 1u;
                }
                if (issuer) ptx::mma_commit_mcast2(acc_full, 0x3);
                __syncwarp();
                acc_ph ^= 1u;
            }
        }
    } else if (warp < T3_EPI_WARP0) {
        // ===================== S2: unpack =====================
        const int ut = threadIdx.x - 64;
        const int q = warp & 3;                 // TMEM lane quarter this warp may write: inputs 32q..32q+31
        const int kh = (warp - 2) >> 2;         // which 32-sample half of the stage this warp transposes
        // ldmatrix row address of this lane: matrix m = lane/16, row r = lane%16 -> sample 32 kh + 16 m + r
        const int lrow = 32 * kh + 16 * (lane >> 4) + (lane & 15);
        const uint32_t lds0 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 0) ^ (lrow & 7)) << 4);
        const uint32_t lds1 = (uint32_t)lrow * 128u + ((uint32_t)((2 * q + 1) ^ (lrow & 7)) << 4);
        const int tbase = 32 * kh + 4 * (lane & 3);  // first sample of this thread's r0/r1 (r2/r3: + 16)
        const uint32_t tdst = tmem + ((uint32_t)(32 * q) << 16) + T3_ACOL0 + 8u * kh;
        int pst = 0, qst = 0;
        uint32_t pph = 0, qph = 0;
        while (tc3_next_segment(p, sit, sg)) {
            const int t_begin = sg.t_begin, t_end = sg.t_end;
            const int t_pad = t_begin + sg.cnt * T3_GROUP;
            for (int t = t_begin; t < t_pad; t += T3_ST) {
                const int rows_valid = t_end - t;  // <= 0 in a padding stage: all-zero operands
                // byte masks of this thread's four samples (zero beyond the slice)
                uint32_t m0 = 0xF0F0F0F0u, m1 = 0xF0F0F0F0u;
                if (rows_valid < T3_ST) {
                    const int v0 = min(4, max(0, rows_valid - tbase)), v1 = min(4, max(0, rows_valid - tbase - 16));
                    m0 = v0 ? (0xF0F0F0F0u >> (32 - 8 * v0)) : 0u;
                    m1 = v1 ? (0xF0F0F0F0u >> (32 - 8 * v1)) : 0u;
                }
                ptx::mbar_wait(pk_full(pst), pph);
                const uint32_t src = pk0 + pst * T3_PK_BYTES;
                // ---- loads first: two transposing loads of the x-block, one 16-byte chunk of the y-half
                uint32_t xa[4], xb[4];
                ptx::ldsm_t_b8_x2(src + lds0, xa[0], xa[1], xa[2], xa[3]);   // inputs 32q + 0..15
                ptx::ldsm_t_b8_x2(src + lds1, xb[0], xb[1], xb[2], xb[3]);   // inputs 32q + 16..31
                const uint4 wy = *reinterpret_cast<const uint4 *>(gbase + (src - base) + T3_XBYTES + ut * 16);
                ptx::mbar_wait_cluster(pl_empty(qst), qph ^ 1u);
                // ---- A planes -> TMEM
                const uint32_t ta = tdst + (uint32_t)qst * T3_ACOLS;
                ptx::tmem_st_16x128b_x2(ta, (xa[0] ^ 0x80808080u) & m0, (xa[1] ^ 0x80808080u) & m0,
                                        (xa[2] ^ 0x80808080u) & m1, (xa[3] ^ 0x80808080u) & m1);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16), (xb[0] ^ 0x80808080u) & m0, (xb[1] ^ 0x80808080u) & m0,
                                        (xb[2] ^ 0x80808080u) & m1, (xb[3] ^ 0x80808080u) & m1);
                ptx::tmem_st_16x128b_x2(ta + 16u, ((xa[0] << 4) ^ 0x80808080u) & m0, ((xa[1] << 4) ^ 0x80808080u) & m0,
                                        ((xa[2] << 4) ^ 0x80808080u) & m1, ((xa[3] << 4) ^ 0x80808080u) & m1);
                ptx::tmem_st_16x128b_x2(ta + (16u << 16) + 16u, ((xb[0] << 4) ^ 0x80808080u) & m0,
                                        ((xb[1] << 4) ^ 0x80808080u) & m0, ((xb[2] << 4) ^ 0x80808080u) & m1,
                                        ((xb[3] << 4) ^ 0x80808080u) & m1);
                // ---- B planes -> shared memory, same physical offsets as the packed y-half
                {
                    uint8_t *dst = gbase + (pl0 - base) + qst * T3_PL_BYTES;
                    const uint32_t off = (uint32_t)ut * 16u;
                    const uint32_t m = ((int)(off >> 6) < rows_valid) ? 0xF0F0F0F0u : 0u;  // 64-B rows
                    uint4 r, i;
                    r.x = (wy.x ^ 0x80808080u) & m; r.y = (wy.y ^ 0x80808080u) & m;
                    r.z = (wy.z ^ 0x80808080u) & m; r.w = (wy.w ^ 0x80808080u) & m;
                    i.x = ((wy.x << 4) ^ 0x80808080u) & m; i.y = ((wy.y << 4) ^ 0x80808080u) & m;
                    i.z = ((wy.z << 4) ^ 0x80808080u) & m; i.w = ((wy.w << 4) ^ 0x80808080u) & m;
                    *reinterpret_cast<uint4 *>(dst + off) = r;
                    *reinterpret_cast<uint4 *>(dst + T3_YPLANE + off) = i;
                }
                ptx::fence_proxy_async_smem();   // B planes: generic-proxy writes, read by the MMA's async proxy
                ptx::tmem_st_wait();             // A planes are in TMEM
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive_cluster(pl_full(qst), 0);  // the leader's barrier
                    ptx::mbar_arrive(pk_empty(pst));
                }
                if (++pst == T3_PK_STAGES) { pst = 0; pph ^= 1u; }
                if (++qst == T3_PL_STAGES) { qst = 0; qph ^= 1u; }
            }
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
        const int h = (warp - T3_EPI_WARP0) >> 2;
        const int row = 32 * q + lane;
        const uint32_t srow = epi0 + (uint32_t)row * T3_EPI_PITCH;
        uint8_t *srow_g = epi_g + row * T3_EPI_PITCH;
        const long long Bn = (long long)p.N * ((long long)p.N + 1) / 2;
        const bool base_add = (p.out_mode != OUT_STORE);
        uint32_t acc_ph = 0;
        bool prev_transposed = false;
        while (tc3_next_segment(p, sit, sg)) {
            // A unit cut by the stream-K schedule is summed in memory.  When the call overwrites (OUT_STORE),
            // the piece that gets to its output FIRST claims the unit (atomic compare-and-swap on the unit's flag),
            // stores, and then marks the flag "stored"; every later piece waits for that mark and adds.  A waiting
            // CTA therefore only ever waits for a CTA that is resident and already in its epilogue: no piece
            // depends on a CTA that has not been scheduled yet, whatever else shares the GPU.
            const bool claim = !base_add && (sg.cnt != sg.len);   // a piece of a cut unit in a call that overwrites
            bool add = base_add, raise_flag = false;
            int *flag = p.flags + 2 * sg.u + (int)rank;
            const int f = sg.f;
            const ushort4 tile = sg.tile;
            const int x0 = (int)(rank ? tile.y : tile.x) * 128, y0 = tile.z * 128;   // rows and columns of the MMA
            const int xw = x0 + q * 32;
            const int x = x0 + row;
            const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
            const bool transposed = (tile.w & TC3_TILE_TRANSPOSED) != 0;
            if (transposed || prev_transposed) {
                // a transposed unit's row images are written by all epilogue threads and sent by others: everybody's
                // previous copies must have left shared memory before anybody writes
                ptx::bulk_wait_read0();
                ptx::named_bar_sync(3, 32 * T3_EPI_WARPS);
            }
            prev_transposed = transposed;
            if (transposed) {
                // ---- transposed block: this thread's MMA row is the baseline's y, the MMA columns are its x,
                // vis(x', y') = conj(D[y'][x']).  For one MMA column the 32 lanes of a warp hold consecutive y', which
                // are consecutive in vis: the image of output row x' = y0 + c is shared-memory row c, written by
                // the lanes side by side (conflict-free), and thread c of the h = 0 warps sends it as one bulk copy.
                ptx::mbar_wait_cluster(acc_full, acc_ph);
                acc_ph ^= 1u;
                ptx::tc_fence_after_sync();
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int col = 64 * h + 16 * c;
                    const int xt0 = y0 + col;   // true x of the chunk's first column
                    const bool skip = (xt0 > xw + 31) || (xt0 >= p.N) || (xw >= p.N);  // warp-uniform
                    if (!skip) {
                        uint32_t ir[16], rr[16], ri[16];
                        ptx::tmem_ld16(trow + col, ir);
                        ptx::tmem_ld16(trow + 128 + col, rr);
                        ptx::tmem_ld16(trow + 256 + col, ri);
                        ptx::tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) {
                            const int xt = xt0 + j;
                            // parity of the 8-byte index of (xt, x0) in vis: slot of MMA row R in image row col + j
                            const long long gi = (long long)f * Bn + (long long)xt * p.N - (long long)xt * (xt - 1) / 2 - xt + x0;
                            const uint32_t parc = (uint32_t)((reinterpret_cast<uintptr_t>(p.vis) >> 3) + (unsigned long long)gi) & 1u;
                            const int re = (int)rr[j] >> 8;
                            const int im = -((int)(ir[j] - ri[j]) >> 8);
                            *reinterpret_cast<int2 *>(epi_g + (col + j) * T3_EPI_PITCH + 8 * (parc + row)) = make_int2(re, im);
                        }
                    }
                }
                // TMEM is free for the next unit
                ptx::tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive_cluster(acc_empty, 0);
                if (claim) add = !tc3_claim_store(flag, claim_g), raise_flag = !add;
                ptx::fence_proxy_async_smem();  // this thread's st.shared -> visible to the bulk-copy engine
                ptx::named_bar_sync(3, 32 * T3_EPI_WARPS);   // every image row is complete
                if (h == 0) {
                    // image row `row` = output row xt, columns yt = x0 + R for R in [rlo, rhi)
                    const int xt = y0 + row;
                    int rlo = max(0, xt - x0), rhi = min(128, p.N - x0);
                    if (xt < p.N && rlo < rhi) {
                        const long long gi = (long long)f * Bn + (long long)xt * p.N - (long long)xt * (xt - 1) / 2 - xt + x0;
                        int2 *grow = reinterpret_cast<int2 *>(p.vis) + gi;
                        const uint32_t parc = (uint32_t)(reinterpret_cast<uintptr_t>(grow) >> 3) & 1u;
                        if ((parc + rlo) & 1) {           // leading baseline on an odd 8-byte slot
                            const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (parc + rlo));
                            if (add) { atomicAdd(&grow[rlo].x, v.x); atomicAdd(&grow[rlo].y, v.y); }
                            else grow[rlo] = v;
                            ++rlo;
                        }
                        if ((rhi - rlo) & 1) {            // trailing baseline
                            --rhi;
                            const int2 v = *reinterpret_cast<const int2 *>(srow_g + 8 * (parc + rhi));
                            if (add) { atomicAdd(&grow[rhi].x, v.x); atomicAdd(&grow[rhi].y, v.y); }
                            else grow[rhi] = v;
                        }
                        if (rlo < rhi) {
                            if (add) ptx::bulk_reduce_add_s32(grow + rlo, srow + 8u * (parc + rlo), 8u * (rhi - rlo));
                            else ptx::bulk_store(grow + rlo, srow + 8u * (parc + rlo), 8u * (rhi - rlo));
                        }
                    }
                }
            } else {
            // 8-byte index of (x, y0) in vis (formal when y0 < x: only its parity and offsets from it are used)
            const long long g0 = (long long)f * Bn + (long long)x * p.N - (long long)x * (x - 1) / 2 - x + y0;
            int2 *grow = reinterpret_cast<int2 *>(p.vis) + g0;
            const uint32_t par = (uint32_t)(reinterpret_cast<uintptr_t>(grow) >> 3) & 1u;
            ptx::bulk_wait_read0();  // this thread's previous row segment has left shared memory
            ptx::mbar_wait_cluster(acc_full, acc_ph);
            acc_ph ^= 1u;
            ptx::tc_fence_after_sync();
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int col = 64 * h + 16 * c;
                const int yc = y0 + col;
                const bool skip = (yc + 15 < xw) || (yc >= p.N) || (xw >= p.N);  // warp-uniform
                if (!skip) {
                    uint32_t ir[16], rr[16], ri[16];
                    ptx::tmem_ld16(trow + col, ir);
                    ptx::tmem_ld16(trow + 128 + col, rr);
                    ptx::tmem_ld16(trow + 256 + col, ri);
                    ptx::tmem_ld_wait();
                    uint8_t *dst = srow_g + 8 * (par + col);
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
            if (lane == 0) ptx::mbar_arrive_cluster(acc_empty, 0);
            // ---- write the row segment [jlo, jhi) of this thread
            int jlo = max(64 * h, x - y0), jhi = min(64 * h + 64, p.N - y0);
            if (claim) add = !tc3_claim_store(flag, claim_g), raise_flag = !add;
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
            }
            ptx::bulk_commit();
            if (raise_flag) {
                ptx::bulk_wait0();                 // this thread's part of the tile is in memory ...
                __threadfence();
                ptx::named_bar_sync(1, 32 * T3_EPI_WARPS);   // ... and so is every other epilogue thread's
                if (threadIdx.x == 32 * T3_EPI_WARP0) ptx::st_release_gpu(flag, TC3_FLAG_STORED);
            }
        }
        ptx::bulk_wait0();  // every row segment has been written before the CTA retires
    }

    __syncwarp();  // lanes that skipped the single-thread roles rejoin here
    ptx::tc_fence_before_sync();
    ptx::cluster_sync();  // no CTA of the pair may exit while its peer still reads its smem / barriers
    if (warp == 1) ptx::tmem_dealloc<2>(tmem, 512);
    // The last CTA to get here clears the flags, so that the next launch (or a replay of this one from a
    // captured CUDA graph) starts from a clean array: nobody reads a flag after its own CTA has counted itself.
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
