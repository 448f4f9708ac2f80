// corr_imma.cuh -- step S4' of the hot path for N = 16, 32, 48, 64: warp-level int8 tensor-core
// MMA (mma.sync.m16n8k32.s8) on whole channels, fed by TMA.
//
// Why not dp4a here: streaming N = 16 inputs at HBM speed needs 4 (N + 1) ops per byte x 6.5 TB/s = 440 effective
// TOPS, and the CUDA-core kernel (one __dp4a per complex MAC, corr_dp4a.cuh) reached 0.37 TB/s on that shape where
// this kernel reaches 4.2 - 4.7 (profiles/r01_sweep.csv, the dp4a figure in profiles/r01_sweep.md).  Warp-level
// mma.sync keeps N = 16 and 32 memory-bound; at N = 48 and 64 it is bound by its own issue rate.  Other N <= 64 run
// here on a stream padded to the next multiple of 16 inputs (corr_pad_kernel below); N = 64 with an even channel
// count goes to single-CTA tcgen05 tiles instead (two channels per tile, corr_api.cu); corr_dp4a.cuh is only
// used on request.  The paper makes the small-N observation for its own tiles at
// PAPER.md:72; the result computed is Eq. 1 summed over time on the
// upper triangle.
//
// Data movement.  The stream [T][F][N] is a plain 2-D byte matrix with rows of F*N bytes, so a CTA
// takes a 128-byte-wide column strip (FB = 128/N whole channels) and a chunk of time samples:
// TMA boxes [128 t][128 B] with 128-byte swizzle into a ring of stages.
//
// Arithmetic.  ldmatrix.m16n16.trans.b8 hands every thread four TIME-consecutive bytes of one
// input, which is both the A fragment (rows = inputs 16mt..16mt+15, K = 32 samples) and, split in
// halves, the B fragments (columns = inputs 8nt..8nt+7) of mma.m16n8k32.  Planes 16*Re =
// (w ^ 0x80) & 0xF0 and 16*Im = ((w << 4) ^ 0x80) & 0xF0 are exact int8; per 32 samples
//     Re[mt][nt] += Pr[mt] Pr[nt]^T + Pi[mt] Pi[nt]^T      only blocks with nt >= 2 mt (upper triangle)
//     IR[mt][nt] += Pi[mt] Pr[nt]^T                         all blocks
// and at the end  Re >> 8,  Im[x][y] = (IR[x][y] - IR[y][x]) >> 8  (sum Re[x] Im[y] = IR[y][x]).
// Three MMAs per block pair instead of four because the whole channel is in one CTA.
//
// Warps: one per (channel of the strip, m-tile set, K-split); partial sums of the K-split warps
// are combined with shared-memory atomics in the ring's memory after the pipeline has drained,
// then written with store / read-add-store / atomicAdd like the other paths.
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_dp4a.cuh"  // OutMode, baseline_index
#include "corr_ptx.cuh"

namespace corr {

constexpr int IM_ROWS = 128;                 // time samples per stage
constexpr int IM_STAGE_BYTES = IM_ROWS * 128;
constexpr int IM_STAGES = 6;
constexpr int IM_MAX_CHUNK = 32768;          // time samples per CTA: 256 * 128 * chunk stays far below 2^31 (multiple of IM_ROWS)
constexpr int IM_SMEM_BYTES = 1024 + IM_STAGES * IM_STAGE_BYTES + 512;   // ring + 2 x IM_STAGES x 4 barriers

template <int NT16> struct ImmaCfg {
    static constexpr int N = 16 * NT16;
    static constexpr int FB = 128 / N;                         // whole channels per 128-byte strip (8, 4, 2, 2)
    static constexpr int STRIP = FB * N;                       // bytes between strips (N = 48: 96, boxes overlap by 32)
    static constexpr int MS = (NT16 == 4) ? 2 : 1;             // warps that share a channel's m-tiles
    static constexpr int SETS = NT16 / MS;                     // m-tiles per warp (1, 2, 3, 2)
    static constexpr int KS = (NT16 == 1) ? 2 : (NT16 == 4) ? 2 : 4;   // K-split
    static constexpr int WARPS = FB * MS * KS;                 // consumer warps (16, 16, 8, 8)
    // + the TMA producer warp (measured 7 % faster than thread 0 issuing the loads between its consumer iterations)
    static constexpr int THREADS = 32 * (WARPS + 1);
};

struct ImmaParams {
    int N, F, T;
    int t_per_chunk;   // multiple of 32
    int out_mode;
    int32_t *vis;
};

__device__ __forceinline__ void mma_s8(int (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// One K-block (32 samples): the products of m-tile MT (accumulator set S of this warp) with every n-tile.
template <int NT16, int MT, int S, int SETS>
__device__ __forceinline__ void imma_mtile(const uint32_t (&pr)[NT16][4], const uint32_t (&pi)[NT16][4],
                                           int (&re)[SETS][2 * NT16][4], int (&ir)[SETS][2 * NT16][4])
{
    // three passes so that the two MMAs that add into the same Re block are far apart in the issue stream
#pragma unroll
    for (int nt = 2 * MT; nt < 2 * NT16; ++nt)        // blocks that touch the upper triangle
        mma_s8(re[S][nt], pr[MT], pr[nt >> 1][nt & 1], pr[nt >> 1][2 + (nt & 1)]);
#pragma unroll
    for (int nt = 0; nt < 2 * NT16; ++nt)
        mma_s8(ir[S][nt], pi[MT], pr[nt >> 1][nt & 1], pr[nt >> 1][2 + (nt & 1)]);
#pragma unroll
    for (int nt = 2 * MT; nt < 2 * NT16; ++nt)
        mma_s8(re[S][nt], pi[MT], pi[nt >> 1][nt & 1], pi[nt >> 1][2 + (nt & 1)]);
}

template <int NT16>
__global__ void __launch_bounds__(ImmaCfg<NT16>::THREADS, 1)
corr_imma_kernel(const __grid_constant__ CUtensorMap tmap, const ImmaParams p)
{
    using C = ImmaCfg<NT16>;
    constexpr int N = C::N;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t *gbase = smem_raw + (base - ptx::smem_u32(smem_raw));
    const uint32_t bar0 = base + IM_STAGES * IM_STAGE_BYTES;
    // One pair of barriers per (ring position, K-split group).  Stage j goes to position j % IM_STAGES and is consumed by the
    // warps of group j % KS only, so with IM_STAGES = 6 and KS = 4 a group comes back to a position every SECOND time round:
    // on a barrier per position it would always wait for the same parity and could not tell "my stage has landed" from
    // "the other group's stage before it has not landed yet" (TMA loads complete out of order): it would read the ring
    // early and arrive on `empty` once too often.  With a barrier of its own every visit is the next phase; a (position,
    // group) pair is used once every PERIOD = lcm(IM_STAGES, KS) stages.
    constexpr int PERIOD = (IM_STAGES % C::KS == 0) ? IM_STAGES : (IM_STAGES * C::KS) / ((IM_STAGES % 2 == 0 && C::KS % 2 == 0) ? 2 : 1);
    static_assert(PERIOD % IM_STAGES == 0 && PERIOD % C::KS == 0 && C::KS <= 4, "PERIOD = lcm(IM_STAGES, KS)");
    auto full = [&](int s, int g) { return bar0 + 8u * (4 * s + g); };
    auto empty = [&](int s, int g) { return bar0 + 8u * (4 * IM_STAGES + 4 * s + g); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int strip = blockIdx.x, chunk = blockIdx.y;
    const int t_begin = chunk * p.t_per_chunk;
    const int t_end = min(p.T, t_begin + p.t_per_chunk);
    const int nstages = (t_end - t_begin + IM_ROWS - 1) / IM_ROWS;

    if (threadIdx.x == 0) {
        ptx::prefetch_tmap(&tmap);
        for (int s = 0; s < IM_STAGES; ++s) {
            for (int g = 0; g < C::KS; ++g) {
                ptx::mbar_init(full(s, g), 1);
                ptx::mbar_init(empty(s, g), C::WARPS / C::KS);   // the warps of the group (see the K-split below)
            }
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();

    // accumulators of this warp: SETS m-tiles x all n-tiles, (16 x 8 int32 per block) / 32 lanes
    int re[C::SETS][2 * NT16][4], ir[C::SETS][2 * NT16][4];
#pragma unroll
    for (int s = 0; s < C::SETS; ++s)
#pragma unroll
        for (int nt = 0; nt < 2 * NT16; ++nt)
#pragma unroll
            for (int j = 0; j < 4; ++j) re[s][nt][j] = ir[s][nt][j] = 0;

    const int ch = warp % C::FB;                    // channel inside the strip
    // N = 64: two warps per channel with m-tiles {0, 3} and {1, 2}: 36 MMAs per K-block each
    const int ms = (warp / C::FB) % C::MS;
    const int ks = warp / (C::FB * C::MS);          // K-split index
    const int f = strip * C::FB + ch;

    auto produce = [&](int j) {
        if (j < nstages) {
            const int sj = j % IM_STAGES;
            if (j >= IM_STAGES) {   // the position's last stage, j - IM_STAGES (another group's when KS = 4), has been consumed
                const int jp = j - IM_STAGES;
                ptx::mbar_wait(empty(sj, jp % C::KS), (uint32_t)(jp / PERIOD) & 1u);
            }
            ptx::mbar_arrive_expect_tx(full(sj, j % C::KS), IM_STAGE_BYTES);
            ptx::tma_load_2d(base + sj * IM_STAGE_BYTES, &tmap, full(sj, j % C::KS), strip * C::STRIP, t_begin + j * IM_ROWS);
        }
    };
    if (warp == C::WARPS) {
        // ===================== TMA producer =====================
        if (lane == 0)
            for (int j = 0; j < nstages; ++j) produce(j);
    } else {
        // ===================== consumers =====================
        const uint32_t c16 = (uint32_t)(ch * N) >> 4;   // first 16-byte chunk of this channel in a 128-byte row
        // K-split by STAGE: warp ks takes the stages it with it % KS == ks, whole.  The warps of one SM
        // sub-partition (same channel, different ks) then wait on different barriers and drift apart, so the
        // load / unpack phase of one overlaps the MMA phase of another instead of all four moving in lockstep.
        for (int it = ks; it < nstages; it += C::KS) {
            const int s = it % IM_STAGES;
            ptx::mbar_wait(full(s, ks), (uint32_t)(it / PERIOD) & 1u);
            const uint32_t stage = base + s * IM_STAGE_BYTES;
            if (f < p.F) {
#pragma unroll
                for (int kb = 0; kb < IM_ROWS / 32; ++kb) {             // K-blocks of 32 samples of the stage
                    const int valid = t_end - (t_begin + it * IM_ROWS + 32 * kb);   // samples of this K-block inside the chunk
                    if (valid <= 0) continue;
                    const uint32_t r = 32u * kb + lane;                   // ldmatrix row of this lane (time sample)
                    uint32_t pr[NT16][4], pi[NT16][4];
#pragma unroll
                    for (int mt = 0; mt < NT16; ++mt) {
                        uint32_t w[4];
                        ptx::ldsm_t_b8_x2(stage + r * 128u + (((c16 + mt) ^ (r & 7u)) << 4), w[0], w[1], w[2], w[3]);
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            pr[mt][j] = (w[j] ^ 0x80808080u) & 0xF0F0F0F0u;
                            pi[mt][j] = ((w[j] << 4) ^ 0x80808080u) & 0xF0F0F0F0u;
                        }
                    }
                    uint32_t mk0 = 0xF0F0F0F0u, mk1 = 0xF0F0F0F0u;
                    if (valid < 32) {   // ragged end of the chunk: zero the samples beyond it (registers 0,1: 4c.., 2,3: 16+4c..)
                        const int c4 = 4 * (lane & 3);
                        const int v0 = min(4, max(0, valid - c4)), v1 = min(4, max(0, valid - c4 - 16));
                        mk0 = v0 ? (0xF0F0F0F0u >> (32 - 8 * v0)) : 0u;
                        mk1 = v1 ? (0xF0F0F0F0u >> (32 - 8 * v1)) : 0u;
#pragma unroll
                        for (int mt = 0; mt < NT16; ++mt) {
                            pr[mt][0] &= mk0; pr[mt][1] &= mk0; pr[mt][2] &= mk1; pr[mt][3] &= mk1;
                            pi[mt][0] &= mk0; pi[mt][1] &= mk0; pi[mt][2] &= mk1; pi[mt][3] &= mk1;
                        }
                    }
                    if constexpr (NT16 == 4) {
                        if (ms == 0) { imma_mtile<4, 0, 0, 2>(pr, pi, re, ir); imma_mtile<4, 3, 1, 2>(pr, pi, re, ir); }
                        else         { imma_mtile<4, 1, 0, 2>(pr, pi, re, ir); imma_mtile<4, 2, 1, 2>(pr, pi, re, ir); }
                    } else if constexpr (NT16 == 3) {
                        imma_mtile<3, 0, 0, 3>(pr, pi, re, ir); imma_mtile<3, 1, 1, 3>(pr, pi, re, ir);
                        imma_mtile<3, 2, 2, 3>(pr, pi, re, ir);
                    } else if constexpr (NT16 == 2) {
                        imma_mtile<2, 0, 0, 2>(pr, pi, re, ir); imma_mtile<2, 1, 1, 2>(pr, pi, re, ir);
                    } else {
                        imma_mtile<1, 0, 0, 1>(pr, pi, re, ir);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty(s, ks));
        }
    }

    // ---- combine the K-split warps in shared memory (the ring is drained: every stage was consumed)
    __syncthreads();
    int *red = reinterpret_cast<int *>(gbase);          // [FB][2][N*N]: Re, IR
    for (int i = threadIdx.x; i < C::FB * 2 * N * N; i += C::THREADS) red[i] = 0;
    __syncthreads();
    if (warp < C::WARPS && f < p.F) {
        int *rre = red + (ch * 2 + 0) * N * N, *rir = red + (ch * 2 + 1) * N * N;
        const int g = lane >> 2, c2 = 2 * (lane & 3);
#pragma unroll
        for (int s = 0; s < C::SETS; ++s) {
            const int mt = (NT16 == 4) ? ((ms == 0) ? (s == 0 ? 0 : 3) : (s == 0 ? 1 : 2)) : s;
#pragma unroll
            for (int nt = 0; nt < 2 * NT16; ++nt) {
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int x = 16 * mt + g + 8 * (j >> 1), y = 8 * nt + c2 + (j & 1);
                    atomicAdd(&rir[x * N + y], ir[s][nt][j]);
                    if (nt >= 2 * mt) atomicAdd(&rre[x * N + y], re[s][nt][j]);
                }
            }
        }
    }
    __syncthreads();

    // ---- S5: form (Re, Im), keep x <= y, write.  p.N is the number of inputs the caller has (the stream may be
    //      padded to the next multiple of 16 with zero samples): it decides the layout of vis.
    const int NL = p.N;
    const size_t B = (size_t)NL * (NL + 1) / 2;
    for (int i = threadIdx.x; i < C::FB * N * N; i += C::THREADS) {
        const int c = i / (N * N), x = (i / N) % N, y = i % N;
        const int fo = strip * C::FB + c;
        if (fo >= p.F || y < x || y >= NL) continue;
        const int *rre = red + (c * 2 + 0) * N * N, *rir = red + (c * 2 + 1) * N * N;
        const int vre = rre[x * N + y] >> 8;
        const int vim = (rir[x * N + y] - rir[y * N + x]) >> 8;
        int32_t *o = p.vis + 2 * ((size_t)fo * B + baseline_index(NL, x, y));
        if (p.out_mode == OUT_STORE) { o[0] = vre; o[1] = vim; }
        else if (p.out_mode == OUT_RMW) { o[0] += vre; o[1] += vim; }
        else { atomicAdd(o, vre); atomicAdd(o + 1, vim); }
    }
}

// Pads a stream of N inputs per (t, f) row to NP = the next multiple of 16 with stored zeros (0x88 = 0 + 0i),
// for the TMA-fed paths, whose global strides must be multiples of 16 bytes.  HBM-bound copy.
__global__ void __launch_bounds__(256)
corr_pad_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, int N, int NP, long long rows)
{
    // a block takes 64 consecutive (t, f) rows at a time; a thread builds 16 output bytes from 16 consecutive
    // input bytes at any alignment (five aligned 32-bit loads and four funnel shifts), or byte by byte at the
    // end of a row and in the last row of the stream (where reading past the 16 bytes could leave the buffer)
    const int chunks = NP >> 4;
    for (long long r0 = (long long)blockIdx.x * 64; r0 < rows; r0 += (long long)gridDim.x * 64) {
        const int nr = (int)min((long long)64, rows - r0);
        for (int i = threadIdx.x; i < nr * chunks; i += 256) {
            const int lr = i / chunks, c = i - lr * chunks;
            const long long r = r0 + lr;
            const uint8_t *src = in + r * N + 16 * c;
            uint32_t v[4];
            if (16 * c + 16 <= N && r + 1 < rows) {
                const uintptr_t a = reinterpret_cast<uintptr_t>(src);
                const uint32_t *al = reinterpret_cast<const uint32_t *>(a & ~(uintptr_t)3);
                const uint32_t sh = 8u * (uint32_t)(a & 3);
                uint32_t w[5];
#pragma unroll
                for (int k = 0; k < 5; ++k) w[k] = __ldg(al + k);
#pragma unroll
                for (int k = 0; k < 4; ++k) v[k] = __funnelshift_r(w[k], w[k + 1], sh);
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    uint32_t x = 0;
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int n = 16 * c + 4 * k + j;
                        x |= (uint32_t)((n < N) ? src[4 * k + j] : (uint8_t)0x88) << (8 * j);
                    }
                    v[k] = x;
                }
            }
            *reinterpret_cast<uint4 *>(out + r * NP + 16 * c) = make_uint4(v[0], v[1], v[2], v[3]);
        }
    }
}

}  // namespace corr
