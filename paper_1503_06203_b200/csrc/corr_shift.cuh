// corr_shift.cuh -- SURVEY section 8(f) item 4: the paper's pre-correlation time shift (PAPER.md:125-131,
// "a kernel ... that modifies the input stream at the raw data level, allowing individual elements to be
// shifted by integer time steps pre-correlation; lags can be generated or compensated for computationally").
//
//     out[t][f][n] = in[t - lag[n]][f][n]   if 0 <= t - lag[n] < T,   else 0x88 (the sample 0 + 0i)
//
// A positive lag delays element n.  Samples shifted in from outside the block are the stored form of zero,
// which adds nothing to any correlation sum.  Same layout in and out ([T][F][N] bytes).
//
// HBM-bound gather.  A tile is (channel, 128 inputs, SH_TB output samples); it needs the input rows
// [t0 - max lag, t0 + SH_TB - min lag) of its 128 inputs, its WINDOW (spread = max lag - min lag over the 128 inputs;
// read amplification (SH_TB + spread) / SH_TB).  One persistent CTA per SM walks the tiles.  A producer warp reads
// the tile's lags, finds the window and fetches it with TMA (boxes of 16 rows x 128 bytes) into a ring of rows in
// shared memory from which every tile takes as many rows as its window has: several windows are in flight whatever
// their size, which is what an HBM-bound copy needs (the first form of this kernel loaded, synchronised and
// assembled per CTA, three CTAs per SM: 3.5 TB/s; profiles/r02_secondary_kernels.md).  Sixteen consumer warps
// assemble the output: a thread one 32-bit word from the rows its four inputs' lags select (one 32-bit load when
// they share a lag), a warp one 128-byte output row per step -- lane l reads bank l whatever row the lag selects.
// A window that does not fit (spread > SH_MAX_ROWS - SH_TB): one tile in four goes through its inputs 16 at a time
// with a 16-byte-wide window that can be eight times longer, for 512 output samples (spreads up to 4096); beyond
// that, and in corr_shift_bytes_kernel for N not a multiple of 16, bytes are gathered one by one from global
// memory (correct, slow).
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "corr_ptx.cuh"

namespace corr {

constexpr int SH_TB = 128;             // output samples per tile
constexpr int SH_CWARPS = 16;          // consumer warps
constexpr int SH_CTHREADS = 32 * SH_CWARPS;
constexpr int SH_THREADS = 32 + SH_CTHREADS;
constexpr int SH_RING_ROWS = 1760;     // rows of 128 bytes in the ring: 220 KB
constexpr int SH_MAX_ROWS = 1280;      // largest window fetched by TMA: spread <= 1024 (tiles of 256 samples)
constexpr int SH_ONE_ROWS = 320;       // largest window of a tile of 128 samples; a wider spread takes tiles of 256
constexpr int SH_WIDE_ROWS = 576;      // ring rows a wide-spread tile uses as its 16-byte-wide window (x 8 rows)
constexpr int SH_SLOTS = 8;            // tiles in flight
constexpr int SH_BOX_ROWS = 16;
constexpr int SH_MAX_GROUPS = 512;     // groups of 128 inputs whose lag range fits the table: N <= 65536
constexpr int SH_SMEM_BYTES = 128 + SH_RING_ROWS * 128 + SH_MAX_GROUPS * 8 + SH_SLOTS * 16 + 2 * SH_SLOTS * 8;
enum { SH_MODE_TMA = 0, SH_MODE_WIDE = 1, SH_MODE_SKIP = 2 };

// one byte per thread and step straight from global memory: any N
__global__ void __launch_bounds__(256)
corr_shift_bytes_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, const int *__restrict__ lags,
                        int N, int F, int T)
{
    const int n0 = blockIdx.x * 128, f = blockIdx.y, t0 = blockIdx.z * SH_TB;
    const int ncols = min(128, N - n0), tcount = min(SH_TB, T - t0);
    for (int idx = threadIdx.x; idx < tcount * ncols; idx += 256) {
        const int tr = idx / ncols, n = idx % ncols;
        const long long tin = (long long)t0 + tr - lags[n0 + n];
        uint8_t b = 0x88;
        if (tin >= 0 && tin < T) b = in[((size_t)tin * F + f) * (size_t)N + n0 + n];
        out[((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + n] = b;
    }
}

// N % 16 == 0.  tmap: the input as the 3-D byte tensor (N, F, T), box (128, 1, SH_BOX_ROWS), no swizzle.
// Column n of a row has the lag lags[n % nlag]: nlag = N, or -- a stream whose N is not a multiple of 16 but whose rows
// are (F * N_stream % 16 == 0), seen as ONE channel of N = F * N_stream columns -- nlag = N_stream.
__global__ void __launch_bounds__(SH_THREADS, 1)
corr_shift_kernel(const __grid_constant__ CUtensorMap tmap, const uint8_t *__restrict__ in, uint8_t *__restrict__ out,
                  const int *__restrict__ lags, int N, int F, int T, int nlag)
{
    extern __shared__ uint8_t sh_raw[];
    const uint32_t base = (ptx::smem_u32(sh_raw) + 127u) & ~127u;
    uint8_t *ring = sh_raw + (base - ptx::smem_u32(sh_raw));
    int2 *glohi = reinterpret_cast<int2 *>(ring + SH_RING_ROWS * 128);       // [G]: (min, max) lag of the group's inputs
    int4 *meta = reinterpret_cast<int4 *>(glohi + SH_MAX_GROUPS);            // [SH_SLOTS]: (first ring row, max lag, min lag, mode)
    const uint32_t bar0 = base + SH_RING_ROWS * 128 + SH_MAX_GROUPS * 8 + SH_SLOTS * 16;
    auto full = [&](int s) { return bar0 + 8u * s; };
    auto empty = [&](int s) { return bar0 + 8u * (SH_SLOTS + s); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = (N + 127) >> 7, ntb = (T + SH_TB - 1) / SH_TB;
    const long long total = (long long)ntb * F * G;

    if (threadIdx.x == 0) {
        ptx::prefetch_tmap(&tmap);
        for (int s = 0; s < SH_SLOTS; ++s) {
            ptx::mbar_init(full(s), 1);
            ptx::mbar_init(empty(s), SH_CWARPS);
        }
        ptx::fence_mbar_init();
    }
    for (int g = warp; g < G; g += SH_THREADS / 32) {
        int lo = 0x7fffffff, hi = (int)0x80000000;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (g * 128 + 4 * lane + j < N) {
                const int l = __ldg(lags + (g * 128 + 4 * lane + j) % nlag);
                lo = min(lo, l);
                hi = max(hi, l);
            }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, o));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, o));
        }
        if (lane == 0) glohi[g] = make_int2(lo, hi);
    }
    __syncthreads();

    // tiles blockIdx.x, blockIdx.x + gridDim.x, ...: tile i = (tb * F + f) * G + g, decoded incrementally
    const int dg = (int)(gridDim.x % G), df = (int)((gridDim.x / G) % F), dtb = (int)(gridDim.x / ((long long)G * F));
    int g = (int)(blockIdx.x % G), f = (int)((blockIdx.x / G) % F), tb = (int)(blockIdx.x / ((long long)G * F));
    auto next_tile = [&]() {
        g += dg;
        if (g >= G) { g -= G; ++f; }
        f += df;
        if (f >= F) { f -= F; ++tb; }
        tb += dtb;
    };

    if (warp == 0) {
        // ===================== producer: window -> TMA =====================
        int head = 0, used = 0;          // next free ring row; rows between the oldest tile in flight and head
        int oldest = 0, k = 0;           // tiles of this CTA: first one in flight, next one
        int span_of = 0;                 // lane s keeps the ring rows slot s holds (its padding included)
        for (long long i = blockIdx.x; i < total; i += gridDim.x, ++k, next_tile()) {
            const int n0 = g * 128, t0 = tb * SH_TB;
            const int2 lh = glohi[g];
            const int lo = lh.x, hi = lh.y;
            const long long rows = (long long)SH_TB + (long long)hi - (long long)lo;
            // time blocks per tile: two when the spread is wide (half the re-reading of the spread; the tiles of
            // the odd time blocks are then empty)
            int mode, need;
            if (rows <= SH_ONE_ROWS) {
                mode = SH_MODE_TMA | (1 << 8);
                need = ((int)rows + SH_BOX_ROWS - 1) / SH_BOX_ROWS * SH_BOX_ROWS;
            } else if (rows + SH_TB <= SH_MAX_ROWS) {
                mode = (tb & 1) ? SH_MODE_SKIP : (SH_MODE_TMA | (2 << 8));
                need = (tb & 1) ? 0 : ((int)rows + SH_TB + SH_BOX_ROWS - 1) / SH_BOX_ROWS * SH_BOX_ROWS;
            } else if ((tb & 3) == 0) {
                mode = SH_MODE_WIDE;
                need = SH_WIDE_ROWS;
            } else {
                mode = SH_MODE_SKIP;
                need = 0;
            }
            // a window is contiguous: one that would run over the end of the ring starts at row 0 and the rows left
            // over count as its own.  Room in the ring and a free slot: tiles finish in order
            int span;
            bool wrap;
            for (;;) {
                wrap = head + need > SH_RING_ROWS;
                span = (wrap ? SH_RING_ROWS - head : 0) + need;
                if (used + span <= SH_RING_ROWS && k - oldest < SH_SLOTS) break;
                const int os = oldest % SH_SLOTS;
                ptx::mbar_wait(empty(os), (uint32_t)((oldest / SH_SLOTS) & 1));
                used -= __shfl_sync(0xffffffffu, span_of, os);
                if (++oldest == k) { head = 0; used = 0; }
            }
            const int slot = k % SH_SLOTS;
            const int row0 = wrap ? 0 : head;
            head = row0 + need;
            used += span;
            if (lane == slot) span_of = span;
            if (lane == 0) {
                meta[slot] = make_int4(row0, hi, lo, mode);
                if ((mode & 255) == SH_MODE_TMA) ptx::mbar_arrive_expect_tx(full(slot), (uint32_t)need * 128u);
                else ptx::mbar_arrive(full(slot));
            }
            __syncwarp();
            if ((mode & 255) == SH_MODE_TMA) {
                // a window a billion samples outside the stream is just outside the stream (the coordinate is 32 bits)
                const long long ts = (long long)t0 - (long long)hi;
                const int tc = (int)max(-(1ll << 30), min(1ll << 30, ts));
                for (int b = lane; b < need / SH_BOX_ROWS; b += 32)
                    ptx::tma_load_3d(base + (uint32_t)(row0 + SH_BOX_ROWS * b) * 128u, &tmap, full(slot), n0, f,
                                     tc + SH_BOX_ROWS * b);
            }
        }
    } else {
        // ===================== consumers: assemble the output rows =====================
        const int cw = warp - 1, ct = threadIdx.x - 32;
        const size_t ostride = (size_t)F * N;
        int k = 0;
        for (long long i = blockIdx.x; i < total; i += gridDim.x, ++k, next_tile()) {
            const int n0 = g * 128, t0 = tb * SH_TB;
            const int ncols = min(128, N - n0);
            const int slot = k % SH_SLOTS;
            int4 lv = make_int4(0, 0, 0, 0);   // the lags of this thread's four inputs
            if (4 * lane < ncols) {
                if (nlag == N) {
                    lv = __ldg(reinterpret_cast<const int4 *>(lags + n0) + lane);
                } else {
                    const int c = n0 + 4 * lane;
                    lv = make_int4(__ldg(lags + c % nlag), __ldg(lags + (c + 1) % nlag), __ldg(lags + (c + 2) % nlag),
                                   __ldg(lags + (c + 3) % nlag));
                }
            }
            ptx::mbar_wait(full(slot), (uint32_t)((k / SH_SLOTS) & 1));
            const int4 m = meta[slot];
            uint8_t *win = ring + m.x * 128;
            const int hi = m.y, lo = m.z;
            if ((m.w & 255) == SH_MODE_TMA) {
                const int l0 = lv.x, l1 = lv.y, l2 = lv.z, l3 = lv.w;
                const int d1 = (l0 - l1) * 128 + 1, d2 = (l0 - l2) * 128 + 2, d3 = (l0 - l3) * 128 + 3;
                const size_t ostep = ostride * SH_CWARPS;
                for (int sb = 0; sb < (m.w >> 8); ++sb) {
                    const int ts = t0 + sb * SH_TB;                 // first sample of this block of SH_TB output rows
                    const int tcount = min(SH_TB, T - ts);
                    if (tcount <= 0 || 4 * lane >= ncols) break;
                    // rows before sample 0 or after sample T - 1 arrive as zero bytes, the stored zero is 0x88
                    const bool edge = ((long long)ts - hi < 0) || ((long long)ts + tcount - 1 - lo >= T);
                    uint8_t *o = out + ((size_t)(ts + cw) * F + f) * (size_t)N + n0 + 4 * lane;
                    const uint8_t *w0 = win + (sb * SH_TB + cw + hi - l0) * 128 + 4 * lane;
                    if (!edge && tcount == SH_TB && d1 == 1 && d2 == 2 && d3 == 3) {
#pragma unroll
                        for (int r = 0; r < SH_TB / SH_CWARPS; ++r)
                            *reinterpret_cast<uint32_t *>(o + r * ostep) =
                                *reinterpret_cast<const uint32_t *>(w0 + r * (SH_CWARPS * 128));
                    } else if (!edge && tcount == SH_TB) {
                        uint32_t v[SH_TB / SH_CWARPS];
#pragma unroll
                        for (int r = 0; r < SH_TB / SH_CWARPS; ++r) {
                            const uint8_t *rowp = w0 + r * (SH_CWARPS * 128);
                            const uint32_t b0 = rowp[0], b1 = rowp[d1], b2 = rowp[d2], b3 = rowp[d3];
                            v[r] = __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                        }
#pragma unroll
                        for (int r = 0; r < SH_TB / SH_CWARPS; ++r) *reinterpret_cast<uint32_t *>(o + r * ostep) = v[r];
                    } else {
                        for (int tr = cw, r = 0; tr < tcount; tr += SH_CWARPS, ++r) {
                            const uint8_t *rowp = w0 + r * (SH_CWARPS * 128);
                            const long long t = (long long)ts + tr;
                            const uint32_t b0 = (t - l0 >= 0 && t - l0 < T) ? rowp[0] : 0x88u;
                            const uint32_t b1 = (t - l1 >= 0 && t - l1 < T) ? rowp[d1] : 0x88u;
                            const uint32_t b2 = (t - l2 >= 0 && t - l2 < T) ? rowp[d2] : 0x88u;
                            const uint32_t b3 = (t - l3 >= 0 && t - l3 < T) ? rowp[d3] : 0x88u;
                            *reinterpret_cast<uint32_t *>(o + r * ostep) = __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                        }
                    }
                }
            } else if ((m.w & 255) == SH_MODE_WIDE) {
                // one group of 16 inputs at a time through a 16-byte-wide window of up to 8 SH_WIDE_ROWS rows, for the
                // 512 output rows of this tile and the three after it along t (their CTAs skip them).  A thread assembles
                // one 32-bit word; a warp covers 8 rows x 4 words = 32 distinct banks (rows are 16 bytes apart)
                const int tcw = min(4 * SH_TB, T - t0);
                const int c16n = ncols >> 4;
                const int w = ct & 3, rl = ct >> 2;
                auto lag_of = [&](int n) { return __ldg(lags + (n0 + n) % nlag); };
                for (int c = 0; c < c16n; ++c) {
                    int glo = 0x7fffffff, ghi = (int)0x80000000;
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const int l = lag_of(16 * c + j);
                        glo = min(glo, l);
                        ghi = max(ghi, l);
                    }
                    const long long grows = (long long)tcw + (long long)ghi - (long long)glo;
                    if (grows <= SH_WIDE_ROWS * 8) {
                        ptx::named_bar_sync(1, SH_CTHREADS);   // the previous group's window is no longer read
                        for (int r = ct; r < (int)grows; r += SH_CTHREADS) {
                            const long long tin = (long long)t0 - ghi + r;
                            uint4 v = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
                            if (tin >= 0 && tin < T)
                                v = __ldg(reinterpret_cast<const uint4 *>(in + ((size_t)tin * F + f) * (size_t)N + n0 + 16 * c));
                            *reinterpret_cast<uint4 *>(win + r * 16) = v;
                        }
                        ptx::named_bar_sync(1, SH_CTHREADS);
                        const int o0 = (ghi - lag_of(16 * c + 4 * w + 0)) * 16 + 4 * w + 0, o1 = (ghi - lag_of(16 * c + 4 * w + 1)) * 16 + 4 * w + 1;
                        const int o2 = (ghi - lag_of(16 * c + 4 * w + 2)) * 16 + 4 * w + 2, o3 = (ghi - lag_of(16 * c + 4 * w + 3)) * 16 + 4 * w + 3;
                        for (int tr = rl; tr < tcw; tr += SH_CTHREADS / 4) {
                            const uint8_t *rowp = win + tr * 16;
                            const uint32_t b0 = rowp[o0], b1 = rowp[o1], b2 = rowp[o2], b3 = rowp[o3];
                            *reinterpret_cast<uint32_t *>(out + ((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + 16 * c + 4 * w) =
                                __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                        }
                    } else {
                        for (int idx = ct; idx < tcw * 16; idx += SH_CTHREADS) {
                            const int tr = idx >> 4, n = 16 * c + (idx & 15);
                            const long long tin = (long long)t0 + tr - lag_of(n);
                            uint8_t b = 0x88;
                            if (tin >= 0 && tin < T) b = in[((size_t)tin * F + f) * (size_t)N + n0 + n];
                            out[((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + n] = b;
                        }
                    }
                }
                ptx::fence_proxy_async_smem();   // the ring rows go back to TMA
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty(slot));
        }
    }
}

}  // namespace corr
