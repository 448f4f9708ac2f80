// corr_shift.cuh -- SURVEY section 8(f) item 4: the paper's pre-correlation time shift (PAPER.md:125-131,
// "a kernel ... that modifies the input stream at the raw data level, allowing individual elements to be
// shifted by integer time steps pre-correlation; lags can be generated or compensated for computationally").
//
//     out[t][f][n] = in[t - lag[n]][f][n]   if 0 <= t - lag[n] < T,   else 0x88 (the sample 0 + 0i)
//
// A positive lag delays element n.  Samples shifted in from outside the block are the stored form of zero,
// which adds nothing to any correlation sum.  Same layout in and out ([T][F][N] bytes).
//
// HBM-bound gather: a CTA owns (channel, 128 inputs, SH_TB output samples); it loads the input rows
// [t0 - max lag, t0 + SH_TB - min lag) of its 128 inputs into shared memory with 16-byte loads, then every
// thread assembles one 32-bit word of an output row from the rows its four inputs' lags select (a single 32-bit
// shared-memory load when they share one lag) and a warp writes the 128-byte row.  Read amplification (SH_TB + spread) / SH_TB, spread = max lag - min lag over the 128 inputs.  When
// the spread does not fit, one CTA in four goes through its inputs 16 at a time with a 16-byte-wide window that can be
// eight times longer, for 512 output samples (spreads up to 4096 samples); beyond that, or when N is not a multiple of 16, it gathers
// byte by byte from global memory (correct, slow).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace corr {

constexpr int SH_TB = 128;          // output samples per CTA
constexpr int SH_THREADS = 256;
constexpr int SH_MAX_ROWS = 576;    // input rows a CTA can stage: 72 KB, three CTAs per SM; spread <= 448
constexpr int SH_SMEM_BYTES = SH_MAX_ROWS * 128 + 128 * 4 + 16;

__global__ void __launch_bounds__(SH_THREADS)
corr_shift_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, const int *__restrict__ lags,
                  int N, int F, int T)
{
    extern __shared__ __align__(16) uint8_t sh_raw[];
    uint8_t *tile = sh_raw;
    int *slag = reinterpret_cast<int *>(sh_raw + SH_MAX_ROWS * 128);
    int *smm = slag + 128;   // [0] = min lag, [1] = max lag of this CTA's inputs

    const int n0 = blockIdx.x * 128, f = blockIdx.y, t0 = blockIdx.z * SH_TB;
    const int ncols = min(128, N - n0);
    const int tid = threadIdx.x;
    if (tid == 0) { smm[0] = 0x7fffffff; smm[1] = (int)0x80000000; }
    __syncthreads();
    if (tid < 128) {
        const int l = (tid < ncols) ? lags[n0 + tid] : 0;
        slag[tid] = l;
        if (tid < ncols) { atomicMin(&smm[0], l); atomicMax(&smm[1], l); }
    }
    __syncthreads();
    const int lo = smm[0], hi = smm[1];
    const long long rows = (long long)SH_TB + (long long)hi - (long long)lo;
    const int tcount = min(SH_TB, T - t0);

    if ((N & 15) == 0 && rows <= SH_MAX_ROWS) {
        // ---- stage rows [t0 - hi, t0 - hi + rows) of the 128 inputs
        const int c16n = ncols >> 4;
#pragma unroll 4
        for (int idx = tid; idx < (int)rows * 8; idx += SH_THREADS) {
            const int r = idx >> 3, c = idx & 7;
            const long long tin = (long long)t0 - hi + r;
            uint4 v = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
            if (c < c16n && tin >= 0 && tin < T)
                v = __ldg(reinterpret_cast<const uint4 *>(in + ((size_t)tin * F + f) * (size_t)N + n0 + 16 * c));
            *reinterpret_cast<uint4 *>(tile + r * 128 + 16 * c) = v;
        }
        __syncthreads();
        // ---- assemble one 32-bit word (4 inputs) per thread: a warp writes one output row of 128 bytes per step.
        //      Lane l owns word l of the row whatever source row its lags select, and the staged rows are 128 bytes
        //      = 32 banks apart, so the byte loads of a warp fall on 32 distinct banks (a thread that gathered 16
        //      bytes met the other rows of its warp on the same banks: 4-way conflicts, profiles/r02_secondary_kernels.md)
        const int wq = tid & 31;            // word of the row: inputs 4 wq .. 4 wq + 3
        const int off0 = (hi - slag[4 * wq + 0]) * 128 + 4 * wq + 0, off1 = (hi - slag[4 * wq + 1]) * 128 + 4 * wq + 1;
        const int off2 = (hi - slag[4 * wq + 2]) * 128 + 4 * wq + 2, off3 = (hi - slag[4 * wq + 3]) * 128 + 4 * wq + 3;
        const bool same = (off1 == off0 + 1) && (off2 == off0 + 2) && (off3 == off0 + 3);   // the four inputs share a lag
        if ((wq >> 2) < c16n) {
            for (int tr = tid >> 5; tr < tcount; tr += SH_THREADS / 32) {
                const uint8_t *rowp = tile + tr * 128;
                uint32_t v;
                if (same) {
                    v = *reinterpret_cast<const uint32_t *>(rowp + off0);
                } else {
                    const uint32_t b0 = rowp[off0], b1 = rowp[off1], b2 = rowp[off2], b3 = rowp[off3];
                    v = __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                }
                *reinterpret_cast<uint32_t *>(out + ((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + 4 * wq) = v;
            }
        }
    } else if ((N & 15) == 0) {
        // ---- wide spread: one group of 16 inputs at a time, so the window is 16 bytes wide and can be 8 x longer.
        //      Four consecutive CTAs along t share the work of one (the other three leave): 512 output rows per
        //      window instead of 128 cut the re-read of the spread by four.  A thread assembles one 32-bit word;
        //      a warp covers 8 rows x 4 words, which fall on 32 distinct banks (rows are 16 bytes = 4 banks apart).
        if (blockIdx.z & 3) return;
        const int tcw = min(4 * SH_TB, T - t0);
        const int c16n = ncols >> 4;
        const int w = tid & 3, rl = tid >> 2;          // word of the group, row inside a block of 64 rows
        for (int c = 0; c < c16n; ++c) {
            int glo = 0x7fffffff, ghi = (int)0x80000000;
#pragma unroll
            for (int j = 0; j < 16; ++j) { glo = min(glo, slag[16 * c + j]); ghi = max(ghi, slag[16 * c + j]); }
            const long long grows = (long long)tcw + (long long)ghi - (long long)glo;
            if (grows <= SH_MAX_ROWS * 8) {
                __syncthreads();   // the previous group's window is no longer read
                for (int r = tid; r < (int)grows; r += SH_THREADS) {
                    const long long tin = (long long)t0 - ghi + r;
                    uint4 v = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
                    if (tin >= 0 && tin < T)
                        v = __ldg(reinterpret_cast<const uint4 *>(in + ((size_t)tin * F + f) * (size_t)N + n0 + 16 * c));
                    *reinterpret_cast<uint4 *>(tile + r * 16) = v;
                }
                __syncthreads();
                const int o0 = (ghi - slag[16 * c + 4 * w + 0]) * 16 + 4 * w + 0, o1 = (ghi - slag[16 * c + 4 * w + 1]) * 16 + 4 * w + 1;
                const int o2 = (ghi - slag[16 * c + 4 * w + 2]) * 16 + 4 * w + 2, o3 = (ghi - slag[16 * c + 4 * w + 3]) * 16 + 4 * w + 3;
                for (int tr = rl; tr < tcw; tr += SH_THREADS / 4) {
                    const uint8_t *rowp = tile + tr * 16;
                    const uint32_t b0 = rowp[o0], b1 = rowp[o1], b2 = rowp[o2], b3 = rowp[o3];
                    *reinterpret_cast<uint32_t *>(out + ((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + 16 * c + 4 * w) =
                        __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                }
            } else {
                for (int idx = tid; idx < tcw * 16; idx += SH_THREADS) {
                    const int tr = idx >> 4, n = 16 * c + (idx & 15);
                    const long long tin = (long long)t0 + tr - slag[n];
                    uint8_t b = 0x88;
                    if (tin >= 0 && tin < T) b = in[((size_t)tin * F + f) * (size_t)N + n0 + n];
                    out[((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + n] = b;
                }
            }
        }
    } else {
        // ---- general path: one byte per thread-iteration straight from global memory
        for (int idx = tid; idx < tcount * ncols; idx += SH_THREADS) {
            const int tr = idx / ncols, n = idx % ncols;
            const long long tin = (long long)t0 + tr - slag[n];
            uint8_t b = 0x88;
            if (tin >= 0 && tin < T) b = in[((size_t)tin * F + f) * (size_t)N + n0 + n];
            out[((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + n] = b;
        }
    }
}

}  // namespace corr
