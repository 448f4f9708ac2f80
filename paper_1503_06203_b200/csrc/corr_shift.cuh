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
// thread assembles 16 output bytes from the rows its inputs' lags select and writes them with one 16-byte
// store (a single 16-byte shared-memory load when the 16 inputs share one lag, the common case of a few
// cable lengths).  Read amplification (SH_TB + spread) / SH_TB, spread = max lag - min lag over the 128 inputs.  When
// the spread does not fit, the CTA goes through its inputs 16 at a time with a 16-byte-wide window that can be
// eight times longer (spreads up to 4480 samples); beyond that, or when N is not a multiple of 16, it gathers
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
        // ---- assemble 16 output bytes per thread
        // (SH_THREADS is a multiple of 8, so a thread keeps its column group c for every row it handles)
        const int c = tid & 7;
        bool same = true;
        int off[16];   // shared-memory offset of this thread's 16 inputs relative to output row 0 (loop invariant)
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            same = same && (slag[16 * c + j] == slag[16 * c]);
            off[j] = (hi - slag[16 * c + j]) * 128 + 16 * c + j;
        }
        if (c < c16n) {
            for (int tr = tid >> 3; tr < tcount; tr += SH_THREADS / 8) {
                uint4 v;
                if (same) {
                    v = *reinterpret_cast<const uint4 *>(tile + tr * 128 + off[0]);
                } else {
                    const uint8_t *rowp = tile + tr * 128;
                    uint32_t w[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const uint32_t b0 = rowp[off[4 * q + 0]], b1 = rowp[off[4 * q + 1]];
                        const uint32_t b2 = rowp[off[4 * q + 2]], b3 = rowp[off[4 * q + 3]];
                        w[q] = __byte_perm(b0 | (b1 << 8), b2 | (b3 << 8), 0x5410);
                    }
                    v = make_uint4(w[0], w[1], w[2], w[3]);
                }
                *reinterpret_cast<uint4 *>(out + ((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + 16 * c) = v;
            }
        }
    } else if ((N & 15) == 0) {
        // ---- wide spread: one group of 16 inputs at a time, so the window is 16 bytes wide and can be
        //      8 x longer (spreads up to SH_MAX_ROWS * 8 - SH_TB rows inside a group of 16 inputs)
        const int c16n = ncols >> 4;
        for (int c = 0; c < c16n; ++c) {
            int glo = 0x7fffffff, ghi = (int)0x80000000;
#pragma unroll
            for (int j = 0; j < 16; ++j) { glo = min(glo, slag[16 * c + j]); ghi = max(ghi, slag[16 * c + j]); }
            const long long grows = (long long)SH_TB + (long long)ghi - (long long)glo;
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
                for (int tr = tid; tr < tcount; tr += SH_THREADS) {
                    uint32_t w[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        uint32_t acc = 0;
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int n = 4 * q + j;
                            acc |= (uint32_t)tile[(tr + ghi - slag[16 * c + n]) * 16 + n] << (8 * j);
                        }
                        w[q] = acc;
                    }
                    *reinterpret_cast<uint4 *>(out + ((size_t)(t0 + tr) * F + f) * (size_t)N + n0 + 16 * c) =
                        make_uint4(w[0], w[1], w[2], w[3]);
                }
            } else {
                for (int idx = tid; idx < tcount * 16; idx += SH_THREADS) {
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
