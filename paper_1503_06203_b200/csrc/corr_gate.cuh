// corr_gate.cuh -- SURVEY section 8(f) item 3: gated correlation ("the correlation kernel has
// also been extended to gate the correlation products on multiple time periods ... useful for analysis of
// data where periodic signals occur (e.g., artificial calibration signals, and pulsars)").
//
// Every time sample belongs to one of G gates (or to none); gate g gets its own correlation matrix
//     A_g[f][x][y] = sum over { t : gate[t] = g } of X_t[x] conj(X_t[y])        (Eq. 1)
// The sum over a subset of the samples is the ordinary correlation of the stream made of exactly those
// samples, so gating is done at the raw data level, like the paper's time shift: this kernel gathers the
// rows (time samples) of each gate into one contiguous run -- an HBM-bound row copy, F*N bytes per row --
// and the ordinary kernels then run once per gate on its run.  No arithmetic of the method lives here.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace corr {

constexpr int GATE_THREADS = 256;

// out row j = in row order[j], rows of row_bytes bytes (a multiple of 16, 16-byte aligned).
__global__ void __launch_bounds__(GATE_THREADS)
corr_gate_gather_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, const int *__restrict__ order,
                        int nrows, int row_vecs)
{
    const long long total = (long long)nrows * row_vecs;
    for (long long i = (long long)blockIdx.x * GATE_THREADS + threadIdx.x; i < total;
         i += (long long)gridDim.x * GATE_THREADS) {
        const int j = (int)(i / row_vecs), v = (int)(i % row_vecs);
        const uint4 *src = reinterpret_cast<const uint4 *>(in) + (size_t)order[j] * row_vecs + v;
        reinterpret_cast<uint4 *>(out)[i] = __ldg(src);
    }
}

// the gates side by side: out row j * G + g = in row order[gates[g].x + j] for j < gates[g].y (the gate's count), else a
// row of stored zeros (0x88: the sample 0 + 0i); j < tmax
__global__ void __launch_bounds__(GATE_THREADS)
corr_gate_gather_merged_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out, const int *__restrict__ order,
                               const int2 *__restrict__ gates, int G, int tmax, int row_vecs)
{
    const long long total = (long long)tmax * G * row_vecs;
    for (long long i = (long long)blockIdx.x * GATE_THREADS + threadIdx.x; i < total;
         i += (long long)gridDim.x * GATE_THREADS) {
        const long long r = i / row_vecs;
        const int v = (int)(i - r * row_vecs), j = (int)(r / G), g = (int)(r - (long long)j * G);
        const int2 sc = __ldg(gates + g);
        uint4 w = make_uint4(0x88888888u, 0x88888888u, 0x88888888u, 0x88888888u);
        if (j < sc.y) w = __ldg(reinterpret_cast<const uint4 *>(in) + (size_t)__ldg(order + sc.x + j) * row_vecs + v);
        reinterpret_cast<uint4 *>(out)[i] = w;
    }
}

// same for rows that are not a multiple of 16 bytes
__global__ void __launch_bounds__(GATE_THREADS)
corr_gate_gather_bytes_kernel(const uint8_t *__restrict__ in, uint8_t *__restrict__ out,
                              const int *__restrict__ order, int nrows, int row_bytes)
{
    const long long total = (long long)nrows * row_bytes;
    for (long long i = (long long)blockIdx.x * GATE_THREADS + threadIdx.x; i < total;
         i += (long long)gridDim.x * GATE_THREADS) {
        const int j = (int)(i / row_bytes), b = (int)(i % row_bytes);
        out[i] = in[(size_t)order[j] * row_bytes + b];
    }
}

}  // namespace corr
