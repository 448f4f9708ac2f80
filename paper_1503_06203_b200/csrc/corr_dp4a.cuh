// corr_dp4a.cuh -- step S4' of the hot path: the CUDA-core dp4a correlation kernel.
//
// Serves small N, where a 128-wide tensor-core tile would waste most of its work
// (the paper makes the same observation for its own tiles: "A tile size of 32x32 ... for large N
// (N >~ 128)"), and every N the tcgen05 path cannot take (N % 16 != 0).
//
// Formulation (Eq. 1): for a pair of time samples (t, t+1) each input n is held
// as two 4 x int8 words
//      P[n] = [ Re(t),  Im(t),  Re(t+1),  Im(t+1) ]
//      Q[n] = [-Im(t),  Re(t), -Im(t+1),  Re(t+1) ]      (the conjugate-rotated copy)
// so that   Re A[x][y] += dp4a(P[x], P[y])   and   Im A[x][y] += dp4a(P[x], Q[y]):
// one dp4a per complex multiply-accumulate (cMAC).
//
// One CTA owns one (channel, tile, T-slab) work unit.  Tiles are TS x TS inputs and only tiles
// on or above the diagonal exist in the tile table.  256 threads; a thread owns
// a 4x4 block of baselines.  For TS < 64 the CTA's threads split into G = 256/(TS/4)^2 groups
// that take different time pairs of a stage and are summed through shared memory at the end.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace corr {

enum OutMode : int { OUT_STORE = 0, OUT_RMW = 1, OUT_ATOMIC = 2 };

constexpr int DP4A_THREADS = 256;
constexpr int DP4A_TK = 32;              // time samples per stage
constexpr int DP4A_PAIRS = DP4A_TK / 2;  // dp4a words per input per stage

__device__ __forceinline__ size_t baseline_index(size_t N, size_t x, size_t y)
{
    return x * N - x * (x - 1) / 2 + (y - x);
}

// 4 consecutive inputs of one (t, f) row as a 32-bit word; anything outside the stream reads as
// 0x88 = 0+0i, which adds nothing to any sum.
__device__ __forceinline__ uint32_t load4(const uint8_t *__restrict__ packed, int N, int F, int T,
                                          int f, int t, int n, bool aligned)
{
    if (t >= T) return 0x88888888u;
    const uint8_t *row = packed + ((size_t)t * F + f) * (size_t)N;
    if (aligned && n + 3 < N) return __ldg(reinterpret_cast<const uint32_t *>(row + n));
    uint32_t w = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        uint32_t b = (n + j < N) ? (uint32_t)__ldg(row + n + j) : 0x88u;
        w |= b << (8 * j);
    }
    return w;
}

// (W0, W1) = 4 inputs at times t and t+1  ->  P[0..3], Q[0..3] as defined above.
__device__ __forceinline__ void make_pq(uint32_t W0, uint32_t W1, uint4 &P, uint4 &Q)
{
    const uint32_t hiA = (W0 >> 4) & 0x0F0F0F0Fu, loA = W0 & 0x0F0F0F0Fu;  // stored Re', Im' at t
    const uint32_t hiB = (W1 >> 4) & 0x0F0F0F0Fu, loB = W1 & 0x0F0F0F0Fu;  // at t+1
    const uint32_t a = __byte_perm(hiA, loA, 0x5140), b = __byte_perm(hiA, loA, 0x7362);
    const uint32_t c = __byte_perm(hiB, loB, 0x5140), d = __byte_perm(hiB, loB, 0x7362);
    uint32_t u[4] = {__byte_perm(a, c, 0x5410), __byte_perm(a, c, 0x7632),
                     __byte_perm(b, d, 0x5410), __byte_perm(b, d, 0x7632)};  // [Re',Im',Re',Im'] per input
    uint32_t p[4], q[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        // stored nibble s in [0,15] -> s-8 as int8: (s + 0x78) ^ 0x80, no carry between bytes
        p[j] = (u[j] + 0x78787878u) ^ 0x80808080u;
        // swap Re'/Im' within each time sample; Im' -> 8-Im' = -Im via (15-s)+0x79, Re' -> Re'-8
        const uint32_t v = __byte_perm(u[j], 0, 0x2301);
        q[j] = ((v ^ 0x000F000Fu) + 0x78797879u) ^ 0x80808080u;
    }
    P = make_uint4(p[0], p[1], p[2], p[3]);
    Q = make_uint4(q[0], q[1], q[2], q[3]);
}

template <int TS>
__global__ void __launch_bounds__(DP4A_THREADS)
corr_dp4a_kernel(const uint8_t *__restrict__ packed, int32_t *__restrict__ vis,
                 const ushort2 *__restrict__ tiles, int ntiles, int N, int F, int T,
                 int t_per_slab, int out_mode, int aligned)
{
    constexpr int NT = TS / 4;                 // threads per tile edge
    constexpr int GS = NT * NT;                // threads per time group
    constexpr int G = DP4A_THREADS / GS;       // time groups
    constexpr int ITEMS = DP4A_PAIRS * NT;     // staging items per block side per stage
    constexpr int IPT = (ITEMS + DP4A_THREADS - 1) / DP4A_THREADS;
    static_assert(G >= 1 && DP4A_PAIRS % G == 0, "bad tile size");

    __shared__ __align__(16) uint32_t sPx[DP4A_PAIRS][TS];
    __shared__ __align__(16) uint32_t sPy[DP4A_PAIRS][TS];
    __shared__ __align__(16) uint32_t sQy[DP4A_PAIRS][TS];
    __shared__ int32_t sRed[(G > 1) ? GS * 32 : 1];

    const int tid = threadIdx.x;
    const int f = blockIdx.x / ntiles;
    const ushort2 tile = tiles[blockIdx.x % ntiles];
    const int x0 = tile.x * TS, y0 = tile.y * TS;
    const bool diag = (tile.x == tile.y);
    const int t_begin = blockIdx.y * t_per_slab;
    const int t_end = min(T, t_begin + t_per_slab);

    const int grp = tid / GS, r = tid % GS;
    const int ty = r / NT, tx = r % NT;
    const bool active = !(diag && ty > tx);    // 4x4 block entirely below the diagonal

    int32_t re[4][4], im[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) re[i][j] = im[i][j] = 0;

    uint32_t wx[IPT][2], wy[IPT][2];
    auto fetch = [&](int t0) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const int it = tid + k * DP4A_THREADS;
            if (it < ITEMS) {
                const int p = it / NT, g = it % NT;
                const int t = t0 + 2 * p;
                const int tl = (t < t_end) ? t : T, tl1 = (t + 1 < t_end) ? t + 1 : T;
                wx[k][0] = load4(packed, N, F, T, f, tl, x0 + 4 * g, aligned);
                wx[k][1] = load4(packed, N, F, T, f, tl1, x0 + 4 * g, aligned);
                if (!diag) {
                    wy[k][0] = load4(packed, N, F, T, f, tl, y0 + 4 * g, aligned);
                    wy[k][1] = load4(packed, N, F, T, f, tl1, y0 + 4 * g, aligned);
                }
            }
        }
    };

    fetch(t_begin);
    for (int t0 = t_begin; t0 < t_end; t0 += DP4A_TK) {
#pragma unroll
        for (int k = 0; k < IPT; ++k) {
            const int it = tid + k * DP4A_THREADS;
            if (it < ITEMS) {
                const int p = it / NT, g = it % NT;
                uint4 P, Q;
                make_pq(wx[k][0], wx[k][1], P, Q);
                *reinterpret_cast<uint4 *>(&sPx[p][4 * g]) = P;
                if (diag) {
                    *reinterpret_cast<uint4 *>(&sPy[p][4 * g]) = P;
                    *reinterpret_cast<uint4 *>(&sQy[p][4 * g]) = Q;
                } else {
                    make_pq(wy[k][0], wy[k][1], P, Q);
                    *reinterpret_cast<uint4 *>(&sPy[p][4 * g]) = P;
                    *reinterpret_cast<uint4 *>(&sQy[p][4 * g]) = Q;
                }
            }
        }
        __syncthreads();
        if (t0 + DP4A_TK < t_end) fetch(t0 + DP4A_TK);
        if (active) {
#pragma unroll
            for (int pp = 0; pp < DP4A_PAIRS / G; ++pp) {
                const int p = grp + pp * G;
                const uint4 a = *reinterpret_cast<const uint4 *>(&sPx[p][4 * ty]);
                const uint4 b = *reinterpret_cast<const uint4 *>(&sPy[p][4 * tx]);
                const uint4 c = *reinterpret_cast<const uint4 *>(&sQy[p][4 * tx]);
                const int av[4] = {(int)a.x, (int)a.y, (int)a.z, (int)a.w};
                const int bv[4] = {(int)b.x, (int)b.y, (int)b.z, (int)b.w};
                const int cv[4] = {(int)c.x, (int)c.y, (int)c.z, (int)c.w};
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        re[i][j] = __dp4a(av[i], bv[j], re[i][j]);
                        im[i][j] = __dp4a(av[i], cv[j], im[i][j]);
                    }
            }
        }
        __syncthreads();
    }

    if (G > 1) {  // sum the time groups
        for (int i = tid; i < GS * 32; i += DP4A_THREADS) sRed[i] = 0;
        __syncthreads();
        if (active) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    // bank = (k*GS + r) % 32: conflict-free across the lanes of a group
                    atomicAdd(&sRed[((i * 4 + j) * 2 + 0) * GS + r], re[i][j]);
                    atomicAdd(&sRed[((i * 4 + j) * 2 + 1) * GS + r], im[i][j]);
                }
        }
        __syncthreads();
        if (grp != 0) return;
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                re[i][j] = sRed[((i * 4 + j) * 2 + 0) * GS + r];
                im[i][j] = sRed[((i * 4 + j) * 2 + 1) * GS + r];
            }
    }
    if (!active) return;

    const size_t B = (size_t)N * ((size_t)N + 1) / 2;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int x = x0 + 4 * ty + i;
        if (x >= N) continue;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int y = y0 + 4 * tx + j;
            if (y >= N || y < x) continue;  // entries below the diagonal do not exist
            int32_t *o = vis + ((size_t)f * B + baseline_index(N, x, y)) * 2;
            if (out_mode == OUT_STORE) {
                *reinterpret_cast<int2 *>(o) = make_int2(re[i][j], im[i][j]);
            } else if (out_mode == OUT_RMW) {
                int2 v = *reinterpret_cast<int2 *>(o);
                v.x += re[i][j];
                v.y += im[i][j];
                *reinterpret_cast<int2 *>(o) = v;
            } else {
                atomicAdd(o + 0, re[i][j]);
                atomicAdd(o + 1, im[i][j]);
            }
        }
    }
}

}  // namespace corr
