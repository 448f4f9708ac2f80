// corr_api.cu -- the C ABI of include/corr.h: plan construction (path choice, triangular tile
// schedule = step S3), TMA tensor-map construction, kernel launches.  Host code only; the
// kernels are in corr_dp4a.cuh (S4') and corr_tc.cuh (S1, S2, S4, S5).
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <vector>

#include "../../include/corr.h"
#include "corr_dp4a.cuh"
#include "corr_gate.cuh"
#include "corr_imma.cuh"
#include "corr_peak.cuh"
#include "corr_shift.cuh"
#include "corr_tc.cuh"
#include "corr_tc3.cuh"
#include "corr_tcd.cuh"
#include "corr_tc5.cuh"

namespace {

thread_local char g_err[512] = "";
thread_local int g_create_rc = 0;   // error code of the last failed corr_plan_create_ex in this thread

void set_err(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

#define CUDA_TRY(expr, code)                                                          \
    do {                                                                              \
        cudaError_t e_ = (expr);                                                      \
        if (e_ != cudaSuccess) {                                                      \
            set_err("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
            return code;                                                              \
        }                                                                             \
    } while (0)

using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                   CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                   CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

int count_tiles(int N, int tx, int ty)
{
    // tile (bx, by) covers x in [bx*tx, (bx+1)*tx), y in [by*ty, (by+1)*ty); it touches the upper
    // triangle iff its largest y is >= its smallest x.
    if (N < 1 || tx < 1 || ty < 1) return -1;
    const int nbx = (N + tx - 1) / tx, nby = (N + ty - 1) / ty;
    int n = 0;
    for (int bx = 0; bx < nbx; ++bx)
        for (int by = 0; by < nby; ++by)
            if (std::min(N, (by + 1) * ty) - 1 >= bx * tx) ++n;
    return n;
}

}  // namespace

// S3, the tail of the schedule (corr_tc3.cuh): the units left after the last whole wave are cut into pieces, one or
// two per CTA pair, so that every pair finishes at the same time.  The cost of a pair is counted in groups of
// T3_GROUP samples: its pieces, a fixed cost per piece (accumulator drain, epilogue, and the output being summed in
// memory) and the extra time its transposed tiles take in the epilogue (~3 and ~0.5 groups; the result is flat
// within 0.3 % for 2..5 and 0..3.5, profiles/r02_tc3_ncu_summary.md).  The first
// piece of a cut unit is marked EARLY: its pair computes it before its whole units, so that its store is long done
// when the other pieces add theirs.  Pieces are handed out in unit order, pair by pair, for the smallest budget
// (binary search) that places every group.
static void tc3_build_pieces(int num_units, int npairs, int slices, int groups_full, int groups_last,
                             const std::vector<ushort4> &tiles4, std::vector<int4> &pieces)
{
    const double E = 3.0, XT = 0.5;
    const int tiles_per_f = (int)tiles4.size();
    pieces.assign((size_t)npairs * corr::TC3_MAX_PIECES, make_int4(0, 0, 0, 0));
    const int waves = num_units / npairs, u0 = waves * npairs;
    if (u0 == num_units) return;
    auto len = [&](int u) { return (u % slices == slices - 1) ? groups_last : groups_full; };
    auto transposed = [&](int u) { return (tiles4[(size_t)((u / slices) % tiles_per_f)].w & corr::TC3_TILE_TRANSPOSED) != 0; };
    std::vector<double> pre((size_t)npairs, 0.0);
    double gt = 0.0;
    for (int pr = 0; pr < npairs; ++pr)
        for (int k = 0; k < waves; ++k)
            if (transposed(pr + k * npairs)) pre[(size_t)pr] += XT;
    for (int u = u0; u < num_units; ++u) gt += len(u);
    auto assign = [&](double B, bool commit) {
        int u = u0, off = 0;
        for (int pr = 0; pr < npairs && u < num_units; ++pr) {
            double budget = B - pre[(size_t)pr];
            for (int np = 0; np < corr::TC3_MAX_PIECES && u < num_units; ++np) {
                const int room = (int)(budget - E);
                if (room < 1) break;
                const int l = len(u), cnt = std::min(l - off, room);
                if (commit)
                    pieces[(size_t)pr * corr::TC3_MAX_PIECES + np] = make_int4(u, off, cnt, (off == 0 && cnt < l && waves > 0) ? 1 : 0);
                budget -= cnt + E + (transposed(u) ? XT * cnt / l : 0.0);
                off += cnt;
                if (off == l) { ++u; off = 0; }
            }
        }
        return u == num_units;
    };
    double lo = 0.0, hi = gt + 2.0 * (E + XT) * corr::TC3_MAX_PIECES + 64.0;
    for (int it = 0; it < 48; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (assign(mid, false)) hi = mid; else lo = mid;
    }
    assign(hi, true);
}

// S3, the tile table of the CTA-pair kernels (corr_tc3.cuh): pair tiles of two row blocks (128 inputs each) against
// one column block.  Column block j needs the row blocks 0..j.  An even count pairs up as (0,1), (2,3), ...; an odd
// count as (1,2), (3,4), ... and leaves block (0, j) over.  The left-over blocks all have row block 0: computed
// transposed (rows = block j, columns = block 0) they share their column operand, so they pair up with each other.
static void tc3_tile_table(int N, std::vector<ushort4> &tiles4)
{
    const int nb = (N + 127) / 128;
    auto us = [](int v) { return (unsigned short)v; };
    std::vector<int> left;
    tiles4.clear();
    for (int j = 0; j < nb; ++j) {
        const int first = ((j + 1) % 2 == 0) ? 0 : 1;
        for (int a = first; a + 1 <= j; a += 2) tiles4.push_back(make_ushort4(us(a), us(a + 1), us(j), 0));
        if (first == 1) left.push_back(j);
    }
    for (size_t i = 0; i < left.size(); i += 2)
        tiles4.push_back(make_ushort4(us(left[i]), (i + 1 < left.size()) ? us(left[i + 1]) : corr::TC3_NO_BLOCK, 0,
                                      corr::TC3_TILE_TRANSPOSED));
}

static bool alloc_pad_buf(struct corr_plan *p);

struct corr_plan {
    int N, F, T, path;
    int n_pad;         // N rounded up to a multiple of 16: the width of the stream the TMA-fed kernels read
    uint8_t *pad_buf;  // T*F*n_pad bytes when n_pad != N (corr_pad_kernel)
    int sm_count;
    // schedule
    int tile;          // tile edge (square tiles)
    int tiles_per_f;
    int slices;        // T-slices per tile
    int t_per_slice;
    int num_units;
    int grid;
    int kernels_per_exec;
    ushort2 *tiles_dev;
    ushort4 *tiles4_dev;   // variant 3: (xa, xb, by, flags), see Tc3Tile in corr_tc3.cuh
    // dp4a only
    int aligned;
    // tcgen05 only
    int pack_sub;      // variant 1: 128, or 64 when two 64-input channels are packed into one 128-tile (see below)
    int variant;       // 1: single-CTA tiles 128x128, both operands' planes in shared memory (corr_tc.cuh; on request);
                       // 2: one diagonal 128-block per channel on one CTA, A operand in TMEM (corr_tcd.cuh; chosen
                       // for N <= 128, where a pair tile would be half empty, and for two 64-input channels per tile);
                       // 3: CTA-pair tiles 256x128, A operand in TMEM (corr_tc3.cuh, default above N = 128);
                       // 5: as 3 with three products per complex MAC (corr_tc5.cuh; CORR_TC_VARIANT=5)
    int win_c, Fs;     // whole channels per window ((128 - 15) / N; > 1: the buffer MUST be aligned); channels as the schedule sees them
    int win_ok;        // variant 2, N % 16 != 0: the unpadded stream can be read through 16-byte aligned windows (corr_tcd.cuh):
                       // N + 15 <= 128 and (F * N) % 16 == 0; used when the caller's buffer is 16-byte aligned, else the padded copy
    int tmap_win;      // the cached tensor map is the window one
    int balanced;      // variant 2: all groups of all channels dealt to the CTAs in equal shares (corr_tcd.cuh), output added
    int groups_full, groups_last;   // variant 3: groups of T3_GROUP samples per full / last slice
    long long total_groups;
    int *flags_dev;    // variant 3: [num_units][2] stream-K flags (corr_tc3.cuh)
    int4 *pieces_dev;  // variant 3: [pairs][TC3_MAX_PIECES] tail pieces of every CTA pair (tc3_build_pieces)
    CUtensorMap tmap;
    CUtensorMap tmap_y;
    const void *tmap_ptr;
    // corr_execute_host staging
    uint8_t *packed_own;
    int32_t *vis_own;
    // corr_execute_host pipeline over groups of channels (copy in | compute | copy out)
    corr_plan *sub;        // plan for host_fg channels, executed once per group
    int host_fg;           // channels per group (divides F); 0 = not pipelined
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_start, ev_in[2], ev_free[2], ev_out[8], ev_comp, ev_done;
    unsigned long long grp_seq;   // channel groups submitted so far (staging buffers alternate across calls)
    unsigned long long calls_submitted;
    // corr_execute_gated: per-gate runs of the gathered stream, plans for their lengths
    uint8_t *gate_buf;     // device: rows regrouped by gate
    size_t gate_buf_bytes;
    int *order_dev;        // device, T row indices, then the (start, count) of every gate (at most GATE_MERGE_MAX_G)
    int *order_pin;        // pinned host copy the upload reads from
    cudaEvent_t ev_gate;   // the upload of order_pin has been consumed
    std::map<long long, corr_plan *> *gate_plans;   // length of a run -> plan (N, F, length); (G << 32 | length) -> plan (N, G*F, length)
};

extern "C" void corr_plan_destroy(corr_plan *p);

// N % 16 != 0 on a TMA-fed path: the padded copy of the stream lives in the plan from creation on, so that
// corr_execute only enqueues work (no allocation, no implicit synchronisation, capturable into a CUDA graph).
static bool alloc_pad_buf(corr_plan *p)
{
    if (p->path == CORR_PATH_DP4A || p->n_pad == p->N || p->win_c > 1) return true;   // (win_c > 1: never padded)
    if (cudaMalloc(&p->pad_buf, (size_t)p->T * p->F * p->n_pad) != cudaSuccess) {
        g_create_rc = CORR_ERR_ALLOC;
        set_err("corr_plan_create: device allocation of the padded stream (%zu bytes) failed: %s",
                (size_t)p->T * p->F * p->n_pad, cudaGetErrorString(cudaGetLastError()));
        corr_plan_destroy(p);
        return false;
    }
    return true;
}

extern "C" {

const char *corr_last_error(void) { return g_err; }

size_t corr_baseline_index(int N, int x, int y)
{
    if (N < 1 || x < 0 || y < x || y >= N) return (size_t)-1;
    return (size_t)x * N - (size_t)x * (x - 1) / 2 + (size_t)(y - x);
}

int corr_count_tiles(int N, int tile_x, int tile_y) { return count_tiles(N, tile_x, tile_y); }

int corr_schedule_pairs(int N, int F, int T, int pairs, int info[8], int *pieces_out)
{
    if (N < 1 || F < 1 || T < 1 || T > 16777215 || pairs < 1 || !info) {
        set_err("corr_schedule_pairs: need N, F, pairs >= 1, 1 <= T <= 16777215 and an info array");
        return CORR_ERR_INVALID_ARG;
    }
    std::vector<ushort4> tiles4;
    tc3_tile_table(N, tiles4);
    const long long units0 = (long long)F * (long long)tiles4.size();
    if (units0 > 0x7fffffffLL / 64) {
        set_err("corr_schedule_pairs: too many work units");
        return CORR_ERR_INVALID_ARG;
    }
    const int Q = corr::T3_GROUP, s = (T + corr::TC_MAX_SLICE - 1) / corr::TC_MAX_SLICE;
    const int tps = ((T + s - 1) / s + Q - 1) / Q * Q, slices = (T + tps - 1) / tps;
    const int num_units = (int)(units0 * slices);
    const int groups_full = tps / Q, groups_last = (T - (slices - 1) * tps + Q - 1) / Q;
    const long long total_groups = units0 * ((long long)(slices - 1) * groups_full + groups_last);
    const int used = (int)std::min<long long>(total_groups, pairs);
    info[0] = (int)tiles4.size(); info[1] = slices; info[2] = num_units; info[3] = groups_full; info[4] = groups_last;
    info[5] = used; info[6] = num_units / used; info[7] = 0;
    for (const ushort4 &t : tiles4) info[7] += (t.w & corr::TC3_TILE_TRANSPOSED) ? 1 : 0;
    if (pieces_out) {
        std::vector<int4> pieces;
        tc3_build_pieces(num_units, used, slices, groups_full, groups_last, tiles4, pieces);
        for (size_t i = 0; i < pieces.size(); ++i) {
            pieces_out[4 * i + 0] = pieces[i].x; pieces_out[4 * i + 1] = pieces[i].y;
            pieces_out[4 * i + 2] = pieces[i].z; pieces_out[4 * i + 3] = pieces[i].w;
        }
    }
    return CORR_OK;
}

size_t corr_input_bytes(const corr_plan *p) { return p ? (size_t)p->T * p->F * p->N : 0; }

size_t corr_vis_elems(const corr_plan *p) { return p ? (size_t)p->F * ((size_t)p->N * (p->N + 1) / 2) * 2 : 0; }

int corr_plan_info(const corr_plan *p, int info[8])
{
    if (!p || !info) {
        set_err("corr_plan_info: NULL argument");
        return CORR_ERR_INVALID_ARG;
    }
    info[0] = p->path;
    info[1] = (p->variant >= 3) ? 256 : p->tile;
    info[2] = p->tile;
    info[3] = p->tiles_per_f;
    info[4] = p->slices;
    info[5] = p->num_units;
    info[6] = p->grid;
    info[7] = p->kernels_per_exec;
    return CORR_OK;
}

void corr_plan_destroy(corr_plan *p)
{
    if (!p) return;
    if (p->pad_buf) cudaFree(p->pad_buf);
    if (p->tiles_dev) cudaFree(p->tiles_dev);
    if (p->tiles4_dev) cudaFree(p->tiles4_dev);
    if (p->flags_dev) cudaFree(p->flags_dev);
    if (p->pieces_dev) cudaFree(p->pieces_dev);
    if (p->host_fg != 0) cudaEventDestroy(p->ev_done);
    if (p->gate_plans) {
        for (auto &kv : *p->gate_plans) corr_plan_destroy(kv.second);
        delete p->gate_plans;
    }
    if (p->gate_buf) cudaFree(p->gate_buf);
    if (p->order_dev) cudaFree(p->order_dev);
    if (p->order_pin) {
        cudaFreeHost(p->order_pin);
        cudaEventDestroy(p->ev_gate);
    }
    if (p->sub) {
        corr_plan_destroy(p->sub);
        cudaStreamDestroy(p->s_in);
        cudaStreamDestroy(p->s_out);
        cudaEventDestroy(p->ev_start);
        cudaEventDestroy(p->ev_comp);
        for (int i = 0; i < 8; ++i) cudaEventDestroy(p->ev_out[i]);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(p->ev_in[i]);
            cudaEventDestroy(p->ev_free[i]);
        }
    }
    if (p->packed_own) cudaFree(p->packed_own);
    if (p->vis_own) cudaFree(p->vis_own);
    delete p;
}

corr_plan *corr_plan_create_ex(int N, int F, int T, int path)
{
    if (N < 1 || F < 1 || T < 1 || T > 16777215) {
        g_create_rc = CORR_ERR_INVALID_ARG; set_err("corr_plan_create: need N >= 1, F >= 1, 1 <= T <= 16777215 (got N=%d F=%d T=%d)", N, F, T);
        return nullptr;
    }
    if (N > 65535 * 16) {
        g_create_rc = CORR_ERR_INVALID_ARG; set_err("corr_plan_create: N=%d too large for the tile table", N);
        return nullptr;
    }
    if (path != CORR_PATH_AUTO && path != CORR_PATH_DP4A && path != CORR_PATH_TCGEN05 && path != CORR_PATH_IMMA) {
        g_create_rc = CORR_ERR_INVALID_ARG; set_err("corr_plan_create: unknown path %d", path);
        return nullptr;
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        g_create_rc = CORR_ERR_CUDA; set_err("corr_plan_create: no usable CUDA device (%s); this library has no CPU fallback",
                cudaGetErrorString(cudaGetLastError()));
        return nullptr;
    }
    if (prop.major != 10) {
        g_create_rc = CORR_ERR_UNSUPPORTED; set_err("corr_plan_create: device '%s' is sm_%d%d; this library is built for sm_100a only", prop.name,
                prop.major, prop.minor);
        return nullptr;
    }
    const int n_pad = (N + 15) / 16 * 16;   // N % 16 != 0: the TMA-fed paths read a zero-padded copy of the stream
    if (path == CORR_PATH_AUTO) {
        const char *force = getenv("CORR_FORCE_PATH");
        if (force && !strcmp(force, "dp4a"))
            path = CORR_PATH_DP4A;
        else if (force && !strcmp(force, "tcgen05"))
            path = CORR_PATH_TCGEN05;
        else if (force && !strcmp(force, "imma"))
            path = CORR_PATH_IMMA;
        else
            // N = 64 with an even number of channels: the stream [T][F][64] IS the stream [T][F/2][128], so a 128-tile
            // holds two whole channels and its two diagonal 64-blocks are their matrices (half of the tensor work is
            // cross-channel and dropped; still 1.45x the warp-MMA kernel, which is MMA-issue-bound at N = 64,
            // profiles/r02_sweep.md)
            // (an odd number of channels: the last tile holds one channel and 64 bytes beyond the row, which TMA fills with
            // zeros; measured against the warp-MMA kernel at T = 65536: F = 3 a tie, F = 5: 19.9 / 26.3 us, F = 63: 82 / 141)
            path = (N == 64 && (F % 2 == 0 || F >= 5)) ? CORR_PATH_TCGEN05 : (n_pad <= 64) ? CORR_PATH_IMMA : CORR_PATH_TCGEN05;
            // N % 16 != 0 below 64 with rows of a multiple of 16 bytes: several whole channels per 16-byte aligned window of
            // corr_tcd_kernel instead of a padded copy + the warp-MMA kernel (N = 37, F = 128, T = 32768: 68 against 224 us)
            if (path == CORR_PATH_IMMA && n_pad != N && ((long long)F * N) % 16 == 0 && !getenv("CORR_TCD_NO_WINDOW")) path = CORR_PATH_TCGEN05;
    }
    const char *v_forced = getenv("CORR_TC_VARIANT");
    const bool v1_forced = v_forced && !strcmp(v_forced, "1");   // corr_tc_kernel reads the packed view through a 3-D map: even F only
    const bool packed64 = (path == CORR_PATH_TCGEN05 && N == 64 && (F % 2 == 0 || (F >= 3 && !v1_forced && !(v_forced && v_forced[0]))));
    if (path == CORR_PATH_IMMA && n_pad > 64) {
        g_create_rc = CORR_ERR_UNSUPPORTED; set_err("corr_plan_create: the warp-MMA path takes N <= 64, got N=%d", N);
        return nullptr;
    }

    corr_plan *p = new (std::nothrow) corr_plan();
    if (!p) {
        g_create_rc = CORR_ERR_ALLOC; set_err("corr_plan_create: out of host memory");
        return nullptr;
    }
    memset(p, 0, sizeof(*p));
    p->N = N;
    p->n_pad = n_pad;
    p->F = F;
    p->T = T;
    p->path = path;
    p->sm_count = prop.multiProcessorCount;

    if (path == CORR_PATH_IMMA) {
        // whole channels per CTA: strips of 128/N channels x chunks of time samples (corr_imma.cuh)
        if (!get_encode_fn()) {
            g_create_rc = CORR_ERR_CUDA; set_err("corr_plan_create: cuTensorMapEncodeTiled not available from the driver");
            delete p;
            return nullptr;
        }
        const int fb = 128 / n_pad;
        const int strips = (F + fb - 1) / fb;
        cudaError_t e = cudaFuncSetAttribute(corr::corr_imma_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::IM_SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::corr_imma_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::IM_SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::corr_imma_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::IM_SMEM_BYTES);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(corr::corr_imma_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::IM_SMEM_BYTES);
        int occ = 1;
        if (e == cudaSuccess) {
            if (n_pad == 16) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, corr::corr_imma_kernel<1>, corr::ImmaCfg<1>::THREADS, corr::IM_SMEM_BYTES);
            else if (n_pad == 32) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, corr::corr_imma_kernel<2>, corr::ImmaCfg<2>::THREADS, corr::IM_SMEM_BYTES);
            else if (n_pad == 48) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, corr::corr_imma_kernel<3>, corr::ImmaCfg<3>::THREADS, corr::IM_SMEM_BYTES);
            else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, corr::corr_imma_kernel<4>, corr::ImmaCfg<4>::THREADS, corr::IM_SMEM_BYTES);
        }
        if (e != cudaSuccess || occ < 1) {
            g_create_rc = CORR_ERR_CUDA; set_err("corr_plan_create: cannot reserve %d B of shared memory: %s", corr::IM_SMEM_BYTES, cudaGetErrorString(e));
            delete p;
            return nullptr;
        }
        // time chunks (>= 512 samples each): the count that fills whole waves of CTA slots best
        // int32 headroom: a chunk accumulates 256 * sum (x16 planes) in registers and in the shared-memory
        // reduction, |256 * 128 * chunk| < 2^31 needs chunk <= 65535; IM_MAX_CHUNK = 32768 leaves a factor 2
        const int slots = p->sm_count * occ;
        const int min_chunks = (T + corr::IM_MAX_CHUNK - 1) / corr::IM_MAX_CHUNK;
        int chunks = min_chunks;
        double best = 0.0;
        for (int c = min_chunks; c <= std::max(min_chunks, std::min(T / 512, 4 * slots / strips + 1)); ++c) {
            const long long units = (long long)strips * c;
            const double eff = (double)units / (double)(((units + slots - 1) / slots) * slots);
            if (eff > best + 0.10) { best = eff; chunks = c; }   // more chunks only for a clearly better fill
        }
        if (const char *cc = getenv("CORR_IMMA_CHUNKS"))   // testing aid
            chunks = std::max(min_chunks, std::min(atoi(cc), std::max(1, T / 128)));
        p->t_per_slice = ((T + chunks - 1) / chunks + corr::IM_ROWS - 1) / corr::IM_ROWS * corr::IM_ROWS;
        p->slices = (T + p->t_per_slice - 1) / p->t_per_slice;
        p->tile = N;
        p->tiles_per_f = 1;
        p->num_units = strips * p->slices;
        p->grid = p->num_units;
        p->kernels_per_exec = (n_pad != N) ? 2 : 1;
        if (!alloc_pad_buf(p)) return nullptr;
        return p;
    }

    // ---- S3: the triangular tile table (only tiles on or above the diagonal)
    if (path == CORR_PATH_DP4A)
        p->tile = (N <= 16) ? 16 : (N <= 32) ? 32 : 64;
    else
        p->tile = corr::TC_BLK;
    p->variant = 0;
    if (path == CORR_PATH_TCGEN05) {
        // N <= 128 is one 128-block per channel: a CTA-pair tile would have an idle half (measured 923 against 1358
        // effective TOPS at N = 128, profiles/r02_sweep.md), so single-CTA tiles take over there
        const char *v = getenv("CORR_TC_VARIANT");   // testing aid: force a kernel
        p->variant = (v && !strcmp(v, "1")) ? 1 : (v && !strcmp(v, "3")) ? 3 : (v && !strcmp(v, "5")) ? 5 : (n_pad <= 128) ? 1 : 3;
        if (packed64) p->variant = 1;
        // one 128-block per channel: the diagonal-block kernel (A operand in TMEM, corr_tcd.cuh) unless variant 1 is forced
        // Two or three blocks per channel (128 < N <= 256): the same kernel with off-diagonal blocks (two packed blocks per
        // stage, the image used by the two halves of a block in turn) beats the pair kernel, which computes one of its two
        // pair tiles next to an empty block there, when the segments are long: measured N = 256: 2384 against 1978 TOPS
        // at F = 32, T = 32768 and 41.5 against 44.7 us on cfg 2, but 53.7 against 49.9 us at F = 128, T = 2048 (segments of
        // 8 groups) and above N = 256 the pair kernel wins (N = 272: 1225 against 1455).  CORR_TCD_MAX_N (testing aid)
        // moves the upper limit.
        const char *mx = getenv("CORR_TCD_MAX_N");
        const int tcd_max = mx ? atoi(mx) : 256;
        {
            const long long nbk = (n_pad + 127) / 128, gpc = (T + corr::TD_GROUP - 1) / corr::TD_GROUP;
            const long long G = (long long)F * (nbk * (nbk + 1) / 2) * gpc;
            const double seg = std::min<double>((double)gpc, (double)G / (double)std::min<long long>(G, p->sm_count));
            if (!(v && v[0]) && !packed64 && n_pad > 128 && n_pad <= tcd_max && (seg >= 16.0 || mx)) p->variant = 1;
        }
        if (p->variant == 1 && (packed64 || n_pad <= std::max(128, tcd_max)) && !(v && !strcmp(v, "1"))) p->variant = 2;
    }
    p->pack_sub = packed64 ? 64 : 128;
    // N % 16 != 0 read through 16-byte aligned windows (corr_tcd.cuh): N <= 113, rows of a multiple of 16 bytes; a window holds
    // (128 - 15) / N whole channels
    int win_c = 0;
    if (p->variant == 2 && !packed64 && n_pad != N && N + 15 <= 128 && ((long long)F * N) % 16 == 0 && !getenv("CORR_TCD_NO_WINDOW"))
        win_c = (128 - 15) / N;
    p->win_c = win_c;
    p->win_ok = win_c > 0 ? 1 : 0;
    const int Ns = packed64 ? 128 : N, Fs = packed64 ? (F + 1) / 2 : (win_c > 1) ? (F + win_c - 1) / win_c : F;   // the shape the tile schedule sees
    p->Fs = Fs;
    const int nb = (Ns + p->tile - 1) / p->tile;
    std::vector<ushort2> tiles;
    std::vector<ushort4> tiles4;
    if (p->variant >= 3) {
        tc3_tile_table(Ns, tiles4);
        tiles.resize(tiles4.size());   // the count is what the schedule below needs
    } else {
        for (int bx = 0; bx < nb; ++bx)
            for (int by = bx; by < nb; ++by) tiles.push_back(make_ushort2((unsigned short)bx, (unsigned short)by));
    }
    p->tiles_per_f = (int)tiles.size();
    const long long units0 = (long long)Fs * p->tiles_per_f;
    if (units0 > 0x7fffffffLL / 64) {
        g_create_rc = CORR_ERR_INVALID_ARG; set_err("corr_plan_create: too many work units");
        delete p;
        return nullptr;
    }

    // ---- split-T: choose the number of T-slices per tile from a wave-count cost model
    const int quantum = (path == CORR_PATH_DP4A) ? corr::DP4A_TK
                        : (p->variant >= 3) ? corr::T3_GROUP  // tc3 / tc5 run whole groups of stages
                        : (p->variant == 2) ? corr::TD_GROUP
                                            : corr::TC_ST;
    const int max_slice = (path == CORR_PATH_DP4A) ? (1 << 22) : (p->variant == 5) ? corr::T5_MAX_SLICE : corr::TC_MAX_SLICE;
    const int ctas_per_wave = (path == CORR_PATH_DP4A) ? 4 * p->sm_count : (p->variant >= 3 ? p->sm_count / 2 : p->sm_count);
    const double per_sample = (path == CORR_PATH_DP4A) ? 40.0 : 8.0;  // cycles per time sample per unit
    const double epi = (path == CORR_PATH_DP4A) ? 1500.0 : 6000.0;    // cycles per unit, fixed
    const int min_slices = (T + max_slice - 1) / max_slice;
    double best_cost = 0;
    int best_s = 0;
    // variant 3 balances the load itself (stream-K over groups of stages): T is split only for int32 headroom
    const int s_max = (p->variant >= 3) ? min_slices : std::max(min_slices, 64);
    for (int s = min_slices; s <= s_max; ++s) {
        int tps = ((T + s - 1) / s + quantum - 1) / quantum * quantum;
        if (s > min_slices && tps < 8 * quantum) break;
        const int s_eff = (T + tps - 1) / tps;
        const double waves = (double)((units0 * s_eff + ctas_per_wave - 1) / ctas_per_wave);
        const double cost = waves * (per_sample * tps + epi * (s_eff > 1 ? 2.0 : 1.0));
        if (best_s == 0 || cost < best_cost * 0.97) {
            best_cost = cost;
            best_s = s;
        }
    }
    p->t_per_slice = ((T + best_s - 1) / best_s + quantum - 1) / quantum * quantum;
    p->slices = (T + p->t_per_slice - 1) / p->t_per_slice;
    p->num_units = (int)(units0 * p->slices);
    p->grid = (path == CORR_PATH_DP4A) ? p->num_units
              : (p->variant >= 3) ? 2 * std::min(p->num_units, p->sm_count / 2)
                                  : std::min(p->num_units, p->sm_count);
    if (p->variant == 2) {
        // few, long channels leave SMs idle (64 channels in two slices: 128 units for 148 SMs): deal the groups of 256
        // samples of all channels to the CTAs in equal shares instead, every share added into a cleared output
        const long long gpc = (T + corr::TD_GROUP - 1) / corr::TD_GROUP, G = units0 * gpc;
        const long long waves = (p->num_units + p->sm_count - 1) / p->sm_count;
        const double extra = 512.0;   // samples' worth of time per segment: accumulator drain, epilogue, pipeline restart
        const double simple_cost = (double)waves * (p->t_per_slice + extra);
        const double shares_cost = (double)((G + p->sm_count - 1) / p->sm_count) * corr::TD_GROUP + 3.0 * extra;
        const char *e = getenv("CORR_TCD_SHARES");   // testing aid: 0 / 1 forces the choice
        // (equal shares put the CTAs at 148 different times of the stream, where units of a wave sweep it together: the
        // tensor map of this schedule asks for 64-byte L2 promotion instead of 256, see build_tmap)
        const double need = 0.97;
        p->balanced = (G >= p->sm_count && shares_cost < need * simple_cost) ? 1 : 0;
        if (e && G >= 1) p->balanced = (e[0] != '0') ? 1 : 0;
        if (p->balanced) p->grid = (int)std::min<long long>(G, p->sm_count);
    }
    p->kernels_per_exec = 1 + ((path != CORR_PATH_DP4A && n_pad != N && !p->win_ok) ? 1 : 0);  // + corr_pad_kernel (with win_ok: only for a misaligned buffer)
    p->aligned = (N % 4 == 0) ? 1 : 0;
    if (p->variant >= 3) {
        p->groups_full = p->t_per_slice / corr::T3_GROUP;
        p->groups_last = (T - (p->slices - 1) * p->t_per_slice + corr::T3_GROUP - 1) / corr::T3_GROUP;
        p->total_groups = units0 * ((long long)(p->slices - 1) * p->groups_full + p->groups_last);
        p->grid = 2 * (int)std::min<long long>(p->total_groups, p->sm_count / 2);
        std::vector<int4> pieces;
        tc3_build_pieces(p->num_units, p->grid / 2, p->slices, p->groups_full, p->groups_last, tiles4, pieces);
        if (cudaMalloc(&p->flags_dev, (2 * (size_t)p->num_units + 1) * sizeof(int)) != cudaSuccess ||
            cudaMemset(p->flags_dev, 0, (2 * (size_t)p->num_units + 1) * sizeof(int)) != cudaSuccess ||
            cudaMalloc(&p->pieces_dev, pieces.size() * sizeof(int4)) != cudaSuccess ||
            cudaMemcpy(p->pieces_dev, pieces.data(), pieces.size() * sizeof(int4), cudaMemcpyHostToDevice) != cudaSuccess) {
            g_create_rc = CORR_ERR_ALLOC; set_err("corr_plan_create: device allocation of the schedule flags failed: %s",
                    cudaGetErrorString(cudaGetLastError()));
            corr_plan_destroy(p);
            return nullptr;
        }
    }

    if (cudaMalloc(&p->tiles_dev, tiles.size() * sizeof(ushort2)) != cudaSuccess ||
        cudaMemcpy(p->tiles_dev, tiles.data(), tiles.size() * sizeof(ushort2), cudaMemcpyHostToDevice) != cudaSuccess ||
        (!tiles4.empty() &&
         (cudaMalloc(&p->tiles4_dev, tiles4.size() * sizeof(ushort4)) != cudaSuccess ||
          cudaMemcpy(p->tiles4_dev, tiles4.data(), tiles4.size() * sizeof(ushort4), cudaMemcpyHostToDevice) != cudaSuccess))) {
        g_create_rc = CORR_ERR_ALLOC; set_err("corr_plan_create: device allocation of the tile table failed: %s",
                cudaGetErrorString(cudaGetLastError()));
        corr_plan_destroy(p);
        return nullptr;
    }
    if (path == CORR_PATH_TCGEN05) {
        if (!get_encode_fn()) {
            g_create_rc = CORR_ERR_CUDA; set_err("corr_plan_create: cuTensorMapEncodeTiled not available from the driver");
            corr_plan_destroy(p);
            return nullptr;
        }
        cudaError_t e1 = cudaFuncSetAttribute(corr::corr_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              corr::TC_SMEM_BYTES);
        cudaError_t e3 = cudaFuncSetAttribute(corr::corr_tc3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              corr::T3_SMEM_BYTES);
        cudaError_t e5 = cudaFuncSetAttribute(corr::corr_tc5_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                              corr::T5_SMEM_BYTES);
        if (e5 == cudaSuccess)
            e5 = cudaFuncSetAttribute(corr::corr_tcd_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::TD_SMEM_BYTES);
        if (e5 == cudaSuccess)
            e5 = cudaFuncSetAttribute(corr::corr_tcd_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::TD_SMEM_BYTES_G);
        if (e1 != cudaSuccess || e3 != cudaSuccess || e5 != cudaSuccess) {
            g_create_rc = CORR_ERR_CUDA; set_err("corr_plan_create: cannot reserve %d / %d / %d B of shared memory: %s", corr::TC_SMEM_BYTES,
                    corr::T3_SMEM_BYTES, corr::T5_SMEM_BYTES, cudaGetErrorString(cudaGetLastError()));
            corr_plan_destroy(p);
            return nullptr;
        }
    }
    if (!alloc_pad_buf(p)) return nullptr;
    return p;
}

corr_plan *corr_plan_create(int N, int F, int T) { return corr_plan_create_ex(N, F, T, CORR_PATH_AUTO); }

int corr_measure_int8_tops(int iters, double *tops_out)
{
    if (iters < 1 || !tops_out) {
        set_err("corr_measure_int8_tops: need iters >= 1 and a result pointer");
        return CORR_ERR_INVALID_ARG;
    }
    int dev = 0;
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDevice(&dev), CORR_ERR_CUDA);
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev), CORR_ERR_CUDA);
    if (prop.major != 10) {
        set_err("corr_measure_int8_tops: needs an sm_100 device");
        return CORR_ERR_UNSUPPORTED;
    }
    CUDA_TRY(cudaFuncSetAttribute(corr::corr_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::PK_SMEM_BYTES),
             CORR_ERR_CUDA);
    const int grid = prop.multiProcessorCount / 2 * 2;
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0), CORR_ERR_CUDA);
    CUDA_TRY(cudaEventCreate(&e1), CORR_ERR_CUDA);
    corr::corr_peak_kernel<<<grid, corr::PK_THREADS, corr::PK_SMEM_BYTES>>>(iters / 8 + 1);   // warm-up
    CUDA_TRY(cudaEventRecord(e0), CORR_ERR_CUDA);
    corr::corr_peak_kernel<<<grid, corr::PK_THREADS, corr::PK_SMEM_BYTES>>>(iters);
    CUDA_TRY(cudaEventRecord(e1), CORR_ERR_CUDA);
    CUDA_TRY(cudaEventSynchronize(e1), CORR_ERR_CUDA);
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1), CORR_ERR_CUDA);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    // per CTA pair and iteration: 4 MMAs of 256 x 128 x 32 multiply-adds
    *tops_out = (double)(grid / 2) * iters * 4.0 * 2.0 * 256.0 * 128.0 * 32.0 / (ms * 1e-3) / 1e12;
    return CORR_OK;
}

int corr_time_shift(int N, int F, int T, const uint8_t *packed_in_dev, const int32_t *lags_dev, uint8_t *packed_out_dev,
                    corr_stream_t stream_)
{
    if (N < 1 || F < 1 || T < 1 || F > 65535 || (T + corr::SH_TB - 1) / corr::SH_TB > 65535) {
        set_err("corr_time_shift: need N >= 1, 1 <= F <= 65535, 1 <= T <= %d (got N=%d F=%d T=%d)", 65535 * corr::SH_TB, N, F, T);
        return CORR_ERR_INVALID_ARG;
    }
    if (!packed_in_dev || !lags_dev || !packed_out_dev || packed_in_dev == packed_out_dev) {
        set_err("corr_time_shift: NULL buffer, or input and output are the same buffer (the shift is not in place)");
        return CORR_ERR_INVALID_ARG;
    }
    if ((N % 16 == 0) && ((reinterpret_cast<uintptr_t>(packed_in_dev) | reinterpret_cast<uintptr_t>(packed_out_dev)) & 15u)) {
        set_err("corr_time_shift: buffers must be 16-byte aligned");
        return CORR_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    // N % 16 != 0 but rows of a multiple of 16 bytes: one channel of F * N columns whose lags repeat with period N
    const bool flat = N % 16 != 0 && ((long long)F * N) % 16 == 0 && (long long)F * N <= 128 * corr::SH_MAX_GROUPS &&
                      !((reinterpret_cast<uintptr_t>(packed_in_dev) | reinterpret_cast<uintptr_t>(packed_out_dev)) & 15u);
    const int Nk = flat ? F * N : N, Fk = flat ? 1 : F;
    if (Nk % 16 != 0 || (Nk + 127) / 128 > corr::SH_MAX_GROUPS) {
        dim3 grid((unsigned)((N + 127) / 128), (unsigned)F, (unsigned)((T + corr::SH_TB - 1) / corr::SH_TB));
        corr::corr_shift_bytes_kernel<<<grid, 256, 0, stream>>>(packed_in_dev, packed_out_dev, lags_dev, N, F, T);
        CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
        return CORR_OK;
    }
    if (!get_encode_fn()) {
        set_err("corr_time_shift: cuTensorMapEncodeTiled not available from the driver");
        return CORR_ERR_CUDA;
    }
    // the input as a 3-D byte tensor, innermost first: (N, F, T); a box is 16 rows of 128 inputs of one channel
    CUtensorMap tmap;
    const cuuint64_t dims[3] = {(cuuint64_t)Nk, (cuuint64_t)Fk, (cuuint64_t)T};
    const cuuint64_t strides[2] = {(cuuint64_t)Nk, (cuuint64_t)Fk * (cuuint64_t)Nk};
    const cuuint32_t box[3] = {128u, 1u, (cuuint32_t)corr::SH_BOX_ROWS};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    CUresult r = get_encode_fn()(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<uint8_t *>(packed_in_dev), dims, strides,
                                 box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_err("corr_time_shift: cuTensorMapEncodeTiled failed with CUresult %d (N=%d F=%d T=%d)", (int)r, N, F, T);
        return CORR_ERR_CUDA;
    }
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev), CORR_ERR_CUDA);
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), CORR_ERR_CUDA);
    // the attribute belongs to the current device's context: set it on every call (a host-side table write)
    CUDA_TRY(cudaFuncSetAttribute(corr::corr_shift_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::SH_SMEM_BYTES),
             CORR_ERR_CUDA);
    const long long tiles = (long long)((Nk + 127) / 128) * Fk * ((T + corr::SH_TB - 1) / corr::SH_TB);
    const unsigned grid = (unsigned)std::min<long long>(tiles, sms);
    corr::corr_shift_kernel<<<grid, corr::SH_THREADS, corr::SH_SMEM_BYTES, stream>>>(tmap, packed_in_dev, packed_out_dev, lags_dev,
                                                                                   Nk, Fk, T, N);
    CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
    return CORR_OK;
}

static int build_tmap(corr_plan *p, const uint8_t *packed_dev, int window = 0)
{
    if (p->tmap_ptr == packed_dev && p->tmap_win == window) return CORR_OK;
    p->tmap_win = window;
    if (p->path == CORR_PATH_IMMA) {
        // packed[T][F][N] as a byte matrix, innermost first: (F*N, T), row stride F*N bytes
        const cuuint64_t dims2[2] = {(cuuint64_t)p->F * (cuuint64_t)p->n_pad, (cuuint64_t)p->T};
        const cuuint64_t strides2[1] = {(cuuint64_t)p->F * (cuuint64_t)p->n_pad};
        const cuuint32_t box2[2] = {128u, (cuuint32_t)corr::IM_ROWS};
        const cuuint32_t estr2[2] = {1u, 1u};
        CUresult r2 = get_encode_fn()(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(packed_dev), dims2,
                                      strides2, box2, estr2, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r2 != CUDA_SUCCESS) {
            set_err("cuTensorMapEncodeTiled (2-D) failed with CUresult %d (N=%d F=%d T=%d)", (int)r2, p->N, p->F, p->T);
            return CORR_ERR_CUDA;
        }
        p->tmap_ptr = packed_dev;
        return CORR_OK;
    }
    if (window) {
        // the unpadded stream as a byte matrix (F * N, T): channel f is read through the box at column f * N rounded down to 16
        const cuuint64_t dims2[2] = {(cuuint64_t)p->F * (cuuint64_t)p->N, (cuuint64_t)p->T};
        const cuuint64_t strides2[1] = {(cuuint64_t)p->F * (cuuint64_t)p->N};
        const cuuint32_t box2[2] = {128u, (cuuint32_t)corr::TD_ST};
        const cuuint32_t estr2[2] = {1u, 1u};
        CUresult r2 = get_encode_fn()(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(packed_dev), dims2, strides2,
                                      box2, estr2, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                      p->balanced ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r2 != CUDA_SUCCESS) {
            set_err("cuTensorMapEncodeTiled (2-D, windows) failed with CUresult %d (N=%d F=%d T=%d)", (int)r2, p->N, p->F, p->T);
            return CORR_ERR_CUDA;
        }
        p->tmap_ptr = packed_dev;
        return CORR_OK;
    }
    if (p->pack_sub == 64 && p->variant == 2) {
        // two channels of 64 inputs per tile (corr_tcd_kernel): the stream as a byte matrix (F * 64, T); tile g is the box
        // at column 128 g, and with an odd F the last tile's second half lies beyond the row and is filled with zeros
        const cuuint64_t dims2[2] = {(cuuint64_t)p->F * 64u, (cuuint64_t)p->T};
        const cuuint64_t strides2[1] = {(cuuint64_t)p->F * 64u};
        const cuuint32_t box2[2] = {128u, (cuuint32_t)corr::TD_ST};
        const cuuint32_t estr2[2] = {1u, 1u};
        CUresult r2 = get_encode_fn()(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(packed_dev), dims2, strides2,
                                      box2, estr2, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                      p->balanced ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r2 != CUDA_SUCCESS) {
            set_err("cuTensorMapEncodeTiled (2-D, two channels per tile) failed with CUresult %d (N=%d F=%d T=%d)", (int)r2, p->N, p->F, p->T);
            return CORR_ERR_CUDA;
        }
        p->tmap_ptr = packed_dev;
        return CORR_OK;
    }
    // packed[T][F][N] bytes as a 3-D tensor, innermost first: (N, F, T), strides (1, N, F*N) bytes.
    // (two 64-input channels packed into one 128-tile: the same bytes seen as (128, F/2, T))
    const cuuint64_t nw = (p->pack_sub == 64) ? 128 : (cuuint64_t)p->n_pad, fw = (p->pack_sub == 64) ? (cuuint64_t)p->F / 2 : (cuuint64_t)p->F;
    const cuuint64_t dims[3] = {nw, fw, (cuuint64_t)p->T};
    const cuuint64_t strides[2] = {nw, fw * nw};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const int st = (p->variant >= 3) ? corr::T3_ST : corr::TC_ST;
    const cuuint32_t box[3] = {128u, 1u, (cuuint32_t)st};
    // L2 promotion: 256-byte lines pay when the neighbouring 128 bytes (the next channel's block at the same sample) are
    // wanted soon, which is so when the CTAs sweep the stream together; the equal-shares schedule of corr_tcd_kernel
    // puts them at 148 different times (ncu: 402 MB read from DRAM for a 268 MB stream with 256-byte promotion; measured
    // with 256 / 128 / 64 bytes / none: 86.2 / 83.1 / 83.0 / 83.2 us at N = 128, F = 64 and 101.0 / 90.6 / 86.5 / 90.6 at N = 112)
    CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
    if (p->variant == 2 && p->balanced) promo = CU_TENSOR_MAP_L2_PROMOTION_L2_64B;
    CUresult r = get_encode_fn()(&p->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<uint8_t *>(packed_dev), dims,
                                 strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                 promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS && p->variant >= 3) {
        const cuuint32_t boxy[3] = {64u, 1u, (cuuint32_t)st};  // half a y-block per CTA of the pair
        r = get_encode_fn()(&p->tmap_y, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<uint8_t *>(packed_dev), dims,
                            strides, boxy, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (r != CUDA_SUCCESS) {
        set_err("cuTensorMapEncodeTiled failed with CUresult %d (N=%d F=%d T=%d)", (int)r, p->N, p->F, p->T);
        return CORR_ERR_CUDA;
    }
    p->tmap_ptr = packed_dev;
    return CORR_OK;
}

int corr_execute(corr_plan *p, const uint8_t *packed_dev, int32_t *vis_dev, int accumulate_flag,
                 corr_stream_t stream_)
{
    if (!p || !packed_dev || !vis_dev) {
        set_err("corr_execute: NULL plan or buffer");
        return CORR_ERR_INVALID_ARG;
    }
    const bool padded = (p->path != CORR_PATH_DP4A && p->n_pad != p->N);
    if ((!padded && (reinterpret_cast<uintptr_t>(packed_dev) & 15u)) || (reinterpret_cast<uintptr_t>(vis_dev) & 7u)) {
        set_err("corr_execute: packed_dev must be 16-byte aligned and vis_dev 8-byte aligned");
        return CORR_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    // N % 16 != 0, N <= 113, rows of a multiple of 16 bytes, an aligned buffer: corr_tcd_kernel reads the stream as it is
    const int window = (padded && p->variant == 2 && p->win_ok && !(reinterpret_cast<uintptr_t>(packed_dev) & 15u)) ? 1 : 0;
    if (padded && p->variant == 2 && p->win_c > 1 && !window) {
        set_err("corr_execute: packed_dev must be 16-byte aligned for this shape (N=%d: %d channels per 128-byte window)", p->N, p->win_c);
        return CORR_ERR_INVALID_ARG;
    }
    if (padded && !window) {
        // N % 16 != 0: the TMA-fed kernels read a copy of the stream padded to n_pad inputs with stored zeros
        const long long rows = (long long)p->T * p->F;
        corr::corr_pad_kernel<<<8 * p->sm_count, 256, 0, stream>>>(packed_dev, p->pad_buf, p->N, p->n_pad, rows);
        CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
        packed_dev = p->pad_buf;
    }
    int out_mode;
    if (p->slices > 1 || p->balanced) {
        out_mode = corr::OUT_ATOMIC;
        if (!accumulate_flag)
            CUDA_TRY(cudaMemsetAsync(vis_dev, 0, corr_vis_elems(p) * sizeof(int32_t), stream), CORR_ERR_CUDA);
    } else {
        out_mode = accumulate_flag ? corr::OUT_RMW : corr::OUT_STORE;
    }

    if (p->path == CORR_PATH_IMMA) {
        int rc = build_tmap(p, packed_dev);
        if (rc != CORR_OK) return rc;
        corr::ImmaParams prm;
        prm.N = p->N;
        prm.F = p->F;
        prm.T = p->T;
        prm.t_per_chunk = p->t_per_slice;
        prm.out_mode = out_mode;
        prm.vis = vis_dev;
        dim3 grid((unsigned)(p->num_units / p->slices), (unsigned)p->slices);
        if (p->n_pad == 16)
            corr::corr_imma_kernel<1><<<grid, corr::ImmaCfg<1>::THREADS, corr::IM_SMEM_BYTES, stream>>>(p->tmap, prm);
        else if (p->n_pad == 32)
            corr::corr_imma_kernel<2><<<grid, corr::ImmaCfg<2>::THREADS, corr::IM_SMEM_BYTES, stream>>>(p->tmap, prm);
        else if (p->n_pad == 48)
            corr::corr_imma_kernel<3><<<grid, corr::ImmaCfg<3>::THREADS, corr::IM_SMEM_BYTES, stream>>>(p->tmap, prm);
        else
            corr::corr_imma_kernel<4><<<grid, corr::ImmaCfg<4>::THREADS, corr::IM_SMEM_BYTES, stream>>>(p->tmap, prm);
    } else if (p->path == CORR_PATH_DP4A) {
        dim3 grid((unsigned)(p->F * p->tiles_per_f), (unsigned)p->slices);
        switch (p->tile) {
        case 16:
            corr::corr_dp4a_kernel<16><<<grid, corr::DP4A_THREADS, 0, stream>>>(
                packed_dev, vis_dev, p->tiles_dev, p->tiles_per_f, p->N, p->F, p->T, p->t_per_slice, out_mode, p->aligned);
            break;
        case 32:
            corr::corr_dp4a_kernel<32><<<grid, corr::DP4A_THREADS, 0, stream>>>(
                packed_dev, vis_dev, p->tiles_dev, p->tiles_per_f, p->N, p->F, p->T, p->t_per_slice, out_mode, p->aligned);
            break;
        default:
            corr::corr_dp4a_kernel<64><<<grid, corr::DP4A_THREADS, 0, stream>>>(
                packed_dev, vis_dev, p->tiles_dev, p->tiles_per_f, p->N, p->F, p->T, p->t_per_slice, out_mode, p->aligned);
            break;
        }
    } else {
        int rc = build_tmap(p, packed_dev, window);
        if (rc != CORR_OK) return rc;
        if (p->variant >= 3) {
            corr::Tc3Params prm;
            prm.N = p->N;
            prm.F = p->F;
            prm.T = p->T;
            prm.tiles_per_f = p->tiles_per_f;
            prm.slices = p->slices;
            prm.t_per_slice = p->t_per_slice;
            prm.num_units = p->num_units;
            prm.out_mode = out_mode;
            prm.groups_full = p->groups_full;
            prm.groups_last = p->groups_last;
            prm.total_groups = p->total_groups;
            prm.flags = p->flags_dev;
            prm.pieces = p->pieces_dev;
            prm.tiles = p->tiles4_dev;
            prm.vis = vis_dev;
            if (p->variant == 5)
                corr::corr_tc5_kernel<<<p->grid, corr::T5_THREADS, corr::T5_SMEM_BYTES, stream>>>(p->tmap, p->tmap_y, prm);
            else
            {
                // programmatic dependent launch: the CTAs of this launch may take the SMs the previous kernel of the
                // stream frees one by one and run their prologue (barriers, TMEM, cluster handshake) there; they touch
                // global memory only after griddepcontrol.wait, i.e. after that kernel has completed
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3((unsigned)p->grid);
                cfg.blockDim = dim3(corr::T3_THREADS);
                cfg.dynamicSmemBytes = corr::T3_SMEM_BYTES;
                cfg.stream = stream;
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
                at[0].val.programmaticStreamSerializationAllowed = getenv("CORR_NO_PDL") ? 0 : 1;
                cfg.attrs = at;
                cfg.numAttrs = 1;
                CUDA_TRY(cudaLaunchKernelEx(&cfg, corr::corr_tc3_kernel, p->tmap, p->tmap_y, prm), CORR_ERR_CUDA);
            }
        } else {
            corr::TcParams prm;
            prm.N = (p->pack_sub == 64) ? 128 : p->N;
            prm.F = p->Fs;
            prm.f_out = p->F;
            prm.win_n = window ? p->N : 0;
            prm.win_c = p->win_c;
            prm.sub = p->pack_sub;
            prm.n_out = p->N;
            prm.T = p->T;
            prm.tiles_per_f = p->tiles_per_f;
            prm.slices = p->balanced ? 0 : p->slices;
            prm.groups_per_f = (p->T + corr::TD_GROUP - 1) / corr::TD_GROUP;
            prm.t_per_slice = p->t_per_slice;
            prm.num_units = p->num_units;
            prm.out_mode = out_mode;
            prm.tiles = p->tiles_dev;
            prm.vis = vis_dev;
            if (p->variant == 2 && p->tiles_per_f > 1)
                corr::corr_tcd_kernel<true><<<p->grid, corr::TD_THREADS, corr::TD_SMEM_BYTES_G, stream>>>(p->tmap, prm);
            else if (p->variant == 2)
                corr::corr_tcd_kernel<false><<<p->grid, corr::TD_THREADS, corr::TD_SMEM_BYTES, stream>>>(p->tmap, prm);
            else
                corr::corr_tc_kernel<<<p->grid, corr::TC_THREADS, corr::TC_SMEM_BYTES, stream>>>(p->tmap, prm);
        }
    }
    CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
    return CORR_OK;
}

constexpr int GATE_MERGE_MAX_G = 1024;   // gates that can share one pass (their starts and counts travel with the row order)

int corr_execute_gated(corr_plan *p, const uint8_t *packed_dev, const int32_t *gate_host, int G, int32_t *vis_dev,
                       int accumulate_flag, corr_stream_t stream_)
{
    if (!p || !packed_dev || !gate_host || !vis_dev || G < 1) {
        set_err("corr_execute_gated: NULL plan or buffer, or G < 1");
        return CORR_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int T = p->T;
    const size_t row_bytes = (size_t)p->F * p->N;
    const size_t vis_per_gate = corr_vis_elems(p);
    // ---- host: rows grouped by gate (stable), run lengths
    std::vector<int> count((size_t)G, 0);
    for (int t = 0; t < T; ++t) {
        const int g = gate_host[t];
        if (g >= G || g < -1) {
            set_err("corr_execute_gated: gate[%d] = %d is outside [-1, %d)", t, g, G);
            return CORR_ERR_INVALID_ARG;
        }
        if (g >= 0) ++count[(size_t)g];
    }
    if (row_bytes % 16 == 0 && (reinterpret_cast<uintptr_t>(packed_dev) & 15u)) {
        set_err("corr_execute_gated: packed_dev must be 16-byte aligned");
        return CORR_ERR_INVALID_ARG;
    }
    if (!p->order_pin) {
        // first gated call of the plan: all of the scratch or none of it (order_pin is the "ready" mark, set last)
        int *pin = nullptr, *odev = nullptr;
        uint8_t *gbuf = nullptr;
        cudaEvent_t ev = nullptr;
        // rows of all gates + alignment padding per run; or the gates side by side, padded to the longest (<= 5/4)
        const size_t gbytes = std::max((size_t)T * row_bytes + 16 * (size_t)T + 16, ((size_t)T + (size_t)T / 4 + 1) * row_bytes);
        const size_t oints = (size_t)T + 2 * (size_t)GATE_MERGE_MAX_G;
        const bool ok = cudaMallocHost(&pin, oints * sizeof(int)) == cudaSuccess &&
                        cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess &&
                        cudaMalloc(&odev, oints * sizeof(int)) == cudaSuccess &&
                        cudaMalloc(&gbuf, gbytes) == cudaSuccess;
        std::map<long long, corr_plan *> *plans = ok ? new (std::nothrow) std::map<long long, corr_plan *>() : nullptr;
        if (!ok || !plans) {
            set_err("corr_execute_gated: allocation of the gating scratch failed: %s", cudaGetErrorString(cudaGetLastError()));
            if (gbuf) cudaFree(gbuf);
            if (odev) cudaFree(odev);
            if (ev) cudaEventDestroy(ev);
            if (pin) cudaFreeHost(pin);
            return CORR_ERR_ALLOC;
        }
        p->ev_gate = ev;
        p->order_dev = odev;
        p->gate_buf = gbuf;
        p->gate_buf_bytes = gbytes;
        p->gate_plans = plans;
        p->order_pin = pin;
    } else {
        CUDA_TRY(cudaEventSynchronize(p->ev_gate), CORR_ERR_CUDA);   // the previous call's upload has left order_pin
    }
    std::vector<int> start((size_t)G + 1, 0);
    for (int g = 0; g < G; ++g) start[(size_t)g + 1] = start[(size_t)g] + count[(size_t)g];
    {
        std::vector<int> fill(start.begin(), start.end() - 1);
        for (int t = 0; t < T; ++t)
            if (gate_host[t] >= 0) p->order_pin[fill[(size_t)gate_host[t]]++] = t;
    }
    const int used = start[(size_t)G];
    // ---- gates of about the same length (a periodic signal cut into G phase bins): ONE pass over all of them.  The
    //      gathered rows are laid out [j][g][F][N] (sample j of gate g; gates shorter than the longest are filled up
    //      with stored zeros, which add nothing), which is the stream of G*F channels and max-length samples, and
    //      its visibilities [G*F][B] are vis[G][F][B]: G times fewer launches, cold starts and tails
    const int tmax = *std::max_element(count.begin(), count.end());
    if (G >= 2 && G <= GATE_MERGE_MAX_G && row_bytes % 16 == 0 && used > 0 && (long long)G * p->F <= 65535 &&
        (long long)tmax * G <= (long long)used + used / 4 && (size_t)tmax * G * row_bytes <= p->gate_buf_bytes &&
        !getenv("CORR_GATED_PER_GATE")) {
        const long long key = ((long long)G << 32) | (long long)tmax;
        auto it = p->gate_plans->find(key);
        if (it == p->gate_plans->end()) {
            if (p->gate_plans->size() >= 64) {
                corr_plan_destroy(p->gate_plans->begin()->second);   // waits for its kernels (cudaFree inside)
                p->gate_plans->erase(p->gate_plans->begin());
            }
            corr_plan *np = corr_plan_create_ex(p->N, G * p->F, tmax, p->path);
            if (!np) return g_create_rc;
            it = p->gate_plans->emplace(key, np).first;
        }
        for (int g = 0; g < G; ++g) {
            p->order_pin[(size_t)T + 2 * (size_t)g] = start[(size_t)g];
            p->order_pin[(size_t)T + 2 * (size_t)g + 1] = count[(size_t)g];
        }
        CUDA_TRY(cudaMemcpyAsync(p->order_dev, p->order_pin, (size_t)used * sizeof(int), cudaMemcpyHostToDevice, stream),
                 CORR_ERR_CUDA);
        CUDA_TRY(cudaMemcpyAsync(p->order_dev + T, p->order_pin + T, 2 * (size_t)G * sizeof(int), cudaMemcpyHostToDevice, stream),
                 CORR_ERR_CUDA);
        CUDA_TRY(cudaEventRecord(p->ev_gate, stream), CORR_ERR_CUDA);
        corr::corr_gate_gather_merged_kernel<<<8 * p->sm_count, corr::GATE_THREADS, 0, stream>>>(
            packed_dev, p->gate_buf, p->order_dev, reinterpret_cast<const int2 *>(p->order_dev + T), G, tmax, (int)(row_bytes / 16));
        CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
        return corr_execute(it->second, p->gate_buf, vis_dev, accumulate_flag, stream_);
    }
    // byte offset of every gate's run in gate_buf: runs start on 16-byte boundaries (corr_execute needs that)
    std::vector<size_t> off((size_t)G, 0);
    {
        size_t o = 0;
        for (int g = 0; g < G; ++g) {
            off[(size_t)g] = o;
            o = (o + (size_t)count[(size_t)g] * row_bytes + 15) & ~(size_t)15;
        }
    }
    if (used > 0) {
        CUDA_TRY(cudaMemcpyAsync(p->order_dev, p->order_pin, (size_t)used * sizeof(int), cudaMemcpyHostToDevice, stream),
                 CORR_ERR_CUDA);
        CUDA_TRY(cudaEventRecord(p->ev_gate, stream), CORR_ERR_CUDA);
        const int blocks = 8 * p->sm_count;
        if (row_bytes % 16 == 0) {   // runs are back to back: one launch for all gates
            corr::corr_gate_gather_kernel<<<blocks, corr::GATE_THREADS, 0, stream>>>(packed_dev, p->gate_buf, p->order_dev, used,
                                                                                     (int)(row_bytes / 16));
        } else {
            for (int g = 0; g < G; ++g)
                if (count[(size_t)g] > 0)
                    corr::corr_gate_gather_bytes_kernel<<<blocks, corr::GATE_THREADS, 0, stream>>>(
                        packed_dev, p->gate_buf + off[(size_t)g], p->order_dev + start[(size_t)g], count[(size_t)g], (int)row_bytes);
        }
        CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
    } else {
        CUDA_TRY(cudaEventRecord(p->ev_gate, stream), CORR_ERR_CUDA);
    }
    // ---- one ordinary correlation per gate on its run of rows
    for (int g = 0; g < G; ++g) {
        int32_t *vis_g = vis_dev + (size_t)g * vis_per_gate;
        const int len = count[(size_t)g];
        if (len == 0) {
            if (!accumulate_flag) CUDA_TRY(cudaMemsetAsync(vis_g, 0, vis_per_gate * sizeof(int32_t), stream), CORR_ERR_CUDA);
            continue;
        }
        auto it = p->gate_plans->find((long long)len);
        if (it == p->gate_plans->end()) {
            if (p->gate_plans->size() >= 64) {
                // bound the cache: drop ONE plan whose run length this call does not use (its kernels, if any are
                // still in flight from an earlier call, are waited for by the cudaFree inside destroy)
                for (auto ev = p->gate_plans->begin(); ev != p->gate_plans->end(); ++ev)
                    if ((ev->first >> 32) != 0 || std::find(count.begin(), count.end(), (int)ev->first) == count.end()) {
                        corr_plan_destroy(ev->second);
                        p->gate_plans->erase(ev);
                        break;
                    }
            }
            corr_plan *np = corr_plan_create_ex(p->N, p->F, len, p->path);
            if (!np) return g_create_rc;   // the sub-plan's own error (message already set)
            it = p->gate_plans->emplace((long long)len, np).first;
        }
        int rc = corr_execute(it->second, p->gate_buf + off[(size_t)g], vis_g, accumulate_flag, stream_);
        if (rc != CORR_OK) return rc;
    }
    return CORR_OK;
}

int corr_submit_host(corr_plan *p, const uint8_t *packed_host, int32_t *vis_host, int accumulate_flag,
                     corr_stream_t stream_)
{
    if (!p || !packed_host || !vis_host) {
        set_err("corr_submit_host: NULL plan or buffer");
        return CORR_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const size_t in_bytes = corr_input_bytes(p), out_bytes = corr_vis_elems(p) * sizeof(int32_t);

    // Large transfers: pipeline over groups of channels (channels are independent), so that the
    // host->device copy of group g+1, the kernels of group g and the device->host copy of group g-1 overlap
    // (PCIe is full duplex) -- inside one call and, because nothing here waits for the device, across
    // successive calls.  Each group's slice of the stream is gathered by a strided 2-D copy into a contiguous
    // [T][Fg][N] staging buffer (two of them, used alternately); its output is contiguous in vis.
    if (p->host_fg == 0) {
        p->host_fg = -1;   // decided once
        bool ok = cudaEventCreateWithFlags(&p->ev_done, cudaEventDisableTiming) == cudaSuccess;
        int groups = 0;
        for (int g = std::min(p->F, 8); g >= 2; --g)
            if (p->F % g == 0) { groups = g; break; }
        if (ok && groups >= 2 && in_bytes + out_bytes >= (size_t)(32 << 20)) {
            corr_plan *sub = corr_plan_create_ex(p->N, p->F / groups, p->T, p->path);
            if (sub) {
                ok = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking) == cudaSuccess &&
                     cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking) == cudaSuccess;
                ok = ok && cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming) == cudaSuccess &&
                     cudaEventCreateWithFlags(&p->ev_comp, cudaEventDisableTiming) == cudaSuccess;
                for (int i = 0; i < 2 && ok; ++i)
                    ok = cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
                         cudaEventCreateWithFlags(&p->ev_free[i], cudaEventDisableTiming) == cudaSuccess;
                for (int i = 0; i < 8 && ok; ++i)
                    ok = cudaEventCreateWithFlags(&p->ev_out[i], cudaEventDisableTiming) == cudaSuccess;
                if (ok) {
                    p->sub = sub;
                    p->host_fg = p->F / groups;
                } else {
                    corr_plan_destroy(sub);
                }
            }
        }
        if (!ok) {
            set_err("corr_submit_host: cannot create the copy streams/events: %s", cudaGetErrorString(cudaGetLastError()));
            p->host_fg = 0;
            return CORR_ERR_CUDA;
        }
    }
    if (p->sub) {
        const int fg = p->host_fg, groups = p->F / fg;
        const size_t grp_in = (size_t)p->T * fg * p->N;
        const size_t grp_out = (size_t)fg * ((size_t)p->N * (p->N + 1) / 2) * 2;   // int32 elements
        if (!p->packed_own) CUDA_TRY(cudaMalloc(&p->packed_own, 2 * grp_in), CORR_ERR_ALLOC);
        if (!p->vis_own) CUDA_TRY(cudaMalloc(&p->vis_own, out_bytes), CORR_ERR_ALLOC);
        CUDA_TRY(cudaEventRecord(p->ev_start, stream), CORR_ERR_CUDA);       // everything follows the caller's stream
        CUDA_TRY(cudaStreamWaitEvent(p->s_in, p->ev_start, 0), CORR_ERR_CUDA);
        CUDA_TRY(cudaStreamWaitEvent(p->s_out, p->ev_start, 0), CORR_ERR_CUDA);
        for (int g = 0; g < groups; ++g, ++p->grp_seq) {
            const int b = (int)(p->grp_seq & 1);
            uint8_t *din = p->packed_own + (size_t)b * grp_in;
            int32_t *dvis = p->vis_own + (size_t)g * grp_out;
            if (p->grp_seq >= 2) CUDA_TRY(cudaStreamWaitEvent(p->s_in, p->ev_free[b], 0), CORR_ERR_CUDA);   // staging buffer b is free again
            CUDA_TRY(cudaMemcpy2DAsync(din, (size_t)fg * p->N, packed_host + (size_t)g * fg * p->N, (size_t)p->F * p->N,
                                       (size_t)fg * p->N, (size_t)p->T, cudaMemcpyHostToDevice, p->s_in), CORR_ERR_CUDA);
            if (p->calls_submitted > 0) {
                // the previous call's copy-out of this group's image has finished (device image and, when the caller
                // chains calls through one host buffer, the host data this call reads back in)
                CUDA_TRY(cudaStreamWaitEvent(p->s_in, p->ev_out[g], 0), CORR_ERR_CUDA);
                CUDA_TRY(cudaStreamWaitEvent(stream, p->ev_out[g], 0), CORR_ERR_CUDA);
            }
            if (accumulate_flag)
                CUDA_TRY(cudaMemcpyAsync(dvis, vis_host + (size_t)g * grp_out, grp_out * sizeof(int32_t),
                                         cudaMemcpyHostToDevice, p->s_in), CORR_ERR_CUDA);
            CUDA_TRY(cudaEventRecord(p->ev_in[b], p->s_in), CORR_ERR_CUDA);
            CUDA_TRY(cudaStreamWaitEvent(stream, p->ev_in[b], 0), CORR_ERR_CUDA);
            int rc = corr_execute(p->sub, din, dvis, accumulate_flag, stream_);
            if (rc != CORR_OK) return rc;
            CUDA_TRY(cudaEventRecord(p->ev_free[b], stream), CORR_ERR_CUDA);
            CUDA_TRY(cudaEventRecord(p->ev_comp, stream), CORR_ERR_CUDA);
            CUDA_TRY(cudaStreamWaitEvent(p->s_out, p->ev_comp, 0), CORR_ERR_CUDA);
            CUDA_TRY(cudaMemcpyAsync(vis_host + (size_t)g * grp_out, dvis, grp_out * sizeof(int32_t),
                                     cudaMemcpyDeviceToHost, p->s_out), CORR_ERR_CUDA);
            CUDA_TRY(cudaEventRecord(p->ev_out[g], p->s_out), CORR_ERR_CUDA);
        }
        CUDA_TRY(cudaEventRecord(p->ev_done, p->s_out), CORR_ERR_CUDA);
        ++p->calls_submitted;
        return CORR_OK;
    }
    if (!p->packed_own) CUDA_TRY(cudaMalloc(&p->packed_own, in_bytes), CORR_ERR_ALLOC);
    if (!p->vis_own) CUDA_TRY(cudaMalloc(&p->vis_own, out_bytes), CORR_ERR_ALLOC);
    CUDA_TRY(cudaMemcpyAsync(p->packed_own, packed_host, in_bytes, cudaMemcpyHostToDevice, stream), CORR_ERR_CUDA);
    if (accumulate_flag)
        CUDA_TRY(cudaMemcpyAsync(p->vis_own, vis_host, out_bytes, cudaMemcpyHostToDevice, stream), CORR_ERR_CUDA);
    int rc = corr_execute(p, p->packed_own, p->vis_own, accumulate_flag, stream_);
    if (rc != CORR_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(vis_host, p->vis_own, out_bytes, cudaMemcpyDeviceToHost, stream), CORR_ERR_CUDA);
    CUDA_TRY(cudaEventRecord(p->ev_done, stream), CORR_ERR_CUDA);
    ++p->calls_submitted;
    return CORR_OK;
}

int corr_wait_host(corr_plan *p)
{
    if (!p) {
        set_err("corr_wait_host: NULL plan");
        return CORR_ERR_INVALID_ARG;
    }
    if (p->calls_submitted == 0) return CORR_OK;
    CUDA_TRY(cudaEventSynchronize(p->ev_done), CORR_ERR_CUDA);   // the last copy-out of the last submitted call
    return CORR_OK;
}

int corr_execute_host(corr_plan *p, const uint8_t *packed_host, int32_t *vis_host, int accumulate_flag,
                      corr_stream_t stream_)
{
    int rc = corr_submit_host(p, packed_host, vis_host, accumulate_flag, stream_);
    if (rc != CORR_OK) return rc;
    return corr_wait_host(p);
}


}  // extern "C"

// ---------------------------------------------------------------- corr_execute_noalloc
// For callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc): the small-N pass without a plan.  What a plan owns for this path is one piece of scratch memory, the
// copy of the stream padded to a multiple of 16 inputs (corr_pad_kernel writes it, corr_imma_kernel reads it through
// TMA); here that scratch is a file-scope array every GPU that loads the library holds until exit.  In host code the
// array's name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress, once per
// device, with that device current.
static __device__ __align__(256) uint8_t g_noalloc_scratch[CORR_NOALLOC_MAX_BYTES];

namespace {
struct NoallocDevice {
    bool ready;
    uint8_t *scratch;   // device address of g_noalloc_scratch on this device
    int sms;
    int occ[4];         // resident CTAs per SM of corr_imma_kernel<1..4>
};
NoallocDevice g_noalloc_dev[CORR_NOALLOC_MAX_DEVICES];
std::mutex g_noalloc_mutex;

template <int NT16> cudaError_t noalloc_setup_kernel(int *occ)
{
    cudaError_t e = cudaFuncSetAttribute(corr::corr_imma_kernel<NT16>, cudaFuncAttributeMaxDynamicSharedMemorySize, corr::IM_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, corr::corr_imma_kernel<NT16>, corr::ImmaCfg<NT16>::THREADS, corr::IM_SMEM_BYTES);
    return e;
}

// Set-up of the current device (first call on it): the scratch array's device address and the launch attributes.
int noalloc_device(const NoallocDevice **out)
{
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev), CORR_ERR_CUDA);
    if (dev < 0 || dev >= CORR_NOALLOC_MAX_DEVICES) {
        set_err("corr_execute_noalloc: device ordinal %d is beyond the %d this entry point keeps state for", dev, CORR_NOALLOC_MAX_DEVICES);
        return CORR_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoallocDevice &d = g_noalloc_dev[dev];
    if (!d.ready) {
        void *ptr = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&ptr, g_noalloc_scratch), CORR_ERR_CUDA);
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u)) {
            set_err("corr_execute_noalloc: cudaGetSymbolAddress gave %p for the scratch array", ptr);
            return CORR_ERR_CUDA;
        }
        CUDA_TRY(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev), CORR_ERR_CUDA);
        CUDA_TRY(noalloc_setup_kernel<1>(&d.occ[0]), CORR_ERR_CUDA);
        CUDA_TRY(noalloc_setup_kernel<2>(&d.occ[1]), CORR_ERR_CUDA);
        CUDA_TRY(noalloc_setup_kernel<3>(&d.occ[2]), CORR_ERR_CUDA);
        CUDA_TRY(noalloc_setup_kernel<4>(&d.occ[3]), CORR_ERR_CUDA);
        for (int i = 0; i < 4; ++i)
            if (d.occ[i] < 1) {
                set_err("corr_execute_noalloc: cannot reserve %d B of shared memory per CTA", corr::IM_SMEM_BYTES);
                return CORR_ERR_CUDA;
            }
        d.scratch = static_cast<uint8_t *>(ptr);
        d.ready = true;
    }
    *out = &d;
    return CORR_OK;
}
}  // namespace

extern "C" {

int corr_execute_noalloc(int N, int F, int T, const uint8_t *packed_dev, int32_t *vis_dev, int accumulate_flag,
                         corr_stream_t stream_)
{
    if (N < 1 || N > 64 || F < 1 || T < 1 || T > 16777215) {
        set_err("corr_execute_noalloc: need 1 <= N <= 64, F >= 1, 1 <= T <= 16777215 (got N=%d F=%d T=%d)", N, F, T);
        return (N > 64) ? CORR_ERR_UNSUPPORTED : CORR_ERR_INVALID_ARG;
    }
    if (!packed_dev || !vis_dev || (reinterpret_cast<uintptr_t>(vis_dev) & 7u)) {
        set_err("corr_execute_noalloc: NULL buffer, or vis_dev not 8-byte aligned");
        return CORR_ERR_INVALID_ARG;
    }
    const int n_pad = (N + 15) / 16 * 16;
    const bool padded = n_pad != N;
    const unsigned long long need = padded ? (unsigned long long)T * (unsigned long long)F * (unsigned long long)n_pad : 0ull;
    if (need > (unsigned long long)CORR_NOALLOC_MAX_BYTES) {
        set_err("corr_execute_noalloc: the padded stream T*F*%d = %llu bytes exceeds the static scratch of %llu bytes "
                "(CORR_NOALLOC_MAX_BYTES); use a plan (corr_plan_create + corr_execute) for this size",
                n_pad, need, (unsigned long long)CORR_NOALLOC_MAX_BYTES);
        return CORR_ERR_UNSUPPORTED;
    }
    if ((unsigned long long)F * (unsigned long long)n_pad > 0x7fffffffull) {
        set_err("corr_execute_noalloc: F*N too large");
        return CORR_ERR_INVALID_ARG;
    }
    if (!padded && (reinterpret_cast<uintptr_t>(packed_dev) & 15u)) {
        set_err("corr_execute_noalloc: packed_dev must be 16-byte aligned when N is a multiple of 16");
        return CORR_ERR_INVALID_ARG;
    }
    if (!get_encode_fn()) {
        set_err("corr_execute_noalloc: cuTensorMapEncodeTiled not available from the driver");
        return CORR_ERR_CUDA;
    }
    const NoallocDevice *d = nullptr;
    int rc = noalloc_device(&d);
    if (rc != CORR_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(stream_);

    // ---- the schedule corr_plan_create makes for this path: strips of 128 / n_pad channels x chunks of time samples
    const int nt16 = n_pad / 16, fb = 128 / n_pad;
    const int strips = (F + fb - 1) / fb;
    const int slots = d->sms * d->occ[nt16 - 1];
    const int min_chunks = (T + corr::IM_MAX_CHUNK - 1) / corr::IM_MAX_CHUNK;   // int32 headroom of a chunk
    int chunks = min_chunks;
    double best = 0.0;
    for (int c = min_chunks; c <= std::max(min_chunks, std::min(T / 512, 4 * slots / strips + 1)); ++c) {
        const long long units = (long long)strips * c;
        const double eff = (double)units / (double)(((units + slots - 1) / slots) * slots);
        if (eff > best + 0.10) { best = eff; chunks = c; }
    }
    const int t_per_chunk = ((T + chunks - 1) / chunks + corr::IM_ROWS - 1) / corr::IM_ROWS * corr::IM_ROWS;
    const int slices = (T + t_per_chunk - 1) / t_per_chunk;
    if (strips > 0x7fffffff / std::max(1, slices) || slices > 65535) {
        set_err("corr_execute_noalloc: too many work units");
        return CORR_ERR_INVALID_ARG;
    }

    // ---- N % 16 != 0: pad into the static scratch.  Every byte the pass reads is written here first, so nothing has
    //      to be cleared although the array keeps the last call's contents
    const uint8_t *src = packed_dev;
    if (padded) {
        corr::corr_pad_kernel<<<8 * d->sms, 256, 0, stream>>>(packed_dev, d->scratch, N, n_pad, (long long)T * F);
        CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
        src = d->scratch;
    }
    int out_mode;
    if (slices > 1) {
        out_mode = corr::OUT_ATOMIC;
        if (!accumulate_flag)
            CUDA_TRY(cudaMemsetAsync(vis_dev, 0, (size_t)F * ((size_t)N * (N + 1) / 2) * 2 * sizeof(int32_t), stream), CORR_ERR_CUDA);
    } else {
        out_mode = accumulate_flag ? corr::OUT_RMW : corr::OUT_STORE;
    }
    // the stream as a byte matrix, innermost first: (F * n_pad, T)
    CUtensorMap tmap;
    const cuuint64_t dims2[2] = {(cuuint64_t)F * (cuuint64_t)n_pad, (cuuint64_t)T};
    const cuuint64_t strides2[1] = {(cuuint64_t)F * (cuuint64_t)n_pad};
    const cuuint32_t box2[2] = {128u, (cuuint32_t)corr::IM_ROWS};
    const cuuint32_t estr2[2] = {1u, 1u};
    CUresult r2 = get_encode_fn()(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(src), dims2, strides2, box2, estr2,
                                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r2 != CUDA_SUCCESS) {
        set_err("corr_execute_noalloc: cuTensorMapEncodeTiled failed with CUresult %d (N=%d F=%d T=%d)", (int)r2, N, F, T);
        return CORR_ERR_CUDA;
    }
    corr::ImmaParams prm;
    prm.N = N;
    prm.F = F;
    prm.T = T;
    prm.t_per_chunk = t_per_chunk;
    prm.out_mode = out_mode;
    prm.vis = vis_dev;
    dim3 grid((unsigned)strips, (unsigned)slices);
    if (nt16 == 1)
        corr::corr_imma_kernel<1><<<grid, corr::ImmaCfg<1>::THREADS, corr::IM_SMEM_BYTES, stream>>>(tmap, prm);
    else if (nt16 == 2)
        corr::corr_imma_kernel<2><<<grid, corr::ImmaCfg<2>::THREADS, corr::IM_SMEM_BYTES, stream>>>(tmap, prm);
    else if (nt16 == 3)
        corr::corr_imma_kernel<3><<<grid, corr::ImmaCfg<3>::THREADS, corr::IM_SMEM_BYTES, stream>>>(tmap, prm);
    else
        corr::corr_imma_kernel<4><<<grid, corr::ImmaCfg<4>::THREADS, corr::IM_SMEM_BYTES, stream>>>(tmap, prm);
    CUDA_TRY(cudaGetLastError(), CORR_ERR_CUDA);
    return CORR_OK;
}

}  // extern "C"
