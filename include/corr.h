/* corr.h -- C ABI of the B200-native X-engine (the O(N^2) hot path of arXiv 1503.06203).
 *
 * For each frequency channel f the library accumulates, over the T time samples of a call,
 *
 *      A_f[x][y] = sum_t X_t[x] * conj(X_t[y])          0 <= x <= y < N
 *
 * i.e. Eq. (1) of the paper, Corr(X,Y) = XY* = (XRe*YRe + XIm*YIm, XIm*YRe - XRe*YIm)
 * (PAPER.md:41-44), accumulated over time, upper triangle only because A is
 * Hermitian (Eq. 2), every channel independent.
 *
 * Input format (PAPER.md:76 and Fig. 2 at :82): time-major, then frequency, then the N input
 * elements; ONE BYTE per complex sample, Re and Im each a 4-bit offset-encoded ("excess-8")
 * integer: stored nibble = value + 8, value in [-8, 7].  The paper's text does not say which
 * nibble is which; this library fixes Re = high nibble, Im = low nibble:
 *      byte = ((Re + 8) << 4) | (Im + 8).
 *
 * Output format ("signed 32+32-bit complex correlation products"): int32 pairs
 * (Re, Im), dense upper triangle in row-major order:
 *      vis[f][b(x,y)][0..1],   b(x,y) = x*N - x*(x-1)/2 + (y - x),   B = N(N+1)/2 per channel.
 * The paper's tile-blocked output addressing and its output lock are not
 * reproduced; see DESIGN.md.
 *
 * All arithmetic is exact integer arithmetic.  One time sample adds at most 128 to |Re| and 120
 * to |Im|, so an output buffer is overflow-free while the TOTAL number of samples accumulated
 * into it (over all calls with accumulate_flag != 0) is <= 16 777 215 = floor((2^31-1)/128).
 * Beyond that the result is two's-complement wraparound; the library cannot see across calls and
 * does not check.
 *
 * Threading: a plan may be executed repeatedly on one stream.  Concurrent corr_execute calls on
 * the SAME plan from different streams or threads are not supported (the plan owns device
 * scratch).  Different plans are independent.  corr_last_error() is thread-local.
 *
 * There is no CPU fallback: every entry point that computes needs a CUDA device of compute
 * capability 10.0 (sm_100a) and fails with CORR_ERR_CUDA / CORR_ERR_UNSUPPORTED otherwise.
 */
#ifndef CORR_B200_H
#define CORR_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct corr_plan corr_plan; /* opaque; owned by the library */

/* CUDA stream handle, passed as a plain pointer (cudaStream_t / CUstream); NULL = default stream. */
typedef void *corr_stream_t;

enum {
    CORR_OK = 0,
    CORR_ERR_INVALID_ARG = 1, /* bad N/F/T, NULL or misaligned pointer, NULL plan */
    CORR_ERR_UNSUPPORTED = 2, /* device is not sm_100, or forced path cannot serve this shape */
    CORR_ERR_ALLOC = 3,       /* host or device allocation failed */
    CORR_ERR_CUDA = 4         /* a CUDA runtime/driver call or kernel launch failed */
};

/* Which kernel family a plan uses (S4 vs S4' of SURVEY.md S8(a)). */
enum {
    CORR_PATH_AUTO = 0,  /* library chooses from (N, F, T) */
    CORR_PATH_DP4A = 1,  /* CUDA-core dp4a kernels; any N (small-N path) */
    CORR_PATH_TCGEN05 = 2, /* TMA + tcgen05 int8 MMA, int32 accumulators in TMEM; any N (padded copy if N % 16 != 0) */
    CORR_PATH_IMMA = 3     /* TMA + warp-level int8 MMA on whole channels; N <= 64 (small-N path) */
};

/* corr_plan_create -- validate the shape, choose the path, build the triangular tile schedule
 * (only tiles on or above the diagonal) and allocate the plan's device scratch.
 *   N  number of input elements,           N >= 1
 *   F  number of frequency channels,       F >= 1
 *   T  time samples per corr_execute call, 1 <= T <= 16 777 215
 * Returns NULL on failure; the reason is in corr_last_error().
 * Automatic choice: N <= 64 -> CORR_PATH_IMMA (except N = 64 with an even F or F >= 5: two channels per tcgen05 tile), larger
 * N -> CORR_PATH_TCGEN05 (one CTA per 128 x 128 block up to N = 128, and up to N = 256 when T is long enough for
 * segments of 4096 samples; CTA-pair 256 x 128 tiles otherwise).  When
 * N % 16 != 0 these two paths first copy the stream to a plan-owned buffer padded to the next multiple of 16 inputs
 * (TMA strides and box start addresses are multiples of 16 bytes) -- except N <= 113 with F*N % 16 == 0 and a
 * 16-byte aligned packed_dev, which the tcgen05 path reads in place through 16-byte aligned windows (the automatic
 * choice for such N below 64 as well; there a misaligned packed_dev is CORR_ERR_INVALID_ARG); CORR_PATH_DP4A takes any N without a copy and is
 * only used on request.  Testing aids (environment, read at plan creation): CORR_FORCE_PATH=dp4a|tcgen05|imma
 * overrides the choice; CORR_TC_VARIANT=1|3|5 forces the tcgen05 kernel (1 single-CTA tiles with both operands in
 * shared memory -- the round-1 kernel the N <= 128 kernel replaced --, 3 CTA pairs, 5 = CTA
 * pairs with three products per complex MAC on the stored bytes and the Eq. 3 offset correction).
 * CORR_NO_PDL (read at every corr_execute) launches the CTA-pair kernel without programmatic stream serialisation. */
corr_plan *corr_plan_create(int N, int F, int T);

/* Same, with the path given explicitly (CORR_PATH_*).  CORR_ERR_UNSUPPORTED -> NULL if the
 * path cannot serve the shape. */
corr_plan *corr_plan_create_ex(int N, int F, int T, int path);

/* corr_execute -- enqueue one correlation pass on `stream` and return without synchronising.
 *   packed_dev  DEVICE pointer, T*F*N bytes, layout [T][F][N], format above; 16-byte aligned;
 *               read only; must stay valid until the stream reaches the end of this call's work.
 *   vis_dev     DEVICE pointer, F*N(N+1)/2*2 int32, layout [F][B][2] above; 8-byte aligned.
 *   accumulate_flag  0: every entry of vis_dev is overwritten (whatever it held, including
 *               Im = 0 on the diagonal); nonzero: the result is added, modulo 2^32, to what
 *               vis_dev holds (the paper's output buffer persists across launches and is added
 *               to).
 *   stream      CUDA stream the work is enqueued on.
 * Returns CORR_OK or an error code; errors found at enqueue time are returned here, later
 * device faults surface at the caller's own synchronisation.  The caller owns both buffers.
 * The call only enqueues kernels and memsets, so it may be captured into a CUDA graph and replayed
 * (with the buffers it was captured with).
 * A plan holds per-call state (the tensor map of the last input pointer, the schedule's flags and
 * call counter, scratch buffers): calls on ONE plan must be issued from one host thread at a time
 * and onto one stream (or streams the caller orders); use one plan per concurrent stream. */
int corr_execute(corr_plan *plan, const uint8_t *packed_dev, int32_t *vis_dev,
                 int accumulate_flag, corr_stream_t stream);

/* corr_execute_host -- the same pass with HOST buffers: copies packed_host to a plan-owned
 * device buffer, runs corr_execute, copies the result back, all on `stream`, then synchronises
 * the stream.  With accumulate_flag != 0 vis_host is first copied to the device and added to.
 * Pinned host memory makes the copies asynchronous; pageable memory works but is slower.
 * For large transfers (>= 32 MB, F > 1) the work is pipelined over groups of channels (channels
 * are independent): the host->device copy of one group, the kernels of the previous
 * one and the device->host copy of the one before run concurrently on plan-owned streams that
 * are ordered after `stream` at entry and joined into it before the final synchronisation. */
int corr_execute_host(corr_plan *plan, const uint8_t *packed_host, int32_t *vis_host,
                      int accumulate_flag, corr_stream_t stream);

/* corr_execute_gated -- gated correlation ("gate the correlation products on multiple time
 * periods", for periodic signals such as calibration sources and pulsars): every time sample t of the
 * call belongs to gate gate[t] in [0, G), or to none (-1), and gate g gets its own matrix
 *     vis[g][f][b(x,y)] (=|+=) sum over { t : gate[t] = g } of X_t[x] conj(X_t[y])
 *   plan        a plan for (N, F, T); T is the length of gate[] and of the stream
 *   packed_dev  DEVICE pointer, [T][F][N] bytes as for corr_execute
 *   gate_host   HOST pointer, T int32; read before the call returns
 *   G           number of gates, >= 1 (at most T distinct run lengths are planned and cached)
 *   vis_dev     DEVICE pointer, G*F*N(N+1)/2*2 int32, layout [G][F][B][2]
 *   accumulate_flag  as for corr_execute, applied to every gate (a gate with no sample is zeroed / left)
 * Enqueues on `stream` (a row gather into plan-owned scratch, then ONE ordinary pass over all gates as G*F
 * channels when the gates hold about the same number of samples -- the longest at most 5/4 of the mean, shorter
 * ones filled up with stored zeros -- else one pass per gate; environment CORR_GATED_PER_GATE forces the
 * latter); may wait for the previous gated call's index upload; the first call with a new run length creates
 * a plan for it.  Returns CORR_OK or an error code. */
int corr_execute_gated(corr_plan *plan, const uint8_t *packed_dev, const int32_t *gate_host, int G,
                       int32_t *vis_dev, int accumulate_flag, corr_stream_t stream);

/* corr_time_shift -- the paper's pre-correlation time shift ("modifies the input stream
 * at the raw data level, allowing individual elements to be shifted by integer time steps
 * pre-correlation"):
 *     out[t][f][n] = in[t - lags[n]][f][n]  if 0 <= t - lags[n] < T,  else 0x88 (the sample 0 + 0i)
 * A positive lag delays element n; samples shifted in from outside the block are stored zeros, which
 * add nothing to any correlation sum.  Not in place.
 *   packed_in_dev, packed_out_dev  DEVICE pointers, T*F*N bytes each, layout [T][F][N] as above,
 *                                  distinct, 16-byte aligned when N % 16 == 0; caller-owned
 *   lags_dev                       DEVICE pointer, N int32 (any values; |lag| >= T empties the element)
 * N % 16 == 0 and N <= 65536 take the TMA-fed kernel (a tensor map of the input is encoded per call, on the
 * host), and so do 16-byte aligned streams with F*N % 16 == 0 and F*N <= 65536 (as one channel of F*N columns);
 * other shapes a byte-by-byte gather.
 * Enqueues on `stream`, does not synchronise.  Returns CORR_OK or an error code. */
int corr_time_shift(int N, int F, int T, const uint8_t *packed_in_dev, const int32_t *lags_dev,
                    uint8_t *packed_out_dev, corr_stream_t stream);

/* corr_measure_int8_tops -- measurement aid, not part of the correlation path: runs a bare issue loop of
 * the hot path's own instruction (tcgen05.mma.cta_group::2.kind::i8, 256 x 128 x 32, A in TMEM, B in shared
 * memory; `iters` x 4 MMAs per CTA pair, one pair per two SMs) on the current device's default stream,
 * synchronises, and stores the achieved dense int8 TOPS (2 ops per multiply-add) in *tops_out (HOST pointer).
 * This is the ceiling the roofline of section 8(d) is also reported against.  Returns CORR_OK or an error. */
int corr_measure_int8_tops(int iters, double *tops_out);

/* corr_submit_host / corr_wait_host -- corr_execute_host split in two, for streaming use: submit enqueues the
 * copies and kernels of one call and returns without waiting for the device, so the copy-in of the next call
 * overlaps the kernels and the copy-out of this one; corr_wait_host blocks until everything submitted on the
 * plan so far has finished (results of ALL submitted calls are then in their vis_host buffers).  Between
 * submit and wait the host buffers of that call must stay valid and untouched; use pinned memory, and a
 * different vis_host per call in flight unless the calls are meant to accumulate into one buffer
 * (accumulate_flag != 0 reads vis_host after the previous call's copy-out to it has finished).  All calls
 * of a plan go on one stream.  corr_execute_host = corr_submit_host + corr_wait_host. */
int corr_submit_host(corr_plan *plan, const uint8_t *packed_host, int32_t *vis_host,
                     int accumulate_flag, corr_stream_t stream);
int corr_wait_host(corr_plan *plan);

/* corr_plan_destroy -- free the plan and its device scratch.  NULL is a no-op. */
void corr_plan_destroy(corr_plan *plan);

/* Thread-local, NUL-terminated description of the last failure in this thread; never NULL;
 * owned by the library. */
const char *corr_last_error(void);

/* Pure host conveniences. */
size_t corr_input_bytes(const corr_plan *plan);        /* T*F*N */
size_t corr_vis_elems(const corr_plan *plan);          /* F * N(N+1)/2 * 2 int32 values */
size_t corr_baseline_index(int N, int x, int y);       /* b(x,y); requires 0 <= x <= y < N, else (size_t)-1 */

/* Plan introspection (host only).  Writes up to 8 ints:
 *   info[0] path actually chosen (CORR_PATH_DP4A / CORR_PATH_TCGEN05 / CORR_PATH_IMMA)
 *   info[1] tile edge in elements along x     info[2] tile edge along y
 *   info[3] tiles per channel on or above the diagonal
 *   info[4] T-slices per tile (split-T factor) info[5] total work units = F*tiles*slices
 *   info[6] CTAs launched by the main kernel  info[7] kernels launched per corr_execute
 * Returns CORR_OK or CORR_ERR_INVALID_ARG. */
int corr_plan_info(const corr_plan *plan, int info[8]);

/* Number of tiles of edge (tile_x, tile_y) that touch the upper triangle of an N x N matrix
 * (host only; the scheduler's counting rule, Fig. 1: N=256, 32x32 -> 36). */
int corr_count_tiles(int N, int tile_x, int tile_y);

/* The schedule of the CTA-pair kernels (step S3; PAPER.md:64-72 for the triangular tiling, PAPER.md:21 for channels as
 * independent work) for a problem (N, F, T) on `pairs` CTA pairs, computed without a device by the same code
 * corr_plan_create runs (host only).  A unit is (channel, pair tile, T-slice) = groups of 256 samples; whole waves of
 * units are dealt round-robin (unit = pair + k * pairs), the units left over are cut into pieces.
 *   info[0] pair tiles per channel        info[1] T-slices                info[2] units
 *   info[3] groups per full slice         info[4] groups in the last slice of a tile
 *   info[5] CTA pairs used (<= pairs)     info[6] whole waves             info[7] transposed tiles per channel
 *   pieces  NULL, or caller-owned int[pairs][4][4]: for every used pair up to 4 pieces (unit, first group, number of
 *           groups, early); entries with 0 groups are unused.  early = 1: the piece is computed before the pair's
 *           whole units (it is the first piece of a cut unit and stores; the others add).
 * Returns CORR_OK or CORR_ERR_INVALID_ARG. */
int corr_schedule_pairs(int N, int F, int T, int pairs, int info[8], int *pieces);

/* corr_execute_noalloc -- one correlation pass (Eq. 1, summed over time PAPER.md:48, upper triangle
 * PAPER.md:50; the same result as corr_execute on a plan for (N, F, T)) for small N WITHOUT a plan and without any
 * allocation: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it).  The scratch memory a plan would own for this path -- the copy of the stream padded to the next
 * multiple of 16 inputs, needed when N % 16 != 0 -- is a static device array of CORR_NOALLOC_MAX_BYTES inside the
 * library, which every GPU that loads the library holds until the process exits.
 *   N           1 <= N <= 64 (the warp-MMA kernel of CORR_PATH_IMMA; larger N: CORR_ERR_UNSUPPORTED, use a plan)
 *   F, T        as for corr_plan_create; when N % 16 != 0 the padded stream T * F * ceil16(N) bytes must fit
 *               CORR_NOALLOC_MAX_BYTES, else CORR_ERR_UNSUPPORTED with the sizes in corr_last_error()
 *   packed_dev  DEVICE pointer, T*F*N bytes, layout [T][F][N]; 16-byte aligned when N % 16 == 0; read only
 *   vis_dev     DEVICE pointer, F*N(N+1)/2*2 int32, layout [F][B][2]; 8-byte aligned; caller-owned
 *   accumulate_flag  as for corr_execute
 * Enqueues on `stream` (the pad copy when needed, a memset of vis_dev when T is split and the call overwrites, the
 * kernel) and returns without synchronising; calls no cudaMalloc / cudaFree or allocating library routine (the first
 * call on a device looks up the array's address and sets kernel attributes).  ALL calls on a device share the one
 * scratch array, which keeps the previous call's contents (every byte a call reads it has written itself first):
 * calls that overlap on the GPU -- two streams, or two host threads on two streams -- race on it; keep them on one
 * stream or order them with events.  Returns CORR_OK or an error code. */
#define CORR_NOALLOC_MAX_BYTES (32u << 20)   /* 32 MiB of device memory per GPU, held from library load to exit */
#define CORR_NOALLOC_MAX_DEVICES 64
int corr_execute_noalloc(int N, int F, int T, const uint8_t *packed_dev, int32_t *vis_dev, int accumulate_flag,
                         corr_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* CORR_B200_H */
