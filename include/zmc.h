/*
 * zmc.h -- C ABI of zmc_scan: batched direct Monte-Carlo integration over a parameter grid.
 *
 * What it computes (ZMCintegral-v5, arXiv 1910.01965; citations are PAPER.md lines):
 *   f(x) = \int dy g(y; x),  y in a box of R^N, x = (x_1..x_M)            (Eq. 1)
 * independently at every point x of the Cartesian product of M value lists,
 * by the direct (plain) Monte-Carlo method, one integration per grid point
 * (PAPER.md:65), with the grid cut into batches and the result returned as the
 * "multi-dimensional grid with each element being the integrated values".
 * HToD / DToH / evaluation times are reported separately as in the paper's tables
 * (PAPER.md:85, :132-140).  Readings of everything the paper leaves open (RNG = Philox4x32-10,
 * stream layout, uniforms, grid order, standard error) are listed in DESIGN.md "Readings".
 *
 * Conventions
 *   - All `const double*` inputs (bounds, lists, consts) are HOST memory, copied before the call
 *     returns; the library keeps no pointer to them.
 *   - out_mean / out_stderr: G' elements each (G' = count of the scanned flat range, default the
 *     whole grid G = prod(lists[i].count)), element r = flat index first_index + r, flat order is
 *     row-major with the LAST list fastest.  Element type and location are set by zmc_options
 *     (default: double, DEVICE memory).  The caller owns them; they must stay valid until
 *     `stream` has been synchronised.
 *   - The call only enqueues work: kernels on `stream`, result copies (host output) on an
 *     internal side stream that is joined back into `stream`.  Results are valid after
 *     cudaStreamSynchronize(stream).  If `timing` is non-NULL the call synchronises before
 *     returning and fills it.
 *   - Argument errors are detected before anything is enqueued and leave the outputs untouched.
 *     No exception crosses this boundary.  There is no CPU fallback: without a usable CUDA device
 *     every compute call returns ZMC_ERR_CUDA.
 *   - Every random word is keyed by (seed, GLOBAL flat grid index, word index), so results do
 *     not depend on batching, sub-ranges or launch shape (bit-identical for a fixed schedule).
 */
#ifndef ZMC_H_
#define ZMC_H_

#ifndef __CUDACC_RTC__      /* NVRTC (user integrands) has no host headers; zmc_compat.h supplies the types */
#include <stdint.h>
#endif

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define ZMC_API __attribute__((visibility("default")))
#else
#define ZMC_API
#endif

#define ZMC_MAX_N 16        /* integration dimensions */
#define ZMC_MAX_M 8         /* parameters */
#define ZMC_MAX_CONSTS 8    /* family constants */
#define ZMC_MAX_FARM_DEVICES 16   /* devices of one node in zmc_scan_farm */
#define ZMC_NOALLOC_MAX_LIST_VALUES 4096   /* zmc_scan_noalloc: most list entries (all M lists together) one call may pass */

typedef enum zmc_status {
    ZMC_OK = 0,
    ZMC_ERR_INVALID_ARG = 1,       /* NULL pointer; N or M out of range; count < 1; !(a_k < b_k); non-finite
                                      bound/value; n_samples < 2 or > 2^32-1 or n_samples*N > 2^34; bad option */
    ZMC_ERR_UNKNOWN_INTEGRAND = 2,
    ZMC_ERR_SHAPE_MISMATCH = 3,    /* (N, M, n_consts) not accepted by that family */
    ZMC_ERR_GRID_TOO_LARGE = 4,    /* prod(count) > 2^48, or one list longer than 2^31-1 */
    ZMC_ERR_OUT_OF_MEMORY = 5,
    ZMC_ERR_CUDA = 6,              /* see zmc_last_cuda_error() */
    ZMC_ERR_COMPILE = 7,           /* zmc_register_integrand: NVRTC missing or the body does not compile; see zmc_last_compile_log() */
    ZMC_ERR_NOALLOC_LIMIT = 8      /* zmc_scan_noalloc only: the value lists hold more than ZMC_NOALLOC_MAX_LIST_VALUES entries in total */
} zmc_status;

/* Integrand families g(y; x), SURVEY.md 8(c) S7 / BASELINE.json configs.  y_k is 0-based. */
enum {
    ZMC_FAM_C1_COS_XY = 1,        /* cos(x1*y0)                                   N=1, M=1 */
    ZMC_FAM_C2_SIN_XY2 = 2,       /* sin(x1*y0 + x2*y1)                           N=2, M=2 */
    ZMC_FAM_C3_OSCILLATORY = 3,   /* cos(2 pi u + sum_k c_k y_k), c_k = x_{(k mod 3)+1}*(k+1); consts = {u}; N>=1, M=3 */
    ZMC_FAM_C4_GAUSS_PEAK = 4,    /* exp(-a^2 sum_k (y_k-w_k)^2), a=x1, w=(x2,x2,x3,x3,x4,x4)   N=6, M=4 */
    ZMC_FAM_C5_DAMPED_COS = 5,    /* exp(-x1 |y|^2) cos(x2 y0+x3 y1+x4 y2) (1+x5 y0 y1 y2)      N=3, M=5 */
    ZMC_FAM_P6_SIN_SUM = 6,       /* sin(sum_k y_k + sum_l x_l): Eq. (2), :120 Eq. (4); any N, M */
    ZMC_FAM_CONST_ONE = 100,      /* 1 (diagnostic) */
    ZMC_FAM_PARAM_ECHO = 101,     /* x_{i+1}, consts = {i} (diagnostic) */
    ZMC_FAM_LIN_Y = 102,          /* y_k, consts = {k} (diagnostic) */
    ZMC_FAM_POLY = 103            /* prod_k y_k (diagnostic) */
};

enum { ZMC_PREC_F64 = 0, ZMC_PREC_F32E = 1 };             /* F32E: fp32 evaluate, fp64 accumulate */
enum { ZMC_OUT_F64 = 0, ZMC_OUT_F32 = 1 };
enum { ZMC_LOC_DEVICE = 0, ZMC_LOC_HOST = 1 };            /* HOST: pinned memory recommended */
enum { ZMC_SCHED_AUTO = 0, ZMC_SCHED_THREAD = 1, ZMC_SCHED_WARP = 2, ZMC_SCHED_CTA = 3 };
enum { ZMC_FAST_MATH_DEFAULT = -1, ZMC_FAST_MATH_OFF = 0, ZMC_FAST_MATH_ON = 1 };
/* zmc_options.flags */
enum {
    ZMC_OPT_EXPLICIT_COUNT = 1,   /* take `count` literally: count == 0 is an EMPTY range (nothing enqueued, nothing written)
                                     instead of "up to the end of the grid" -- for callers whose shard may be empty */
    ZMC_OPT_FRESH_LISTS = 2       /* upload the value lists even if an identical copy is cached on the device (timing runs
                                     that must contain the HToD copy) */
};
/* zmc_register_integrand_ex flags */
enum { ZMC_USER_FAST_MATH = 1 };  /* compile the user body with NVRTC --use_fast_math (fp32 only: sinf -> MUFU etc.) */

/* One parameter's value list.  Host memory. */
typedef struct zmc_param_list {
    const double* values;
    int64_t count;
} zmc_param_list;

/* Options of zmc_scan_ex.  Zero-initialise, set struct_size = sizeof(zmc_options), override fields. */
typedef struct zmc_options {
    uint32_t struct_size;
    int32_t precision;       /* ZMC_PREC_*: arithmetic of the integrand evaluation (sums are always fp64) */
    int32_t out_dtype;       /* ZMC_OUT_*: element type of out_mean / out_stderr */
    int32_t out_location;    /* ZMC_LOC_*: where out_mean / out_stderr live */
    int32_t schedule;        /* ZMC_SCHED_*: lanes per grid point (1 / 32 / one CTA); AUTO picks by (count, n_samples) */
    int32_t fast_math;       /* ZMC_FAST_MATH_*: F32E only -- MUFU sin/cos/ex2 (default ON); ignored for F64 */
    uint64_t batch_points;   /* grid points per batch; 0 = one batch */
    uint64_t first_index;    /* scan only flat indices [first_index, first_index+count) ... */
    uint64_t count;          /* ... 0 = up to the end of the grid (unless flags has ZMC_OPT_EXPLICIT_COUNT: then 0 = empty) */
    const double* consts;    /* family constants (host), n_consts of them */
    int32_t n_consts;
    int32_t flags;           /* ZMC_OPT_* bits, 0 = none */
} zmc_options;

/* Where the time went (the paper's HToD / DToH / GPU evaluation split). */
typedef struct zmc_timing {
    double h2d_ms;           /* staging of the value lists (device time; ~0 when the lists were already cached on the device) */
    double kernel_ms;        /* sum of the batch kernels' device time */
    double d2h_ms;           /* sum of the result copies' device time (host output only) */
    double exposed_d2h_ms;   /* max(0, wall - h2d - kernel): copy time NOT hidden behind compute */
    double wall_ms;          /* first enqueue to last completion, device time on `stream` */
    int64_t n_batches;
    int64_t gpu_launches;    /* kernels of this library launched by the call */
    uint64_t d2h_bytes;
    uint64_t h2d_bytes;      /* bytes this call copied host -> device (0 on a list-cache hit) */
    int32_t schedule;        /* the schedule actually used */
    int32_t host_out_pinned; /* HOST outputs: 1 = page-locked (copies overlap compute), 0 = pageable (cudaMemcpyAsync then runs
                                synchronously on the host: no overlap, exposed_d2h_ms is the whole copy); 2 = page-locked and
                                small (one batch, <= 1 MiB of results): the kernel wrote them straight into host memory, no
                                staging and no copy -- d2h_bytes counts them, d2h_ms stays 0; -1 = device outputs */
} zmc_timing;

/* What zmc_scan_farm did (the paper's allocation / evaluation view of Table 2). Host wall clock. */
typedef struct zmc_farm_timing {
    double wall_ms;                                  /* whole call */
    int64_t n_batches;
    uint64_t batch_points;
    int32_t n_devices;
    int32_t reserved;
    int64_t batches_done[ZMC_MAX_FARM_DEVICES];      /* batches each device slot ended up taking (dynamic assignment) */
    double busy_ms[ZMC_MAX_FARM_DEVICES];            /* first pull to last completion, per device slot */
} zmc_farm_timing;

typedef struct zmc_integrand_info {
    int32_t id;
    const char* name;
    int32_t N_min, N_max;    /* accepted integration dimensions */
    int32_t M_min, M_max;    /* accepted parameter counts */
    int32_t n_consts;
    int32_t has_closed_form;
} zmc_integrand_info;

#ifndef __CUDACC_RTC__      /* the entry points are host functions: not part of what NVRTC compiles */
/*
 * zmc_scan -- mean and standard error of the plain Monte-Carlo estimate at every grid point
 * (PAPER.md:55-65).  Defaults: fp64 path, double outputs in DEVICE memory, one batch, AUTO schedule.
 *   integrand_id  ZMC_FAM_*                       N        box dimensions, 1..ZMC_MAX_N
 *   bounds        2N doubles a_0,b_0,..           M        number of lists, 1..ZMC_MAX_M
 *   lists         M value lists                   n_samples samples per grid point (>= 2)
 *   seed          Philox key                      stream   cudaStream_t (as void*), may be 0
 * mean = V * avg(g),  stderr = V * sqrt(s^2 / n) with the unbiased (n-1) sample variance,
 * V = prod_k (b_k - a_k).
 * Accuracy against an exact evaluation of the same sample stream: fp64 path |d mean| <= 1e-10 max(|mean|,
 * stderr) and |d stderr| <= 1e-10 stderr + V eps_g / sqrt(n-1) with eps_g = 4.6e-16 -- the second term only matters for a
 * nearly constant integrand (spread of g below ~4e-6 |g|), where the last-bit rounding of g itself is no longer 1e-10 of the
 * spread; F32E path |d| <= 1e-4 |value| + 1e-6 max(1, V/8).
 */
ZMC_API zmc_status zmc_scan(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                    uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream);

/* Same, with options (may be NULL = defaults) and an optional timing report (may be NULL).
 * CUDA graphs: with DEVICE outputs, timing == NULL and value lists the library already holds on the device (any earlier
 * call with the same lists, not yet displaced by 8 other sets), the call enqueues one kernel per launch on `stream` and
 * nothing else, so it may be issued while `stream` is being captured.  The captured kernels read the library's cached
 * copy of the lists; the library therefore keeps that copy untouched -- never evicted, overwritten or freed -- until
 * zmc_shutdown, so the graph can be replayed at any later time, whatever is scanned in between.  At most 7 different
 * sets of value lists can be held for graphs per device.  A call issued during capture that cannot be captured (lists
 * not cached, an 8th set, host outputs, timing != NULL) returns ZMC_ERR_CUDA with zmc_last_cuda_error() =
 * cudaErrorStreamCaptureUnsupported (900) and enqueues nothing. */
ZMC_API zmc_status zmc_scan_ex(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                       uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream,
                       const zmc_options* opt, zmc_timing* timing);

/*
 * zmc_scan_noalloc -- zmc_scan_ex for callers that must not allocate GPU memory.
 * Some programs cannot let a library call cudaMalloc / cudaFree on their behalf: a server or framework that gave all
 * device memory to its own pool at start-up (a hidden allocation can turn into the owner's out-of-memory error later), a
 * latency-critical loop (both calls take a driver lock and may synchronise the whole device, stalling every stream), or a
 * deployment whose buffer plan was fixed in advance.  zmc_scan_ex keeps its device copy of the value lists in memory it
 * allocates on demand; this entry point keeps it in a fixed array that is part of the library image instead
 * (ZMC_NOALLOC_MAX_LIST_VALUES doubles = 32 KiB on every GPU that loads the library, held until the process exits).
 * It calls no cudaMalloc, cudaFree, cudaMallocHost, stream / event creation or other allocating routine: it only
 * launches kernels on `stream` (the list values travel as kernel arguments, so `lists` is free again on return).
 *   Arguments   as zmc_scan_ex, without `timing`.  out_mean / out_stderr are DEVICE memory owned by the caller
 *               (opt->out_location must be ZMC_LOC_DEVICE; opt may be NULL).  Built-in families only (ids < 1000).
 *               opt->batch_points is ignored (batches exist to stream results to the host); ZMC_OPT_FRESH_LISTS has no
 *               effect (the lists are written into the array by every call).
 *   Results     bit-identical to zmc_scan_ex with the same arguments and schedule (tests/test_zz_no_alloc.py).
 *   Errors      those of zmc_scan_ex, detected before anything is enqueued, plus ZMC_ERR_NOALLOC_LIMIT when
 *               sum_i lists[i].count > ZMC_NOALLOC_MAX_LIST_VALUES (use zmc_scan_ex for longer lists).
 *   First call  the first call on each device looks up the array's device address (the device must be current, as
 *               for every call) and loads the kernels it launches; make that first call during start-up, before any
 *               stream capture is begun on that device.
 *   Sharing     every call on a device uses the same array and finds in it whatever the previous call left; each call
 *               overwrites the entries it reads, so nothing has to be cleared between calls.  Calls issued one after
 *               another on ONE stream are ordered by the stream.  Calls whose GPU work may overlap -- two streams, or
 *               two host threads on the same device -- race on the array and give undefined results: serialise them.
 *               (zmc_scan_ex does not use this array and may run concurrently.)
 */
ZMC_API zmc_status zmc_scan_noalloc(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                            uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, void* stream,
                            const zmc_options* opt);

/* Pure host helpers (no GPU needed). */
ZMC_API int zmc_integrand_count(void);
ZMC_API zmc_status zmc_integrand_info_at(int index, zmc_integrand_info* info);   /* index in [0, count) */
ZMC_API zmc_status zmc_integrand_info_by_id(int integrand_id, zmc_integrand_info* info);
ZMC_API const char* zmc_status_string(zmc_status s);
ZMC_API int zmc_last_cuda_error(void);          /* cudaError_t of the last ZMC_ERR_CUDA on this thread */
ZMC_API const char* zmc_version(void);
/* Validate arguments exactly as zmc_scan_ex does, enqueue nothing; writes G (whole grid) if non-NULL. */
ZMC_API zmc_status zmc_validate(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                        uint64_t n_samples, const zmc_options* opt, uint64_t* grid_points);
/* The schedule AUTO would pick for `count` points of `n_samples` samples in N dimensions (fp64 path; _ex: either
 * precision -- the fp32-evaluate kernels keep more threads resident, so their thresholds are higher).  The thresholds
 * scale with the SM count of the CURRENT device (148 if none is visible).  The schedule fixes the order of the sums,
 * hence the last bits of the results: for bit-identical results across different GPUs pass an explicit schedule. */
ZMC_API int zmc_pick_schedule(uint64_t count, uint64_t n_samples, int N);
ZMC_API int zmc_pick_schedule_ex(uint64_t count, uint64_t n_samples, int N, int precision);
/* Batch b of a range cut into batches of batch_points: writes its (first, count). Returns the number of batches. */
ZMC_API int64_t zmc_batch_range(uint64_t first_index, uint64_t count, uint64_t batch_points, int64_t b,
                        uint64_t* batch_first, uint64_t* batch_count);
/*
 * zmc_scan_adaptive -- per-point adaptive sample count (the paper asks the user to "determine the number
 * of sample points based on the desired accuracy ... increase this value" by hand).  Every grid point is sampled up to
 * the checkpoints n_first, 2 n_first, 4 n_first, ... (clipped to n_max) and stops at the first one whose standard
 * error is <= target_stderr.  Because the sample stream is keyed by (seed, global index, word index), the estimate at
 * a checkpoint uses exactly the first n samples: the outputs equal zmc_scan_ex(n_samples = out_n[point],
 * schedule = ZMC_SCHED_WARP) bit for bit.
 *   n_first   first checkpoint, a multiple of 256 (>= 256)      n_max  last checkpoint, a multiple of 8, >= n_first
 *   out_n     samples used per point (uint32, indexed like out_mean, in the SAME memory as out_mean: device, or host
 *             with opt->out_location = ZMC_LOC_HOST -- it is then streamed batch by batch with the results)
 * opt->schedule is ignored (one warp per point); batching, sub-ranges, precision, out_dtype, out_location and timing behave
 * as in zmc_scan_ex.
 */
ZMC_API zmc_status zmc_scan_adaptive(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                             uint64_t n_first, uint64_t n_max, double target_stderr, uint64_t seed, void* out_mean,
                             void* out_stderr, uint32_t* out_n, void* stream, const zmc_options* opt, zmc_timing* timing);

/*
 * zmc_scan_farm -- the same scan farmed over several GPUs of one node ("Each batch is fed into one GPU
 * device", :81, Table 2 :132-140).  The flat range is cut into batches of opt->batch_points (0 = about 8 per device);
 * one host thread per entry of `devices` pulls batches from a shared counter and scans them on its device into
 * out_mean / out_stderr, which must be HOST memory (pinned recommended; opt->out_location is ignored) of the scanned
 * range's length.  SYNCHRONOUS: returns when every batch has landed.  No inter-device traffic; results are
 * bit-identical to a one-device zmc_scan_ex with the same schedule, whichever device takes which batch.
 * A device may be listed more than once (two feeder threads on one GPU).  timing may be NULL.
 */
ZMC_API zmc_status zmc_scan_farm(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                         uint64_t n_samples, uint64_t seed, void* out_mean, void* out_stderr, const int* devices,
                         int n_devices, const zmc_options* opt, zmc_farm_timing* timing);

/* zmc_scan_farm with a per-point adaptive sample count (zmc_scan_adaptive's n_first / n_max / target_stderr); out_n is a
 * host array like out_mean.  Bit-identical to zmc_scan_adaptive on one device. */
ZMC_API zmc_status zmc_scan_farm_adaptive(int integrand_id, int N, const double* bounds, int M, const zmc_param_list* lists,
                                  uint64_t n_first, uint64_t n_max, double target_stderr, uint64_t seed, void* out_mean,
                                  void* out_stderr, uint32_t* out_n, const int* devices, int n_devices,
                                  const zmc_options* opt, zmc_farm_timing* timing);

/*
 * zmc_register_integrand -- a user-defined integrand ("users have a full flexibility to define their own
 * integrands", :49, :162; the paper JIT-compiles a Python function, here it is CUDA C++ compiled with NVRTC for
 * sm_100a into the same kernel the built-in families use).
 *   body   the body of   template <typename R> __device__ R g(const R* y, const R* x, const R* c)
 *          y: the N sample coordinates y_k = a_k + (b_k - a_k) u_k, x: the M parameter values of the grid point,
 *          c: the n_consts constants of zmc_options.consts; R is double (ZMC_PREC_F64) or float (ZMC_PREC_F32E).
 *          Example: "return exp(-x[0] * y[0] * y[0]) * cos(x[1] * y[1] + c[0]);"
 *   N, M, n_consts   the shape the integrand accepts (anything else is ZMC_ERR_SHAPE_MISMATCH at scan time)
 *   integrand_id     out: an id >= 1000 to pass to zmc_scan / zmc_scan_ex (valid until zmc_unregister_integrand / zmc_shutdown)
 * The body may call the transcendentals the built-in families use (branch-free, no table loads, no slow path), overloaded
 * for R = double and R = float:  zmc_sin(v) zmc_cos(v) [radians], zmc_sinpi(v) zmc_cospi(v) [argument in units of pi],
 * zmc_exp(v), zmc_exp2(v).  double: sin/cos to |error| <= 3e-16 (1 + |v|) (own polynomial after an exact reduction),
 * exp/exp2 = libdevice.  float: sinf/cosf/expf accuracy by default; with ZMC_USER_FAST_MATH (zmc_register_integrand_ex)
 * the MUFU forms after an exact range reduction (absolute error ~1e-6) and NVRTC --use_fast_math for the rest of the body.
 * Plain sin()/cos()/exp() work too (libdevice), at about half the speed in fp64.
 * Compiled integrands are CACHED by the hash of (body, N, M, n_consts, flags): registering the same integrand again costs
 * microseconds and returns the same id (with the first registrant's name), counted: see zmc_unregister_integrand.  Host strings are copied.  ZMC_ERR_COMPILE: libnvrtc.so.12 not found or compilation
 * failed (log below); ZMC_ERR_CUDA: compiled, but the code could not be loaded (no usable device).  zmc_options.fast_math is
 * ignored for user integrands (use ZMC_USER_FAST_MATH at registration).
 */
ZMC_API zmc_status zmc_register_integrand(const char* name, const char* body, int N, int M, int n_consts, int* integrand_id);
ZMC_API zmc_status zmc_register_integrand_ex(const char* name, const char* body, int N, int M, int n_consts, int flags,
                                     int* integrand_id);
/* Give up one registration of a user integrand.  An id handed out more than once (the same integrand registered again,
 * possibly by another part of the program) stays valid until it has been unregistered as many times as it was registered;
 * the last call forgets the id and unloads the code.  Scans already enqueued are safe: the library waits for the devices
 * that are running the integrand's kernels before unloading, and a scan call in progress on another thread keeps the code
 * loaded until it returns.  ZMC_ERR_UNKNOWN_INTEGRAND if the id is not (or no longer) registered. */
ZMC_API zmc_status zmc_unregister_integrand(int integrand_id);
ZMC_API const char* zmc_last_compile_log(void);   /* NVRTC log of the last zmc_register_integrand on this thread */
/* Free the cached per-device scratch (staging buffers, streams, events) and unload user integrands. */
ZMC_API void zmc_shutdown(void);
#endif /* !__CUDACC_RTC__ */

#ifdef __cplusplus
}
#endif
#endif /* ZMC_H_ */
