/* skel.h — C ABI of the B200-native data-parallel skeleton library.
 *
 * What it is. arxiv 1405.2915 (Kessler, Dastgeer, Li) reviews SkePU, a library of "pre-defined
 * generic software components derived from higher-order functions such as map, farm, scan and
 * reduce, which can be parameterized in problem-specific user code" (§III); its
 * data-parallel skeletons are "map, mapoverlap, scan, reduce, ..." and "all
 * non-scalar operands of SkePU skeleton calls are passed in smart containers" (§IV,
 * PAPER.md L111-L123). A *skeleton instance* is "a combination of a skeleton and parameterizing
 * user function(s)". This header is that model as a C ABI: every skeleton call takes
 * an enum-selected user function and smart_vector / smart_matrix handles. The paper prints no
 * formulas; the exact semantics are the readings of DESIGN.md.
 *
 * Conventions.
 *  - Every function returns skel_status (0 = SKEL_OK). Results come back through out-pointers.
 *  - Handles are opaque, owned by the library, released by the matching *_destroy.
 *    NULL handles -> SKEL_ERR_INVALID_ARG.
 *  - skel_last_error(ctx) returns a string owned by the context, valid until the next call on it.
 *  - A context is used from one host thread at a time.
 *  - All skeleton calls are ASYNCHRONOUS on the context's CUDA stream (containers
 *    track dependences so that calls can be asynchronous) and execute in call order. Only the
 *    forms that return a scalar to a HOST pointer (skel_reduce, skel_mapreduce) and host access
 *    to a container (*_host_acquire) block.
 *  - A CUDA failure is sticky: it is returned as SKEL_ERR_CUDA by that call or the next one.
 *  - There is no CPU fallback: every skeleton runs as hand-written CUDA for sm_100a.
 *  - "host pointer" / "device pointer" is stated for every plain-pointer argument.
 */
#ifndef SKEL_H_
#define SKEL_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SKEL_ABI_VERSION 2

/* ---- enums (values are ABI) ------------------------------------------------------------- */
typedef enum {
  SKEL_OK = 0,
  SKEL_ERR_INVALID_ARG = 1,   /* NULL handle/pointer, bad enum value, handle of another context */
  SKEL_ERR_SIZE_MISMATCH = 2, /* operand sizes/shapes differ */
  SKEL_ERR_DTYPE = 3,         /* operand element types differ, or fn not defined for the dtype */
  SKEL_ERR_UNSUPPORTED = 4,   /* radius out of range, fn not valid in this position, ... */
  SKEL_ERR_EMPTY = 5,         /* Reduce / MapReduce of n == 0 (no identity is passed) */
  SKEL_ERR_ALIAS = 6,         /* out aliases in where that is not allowed (MapOverlap) */
  SKEL_ERR_UNINIT = 7,        /* reading a container that was never written */
  SKEL_ERR_OOM = 8,
  SKEL_ERR_CUDA = 9,
  SKEL_ERR_BUSY = 10,         /* ctx destroyed with live containers; host access still held */
  SKEL_ERR_IO = 11            /* plan file could not be read / written / parsed */
} skel_status;

/* SKEL_F64: 8-byte elements; every skeleton has ONE kernel for them (no variants to select, nothing
 * to tune): Map, skel_map3, Reduce, MapReduce (blocking, _to and _async forms; the scalar is a double), Scan, MapOverlap
 * through skel_mapoverlap_*_f64. Not offered for fp64: skel_reduce_rows, skel_mapoverlap_separable, cross-call fusion
 * (such chains run call by call). Tolerances: DESIGN.md section 7. */
typedef enum { SKEL_F32 = 0, SKEL_I32 = 1, SKEL_F64 = 2 } skel_dtype;

/* user functions (BASELINE.json L5: "add, mult, max, saxpy, weighted stencil").
 * Map:      ADD a+b, MULT a*b, MAX max(a,b), SAXPY c*a+b (one fused multiply-add for f32).
 * Reduce / Scan operator, MapReduce reduce operator: ADD, MULT, MAX only.
 * WSTENCIL is the user function of MapOverlap (weights passed with the call); it is accepted
 * nowhere else. */
typedef enum {
  SKEL_FN_ADD = 0, SKEL_FN_MULT = 1, SKEL_FN_MAX = 2, SKEL_FN_SAXPY = 3, SKEL_FN_WSTENCIL = 4,
  SKEL_FN_MULADD = 5  /* three-vector Map only (skel_map3): in0 * in1 + in2 */
} skel_fn;

/* edge policy of MapOverlap: out-of-range neighbours read `pad` (CONSTANT), the nearest in-range
 * element, each index clamped independently (DUPLICATE), or wrap around, each index taken modulo
 * its extent with the non-negative remainder (CYCLIC; reading 19). */
typedef enum { SKEL_EDGE_CONSTANT = 0, SKEL_EDGE_DUPLICATE = 1, SKEL_EDGE_CYCLIC = 2 } skel_edge;
typedef enum { SKEL_SCAN_INCLUSIVE = 0, SKEL_SCAN_EXCLUSIVE = 1 } skel_scan_mode;
typedef enum { SKEL_AXIS_ROW = 0, SKEL_AXIS_COL = 1 } skel_axis;
typedef enum { SKEL_READ = 0, SKEL_WRITE = 1, SKEL_READWRITE = 2 } skel_access;
/* LAZY: the coherence protocol of PAPER.md L121-L123 (valid copies are reused, transfers happen
 * only when the accessing side has no valid copy). EAGER: the "no smart containers" baseline:
 * every skeleton call uploads each input that has a valid host copy and downloads each output. */
typedef enum { SKEL_LAZY = 0, SKEL_EAGER = 1 } skel_coherence;

/* skeleton ids (selector keys, skel_force_variant, skel_last_variant) */
typedef enum {
  SKEL_SK_MAP = 0, SKEL_SK_REDUCE = 1, SKEL_SK_MAPREDUCE = 2, SKEL_SK_SCAN = 3,
  SKEL_SK_OVERLAP1D = 4,      /* vector, and row-wise on a matrix */
  SKEL_SK_OVERLAP1D_COL = 5,  /* column-wise on a matrix */
  SKEL_SK_OVERLAP2D = 6,
  SKEL_SK_SEPARABLE = 7,      /* skel_mapoverlap_separable (variant 0 = the two 1D passes) */
  SKEL_SK_REDUCE_ROWS = 8,    /* skel_reduce_rows */
  SKEL_SK_COUNT = 9
} skel_skeleton;

typedef struct skel_ctx skel_ctx;
typedef struct skel_vector skel_vector;
typedef struct skel_matrix skel_matrix;
typedef struct skel_future skel_future; /* the scalar result of a skel_*_async call (below) */

/* ---- context ---------------------------------------------------------------------------- */
/* Device-memory callbacks (e.g. PyTorch's caching allocator). alloc returns a device pointer
 * (NULL on failure) usable on `stream`; free releases it. Both NULL -> cudaMalloc / cudaFree. */
typedef void* (*skel_alloc_fn)(size_t bytes, void* stream, void* user);
typedef void (*skel_free_fn)(void* dptr, void* user);

/* cuda_stream: a cudaStream_t (NULL = the legacy default stream) owned by the caller; all device
 * work of the context is enqueued on it. The library owns plans, scratch and statistics. */
skel_status skel_ctx_create(void* cuda_stream, skel_alloc_fn alloc, skel_free_fn free_, void* user, skel_ctx** out);
/* Synchronises the stream and frees scratch. Live containers -> SKEL_ERR_BUSY (nothing freed). */
skel_status skel_ctx_destroy(skel_ctx* ctx);
skel_status skel_ctx_sync(skel_ctx* ctx);
skel_status skel_ctx_set_coherence(skel_ctx* ctx, skel_coherence mode);
/* Cross-call fusion (the GPU-only analogue of PAPER.md L137/L149: compose over a
 * chain of dependent calls instead of call by call). Off by default. When enabled, the kernel launch
 * of a call that can be part of the chain
 *     skel_map(f in {ADD, MULT, MAX}, constant c, in1 = NULL, f32)  ->  skel_mapoverlap_1d (r in
 *     {1,2,3,4,8,16}) on the Map's output  ->  skel_reduce / skel_reduce_to (ADD or MAX) on the
 *     MapOverlap's output
 * is held back (argument checks, coherence bookkeeping and transfers still happen inside the call).
 * When the Reduce arrives the chain runs as ONE kernel that reads the input once (12 B/elem instead
 * of 20); a Map -> MapOverlap1D or MapOverlap1D -> Reduce pair fuses the same way. Anything else
 * (another call, a host access, a transfer, skel_ctx_sync, skel_ctx_flush, a destroy, a forced
 * variant) first launches what is held back, call by call, so results never depend on the setting
 * beyond the rounding differences between kernel variants (same tolerances). Consequences while
 * fusion is on: (1) a launch error of a held-back call is reported by the call that flushes it;
 * (2) callers that enqueue their own work on the context's stream (events, kernels) must call
 * skel_ctx_flush first; (3) a fused IN-PLACE Map writes into a library buffer that is then swapped
 * with the container's device buffer: a pointer obtained from skel_vector_device_ptr is valid only
 * until the next skeleton call that writes the container (adopted buffers are never swapped; such a
 * chain runs call by call); (4) skel_last_variant reports variant -2 for a fused launch. */
skel_status skel_ctx_set_fusion(skel_ctx* ctx, int enable);
/* L2-aware traversal (default: on). A skeleton kernel streams its operands front to back, so when it ends the L2
 * (126 MB on B200) holds the TAIL of what it read. With the setting on, a Reduce / MapReduce whose first operand is the
 * buffer the context's previous launch also read walks that buffer in the OPPOSITE direction, so that its first chunks
 * hit L2 instead of HBM (chained calls on one smart container, P:L123 / L137: the container layer knows what the last
 * call touched). The result has the same bits in either direction (a block's partial belongs to its chunk, the fold
 * order is by chunk). Off: every kernel walks forward. */
skel_status skel_ctx_set_l2_reuse(skel_ctx* ctx, int enable);
/* Launch everything that fusion holds back (no synchronisation). */
skel_status skel_ctx_flush(skel_ctx* ctx);
const char* skel_last_error(skel_ctx* ctx);
int skel_abi_version(void);

/* ---- smart containers ------------------------------------------ */
/* A container owns a pinned host buffer (allocated on first host use) and a device buffer
 * (allocated on first device use) and tracks which of the two copies is valid.
 *   create:       contents undefined, state UNINIT.
 *   create_from:  copies n elements from caller HOST memory `src` at call time; state HOST.
 *   adopt_device: wraps a caller-owned DEVICE buffer of n elements as the device copy; state
 *                 DEVICE. The caller keeps it alive and does not touch it while calls are in
 *                 flight; the library never frees it.
 * n == 0 is legal. */
skel_status skel_vector_create(skel_ctx* ctx, skel_dtype dt, size_t n, skel_vector** out);
skel_status skel_vector_create_from(skel_ctx* ctx, skel_dtype dt, size_t n, const void* src, skel_vector** out);
skel_status skel_vector_adopt_device(skel_ctx* ctx, skel_dtype dt, size_t n, void* dptr, skel_vector** out);
skel_status skel_vector_destroy(skel_vector* v);
skel_status skel_vector_size(const skel_vector* v, size_t* n);
/* Host access (replaces SkePU's operator-overloaded element access). Blocks until
 * the device work that the access depends on has finished; READ / READWRITE download the data
 * if only the device copy is valid. *host_ptr (HOST memory, n elements, library-owned pinned
 * buffer) stays valid until host_release. WRITE means the caller overwrites ALL elements.
 * Skeleton calls on a container whose host access is held -> SKEL_ERR_BUSY. */
skel_status skel_vector_host_acquire(skel_vector* v, skel_access mode, void** host_ptr);
skel_status skel_vector_host_release(skel_vector* v);
/* Start downloading the container to its host copy NOW, asynchronously, on a copy stream of the context, if only
 * the device copy is valid (otherwise nothing happens). The download is ordered after everything enqueued so far and
 * overlaps later skeleton calls and their uploads (PCIe is full duplex); a later host access waits for it instead of
 * starting its own copy, a later device write to the container waits for it before it overwrites the buffer.
 * The communication-optimisation service of PAPER.md L117, made explicit: the lazy protocol alone would start the
 * download only at the host access. */
skel_status skel_vector_prefetch_host(skel_vector* v);
/* Range-granular host access (single-GPU half; partial copies, "multiple data
 * transfers ... when accessing a given range of elements"). *host_ptr points at element `offset` of the library's
 * pinned host copy and is valid for `count` elements until skel_vector_host_release.
 *   READ:      if the host copy is not valid only this range is downloaded; the container's state does not change
 *              (a later whole-container host access still downloads everything).
 *   WRITE / READWRITE: the range becomes newer on the host than on the device. If the device copy is valid it STAYS
 *              valid: the next skeleton call that reads the container uploads just the written ranges (ranges merge;
 *              a whole-container device write discards them), instead of the whole container as after
 *              skel_vector_host_acquire(WRITE).
 * The container must have been written before (UNINIT -> SKEL_ERR_UNINIT); offset + count <= n; count > 0. */
skel_status skel_vector_host_acquire_range(skel_vector* v, skel_access mode, size_t offset, size_t count, void** host_ptr);
/* Device pointer of the current device copy for inspection/interop (NULL if none); *valid = 1
 * if the device copy is valid. No transfer, no state change. */
skel_status skel_vector_device_ptr(const skel_vector* v, void** dptr, int* valid);
/* 0 UNINIT, 1 HOST, 2 DEVICE, 3 SHARED (bit 0 = host valid, bit 1 = device valid) */
skel_status skel_vector_state(const skel_vector* v, int* state);

/* matrices: row-major rows x cols, contiguous (pitch = cols) */
skel_status skel_matrix_create(skel_ctx* ctx, skel_dtype dt, size_t rows, size_t cols, skel_matrix** out);
skel_status skel_matrix_create_from(skel_ctx* ctx, skel_dtype dt, size_t rows, size_t cols, const void* src, skel_matrix** out);
skel_status skel_matrix_adopt_device(skel_ctx* ctx, skel_dtype dt, size_t rows, size_t cols, void* dptr, skel_matrix** out);
skel_status skel_matrix_destroy(skel_matrix* m);
skel_status skel_matrix_shape(const skel_matrix* m, size_t* rows, size_t* cols);
skel_status skel_matrix_host_acquire(skel_matrix* m, skel_access mode, void** host_ptr);
skel_status skel_matrix_host_release(skel_matrix* m);
skel_status skel_matrix_prefetch_host(skel_matrix* m);
/* the same for whole rows row0 .. row0 + nrows - 1 of a matrix */
skel_status skel_matrix_host_acquire_rows(skel_matrix* m, skel_access mode, size_t row0, size_t nrows, void** host_ptr);
/* A flattened alias (rows*cols elements) sharing storage and coherence state with the matrix;
 * destroy it like any vector (the storage lives until the last handle is destroyed). */
skel_status skel_matrix_as_vector(skel_matrix* m, skel_vector** view);

/* ---- skeletons ---------------------------------------------------------------------------- */
/* `c` is the scalar constant of the user function, converted to the element type on entry
 * (round-to-nearest to f32; for i32 it must be an integer in int32 range, else INVALID_ARG). */

/* Map: out[i] = f(in0[i], b_i), b_i = in1[i], or the constant c when in1 == NULL.
 * SAXPY: out[i] = c*in0[i] + in1[i] (in1 required). out may alias in0 and/or in1 (in place). */
skel_status skel_map(skel_ctx* ctx, skel_fn f, double c, const skel_vector* in0, const skel_vector* in1, skel_vector* out);
/* Three-vector Map. f must be SKEL_FN_MULADD: out[i] = in0[i] * in1[i] + in2[i] (f32: one fused
 * multiply-add, <= 1 ulp of the fp64 value rounded to f32; i32 wraps modulo 2^32). out may alias any input. */
skel_status skel_map3(skel_ctx* ctx, skel_fn f, const skel_vector* in0, const skel_vector* in1, const skel_vector* in2,
                      skel_vector* out);

/* Reduce: in[0] (+) ... (+) in[n-1], (+) in {ADD, MULT, MAX}; i32 ADD/MULT wrap mod 2^32.
 * skel_reduce writes one element of the element type to HOST memory `host_result` and blocks.
 * skel_reduce_to writes it to out[out_index] on the device and does not block. */
skel_status skel_reduce(skel_ctx* ctx, skel_fn op, const skel_vector* in, void* host_result);
skel_status skel_reduce_to(skel_ctx* ctx, skel_fn op, const skel_vector* in, skel_vector* out, size_t out_index);

/* MapReduce: (+)_i map_f(in0[i], b_i), fused: the mapped vector is never materialised. */
skel_status skel_mapreduce(skel_ctx* ctx, skel_fn map_f, skel_fn red_op, double c, const skel_vector* in0,
                           const skel_vector* in1, void* host_result);
skel_status skel_mapreduce_to(skel_ctx* ctx, skel_fn map_f, skel_fn red_op, double c, const skel_vector* in0,
                              const skel_vector* in1, skel_vector* out, size_t out_index);

/* Asynchronous forms ("asynchronous skeleton calls ... allow the runtime to run ahead", L116 "data
 * dependence tracking"): the call returns at once with a future; the scalar lands in a pinned host slot the kernel
 * writes directly (zero-copy). skel_future_wait blocks until THAT reduction has finished - an event recorded right
 * after its kernel, not the whole stream - and copies one element of the element type to HOST memory `host_result`;
 * it may be called more than once. skel_future_ready polls (*ready = 1 when the result is there). A loop that calls
 * Map -> MapOverlap -> skel_reduce_async and waits for the futures afterwards (or a few iterations late) keeps
 * several iterations in flight. Futures belong to the context, must be destroyed before it (SKEL_ERR_BUSY otherwise),
 * and at most 1024 may be outstanding per context (SKEL_ERR_BUSY). Same checks and results as the blocking forms. */
skel_status skel_reduce_async(skel_ctx* ctx, skel_fn op, const skel_vector* in, skel_future** out);
skel_status skel_mapreduce_async(skel_ctx* ctx, skel_fn map_f, skel_fn red_op, double c, const skel_vector* in0,
                                 const skel_vector* in1, skel_future** out);
skel_status skel_future_wait(skel_future* f, void* host_result);
skel_status skel_future_ready(skel_future* f, int* ready);
skel_status skel_future_destroy(skel_future* f);

/* Row-wise Reduce on a matrix: out[i] = in[i][0] (+) ... (+) in[i][cols-1] for every row i.
 * `out` has `rows` elements of the matrix's element type (f32 or i32; i32 add / mult wrap modulo 2^32);
 * (+) in {ADD, MULT, MAX}. cols == 0 with rows > 0 -> SKEL_ERR_EMPTY. f32: each row within the Reduce tolerance,
 * deterministic for a given shape and variant. */
skel_status skel_reduce_rows(skel_ctx* ctx, skel_fn op, const skel_matrix* in, skel_vector* out);

/* MapOverlap 1D (f32 only): out[i] = sum_{k=-r..r} w[k+r] * x~[i+k] (correlation: w[0]
 * multiplies the left-most neighbour). w: HOST pointer to 2r+1 floats, copied at call time.
 * 0 <= r <= SKEL_MAX_RADIUS_1D. out must not alias in. `pad` is used by SKEL_EDGE_CONSTANT. */
#define SKEL_MAX_RADIUS_1D 64
#define SKEL_MAX_RADIUS_2D 8
skel_status skel_mapoverlap_1d(skel_ctx* ctx, const float* w, int r, skel_edge edge, double pad,
                               const skel_vector* in, skel_vector* out);
/* the same along every row (SKEL_AXIS_ROW) or every column (SKEL_AXIS_COL) of a matrix */
skel_status skel_mapoverlap_1d_matrix(skel_ctx* ctx, const float* w, int r, skel_edge edge, double pad,
                                      skel_axis axis, const skel_matrix* in, skel_matrix* out);
/* MapOverlap 2D (f32 only): out[i][j] = sum_a sum_b W[a+ry][b+rx] * X~[i+a][j+b].
 * W: HOST pointer, (2ry+1)*(2rx+1) floats row-major. 0 <= ry, rx <= SKEL_MAX_RADIUS_2D. */
skel_status skel_mapoverlap_2d(skel_ctx* ctx, const float* W, int ry, int rx, skel_edge edge, double pad,
                               const skel_matrix* in, skel_matrix* out);

/* MapOverlap on int32 containers (the skeletons are generic in the element type, PAPER.md L75, L81;
 * DESIGN.md reading 26): the same three calls with int32 data, int32 weights (HOST pointer, copied at call time)
 * and an int32 pad value. Every product and every sum wraps modulo 2^32 (like the int32 Map / Reduce / Scan), so the
 * result does not depend on the summation order and is bit-exact against the definition. Same radii, edge policies,
 * aliasing and shape rules; f32 containers -> SKEL_ERR_DTYPE (and int32 containers in the f32 calls likewise).
 * Kernels: the direct, register-window and TMA-fed variants with an integer multiply-add. */
skel_status skel_mapoverlap_1d_i32(skel_ctx* ctx, const int32_t* w, int r, skel_edge edge, int32_t pad,
                                   const skel_vector* in, skel_vector* out);
skel_status skel_mapoverlap_1d_matrix_i32(skel_ctx* ctx, const int32_t* w, int r, skel_edge edge, int32_t pad,
                                          skel_axis axis, const skel_matrix* in, skel_matrix* out);
skel_status skel_mapoverlap_2d_i32(skel_ctx* ctx, const int32_t* W, int ry, int rx, skel_edge edge, int32_t pad,
                                   const skel_matrix* in, skel_matrix* out);

/* MapOverlap on fp64 containers (SKEL_F64): fp64 data, fp64 weights (HOST pointer, copied at call time), fp64 pad.
 * One fused multiply-add (DFMA) per tap in ascending tap order, chains of at most 33 taps (2D: one chain per filter
 * row, the row sums added): |error| <= 33 * 2^-53 * sum|w x~| against the exact value. One kernel each (direct form). */
skel_status skel_mapoverlap_1d_f64(skel_ctx* ctx, const double* w, int r, skel_edge edge, double pad, const skel_vector* in,
                                   skel_vector* out);
skel_status skel_mapoverlap_1d_matrix_f64(skel_ctx* ctx, const double* w, int r, skel_edge edge, double pad, skel_axis axis,
                                          const skel_matrix* in, skel_matrix* out);
skel_status skel_mapoverlap_2d_f64(skel_ctx* ctx, const double* W, int ry, int rx, skel_edge edge, double pad,
                                   const skel_matrix* in, skel_matrix* out);
/* Separable MapOverlap (BASELINE.json configs[3] "separable row-then-column 1D
 * passes"): out = colpass(w_col, r_col, T), T = RN_f32(rowpass(w_row, r_row, in)), each pass with the
 * edge policy, i.e. by definition the result of skel_mapoverlap_1d_matrix(ROW) into a temporary
 * matrix followed by skel_mapoverlap_1d_matrix(COL). When r_row == r_col is one of {1,2,3,4,8} the
 * two passes run as ONE kernel that keeps T in shared memory (8 instead of 16 bytes per element of
 * HBM traffic); otherwise (variant 0, "two_pass") the library runs the two 1D kernels through a
 * temporary device matrix of its own. w_row, w_col: HOST pointers (2r+1 floats each).
 * out must not alias in. */
skel_status skel_mapoverlap_separable(skel_ctx* ctx, const float* w_row, int r_row, const float* w_col, int r_col,
                                      skel_edge edge, double pad, const skel_matrix* in, skel_matrix* out);

/* Scan: inclusive out[i] = x[0] (+)...(+) x[i]; exclusive out[0] = init, out[i] = init (+) x[0]
 * (+)...(+) x[i-1]. (+) in {ADD, MULT, MAX}. `init` is ignored for inclusive. out may alias in. */
skel_status skel_scan(skel_ctx* ctx, skel_fn op, skel_scan_mode mode, double init, const skel_vector* in, skel_vector* out);

/* ---- variant selector ("execution plan"; L53 off-line tuned dispatch) --------- */
/* A skeleton instance: the key an execution plan is attached to. Unused fields are 0. */
typedef struct {
  int32_t skeleton; /* skel_skeleton */
  int32_t fn;       /* Map/MapReduce: map function; Reduce/Scan: operator; MapOverlap: WSTENCIL */
  int32_t fn2;      /* MapReduce: reduce operator */
  int32_t dtype;    /* skel_dtype */
  int32_t r0;       /* MapOverlap 1D: r; 2D: ry */
  int32_t r1;       /* 2D: rx */
  int32_t edge;     /* skel_edge */
  int32_t mode;     /* Scan: skel_scan_mode; Map/MapReduce: 1 if in1 is a vector, 0 if it is the constant;
                       MapOverlap 1D (row-wise): shape class, 0 = vector, 1 = rows of a matrix */
} skel_instance;

/* Number of kernel variants of a skeleton and the name of one (static string). */
int skel_variant_count(int skeleton);
const char* skel_variant_name(int skeleton, int variant);
/* The plan is a dispatch TREE over the call context ("tree-based dispatch structure for fast runtime
 * lookup"): skeleton -> dtype -> (fn, fn2) -> mode / shape class -> r0 -> r1 -> edge -> size breakpoints. A call whose
 * own context was never tuned takes, level by level, the nearest tuned child (radii: nearest in log2(r + 1), ties to
 * the larger one; categorical levels: the first child); skeleton and dtype must match. So r = 5 runs what was tuned
 * for r = 4, r = 12 what was tuned for r = 16, and only a (skeleton, dtype) without any tuned point falls back to
 * the built-in preference list. The variant found is used if it is applicable to the call (alignment, shape).
 *
 * skel_tune_instance: measure every applicable variant of `inst` at n = 2^k, k = log2_lo..log2_hi (vectors), mean of
 * the middle half of `reps` launches (event timestamps tick in about 2 us steps: a median would be quantised), variants interleaved, timed with CUDA events on the context stream UNDER THE CONDITIONS OF A
 * SUSTAINED RUN: operands rotate through arenas larger than the L2 cache (so no launch finds its input there) and
 * every timed launch is preceded by a writer that leaves the L2 full of dirty lines, as the previous skeleton call
 * of a real sequence does. Size breakpoints are stored in the context's plan. Where the winner changes between two sampled sizes the interval is
 * bisected (only the two contenders are timed) until it is narrower than 2^(1/4), so breakpoints
 * are not confined to powers of two (adaptive sampling). For matrix skeletons `cols`
 * gives the row length (rows = n/cols); pass 0 for vectors. Blocks. */
skel_status skel_tune_instance(skel_ctx* ctx, const skel_instance* inst, int log2_lo, int log2_hi, size_t cols, int reps);
skel_status skel_plan_save(skel_ctx* ctx, const char* path);
skel_status skel_plan_load(skel_ctx* ctx, const char* path);
skel_status skel_plan_clear(skel_ctx* ctx);
/* Pure host lookup (no GPU needed): which variant would the plan run for `inst` at n elements?
 * Alignment- or radius-driven fallbacks are applied at launch time and reported by
 * skel_last_variant. */
skel_status skel_plan_lookup(skel_ctx* ctx, const skel_instance* inst, size_t n, int* variant);
/* The same, and how it was found: *exact = 1 if the instance's own key has a tuned entry, 0 if the variant was
 * inherited from the nearest tuned neighbour in the dispatch tree or comes from the preference list
 * (*variant_from_plan = 0 in the latter case). Pure host code. */
skel_status skel_plan_explain(skel_ctx* ctx, const skel_instance* inst, size_t n, int* variant, int* exact,
                              int* variant_from_plan);
/* Insert one breakpoint by hand: variant `variant` from n >= n_min (until the next breakpoint). */
skel_status skel_plan_set(skel_ctx* ctx, const skel_instance* inst, size_t n_min, int variant);
/* Measurement hook for the overhead of the container layer (the smart containers' overhead is
 * "negligible (less than 1 %)"; time through skel_* on containers / time of the same kernel
 * launches on raw pointers - 1). skel_replay_begin starts recording the skeleton calls made on the context
 * (fusion must be off), skel_replay_end stops (*ncalls = calls recorded). skel_replay_run then runs the recorded
 * sequence `reps` times, timed inside the library (host: clock around the enqueue loop; device: CUDA events on the
 * context's stream), either
 *   raw = 0: through the container layer - operand acquisition (coherence look-up, transfers if a copy is stale),
 *            execution-plan look-up, launch, publish, event record - i.e. what the public calls do after argument
 *            validation, or
 *   raw = 1: as bare kernel launches on the recorded device pointers with the recorded variants.
 * The containers of the recorded calls must still be alive. Blocks until the sequence has finished. */
skel_status skel_replay_begin(skel_ctx* ctx);
skel_status skel_replay_end(skel_ctx* ctx, int* ncalls);
skel_status skel_replay_run(skel_ctx* ctx, int raw, int reps, double* host_us_per_pass, double* device_us_per_pass);

/* Timing table of the last skel_tune_instance: times_us[(k-log2_lo)*nvariants + v], NaN where a
 * variant is not applicable. Copies at most `capacity` floats; *count = number available. */
skel_status skel_tune_table(skel_ctx* ctx, float* times_us, size_t capacity, size_t* count);
/* Force a variant for a skeleton (variant -1 = back to the plan). A forced variant that is not
 * applicable to a call (dtype, radius, alignment) makes the call fail with UNSUPPORTED. */
skel_status skel_force_variant(skel_ctx* ctx, int skeleton, int variant);
skel_status skel_last_variant(skel_ctx* ctx, int* skeleton, int* variant);

/* ---- observability -------------------------------------------------------------------------- */
typedef struct {
  uint64_t h2d_bytes, h2d_count;     /* container uploads */
  uint64_t d2h_bytes, d2h_count;     /* container downloads */
  uint64_t h2d_elided;               /* device reads served by an already valid device copy */
  uint64_t d2h_elided;               /* outputs left on the device (EAGER would download them) */
  uint64_t scalar_d2h_count;         /* Reduce / MapReduce scalars returned to the host */
  uint64_t launches;                 /* kernels launched by the library */
  uint64_t fused_launches;           /* fused-chain kernels (skel_ctx_set_fusion) */
  uint64_t fused_calls;              /* skeleton calls that ran inside a fused-chain kernel */
} skel_stats;
skel_status skel_get_stats(skel_ctx* ctx, skel_stats* out);
/* Measures the FP32 fused-multiply-add throughput of the device with a register-only FFMA kernel
 * (median of `reps` launches, CUDA events on the context's stream; synchronises): *fma_per_s = FMAs per
 * second (x 2 = FLOP/s). The roofline of the arithmetic-bound MapOverlap instances. */
skel_status skel_probe_fma_peak(skel_ctx* ctx, int reps, double* fma_per_s);
/* The same for a stream of packed FFMA2 (72 per iteration = 144 FMA-pipe cycles per warp) interleaved with
 * `lds128_per_iter` in {0, 1, 2, 4, 8} 128-bit shared-memory loads per iteration, three resident blocks per SM:
 * measures what a load returning into the register file costs the FMA pipe (the ceiling of the arithmetic-bound
 * dense 9x9 MapOverlap). Any other count -> SKEL_ERR_INVALID_ARG. */
skel_status skel_probe_fma_with_loads(skel_ctx* ctx, int lds128_per_iter, int reps, double* fma_per_s);
skel_status skel_reset_stats(skel_ctx* ctx);

/* ---- no-allocation entry point ----------------------------------------------------------------
 * Reduce (PAPER.md L81 skeleton list; reading 2) for callers that may not allocate: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc. Needs no context. The scratch of the reduction
 * (one partial per block + the ticket) lives in a file-scope __device__ array of skel_noalloc_scratch_bytes() = 33 024
 * bytes, which every GPU that loads the library holds until the process exits; the call itself calls no cudaMalloc,
 * cudaFree or allocating library routine.
 *   op             SKEL_FN_ADD, SKEL_FN_MULT or SKEL_FN_MAX (anything else -> SKEL_ERR_INVALID_ARG)
 *   device_in      DEVICE pointer, n floats, owned by the caller, read only (any 4-byte alignment)
 *   n              1 .. skel_noalloc_max_elements() = 2^26; 0 -> SKEL_ERR_EMPTY; more -> SKEL_ERR_UNSUPPORTED
 *   device_result  DEVICE pointer to one float, owned by the caller, written by the kernel
 *   cuda_stream    a cudaStream_t (NULL = the legacy default stream); the call is asynchronous on it
 * The device of the call is the CURRENT device. Same arithmetic as skel_reduce (f32 accumulators, fixed order,
 * deterministic for a given n), within the Reduce tolerance of DESIGN.md section 7; not bitwise equal to skel_reduce,
 * whose order depends on the tuned variant. Every call shares the one array: calls on one stream are ordered and
 * safe, calls that overlap on the GPU (two streams, two host threads) RACE on it. skel_noalloc_last_error() returns
 * the calling thread's message of its last failed no-alloc call (static storage). */
skel_status skel_reduce_f32_noalloc(skel_fn op, const float* device_in, size_t n, float* device_result, void* cuda_stream);
size_t skel_noalloc_max_elements(void);
size_t skel_noalloc_scratch_bytes(void);
const char* skel_noalloc_last_error(void);

/* The range list of the range-granular host access as a pure function (no GPU needed): merges [begin, end) into
 * the sorted list of `*count` disjoint ranges stored as pairs ranges[2k], ranges[2k+1] (capacity in pairs). */
skel_status skel_ranges_add(uint64_t* ranges, size_t* count, size_t capacity, uint64_t begin, uint64_t end);

/* The coherence protocol as a pure function (used by the library itself
 * and exposed so that it can be tested without a GPU).
 * state: bit 0 host valid, bit 1 device valid. actor: 0 = device (skeleton operand), 1 = host.
 * mode: LAZY or EAGER. Outputs: *new_state (once the access / the kernel is done); *transfer: bit
 * mask, 1 = H2D before the kernel, 2 = D2H (host actor: before the access; device actor, EAGER
 * only: after the kernel). Returns SKEL_ERR_UNINIT when the access would read a container with no
 * valid copy. */
skel_status skel_coherence_step(int state, int actor, skel_access access, skel_coherence mode, int* new_state, int* transfer);

#ifdef __cplusplus
}
#endif
#endif /* SKEL_H_ */
