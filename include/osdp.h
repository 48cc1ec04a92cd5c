/* osdp.h — C ABI of osdp-b200: operator-split transformer MLP for one NVIDIA B200 (sm_100a).
 *
 * Method: OSDP (arxiv 2305.09940).  Operator splitting (§3.3): a huge operator is
 * partitioned into slices that are "executed sequentially", their memory "released serially", and "all
 * computation results are summed as the final output".  This library applies it to the transformer MLP
 * operator  Y = gelu(X W1 + b1) W2 + b2  over k TOKEN slices (reading S1), forward and backward,
 * so that the tokens x ffn intermediate never exists whole, and evaluates the paper's per-operator cost
 * model (Eq. 1) to choose k per operator under a memory limit (Algorithm 1).
 *
 * Conventions (all calls)
 *   - Tensors are dense row-major, no padding.  X, Y, dY, dX: [tokens x hidden]; W1: [hidden x ffn];
 *     W2: [ffn x hidden]; b1: [ffn]; b2: [hidden].  Weights are [in x out].
 *   - dtype = storage type of X, W1, b1, W2, b2, dY, Y, dX and of the workspace tensors.  Products
 *     accumulate in fp32.  dW1, dW2, db1, db2 are ALWAYS fp32.
 *   - "device pointer" = CUDA device memory of the current device, owned by the caller, 16-byte aligned
 *     (workspace: 256-byte aligned).  The library never allocates, frees or synchronises device memory; it
 *     only enqueues work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream).  Its own
 *     device state is static module memory: 256 wave-sync counters per device (a scheduling hint with a 200 us give-up,
 *     never a correctness dependency) and the scratch of osdp_bias_grad_static.  The tile counter and flags of the
 *     one-kernel-per-slice path live in the caller's workspace (counted by the *_workspace_bytes queries), so a workspace
 *     must be exclusive to ONE call in flight: calls that may overlap on the GPU - other streams, or captured graphs
 *     replayed side by side - each need their own.  Any number of such calls may be in flight.
 *     Outputs must not alias inputs or each other.
 *   - Every call returns an osdp_status; OSDP_OK = 0.  Nothing is printed, nothing aborts.  On any error
 *     before the first launch the outputs are untouched.
 *   - Re-entrant for distinct streams/workspaces, from any number of host threads, on any device with ordinal < 64:
 *     launch state (SM count, shared-memory opt-in, resident cluster count, wave-sync counters) is kept per device
 *     ordinal; the device used is the one current to the calling thread, which must own every pointer passed.  Only
 *     the osdp_set_tuning knobs are process-wide.  After one warm-up call per (dtype, tile shape, device) the calls
 *     are CUDA-graph capturable (they only enqueue kernels on `stream`).
 */
#ifndef OSDP_H_
#define OSDP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)
#endif

typedef enum osdp_status {
  OSDP_OK = 0,
  OSDP_ERR_NULL = 1,        /* a required pointer is NULL */
  OSDP_ERR_SHAPE = 2,       /* tokens/hidden/ffn < 1, or hidden/ffn not a multiple of 16 bytes / sizeof(dtype) */
  OSDP_ERR_K = 3,           /* k < 1 or k > tokens */
  OSDP_ERR_DTYPE = 4,       /* dtype is not OSDP_F32 / OSDP_BF16 */
  OSDP_ERR_WORKSPACE = 5,   /* workspace smaller than osdp_split_mlp_workspace_bytes, or not 256 B aligned */
  OSDP_ERR_ALIGN = 6,       /* a tensor pointer is not 16 B aligned */
  OSDP_ERR_ARCH = 7,        /* current device is not compute capability 10.x (bf16 path needs tcgen05/TMA) */
  OSDP_ERR_CUDA = 8,        /* CUDA runtime/driver error; see osdp_last_cuda_error() */
  OSDP_ERR_INFEASIBLE = 9,  /* planner: no plan fits the memory limit (Algorithm 1 lines 12-14) */
  OSDP_ERR_ARG = 10,        /* other invalid argument (pass, mode, n, candidate list, ...) */
  OSDP_ERR_SEARCH_LIMIT = 11, /* planner: node budget exhausted before the search completed */
  OSDP_ERR_STATIC_LIMIT = 12, /* osdp_bias_grad_static: cols > OSDP_BIAS_GRAD_STATIC_MAX_COLS (the static scratch is too small) */
  OSDP_ERR_COMM = 13          /* osdp_zdp_*: a caller-supplied collective returned non-zero.  Work enqueued before it stays
                                 enqueued, comm_stream is joined back into compute_stream, the outputs are UNDEFINED */
} osdp_status;

typedef enum osdp_dtype { OSDP_F32 = 0, OSDP_BF16 = 1 } osdp_dtype;
typedef enum osdp_pass { OSDP_FWD = 0, OSDP_BWD = 1 } osdp_pass;
typedef enum osdp_mode { OSDP_DP = 0, OSDP_ZDP = 1 } osdp_mode;

/* One MLP operator and its split count.  k = number of token slices ("slice granularity", PAPER.md:165;
 * the paper's granularity 0 = "no splitting" is k = 1 here).  Slice s covers rows
 * [floor(s*tokens/k), floor((s+1)*tokens/k))  (reading S7: ragged slices allowed). */
typedef struct osdp_mlp_desc {
  int64_t tokens;   /* T >= 1 */
  int64_t hidden;   /* h; multiple of 8 (bf16) / 4 (f32) */
  int64_t ffn;      /* f; multiple of 8 (bf16) / 4 (f32) */
  int32_t dtype;    /* osdp_dtype */
  int32_t k;        /* 1 <= k <= tokens */
} osdp_mlp_desc;

const char* osdp_status_string(int status);   /* static string, never NULL */
const char* osdp_last_cuda_error(void);       /* text of the last CUDA error seen by the calling thread ("" if none) */
const char* osdp_version(void);

/* ---- A10: workspace accounting (PAPER.md:84-86 M_extra; PAPER.md:167 size/slice_granularity) ----------
 * Bytes of caller workspace one forward (OSDP_FWD) or backward (OSDP_BWD) call needs.  Pure host function.
 *   FWD: one [T_s x f] tensor (H_s);  BWD: two (Z_s, overwritten by dZ_s; H_s) + the fp32 column-sum partials:
 *   ceil(T_s / 32) x ffn floats (one row per 32-row band of dZ_s, written by the A4 epilogue: db1) and 32 x hidden
 *   floats (db2); both passes, bf16: + the tile counter and flag words of the one-kernel-per-slice path,
 *   4 k (4 + 2 t) bytes, t = the 256 x 256 tiles of a [T_s x ffn] tensor, when that is <= 128 KiB, else none;
 *   T_s = ceil(T/k); each part rounded up to 256 B.  Returns 0 on an invalid descriptor. */
size_t osdp_split_mlp_workspace_bytes(const osdp_mlp_desc* desc, int pass);

/* ---- A0-A2: forward (DESIGN.md steps A1, A2) ---------------------------------------------
 * for s in 0..k-1 (in order):  H_s = gelu(X_s W1 + b1)  (workspace, storage dtype; Z never stored)
 *                               Y_s = H_s W2 + b2        (rows of Y, storage dtype)
 * gelu = tanh approximation (reading S2).  All tensor arguments are device pointers; Y [T x h] is overwritten. */
int osdp_split_mlp_forward(const osdp_mlp_desc* desc,
                           const void* X, const void* W1, const void* b1, const void* W2, const void* b2,
                           void* Y, void* workspace, size_t workspace_bytes, void* stream);

/* ---- A0, A3-A8: backward (DESIGN.md steps A3-A8) -------------------------------------------------------
 * Takes no saved activations.  for s in 0..k-1 (in order):
 *   Z_s = X_s W1 + b1, H_s = gelu(Z_s)                       (recomputed, workspace)
 *   dZ_s = (dY_s W2^T) (.) gelu'(Z_s)                        (overwrites Z_s)
 *   dW2 (+)= H_s^T dY_s;  dW1 (+)= X_s^T dZ_s                (fp32; "=" on slice 0, "+=" after: "summed")
 *   db1 (+)= colsum(dZ_s)                                    (fp32; 32-row band sums from the dZ_s epilogue, then a
 *                                                             fixed-order sum over bands)
 *   db2 = colsum(dY)                                         (fp32, fixed reduction order, once per call: dY is whole)
 *   dX_s = dZ_s W1^T                                         (rows of dX, storage dtype)
 * dX [T x h] storage dtype; dW1 [h x f], db1 [f], dW2 [f x h], db2 [h] fp32; all OVERWRITTEN (reading S11).
 * b2 is unused and may be NULL (reading S4). */
int osdp_split_mlp_backward(const osdp_mlp_desc* desc,
                            const void* X, const void* W1, const void* b1, const void* W2, const void* b2,
                            const void* dY,
                            void* dX, float* dW1, float* db1, float* dW2, float* db2,
                            void* workspace, size_t workspace_bytes, void* stream);

/* ---- ffn-axis split: the paper-literal operator splitting applied to the MLP pair -------------------------
 * PAPER.md:165 (section 3.3): "both the last dimension of the input data and the first dimension of the operator
 * are partitioned into multiple slices ... the computation of each slice is executed sequentially ... all
 * computation results are summed as the final output".  For Linear2 (Y = H W2) the contraction axis is ffn, so
 * slice s owns ffn columns [lo_s, lo_{s+1}) and
 *     forward : H_s = gelu(X W1[:, lo_s:lo_{s+1}] + b1[lo_s:lo_{s+1}])   [tokens x f_s]  (workspace)
 *               Y  += H_s W2[lo_s:lo_{s+1}, :]                            summed over slices in fp32, then + b2
 *     backward: Z_s, H_s recomputed; dZ_s = (dY W2[lo_s:lo_{s+1}, :]^T) (.) gelu'(Z_s)
 *               dW2[lo_s:lo_{s+1}, :] = H_s^T dY;  dW1[:, lo_s:lo_{s+1}] = X^T dZ_s;  db1[lo_s:lo_{s+1}] = colsum(dZ_s)
 *               (each written once: slices own disjoint parts of the weight gradients)
 *               dX += dZ_s W1[:, lo_s:lo_{s+1}]^T                         summed over slices in fp32;  db2 = colsum(dY)
 * The tokens x ffn intermediate never exists whole (only tokens x ceil(ffn/k)), exactly as in the token split,
 * but the only tensors that span slices are Y and dX (tokens x hidden) instead of dW1 and dW2 (hidden x ffn):
 * the cross-slice read-modify-write traffic falls by hidden*ffn / (tokens*hidden) and every weight is read once per pass
 * (DESIGN.md section 10).
 * Same arguments, dtypes, layouts, ownership and error behaviour as osdp_split_mlp_forward/backward, except:
 *   - desc->k = number of ffn slices, 1 <= k <= ffn / (16 / sizeof(dtype));  lo_s = floor(s * units / k) * unit with
 *     unit = 16 bytes of elements and units = ffn / unit (slices are whole 16-byte column groups);
 *   - workspace (osdp_ffn_split_mlp_workspace_bytes): FWD one [tokens x f_max] tensor, BWD two, f_max = the widest
 *     slice; for k > 1 plus one fp32 [tokens x hidden] accumulator (Y or dX); BWD plus the column-sum partials
 *     (ceil(tokens / 32) x f_max floats for db1, 32 x hidden floats for db2).
 *     Each part rounded up to 256 B.
 *   - results: Y and dX differ across k only by fp32 re-association of the slice sums (then one rounding to the
 *     storage dtype); dW1, dW2, db1, db2 are bit-identical for every k.
 * osdp_ffn_split_mlp_op_cost fills the cost-model factors of this variant for osdp_cost_eval / osdp_plan
 * (extra_fixed includes the fp32 accumulator, i.e. it describes k > 1). */
size_t osdp_ffn_split_mlp_workspace_bytes(const osdp_mlp_desc* desc, int pass);
int osdp_ffn_split_mlp_forward(const osdp_mlp_desc* desc,
                               const void* X, const void* W1, const void* b1, const void* W2, const void* b2,
                               void* Y, void* workspace, size_t workspace_bytes, void* stream);
int osdp_ffn_split_mlp_backward(const osdp_mlp_desc* desc,
                                const void* X, const void* W1, const void* b1, const void* W2, const void* b2,
                                const void* dY,
                                void* dX, float* dW1, float* db1, float* dW2, float* db2,
                                void* workspace, size_t workspace_bytes, void* stream);

/* ---- Linear operator: the other operator type of the paper's models -----------------------------------------
 * Table 1 counts two operators per layer, an attention block and an MLP block; the MatMuls of the
 * attention block are plain Linear operators (minGPT's hidden -> 3 hidden QKV projection and hidden -> hidden output
 * projection).  Operator splitting applies to them as to any MatMul:
 *     forward : Y  = X W + b                 X [tokens x in], W [in x out], b [out] (optional), Y [tokens x out]
 *     backward: dX = dY W^T [tokens x in];   dW = X^T dY [in x out] fp32;   db = colsum(dY) [out] fp32
 * axis = OSDP_SPLIT_CONTRACTION (the paper-literal split: "the last dimension of the input data and the first
 *   dimension of the operator are partitioned ... all computation results are summed"): slice s owns input features
 *   [lo_s, lo_{s+1}), lo_s = floor(s * units / k) * unit, unit = 16 bytes of elements, units = in / unit.
 *   Forward: Y (+)= X[:, lo:hi] W[lo:hi, :] summed over slices in an fp32 [tokens x out] accumulator (workspace, k > 1),
 *   then + b and one rounding.  Backward: dX[:, lo:hi] and dW[lo:hi, :] belong to one slice each (written once).
 * axis = OSDP_SPLIT_TOKENS (the north_star's axis): slice s = rows [floor(s T / k), floor((s+1) T / k)); Y_s, dX_s
 *   are rows of the outputs, dW and db are summed over slices in fp32 ("=" on slice 0, "+=" after).
 * Same conventions as the MLP calls (device pointers of the current device, 16-byte aligned, workspace 256-byte
 * aligned and caller-owned, nothing allocated, only `stream` is used from the caller's point of view, status codes).
 * b and db may be NULL when has_bias = 0.  dW, db are OVERWRITTEN.  workspace may be NULL when the size query says 0.
 * osdp_split_linear_workspace_bytes: FWD = the fp32 accumulator (contraction axis, k > 1) else 0; BWD = the column-sum
 * scratch 32 x out floats (has_bias) else 0; each rounded up to 256 B.  Returns a status; *bytes is written on OSDP_OK.
 * osdp_linear_op_cost: cost-model factors of one call (like osdp_mlp_op_cost): model_bytes = W, b (+ fp32 dW, db in the
 * backward), act_bytes = the tokens x in / tokens x out tensors of the call (one unit of batch = desc->tokens tokens),
 * extra_fixed = the workspace, S = (in out + out) sizeof(dtype). */
typedef enum osdp_split_axis { OSDP_SPLIT_TOKENS = 0, OSDP_SPLIT_CONTRACTION = 1 } osdp_split_axis;
typedef struct osdp_linear_desc {
  int64_t tokens;        /* T >= 1 */
  int64_t in_features;   /* multiple of 8 (bf16) / 4 (f32) */
  int64_t out_features;  /* multiple of 8 (bf16) / 4 (f32) */
  int32_t dtype;         /* osdp_dtype */
  int32_t k;             /* slices: 1 <= k <= tokens (token axis) or <= in_features / unit (contraction axis) */
  int32_t axis;          /* osdp_split_axis */
  int32_t has_bias;      /* 0 / 1 */
} osdp_linear_desc;
int osdp_split_linear_workspace_bytes(const osdp_linear_desc* desc, int pass, size_t* bytes);
int osdp_split_linear_forward(const osdp_linear_desc* desc, const void* X, const void* W, const void* b, void* Y,
                              void* workspace, size_t workspace_bytes, void* stream);
int osdp_split_linear_backward(const osdp_linear_desc* desc, const void* X, const void* W, const void* dY,
                               void* dX, float* dW, float* db, void* workspace, size_t workspace_bytes, void* stream);
/* (osdp_linear_op_cost is declared below, after osdp_op_cost.) */

/* ---- A8 without a workspace: the bias gradient for callers that cannot allocate device memory -------------------
 * db[c] = sum over r of dY[r, c]  ("all computation results are summed": the bias gradient of a Linear
 * is the sum of the output gradient over the tokens; db2 of the MLP backward, db of the Linear backward), fp32, with
 * the same fixed summation order as osdp_split_mlp_backward's db2, so the bits agree with that call.
 *
 * Who this is for: a caller that holds dY and db but has no device memory to lend as a workspace and may not get
 * any - it runs where the CUDA allocator must not be entered (inside another library's callback or allocator hook,
 * on a device whose memory is wholly owned by a pool the caller cannot draw from), or its embedder hands it nothing
 * but the input and output pointers.  All other entry points need a caller workspace; this one needs none, and it
 * calls no cudaMalloc / cudaFree / allocating routine itself.  The 32 x cols floats of partial sums live in a static
 * __device__ array inside the library (2 MiB, reserved on every GPU that loads the library until the process exits),
 * hence the limit: cols <= OSDP_BIAS_GRAD_STATIC_MAX_COLS, otherwise OSDP_ERR_STATIC_LIMIT and nothing is launched.
 *
 *   dY     device pointer, [rows x cols] dense row-major of `dtype` (osdp_dtype), 16-byte aligned; read only
 *   rows   >= 1;  cols >= 1 and a multiple of 8 (bf16) / 4 (f32)
 *   db     device pointer, [cols] fp32, 16-byte aligned; OVERWRITTEN.  Must not alias dY
 *   stream cudaStream_t as void* (NULL = legacy default stream); two kernels are enqueued on it, nothing else
 * The first call on each device looks up the array's device address (cudaGetSymbolAddress, under a mutex, with the
 * calling thread's current device) and checks the compute capability; make that first call before any stream
 * capture begins on that device.  Later calls only enqueue the two kernels.
 * The array is SHARED by every call on a device and keeps the previous call's partial sums.  That needs no
 * clearing (stage 1 writes every word stage 2 reads), but two calls that overlap on the GPU - different streams
 * without an ordering between them, or several host threads on several streams - race on it and give wrong sums.
 * Calls on one stream, or ordered by events, are safe.  Calls on different devices never share (one array per GPU).
 * Errors: OSDP_ERR_NULL, OSDP_ERR_DTYPE, OSDP_ERR_SHAPE, OSDP_ERR_STATIC_LIMIT, OSDP_ERR_ALIGN, OSDP_ERR_ARCH,
 * OSDP_ERR_ARG (device ordinal >= 64), OSDP_ERR_CUDA; db is untouched on every one of them but a launch failure. */
#define OSDP_BIAS_GRAD_STATIC_MAX_COLS 16384
int osdp_bias_grad_static(const void* dY, int64_t rows, int64_t cols, int32_t dtype, float* db, void* stream);

/* Number of kernel launches the last forward/backward call of the calling thread enqueued (for bench.py's
 * gpu_launches claim). */
int64_t osdp_last_launch_count(void);

/* ---- kernel selection knobs (process-wide; defaults are what bench.py measures) ---------------------------
 * The bf16 slice GEMM has two tile shapes: pair tiles of 256 x 256 with the epilogue
 * overlapped (MT = 1) and of 512 x 256 with 25 % less operand traffic and an exposed epilogue (MT = 2), the
 * latter with the producers of all CTA pairs lined up at every tile boundary ("wave sync").  A launch takes
 * MT = 2 when K >= OSDP_TUNE_MT2_MIN_K and either OSDP_TUNE_MT2_MIN_TILES = 0 and the 512 x 256 tiling idles at
 * most ~10 % more MMA slots than the 256 x 256 one (row padding, fill of the last wave), or it has at least
 * OSDP_TUNE_MT2_MIN_TILES > 0 such tiles.  OSDP_TUNE_WAVE_SYNC (MT = 2 launches of more than one wave): 0 off,
 * 1 at tile boundaries, q > 1 also every q k-blocks (64 contraction elements each) inside a tile.  OSDP_TUNE_BAND_MIB: 0 = raster bands that make one wave of
 * resident CTA pairs cover a square-ish block of output tiles (least unique operand bytes per wave); n > 0 = bands whose A
 * rows fit n MiB of L2 (round 1's rule).
 * OSDP_TUNE_CLUSTER_MIN_TILES: n > 0 = launches of at least n pair tiles run as 4-CTA clusters (two CTA pairs that
 * TMA-multicast the A rows they share); 0 = never (clusters of 4 CTAs can occupy only 132 of the 148 SMs).  Results do not depend on
 * any knob beyond fp32 summation order inside a tile (there is none: one owner per output tile).
 * Returns OSDP_ERR_ARG for an unknown key or a value out of range.  osdp_get_tuning returns -1 for an unknown key. */
typedef enum osdp_tune_key {
  OSDP_TUNE_MT2_MIN_K = 0,      /* default 4096 */
  OSDP_TUNE_MT2_MIN_TILES = 1,  /* default 0 (= efficiency rule) */
  OSDP_TUNE_WAVE_SYNC = 2,      /* default 1 */
  OSDP_TUNE_BAND_MIB = 3,       /* default 0 */
  OSDP_TUNE_CLUSTER_MIN_TILES = 4, /* default 0 (multicast clusters off) */
  OSDP_TUNE_MT2_MIN_K_ACC = 5,     /* OSDP_TUNE_MT2_MIN_K for the fp32-accumulate launches (dW GEMMs, K = slice rows) */
  OSDP_TUNE_FORK_MAX_TILES = 6,    /* default 256: in the token-split backward, the launches that only depend on dZ_s
                                      (dW2, dW1, dX, column sums) are enqueued side by side on helper streams that fork
                                      from and join `stream` when each GEMM has at most this many 256 x 256 output tiles
                                      (small slices: every launch is a wave or two; measured +4-8 % at C2, +5 % at the
                                      C5 layer shape, neutral to -1 % at C3 / C4, which the default excludes); 0 = always
                                      in sequence */
  OSDP_TUNE_SLICE_KERNEL_MAX_TILES = 7,
                                   /* default 128.  Token split, bf16: when the [T_s x ffn] GEMMs of a slice have at most
                                      this many 256 x 256 output tiles (small slices: about one wave), the whole slice
                                      runs as ONE persistent kernel (forward A1 -> A2; backward (A3 + A4 fused per tile)
                                      -> A7 | A5 | A6 and the db1 sum): CTA pairs claim tiles of all GEMMs from one list
                                      and a tile waits only for the producer tiles it reads (csrc/slice_sm100.cuh,
                                      DESIGN.md section 6.5).  Results are bit-identical to the launch-per-GEMM path.
                                      If the workspace passed to the forward has room for two slice buffers (the
                                      backward's size), consecutive forward slices alternate buffers and overlap.
                                      0 = never */
  OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES = 8,
                                   /* default 0 (off).  The same path for the ffn-axis split (osdp_ffn_split_mlp_*), taken
                                      when the [tokens x f_s] GEMMs of a slice have at most this many 256 x 256 tiles.
                                      Bit-identical results; faster for many narrow slices of a long token axis (C3
                                      k = 64 +35 %, C5 layer shape k = 16 / 32 +31 / +37 %), slower on C2 and on C4 at
                                      k = 32 (-10 ... -17 %), hence opt-in */
  OSDP_TUNE_BALANCE_N = 9          /* default 1.  The dX GEMM (A7; K-major B, plain epilogue) takes pair tiles of 240 / 224 /
                                      208 / 192 instead of 256 columns when that makes its tile count fill the last wave
                                      of CTA pairs and saves at least 5 % of the launch (C4 k = 4: 128 tiles = 1.73 waves
                                      -> 148 tiles of 224 columns = 2 waves of 0.875).  Results do not change.  0 = always
                                      256 columns */
} osdp_tune_key;
int osdp_set_tuning(int key, int64_t value);
int64_t osdp_get_tuning(int key);

/* ---- per-launch timing (measurement aid; bench.py's roofline) -------------------------------------------
 * osdp_trace_enable(1): from now on every kernel launch of the calling thread's forward/backward calls is
 * bracketed by two CUDA events recorded on the call's stream (nothing else changes; no synchronisation).
 * osdp_trace_read: waits for the recorded events, writes up to max_entries (step id, milliseconds) pairs in
 * launch order, clears the trace and returns the number of launches recorded since the last read (which may
 * exceed max_entries), or -1 on a CUDA error.  Step ids: 1..7 = A1..A7 GEMMs, 8 = the db2 and db1
 * column sums (A8; two launches serve both).  osdp_step_name(id) returns a static string. */
int osdp_trace_enable(int on);
int64_t osdp_trace_read(int64_t max_entries, int32_t* step_ids, float* ms);
const char* osdp_step_name(int step_id);

/* ---- A9: cost model and planner (host only) ------------------------------------------------------------
 * Per-operator record = the paper's "model description" entry: S_i and the three
 * memory factors, with M_extra divided into a part splitting does not shrink and two sliceable parts
 * (reading P6: summed over operators as in Eq. 1, or transient = live for one operator at a time because
 * slices are "released serially"). */
typedef struct osdp_op_cost {
  double   S;                /* parameter bytes one collective moves (S_i) */
  uint64_t model_bytes;      /* M_i^(model): parameters + gradients + optimizer states */
  uint64_t act_bytes;        /* M_i^(act) per unit batch */
  uint64_t extra_fixed;      /* M_i^(extra), not sliceable */
  uint64_t extra_summed;     /* M_i^(extra), sliceable, summed over operators */
  uint64_t extra_transient;  /* M_i^(extra), sliceable, max over operators */
  double   gamma;            /* computation seconds per unit batch (gamma_i) */
  double   delta;            /* seconds per extra slice (reading P2; 0 = the paper's model) */
} osdp_op_cost;

/* "Device information".  The last three fields describe activation checkpointing (PAPER.md:51,
 * :251-253; reading P12) and may be left zero (= the paper's plain cost model): with checkpointing != 0
 *   - a ZDP operator needs FOUR collectives: "the recomputation process before backward propagation requires an
 *     additional round of gathering since each GPU does not maintain a full copy of model states";
 *     DP operators keep their two - which is why OSDP "can leave operators with smaller memory overhead in DP mode";
 *   - computation costs (1 + recompute_fraction) b gamma ("about 30% extra computation overhead");
 *   - only act_keep_fraction of b M_act stays resident (the checkpoints). */
typedef struct osdp_device {
  int32_t  N;                /* parallelism degree >= 1 */
  double   alpha;            /* network latency, seconds */
  double   beta;             /* transfer seconds per byte */
  uint64_t mem_limit_bytes;  /* M_limit */
  int32_t  checkpointing;    /* 0 = off */
  double   recompute_fraction;   /* >= 0; the paper's figure is ~0.3 */
  double   act_keep_fraction;    /* in [0, 1] */
} osdp_device;

/* M_i and T_i of one operator (readings P1, P2):
 *   persist   = model/(N if ZDP else 1, rounded up) + batch*act + extra_fixed + ceil(extra_summed/k)
 *   transient = ceil(extra_transient/k)
 *   seconds   = c (N-1)(alpha + S beta/N) + batch*gamma + (k-1) delta,  c = 2 (DP) / 3 (ZDP)
 * With dev->checkpointing: c = 2 / 4, batch*gamma*(1 + recompute_fraction), ceil(batch*act*act_keep_fraction).
 * Any output pointer may be NULL. */
int osdp_cost_eval(const osdp_op_cost* op, int mode, int32_t k, int64_t batch, const osdp_device* dev,
                   uint64_t* persist_bytes, uint64_t* transient_bytes, double* seconds);

/* Fills an osdp_op_cost for this library's MLP operator as ONE call sees it:
 * pass = OSDP_FWD / OSDP_BWD.  model_bytes = the model states live during the call (W1, W2, b1, b2; in the backward
 * also the fp32 gradients dW1, dW2, db1, db2) - the part ZDP divides by N; act_bytes = the tokens x hidden tensors
 * of the call (X, Y forward; X, dY, dX backward) per unit batch, ONE UNIT OF BATCH = desc->tokens TOKENS (evaluate
 * with batch = 1 for the call as described); extra_transient = workspace at k = 1 minus the fixed scratch;
 * extra_fixed = that scratch; S = (2 h f + f + h) * sizeof(dtype); gamma/delta = 0 (the caller calibrates them).
 * The ZDP rows of the planner describe a sharded placement of the model states; on one GPU (N = 1) they coincide
 * with DP, and the multi-GPU execution of a ZDP decision is osdp_zdp_ffn_split_mlp_* below. */
int osdp_mlp_op_cost(const osdp_mlp_desc* desc, int pass, osdp_op_cost* out);
int osdp_ffn_split_mlp_op_cost(const osdp_mlp_desc* desc, int pass, osdp_op_cost* out);   /* ffn-axis split, see above */
int osdp_linear_op_cost(const osdp_linear_desc* desc, int pass, osdp_op_cost* out);        /* Linear operator, see above */

/* Search engine (Algorithm 1 lines 4-11 at a fixed batch; PAPER.md:149 DFS with two prunings).
 * Decision per operator: mode in {DP, ZDP} x k in k_candidates (ascending, each >= 1).  Minimises
 * sum_i T_i subject to  sum_i persist_i + max_i transient_i <= mem_limit_bytes.  Plans are traversed
 * depth-first in lexicographic order of option index (DP before ZDP, k ascending) and the incumbent is
 * replaced only on a strictly smaller time, so ties resolve to the first plan in that order.
 * Outputs: k_out[n], mode_out[n], *est_seconds, *est_peak_bytes (NULL allowed for the last two).
 * Returns OSDP_ERR_INFEASIBLE (outputs untouched) when no plan fits. */
int osdp_plan(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch,
              const int32_t* k_candidates, int32_t n_cand,
              int32_t* k_out, int32_t* mode_out, double* est_seconds, uint64_t* est_peak_bytes);

/* Slice-level mode mixing ("partition the operator into 4 slices and process 1 of them in the ZDP
 * mode and 3 of them in the DP mode ... a more fine-grained execution plan").  An operator cut into k slices runs
 * zdp_slices of them in ZDP mode and the rest in DP mode (reading P10): each slice carries 1/k of the operator's
 * model states and parameters, so
 *   persist   = (model - zs) + ceil(zs / N) + batch*act + extra_fixed + ceil(extra_summed / k),  zs = ceil(model*zdp_slices / k)
 *   transient = ceil(extra_transient / k)
 *   seconds   = (2 + zdp_slices/k) (N-1)(alpha + S beta/N) + batch*gamma + (k-1) delta
 * zdp_slices = 0 / = k are osdp_cost_eval's DP / ZDP values exactly.  OSDP_ERR_ARG unless 0 <= zdp_slices <= k.
 * osdp_plan_mixed searches per operator over k in k_candidates (each <= 1024) x zdp_slices in 0..k, options ordered
 * k ascending then zdp_slices ascending, otherwise exactly like osdp_plan (same prunings, strict "<", first optimum
 * in traversal order).  Its optimum is never slower than osdp_plan's (a superset of plans). */
int osdp_cost_eval_mixed(const osdp_op_cost* op, int32_t k, int32_t zdp_slices, int64_t batch, const osdp_device* dev,
                         uint64_t* persist_bytes, uint64_t* transient_bytes, double* seconds);
int osdp_plan_mixed(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch,
                    const int32_t* k_candidates, int32_t n_cand,
                    int32_t* k_out, int32_t* zdp_slices_out, double* est_seconds, uint64_t* est_peak_bytes);

/* Scheduler (Algorithm 1 in full): batch = 1, 2, 3, ... up to batch_max; stops at the first
 * batch with no feasible plan; returns the candidate minimising est_seconds / batch (Eq. 1) in *batch_out. */
int osdp_plan_batch(const osdp_op_cost* ops, int32_t n, const osdp_device* dev, int64_t batch_max,
                    const int32_t* k_candidates, int32_t n_cand,
                    int32_t* k_out, int32_t* mode_out, int64_t* batch_out,
                    double* est_seconds, uint64_t* est_peak_bytes);

/* ---- ZDP mode across GPUs with weight-slice gathering -----------------------------------
 * in ZDP mode the model states of an operator are sharded over the N data-parallel ranks, the parameters
 * are all-gathered before the forward and again before the backward, and the gradients are reduce-scattered (three
 * collectives).  PAPER.md:163-167: gathering a huge operator whole is the memory surge operator splitting
 * removes - "Combined with ZDP, operator splitting amortizes the memory from size(MatMul) to
 * size(MatMul) / slice_granularity".  These calls run the ffn-axis split MLP (osdp_ffn_split_mlp_*) in that mode: slice
 * s + 1 of the weights is gathered on `comm_stream` while slice s computes on `compute_stream` ("our
 * distributed training deployment supports the overlapping between computation and communication"), and the slice's
 * weight gradients are reduce-scattered while the next slice computes.  Each rank runs the call on its own token batch.
 *
 * Slices and shards.  unit = 16 bytes of elements.  Slice s = ffn columns [lo_s, lo_{s+1}), lo_s = floor(s G / k) N unit
 * with G = ffn / (N unit): whole groups of N units, so every rank's piece is whole 16-byte units.  Requires
 * hidden % (N unit) == 0, ffn % (N unit) == 0, 1 <= k <= G.  A rank's PARAMETER SHARD is one dense buffer of
 * osdp_zdp_shard_elems() elements of the storage dtype: for s = 0..k-1 the pieces
 *     W1[r h/N : (r+1) h/N, lo:hi]   ((h/N) x fs, row-major)      - gathered: rows concatenate to [h x fs]
 *     b1[lo + r fs/N : lo + (r+1) fs/N]
 *     W2[lo + r fs/N : lo + (r+1) fs/N, :]   ((fs/N) x h)          - gathered: rows concatenate to [fs x h]
 * then b2[r h/N : (r+1) h/N].  osdp_zdp_slice_layout gives the element offsets (s = k: the b2 piece, in b1_off/b1_elems).
 * The GRADIENT SHARD is an fp32 buffer with the same element offsets; it receives the SUM over ranks (data parallelism)
 * of this rank's pieces of dW1, db1, dW2, db2 and is OVERWRITTEN.
 *
 * Collectives come from the caller (osdp_comm): all_gather(send, recv, bytes_per_rank) writes the ranks' send buffers
 * in rank order into recv; reduce_scatter_f32(send, recv, floats_per_rank) sums send (N chunks) over ranks and writes
 * chunk `rank` to recv; both enqueue on the given stream and return 0 on success.  The binding provides them over
 * torch.distributed (NCCL over NVLink / NVSwitch).  comm may be NULL when world == 1 (the collectives are device copies).
 * compute_stream / comm_stream: two cudaStream_t of the current device; the call forks comm_stream from compute_stream
 * at entry and joins it back before returning (in stream order: no host synchronisation); they may be the same stream
 * (no overlap).  Workspace (osdp_zdp_ffn_split_mlp_workspace_bytes): TWO gathered slice buffers (the paper's
 * size / slice_granularity, double-buffered) + in the backward two fp32 gradient staging slices + the ffn-split
 * workspace of one slice.  osdp_zdp_schedule returns the steps of one call in enqueue order (pure host function; the
 * calls walk exactly this list): gathers, slice computations, reduce-scatters, each with the slice, the buffer it uses
 * and the bytes one rank contributes (slice = k: the b2 / db2 vector).  osdp_zdp_ffn_split_mlp_op_cost: cost-model
 * factors of the ZDP execution: model_bytes = the WHOLE operator's model states (osdp_cost_eval divides them by N in
 * ZDP mode), extra_transient = two gathered slices at k = 1 (sliceable: / k), extra_fixed / act_bytes as the ffn split.
 * Status on one B200: N = 1 is parity-tested on the GPU; N = 2 and 3 run the same executor as host threads of one
 * process on one GPU over an in-process loopback communicator (tests/test_gpu_zdp.py), and a world_size-2 CPU run covers
 * the schedule and layout (tests/test_zdp.py); no multi-GPU timing exists.
 * A collective that returns non-zero ends the call with OSDP_ERR_COMM: comm_stream is still joined back into
 * compute_stream, the outputs are undefined. */
typedef struct osdp_zdp_desc {
  osdp_mlp_desc mlp;   /* tokens = THIS rank's token batch; k = number of ffn slices */
  int32_t world;       /* N >= 1 */
  int32_t rank;        /* 0 <= rank < N */
} osdp_zdp_desc;
typedef struct osdp_zdp_slice {
  int64_t lo, hi;               /* ffn columns of the slice */
  int64_t w1_off, w1_elems;     /* element offset / count of the pieces inside a rank's shard */
  int64_t b1_off, b1_elems;
  int64_t w2_off, w2_elems;
} osdp_zdp_slice;
typedef struct osdp_comm {
  void* ctx;
  int (*all_gather)(void* ctx, const void* send, void* recv, size_t bytes_per_rank, void* stream);
  int (*reduce_scatter_f32)(void* ctx, const void* send, void* recv, size_t floats_per_rank, void* stream);
} osdp_comm;
typedef enum osdp_zdp_op { OSDP_ZDP_GATHER = 0, OSDP_ZDP_COMPUTE = 1, OSDP_ZDP_REDUCE_SCATTER = 2 } osdp_zdp_op;
typedef struct osdp_zdp_step {
  int32_t op;                /* osdp_zdp_op */
  int32_t slice;             /* 0..k-1; k = the b2 (forward gather) / db2 (backward reduce-scatter) vector */
  int32_t buffer;            /* which of the two gathered (GATHER, COMPUTE) / gradient staging (REDUCE_SCATTER) buffers */
  int32_t on_comm_stream;    /* 1: enqueued on comm_stream, 0: on compute_stream */
  uint64_t bytes_per_rank;   /* collectives: bytes one rank contributes = bytes it receives from each peer; COMPUTE: 0 */
} osdp_zdp_step;
int osdp_zdp_shard_elems(const osdp_zdp_desc* desc, int64_t* elems);
int osdp_zdp_slice_layout(const osdp_zdp_desc* desc, int32_t s, osdp_zdp_slice* out);
int64_t osdp_zdp_schedule(const osdp_zdp_desc* desc, int pass, int64_t max_steps, osdp_zdp_step* steps);   /* count, or -status */
int osdp_zdp_ffn_split_mlp_workspace_bytes(const osdp_zdp_desc* desc, int pass, size_t* bytes);
int osdp_zdp_ffn_split_mlp_forward(const osdp_zdp_desc* desc, const void* param_shard, const void* X, void* Y,
                                   void* workspace, size_t workspace_bytes, const osdp_comm* comm,
                                   void* compute_stream, void* comm_stream);
int osdp_zdp_ffn_split_mlp_backward(const osdp_zdp_desc* desc, const void* param_shard, const void* X, const void* dY,
                                    void* dX, float* grad_shard, void* workspace, size_t workspace_bytes,
                                    const osdp_comm* comm, void* compute_stream, void* comm_stream);
int osdp_zdp_ffn_split_mlp_op_cost(const osdp_zdp_desc* desc, int pass, osdp_op_cost* out);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* OSDP_H_ */
