// bias_grad_static.cu — osdp_bias_grad_static (include/osdp.h): the bias gradient db = column sums of dY (step A8,
// the db2 of the MLP backward and the db of the Linear backward) for callers that have no device memory to lend.
//
// Why it exists.  Every other entry point takes its scratch from a caller-supplied workspace, which the caller got
// from cudaMalloc or from a framework allocator.  Some callers cannot do either at the point where they need the
// bias gradient: code running inside a region where the CUDA allocator must not be entered (a stream-ordered
// callback, a hook invoked while another library holds the allocator lock, a process whose whole device memory was
// handed to a pool it does not own), or a host that is only given the input and output pointers by its embedder.
// For them the 32 x cols floats of partial sums the two-stage reduction needs live in the library's own module
// memory: the file-scope __device__ array below, reserved on every GPU that loads the library until the process
// exits.  That is why the maximum is modest (OSDP_BIAS_GRAD_STATIC_MAX_COLS columns = 2 MiB).
//
// The arithmetic is the one of reduce.cuh (same chunking, same summation order inside a CTA and across chunks), as
// kernels of this file, so the result has the same bits as the db2 of osdp_split_mlp_backward.  Nothing in this file
// calls cudaMalloc, cudaFree or a library routine that allocates; it does not touch the launch trace either (the trace
// creates events on demand).
//
// g_bias_grad_scratch in HOST code is only a handle for the runtime's symbol table, not a device address: the address
// the kernels get is looked up with cudaGetSymbolAddress, once per device, with that device current.
#include <mutex>

#include "common.cuh"

namespace osdp {
namespace {

constexpr int kChunks = 32;      // partial rows: the rows of dY go into 32 equal chunks (reduce.cuh: kReduceRowChunks)
constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;  // device ordinals the library keeps state for (include/osdp.h, conventions)

static __device__ __align__(256) float g_bias_grad_scratch[(size_t)kChunks * OSDP_BIAS_GRAD_STATIC_MAX_COLS];

template <typename T> struct Vec;
template <> struct Vec<float> {
  static constexpr int N = 4;
  __device__ static void load(const float* p, float (&v)[4]) {
    const float4 x = *reinterpret_cast<const float4*>(p);
    v[0] = x.x; v[1] = x.y; v[2] = x.z; v[3] = x.w;
  }
};
template <> struct Vec<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ static void load(const __nv_bfloat16* p, float (&v)[8]) {
    const uint4 x = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(w[i] << 16);
      v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
};

// Stage 1: grid (column blocks, chunks).  A warp owns whole rows (lanes across 16-byte column vectors), rows
// ascending in steps of 8; the 8 warps are then added in warp order.  partial[chunk][col] is WRITTEN for every column
// of every chunk of the grid, so the shared scratch needs no clearing between calls.
template <typename T>
__global__ void __launch_bounds__(kThreads) bias_grad_partial_kernel(const T* __restrict__ dY, int64_t rows, int cols,
                                                                     int64_t rows_per_chunk, float* __restrict__ partial) {
  constexpr int V = Vec<T>::N;
  constexpr int kWarps = kThreads / 32;
  __shared__ float red[kWarps][32 * V];
  const int lane = threadIdx.x % 32, warp = threadIdx.x / 32;
  const int c = ((int)blockIdx.x * 32 + lane) * V;
  const int64_t r_begin = (int64_t)blockIdx.y * rows_per_chunk;
  const int64_t r_end = r_begin + rows_per_chunk < rows ? r_begin + rows_per_chunk : rows;
  float acc[V];
#pragma unroll
  for (int i = 0; i < V; ++i) acc[i] = 0.0f;
  if (c < cols) {
    for (int64_t r = r_begin + warp; r < r_end; r += kWarps) {
      float v[V];
      Vec<T>::load(dY + r * cols + c, v);
#pragma unroll
      for (int i = 0; i < V; ++i) acc[i] += v[i];
    }
  }
#pragma unroll
  for (int i = 0; i < V; ++i) red[warp][lane * V + i] = acc[i];
  __syncthreads();
  for (int j = threadIdx.x; j < 32 * V; j += kThreads) {
    float s = 0.0f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) s += red[w][j];
    const int col = (int)blockIdx.x * 32 * V + j;
    if (col < cols) partial[(int64_t)blockIdx.y * cols + col] = s;
  }
}

// Stage 2: one thread per column adds the chunk partials in chunk order and overwrites db.
__global__ void bias_grad_final_kernel(const float* __restrict__ partial, int cols, int chunks, float* __restrict__ db) {
  const int col = (int)blockIdx.x * (int)blockDim.x + (int)threadIdx.x;
  if (col >= cols) return;
  float s = 0.0f;
#pragma unroll 8
  for (int r = 0; r < chunks; ++r) s += partial[(int64_t)r * cols + col];
  db[col] = s;
}

// Device address of g_bias_grad_scratch on the current device (set-up once per device ordinal, under a mutex).
struct DeviceSetup {
  bool done = false;
  int status = OSDP_OK;
  float* scratch = nullptr;
};
std::mutex g_setup_mutex;
DeviceSetup g_setup[kMaxDevices];

int scratch_of_current_device(float** out) {
  int dev = -1;
  OSDP_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return OSDP_ERR_ARG;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  DeviceSetup& s = g_setup[dev];
  if (!s.done) {
    int major = 0;
    OSDP_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) {
      s.status = OSDP_ERR_ARCH;
    } else {
      float* p = nullptr;
      OSDP_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_bias_grad_scratch));
      s.scratch = p;
    }
    s.done = true;   // a CUDA failure above returns before this line, so the next call tries again
  }
  *out = s.scratch;
  return s.status;
}

inline bool misaligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }

template <typename T>
int launch(const T* dY, int64_t rows, int cols, float* db, float* scratch, cudaStream_t st) {
  constexpr int V = Vec<T>::N;
  const int64_t rows_per_chunk = (rows + kChunks - 1) / kChunks;
  const int chunks = (int)((rows + rows_per_chunk - 1) / rows_per_chunk);
  const int col_blocks = (cols + 32 * V - 1) / (32 * V);
  bias_grad_partial_kernel<T><<<dim3(col_blocks, chunks), kThreads, 0, st>>>(dY, rows, cols, rows_per_chunk, scratch);
  OSDP_CUDA_TRY(cudaGetLastError());
  bias_grad_final_kernel<<<(cols + 255) / 256, 256, 0, st>>>(scratch, cols, chunks, db);
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace
}  // namespace osdp

extern "C" int osdp_bias_grad_static(const void* dY, int64_t rows, int64_t cols, int32_t dtype, float* db, void* stream) {
  using namespace osdp;
  if (!dY || !db) return OSDP_ERR_NULL;
  if (dtype != OSDP_F32 && dtype != OSDP_BF16) return OSDP_ERR_DTYPE;
  const int64_t unit = dtype == OSDP_BF16 ? 8 : 4;   // 16 bytes of elements
  if (rows < 1 || cols < 1 || cols % unit != 0) return OSDP_ERR_SHAPE;
  if (cols > OSDP_BIAS_GRAD_STATIC_MAX_COLS) return OSDP_ERR_STATIC_LIMIT;   // the partials would not fit the static array
  if (misaligned16(dY) || misaligned16(db)) return OSDP_ERR_ALIGN;
  float* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch);
  if (rc != OSDP_OK) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (dtype == OSDP_BF16) return launch<__nv_bfloat16>(static_cast<const __nv_bfloat16*>(dY), rows, (int)cols, db, scratch, st);
  return launch<float>(static_cast<const float*>(dY), rows, (int)cols, db, scratch, st);
}
