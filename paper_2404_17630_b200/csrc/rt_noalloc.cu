// rt_stored_photons_noalloc: the photon budget's "stored" row (sum over cells of V N per group, the left side
// of the identity in include/rt.h) for callers that may not allocate: code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc.  The existing path (k_stored + k_reduce behind
// rt_ledger_read) keeps its per-block partial sums in the caller's workspace; this variant keeps them in a
// file-scope device array of a fixed size, so the call needs no context, no workspace and no allocation.
//
// The scratch array is shared by every call on a device and keeps the last call's contents.  Nothing in it has
// to start at zero: a call writes every row it later reads (rows 0 .. ceil(C / 256) - 1) before it reads them,
// in stream order.  Two calls that overlap on the GPU (different streams, no dependency) race on it.
#include <mutex>
#include "rt_internal.cuh"

#define RT_NA_BLOCK 256
#define RT_NA_ROWS (RT_NOALLOC_MAX_CELLS / RT_NA_BLOCK)

// [RT_NA_ROWS][RT_MAXG] partial sums: 4 MiB, held by every GPU that loads the library until the process exits
static __device__ __align__(256) double na_scratch[(size_t)RT_NA_ROWS * RT_MAXG];

// part[row][g] = sum over the block's cells of V N_g (fixed order: warp shuffles, then the warps in order)
__global__ void __launch_bounds__(RT_NA_BLOCK) k_na_partial(int64_t C, int G, const double *__restrict__ N,
                                                             const double *__restrict__ V, double *__restrict__ part) {
  __shared__ double sm[RT_MAXG][RT_NA_BLOCK / 32];
  const int64_t i = (int64_t)blockIdx.x * RT_NA_BLOCK + threadIdx.x;
  const double vol = i < C ? V[i] : 0.0;
  for (int g = 0; g < G; g++) {
    double v = i < C ? vol * N[(size_t)g * C + i] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sm[g][threadIdx.x >> 5] = v;
  }
  __syncthreads();
  if (threadIdx.x < G) {
    double t = 0.0;
    for (int k = 0; k < RT_NA_BLOCK / 32; k++) t += sm[threadIdx.x][k];
    part[(size_t)blockIdx.x * G + threadIdx.x] = t;
  }
}

// out[g] = sum of the rows, one block per group: compensated (Neumaier) per thread over rows tid, tid + 1024, ...,
// then a fixed tree: the result does not depend on the scheduling
__global__ void __launch_bounds__(1024) k_na_final(int64_t nrows, int G, const double *__restrict__ part, double *__restrict__ out) {
  __shared__ double sm[1024];
  const int g = blockIdx.x;
  double s = 0.0, c = 0.0;
  for (int64_t r = threadIdx.x; r < nrows; r += 1024) {
    const double x = part[(size_t)r * G + g], t = s + x;
    c += fabs(s) >= fabs(x) ? (s - t) + x : (x - t) + s;
    s = t;
  }
  sm[threadIdx.x] = s + c;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[g] = sm[0];
}

// the device address of na_scratch, looked up once per device with that device current.  (In host code the
// name na_scratch is a host-side stand-in, not a device address: a kernel must be given this pointer.)
#define RT_NA_MAXDEV 64
static double *na_ptr[RT_NA_MAXDEV];
static std::mutex na_mutex;

static int na_fail(char *err, int errlen, int code, const char *msg, const char *detail) {
  if (err && errlen > 0) snprintf(err, (size_t)errlen, "%s%s%s", msg, detail ? ": " : "", detail ? detail : "");
  return code;
}

extern "C" int rt_stored_photons_noalloc(int device, void *stream, int64_t ncell, int ngroup, const double *N_dev,
                                         const double *volume_dev, double *stored_dev, char *err, int errlen) {
  if (err && errlen > 0) err[0] = 0;
  if (device < 0 || device >= RT_NA_MAXDEV) return na_fail(err, errlen, RT_EINVAL, "device index out of range", nullptr);
  if (ngroup < 1 || ngroup > RT_MAXG) return na_fail(err, errlen, RT_EINVAL, "ngroup must be in [1, 8]", nullptr);
  if (ncell < 0) return na_fail(err, errlen, RT_EINVAL, "ncell must not be negative", nullptr);
  if (ncell > (int64_t)RT_NOALLOC_MAX_CELLS) {
    char buf[160];
    snprintf(buf, sizeof buf, "%lld cells, the static scratch holds partial sums for at most %lld (RT_NOALLOC_MAX_CELLS); use rt_ledger_read",
             (long long)ncell, (long long)RT_NOALLOC_MAX_CELLS);
    return na_fail(err, errlen, RT_EINVAL, "too many cells for the no-allocation entry point", buf);
  }
  if (!stored_dev || (ncell > 0 && (!N_dev || !volume_dev))) return na_fail(err, errlen, RT_EINVAL, "null pointer", nullptr);
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
  if (e != cudaSuccess) return na_fail(err, errlen, RT_ECUDA, "cudaSetDevice", cudaGetErrorString(e));
  double *scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(na_mutex);
    if (!na_ptr[device]) {
      e = cudaGetSymbolAddress((void **)&na_ptr[device], na_scratch);
      if (e != cudaSuccess) {
        na_ptr[device] = nullptr;
        if (prev >= 0 && prev != device) cudaSetDevice(prev);
        return na_fail(err, errlen, RT_ECUDA, "cudaGetSymbolAddress(na_scratch)", cudaGetErrorString(e));
      }
    }
    scratch = na_ptr[device];
  }
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t nrows = (ncell + RT_NA_BLOCK - 1) / RT_NA_BLOCK;
  if (nrows > 0) k_na_partial<<<(unsigned)nrows, RT_NA_BLOCK, 0, st>>>(ncell, ngroup, N_dev, volume_dev, scratch);
  k_na_final<<<ngroup, 1024, 0, st>>>(nrows, ngroup, scratch, stored_dev);
  e = cudaGetLastError();
  if (prev >= 0 && prev != device) cudaSetDevice(prev);
  if (e != cudaSuccess) return na_fail(err, errlen, RT_ECUDA, "kernel launch", cudaGetErrorString(e));
  return RT_OK;
}
