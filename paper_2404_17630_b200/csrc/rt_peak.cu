// rt_debug_alu_peak: micro-benchmarks of the fp64 pipe and of shared memory on the device the context
// lives on.  They place the ALU ceiling beside the HBM roofline of the transport kernels (DESIGN.md
// 7.2): every figure is measured, not taken from a data sheet.  Not part of the subcycle.
#include "rt_internal.cuh"

enum { PK_DFMA = 0, PK_DADD, PK_DMUL, PK_DMAX, PK_RCP_SEED, PK_RCP_FULL, PK_RSQ_SEED, PK_DDIV, PK_DSQRT, PK_LDS128, PK_LDS128_B3, PK_LDS128_B8,
       PK_LDS128_RND, PK_N };

template <int OP>
__device__ __forceinline__ double peak_op(double x, double a, double b) {
  if (OP == PK_DFMA) return fma(x, a, b);
  if (OP == PK_DADD) return x + a;
  if (OP == PK_DMUL) return x * a;
  if (OP == PK_DMAX) return x > a ? x : a + b;  // DSETP + select of the two halves (+ DADD off the chain)
  if (OP == PK_RCP_SEED) { double r; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
  if (OP == PK_RCP_FULL) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    return fma(r, e, r);
  }
  if (OP == PK_RSQ_SEED) { double r; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x)); return r; }
  if (OP == PK_DDIV) return a / x;
  return sqrt(x);
}

// CH independent dependency chains per thread, IT operations each
template <int OP, int CH>
__global__ void __launch_bounds__(256) k_peak(int it, double a, double b, double *out) {
  double x[CH];
#pragma unroll
  for (int c = 0; c < CH; c++) x[c] = 1.0 + 1e-3 * (threadIdx.x + c);
  for (int i = 0; i < it; i++) {
#pragma unroll
    for (int c = 0; c < CH; c++) x[c] = peak_op<OP>(x[c], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int c = 0; c < CH; c++) s += x[c];
  if (s == 123.456) out[0] = s;  // keeps the chains alive
}

// 16-byte shared-memory loads, 8 dependent rounds in flight per thread.  MODE 0: lane l reads chunk l
// (32 distinct chunks, conflict-free); 1: lanes 3k, 3k+1, 3k+2 read the same chunk (11 distinct);
// 2: groups of 8 lanes read one chunk (4 distinct); 3: a pseudo-random chunk per lane.
// The next offset depends on the loaded value, so that the compiler cannot hoist the loads.
template <int MODE>
__global__ void __launch_bounds__(256) k_peak_lds(int it, double *out) {
  __shared__ __align__(16) double sm[2 * 512 * 4];
  for (int k = threadIdx.x; k < 2 * 512 * 4; k += 256) sm[k] = 1.0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int chunk = lane;
  if (MODE == 1) chunk = lane / 3;
  if (MODE == 2) chunk = lane / 8;
  if (MODE == 3) chunk = (int)((lane * 2654435761u) >> 23) & 511;
  const double2 *p = reinterpret_cast<const double2 *>(sm) + ((w * 32 + chunk) & 511);
  double s0 = 0.0, s1 = 0.0;
  int off = 0;
  for (int i = 0; i < it; i++) {
#pragma unroll
    for (int c = 0; c < 8; c++) {
      const double2 v = p[512 * off];
      s0 += v.x; s1 += v.y;
      off = (off + __double2int_rn(v.x)) & 3;
    }
  }
  if (s0 + s1 == 123.456) out[0] = s0;
}

template <int OP>
static float time_peak(cudaStream_t st, int blocks, int it, double *scratch) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; rep++) {
    cudaEventRecord(e0, st);
    if (OP == PK_LDS128) k_peak_lds<0><<<blocks, 256, 0, st>>>(it, scratch);
    else if (OP == PK_LDS128_B3) k_peak_lds<1><<<blocks, 256, 0, st>>>(it, scratch);
    else if (OP == PK_LDS128_B8) k_peak_lds<2><<<blocks, 256, 0, st>>>(it, scratch);
    else if (OP == PK_LDS128_RND) k_peak_lds<3><<<blocks, 256, 0, st>>>(it, scratch);
    else k_peak<OP, 8><<<blocks, 256, 0, st>>>(it, 1.0000001, 1e-9, scratch);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}

extern "C" int rt_debug_alu_peak(rt_ctx *c, double *out) {
  if (!c || !out) return RT_EINVAL;
  RT_CUDA(c, cudaSetDevice(c->device));
  cudaDeviceProp prop;
  RT_CUDA(c, cudaGetDeviceProperties(&prop, c->device));
  double *scratch = nullptr;
  RT_CUDA(c, cudaMalloc(&scratch, 64));  // (a debug call: the one allocation outside the caller's workspace)
  const int blocks = prop.multiProcessorCount * 8, it = 4096;
  const double ops = (double)blocks * 256 * 8 * it;  // operations per launch
  float ms[PK_N];
  ms[PK_DFMA] = time_peak<PK_DFMA>(c->stream, blocks, it, scratch);
  ms[PK_DADD] = time_peak<PK_DADD>(c->stream, blocks, it, scratch);
  ms[PK_DMUL] = time_peak<PK_DMUL>(c->stream, blocks, it, scratch);
  ms[PK_DMAX] = time_peak<PK_DMAX>(c->stream, blocks, it, scratch);
  ms[PK_RCP_SEED] = time_peak<PK_RCP_SEED>(c->stream, blocks, it, scratch);
  ms[PK_RCP_FULL] = time_peak<PK_RCP_FULL>(c->stream, blocks, it, scratch);
  ms[PK_RSQ_SEED] = time_peak<PK_RSQ_SEED>(c->stream, blocks, it, scratch);
  ms[PK_DDIV] = time_peak<PK_DDIV>(c->stream, blocks, it / 8, scratch);
  ms[PK_DSQRT] = time_peak<PK_DSQRT>(c->stream, blocks, it / 8, scratch);
  ms[PK_LDS128] = time_peak<PK_LDS128>(c->stream, blocks, it / 4, scratch);
  ms[PK_LDS128_B3] = time_peak<PK_LDS128_B3>(c->stream, blocks, it / 4, scratch);
  ms[PK_LDS128_B8] = time_peak<PK_LDS128_B8>(c->stream, blocks, it / 4, scratch);
  ms[PK_LDS128_RND] = time_peak<PK_LDS128_RND>(c->stream, blocks, it / 4, scratch);
  cudaFree(scratch);
  RT_CUDA(c, cudaGetLastError());
  for (int k = 0; k < PK_N; k++) {
    const double n = (k == PK_DDIV || k == PK_DSQRT) ? ops / 8 : (k >= PK_LDS128 ? ops / 4 : ops);
    out[k] = n / (ms[k] * 1e-3);  // operations (16-byte loads for LDS128) per second
  }
  out[PK_N] = (double)prop.multiProcessorCount;
  return RT_OK;
}
