// gst_diag.cu -- the diagnostics of include/gst_diag.h: T3, the DFMA-chain microbenchmarks behind the roofline
// denominators; the accuracy self-test of the kernels' reciprocal routines; kernel resource queries.
// (gst_diag_chain_poll_limit sits in gst_api.cu, next to the bunch handle it sets.)
#include "../../include/gst_diag.h"

#include <cuda_runtime.h>

#include <cstring>

#include "gst_internal.h"
#include "track_launch.cuh"

namespace gst {

// T3: PEAK_CHAINS independent DFMA chains per thread, all operands in registers.
constexpr int PEAK_BLOCK = 256;
constexpr int PEAK_CHAINS = 8;
constexpr int PEAK_UNROLL = 16;
__global__ void __launch_bounds__(PEAK_BLOCK) dfma_peak_kernel(double* out, int iters, double m) {
  double x[PEAK_CHAINS];
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) x[k] = 1e-3 * (threadIdx.x + k);
  const double b = 1e-7;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u)
#pragma unroll
      for (int k = 0; k < PEAK_CHAINS; ++k) x[k] = fma(x[k], m, b);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) s += x[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// T3b: the same chains with THREE distinct register operands per DFMA (x = y*z + x).  On B200 such a
// DFMA occupies the sub-partition for 3 cycles instead of 2 (one cycle per distinct 64-bit register source;
// DMUL/DADD and DFMAs with a constant, immediate or repeated operand take 2): the ceiling of code whose
// multiply-adds all take three registers is 2/3 of the T3 figure.
__global__ void __launch_bounds__(PEAK_BLOCK) dfma_rrr_kernel(double* out, int iters, double m) {
  double x[PEAK_CHAINS], y[PEAK_CHAINS], z[PEAK_CHAINS];
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) {
    x[k] = 1e-3 * (threadIdx.x + k);
    y[k] = m + 1e-9 * (threadIdx.x + k);
    z[k] = 1e-9 * (k + 1) + 1e-12 * threadIdx.x;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PEAK_UNROLL; ++u)
#pragma unroll
      for (int k = 0; k < PEAK_CHAINS; ++k) x[k] = fma(y[(k + 1) % PEAK_CHAINS], z[(k + 3) % PEAK_CHAINS], x[k]);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < PEAK_CHAINS; ++k) s += x[k] + y[k] + z[k];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// max relative error (in units of 2^-53) of the branch-free reciprocal / reciprocal square root
__global__ void math_selftest_kernel(unsigned long long* out, int n) {
  double worst_rcp = 0.0, worst_rsq = 0.0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    double x = exp2(-2.0 + 4.0 * ((double)i + 0.37) / (double)n);     // [0.25, 4)
    double r = rcp_nr(x), q = rsqrt_nr(x);
    double er = fabs(fma(r, x, -1.0));                                 // |r x - 1|, exact residual
    double eq = fabs(fma(q * q, x, -1.0)) * 0.5;                       // ~ |q sqrt(x) - 1|
    worst_rcp = fmax(worst_rcp, er);
    worst_rsq = fmax(worst_rsq, eq);
  }
  atomicMax(out, (unsigned long long)__double_as_longlong(worst_rcp));
  atomicMax(out + 1, (unsigned long long)__double_as_longlong(worst_rsq));
}

// The rotation-vector ring of track_split_kernel.cuh on its own: warp 0 pushes n entries, warp 1 pops and checks them.
// Both start their entry counter at `start` (a multiple of the ring length), e.g. just below the wrap of 32 bits.
__global__ void __launch_bounds__(SPLIT_BLOCK) ring_selftest_kernel(unsigned start, unsigned n, unsigned long long* bad) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31;
  RotvecRing ring;
  ring.attach(smem_raw, lane);
  ring.s = start;
  if (threadIdx.x < 32) {
    for (unsigned i = 0; i < n; ++i) ring.push(1.0 * i + 0.001 * lane, -2.0 * i + lane, 0.5 * i);
    ring.flush();
  } else {
    ring.open();
    unsigned long long wrong = 0;
    for (unsigned i = 0; i < n; ++i) {
      double x, y, z;
      ring.pop(x, y, z);
      wrong += (x != 1.0 * i + 0.001 * lane) + (y != -2.0 * i + lane) + (z != 0.5 * i);
    }
    if (wrong) atomicAdd(bad, wrong);
  }
}

}  // namespace gst

namespace {
using gst::fail;

gst_status fp64_peak_impl(bool three_registers, double* out_tflops, double* out_ms) {
  if (!out_tflops) return fail(GST_EINVAL, "null argument");
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* d_out = nullptr;
  CUDA_TRY(cudaMalloc(&d_out, sizeof(double) * sms * 8 * gst::PEAK_BLOCK));
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  const int iters = 1 << 14;
  float best = 1e30f;
  for (int rep = 0; rep < 6; ++rep) {
    cudaEventRecord(e0);
    if (three_registers) gst::dfma_rrr_kernel<<<sms * 8, gst::PEAK_BLOCK>>>(d_out, iters, 1.0 + 1e-9 * rep);
    else gst::dfma_peak_kernel<<<sms * 8, gst::PEAK_BLOCK>>>(d_out, iters, 1.0 + 1e-9 * rep);
    cudaEventRecord(e1);
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d_out);
  CUDA_TRY(cudaGetLastError());
  double flops = 2.0 * gst::PEAK_CHAINS * (double)iters * gst::PEAK_UNROLL * (double)sms * 8 * gst::PEAK_BLOCK;
  *out_tflops = flops / (best * 1e-3) / 1e12;
  if (out_ms) *out_ms = best;
  return GST_OK;
}

}  // namespace

extern "C" {

gst_status gst_diag_fp64_peak(double* out_tflops, double* out_ms) { return fp64_peak_impl(false, out_tflops, out_ms); }
gst_status gst_diag_fp64_peak_rrr(double* out_tflops, double* out_ms) { return fp64_peak_impl(true, out_tflops, out_ms); }

gst_status gst_diag_selftest_math(double out[2]) {
  if (!out) return fail(GST_EINVAL, "null argument");
  unsigned long long* d = nullptr;
  CUDA_TRY(cudaMalloc(&d, 16));
  CUDA_TRY(cudaMemset(d, 0, 16));
  gst::math_selftest_kernel<<<296, 256>>>(d, 1 << 24);
  unsigned long long h[2];
  cudaError_t ce = cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (ce != cudaSuccess) return fail(GST_ECUDA, "selftest: %s", cudaGetErrorString(ce));
  for (int k = 0; k < 2; ++k) {
    double v;
    std::memcpy(&v, &h[k], 8);
    out[k] = v / 1.1102230246251565e-16;      // in units of 2^-53
  }
  return GST_OK;
}

#ifndef GST_KERNEL_SOURCE_HASH
#define GST_KERNEL_SOURCE_HASH "unknown"
#endif
gst_status gst_diag_selftest_ring(uint32_t start_count, uint32_t n_entries, int64_t* out_mismatches) {
  if (!out_mismatches) return fail(GST_EINVAL, "null argument");
  if (start_count % (2 * gst::SPLIT_HALF) != 0) return fail(GST_EINVAL, "start_count must be a multiple of the ring length, %d", 2 * gst::SPLIT_HALF);
  unsigned long long* d = nullptr;
  CUDA_TRY(cudaMalloc(&d, 8));
  CUDA_TRY(cudaMemset(d, 0, 8));
  gst::ring_selftest_kernel<<<1, gst::SPLIT_BLOCK, gst::SPLIT_RING_BYTES>>>(start_count, n_entries, d);
  unsigned long long h = 0;
  cudaError_t ce = cudaMemcpy(&h, d, 8, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (ce != cudaSuccess) return fail(GST_ECUDA, "ring selftest: %s", cudaGetErrorString(ce));
  *out_mismatches = (int64_t)h;
  return GST_OK;
}

const char* gst_diag_kernel_source_hash(void) { return GST_KERNEL_SOURCE_HASH; }

gst_status gst_diag_kernel_info(gst_split split, int romberg_depth, int variant, int* out_registers, int* out_local_bytes,
                                int* out_max_blocks_per_sm) {
  if ((int)split < 0 || (int)split > 5 || romberg_depth < 1 || romberg_depth > 6) return fail(GST_EINVAL, "unknown split or depth");
  const int order = (int)split >= 3 ? 4 : 2;
  if (variant < 0 || variant > 3) return fail(GST_EINVAL, "unknown kernel variant %d", variant);
  if ((variant == 1 || variant == 3) && order == 4)
    return fail(GST_EINVAL, "the rotating launch and the two-warp kernel exist for the second-order splits only");
  gst::KernelInfo ki;
  const cudaError_t ce = gst::kernel_info_of((int)split % 3, order, romberg_depth, variant, &ki);
  if (ce != cudaSuccess) return fail(GST_ECUDA, "kernel attributes: %s", cudaGetErrorString(ce));
  if (out_registers) *out_registers = ki.registers;
  if (out_local_bytes) *out_local_bytes = ki.local_bytes;
  if (out_max_blocks_per_sm) *out_max_blocks_per_sm = ki.blocks_per_sm;
  return GST_OK;
}

}  // extern "C"
