// gst_noalloc.cu -- gst_polarization_noalloc: the bunch polarization (a13, reading A18) for callers that cannot
// allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The regular path
// (gst_bunch_init + gst_polarization) keeps its per-block partial sums in memory that gst_bunch_init cudaMallocs; this
// variant of the same two-stage reduction keeps them in a file-scope device array, so the call allocates NOTHING: no
// cudaMalloc / cudaFree / cudaMallocHost, no allocating library routine, no handle.  It does not synchronise either:
// the result goes to a DEVICE buffer of the caller's.
//
// The scratch: NOALLOC_MAX_BLOCKS records of four doubles, one per block of 256 particles -- 128 KiB that every GPU
// which loads libgst.so holds until the process exits.  That fixes the maximum: GST_NOALLOC_MAX_PARTICLES = 2^20
// particles (BASELINE's largest bunch); larger requests are refused with GST_EINVAL.
// Every call on a device shares the one array and finds the previous call's records in it.  Nothing in it has to start
// at zero: a call with B blocks overwrites records 0..B-1 and its second stage reads exactly those, never the stale ones
// behind them.  Calls that OVERLAP on one GPU (two streams, two host threads) race on the array; calls on one stream, or
// ordered by events, are safe.
//
// In host code the array's name is a host-side stand-in, not a device address (a kernel handed it would fault, or, where
// the GPU can reach host memory, silently use the wrong memory): the address comes from cudaGetSymbolAddress, asked once
// per device with that device current, and is what the first-stage kernel receives.  Device code of this file may name
// the array directly, which the second stage does.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "../../include/gst.h"
#include "gst_internal.h"

namespace gst {

constexpr int NOALLOC_BLOCK = 256;
constexpr int NOALLOC_WIDTH = 4;                                  // {sum Sx, sum Sy, sum Ss, alive}
constexpr long long NOALLOC_MAX_PARTICLES = GST_NOALLOC_MAX_PARTICLES;
constexpr int NOALLOC_MAX_BLOCKS = (int)(NOALLOC_MAX_PARTICLES / NOALLOC_BLOCK);      // 4096
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) double g_noalloc_partials[NOALLOC_MAX_BLOCKS * NOALLOC_WIDTH];    // 128 KiB

__device__ __forceinline__ double noalloc_warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// block-wide sums of the NOALLOC_WIDTH values of every thread; valid in thread 0 (the order of reduce_kernel.cuh)
__device__ __forceinline__ void noalloc_block_sum(double (&v)[NOALLOC_WIDTH], double* out) {
  __shared__ double sh[NOALLOC_BLOCK / 32][NOALLOC_WIDTH];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NOALLOC_WIDTH; ++k) v[k] = noalloc_warp_sum(v[k]);
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < NOALLOC_WIDTH; ++k) sh[warp][k] = v[k];
  __syncthreads();
  if (warp == 0) {
#pragma unroll
    for (int k = 0; k < NOALLOC_WIDTH; ++k) {
      double x = lane < NOALLOC_BLOCK / 32 ? sh[lane][k] : 0.0;
      x = noalloc_warp_sum(x);
      if (lane == 0) out[k] = x;
    }
  }
}

// stage 1: block b sums the spins of particles 256 b .. 256 b + 255 that are not lost into record b of `partials`
__global__ void __launch_bounds__(NOALLOC_BLOCK) spin_moments_noalloc_kernel(const double* sx, const double* sy,
                                                                             const double* ss, const uint8_t* lost,
                                                                             long long n, double* partials) {
  double v[NOALLOC_WIDTH] = {0.0, 0.0, 0.0, 0.0};
  const long long j = (long long)blockIdx.x * NOALLOC_BLOCK + threadIdx.x;
  if (j < n && !(lost && lost[j])) {
    v[0] = sx[j]; v[1] = sy[j]; v[2] = ss[j]; v[3] = 1.0;
  }
  noalloc_block_sum(v, partials + (size_t)blockIdx.x * NOALLOC_WIDTH);
}

// stage 2 (one block): sums records 0..blocks-1 of the scratch -- named directly: this is device code -- and writes
// out = {Px, Py, Ps, |P|, alive}
__global__ void __launch_bounds__(NOALLOC_BLOCK) spin_finalize_noalloc_kernel(int blocks, double* out) {
  double v[NOALLOC_WIDTH] = {0.0, 0.0, 0.0, 0.0};
  for (int b = threadIdx.x; b < blocks; b += NOALLOC_BLOCK)
#pragma unroll
    for (int k = 0; k < NOALLOC_WIDTH; ++k) v[k] += g_noalloc_partials[(size_t)b * NOALLOC_WIDTH + k];
  __shared__ double tot[NOALLOC_WIDTH];
  noalloc_block_sum(v, tot);
  if (threadIdx.x == 0) {
    const double alive = tot[3];
    const double inv = alive > 0.0 ? 1.0 / alive : 0.0;
    const double px = tot[0] * inv, py = tot[1] * inv, ps = tot[2] * inv;
    out[0] = px; out[1] = py; out[2] = ps;
    out[3] = sqrt(px * px + py * py + ps * ps);
    out[4] = alive;
  }
}

}  // namespace gst

namespace {

// device address of the scratch, asked once per device (0 = not asked yet)
std::mutex g_noalloc_mu;
double* g_noalloc_ptr[gst::NOALLOC_MAX_DEVICES] = {};

// with `device` current
gst_status noalloc_scratch(int device, double** out) {
  if (device < 0 || device >= gst::NOALLOC_MAX_DEVICES) return gst::fail(GST_EINVAL, "device ordinal %d out of range", device);
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  if (!g_noalloc_ptr[device]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, gst::g_noalloc_partials);
    if (e != cudaSuccess || !p)
      return gst::fail(GST_ECUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", device, cudaGetErrorString(e));
    g_noalloc_ptr[device] = p;
  }
  *out = g_noalloc_ptr[device];
  return GST_OK;
}

}  // namespace

extern "C" gst_status gst_polarization_noalloc(const double* sx, const double* sy, const double* ss, const uint8_t* lost,
                                               size_t n, double* out_dev, void* cuda_stream) {
  if (!out_dev || (n > 0 && (!sx || !sy || !ss))) return gst::fail(GST_EINVAL, "null argument");
  if (n > (size_t)gst::NOALLOC_MAX_PARTICLES)
    return gst::fail(GST_EINVAL, "gst_polarization_noalloc: %zu particles exceed GST_NOALLOC_MAX_PARTICLES = %lld (the scratch is a "
                     "fixed device array); use gst_bunch_init + gst_polarization", n, gst::NOALLOC_MAX_PARTICLES);
  cudaPointerAttributes at;
  CUDA_TRY(cudaPointerGetAttributes(&at, out_dev));
  if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged) return gst::fail(GST_EINVAL, "out_dev must be device memory");
  GUARD_DEVICE(at.device);                           // the device that owns the output; the inputs must live there too
  double* scratch = nullptr;
  const gst_status s = noalloc_scratch(at.device, &scratch);
  if (s != GST_OK) return s;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int blocks = (int)((n + gst::NOALLOC_BLOCK - 1) / gst::NOALLOC_BLOCK);
  if (blocks > 0)
    gst::spin_moments_noalloc_kernel<<<blocks, gst::NOALLOC_BLOCK, 0, st>>>(sx, sy, ss, lost, (long long)n, scratch);
  gst::spin_finalize_noalloc_kernel<<<1, gst::NOALLOC_BLOCK, 0, st>>>(blocks, out_dev);
  CUDA_TRY(cudaGetLastError());
  return GST_OK;
}
