// reduce_kernel.cuh -- T2: bunch polarization / emittance reductions (a13) with warp shuffles and a
// block tree, deterministic (no atomics).
#pragma once
#include <cstdint>

namespace gst {

constexpr int RED_BLOCK = 256;
constexpr int RED_WIDTH = 8;          // doubles per partial record
constexpr int RED_MAX_BLOCKS = 1184;  // 148 SMs x 8

struct RedArgs {
  const double* p[9];
  const uint8_t* lost;
  long long n;
  double* partials;   // [blocks][RED_WIDTH]
  double* result;     // [2][RED_WIDTH]: pass 0 sums, pass 1 central second moments
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

// block-wide sum of W values per thread; result valid in thread 0
template <int W>
__device__ __forceinline__ void block_sum(double (&v)[W], double* out) {
  __shared__ double sh[RED_BLOCK / 32][W];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < W; ++k) v[k] = warp_sum(v[k]);
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < W; ++k) sh[warp][k] = v[k];
  __syncthreads();
  if (warp == 0) {
#pragma unroll
    for (int k = 0; k < W; ++k) {
      double x = lane < RED_BLOCK / 32 ? sh[lane][k] : 0.0;
      x = warp_sum(x);
      if (lane == 0) out[k] = x;
    }
  }
}

// pass 0 (SECOND = false): {sum Sx, Sy, Ss, alive, sum X, Px, Y, Py}
// pass 1 (SECOND = true):  {sum dX^2, dPx^2, dX dPx, dY^2, dPy^2, dY dPy, 0, 0} about the pass-0 means
template <bool SECOND>
__global__ void __launch_bounds__(RED_BLOCK) moments_kernel(const RedArgs a) {
  double v[RED_WIDTH];
#pragma unroll
  for (int k = 0; k < RED_WIDTH; ++k) v[k] = 0.0;
  double mx = 0, mpx = 0, my = 0, mpy = 0;
  if (SECOND) {
    double alive = a.result[3];
    double inv = alive > 0 ? 1.0 / alive : 0.0;
    mx = a.result[4] * inv; mpx = a.result[5] * inv; my = a.result[6] * inv; mpy = a.result[7] * inv;
  }
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < a.n; j += stride) {
    if (a.lost[j]) continue;
    if (!SECOND) {
      v[0] += a.p[6][j]; v[1] += a.p[7][j]; v[2] += a.p[8][j]; v[3] += 1.0;
      v[4] += a.p[0][j]; v[5] += a.p[1][j]; v[6] += a.p[2][j]; v[7] += a.p[3][j];
    } else {
      double dx = a.p[0][j] - mx, dp = a.p[1][j] - mpx, dy = a.p[2][j] - my, dq = a.p[3][j] - mpy;
      v[0] = fma(dx, dx, v[0]); v[1] = fma(dp, dp, v[1]); v[2] = fma(dx, dp, v[2]);
      v[3] = fma(dy, dy, v[3]); v[4] = fma(dq, dq, v[4]); v[5] = fma(dy, dq, v[5]);
    }
  }
  block_sum<RED_WIDTH>(v, a.partials + (size_t)blockIdx.x * RED_WIDTH);
}

__global__ void __launch_bounds__(RED_BLOCK) finalize_kernel(const double* partials, int blocks, double* result, int pass) {
  double v[RED_WIDTH];
#pragma unroll
  for (int k = 0; k < RED_WIDTH; ++k) v[k] = 0.0;
  for (int b = threadIdx.x; b < blocks; b += blockDim.x)
#pragma unroll
    for (int k = 0; k < RED_WIDTH; ++k) v[k] += partials[(size_t)b * RED_WIDTH + k];
  block_sum<RED_WIDTH>(v, result + pass * RED_WIDTH);
}

}  // namespace gst
