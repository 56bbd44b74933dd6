// bench_atomic_peak.cu — measurement support, NOT part of the product library: the
// denominator of the tally-atomic roofline is not published, so it is measured on the box.  Times
// n_ops no-return fp64 atomic adds (RED.ADD.F64) at pseudo-random addresses of arr_dev[n_bins].
// Built by bench_atomic_peak.py into libbench_atomic_peak.so (sm_100a).
#include <cstdint>
#include <cuda_runtime.h>

// leader_only != 0: only lane 0 of every warp adds (the pattern of a warp-aggregated tally: one RED per warp and round)
__global__ void __launch_bounds__(256) k_atomic_peak(double *arr, unsigned long long n_bins, unsigned long long n_ops, int leader_only)
{
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n_ops; i += stride) {
    if (leader_only && (threadIdx.x & 31)) continue;
    unsigned long long h = i * 0x9E3779B97F4A7C15ull;      // Weyl/xorshift mix: spreads lanes over the array
    h ^= h >> 29; h *= 0xBF58476D1CE4E5B9ull; h ^= h >> 32;
    atomicAdd(arr + (h % n_bins), 1.0);
  }
}

// returns 0 and the device time of the timed launch in *ms_out; 1 on a CUDA error
// (with leader_only, n_ops / 32 adds are made)
extern "C" int bench_atomic_peak(void *arr_dev, uint64_t n_bins, uint64_t n_ops, int leader_only, void *cuda_stream, double *ms_out)
{
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 1;
  k_atomic_peak<<<sms * 8, 256, 0, s>>>((double *)arr_dev, n_bins, n_ops / 8, leader_only);      // warm-up
  cudaEventRecord(e0, s);
  k_atomic_peak<<<sms * 8, 256, 0, s>>>((double *)arr_dev, n_bins, n_ops, leader_only);
  cudaEventRecord(e1, s);
  if (cudaEventSynchronize(e1) != cudaSuccess) return 1;
  float ms = 0.f;
  cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *ms_out = ms;
  return 0;
}
