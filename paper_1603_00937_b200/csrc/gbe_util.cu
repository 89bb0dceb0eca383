// Small device utilities: exclusive scans used while sizing CSR outputs (not on the per-iteration path).
#include "gbe_internal.cuh"

// ---------------------------------------------------------------------------------------------- allocator
namespace {
thread_local cudaStream_t t_alloc_stream = nullptr;
}
void gbe_set_alloc_stream(cudaStream_t s) {
  static bool pool_ready = false;  // benign race: setting the attribute twice is harmless
  if (!pool_ready) {
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      uint64_t keep = UINT64_MAX;  // keep freed blocks in the pool across synchronisations
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
    pool_ready = true;
  }
  t_alloc_stream = s;
}
cudaStream_t gbe_alloc_stream() { return t_alloc_stream; }
int gbe_dev_alloc(void** p, size_t bytes) {
  cudaError_t e = cudaMallocAsync(p, bytes ? bytes : 16, t_alloc_stream);
  if (e != cudaSuccess) {
    gbe_set_cuda_error(e, "cudaMallocAsync", __LINE__);
    *p = nullptr;
    return GBE_ENOMEM;
  }
  return GBE_OK;
}
void gbe_dev_free(void* p) {
  if (p) cudaFreeAsync(p, t_alloc_stream);
}

namespace {
template <typename TI>
__global__ void __launch_bounds__(1024) k_scan_single_block(const TI* __restrict__ in, int64_t* __restrict__ out,
                                                            int64_t n) {
  __shared__ int64_t part[1024];
  const int t = threadIdx.x;
  const int64_t chunk = (n + 1023) / 1024;
  const int64_t b = (int64_t)t * chunk, e = min(n, b + chunk);
  int64_t s = 0;
  for (int64_t i = b; i < e; ++i) s += (int64_t)in[i];
  part[t] = s;
  __syncthreads();
  // Hillis-Steele inclusive scan over the 1024 chunk sums
  for (int o = 1; o < 1024; o <<= 1) {
    int64_t v = (t >= o) ? part[t - o] : 0;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  int64_t run = part[t] - s;
  for (int64_t i = b; i < e; ++i) {
    int64_t v = (int64_t)in[i];
    out[i] = run;
    run += v;
  }
  if (t == 1023) out[n] = part[1023];
}
}  // namespace

int gbe_exclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, cudaStream_t s) {
  k_scan_single_block<int32_t><<<1, 1024, 0, s>>>(in, out, n);
  GBE_LAUNCHED();
  return GBE_OK;
}
