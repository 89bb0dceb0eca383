// Small device utilities: exclusive scans used while sizing CSR outputs (not on the per-iteration path).
#include <cstdlib>

#include "gbe_internal.cuh"

// ---------------------------------------------------------------------------------------------- allocator
namespace {
thread_local cudaStream_t t_alloc_stream = nullptr;
}
bool gbe_device_once::first() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 256) return true;  // unknown device: set up every time
  const uint64_t bit = 1ull << (dev & 63);
  return (mask[dev >> 6].fetch_or(bit, std::memory_order_acq_rel) & bit) == 0;
}
int gbe_sm_count() {
  static std::atomic<int> cached[256] = {};
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 1;
  if (dev >= 0 && dev < 256 && (n = cached[dev].load(std::memory_order_relaxed)) > 0) return n;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 1;
  if (dev >= 0 && dev < 256) cached[dev].store(n, std::memory_order_relaxed);
  return n;
}
// programmatic dependent launch (gbe_internal.cuh), process-wide: on unless GBE_PDL=0 is in the environment when the
// library is loaded; gbe_set_dependent_launch (gbe.h) changes it
static std::atomic<int> g_pdl{[] { const char* e = getenv("GBE_PDL"); return e ? (atoi(e) != 0 ? 1 : 0) : 1; }()};
bool gbe_pdl_enabled() { return g_pdl.load(std::memory_order_relaxed) != 0; }
int gbe_pdl_set(int on) { return g_pdl.exchange(on ? 1 : 0, std::memory_order_relaxed); }

void gbe_set_alloc_stream(cudaStream_t s) {
  static gbe_device_once pool_ready;  // per device: the release threshold belongs to the device's default pool
  if (pool_ready.first()) {
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      uint64_t keep = UINT64_MAX;  // keep freed blocks in the pool across synchronisations
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    cudaGetLastError();
  }
  t_alloc_stream = s;
}
cudaStream_t gbe_alloc_stream() { return t_alloc_stream; }

// A few pinned host words per thread (allocated once, kept): a device-to-host copy into them does not block the host,
// unlike a copy into pageable memory, so a flag can be fetched now and looked at after a later synchronisation.
int32_t* gbe_pinned_words() {
  thread_local int32_t* w = nullptr;
  if (!w && cudaHostAlloc((void**)&w, 64 * sizeof(int32_t), cudaHostAllocDefault) != cudaSuccess) {
    (void)cudaGetLastError();
    w = nullptr;
  }
  return w;
}
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
// One CTA walks the array in tiles of 16,384: every thread takes SCAN_EPT = 16 consecutive elements (four 16-byte loads
// in flight), warp scans by shuffle, one scan over the 32 warp sums, a running carry between tiles.  (The graph build
// calls this eight times on n counts; with 4 elements per thread the 24,576-orbital box took six tiles and 20 us a call.)
constexpr int SCAN_EPT = 16;
template <typename TI>
__global__ void __launch_bounds__(1024) k_scan_single_block(const TI* __restrict__ in, int64_t* __restrict__ out,
                                                            int64_t n, int want_max) {
  __shared__ int64_t wsum[32];
  __shared__ int64_t tile_total;
  const int t = threadIdx.x, lane = t & 31, w = t >> 5;
  int64_t carry = 0;
  int64_t vmax = 0;  // want_max: out[n + 1] = max(0, max_i in[i])
  const bool vec_ok = sizeof(TI) == 4 && (reinterpret_cast<uintptr_t>(in) & 15) == 0;
  const bool vec_out = (reinterpret_cast<uintptr_t>(out) & 15) == 0;
  for (int64_t base = 0; base < n; base += (int64_t)SCAN_EPT * 1024) {
    const int64_t i0 = base + (int64_t)SCAN_EPT * t;
    TI v[SCAN_EPT];
    if (vec_ok && i0 + SCAN_EPT <= n) {
#pragma unroll
      for (int k = 0; k < SCAN_EPT / 4; ++k) {
        const int4 q = reinterpret_cast<const int4*>(in + i0)[k];
        v[4 * k] = (TI)q.x; v[4 * k + 1] = (TI)q.y; v[4 * k + 2] = (TI)q.z; v[4 * k + 3] = (TI)q.w;
      }
    } else {
#pragma unroll
      for (int k = 0; k < SCAN_EPT; ++k) v[k] = i0 + k < n ? in[i0 + k] : (TI)0;
    }
    int64_t s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_EPT; ++k) {
      s += (int64_t)v[k];
      vmax = max(vmax, (int64_t)v[k]);
    }
    int64_t x = s;  // inclusive scan over the warp
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int64_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) wsum[w] = x;
    __syncthreads();
    if (w == 0) {
      const int64_t ws = wsum[lane];
      int64_t z = ws;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int64_t y = __shfl_up_sync(0xffffffffu, z, o);
        if (lane >= o) z += y;
      }
      wsum[lane] = z - ws;  // exclusive over the warps
      if (lane == 31) tile_total = z;
    }
    __syncthreads();
    int64_t run = carry + wsum[w] + (x - s);
    if (vec_out && i0 + SCAN_EPT <= n) {
#pragma unroll
      for (int k = 0; k < SCAN_EPT; k += 2) {  // (i0 is even)
        const int64_t r1 = run + (int64_t)v[k];
        *reinterpret_cast<longlong2*>(out + i0 + k) = make_longlong2(run, r1);
        run = r1 + (int64_t)v[k + 1];
      }
    } else {
#pragma unroll
      for (int k = 0; k < SCAN_EPT; ++k)
        if (i0 + k < n) {
          out[i0 + k] = run;
          run += (int64_t)v[k];
        }
    }
    carry += tile_total;
    __syncthreads();  // wsum and tile_total are rewritten by the next tile
  }
  if (t == 0) out[n] = carry;
  if (want_max) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, (int64_t)__shfl_xor_sync(0xffffffffu, vmax, o));
    if (lane == 0) wsum[w] = vmax;
    __syncthreads();
    if (t == 0) {
      int64_t m = 0;
      for (int k = 0; k < 32; ++k) m = max(m, wsum[k]);
      out[n + 1] = m;
    }
  }
}
}  // namespace

int gbe_exclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, cudaStream_t s) {
  k_scan_single_block<int32_t><<<1, 1024, 0, s>>>(in, out, n, 0);
  GBE_LAUNCHED();
  return GBE_OK;
}
// as above, and out[n + 1] = max(0, max_i in[i]) (out has n + 2 entries)
int gbe_exclusive_scan_i32_to_i64_max(const int32_t* in, int64_t* out, int64_t n, cudaStream_t s) {
  k_scan_single_block<int32_t><<<1, 1024, 0, s>>>(in, out, n, 1);
  GBE_LAUNCHED();
  return GBE_OK;
}
