// Observables of the assembled density matrix (not on the per-iteration path).
//
//     <A> = Tr[D A] = sum_{k,i} D_ki A_ik                                    ("expectation values"; P:L76 E_band = Tr[DH])
// D is the CSR matrix produced by gbe_density on the pattern S' of the graph (not symmetric, obs. (i) P:L65), A any CSR
// matrix of the same dimension with ascending columns (the Hamiltonian for the band energy).
// Warp per row k of D, lanes over its stored entries (k, i); A_ik is found by binary search of column k in row i of A.
// Reduction in a fixed order (lane-strided sums, shuffle tree, per-row partials, one CTA for the final sum): reproducible.
// Bound: L2 latency (one dependent binary search per stored entry of D).
#include "gbe_internal.cuh"

namespace {
__global__ void __launch_bounds__(256) k_expect_rows(int64_t n, const int64_t* __restrict__ D_rp,
                                                     const int32_t* __restrict__ D_col, const double* __restrict__ D_val,
                                                     const int64_t* __restrict__ A_rp, const int32_t* __restrict__ A_col,
                                                     const double* __restrict__ A_val, double* __restrict__ row_sum) {
  const int lane = threadIdx.x & 31;
  const int64_t k = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (k >= n) return;
  double acc = 0.0;
  for (int64_t e = D_rp[k] + lane; e < D_rp[k + 1]; e += 32) {
    const int i = D_col[e];
    int64_t lo = A_rp[i], hi = A_rp[i + 1];
    const int64_t end = hi;
    while (lo < hi) {
      const int64_t mid = (lo + hi) >> 1;
      if (A_col[mid] < k) lo = mid + 1; else hi = mid;
    }
    if (lo < end && A_col[lo] == k) acc += D_val[e] * A_val[lo];
  }
  acc = warp_sum(acc);
  if (lane == 0) row_sum[k] = acc;
}

__global__ void __launch_bounds__(1024) k_expect_final(int64_t n, const double* __restrict__ row_sum, double* __restrict__ out) {
  __shared__ double sh[1024];
  const int t = threadIdx.x;
  double a = 0.0;
  for (int64_t i = t; i < n; i += 1024) a += row_sum[i];
  sh[t] = a;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (t < o) sh[t] += sh[t + o];
    __syncthreads();
  }
  if (t == 0) out[0] = sh[0];
}
}  // namespace

int gbe_launch_expectation(const gbe_graph* g, const double* D_val, const gbe_csr_view& A, double* row_sum, double* out,
                           cudaStream_t s) {
  const int64_t n = g->n;
  k_expect_rows<<<(unsigned)((n + 7) / 8), 256, 0, s>>>(n, g->D_row_ptr, g->D_col, D_val, A.row_ptr, A.col_idx, A.val,
                                                       row_sum);
  GBE_LAUNCHED();
  k_expect_final<<<1, 1024, 0, s>>>(n, row_sum, out);
  GBE_LAUNCHED();
  return GBE_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Error of the assembled D against a dense reference (Fig.2: "the error in the calculated density matrix ... as
// measured by the Frobenius norm (normalized per atom)"):
//     out[0] = max |D_ki - R_ki| over the stored entries of D,   out[1] = sum (D_ki - R_ki)^2 over the stored entries,
//     out[2] = ||D - R||_F^2 over the full matrix (D is zero where it stores nothing, obs. (iv) P:L65).
// Warp per row: the stored entries lane-strided, then the gaps between consecutive stored columns summed directly
// (no ||R||^2 - sum cancellation).  Fixed-order reductions: reproducible.  Bound: HBM (one pass over the n x n reference).
namespace {
__global__ void __launch_bounds__(256) k_error_rows(int64_t n, const int64_t* __restrict__ D_rp,
                                                    const int32_t* __restrict__ D_col, const double* __restrict__ D_val,
                                                    const double* __restrict__ R, int64_t ld,
                                                    double* __restrict__ row_out /* 3 n */) {
  const int lane = threadIdx.x & 31;
  const int64_t k = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (k >= n) return;
  const double* __restrict__ r = R + k * ld;
  const int64_t e0 = D_rp[k], e1 = D_rp[k + 1];
  double mx = 0.0, in2 = 0.0, out2 = 0.0;
  for (int64_t e = e0 + lane; e < e1; e += 32) {
    const double d = D_val[e] - r[D_col[e]];
    mx = fmax(mx, fabs(d));
    in2 += d * d;
  }
  int prev = -1;  // last stored column seen (n < 2^31: columns are int32)
  for (int64_t b = e0; b <= e1; b += 32) {  // 32 stored columns at a time; the sentinel n closes the last gap
    const int64_t e = b + lane;
    const int mine = e < e1 ? D_col[e] : (int)n;
    const int cnt = (int)min((int64_t)32, e1 - b + 1);
    for (int u = 0; u < cnt; ++u) {
      const int next = __shfl_sync(0xffffffffu, mine, u);
      for (int c = prev + 1 + lane; c < next; c += 32) {
        const double x = r[c];
        out2 += x * x;
      }
      prev = next;
    }
  }
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  in2 = warp_sum(in2);
  out2 = warp_sum(out2);
  if (lane == 0) {
    row_out[k] = mx;
    row_out[n + k] = in2;
    row_out[2 * n + k] = in2 + out2;
  }
}

__global__ void __launch_bounds__(1024) k_error_final(int64_t n, const double* __restrict__ row_out,
                                                      double* __restrict__ out) {
  __shared__ double sh[3][1024];
  const int t = threadIdx.x;
  double mx = 0.0, a = 0.0, b = 0.0;
  for (int64_t i = t; i < n; i += 1024) {
    mx = fmax(mx, row_out[i]);
    a += row_out[n + i];
    b += row_out[2 * n + i];
  }
  sh[0][t] = mx;
  sh[1][t] = a;
  sh[2][t] = b;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (t < o) {
      sh[0][t] = fmax(sh[0][t], sh[0][t + o]);
      sh[1][t] += sh[1][t + o];
      sh[2][t] += sh[2][t + o];
    }
    __syncthreads();
  }
  if (t == 0) { out[0] = sh[0][0]; out[1] = sh[1][0]; out[2] = sh[2][0]; }
}
}  // namespace

int gbe_launch_error_norms(const gbe_graph* g, const double* D_val, const double* D_ref, int64_t ld_ref, double* row_out,
                           double* out, cudaStream_t s) {
  const int64_t n = g->n;
  k_error_rows<<<(unsigned)((n + 7) / 8), 256, 0, s>>>(n, g->D_row_ptr, g->D_col, D_val, D_ref, ld_ref, row_out);
  GBE_LAUNCHED();
  k_error_final<<<1, 1024, 0, s>>>(n, row_out, out);
  GBE_LAUNCHED();
  return GBE_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// gbe_expectation_static: <A> = Tr[D A] for callers that may not allocate (gbe.h).  The same two kernels as
// gbe_launch_expectation; the n per-row partial sums go to a FILE-SCOPE device array instead of a pool allocation.
//   - GBE_STATIC_MAX_N doubles = 1 MiB of device memory, held by every GPU that loads the library until the process exits;
//   - in host code the NAME g_expect_scratch is a host-side stand-in of the symbol, not a device address: the address is
//     looked up once per device, with that device current (cudaGetSymbolAddress), and handed to the kernels;
//   - nothing in the array has to start at zero: k_expect_rows writes row_sum[k] for every k < n before k_expect_final
//     reads exactly those n words, so whatever the previous call (or a larger n) left behind is never read;
//   - every call on a device shares the array: two calls that overlap on the GPU (different streams, no dependency
//     between them) race on it.
static __device__ __align__(256) double g_expect_scratch[GBE_STATIC_MAX_N];

namespace {
int expect_scratch_address(double** out) {
  static std::atomic<double*> cached[256] = {};  // per device
  int dev = 0;
  GBE_CUDA(cudaGetDevice(&dev));
  const bool slot = dev >= 0 && dev < 256;
  double* p = slot ? cached[dev].load(std::memory_order_acquire) : nullptr;
  if (!p) {
    GBE_CUDA(cudaGetSymbolAddress((void**)&p, g_expect_scratch));
    if (!p) return GBE_ECUDA;
    if (slot) cached[dev].store(p, std::memory_order_release);
  }
  *out = p;
  return GBE_OK;
}
}  // namespace

int gbe_launch_expectation_static(const gbe_graph* g, const double* D_val, const gbe_csr_view& A, double* out_dev,
                                  cudaStream_t s) {
  if (g->n > GBE_STATIC_MAX_N) return GBE_ELIMIT;
  double* row_sum = nullptr;
  GBE_TRY(expect_scratch_address(&row_sum));
  return gbe_launch_expectation(g, D_val, A, row_sum, out_dev, s);
}
