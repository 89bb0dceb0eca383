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
