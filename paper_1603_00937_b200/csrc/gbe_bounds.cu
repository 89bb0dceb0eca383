// Step 0 - spectral bounds (row 0; reading A-5).
//   eps_min = min_i (H_ii - sum_{j != i} |H_ij|),  eps_max = max_i (H_ii + sum_{j != i} |H_ij|)
// over all stored entries of the global H.  A row without a stored diagonal has H_ii = 0 (A-12).
// The recursive expansion of theta(mu I - H) needs the spectrum in [0,1]; X0 = (eps_max I - H)/(eps_max - eps_min)
// is never stored - the gather and the graph kernels form it on the fly from these two doubles.
//
// Warp per row, 32-bit/64-bit coalesced loads along the row, fixed shuffle tree (deterministic).
// Bound: HBM, 12 B per stored entry.
#include "gbe_internal.cuh"

namespace {
constexpr int BLK = 256;

__global__ void __launch_bounds__(BLK) k_row_bounds(int64_t n, const int64_t* __restrict__ row_ptr,
                                                    const int32_t* __restrict__ col, const double* __restrict__ val,
                                                    double* __restrict__ block_lo, double* __restrict__ block_hi) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t warp0 = (int64_t)blockIdx.x * (BLK / 32) + w, nwarps = (int64_t)gridDim.x * (BLK / 32);
  double lo = INFINITY, hi = -INFINITY;
  for (int64_t i = warp0; i < n; i += nwarps) {
    const int64_t a = row_ptr[i], b = row_ptr[i + 1];
    double d = 0.0, r = 0.0;
    for (int64_t e = a + lane; e < b; e += 32) {
      const double v = val[e];
      if (col[e] == i) d += v; else r += fabs(v);
    }
    d = warp_sum(d);
    r = warp_sum(r);
    lo = fmin(lo, d - r);
    hi = fmax(hi, d + r);
  }
  __shared__ double slo[BLK / 32], shi[BLK / 32];
  if (lane == 0) { slo[w] = lo; shi[w] = hi; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < BLK / 32; ++k) { lo = fmin(lo, slo[k]); hi = fmax(hi, shi[k]); }
    block_lo[blockIdx.x] = lo;
    block_hi[blockIdx.x] = hi;
  }
}

__global__ void k_bounds_final(const double* __restrict__ block_lo, const double* __restrict__ block_hi, int nb,
                               gbe_state* st) {
  double lo = INFINITY, hi = -INFINITY;
  for (int k = threadIdx.x; k < nb; k += 32) { lo = fmin(lo, block_lo[k]); hi = fmax(hi, block_hi[k]); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (threadIdx.x == 0) {
    st->eps_min = lo;
    st->eps_max = hi;
    st->degenerate = !(hi > lo);
  }
}
}  // namespace

int gbe_launch_bounds(const gbe_csr_view& H, double* block_lo, double* block_hi, int max_blocks, gbe_state* st,
                      cudaStream_t s) {
  int64_t want = (H.n + (BLK / 32) - 1) / (BLK / 32);
  int nb = (int)(want < max_blocks ? want : max_blocks);
  if (nb < 1) nb = 1;
  k_row_bounds<<<nb, BLK, 0, s>>>(H.n, H.row_ptr, H.col_idx, H.val, block_lo, block_hi);
  GBE_LAUNCHED();
  k_bounds_final<<<1, 32, 0, s>>>(block_lo, block_hi, nb, st);
  GBE_LAUNCHED();
  return GBE_OK;
}
