// Step 5 - global trace and SP2 branch choice (row 5).
//
//     t1 = sum_p sum_{i<ncore_p} (X_n)_ii,   t2 = sum_p sum_{i<ncore_p} (X_n^2)_ii      (fixed-order reduction)
//     [idem_tol >= 0 and n >= 1 and |t1 - t2| <= idem_tol: stop]                          (A-7)
//     branch_n = X^2 if |t2 - n_occ| < |2 t1 - t2 - n_occ| else 2X - X^2 (tie -> 2X - X^2)  (A-6)
// One polynomial for every subgraph (Eq.(4); "the same for each subgraph expansion ... for the correct
// total occupation").  The paper pre-sets the sequence from a gap estimate (ref. 41); north_star
// asks for the choice from the global trace, taken on the device with no host round trip.
// A single CTA sums the partials (one pair per gather CTA, or per X^2 tile with a core row) in a fixed order (no
// floating-point atomics): reproducible.
// Bound: latency (16 B per partial).
#include "gbe_internal.cuh"

namespace {
constexpr int TB = 1024;

__global__ void __launch_bounds__(TB) k_trace_branch(gbe_state* st, const double* __restrict__ partials, int n) {
  __shared__ double s1[32], s2[32];
  const int t = threadIdx.x;
  // programmatic dependent launch (gbe_internal.cuh): this CTA may be resident before the kernel that writes the partials
  // has finished - wait for it; the next kernel of the stream is let go at the very end, after the decision
  // the state this kernel decides from is written by kernels of its own kind only (and before the first X^2 launch):
  // thread 0 requests it before the wait, so that the decision costs no load after the sums
  gbe_decide_in din = {};
  int stopped = 0;
  if (t == 0) {
    din = gbe_trace_decide_load(st);
    stopped = __ldcg(&st->stop);
  }
  gbe_griddep_wait();
  // the kernel is one CTA and latency bound: 8 independent 16-byte loads in flight per thread, summed in a fixed order
  double a1 = 0.0, a2 = 0.0;
  const double2* __restrict__ p2 = reinterpret_cast<const double2*>(partials);
  for (int i = t; i < n; i += 8 * TB) {
    double2 v[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) v[u] = i + u * TB < n ? p2[i + u * TB] : make_double2(0.0, 0.0);
#pragma unroll
    for (int u = 0; u < 8; ++u) { a1 += v[u].x; a2 += v[u].y; }
  }
  // fixed-order reduction: butterfly inside each warp, then warp 0 over the 32 warp sums
  a1 = warp_sum(a1);
  a2 = warp_sum(a2);
  if ((t & 31) == 0) { s1[t >> 5] = a1; s2[t >> 5] = a2; }
  __syncthreads();
  if (t < 32) {
    a1 = warp_sum(s1[t]);
    a2 = warp_sum(s2[t]);
  }
  if (t == 0) {
    if (!stopped) gbe_trace_decide(st, a1, a2, din);
    // the X^2 launch behind this kernel (launched with the attribute) never waits: it may start only now, when X_{n+1}
    // is complete (the wait above) and the decision is visible device-wide
    __threadfence();
    gbe_griddep_launch();
  }
}
}  // namespace

int gbe_launch_trace_branch(gbe_state* st, const double* partials, int n_partials, cudaStream_t s, int pdl) {
  GBE_CUDA(gbe_launch_kernel(k_trace_branch, dim3(1), dim3(TB), 0, s, pdl != GBE_PDL_NONE, st, partials, n_partials));
  GBE_LAUNCHED();
  return GBE_OK;
}
