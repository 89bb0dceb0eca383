// Steps 4 + 5 for SMALL subgraphs: the whole SP2 loop in one kernel, X_p resident in shared memory.
//
//     for n = 0 .. iters - 1:  t1, t2 (global, over core diagonals);  branch_n;  X_p <- X_p^2  or  2 X_p - X_p^2
// (one sequence for every subgraph).  A system of a few dozen small communities (config 1: 16 blocks
// of 48 x 48) is launch bound on the tiled path: 2 launches of a few microseconds per iteration, each iteration streaming
// 18 KB per matrix through L2.  Here one CTA owns one community for all iterations:
//   - X_p (m_p <= 160) sits in shared memory, row stride ld_p + 4 doubles (conflict-free 64-bit fragment loads);
//   - Y = X X^T on FP64 tensor cores (mma.sync.m8n8k4.f64): a work unit is one 8-row block x up to four 8-column blocks
//     on or above the diagonal, the units are dealt round robin to the 16 warps (at most 4 each), accumulators stay in
//     registers until every warp has finished reading X, then X is overwritten in place (direct + mirrored store).
//     Rows and columns beyond m_p are zero in shared memory and stay zero under both updates: no predicates;
//   - the global traces need one grid-wide exchange per iteration (P:L90 pre-sets the sequence to avoid it; north_star
//     takes the decision from the trace).  <= 16 communities: the grid is one thread-block cluster, every CTA stores its
//     (t1_p, t2_p) into each peer's shared memory (DSMEM) and the hardware cluster barrier orders it.  More communities
//     (cooperative launch: all CTAs are co-resident): the pairs go to global memory, the CTAs arrive at a counter with
//     a release reduction and acquire it.  Either way EVERY CTA sums all pairs in the same fixed order and takes the same
//     decision - no broadcast, no floating-point atomics, reproducible.  The squaring does not depend on the branch and
//     runs between arrive and wait;
//   - with a pre-determined sequence and no per-iteration trace log (gbe_density_preset, trace_every_iteration = 0)
//     the CTAs never communicate: a plain launch, any number of communities.
// Bound: latency (the grid barrier, ~2 us per iteration) - the FP64 work of config 1 is under 1 us per iteration.
#include <cooperative_groups.h>

#include "gbe_internal.cuh"

namespace {
namespace cg = cooperative_groups;

constexpr int RS_WARPS = 16;
constexpr int RS_THREADS = RS_WARPS * 32;
constexpr int RS_MAXU = 4;    // work units per warp
constexpr int RS_UCOLS = 4;   // 8-column blocks per unit
constexpr int RS_MAX_UNITS = RS_WARPS * RS_MAXU;
constexpr int RS_CLUSTER_MAX = 16;  // largest thread-block cluster (non-portable size)

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
  unsigned v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// All CTAs of the (cooperative) grid arrive; `target` = arrivals expected since the counter was reset by k_init_state.
// The grid barrier is split: arrive (release: the partials this thread wrote are visible before the arrival) and wait
// (acquire: those of the others after it), so that work that does not depend on the exchange runs in between.
// (An exchange without the counter - every CTA polling one epoch flag per community - was measured slower: n_part^2
// acquire loads per iteration; 369 us instead of 229 us per 40 iterations at 148 communities.)
__device__ __forceinline__ void grid_arrive(unsigned* bar) {
  asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
}
__device__ __forceinline__ void grid_wait(const unsigned* bar, unsigned target) {
  while (ld_acquire(bar) < target) {}
}

// upper-triangle work units of an R x R grid of 8 x 8 blocks
__host__ __device__ inline int rs_units(int R) {
  int n = 0;
  for (int bi = 0; bi < R; ++bi) n += (R - bi + RS_UCOLS - 1) / RS_UCOLS;
  return n;
}

template <int NB>
__device__ __forceinline__ void rs_unit_mma(double (&acc)[RS_UCOLS][2], const double* __restrict__ pa,
                                            const double* __restrict__ pb, int ld, int stride) {
#pragma unroll 4
  for (int k0 = 0; k0 < ld; k0 += 4) {
    const double a = pa[k0];
    double b[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) b[j] = pb[j * 8 * stride + k0];
#pragma unroll
    for (int j = 0; j < NB; ++j) dmma884(acc[j][0], acc[j][1], a, b[j]);
  }
}

// mode 0: branch from the global trace; 1: preset sequence, traces logged every iteration (both: cooperative launch);
// mode 2: preset sequence, no exchange; the final partials go to partials[p] for one k_trace_branch launch afterwards.
__global__ void __launch_bounds__(RS_THREADS, 1)
    k_sp2_resident(const int32_t* __restrict__ msize, const int32_t* __restrict__ ncore,
                   const int64_t* __restrict__ dense_off, gbe_state* st, double* X0, double* X1, double* partials,
                   int n_part, int mode, int cl) {
  extern __shared__ __align__(16) double xs[];  // R8 rows x stride
  __shared__ double red[2 * RS_WARPS];
  __shared__ double tot[2];
  __shared__ short2 units[RS_MAX_UNITS];
  __shared__ int n_units_s;
  __shared__ double cl_slots[2][RS_CLUSTER_MAX][2];  // [iteration parity][community] = (t1, t2), written by the peers

  const int p = blockIdx.x;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, g = lane >> 2, q = lane & 3;
  const int m = msize[p], nc = ncore[p];
  const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN, stride = ld + 4;
  const int R = (m + 7) >> 3;
  const int64_t doff = dense_off[p];
  const int iters = st->iters;
  const double n_occ = st->n_occ, idem_tol = st->idem_tol;

  // ---- load X_0 (written by the gather), zero the rows [m, 8R)
  {
    const double2* __restrict__ src = reinterpret_cast<const double2*>(X0 + doff);
    const int h = ld >> 1;
    for (int i = t; i < m * h; i += RS_THREADS) {
      const int r = i / h, c2 = i - r * h;
      *reinterpret_cast<double2*>(xs + (size_t)r * stride + 2 * c2) = src[i];
    }
    for (int i = m * stride + t; i < 8 * R * stride; i += RS_THREADS) xs[i] = 0.0;
    if (t == 0) {
      int n = 0;
      for (int bi = 0; bi < R; ++bi)
        for (int bj = bi; bj < R; bj += RS_UCOLS) units[n++] = make_short2((short)bi, (short)bj);
      n_units_s = n;
    }
  }
  __syncthreads();
  const int n_units = n_units_s;
  // distributed shared memory may only be touched once every CTA of the cluster has started executing
  if (cl) cg::this_cluster().sync();

  // (t1_p, t2_p) of the X in shared memory: core diagonal and squared core rows (Tr_core X^2 for symmetric X);
  // the result is valid in every lane of warp 0
  auto core_traces = [&](double& o1, double& o2) {
    double s1 = 0.0, s2 = 0.0;
    for (int i = wid; i < nc; i += RS_WARPS) {
      const double* __restrict__ row = xs + (size_t)i * stride;
      for (int c = lane; c < ld; c += 32) {
        const double x = row[c];
        s2 += x * x;
        if (c == i) s1 += x;
      }
    }
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) { red[wid] = s1; red[RS_WARPS + wid] = s2; }
    __syncthreads();
    if (wid == 0) {  // every lane of warp 0 ends up with both sums (fixed butterfly order)
      o1 = warp_sum(lane < RS_WARPS ? red[lane] : 0.0);
      o2 = warp_sum(lane < RS_WARPS ? red[RS_WARPS + lane] : 0.0);
    }
  };

  // One update X <- X^2 (b = 0) or 2X - X^2 (b = 1), in place, in two halves: square() forms this warp's part of
  // Y = X X^T in registers and does not depend on the branch, so it runs while the traces of the other communities are
  // still on their way; apply(b) overwrites X once every warp of the CTA is done reading it (a barrier in between).
  double acc[RS_MAXU][RS_UCOLS][2];
  auto square = [&]() {
#pragma unroll
    for (int u = 0; u < RS_MAXU; ++u)
#pragma unroll
      for (int j = 0; j < RS_UCOLS; ++j) acc[u][j][0] = acc[u][j][1] = 0.0;
#pragma unroll
    for (int u = 0; u < RS_MAXU; ++u) {
      const int ui = wid + u * RS_WARPS;
      if (ui < n_units) {
        const short2 un = units[ui];
        const int nb = min(RS_UCOLS, R - un.y);
        const double* pa = xs + (size_t)(un.x * 8 + g) * stride + q;
        const double* pb = xs + (size_t)(un.y * 8 + g) * stride + q;
        switch (nb) {
          case 4: rs_unit_mma<4>(acc[u], pa, pb, ld, stride); break;
          case 3: rs_unit_mma<3>(acc[u], pa, pb, ld, stride); break;
          case 2: rs_unit_mma<2>(acc[u], pa, pb, ld, stride); break;
          default: rs_unit_mma<1>(acc[u], pa, pb, ld, stride); break;
        }
      }
    }
  };
  auto apply = [&](int b) {
#pragma unroll
    for (int u = 0; u < RS_MAXU; ++u) {
      const int ui = wid + u * RS_WARPS;
      if (ui < n_units) {
        const short2 un = units[ui];
        const int nb = min(RS_UCOLS, R - un.y);
        const int r = un.x * 8 + g;
#pragma unroll
        for (int j = 0; j < RS_UCOLS; ++j) {
          if (j < nb) {
            const int c = (un.y + j) * 8 + 2 * q;
            double* xr = xs + (size_t)r * stride + c;
            double v0 = acc[u][j][0], v1 = acc[u][j][1];
            if (b) {  // only this lane touches (r, c), (r, c + 1) and their mirror images
              const double2 x = *reinterpret_cast<const double2*>(xr);
              v0 = 2.0 * x.x - v0;
              v1 = 2.0 * x.y - v1;
            }
            *reinterpret_cast<double2*>(xr) = make_double2(v0, v1);
            if (un.y + j != un.x) {  // off-diagonal block: mirror (the diagonal block is computed whole)
              xs[(size_t)c * stride + r] = v0;
              xs[(size_t)(c + 1) * stride + r] = v1;
            }
          }
        }
      }
    }
    __syncthreads();
  };

  double* const pbuf[2] = {partials, partials + 2 * (size_t)n_part};
  int k = 0;
  if (mode == 2) {  // pre-determined sequence, no exchange
    for (; k < iters; ++k) {
      square();
      __syncthreads();
      apply((int)st->br[k]);
    }
    double a = 0.0, b = 0.0;
    core_traces(a, b);
    if (t == 0) { partials[2 * (size_t)p] = a; partials[2 * (size_t)p + 1] = b; }
  } else {
    unsigned arrivals = 0;
    for (;;) {
      double a = 0.0, b = 0.0, t1, t2;
      core_traces(a, b);
      if (cl) {
        // <= 16 communities: the grid is ONE thread-block cluster; the sums travel through distributed shared memory and
        // the hardware cluster barrier (arrive.release / wait.acquire) replaces the round trips through L2
        cg::cluster_group cluster = cg::this_cluster();
        if (t < n_part) {  // lanes of warp 0: lane t delivers this community's pair to peer t
          double* dst = cluster.map_shared_rank(&cl_slots[k & 1][p][0], t);
          dst[0] = a;
          dst[1] = b;
        }
        __syncwarp();  // the cluster barrier is .aligned: warp 0 must be converged again
        cluster.barrier_arrive();
        if (k < iters) square();
        cluster.barrier_wait();  // every peer's pair has landed here
        __syncthreads();         // every warp is done reading X_k (the arrivals were counted BEFORE the squaring)
        // every warp sums the pairs itself, in the same butterfly order: no broadcast, no further barrier
        t1 = warp_sum(lane < n_part ? cl_slots[k & 1][lane][0] : 0.0);
        t2 = warp_sum(lane < n_part ? cl_slots[k & 1][lane][1] : 0.0);
      } else {
        double* pb = pbuf[k & 1];
        arrivals += gridDim.x;
        if (t == 0) {
          pb[2 * (size_t)p] = a;
          pb[2 * (size_t)p + 1] = b;
          grid_arrive(&st->bar);
        }
        if (k < iters) square();  // Y = X_k X_k^T, whichever branch is taken (unused if the idempotency stop fires)
        if (t == 0) grid_wait(&st->bar, arrivals);
        __syncthreads();  // all partials are visible; every warp is done reading X_k
        if (wid == 0) {  // the same fixed-order sum of all partials in every CTA, read from L2 by one warp
          double s1 = 0.0, s2 = 0.0;
          const double2* __restrict__ p2 = reinterpret_cast<const double2*>(pb);
          for (int i = lane; i < n_part; i += 32) {
            const double2 v = __ldcg(p2 + i);
            s1 += v.x;
            s2 += v.y;
          }
          s1 = warp_sum(s1);
          s2 = warp_sum(s2);
          if (lane == 0) { tot[0] = s1; tot[1] = s2; }
        }
        __syncthreads();
        t1 = tot[0];
        t2 = tot[1];
      }
      const bool stop = k >= iters || (idem_tol >= 0.0 && k >= 1 && fabs(t1 - t2) <= idem_tol);
      int br = 0;
      if (!stop) br = mode == 1 ? (int)st->br[k] : ((fabs(t2 - n_occ) < fabs(2.0 * t1 - t2 - n_occ)) ? 0 : 1);
      if (p == 0 && t == 0) {  // the log, exactly as k_trace_branch keeps it
        st->t1[k] = t1;
        st->t2[k] = t2;
        st->iters_done = k;
        if (stop) {
          st->stop = 1;
        } else {
          st->branch = br;
          st->br[k] = (uint8_t)br;
          st->iter = k + 1;
        }
      }
      if (stop) break;
      apply(br);
      ++k;
    }
  }

  // ---- the final X goes to buffer (updates applied) & 1, where the scatter looks for it
  {
    double2* __restrict__ dst = reinterpret_cast<double2*>(((k & 1) ? X1 : X0) + doff);
    const int h = ld >> 1;
    for (int i = t; i < m * h; i += RS_THREADS) {
      const int r = i / h, c2 = i - r * h;
      dst[i] = *reinterpret_cast<const double2*>(xs + (size_t)r * stride + 2 * c2);
    }
  }
}

size_t rs_smem_bytes(int max_m) {
  const int ld = (max_m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  const int R = (max_m + 7) / 8;
  return (size_t)std::max(1, 8 * R) * (ld + 4) * sizeof(double);
}
}  // namespace

// Can the resident kernel hold the largest community of this graph, and how many CTAs are co-resident on the device?
int gbe_resident_capacity(const gbe_graph* g, int* fits, int* coresident, int* cluster) {
  *fits = 0;
  *coresident = 0;
  *cluster = 0;
  if (g->n_part <= 0 || g->max_m <= 0) return GBE_OK;
  if (rs_units((g->max_m + 7) / 8) > RS_MAX_UNITS) return GBE_OK;
  int dev = 0, smem_max = 0, sms = 0;
  GBE_CUDA(cudaGetDevice(&dev));
  GBE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  GBE_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t smem = rs_smem_bytes(g->max_m);
  cudaFuncAttributes fa;
  GBE_CUDA(cudaFuncGetAttributes(&fa, k_sp2_resident));
  if (smem + fa.sharedSizeBytes > (size_t)smem_max) return GBE_OK;  // dynamic + the kernel's static shared memory
  GBE_CUDA(cudaFuncSetAttribute(k_sp2_resident, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  GBE_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sp2_resident, RS_THREADS, smem));
  *fits = per_sm > 0;
  *coresident = per_sm * sms;
  *cluster = 0;
  if (*fits && g->n_part <= RS_CLUSTER_MAX) {  // can one cluster of n_part CTAs be scheduled?
    GBE_CUDA(cudaFuncSetAttribute(k_sp2_resident, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(g->n_part);
    cfg.blockDim = dim3(RS_THREADS);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)g->n_part;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    int n_clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&n_clusters, k_sp2_resident, &cfg) == cudaSuccess) *cluster = n_clusters > 0;
    else (void)cudaGetLastError();
  }
  return GBE_OK;
}

int gbe_launch_sp2_resident(const gbe_graph* g, gbe_state* st, double* X0, double* X1, double* partials, int mode,
                            cudaStream_t s) {
  const size_t smem = rs_smem_bytes(g->max_m);
  GBE_CUDA(cudaFuncSetAttribute(k_sp2_resident, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int32_t* msize = g->msize;
  const int32_t* ncore = g->ncore;
  const int64_t* doff = g->dense_off;
  int n_part = g->n_part;
  int cl = 0;
  if (mode == 2) {
    k_sp2_resident<<<n_part, RS_THREADS, smem, s>>>(msize, ncore, doff, st, X0, X1, partials, n_part, mode, cl);
  } else if (g->resident_cluster) {
    // one thread-block cluster holds every community: exchange through distributed shared memory
    cl = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(n_part);
    cfg.blockDim = dim3(RS_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)n_part;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, k_sp2_resident, msize, ncore, doff, st, X0, X1, partials, n_part, mode, cl);
    if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources) {
      (void)cudaGetLastError();
      return GBE_RESIDENT_UNAVAILABLE;
    }
    GBE_CUDA(e);
  } else {
    void* args[] = {&msize, &ncore, &doff, &st, &X0, &X1, &partials, &n_part, &mode, &cl};
    // the co-residency was established at build time on an otherwise idle device: if the device is shared now and the
    // grid no longer fits, the caller falls back to the kernels that need no grid barrier
    const cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_sp2_resident, dim3(n_part), dim3(RS_THREADS), args, smem, s);
    if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources) {
      (void)cudaGetLastError();
      return GBE_RESIDENT_UNAVAILABLE;
    }
    GBE_CUDA(e);
  }
  GBE_LAUNCHED();
  return GBE_OK;
}
