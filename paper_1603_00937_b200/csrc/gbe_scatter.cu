// Step 6 - core-column scatter (row 6).
//
//     D[s_p[r], s_p[c]] = (X_p)[r, c],  r < m_p, c < ncore_p                                (A-9, A-10)
// Column i of P_tau(H) is column j of P(x[s]) (Eq.(6)); P(x[s]) is symmetric, so the kernel reads ROW
// segments instead (contiguous): for dense row (p, r) the ncore_p leading entries go to one contiguous run of
// D.val when every core is an index range, else through a per-entry position map.  D is NOT symmetrised
// (obs. (i) P:L65).  The final X lives in buffer (iters_done & 1) - in buffer 0 when the SP2 loop ran in place - read from
// the device state.
// Bound: HBM - 8 B read + 8 B written per stored entry of D (+ 8 B map in the general case).
// BULK variant (index-range cores, every core size even, D.val 16-byte aligned: every run then is a whole number of
// 16-byte pieces on both sides): the copy engine moves the runs, global -> shared -> global (cp.async.bulk, UBLKCP), one
// run per lane and 32 runs per warp in flight, with no register staging - a persistent grid of one 16-warp CTA per SM
// holds ~200 KB of runs in flight per SM, twice what the register variant reaches, at a fifth of its instructions.
#include "gbe_internal.cuh"

namespace {
template <bool CONTIG>
__global__ void __launch_bounds__(256, 4) k_scatter(int64_t sum_m, const int64_t* __restrict__ row_src,
                                                 const int32_t* __restrict__ row_nc,
                                                 const int64_t* __restrict__ scat_base,
                                                 const int64_t* __restrict__ scat_ofs,
                                                 const int64_t* __restrict__ scat_pos, const gbe_state* __restrict__ st,
                                                 const double* __restrict__ X0, const double* __restrict__ X1,
                                                 double* __restrict__ D_val) {
  const int lane = threadIdx.x & 31;
  const int64_t warp = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5), nwarps = (int64_t)gridDim.x * 8;
  const double* __restrict__ X = (!st->inplace && (st->iters_done & 1)) ? X1 : X0;  // in place: X never left X0
  constexpr int R = 8;  // dense rows per warp iteration: their metadata is fetched by 8 lanes at once and the loads
                        // of all 8 rows are issued before the first store (the kernel is latency bound otherwise)
  for (int64_t q0 = warp * R; q0 < sum_m; q0 += nwarps * R) {
    int nc_l = 0;
    int64_t src_l = 0, dst_l = 0;
    if (lane < R && q0 + lane < sum_m) {
      const int64_t q = q0 + lane;
      nc_l = row_nc[q];
      src_l = row_src[q];
      dst_l = CONTIG ? scat_base[q] : scat_ofs[q];
    }
    // phase 1: all loads of the 8 rows; 16-byte loads when the row can be moved as aligned pairs
    double2 v[R];
    bool vec[R];
#pragma unroll
    for (int l = 0; l < R; ++l) {
      const int nc = __shfl_sync(0xffffffffu, nc_l, l);
      const int64_t so = __shfl_sync(0xffffffffu, src_l, l);
      const int64_t dofs = __shfl_sync(0xffffffffu, dst_l, l);
      const double* src = X + so;  // 128-byte aligned: rows of a dense block start on a line
      vec[l] = CONTIG && nc <= 64 && !(nc & 1) && !((reinterpret_cast<uintptr_t>(D_val + dofs)) & 15);
      v[l] = make_double2(0.0, 0.0);
      if (vec[l]) {
        if (2 * lane < nc) v[l] = *reinterpret_cast<const double2*>(src + 2 * lane);
      } else {
        if (lane < nc) v[l].x = src[lane];
        if (lane + 32 < nc) v[l].y = src[lane + 32];
      }
    }
    // phase 2: all stores
#pragma unroll
    for (int l = 0; l < R; ++l) {
      const int nc = __shfl_sync(0xffffffffu, nc_l, l);
      const int64_t dofs = __shfl_sync(0xffffffffu, dst_l, l);
      if (CONTIG) {
        double* dst = D_val + dofs;
        if (vec[l]) {
          if (2 * lane < nc) *reinterpret_cast<double2*>(dst + 2 * lane) = v[l];
        } else {
          if (lane < nc) dst[lane] = v[l].x;
          if (lane + 32 < nc) dst[lane + 32] = v[l].y;
          if (nc > 64) {
            const double* src = X + __shfl_sync(0xffffffffu, src_l, l);
            for (int c = lane + 64; c < nc; c += 32) dst[c] = src[c];
          }
        }
      } else {
        const int64_t* pos = scat_pos + dofs;
        if (lane < nc) D_val[pos[lane]] = v[l].x;
        if (lane + 32 < nc) D_val[pos[lane + 32]] = v[l].y;
        if (nc > 64) {
          const double* src = X + __shfl_sync(0xffffffffu, src_l, l);
          for (int c = lane + 64; c < nc; c += 32) D_val[pos[c]] = src[c];
        }
      }
    }
  }
}

__device__ __forceinline__ void sc_mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(mbar), "r"(parity)
        : "memory");
  }
}

constexpr int SCB_WARPS = 16;

__global__ void __launch_bounds__(SCB_WARPS * 32, 1)
    k_scatter_bulk(int64_t sum_m, int slot_doubles, const int64_t* __restrict__ row_src, const int32_t* __restrict__ row_nc,
                   const int64_t* __restrict__ scat_base, const gbe_state* __restrict__ st, const double* __restrict__ X0,
                   const double* __restrict__ X1, double* __restrict__ D_val) {
  extern __shared__ __align__(128) double stage[];  // warps x 32 slots of slot_doubles
  __shared__ __align__(8) unsigned long long bars[SCB_WARPS];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const double* __restrict__ X = (!st->inplace && (st->iters_done & 1)) ? X1 : X0;  // in place: X never left X0
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&bars[wid]);
  if (lane == 0) {  // one barrier per warp: every lane arrives once per group of 32 runs
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(32) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncwarp();
  double* const slot = stage + ((size_t)wid * 32 + lane) * slot_doubles;
  const uint32_t slot_s = (uint32_t)__cvta_generic_to_shared(slot);
  uint32_t parity = 0;
  const int64_t stride = (int64_t)gridDim.x * nw * 32;
  int64_t q = ((int64_t)blockIdx.x * nw + wid) * 32 + lane;
  // this lane's run of the first group; inside the loop the next group's is requested before this one is waited for
  int nc = 0;
  int64_t so = 0, dofs = 0;
  if (q < sum_m) { nc = row_nc[q]; so = row_src[q]; dofs = scat_base[q]; }
  for (; q - lane < sum_m; q += stride) {  // (warp-uniform trip count)
    const uint32_t bytes = (uint32_t)nc * 8u;
    const double* const src = X + so;  // 128-byte aligned: rows of a dense block start on a line
    double* const dst = D_val + dofs;
    int nc1 = 0;
    int64_t so1 = 0, dofs1 = 0;
    if (q + stride < sum_m) { nc1 = row_nc[q + stride]; so1 = row_src[q + stride]; dofs1 = scat_base[q + stride]; }
    // the engine has read the slot's previous run
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    if (bytes) {
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(slot_s),
                   "l"(src), "r"(bytes), "r"(bar)
                   : "memory");
    } else {
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
    }
    sc_mbar_wait(bar, parity);  // all 32 runs of the group have landed
    parity ^= 1u;
    if (bytes) {
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(slot_s), "r"(bytes) : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    nc = nc1; so = so1; dofs = dofs1;
  }
  asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // the slots live as long as the CTA
}
}  // namespace

// row0, n_rows: a sub-range of the dense rows (one wave of communities); n_rows < 0: all of them
int gbe_launch_scatter(const gbe_graph* g, const gbe_state* st, const double* X0, const double* X1, double* D_val,
                       cudaStream_t s, int64_t row0, int64_t n_rows) {
  if (n_rows < 0) { row0 = 0; n_rows = g->sum_m; }
  if (n_rows == 0) return GBE_OK;
  const int64_t want = (n_rows + 63) / 64;  // 8 warps x 8 rows per CTA iteration
  const int grid = (int)std::min<int64_t>(want, (int64_t)gbe_sm_count() * 64);
  // bulk variant: index-range cores of even size (every run starts and ends on a 16-byte boundary of D.val) whose 32-run
  // groups fit shared memory at four warps or more
  const int slot_doubles = (g->max_ncore + 1) / 2 * 2;
  const int bulk_warps = slot_doubles > 0 ? (int)std::min<size_t>(SCB_WARPS, (size_t)200 * 1024 / ((size_t)32 * slot_doubles * 8)) : 0;
  if (g->contiguous && g->ncore_all_even && bulk_warps >= 4 && !(reinterpret_cast<uintptr_t>(D_val) & 15) && g->scatter_path != 1) {
    const size_t smem = (size_t)bulk_warps * 32 * slot_doubles * 8;
    GBE_CUDA(cudaFuncSetAttribute(k_scatter_bulk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int64_t groups = (n_rows + 32 * bulk_warps - 1) / (32 * bulk_warps);
    const int bgrid = (int)std::min<int64_t>(groups, gbe_sm_count());
    k_scatter_bulk<<<bgrid, bulk_warps * 32, smem, s>>>(n_rows, slot_doubles, g->row_src + row0, g->row_nc + row0,
                                                        g->scat_base + row0, st, X0, X1, D_val);
  } else if (g->contiguous)
    k_scatter<true><<<grid, 256, 0, s>>>(n_rows, g->row_src + row0, g->row_nc + row0, g->scat_base + row0, nullptr,
                                         nullptr, st, X0, X1, D_val);
  else
    k_scatter<false><<<grid, 256, 0, s>>>(n_rows, g->row_src + row0, g->row_nc + row0, nullptr, g->scat_ofs + row0,
                                          g->scat_pos, st, X0, X1, D_val);
  GBE_LAUNCHED();
  return GBE_OK;
}
