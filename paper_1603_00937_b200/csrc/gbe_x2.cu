// Step 4 - one SP2 iteration over the whole batch (row 4): the dense contraction of the path.
//
//     Y_p = X_p X_p for every community p;  X_p <- Y_p  or  2 X_p - Y_p        (obs. (x) P:L65)
// with the SAME branch for every p, read from the device-side state written by step 5.
//
// X_p is symmetric, so Y = X X^T: both operand panels are ROW panels of X (K contiguous, identical load
// pattern, no transpose) and only tiles (ti <= tj) are computed; the result is mirrored on store.
// FP64 tensor cores: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4 - tcgen05 has no f64 kind), fed from shared memory
// with conflict-free 64-bit loads (row stride 20 doubles), panels staged by a 4-stage cp.async pipeline in
// 128-byte rows (K chunk = 16 doubles).  Ragged edges: loads of rows >= m_p are zero-filled, stores predicated;
// pad columns [m_p, ld_p) stay zero by construction.
//
// Fused epilogue (warp-shuffle partials, north_star item 3): while X_{n+1} is written, accumulate over the core
// rows  t1 = sum_i X_ii  and  t2 = sum_i sum_c X_ic^2 (= Tr_core(X^2) for symmetric X), one fixed-order partial
// per work item, so that the branch of the NEXT iteration is known before its GEMM starts.
// Bound: FP64 tensor pipe - 2 m^3 algorithmic flop per community per iteration (m^3 executed thanks to symmetry).
#include "gbe_internal.cuh"

namespace {

constexpr int X2_STRIDE = GBE_KC + 4;  // doubles per shared-memory row: 20 -> 8*row mod 32 banks, conflict-free

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, bool pred) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  const int sz = pred ? 16 : 0;  // src-size 0: the 16 bytes are zero-filled
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

// CTA tile BM x BN, WARPS_M x WARPS_N warps, warp tile (BM/WARPS_M) x (BN/WARPS_N)
template <int BM, int BN, int WARPS_M, int WARPS_N, int STAGES>
__global__ void __launch_bounds__(WARPS_M* WARPS_N * 32, 1)
    k_x2(const gbe_tile_item* __restrict__ items, const int64_t* __restrict__ sub_ptr,
         const int32_t* __restrict__ ncore_arr, const int64_t* __restrict__ dense_off,
         const gbe_state* __restrict__ st, const double* __restrict__ Xin, double* __restrict__ Xout,
         double* __restrict__ partials) {
  static_assert(BM == BN, "square tiles: the mirror store assumes it");
  constexpr int NT = WARPS_M * WARPS_N * 32;
  constexpr int WM = BM / WARPS_M, WN = BN / WARPS_N;
  constexpr int MI = WM / 8, NJ = WN / 8;
  constexpr int STAGE_ELEMS = (BM + BN) * X2_STRIDE;
  extern __shared__ __align__(16) double smem[];
  __shared__ double red[2 * WARPS_M * WARPS_N];

  if (st->stop) return;  // idempotency stop already fired (A-7): X is final
  const int branch = st->branch;

  const gbe_tile_item it = items[blockIdx.x];
  const int p = it.p, ti = it.ti, tj = it.tj;
  const int m = (int)(sub_ptr[p + 1] - sub_ptr[p]);
  const int nc = ncore_arr[p];
  const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  const double* __restrict__ X = Xin + dense_off[p];
  double* __restrict__ Y = Xout + dense_off[p];
  const bool diag = (ti == tj);
  const int row0 = ti * BM, col0 = tj * BN;
  const int nchunks = ld / GBE_KC;

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int wm = wid / WARPS_N, wn = wid % WARPS_N;
  const int g = lane >> 2, q = lane & 3;

  auto load_stage = [&](int stage, int kc) {
    double* sA = smem + (size_t)stage * STAGE_ELEMS;
    double* sB = sA + BM * X2_STRIDE;
    const int k0 = kc * GBE_KC;
#pragma unroll
    for (int c = t; c < BM * 8; c += NT) {
      const int r = c >> 3, ch = c & 7;
      const int gr = row0 + r;
      const bool ok = gr < m;
      cp_async16(sA + r * X2_STRIDE + ch * 2, X + (size_t)(ok ? gr : 0) * ld + k0 + ch * 2, ok);
    }
    if (!diag) {
#pragma unroll
      for (int c = t; c < BN * 8; c += NT) {
        const int r = c >> 3, ch = c & 7;
        const int gr = col0 + r;
        const bool ok = gr < m;
        cp_async16(sB + r * X2_STRIDE + ch * 2, X + (size_t)(ok ? gr : 0) * ld + k0 + ch * 2, ok);
      }
    }
  };

  double acc[MI][NJ][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int j = 0; j < NJ; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // prologue
#pragma unroll
  for (int s = 0; s < STAGES - 1; ++s) {
    if (s < nchunks) load_stage(s, s);
    cp_async_commit();
  }

  for (int kc = 0; kc < nchunks; ++kc) {
    cp_async_wait<STAGES - 2>();
    __syncthreads();
    {
      const int nk = kc + STAGES - 1;
      if (nk < nchunks) load_stage(nk % STAGES, nk);
      cp_async_commit();
    }
    const double* sA = smem + (size_t)(kc % STAGES) * STAGE_ELEMS;
    const double* sB = diag ? sA : sA + BM * X2_STRIDE;
    const double* pa = sA + (wm * WM + g) * X2_STRIDE + q;
    const double* pb = sB + (wn * WN + g) * X2_STRIDE + q;
#pragma unroll
    for (int ks = 0; ks < GBE_KC / 4; ++ks) {
      double a[MI], b[NJ];
#pragma unroll
      for (int i = 0; i < MI; ++i) a[i] = pa[i * 8 * X2_STRIDE + ks * 4];
#pragma unroll
      for (int j = 0; j < NJ; ++j) b[j] = pb[j * 8 * X2_STRIDE + ks * 4];
#pragma unroll
      for (int i = 0; i < MI; ++i)
#pragma unroll
        for (int j = 0; j < NJ; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
    }
  }
  cp_async_wait<0>();

  // epilogue: X_{n+1} = Y or 2 X_n - Y, mirrored store, core-row trace partials
  double s1 = 0.0, s2 = 0.0;
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int r = row0 + wm * WM + i * 8 + g;
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int c = col0 + wn * WN + j * 8 + 2 * q;
      if (r < m && c < ld) {
        double v0 = acc[i][j][0], v1 = acc[i][j][1];
        if (branch) {
          const double2 x = *reinterpret_cast<const double2*>(X + (size_t)r * ld + c);
          v0 = 2.0 * x.x - v0;
          v1 = 2.0 * x.y - v1;
        }
        *reinterpret_cast<double2*>(Y + (size_t)r * ld + c) = make_double2(v0, v1);
        if (r < nc) {
          s2 += v0 * v0 + v1 * v1;
          if (diag) {
            if (r == c) s1 += v0;
            if (r == c + 1) s1 += v1;
          }
        }
        if (!diag) {
          if (c < m) {
            Y[(size_t)c * ld + r] = v0;
            if (c < nc) s2 += v0 * v0;
          }
          if (c + 1 < m) {
            Y[(size_t)(c + 1) * ld + r] = v1;
            if (c + 1 < nc) s2 += v1 * v1;
          }
        }
      }
    }
  }
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) { red[wid] = s1; red[WARPS_M * WARPS_N + wid] = s2; }
  __syncthreads();
  if (t == 0) {
    double a1 = 0.0, a2 = 0.0;
#pragma unroll
    for (int w = 0; w < WARPS_M * WARPS_N; ++w) { a1 += red[w]; a2 += red[WARPS_M * WARPS_N + w]; }
    partials[2 * (size_t)blockIdx.x] = a1;
    partials[2 * (size_t)blockIdx.x + 1] = a2;
  }
}

}  // namespace

int gbe_launch_x2(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                  cudaStream_t s) {
  (void)iter;
  if (g->n_items == 0) return GBE_OK;
  constexpr int BM = 128, WMN = 2, WNN = 4, STAGES = 4;
  auto kern = k_x2<BM, BM, WMN, WNN, STAGES>;
  const size_t smem = (size_t)STAGES * (BM + BM) * X2_STRIDE * sizeof(double);
  static bool configured = false;
  if (!configured) {
    GBE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = true;
  }
  kern<<<g->n_items, WMN * WNN * 32, smem, s>>>(g->items, g->sub_ptr, g->ncore, g->dense_off, st, Xin, Xout, partials);
  GBE_LAUNCHED();
  return GBE_OK;
}
