// Step 4 - one SP2 iteration over the whole batch (row 4): the dense contraction of the path.
//
//     Y_p = X_p X_p for every community p;  X_p <- Y_p  or  2 X_p - Y_p        (obs. (x) P:L65)
// with the SAME branch for every p, read from the device-side state written by step 5.
//
// X_p is symmetric, so Y = X X^T: both operand panels are ROW panels of X (K contiguous, identical load
// pattern, no transpose) and only the upper triangle is computed; the result is mirrored on store.
// FP64 tensor cores: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4 - tcgen05 has no f64 kind).  The DMMA pipe is the
// bound (37 TFLOP/s measured, one DMMA per 16 cycles per SM sub-partition), so the design spends everything else
// to keep that pipe on USEFUL flops:
//   - 64x64 CTA tiles, 4 warps of 32x32 (16 accumulator pairs), 3 CTAs per SM: the epilogue of one CTA (stores,
//     mirrored stores, the X read of the 2X - X^2 branch) overlaps the main loops of the other two;
//   - work skipped at 8x8 granularity with warp-uniform masks: sub-tiles strictly below the diagonal (their values
//     arrive by the mirrored store) and sub-tiles beyond the ragged edge m_p.  Executed flops ~ 0.52 x 2 m^3;
//   - in a diagonal CTA the warp whose 32x32 block lies below the diagonal is idle; the warp -> block map rotates
//     with the CTA index so that the idle warp does not always sit on the same SM sub-partition;
//   - panels staged by a 3-stage cp.async pipeline in 128-byte rows (K chunk = 16 doubles), read with conflict-free
//     64-bit loads (row stride 20 doubles).  Loads of rows >= m_p are zero-filled, stores predicated; pad columns
//     [m_p, ld_p) stay zero by construction.
//
// Fused epilogue (warp-shuffle partials, north_star item 3): while X_{n+1} is written, accumulate over the core
// rows  t1 = sum_i X_ii  and  t2 = sum_i sum_c X_ic^2 (= Tr_core(X^2) for symmetric X), one fixed-order partial
// per work item, so that the branch of the NEXT iteration is known before its GEMM starts.
// Bound: FP64 tensor pipe - 2 m^3 algorithmic flop per community per iteration (~m^3 executed thanks to symmetry).
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

constexpr int X2_BT = 64;       // CTA tile edge
constexpr int X2_WT = 32;       // warp tile edge (2 x 2 warps)
constexpr int X2_THREADS = 128;

template <int STAGES>
__global__ void __launch_bounds__(X2_THREADS, 3)
    k_x2(const gbe_tile_item* __restrict__ items, const int64_t* __restrict__ sub_ptr,
         const int32_t* __restrict__ ncore_arr, const int64_t* __restrict__ dense_off,
         const gbe_state* __restrict__ st, const double* __restrict__ Xin, double* __restrict__ Xout,
         double* __restrict__ partials) {
  constexpr int SUB = X2_WT / 8;  // 4 x 4 sub-tiles of 8 x 8 per warp
  constexpr int STAGE_ELEMS = 2 * X2_BT * X2_STRIDE;
  extern __shared__ __align__(16) double smem[];
  __shared__ double red[8];

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
  const int row0 = ti * X2_BT, col0 = tj * X2_BT;
  const int nchunks = ld / GBE_KC;

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int role = (wid + blockIdx.x) & 3;  // rotate: the idle warp of a diagonal CTA changes sub-partition
  const int wm = role >> 1, wn = role & 1;
  const int g = lane >> 2, q = lane & 3;
  const int wr0 = row0 + wm * X2_WT, wc0 = col0 + wn * X2_WT;  // first row / column of the warp tile

  // warp-uniform masks over the 4 x 4 sub-tiles: bit (i * 4 + j)
  //   active: rows < m, columns < ld, and not strictly below the diagonal;  mirrored: strictly above the diagonal
  unsigned active = 0, mirror = 0;
#pragma unroll
  for (int i = 0; i < SUB; ++i)
#pragma unroll
    for (int j = 0; j < SUB; ++j) {
      const int r8 = wr0 + 8 * i, c8 = wc0 + 8 * j;
      if (r8 < m && c8 < ld && r8 <= c8) {
        active |= 1u << (i * 4 + j);
        if (r8 < c8) mirror |= 1u << (i * 4 + j);
      }
    }

  auto load_stage = [&](int stage, int kc) {
    double* sA = smem + (size_t)stage * STAGE_ELEMS;
    double* sB = sA + X2_BT * X2_STRIDE;
    const int k0 = kc * GBE_KC;
#pragma unroll
    for (int c = t; c < X2_BT * 8; c += X2_THREADS) {
      const int r = c >> 3, ch = c & 7;
      const int gr = row0 + r;
      const bool ok = gr < m;
      cp_async16(sA + r * X2_STRIDE + ch * 2, X + (size_t)(ok ? gr : 0) * ld + k0 + ch * 2, ok);
    }
    if (!diag) {
#pragma unroll
      for (int c = t; c < X2_BT * 8; c += X2_THREADS) {
        const int r = c >> 3, ch = c & 7;
        const int gr = col0 + r;
        const bool ok = gr < m;
        cp_async16(sB + r * X2_STRIDE + ch * 2, X + (size_t)(ok ? gr : 0) * ld + k0 + ch * 2, ok);
      }
    }
  };

  double acc[SUB][SUB][2];
#pragma unroll
  for (int i = 0; i < SUB; ++i)
#pragma unroll
    for (int j = 0; j < SUB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

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
    if (active == 0) continue;  // warp-uniform: this warp's block lies below the diagonal or beyond the edge
    const double* sA = smem + (size_t)(kc % STAGES) * STAGE_ELEMS;
    const double* sB = diag ? sA : sA + X2_BT * X2_STRIDE;
    const double* pa = sA + (wm * X2_WT + g) * X2_STRIDE + q;
    const double* pb = sB + (wn * X2_WT + g) * X2_STRIDE + q;
    if (active == 0xFFFFu) {
#pragma unroll
      for (int ks = 0; ks < GBE_KC / 4; ++ks) {
        double a[SUB], b[SUB];
#pragma unroll
        for (int i = 0; i < SUB; ++i) a[i] = pa[i * 8 * X2_STRIDE + ks * 4];
#pragma unroll
        for (int j = 0; j < SUB; ++j) b[j] = pb[j * 8 * X2_STRIDE + ks * 4];
#pragma unroll
        for (int i = 0; i < SUB; ++i)
#pragma unroll
          for (int j = 0; j < SUB; ++j) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
      }
    } else {
#pragma unroll
      for (int ks = 0; ks < GBE_KC / 4; ++ks) {
        double a[SUB], b[SUB];
#pragma unroll
        for (int i = 0; i < SUB; ++i) a[i] = pa[i * 8 * X2_STRIDE + ks * 4];
#pragma unroll
        for (int j = 0; j < SUB; ++j) b[j] = pb[j * 8 * X2_STRIDE + ks * 4];
#pragma unroll
        for (int i = 0; i < SUB; ++i)
#pragma unroll
          for (int j = 0; j < SUB; ++j)
            if (active & (1u << (i * 4 + j))) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
      }
    }
  }
  cp_async_wait<0>();

  // epilogue: X_{n+1} = Y or 2 X_n - Y, direct + mirrored store, core-row trace partials
  double s1 = 0.0, s2 = 0.0;
#pragma unroll
  for (int i = 0; i < SUB; ++i) {
    const int r = wr0 + i * 8 + g;
#pragma unroll
    for (int j = 0; j < SUB; ++j) {
      if (!(active & (1u << (i * 4 + j)))) continue;
      const int c = wc0 + j * 8 + 2 * q;
      if (r < m) {  // c < ld holds for every active sub-tile
        double v0 = acc[i][j][0], v1 = acc[i][j][1];
        if (branch) {
          const double2 x = *reinterpret_cast<const double2*>(X + (size_t)r * ld + c);
          v0 = 2.0 * x.x - v0;
          v1 = 2.0 * x.y - v1;
        }
        *reinterpret_cast<double2*>(Y + (size_t)r * ld + c) = make_double2(v0, v1);
        if (r < nc) {
          s2 += v0 * v0 + v1 * v1;
          if (r == c) s1 += v0;
          if (r == c + 1) s1 += v1;
        }
        if (mirror & (1u << (i * 4 + j))) {
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
  if (lane == 0) { red[role] = s1; red[4 + role] = s2; }  // indexed by block position: order independent of the rotation
  __syncthreads();
  if (t == 0) {
    partials[2 * (size_t)blockIdx.x] = (red[0] + red[1]) + (red[2] + red[3]);
    partials[2 * (size_t)blockIdx.x + 1] = (red[4] + red[5]) + (red[6] + red[7]);
  }
}

}  // namespace

int gbe_launch_x2(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                  cudaStream_t s) {
  (void)iter;
  if (g->n_items == 0) return GBE_OK;
  constexpr int STAGES = 3;
  auto kern = k_x2<STAGES>;
  const size_t smem = (size_t)STAGES * 2 * X2_BT * X2_STRIDE * sizeof(double);
  static bool configured = false;
  if (!configured) {
    GBE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    GBE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    configured = true;
  }
  kern<<<g->n_items, X2_THREADS, smem, s>>>(g->items, g->sub_ptr, g->ncore, g->dense_off, st, Xin, Xout, partials);
  GBE_LAUNCHED();
  return GBE_OK;
}
