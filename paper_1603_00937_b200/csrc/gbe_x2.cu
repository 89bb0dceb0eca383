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
//   - 64x64 CTA tiles, 4 warps with 16 accumulator pairs each, 4 CTAs per SM: the epilogue of one CTA (stores,
//     mirrored stores, the X read of the 2X - X^2 branch) overlaps the main loops of the other three;
//   - work skipped at 8x8 granularity with warp-uniform masks: sub-tiles strictly below the diagonal (their values
//     arrive by the mirrored store) and sub-tiles beyond the ragged edge m_p.  Executed flops ~ 0.52 x 2 m^3;
//   - a CTA runs in lockstep (one barrier per K chunk), so its four warps - one per SM sub-partition, each with its
//     own DMMA pipe - must carry equal work or the lighter sub-partitions idle: warp w owns the 8-row blocks
//     {w, 7 - w} x all eight 8-column blocks, which gives every warp 9 of the 36 upper-triangle sub-tiles of a
//     diagonal tile and an equal share of a ragged right edge; the map rotates with the CTA index;
//   - measured on B200 (profiles/r01_fp64_peak_probe.md): every non-DMMA ALU instruction a warp issues costs ~1.4
//     cycles of its sub-partition's DMMA pipe (shared-memory loads cost almost nothing), so the main loop is pared
//     down to 64 DMMA + 32 LDS.64 + 8 LDGSTS per K chunk: per-thread copy pointers live in registers, rows beyond
//     the ragged edge are clamped to row m_p - 1 instead of predicated (their products are never stored), stage
//     and K offsets are immediates of a loop unrolled over the two stages, and the sub-tile masks are compile-time
//     patterns (full / upper triangle) with a predicated fallback for edge tiles only;
//   - panels staged by a 2-stage cp.async pipeline in 128-byte rows (K chunk = 16 doubles), read with conflict-free
//     64-bit loads (row stride 20 doubles).  Stores are predicated; pad columns [m_p, ld_p) are written as zeros.
//
// Fused epilogue (warp-shuffle partials, north_star item 3): while X_{n+1} is written, accumulate over the core
// rows  t1 = sum_i X_ii  and  t2 = sum_i sum_c X_ic^2 (= Tr_core(X^2) for symmetric X), one fixed-order partial
// per tile with a core row (packed: the other tiles carry no trace and write none), so that the branch of the NEXT
// iteration is known before its GEMM starts.
// Bound: FP64 tensor pipe - 2 m^3 algorithmic flop per community per iteration (~m^3 executed thanks to symmetry).
#include <cuda.h>

#include <cstdlib>
#include <type_traits>

#include "gbe_internal.cuh"

// Optional instrumentation (python -m paper_1603_00937_b200.build --stamps -> libgbe_stamps.so; bench.py --timeline x2):
// %globaltimer per CTA of k_x2_tma at its start, after its main loop and after its epilogue, plus the SM it ran on, for
// the launches of two consecutive iterations.  Compiled out of libgbe.so.
#ifdef GBE_STAMPS
constexpr int X2_ST_IT0 = 10, X2_ST_ITERS = 2, X2_ST_CTAS = 32768, X2_ST_W = 4;
static __device__ unsigned long long g_x2_stamps[(size_t)X2_ST_ITERS * X2_ST_CTAS * X2_ST_W];
#define X2_STAMP(k)                                                                                             \
  do {                                                                                                          \
    if (threadIdx.x == 0 && iter >= X2_ST_IT0 && iter < X2_ST_IT0 + X2_ST_ITERS && blockIdx.x < X2_ST_CTAS) {   \
      unsigned long long now_;                                                                                  \
      unsigned smid_;                                                                                           \
      asm volatile("mov.u64 %0, %globaltimer;" : "=l"(now_));                                                   \
      asm volatile("mov.u32 %0, %smid;" : "=r"(smid_));                                                         \
      unsigned long long* e_ = g_x2_stamps + ((size_t)(iter - X2_ST_IT0) * X2_ST_CTAS + blockIdx.x) * X2_ST_W;  \
      e_[k] = now_;                                                                                             \
      e_[3] = smid_;                                                                                            \
    }                                                                                                           \
  } while (0)
extern "C" int gbe_stamps_x2(unsigned long long* host, size_t bytes) {
  if (bytes < sizeof(g_x2_stamps)) return -1;
  return (int)cudaMemcpyFromSymbol(host, g_x2_stamps, sizeof(g_x2_stamps));
}
extern "C" int gbe_stamps_x2_shape(int* iter0, int* iters, int* ctas, int* width) {
  *iter0 = X2_ST_IT0; *iters = X2_ST_ITERS; *ctas = X2_ST_CTAS; *width = X2_ST_W;
  return 0;
}
#else
#define X2_STAMP(k) do { } while (0)
#endif

namespace {


__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N)); }

constexpr int X2_BT = 64;       // CTA tile edge
constexpr int X2_THREADS = 128;
constexpr int X2_KC = GBE_KC;                    // K chunk: 16 doubles = one 128-byte line per row
constexpr int X2_STRIDE = X2_KC + 4;             // doubles per shared-memory row: 8 banks mod 32 -> conflict-free LDS.64
constexpr int X2_PANEL = X2_BT * X2_STRIDE;      // doubles per panel per stage
constexpr int X2_STAGE = 2 * X2_PANEL;           // A panel + B panel
constexpr unsigned X2_FULL = 0xFFFFu;

// Sub-tile masks, bit (i * 8 + j): the warp with role w owns the 8-row blocks {w, 7 - w} (i = 0, 1) and all eight
// 8-column blocks j of the 64 x 64 tile.  In a diagonal tile row block b needs the columns j >= b only, so every
// warp has exactly 9 of the 36 upper-triangle sub-tiles: the four warps (one per SM sub-partition) stay balanced.
__host__ __device__ constexpr unsigned x2_diag_mask(int w) {
  return ((0xFFu << w) & 0xFFu) | (((0xFFu << (7 - w)) & 0xFFu) << 8);
}

__host__ __device__ constexpr unsigned x2_cols_mask(int nb) {  // the first nb column blocks of both row blocks
  return ((1u << nb) - 1u) | (((1u << nb) - 1u) << 8);
}

// one K chunk of the warp's 2 x 8 sub-tiles: 4 k-steps of 10 LDS.64 + (up to) 16 DMMA; MASK is a compile-time
// pattern, MASK == 0 means "use the run-time mask"
template <unsigned MASK>
__device__ __forceinline__ void x2_chunk(double (&acc)[2][8][2], const double* __restrict__ pa0,
                                         const double* __restrict__ pa1, const double* __restrict__ pb,
                                         unsigned rt_mask) {
#pragma unroll
  for (int ks = 0; ks < X2_KC / 4; ++ks) {
    double a[2], b[8];
    a[0] = pa0[ks * 4];
    a[1] = pa1[ks * 4];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const bool need = MASK == 0 || ((MASK | (MASK >> 8)) & (1u << j));
      if (need) b[j] = pb[j * 8 * X2_STRIDE + ks * 4];
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (MASK != 0) {
          if (MASK & (1u << (i * 8 + j))) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        } else {
          if (rt_mask & (1u << (i * 8 + j))) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
      }
  }
}

// OP 0: one SP2 iteration, Y = X X^T then X' = Y or 2X - Y (Xin -> Xout).
// OP 1: one step of the Chebyshev recurrence of the finite-temperature expansion (Eq.(7); Eq.(5) P:L51-56 with
//       its alpha_n): T_{n+1} = 2 Xt T_n - T_{n-1}, D += c_{n+1} T_{n+1}.  Xin = Xt (A operand), Xb = T_n (B operand),
//       Xout holds T_{n-1} on entry and T_{n+1} on exit (every element is read and written by the same thread), Dacc
//       the running sum, coef[iter] = c_{n+1}.  Xt and T_n are symmetric and commute, so the product is symmetric and
//       the same upper-triangle / mirrored-store scheme applies; only the B panel now comes from another matrix.
template <int MINB, int OP, bool HYB>
__global__ void __launch_bounds__(X2_THREADS, MINB)
    k_x2(const gbe_tile_item* __restrict__ items, const gbe_state* __restrict__ st, const double* __restrict__ Xin,
         double* __restrict__ Xout, double* __restrict__ partials, int iter, const double* __restrict__ Xb,
         double* __restrict__ Dacc, const double* __restrict__ coef) {
  extern __shared__ __align__(16) double smem[];  // 2 stages x (A panel, B panel)
  __shared__ double red[8];

  // programmatic dependent launch (gbe_internal.cuh): the next kernel of the stream (k_trace_branch, or the packed
  // kernel) may become resident from here on; it waits for this grid in its own code.  This kernel itself never waits:
  // launched behind k_trace_branch with the attribute it starts when that kernel lets it go - AFTER it has waited for
  // the previous X^2 launch, taken the decision and fenced - so X_n, the branch and the stop flag are all final.  The
  // state is read with uncached loads (a line of it may sit in this SM's L1 from the previous launch), requested here
  // and looked at after the tile's own set-up so that their latency costs nothing.
  gbe_griddep_launch();
  // hyb (mixed graph: this launch runs next to the packed launch of the same iteration, whose first bin takes the
  // decision): until the branch of THIS iteration is published (iter advanced) or the stop flag is up
  if (OP == 0 && HYB)
    while (gbe_ld_acquire(&st->iter) != iter + 1 && !gbe_ld_state(&st->stop)) __nanosleep(200);
  const int stop0 = OP == 0 ? gbe_ld_state(&st->stop) : 0;
  const int br_preset = OP == 0 ? gbe_ld_state(&st->preset) : 0;
  const int br_given = OP == 0 && iter < GBE_MAX_ITERS ? gbe_ld_state(&st->br[iter]) : 0;
  const int br_chosen = OP == 0 ? gbe_ld_state(&st->branch) : 0;
  const double cn = OP == 1 ? coef[iter] : 0.0;

  const int4 it0 = reinterpret_cast<const int4*>(items)[2 * (size_t)blockIdx.x];      // pidx, ti | tj << 16, p, m
  const int4 it1 = reinterpret_cast<const int4*>(items)[2 * (size_t)blockIdx.x + 1];  // nc, ld, dense_off
  const int ti = it0.y & 0xFFFF, tj = it0.y >> 16, m = it0.w, nc = it1.x, ld = it1.y;
  const int64_t doff = ((int64_t)(uint32_t)it1.z) | ((int64_t)it1.w << 32);
  const double* __restrict__ X = Xin + doff;
  double* __restrict__ Y = Xout + doff;
  const double* __restrict__ XB = OP == 1 ? Xb + doff : X;  // rows of the B operand
  double* __restrict__ DA = OP == 1 ? Dacc + doff : nullptr;
  // OP 1: the sum D is read again only at its core columns (scatter, occupation; Eq.(6)), and with the mirrored
  // store those all lie in the tiles with a core row - the ones that carry a trace partial (pidx >= 0).  The other tiles
  // (four fifths on the water box) skip the read-modify-write of D; there D keeps c_0 T_0 + c_1 T_1 and is never read.
  const bool acc_d = OP == 1 && it0.x >= 0;
  const bool diag = (ti == tj);
  const bool share = diag && OP == 0;  // X X^T on a diagonal tile: the B panel is the A panel
  const int row0 = ti * X2_BT, col0 = tj * X2_BT;
  const int nchunks = ld / X2_KC;

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int role = (wid + blockIdx.x) & 3;  // rotate the warp -> row-block map over the SM sub-partitions
  const int g = lane >> 2, q = lane & 3;
  const int rblk[2] = {role, 7 - role};

  // warp-uniform masks over the 2 x 8 sub-tiles, bit (i * 8 + j):
  //   active: rows < m, columns < ld, not strictly below the diagonal;  mirror: strictly above the diagonal
  unsigned active, mirror;
  {  // lane L < 16 evaluates bit L = (i, j); two ballots build the masks
    const int i = (lane >> 3) & 1, j = lane & 7;
    const int r8 = row0 + 8 * (i ? 7 - role : role), c8 = col0 + 8 * j;
    const bool on = lane < 16 && r8 < m && c8 < ld && r8 <= c8;
    active = __ballot_sync(0xffffffffu, on);
    mirror = __ballot_sync(0xffffffffu, on && r8 < c8);
  }

  // copy slots of this thread: rows (t >> 3) + 16 u, u = 0..3, 16-byte chunk (t & 7) of each K chunk.
  // Rows beyond the edge are clamped to row m - 1: finite data whose products are never stored.
  const double* gA[4];
  const double* gB[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int r = (t >> 3) + 16 * u;
    gA[u] = X + (size_t)min(row0 + r, m - 1) * ld + (t & 7) * 2;
    gB[u] = XB + (size_t)min(col0 + r, m - 1) * ld + (t & 7) * 2;
  }
  double* const sdst = smem + (t >> 3) * X2_STRIDE + (t & 7) * 2;  // slot 0 of the A panel of stage 0

  auto issue = [&](int stage, int kofs) {  // both arguments are compile-time constants after unrolling
#pragma unroll
    for (int u = 0; u < 4; ++u)
      cp_async16(sdst + stage * X2_STAGE + u * 16 * X2_STRIDE, gA[u] + kofs);
    if (!share) {
#pragma unroll
      for (int u = 0; u < 4; ++u)
        cp_async16(sdst + stage * X2_STAGE + X2_PANEL + u * 16 * X2_STRIDE, gB[u] + kofs);
    }
    cp_async_commit();
  };

  double acc[2][8][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  const double* const pa0 = smem + (rblk[0] * 8 + g) * X2_STRIDE + q;
  const double* const pa1 = smem + (rblk[1] * 8 + g) * X2_STRIDE + q;
  const double* const pb0 = smem + (share ? 0 : X2_PANEL) + g * X2_STRIDE + q;
  // warp-uniform code path: 0 full, 1..4 the diagonal pattern of role 0..3, 5..11 the first 1..7 column blocks of
  // both row blocks (ragged right edge), 12 run-time mask (the last diagonal tile), 13 idle
  int pattern = active ? 12 : 13;
  if (active == X2_FULL) pattern = 0;
  else if (active == x2_diag_mask(role)) pattern = 1 + role;
  else {
#pragma unroll
    for (int nb = 1; nb < 8; ++nb)
      if (active == x2_cols_mask(nb)) pattern = 4 + nb;
  }
  auto compute = [&](int stage) {
    const double* a0 = pa0 + stage * X2_STAGE;
    const double* a1 = pa1 + stage * X2_STAGE;
    const double* pb = pb0 + stage * X2_STAGE;
    switch (pattern) {
      case 0: x2_chunk<X2_FULL>(acc, a0, a1, pb, 0); break;
      case 1: x2_chunk<x2_diag_mask(0)>(acc, a0, a1, pb, 0); break;
      case 2: x2_chunk<x2_diag_mask(1)>(acc, a0, a1, pb, 0); break;
      case 3: x2_chunk<x2_diag_mask(2)>(acc, a0, a1, pb, 0); break;
      case 4: x2_chunk<x2_diag_mask(3)>(acc, a0, a1, pb, 0); break;
      case 5: x2_chunk<x2_cols_mask(1)>(acc, a0, a1, pb, 0); break;
      case 6: x2_chunk<x2_cols_mask(2)>(acc, a0, a1, pb, 0); break;
      case 7: x2_chunk<x2_cols_mask(3)>(acc, a0, a1, pb, 0); break;
      case 8: x2_chunk<x2_cols_mask(4)>(acc, a0, a1, pb, 0); break;
      case 9: x2_chunk<x2_cols_mask(5)>(acc, a0, a1, pb, 0); break;
      case 10: x2_chunk<x2_cols_mask(6)>(acc, a0, a1, pb, 0); break;
      case 11: x2_chunk<x2_cols_mask(7)>(acc, a0, a1, pb, 0); break;
      case 12: x2_chunk<0>(acc, a0, a1, pb, active); break;
      default: break;
    }
  };

  if (stop0) {  // idempotency stop already fired (A-7): X is final
    if (OP == 0 && HYB) gbe_griddep_wait();
    return;
  }
  const int branch = br_preset ? br_given : br_chosen;  // preset sequence or the on-device choice
  issue(0, 0);
  for (int kc = 0; kc < nchunks; kc += 2) {
    cp_async_wait<0>();
    __syncthreads();  // chunk kc has landed for every thread; every warp is done with the other stage
    if (kc + 1 < nchunks) issue(1, X2_KC);
    compute(0);
    if (kc + 1 >= nchunks) break;
    cp_async_wait<0>();
    __syncthreads();
    if (kc + 2 < nchunks) issue(0, 2 * X2_KC);
    compute(1);
#pragma unroll
    for (int u = 0; u < 4; ++u) { gA[u] += 2 * X2_KC; gB[u] += 2 * X2_KC; }
  }

  // epilogue: X_{n+1} = Y or 2 X_n - Y, direct + mirrored store, core-row trace partials.
  // Interior tiles (no ragged edge, no core row or column: most of them) take the path without any predicate.
  double s1 = 0.0, s2 = 0.0;
  auto epilogue = [&](auto edge_c, auto trace_c, auto full_c) {
    constexpr bool EDGE = decltype(edge_c)::value, TRACE = decltype(trace_c)::value;
    constexpr bool FULL = decltype(full_c)::value;  // every sub-tile active and strictly above the diagonal
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int r = row0 + rblk[i] * 8 + g;
      if (EDGE && r >= m) continue;
      const double* __restrict__ xr = X + (size_t)r * ld + col0 + 2 * q;
      double* __restrict__ yr = Y + (size_t)r * ld + col0 + 2 * q;
      double* __restrict__ ym0 = Y + (size_t)(col0 + 2 * q) * ld + r;  // mirrored position (c, r) of column block 0
      double* __restrict__ ym1 = ym0 + ld;                            // and (c + 1, r); both advance by 8 rows per j
      const size_t mstep = (size_t)8 * ld;
      double* __restrict__ dr = OP == 1 ? DA + (size_t)r * ld + col0 + 2 * q : nullptr;
      double* __restrict__ dm0 = OP == 1 ? DA + (size_t)(col0 + 2 * q) * ld + r : nullptr;
      double* __restrict__ dm1 = dm0 + ld;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (!FULL && !(active & (1u << (i * 8 + j)))) {  // c < ld holds for every active sub-tile
          ym0 += mstep;
          ym1 += mstep;
          if (OP == 1) { dm0 += mstep; dm1 += mstep; }
          continue;
        }
        const int c = col0 + j * 8 + 2 * q;
        double v0 = acc[i][j][0], v1 = acc[i][j][1];
        if (OP == 1) {  // T_{n+1} = 2 (Xt T_n) - T_{n-1}; T_{n-1} sits where T_{n+1} goes
          const double2 told = *reinterpret_cast<const double2*>(yr + j * 8);
          v0 = 2.0 * v0 - told.x;
          v1 = 2.0 * v1 - told.y;
        } else if (branch) {
          const double2 x = *reinterpret_cast<const double2*>(xr + j * 8);
          v0 = 2.0 * x.x - v0;
          v1 = 2.0 * x.y - v1;
        }
        if (EDGE) {  // pad columns [m, ld) stay zero (the clamped rows above put finite junk here)
          if (c >= m) v0 = 0.0;
          if (c + 1 >= m) v1 = 0.0;
        }
        *reinterpret_cast<double2*>(yr + j * 8) = make_double2(v0, v1);
        if (OP == 1 && acc_d) {  // D += c_{n+1} T_{n+1}
          double2 d = *reinterpret_cast<const double2*>(dr + j * 8);
          d.x = fma(cn, v0, d.x);
          d.y = fma(cn, v1, d.y);
          *reinterpret_cast<double2*>(dr + j * 8) = d;
        }
        if (TRACE && r < nc) {
          s2 += v0 * v0 + v1 * v1;
          if (r == c) s1 += v0;
          if (r == c + 1) s1 += v1;
        }
        if (FULL || (mirror & (1u << (i * 8 + j)))) {
          if (!EDGE || c < m) {
            *ym0 = v0;
            if (OP == 1 && acc_d) *dm0 = fma(cn, v0, *dm0);
            if (TRACE && c < nc) s2 += v0 * v0;
          }
          if (!EDGE || c + 1 < m) {
            *ym1 = v1;
            if (OP == 1 && acc_d) *dm1 = fma(cn, v1, *dm1);
            if (TRACE && c + 1 < nc) s2 += v1 * v1;
          }
        }
        ym0 += mstep;
        ym1 += mstep;
        if (OP == 1) { dm0 += mstep; dm1 += mstep; }
      }
    }
  };
  const bool edge = col0 + X2_BT > m;             // row0 <= col0: the row edge implies the column edge
  const bool trace = OP == 0 && (row0 < nc || col0 < nc);  // a core row, directly or through the mirror
  if (edge || trace) {
    if (edge) epilogue(std::true_type{}, std::true_type{}, std::false_type{});
    else epilogue(std::false_type{}, std::true_type{}, std::false_type{});
  } else if (active == X2_FULL && mirror == X2_FULL) {
    epilogue(std::false_type{}, std::false_type{}, std::true_type{});
  } else {
    epilogue(std::false_type{}, std::false_type{}, std::false_type{});
  }
  // only the tiles with a core row carry a trace; their partials are packed (pidx), so that step 5 reads n_tiles_last
  // pairs instead of one per tile
  const int pidx = it0.x;
  if (!HYB && (OP != 0 || pidx < 0)) return;
  if (OP == 0 && pidx >= 0) {
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) { red[role] = s1; red[4 + role] = s2; }  // indexed by block position: order independent of the rotation
    __syncthreads();
    if (t == 0) {
      partials[2 * (size_t)pidx] = (red[0] + red[1]) + (red[2] + red[3]);
      partials[2 * (size_t)pidx + 1] = (red[4] + red[5]) + (red[6] + red[7]);
    }
  }
  // hyb: this grid must not count as complete before the packed launch next to it is (the launch behind this one waits
  // for THIS grid only, and needs both)
  if (OP == 0 && HYB) gbe_griddep_wait();
}

// ---------------------------------------------------------------------------------------------------------------------
// The same tile with the panels staged by 2-D TMA instead of cp.async: what one SP2 iteration runs (OP 0).
//   - one tensor map per community and dense buffer ([m rows][ld doubles], box 64 rows x 16 doubles = one K chunk of one
//     panel, 128-byte swizzle, rows beyond m zero-filled by the TMA unit: no clamping);
//   - 3 stages, mbarrier full / empty pairs: thread 0 issues the 1-2 tensor copies of a chunk (UTMALDG) two chunks ahead,
//     the four DMMA warps issue no copy instruction and meet no CTA-wide barrier in the main loop;
//   - conflict-free 64-bit fragment loads from the swizzled panels need the K order {2ks, 2ks+1, 2ks+8, 2ks+9} within a
//     chunk (lanes q = 0, 1 read 16-byte unit ks, lanes q = 2, 3 unit ks + 4; the unit index is XORed with the row's low
//     three bits): A and B are permuted alike, the sum over k only changes its order.
// Measured on the 24,576-orbital box: 2.019 ms per launch against 2.083 ms for the cp.async kernel (DMMA sub-pipe 92 %
// active); results agree with the cp.async kernel to rounding (another order of the sum over k).  Tried, slower: one polling
// lane per warp (2.054), the four warps taking turns as producer (2.019 / 2.043), the refill issued before the products
// (2.039), four stages at three CTAs per SM (2.126).
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t mbar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(mbar), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t mbar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(mbar)
      : "memory");
}

constexpr int XT_NST = 3;                          // stages (48 KB: four CTAs per SM)
constexpr int XT_ROW = 16;                         // doubles per panel row (128 bytes, swizzled)
constexpr int XT_PANEL = X2_BT * XT_ROW;           // doubles per panel
constexpr int XT_STAGE = 2 * XT_PANEL;             // A panel + B panel (16 KB)

// one K chunk from swizzled panels; off[ks]: this lane's offset (doubles) inside a row for k-step ks
template <unsigned MASK>
__device__ __forceinline__ void xt_chunk(double (&acc)[2][8][2], const double* __restrict__ pa0,
                                         const double* __restrict__ pa1, const double* __restrict__ pb,
                                         const int (&off)[4], unsigned rt_mask) {
#pragma unroll
  for (int ks = 0; ks < X2_KC / 4; ++ks) {
    double a[2], b[8];
    a[0] = pa0[off[ks]];
    a[1] = pa1[off[ks]];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const bool need = MASK == 0 || ((MASK | (MASK >> 8)) & (1u << j));
      if (need) b[j] = pb[j * 8 * XT_ROW + off[ks]];
    }
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (MASK != 0) {
          if (MASK & (1u << (i * 8 + j))) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        } else {
          if (rt_mask & (1u << (i * 8 + j))) dmma884(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
      }
  }
}

template <int MINB, bool HYB>
__global__ void __launch_bounds__(X2_THREADS, MINB)
    k_x2_tma(const gbe_tile_item* __restrict__ items, const gbe_state* __restrict__ st, const double* __restrict__ Xin,
             double* __restrict__ Xout, double* __restrict__ partials, int iter, const CUtensorMap* __restrict__ maps) {
  extern __shared__ __align__(1024) double smem_t[];  // 3 stages x (A panel, B panel), every panel 1024-byte aligned
  __shared__ double red[8];
  __shared__ __align__(8) unsigned long long bars[2 * XT_NST];  // full[0..2], empty[0..2]

  X2_STAMP(0);
  // programmatic dependent launch, hyb and state loads: as in k_x2
  gbe_griddep_launch();
  if (HYB)
    while (gbe_ld_acquire(&st->iter) != iter + 1 && !gbe_ld_state(&st->stop)) __nanosleep(200);
  const int stop0 = gbe_ld_state(&st->stop);  // requested here, looked at after the mbarrier set-up
  const int br_preset = gbe_ld_state(&st->preset);
  const int br_given = iter < GBE_MAX_ITERS ? gbe_ld_state(&st->br[iter]) : 0;
  const int br_chosen = gbe_ld_state(&st->branch);

  const int4 it0 = reinterpret_cast<const int4*>(items)[2 * (size_t)blockIdx.x];      // pidx, ti | tj << 16, p, m
  const int4 it1 = reinterpret_cast<const int4*>(items)[2 * (size_t)blockIdx.x + 1];  // nc, ld, dense_off
  const int ti = it0.y & 0xFFFF, tj = it0.y >> 16, m = it0.w, nc = it1.x, ld = it1.y;
  const int64_t doff = ((int64_t)(uint32_t)it1.z) | ((int64_t)it1.w << 32);
  const CUtensorMap* const map = maps + it0.z;
  const double* __restrict__ X = Xin + doff;
  double* __restrict__ Y = Xout + doff;
  const bool share = (ti == tj);  // X X^T on a diagonal tile: the B panel is the A panel
  const int row0 = ti * X2_BT, col0 = tj * X2_BT;
  const int nchunks = ld / X2_KC;

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int role = (wid + blockIdx.x) & 3;
  const int g = lane >> 2, q = lane & 3;
  const int rblk[2] = {role, 7 - role};
  const uint32_t bar0 = (uint32_t)__cvta_generic_to_shared(bars);
  const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem_t);
  if (t == 0) {
#pragma unroll
    for (int s = 0; s < XT_NST; ++s) {
      mbar_init(bar0 + 8 * s, 1);             // full: the producer's arrive.expect_tx
      mbar_init(bar0 + 8 * (XT_NST + s), 4);  // empty: one arrival per warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (stop0) {  // idempotency stop already fired (A-7): X is final
    if (HYB) gbe_griddep_wait();
    return;
  }
  const int branch = br_preset ? br_given : br_chosen;
  const uint32_t stage_bytes = share ? XT_PANEL * 8u : XT_STAGE * 8u;
  auto produce = [&](int s, int kc) {  // thread 0: chunk kc -> stage s
    mbar_expect_tx(bar0 + 8 * s, stage_bytes);
    tma_load_2d(smem0 + s * XT_STAGE * 8, map, kc * X2_KC, row0, bar0 + 8 * s);
    if (!share) tma_load_2d(smem0 + (s * XT_STAGE + XT_PANEL) * 8, map, kc * X2_KC, col0, bar0 + 8 * s);
  };
  if (t == 0) {  // all stages are free: chunks 0 .. XT_NST - 1
    asm volatile("fence.proxy.tensormap::generic.acquire.gpu [%0], 128;" ::"l"(map) : "memory");
#pragma unroll
    for (int s = 0; s < XT_NST; ++s)
      if (s < nchunks) produce(s, s);
  }

  unsigned active, mirror;
  {
    const int i = (lane >> 3) & 1, j = lane & 7;
    const int r8 = row0 + 8 * (i ? 7 - role : role), c8 = col0 + 8 * j;
    const bool on = lane < 16 && r8 < m && c8 < ld && r8 <= c8;
    active = __ballot_sync(0xffffffffu, on);
    mirror = __ballot_sync(0xffffffffu, on && r8 < c8);
  }
  double acc[2][8][2];
#pragma unroll
  for (int i = 0; i < 2; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // swizzled fragment offsets: k-step ks reads k = {2ks, 2ks+1, 2ks+8, 2ks+9}: 16-byte unit ks (q < 2) or ks + 4, XOR row & 7
  int off[4];
#pragma unroll
  for (int ks = 0; ks < 4; ++ks) off[ks] = (((ks + 4 * (q >> 1)) ^ g) << 1) + (q & 1);
  const double* const pa0 = smem_t + (rblk[0] * 8 + g) * XT_ROW;
  const double* const pa1 = smem_t + (rblk[1] * 8 + g) * XT_ROW;
  const double* const pb0 = smem_t + (share ? 0 : XT_PANEL) + g * XT_ROW;
  int pattern = active ? 12 : 13;
  if (active == X2_FULL) pattern = 0;
  else if (active == x2_diag_mask(role)) pattern = 1 + role;
  else {
#pragma unroll
    for (int nb = 1; nb < 8; ++nb)
      if (active == x2_cols_mask(nb)) pattern = 4 + nb;
  }
  auto compute = [&](int stage) {
    const double* a0 = pa0 + stage * XT_STAGE;
    const double* a1 = pa1 + stage * XT_STAGE;
    const double* pb = pb0 + stage * XT_STAGE;
    switch (pattern) {
      case 0: xt_chunk<X2_FULL>(acc, a0, a1, pb, off, 0); break;
      case 1: xt_chunk<x2_diag_mask(0)>(acc, a0, a1, pb, off, 0); break;
      case 2: xt_chunk<x2_diag_mask(1)>(acc, a0, a1, pb, off, 0); break;
      case 3: xt_chunk<x2_diag_mask(2)>(acc, a0, a1, pb, off, 0); break;
      case 4: xt_chunk<x2_diag_mask(3)>(acc, a0, a1, pb, off, 0); break;
      case 5: xt_chunk<x2_cols_mask(1)>(acc, a0, a1, pb, off, 0); break;
      case 6: xt_chunk<x2_cols_mask(2)>(acc, a0, a1, pb, off, 0); break;
      case 7: xt_chunk<x2_cols_mask(3)>(acc, a0, a1, pb, off, 0); break;
      case 8: xt_chunk<x2_cols_mask(4)>(acc, a0, a1, pb, off, 0); break;
      case 9: xt_chunk<x2_cols_mask(5)>(acc, a0, a1, pb, off, 0); break;
      case 10: xt_chunk<x2_cols_mask(6)>(acc, a0, a1, pb, off, 0); break;
      case 11: xt_chunk<x2_cols_mask(7)>(acc, a0, a1, pb, off, 0); break;
      case 12: xt_chunk<0>(acc, a0, a1, pb, off, active); break;
      default: break;
    }
  };

  // main loop: chunk kc lives in stage kc % XT_NST; after computing chunk kc the warp releases its stage, and the producer
  // refills the stage released one chunk EARLIER (chunk kc - 1) with chunk kc - 1 + XT_NST: the other warps have a whole
  // chunk to release it, so the producer hardly ever waits
  for (int kc0 = 0; kc0 < nchunks; kc0 += XT_NST) {
    const uint32_t par = (uint32_t)(kc0 / XT_NST) & 1u;
#pragma unroll
    for (int s = 0; s < XT_NST; ++s) {
      const int kc = kc0 + s;
      if (kc >= nchunks) break;
      mbar_wait(bar0 + 8 * s, par);
      compute(s);
      __syncwarp();
      if (lane == 0) mbar_arrive(bar0 + 8 * (XT_NST + s));
      if (t == 0 && kc >= 1 && kc - 1 + XT_NST < nchunks) {
        const int sp = (s + XT_NST - 1) % XT_NST;                // stage of chunk kc - 1
        const uint32_t pp = (uint32_t)((kc - 1) / XT_NST) & 1u;  // its round
        mbar_wait(bar0 + 8 * (XT_NST + sp), pp);
        produce(sp, kc - 1 + XT_NST);
      }
    }
  }

  X2_STAMP(1);
  // epilogue: as k_x2 (OP 0)
  double s1 = 0.0, s2 = 0.0;
  auto epilogue = [&](auto edge_c, auto trace_c, auto full_c) {
    constexpr bool EDGE = decltype(edge_c)::value, TRACE = decltype(trace_c)::value;
    constexpr bool FULL = decltype(full_c)::value;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      const int r = row0 + rblk[i] * 8 + g;
      if (EDGE && r >= m) continue;
      const double* __restrict__ xr = X + (size_t)r * ld + col0 + 2 * q;
      double* __restrict__ yr = Y + (size_t)r * ld + col0 + 2 * q;
      double* __restrict__ ym0 = Y + (size_t)(col0 + 2 * q) * ld + r;
      double* __restrict__ ym1 = ym0 + ld;
      const size_t mstep = (size_t)8 * ld;
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (!FULL && !(active & (1u << (i * 8 + j)))) {
          ym0 += mstep;
          ym1 += mstep;
          continue;
        }
        const int c = col0 + j * 8 + 2 * q;
        double v0 = acc[i][j][0], v1 = acc[i][j][1];
        if (branch) {
          const double2 x = *reinterpret_cast<const double2*>(xr + j * 8);
          v0 = 2.0 * x.x - v0;
          v1 = 2.0 * x.y - v1;
        }
        if (EDGE) {
          if (c >= m) v0 = 0.0;
          if (c + 1 >= m) v1 = 0.0;
        }
        *reinterpret_cast<double2*>(yr + j * 8) = make_double2(v0, v1);
        if (TRACE && r < nc) {
          s2 += v0 * v0 + v1 * v1;
          if (r == c) s1 += v0;
          if (r == c + 1) s1 += v1;
        }
        if (FULL || (mirror & (1u << (i * 8 + j)))) {
          if (!EDGE || c < m) {
            *ym0 = v0;
            if (TRACE && c < nc) s2 += v0 * v0;
          }
          if (!EDGE || c + 1 < m) {
            *ym1 = v1;
            if (TRACE && c + 1 < nc) s2 += v1 * v1;
          }
        }
        ym0 += mstep;
        ym1 += mstep;
      }
    }
  };
  const bool edge = col0 + X2_BT > m;
  const bool trace = row0 < nc || col0 < nc;
  if (edge || trace) {
    if (edge) epilogue(std::true_type{}, std::true_type{}, std::false_type{});
    else epilogue(std::false_type{}, std::true_type{}, std::false_type{});
  } else if (active == X2_FULL && mirror == X2_FULL) {
    epilogue(std::false_type{}, std::false_type{}, std::true_type{});
  } else {
    epilogue(std::false_type{}, std::false_type{}, std::false_type{});
  }
  X2_STAMP(2);
  const int pidx = it0.x;
  if (!HYB && pidx < 0) return;
  if (pidx >= 0) {
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) { red[role] = s1; red[4 + role] = s2; }
    __syncthreads();
    if (t == 0) {
      partials[2 * (size_t)pidx] = (red[0] + red[1]) + (red[2] + red[3]);
      partials[2 * (size_t)pidx + 1] = (red[4] + red[5]) + (red[6] + red[7]);
    }
  }
  if (HYB) gbe_griddep_wait();
}

// Tensor maps.  A map describes ONE community's X_p in ONE dense buffer ([m_p rows][ld_p doubles], box 64 x 16, 128-byte
// swizzle).  Shapes are fixed by the graph, so the maps are encoded once, on the host, when the graph is built
// (cuTensorMapEncodeTiled through the runtime's driver entry point - no link against libcuda) with a placeholder address;
// the dense buffers live in the caller's workspace, so every density call sets the addresses ON THE DEVICE
// (tensormap.replace.tile.global_address, one thread per map, 2 n_part maps): no host work per call, nothing to
// synchronise, capturable in a CUDA graph.  The kernels acquire the map through the tensormap proxy fence before use.
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

__global__ void k_patch_tmaps(CUtensorMap* __restrict__ maps, const int64_t* __restrict__ dense_off,
                              const int32_t* __restrict__ msize, int n_part, const double* X0, const double* X1) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 2 * n_part) return;
  const int p = i < n_part ? i : i - n_part;
  if (msize[p] == 0) return;  // an empty community has no tiles
  const double* base = (i < n_part ? X0 : X1) + dense_off[p];
  asm volatile("tensormap.replace.tile.global_address.global.b1024.b64 [%0], %1;" ::"l"(maps + i), "l"(base) : "memory");
}
}  // namespace

// Encodes the 2 n_part maps of a graph (both halves identical until gbe_x2_prepare sets the addresses); leaves
// g->tmaps null if the driver has no tensor-map encoder (then the cp.async kernel runs)
int gbe_x2_build_tmaps(gbe_graph* g, cudaStream_t s) {
  g->tmaps = nullptr;
  if (g->n_items == 0) return GBE_OK;
  // Which kernel stages the panels.  Measured on the tau x partition grid of the 24,576-orbital box (profiles/
  // r02_sweep_config5.md): the TMA kernel wins where the K loops are long (work-weighted mean m >~ 350: -3 % per launch at
  // m ~ 490, -2 % at m ~ 1,800) and loses where a tile has fewer than ~20 K chunks (m ~ 170: +20 %) - its per-tile set-up
  // (mbarrier initialisation, tensor-map fetch, three chunks requested by one thread) is longer than the cp.async kernel's.
  {
    double w = 0.0, wm = 0.0;
    for (int p = 0; p < g->n_part; ++p) {
      const double m = (double)g->h_m[p];
      w += m * m * m;
      wm += m * m * m * m;
    }
    if (w <= 0.0 || wm / w < 360.0) return GBE_OK;  // short K loops: the cp.async kernel
  }
  static std::atomic<PFN_encodeTiled> encode_p{nullptr};
  PFN_encodeTiled encode = encode_p.load();
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
      (void)cudaGetLastError();
      return GBE_OK;
    }
    encode = reinterpret_cast<PFN_encodeTiled>(fn);
    encode_p.store(encode);
  }
  std::vector<CUtensorMap> h(2 * (size_t)g->n_part);
  memset(h.data(), 0, h.size() * sizeof(CUtensorMap));
  for (int p = 0; p < g->n_part; ++p) {
    const int m = g->h_m[p];
    if (m == 0) continue;
    const cuuint64_t ld = (cuuint64_t)((m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN);
    const cuuint64_t dims[2] = {ld, (cuuint64_t)m};
    const cuuint64_t strides[1] = {ld * 8};
    const cuuint32_t box[2] = {(cuuint32_t)X2_KC, (cuuint32_t)X2_BT};
    const cuuint32_t es[2] = {1, 1};
    void* placeholder = g->dense_off;  // any 16-byte aligned device address: replaced before the first use
    if (encode(&h[p], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, placeholder, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return GBE_OK;  // no maps: the cp.async kernel runs
    h[(size_t)g->n_part + p] = h[p];
  }
  GBE_TRY(gbe_dev_alloc(&g->tmaps, h.size() * sizeof(CUtensorMap)));
  GBE_CUDA(cudaMemcpyAsync(g->tmaps, h.data(), h.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, s));  // pageable: staged
  return GBE_OK;
}

// Before the tiled SP2 loop of a density call: point the maps at this call's dense buffers
int gbe_x2_prepare(const gbe_graph* g, const double* X0, const double* X1, cudaStream_t s) {
  if (!g->tmaps || g->n_items == 0) return GBE_OK;
  const int n = 2 * g->n_part;
  k_patch_tmaps<<<(n + 127) / 128, 128, 0, s>>>(reinterpret_cast<CUtensorMap*>(g->tmaps), g->dense_off, g->msize, g->n_part,
                                               X0, X1);
  GBE_LAUNCHED();
  return GBE_OK;
}

namespace {
template <int MINB, int OP, bool HYB>
int launch_x2(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
              const double* Xb, double* Dacc, const double* coef, const gbe_tile_item* items, int n_items,
              cudaStream_t s, int pdl) {
  auto kern = k_x2<MINB, OP, HYB>;
  const size_t smem = (size_t)2 * X2_STAGE * sizeof(double);
  static gbe_device_once configured;  // one per template instance; function attributes are per device
  if (configured.first()) {
    GBE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    GBE_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
  }
  GBE_CUDA(gbe_launch_kernel(kern, dim3((unsigned)n_items), dim3(X2_THREADS), smem, s, pdl != GBE_PDL_NONE, items, st, Xin,
                             Xout, partials, iter, Xb, Dacc, coef));
  GBE_LAUNCHED();
  return GBE_OK;
}
}  // namespace

int gbe_launch_x2(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                  bool last, bool hybrid, int buffer, cudaStream_t s, int pdl, bool hyb) {
  // the last SP2 iteration computes the tiles with a core row only: the scatter keeps core columns (Eq.(6));
  // hybrid: the communities with m <= GBE_PK_MAX_M are the packed kernel's (gbe_small.cu), only the others are tiled
  const gbe_tile_item* items = hybrid ? (last ? g->items_last_h : g->items_h) : (last ? g->items_last : g->items);
  const int n_items = hybrid ? (last ? g->n_items_last_h : g->n_items_h) : (last ? g->n_items_last : g->n_items);
  return gbe_launch_x2_items(g, st, Xin, Xout, partials, iter, items, n_items, buffer, s, pdl, hyb);
}

int gbe_launch_x2_items(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                        const gbe_tile_item* items, int n_items, int buffer, cudaStream_t s, int pdl, bool hyb) {
  if (n_items == 0) return GBE_OK;
  if (g->tmaps) {  // panels staged by 2-D TMA (k_x2_tma); X_n is in buffer 0 for even iterations, in buffer 1 for odd ones
    const CUtensorMap* maps = reinterpret_cast<const CUtensorMap*>(g->tmaps) + (buffer ? g->n_part : 0);
    const size_t smem = (size_t)XT_NST * XT_STAGE * sizeof(double) + 1024;
    static gbe_device_once configured;
    if (configured.first()) {
      GBE_CUDA(cudaFuncSetAttribute(k_x2_tma<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GBE_CUDA(cudaFuncSetAttribute(k_x2_tma<4, false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
      GBE_CUDA(cudaFuncSetAttribute(k_x2_tma<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      GBE_CUDA(cudaFuncSetAttribute(k_x2_tma<4, true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    }
    // (HYB is a template parameter: the kernel of the bench workload carries none of the mixed-graph code)
    GBE_CUDA(gbe_launch_kernel(hyb ? k_x2_tma<4, true> : k_x2_tma<4, false>, dim3((unsigned)n_items), dim3(X2_THREADS), smem,
                               s, pdl != GBE_PDL_NONE, items, st, Xin, Xout, partials, iter, maps));
    GBE_LAUNCHED();
    return GBE_OK;
  }
  if (hyb) return launch_x2<4, 0, true>(g, st, Xin, Xout, partials, iter, nullptr, nullptr, nullptr, items, n_items, s, pdl);
  return launch_x2<4, 0, false>(g, st, Xin, Xout, partials, iter, nullptr, nullptr, nullptr, items, n_items, s, pdl);
}

int gbe_launch_cheb_step(const gbe_graph* g, gbe_state* st, const double* Xt, const double* Tn, double* Tio, double* Dacc,
                         const double* coef, int iter, double* partials, cudaStream_t s, bool last) {
  if (g->n_items == 0) return GBE_OK;
  // last: T_M feeds D only, and D is read at its core columns only - the tiles with a core row suffice
  return launch_x2<4, 1, false>(g, st, Xt, Tio, partials, iter, Tn, Dacc, coef, last ? g->items_last : g->items,
                                last ? g->n_items_last : g->n_items, s, GBE_PDL_NONE);
}
