// Step 4 (+ 5) for SMALL subgraphs, any number of them: one SP2 iteration per launch, whole matrices in shared memory.
//
//     Y_p = X_p X_p;  X_p <- Y_p  or  2 X_p - Y_p   for every community p with m_p <= 160
//
// The cost law of the paper (more partitions -> smaller core+halo size m) puts a whole regime of the method at
// m ~ 30 - 130 with a thousand or more communities (BASELINE.json configs[4], tau = 1e-3).  There a 64 x 64 tile of the
// tiled kernel (gbe_x2.cu) is mostly mask and its two launches per iteration are mostly launch latency, and the resident
// kernel (gbe_resident.cu) cannot run: its grid barrier needs all communities co-resident.  Here:
//   - a CTA (32 warps, one per SM) owns a BIN of 1..16 communities for one iteration.  The bins are packed once per graph
//     on the host: longest processing time first onto exactly k x SM-count bins (a launch is k equally heavy waves),
//     bounded by shared memory;
//   - every X_p of the bin is copied to shared memory by TMA: one bulk copy (cp.async.bulk, SASS UBLKCP) per matrix row,
//     described by a per-bin ROW TABLE built with the graph (shared-memory offset, dense offset, bytes, community): a
//     thread reads its entry before the launch dependency resolves and issues one copy - no per-community loops.  UBLKCP
//     takes uniform operands, so a warp issues its lanes' copies one by one: the rows are dealt over all 32 warps.  Each
//     community counts its bytes on an mbarrier of its own, and a work unit waits for ITS community only (the largest
//     sits in slot 0 and lands first).  Row stride ld_p + 4 doubles: conflict-free 64-bit fragment loads.  The batch is
//     read exactly once per iteration;
//   - Y = X X^T on FP64 tensor cores (mma.sync.m8n8k4.f64): a work unit is two 8-row blocks x up to four 8-column blocks
//     on or above the diagonal (6 fragment loads per 8 DMMA); the host deals the units of the bin, longest first, to the
//     least loaded warp, ties to the least loaded SM sub-partition (each has its own DMMA pipe).  A unit's part of
//     X_{n+1} goes straight from the accumulators to the dense buffer (direct + mirrored store; X_n in shared memory
//     stays intact), with the core-row traces of X_{n+1} (t1 = sum X_ii, t2 = sum_c X_ic^2 = Tr_core X^2 for symmetric
//     X) taken on the way and summed per bin in a fixed order;
//   - a unit stores to X_p only after all of X_p is in shared memory (its mbarrier), so when every community of the
//     graph is packed the iteration runs IN PLACE in one dense buffer;
//   - programmatic dependent launch: the bins of iteration n + 1 are handed to the SMs while the last bins of iteration
//     n still run, set themselves up (description, row table entry, mbarriers, zero rows) and wait in the kernel
//     (griddepcontrol.wait) for iteration n to complete;
//   - step 5 LAZY (every community packed): a bin ends by storing its trace pair, nothing else.  Every bin of the NEXT
//     launch starts by summing all pairs of the previous one - the same fixed order in every bin, so bitwise the same
//     t1, t2 and the same branch everywhere - while its rows land; bin 0 also writes the decision to the state and the
//     log.  No fence, no ticket, no serial tail after the last bin; one k_trace_branch after the last launch.  (With
//     larger communities in the same graph the tiled kernel runs first in the iteration and the decision is taken by the
//     bin that publishes its pair LAST - one ticket per bin; its pairs sit in front of the bins' and enter the same
//     sum.)  Either way ONE launch per SP2 iteration instead of two, and results reproducible bit for bit.
// Measured on B200 (profiles/r02_small_m_ncu.md; per-warp %globaltimer stamps in a throw-away build): 1,024 communities of
// m = 28/69/123 take 1.40 ms per density call (tiled kernels 2.55 ms, first version of this kernel 1.85 ms).  Per bin:
// ~1.4 us set-up (hidden behind the previous launch for the first wave), rows landed 2.3 - 2.6 us after the dependency
// resolves (the pair sum runs meanwhile), 10 - 11 us of products and stores, 0.4 us for the pair.  In the product phase
// the FP64 tensor pipe is busy about 60 % of the time (43 % over the launch): every non-DMMA instruction costs the
// sub-partition ~1.4 DMMA-pipe cycles, and with K = m ~ 70 a unit is 18 k-steps of 8 DMMA against ~70 instructions of
// unit decode, update and store per 8 x 8 block.
// Tried and dropped, none faster: 16 warps and two bins per SM (the two start in phase and share the pipes); copies in
// column quarters with the first unit started on the first quarter; self-scheduling of the units through a shared-memory
// counter; persistent CTAs with two half-size buffers (the next bin copied in under the products of this one); every
// warp summing all pairs itself (no CTA barrier, but 32 x the pair traffic: 1.9 ms); 128-bit fragment loads feeding two
// k-steps (row stride ld + 8, k order 0 2 4 6 | 1 3 5 7, addresses formed in the asm: half the LDS and a third fewer
// instructions in the main loop, yet 5 - 9 % slower end to end).
// Bound: FP64 tensor pipe + instruction issue inside a bin; per-bin latencies around it.
#include <algorithm>
#include <cstdlib>
#include <numeric>
#include <queue>

#include "gbe_internal.cuh"

// Optional instrumentation (python -m paper_1603_00937_b200.build --stamps -> libgbe_stamps.so; bench.py --timeline packed):
// %globaltimer stamps per bin at a few points of the kernel.  Compiled out of libgbe.so.
#ifdef GBE_STAMPS
constexpr int PK_ST_ITERS = 40, PK_ST_BINS = 1024, PK_ST_W = 64;
static __device__ unsigned long long g_pk_stamps[(size_t)PK_ST_ITERS * PK_ST_BINS * PK_ST_W];
__device__ __forceinline__ unsigned long long pk_gtime() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
// slot k of bin blockIdx.x in launch `iter`: 0 CTA start, 1 set-up done, 2 dependency resolved, 3 copies issued,
// 4 first unit of thread 0 starts, 5 pair published, 7 step 5 done, 8 + w warp w has computed and stored its units,
// 40 + s the rows of community s have landed
#define PK_STAMP(k)                                                                                   \
  do {                                                                                                \
    if (iter < PK_ST_ITERS && blockIdx.x < PK_ST_BINS)                                                \
      g_pk_stamps[((size_t)iter * PK_ST_BINS + blockIdx.x) * PK_ST_W + (k)] = pk_gtime();             \
  } while (0)
extern "C" int gbe_stamps_packed(unsigned long long* host, size_t bytes) {
  if (bytes < sizeof(g_pk_stamps)) return -1;
  return (int)cudaMemcpyFromSymbol(host, g_pk_stamps, sizeof(g_pk_stamps));
}
extern "C" int gbe_stamps_packed_shape(int* iters, int* bins, int* width) {
  *iters = PK_ST_ITERS; *bins = PK_ST_BINS; *width = PK_ST_W;
  return 0;
}
#else
#define PK_STAMP(k) do { } while (0)
#endif

namespace {

constexpr int PK_WARPS = 32;             // 1,024 threads, 64 registers each, one CTA per SM
constexpr int PK_THREADS = PK_WARPS * 32;
constexpr int PK_UCOLS = 4;              // 8-column blocks per work unit
constexpr int PK_MAX_ROUNDS = 32;        // units per warp (lane j of a warp fetches the code of its j-th unit)
constexpr unsigned PK_NONE = 0xFFFFu;
constexpr int PK_PAD = 4;                // shared-memory row stride = ld + 4 doubles (ld is a multiple of 16): the 16 doubles a
                                         // half warp loads with LDS.64 (4 rows x 4 columns) fall into distinct banks

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
// TALL: the unit spans two 8-row blocks (bi, bi + 1); FIRST: its first column block is bi, so the block (bi + 1, bi) lies
// below the diagonal and is left out (its values arrive through the mirror of (bi, bi + 1))
template <int NB, bool TALL, bool FIRST>
__device__ __forceinline__ void pk_unit_mma(double (&acc)[2][PK_UCOLS][2], const double* __restrict__ pa,
                                            const double* __restrict__ pb, int kmax, int stride) {
#pragma unroll 2
  for (int k0 = 0; k0 < kmax; k0 += 4) {
    const double a0 = pa[k0];
    const double a1 = TALL ? pa[8 * stride + k0] : 0.0;
    double b[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) b[j] = pb[j * 8 * stride + k0];
#pragma unroll
    for (int j = 0; j < NB; ++j) dmma884(acc[0][j][0], acc[0][j][1], a0, b[j]);
    if (TALL) {
#pragma unroll
      for (int j = FIRST ? 1 : 0; j < NB; ++j) dmma884(acc[1][j][0], acc[1][j][1], a1, b[j]);
    }
  }
}
template <bool TALL, bool FIRST>
__device__ __forceinline__ void pk_unit_mma_nb(int nb, double (&acc)[2][PK_UCOLS][2], const double* __restrict__ pa,
                                               const double* __restrict__ pb, int kmax, int stride) {
  switch (nb) {
    case 4: pk_unit_mma<4, TALL, FIRST>(acc, pa, pb, kmax, stride); break;
    case 3: pk_unit_mma<3, TALL, FIRST>(acc, pa, pb, kmax, stride); break;
    case 2: pk_unit_mma<2, TALL, FIRST>(acc, pa, pb, kmax, stride); break;
    default: pk_unit_mma<1, TALL, FIRST>(acc, pa, pb, kmax, stride); break;
  }
}

// TMA bulk copy of one row (global -> shared), completion counted in bytes on an mbarrier
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_row_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(mbar)
               : "memory");
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

// unit code: slot (4 bits) | row block bi (5) | first column block as (bj - bi) / 4 (3) | blocks - 1 (2) | tall (1)
__host__ __device__ inline uint16_t pk_encode(int slot, int bi, int bj, int nb, int tall) {
  return (uint16_t)(slot | (bi << 4) | (((bj - bi) >> 2) << 9) | ((nb - 1) << 12) | (tall << 14));
}

// one unit's part of X_{n+1}: direct + mirrored store, traces of the core rows.  EDGE: the unit touches rows or columns
// >= m (ragged last block); TRACE: it touches a core row, directly or through the mirror
template <bool EDGE, bool TRACE>
__device__ __forceinline__ void pk_unit_store(const double (&acc)[PK_UCOLS][2], int j0, const double* __restrict__ x0,
                                              double* __restrict__ Y, int bi, int bj, int nb, int g, int q, int m,
                                              int nc, int ld, int stride, int branch, double& s1, double& s2) {
  const int r = bi * 8 + g;
  if (EDGE && r >= m) return;
  const double* __restrict__ xr = x0 + (size_t)r * stride + bj * 8 + 2 * q;
  double* __restrict__ yr = Y + (size_t)r * ld + bj * 8 + 2 * q;
  double* __restrict__ ym = Y + (size_t)(bj * 8 + 2 * q) * ld + r;  // mirrored position (c, r); (c + 1, r) is ld further
#pragma unroll
  for (int j = 0; j < PK_UCOLS; ++j) {
    if (j >= j0 && j < nb) {
      const int c = (bj + j) * 8 + 2 * q;
      double v0 = acc[j][0], v1 = acc[j][1];
      if (branch) {
        const double2 x = *reinterpret_cast<const double2*>(xr + j * 8);
        v0 = 2.0 * x.x - v0;
        v1 = 2.0 * x.y - v1;
      }
      *reinterpret_cast<double2*>(yr + j * 8) = make_double2(v0, v1);
      if (TRACE && r < nc) {
        s2 += v0 * v0 + v1 * v1;
        if (r == c) s1 += v0;
        if (r == c + 1) s1 += v1;
      }
      if (bj + j != bi) {  // off-diagonal block: mirror (the diagonal block is computed whole)
        if (!EDGE || c < m) {
          ym[(size_t)j * 8 * ld] = v0;
          if (TRACE && c < nc) s2 += v0 * v0;
        }
        if (!EDGE || c + 1 < m) {
          ym[(size_t)j * 8 * ld + ld] = v1;
          if (TRACE && c + 1 < nc) s2 += v1 * v1;
        }
      }
    }
  }
}

// Step 5, three ways (`fused`):
//   0  no decision here (pre-set sequence without traces, or k_trace_branch follows);
//   1  TICKET: the last bin to publish its partial reduces all n_partials pairs and takes the decision;
//   2  LAZY: nobody does at the end - EVERY bin of the next launch starts by summing the lazy_n pairs this launch left at
//      partials[lazy_base ...] (same fixed order in every bin: bitwise the same t1, t2, the same decision), bin 0 also
//      writes it to the state and the log.  No fence, no ticket, no serial tail; the sums run while the rows land.  The
//      pairs of consecutive launches alternate between two halves of `partials` (a late bin of launch n + 1 still reads
//      the pairs of launch n while early bins of n + 1 publish theirs).  lazy_n == 0 (first launch): the decision is in
//      the state already (k_trace_branch after the gather); after the last launch the host runs k_trace_branch once.
__global__ void __launch_bounds__(PK_THREADS, 1)
    k_sp2_packed(const gbe_pk_cta* __restrict__ ctas, const uint16_t* __restrict__ ucodes,
                 const gbe_pk_row* __restrict__ rows, gbe_state* st,
                 const double* Xin, double* Xout, double* __restrict__ partials,  // Xin == Xout when the loop runs in place
                 int partial_base, int n_partials, int iter, int last, int fused, int code_stride, int rounds_max,
                 int lazy_base, int lazy_n) {
  extern __shared__ __align__(16) double xs[];  // the X_p of the bin
  __shared__ gbe_pk_cta me;
  __shared__ double red[2 * PK_WARPS], lazy_red[2 * PK_WARPS];
  __shared__ int is_last;
  __shared__ __align__(8) unsigned long long load_bar[GBE_PK_MAX_SLOTS];  // one per community of the bin

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, g = lane >> 2, q = lane & 3;
  if (t == 0) PK_STAMP(0);
  // the bin's description (one coalesced read), this warp's unit codes (dealt on the host, longest first, to the least
  // loaded warp; lane j holds the j-th one; fixed stride per bin, so the address does not wait for the description):
  // independent loads, all in flight
  if (t < (int)(sizeof(gbe_pk_cta) / 4)) reinterpret_cast<int*>(&me)[t] = reinterpret_cast<const int*>(ctas + blockIdx.x)[t];
  const unsigned my_code = lane < rounds_max ? ucodes[(size_t)blockIdx.x * code_stride + lane * PK_WARPS + wid] : PK_NONE;
  __syncthreads();
  const int n_slots = me.n_slots, n_rounds = me.n_rounds, n_rows = me.n_rows;
  // ---- everything that does not depend on the previous launch: the mbarriers, the zero rows [m, 8R) of shared memory,
  //      this thread's entry of the row table (the rows of the bin are dealt warp by warp: entry i goes to lane i / 32 of
  //      warp i % 32.  UBLKCP takes its operands from uniform registers, so a warp issues the copies of its lanes one
  //      after the other: every warp gets a few, none a whole column - that warp would start its products late)
  const uint32_t mbar0 = (uint32_t)__cvta_generic_to_shared(load_bar);
  const uint32_t xs0 = (uint32_t)__cvta_generic_to_shared(xs);
  if (t < n_slots) {
    mbar_init(mbar0 + 8u * t, 1);
    mbar_expect_tx(mbar0 + 8u * t, (uint32_t)(me.slot[t].m * me.slot[t].ld) * 8u);
  }
  const int ridx = wid + PK_WARPS * lane;
  gbe_pk_row my_row = {0u, 0u, 0};
  if (ridx < n_rows) my_row = rows[me.row0 + ridx];
  for (int s = 0; s < n_slots; ++s) {
    const int m = me.slot[s].m, stride = me.slot[s].ld + PK_PAD;
    for (int i = m * stride + t; i < 8 * me.slot[s].R * stride; i += PK_THREADS) xs[me.slot[s].soff + i] = 0.0;
  }
  // Programmatic dependent launch (the launcher sets the stream-serialisation attribute): the bins of iteration n + 1 are
  // handed to the SMs while the last bins of iteration n still run, do the set-up above, and wait HERE until that grid
  // has completed and its X_{n+1}, partials and state are visible.  Nothing above reads or writes what a launch produces
  // (the description, the unit codes and the row table belong to the graph).  Without the attribute both instructions
  // are no-ops.
  if (t == 0) PK_STAMP(1);
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (t == 0) PK_STAMP(2);
  // the state and (lazy step 5) this thread's pair(s) of the previous launch: all requested at once, used after the
  // copies are issued
  int stop = st->stop;
  const int preset = st->preset, br_state = st->branch, br_preset = iter < GBE_MAX_ITERS ? (int)st->br[iter] : 0;
  const double idem_tol = st->idem_tol, n_occ = st->n_occ;
  double a1 = 0.0, a2 = 0.0;
  if (lazy_n > 0) {
    const double2* __restrict__ p2 = reinterpret_cast<const double2*>(partials) + lazy_base;
    for (int i = t; i < lazy_n; i += PK_THREADS) {
      const double2 v = __ldcg(p2 + i);
      a1 += v.x;
      a2 += v.y;
    }
  }
  int branch = preset ? br_preset : br_state;
  __syncthreads();   // the mbarriers are initialised
  if (stop) return;  // idempotency stop already fired (A-7): X is final

  // ---- X_n of every community of the bin -> shared memory: one TMA bulk copy per row (row stride ld + 4 doubles in
  //      shared memory: conflict-free 64-bit fragment loads), completion counted in bytes on the community's mbarrier
  //      - no per-piece instructions.  Rows [m, 8R) are zero: no predicate in the products.
  if (ridx < n_rows)
    bulk_row_g2s(xs0 + my_row.soff, Xin + my_row.goff, my_row.bytes & 0xFFFFFFu, mbar0 + 8u * (my_row.bytes >> 24));
  for (int i = ridx + PK_THREADS; i < n_rows; i += PK_THREADS) {  // bins of more than 1,024 rows
    const gbe_pk_row e = rows[me.row0 + i];
    bulk_row_g2s(xs0 + e.soff, Xin + e.goff, e.bytes & 0xFFFFFFu, mbar0 + 8u * (e.bytes >> 24));
  }
  if (Xin != Xout) {
    // pad columns [8R, ld) of the OUTPUT stay zero (no work unit covers them; [m, 8R) come out of the products as zeros);
    // in place they are zero since the gather and nobody writes them
    for (int s = 0; s < n_slots; ++s) {
      const int m = me.slot[s].m, ld = me.slot[s].ld;
      if (ld > 8 * me.slot[s].R) {
        double* __restrict__ out = Xout + me.slot[s].dense_off + 8 * me.slot[s].R;
        for (int i = t; i < m * 8; i += PK_THREADS) out[(size_t)(i >> 3) * ld + (i & 7)] = 0.0;
      }
    }
  }
  if (t == 0) PK_STAMP(3);
  if (lazy_n > 0) {
    // LAZY step 5: t1, t2 of X_iter from the pairs of the previous launch
    if (wid * 32 < lazy_n) {  // (a warp without pairs holds zeros)
      a1 = warp_sum(a1);
      a2 = warp_sum(a2);
    }
    if (lane == 0) { lazy_red[wid] = a1; lazy_red[PK_WARPS + wid] = a2; }
    __syncthreads();
    a1 = warp_sum(lazy_red[lane]);  // every warp: the same 32 numbers in the same order
    a2 = warp_sum(lazy_red[PK_WARPS + lane]);
    // gbe_trace_decide's rule (A-6, A-7) with k = iter (the state's counter is bin 0's to advance, below)
    if (idem_tol >= 0.0 && iter >= 1 && fabs(a1 - a2) <= idem_tol) stop = 1;
    else if (!preset) branch = (fabs(a2 - n_occ) < fabs(2.0 * a1 - a2 - n_occ)) ? 0 : 1;
    if (blockIdx.x == 0 && t == 0) gbe_trace_decide(st, a1, a2);
    if (stop) {  // X_iter is final; no copy may be in flight when the CTA retires
      __syncthreads();
      if (t < n_slots) mbar_wait(mbar0 + 8u * t, 0);
      return;
    }
  }
  if (t == 0) PK_STAMP(7);
#ifdef GBE_STAMPS
  if (wid == PK_WARPS - 1)  // (instrumented build only: the last warp watches the communities land before it starts)
    for (int s = 0; s < n_slots; ++s) {
      mbar_wait(mbar0 + 8u * s, 0);
      if (lane == 0) PK_STAMP(40 + s);
    }
#endif
  // (no wait here: a unit waits for the rows of ITS community only - the largest community of a bin sits in slot 0, its
  //  copies are issued first and its units are the first of every warp's list, so the products start while the rest lands)

  // ---- Y = X X^T unit by unit (one 8-row block x up to four 8-column blocks on or above the diagonal); the unit's part
  //      of X_{n+1} = Y or 2 X_n - Y goes straight from the accumulators to the other dense buffer, direct + mirrored,
  //      with the core-row traces of X_{n+1} taken on the way (X_n in shared memory stays intact: nothing is in place).
  double s1 = 0.0, s2 = 0.0;
#pragma unroll 1
  for (int round = 0; round < n_rounds; ++round) {
    const unsigned code = __shfl_sync(0xffffffffu, my_code, round);
    const int s = code & 15, bi = (code >> 4) & 31, bj = bi + 4 * ((code >> 9) & 7), nb = 1 + ((code >> 12) & 3);
    const bool tall = (code >> 14) & 1, firstu = bj == bi;
    const int nc = me.slot[s].nc, m = me.slot[s].m, ld = me.slot[s].ld, stride = ld + PK_PAD;
    const int kmax = (m + 3) & ~3;  // columns >= m are zero
    // the last iteration needs the core rows and (through the mirror) the core columns only (Eq.(6))
    if (code == PK_NONE || (last && bi * 8 >= nc)) continue;
    mbar_wait(mbar0 + 8u * s, 0);
    if (round == 0 && t == 0) PK_STAMP(4);
    const double* x0 = xs + me.slot[s].soff;
    const double* pa = x0 + (size_t)(bi * 8 + g) * stride + q;
    const double* pb = x0 + (size_t)(bj * 8 + g) * stride + q;
    double acc[2][PK_UCOLS][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
      for (int j = 0; j < PK_UCOLS; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    if (!tall) pk_unit_mma_nb<false, false>(nb, acc, pa, pb, kmax, stride);
    else if (firstu) pk_unit_mma_nb<true, true>(nb, acc, pa, pb, kmax, stride);
    else pk_unit_mma_nb<true, false>(nb, acc, pa, pb, kmax, stride);
    double* __restrict__ Y = Xout + me.slot[s].dense_off;
    const bool edge = (bj + nb) * 8 > m;  // bi <= bj: the row edge implies the column edge
    const bool trace = bi * 8 < nc;       // bi <= bj: a core column implies a core row
#pragma unroll
    for (int i = 0; i < 2; ++i) {
      if (i == 1 && !tall) break;
      const int j0 = (i == 1 && firstu) ? 1 : 0;  // block (bi + 1, bi) was not formed
      if (edge) pk_unit_store<true, true>(acc[i], j0, x0, Y, bi + i, bj, nb, g, q, m, nc, ld, stride, branch, s1, s2);
      else if (trace) pk_unit_store<false, true>(acc[i], j0, x0, Y, bi + i, bj, nb, g, q, m, nc, ld, stride, branch, s1, s2);
      else pk_unit_store<false, false>(acc[i], j0, x0, Y, bi + i, bj, nb, g, q, m, nc, ld, stride, branch, s1, s2);
    }
  }

  // ---- core-row traces of X_{n+1}: per warp in the (fixed) order of its unit list, then over the warps: one pair per bin
  if (lane == 0) PK_STAMP(8 + wid);
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) { red[wid] = s1; red[PK_WARPS + wid] = s2; }
  if (wid == 1 && lane < n_slots) mbar_wait(mbar0 + 8u * lane, 0);  // no copy in flight when the CTA retires
  __syncthreads();
  if (wid == 0) {
    const double a = warp_sum(red[lane]);
    const double b = warp_sum(red[PK_WARPS + lane]);
    if (lane == 0) {
      double* out = partials + 2 * (size_t)(partial_base + blockIdx.x);
      out[0] = a;
      out[1] = b;
      int lastflag = 0;
      if (fused == 1) {
        __threadfence();  // the pair is visible before the ticket is taken
        lastflag = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
      }
      is_last = lastflag;
      PK_STAMP(5);
    }
  }
  if (fused != 1) return;
  __syncthreads();
  if (!is_last) return;

  // ---- step 5, by the bin that arrived last: all partials of this iteration (tiled kernel's and bins') in a fixed order
  __threadfence();
  a1 = a2 = 0.0;
  const double2* __restrict__ p2 = reinterpret_cast<const double2*>(partials);
  for (int i = t; i < n_partials; i += PK_THREADS) {
    const double2 v = __ldcg(p2 + i);
    a1 += v.x;
    a2 += v.y;
  }
  a1 = warp_sum(a1);
  a2 = warp_sum(a2);
  if (lane == 0) { red[wid] = a1; red[PK_WARPS + wid] = a2; }
  __syncthreads();
  if (wid == 0) {
    a1 = warp_sum(red[lane]);
    a2 = warp_sum(red[PK_WARPS + lane]);
    if (lane == 0) {
      st->ticket = 0;
      gbe_trace_decide(st, a1, a2);
    }
  }
}

struct Unit { int slot, bi, bj, nb, tall, cost; };

inline int units_of(int R) {
  int n = 0;
  for (int bi = 0; bi < R; bi += 2) n += (R - bi + PK_UCOLS - 1) / PK_UCOLS;
  return n;
}
inline int64_t dmma_of(int m, int /*ld*/) {  // DMMA instructions of one X X^T: 8 x 8 blocks on or above the diagonal x ceil(m / 4)
  const int64_t R = (m + 7) / 8;
  return R * (R + 1) / 2 * ((m + 3) / 4);
}
inline size_t smem_doubles_of(int m, int ld) { return (size_t)((m + 7) / 8 * 8) * (ld + PK_PAD); }  // 8R rows of ld + 4 doubles

template <typename T>
int upload(const std::vector<T>& h, T** d, cudaStream_t s) {
  GBE_TRY(gbe_dev_alloc((void**)d, std::max<size_t>(16, h.size() * sizeof(T))));
  if (!h.empty()) GBE_CUDA(cudaMemcpyAsync(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, s));
  return GBE_OK;
}
}  // namespace

namespace {
struct Bin { int64_t load = 0; size_t smem = 0; int units = 0; std::vector<int> ps; };

// Longest processing time first onto EXACTLY n bins (no bin is opened on the way: a launch is a whole number of waves);
// false if a community finds no bin with room (shared memory, slots, unit codes)
bool lpt(const gbe_graph* g, const std::vector<int>& cs, int n, size_t smem_cap, int warps, std::vector<Bin>* out) {
  std::vector<Bin>& bins = *out;
  bins.assign(n, Bin());
  using QE = std::pair<int64_t, int>;  // (load, bin): least loaded first, ties by index
  std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
  for (int b = 0; b < n; ++b) pq.push({0, b});
  std::vector<QE> aside;
  for (int p : cs) {
    const int m = g->h_m[p], ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    const size_t need = smem_doubles_of(m, ld);
    const int nu = units_of((m + 7) / 8);
    aside.clear();
    int chosen = -1;
    while (!pq.empty()) {
      const QE e = pq.top();
      pq.pop();
      const Bin& b = bins[e.second];
      if (b.units + nu <= PK_MAX_ROUNDS * warps / 2 && b.smem + need <= smem_cap && (int)b.ps.size() < GBE_PK_MAX_SLOTS) {
        chosen = e.second;
        break;
      }
      aside.push_back(e);
    }
    for (const QE& e : aside) pq.push(e);
    if (chosen < 0) return false;
    Bin& b = bins[chosen];
    b.ps.push_back(p);
    b.units += nu;
    b.smem += need;
    b.load += dmma_of(m, ld);
    pq.push({b.load, chosen});
  }
  return true;
}

}  // namespace

// Packs the communities with 0 < m_p <= g->pk_max_m into bins (host; once per graph) and uploads the work description.
int gbe_build_packed(gbe_graph* g, cudaStream_t s) {
  g->n_pk_ctas = 0;
  g->pk_n_small = 0;
  g->pk[0] = gbe_pk_class();
  int dev = 0, smem_max = 0;
  GBE_CUDA(cudaGetDevice(&dev));
  GBE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  const int sms = gbe_sm_count();
  const size_t smem_cap = (size_t)std::max(0, smem_max - 2048) / sizeof(double);  // doubles; static shared memory aside
  std::vector<int> cs;
  int64_t total = 0;
  for (int p = 0; p < g->n_part; ++p) {
    const int m = g->h_m[p];
    if (m <= 0 || m > g->pk_max_m) continue;
    const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    if (smem_doubles_of(m, ld) > smem_cap) continue;
    cs.push_back(p);
    total += dmma_of(m, ld);
  }
  g->pk_n_small = (int32_t)cs.size();
  if (cs.empty()) return GBE_OK;
  auto cost = [&](int p) { return dmma_of(g->h_m[p], 0); };
  std::stable_sort(cs.begin(), cs.end(), [&](int a, int b) { return cost(a) > cost(b); });
  // k waves of one bin per SM: the smallest k the communities fit into, and at least so many that a bin carries no more
  // than ~3,000 DMMA (6 us of tensor work on one SM); a launch is a whole number of equally heavy waves
  std::vector<Bin> bins;
  for (int k = (int)std::max<int64_t>(1, (total / sms + 1500) / 3000);; ++k) {
    const int n = (int)std::min<int64_t>((int64_t)cs.size(), (int64_t)k * sms);
    if (lpt(g, cs, n, smem_cap, PK_WARPS, &bins)) break;
    if (n == (int)cs.size()) return GBE_EINVAL;  // cannot happen: every community fits a bin of its own
  }
  // heavy bins first in launch order
  std::vector<int> border(bins.size());
  std::iota(border.begin(), border.end(), 0);
  std::stable_sort(border.begin(), border.end(), [&](int a, int b) { return bins[a].load > bins[b].load; });
  std::vector<gbe_pk_cta> h_ctas;
  std::vector<gbe_pk_row> h_rows;
  std::vector<std::vector<uint16_t>> grids;
  size_t smem_need = 0;
  int rounds_max = 0;
  for (int bi_ : border) {
    const Bin& b = bins[bi_];
    if (b.ps.empty()) continue;
    gbe_pk_cta c = {};
    c.n_slots = (int32_t)b.ps.size();
    c.row0 = (int32_t)h_rows.size();
    std::vector<Unit> units;
    size_t soff = 0;
    for (int k = 0; k < (int)b.ps.size(); ++k) {
      const int p = b.ps[k], m = g->h_m[p], ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN, R = (m + 7) / 8;
      c.slot[k] = {p, m, g->h_ncore[p], ld, (int32_t)soff, (int16_t)R, 0, 0, 0, g->h_dense_off[p]};
      for (int r = 0; r < m; ++r)
        h_rows.push_back({(uint32_t)((soff + (size_t)r * (ld + PK_PAD)) * 8), (uint32_t)(ld * 8) | ((uint32_t)k << 24),
                          g->h_dense_off[p] + (int64_t)r * ld});
      soff += (size_t)(8 * R) * (ld + PK_PAD);
      // row blocks in pairs (2 x up to 4 blocks per unit: 6 fragment loads per 8 DMMA); an odd last row block alone
      for (int bi = 0; bi < R; bi += 2) {
        const int tall = bi + 1 < R ? 1 : 0;
        for (int bj = bi; bj < R; bj += PK_UCOLS) {
          const int nb = std::min(PK_UCOLS, R - bj);
          units.push_back({k, bi, bj, nb, tall, ((1 + tall) * nb - (tall && bj == bi ? 1 : 0)) * ((m + 3) / 4)});
        }
      }
    }
    c.n_rows = (int32_t)h_rows.size() - c.row0;
    smem_need = std::max(smem_need, soff * sizeof(double));
    // the units of the bin onto the 32 warps: longest first, always to the least loaded warp - ties to the warp whose SM
    // sub-partition (warp index mod 4: each has its own FP64 tensor pipe) carries the least; codes stored round-major
    std::stable_sort(units.begin(), units.end(), [](const Unit& a, const Unit& b) { return a.cost > b.cost; });
    int wload[PK_WARPS] = {0}, wcnt[PK_WARPS] = {0}, sub[4] = {0};
    std::vector<uint16_t> grid((size_t)PK_MAX_ROUNDS * PK_WARPS, (uint16_t)PK_NONE);
    int rounds = 0;
    for (const Unit& un : units) {
      int best = -1;
      for (int w = 0; w < PK_WARPS; ++w) {
        if (wcnt[w] >= PK_MAX_ROUNDS) continue;
        if (best < 0 || wload[w] < wload[best] || (wload[w] == wload[best] && sub[w & 3] < sub[best & 3])) best = w;
      }
      if (best < 0) return GBE_EINVAL;  // cannot happen: a bin holds at most 16 x 32 units
      grid[(size_t)wcnt[best] * PK_WARPS + best] = pk_encode(un.slot, un.bi, un.bj, un.nb, un.tall);
      rounds = std::max(rounds, ++wcnt[best]);
      wload[best] += un.cost;
      sub[best & 3] += un.cost;
    }
    c.n_rounds = rounds;
    rounds_max = std::max(rounds_max, rounds);
    grids.push_back(std::move(grid));
    h_ctas.push_back(c);
  }
  std::vector<uint16_t> h_codes;
  for (const auto& gr : grids) h_codes.insert(h_codes.end(), gr.begin(), gr.begin() + (size_t)rounds_max * PK_WARPS);
  gbe_pk_class& out = g->pk[0];
  out.n_ctas = (int32_t)h_ctas.size();
  out.warps = PK_WARPS;
  out.smem_bytes = smem_need;
  out.rounds_max = rounds_max;
  out.code_stride = rounds_max * PK_WARPS;
  GBE_TRY(upload(h_ctas, &out.ctas, s));
  GBE_TRY(upload(h_codes, &out.codes, s));
  GBE_TRY(upload(h_rows, &out.rows, s));
  g->n_pk_ctas = out.n_ctas;
  return GBE_OK;
}

// One SP2 iteration of the packed communities.  partial_base: index of the first bin's pair in `partials` (the pairs of the
// tiled kernel, if it runs in the same iteration, sit in front); n_partials: all pairs of the iteration.
int gbe_launch_sp2_packed(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials,
                          int partial_base, int n_partials, int iter, bool last, int fused, int lazy_base, int lazy_n,
                          cudaStream_t s) {
  if (g->n_pk_ctas == 0) return GBE_OK;
  static gbe_device_once configured;
  if (configured.first()) {
    int dev = 0, smem_max = 0;
    GBE_CUDA(cudaGetDevice(&dev));
    GBE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    GBE_CUDA(cudaFuncSetAttribute(k_sp2_packed, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - 2048));
    GBE_CUDA(cudaFuncSetAttribute(k_sp2_packed, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
  }
  const gbe_pk_class& a = g->pk[0];
  // programmatic stream serialisation: the grid may be scheduled before the previous kernel of the stream has finished;
  // it synchronises with it in the kernel (griddepcontrol.wait) after its set-up
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)a.n_ctas);
  cfg.blockDim = dim3(PK_THREADS);
  cfg.dynamicSmemBytes = a.smem_bytes;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = gbe_pdl_enabled() ? 1 : 0;
  GBE_CUDA(cudaLaunchKernelEx(&cfg, k_sp2_packed, (const gbe_pk_cta*)a.ctas, (const uint16_t*)a.codes,
                              (const gbe_pk_row*)a.rows, st, Xin, Xout,
                              partials, partial_base, n_partials, iter, last ? 1 : 0, fused, (int)a.code_stride,
                              (int)a.rounds_max, lazy_base, lazy_n));
  GBE_LAUNCHED();
  return GBE_OK;
}
