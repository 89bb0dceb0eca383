// Step 1 - the data-dependency graph S_tau (row 1).
//
// Reading A-1 of Eq.(2) P:L38-40 (in the spirit of Eq.(8)):
//     A = floor(X0)_tau,  X0 = (eps_max I - H)/(eps_max - eps_min)       (|value| >= tau kept, A-3)
//     T^(1) = A,  T^(n) = floor(A T^(n-1))_tau,  n = 2..power
//     S = I u pat(T^(1)) u ... u pat(T^(power)),  then S u S^T          (self loops: T^(0) = I, A-4)
//
// Every kernel is warp-per-row CSR work with a per-warp bitmap over the n columns in shared memory:
//   - the thresholded product is a row-wise (Gustavson, ref. 18 P:L132) accumulation: pass 1 marks the candidate
//     columns in the bitmap, a popcount prefix turns the bitmap into a compact slot index, pass 2 accumulates
//     a_ik * t_kj into the compact accumulator with k ASCENDING and a separate multiply and add, so the value of
//     every entry does not depend on scheduling (and A A is bitwise symmetric when H is);
//   - walking the bitmap emits the columns in ascending order, so no sort is ever needed;
//   - the candidate bitmaps of pass 1 are computed once (the sizing pass keeps them in global memory for the numeric
//     pass, gbe_set_build_scratch_limit), and with the default power 2 only the upper triangle of A A is formed, each
//     walk starting at the first column >= i of every T row (k_first_upper).
// Bound: instruction issue and the latency of dependent L2 loads at 3-4 warps per scheduler (the bitmap, its ranks and
// the accumulator of every warp live in shared memory); ncu counters in profiles/r01_spgemm_ncu.md.
#include "gbe_internal.cuh"

static std::atomic<size_t> g_bm_save_max{(size_t)8 << 30};  // gbe_set_build_scratch_limit
size_t gbe_set_build_scratch_limit(size_t bytes) { return g_bm_save_max.exchange(bytes); }

namespace {


__device__ __forceinline__ double x0_entry(double h, bool diag, double eps_max, double delta) {
  return ((diag ? eps_max : 0.0) - h) / delta;
}

// ---------------------------------------------------------------- A = floor(X0)_tau with an explicit diagonal
template <bool FILL>
__global__ void __launch_bounds__(256) k_materialise_A(int64_t n, const int64_t* __restrict__ rp,
                                                       const int32_t* __restrict__ col, const double* __restrict__ val,
                                                       const gbe_state* __restrict__ st, double tau,
                                                       int32_t* __restrict__ cnt, const int64_t* __restrict__ out_rp,
                                                       int32_t* __restrict__ out_col, double* __restrict__ out_val) {
  const int lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (i >= n) return;
  const double eps_max = st->eps_max, delta = st->eps_max - st->eps_min;
  const int64_t a = rp[i], b = rp[i + 1];
  // does the row store its diagonal?  (A-12: a missing diagonal means H_ii = 0, X0_ii = eps_max/delta)
  int has = 0;
  for (int64_t e = a + lane; e < b; e += 32) has |= (col[e] == i);
  has = __any_sync(0xffffffffu, has);
  const double dmiss = x0_entry(0.0, true, eps_max, delta);
  const bool ins = !has && fabs(dmiss) >= tau;
  int kept = 0, less = 0;  // kept entries so far; kept entries with column < i
  const int64_t ob = FILL ? out_rp[i] : 0;
  for (int64_t e0 = a; e0 < b; e0 += 32) {
    const int64_t e = e0 + lane;
    int c = -1;
    double x = 0.0;
    bool keep = false;
    if (e < b) {
      c = col[e];
      x = x0_entry(val[e], c == i, eps_max, delta);
      keep = fabs(x) >= tau;
    }
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    const unsigned ml = __ballot_sync(0xffffffffu, keep && c < i);
    if (FILL && keep) {
      const int pos = kept + __popc(m & ((1u << lane) - 1)) + ((ins && c > i) ? 1 : 0);
      out_col[ob + pos] = c;
      out_val[ob + pos] = x;
    }
    kept += __popc(m);
    less += __popc(ml);
  }
  if (lane == 0) {
    if (FILL) {
      if (ins) { out_col[ob + less] = (int32_t)i; out_val[ob + less] = dmiss; }
    } else {
      cnt[i] = kept + (ins ? 1 : 0);
    }
  }
}

// ---------------------------------------------------------------- T_next = floor(A T)_tau
// Walks every product a_ik * t_kj of row i (k ascending; the entries of one T row spread over the lanes) and calls
// fn(aik, j[4], t_kj[4]) once per ROUND of up to 128 entries of one T row (4 per lane; j = -1 marks an empty slot).
// The kernels around it are bound by instruction issue and by the latency of dependent loads from L2 (ncu: the
// integer and branch instructions around each product were ~10 times the useful ones), so the walk is written to
// be cheap and flat: the 32 lanes fetch the row pointers of 32 neighbours k at once (and the neighbour indices of
// the NEXT 32 while these are walked); a warp scan numbers the rounds of the 32 T rows, so that round r is located
// with one ballot and two shuffles instead of a search loop; each round costs one 64-bit address per array and
// predicated loads at immediate offsets with 32-bit bounds; the loads of round r + 1 are in flight while round r is
// processed.  ORDERED: a __syncwarp follows every round, because the next k may hit the accumulator slots of this one.
template <bool NEED_VAL, bool ORDERED, bool CONSEC, typename F>
__device__ __forceinline__ void walk_products(int lane, int64_t a, int64_t b, const int32_t* __restrict__ A_col,
                                              const double* __restrict__ A_val, const int64_t* __restrict__ T_rp,
                                              const int32_t* __restrict__ T_col, const double* __restrict__ T_val,
                                              const int64_t* __restrict__ T_start, F&& fn) {
  // T_start (may be null): per entry e = (i, k) of the A row, the offset in T of the first entry of row k that counts
  // (k_first_upper: the first column >= i when only the upper triangle is formed); null: the whole row, from T_rp[k]
  constexpr unsigned FULL = 0xffffffffu;
  struct Buf {
    int j[4];
    double v[4];
    int q;
  };
  int kk_n = a + lane < b ? A_col[a + lane] : -1;
  double av_n = (NEED_VAL && a + lane < b) ? A_val[a + lane] : 0.0;
  for (int64_t e0 = a; e0 < b; e0 += 32) {
    const int kk = kk_n;
    const double av = av_n;
    const int64_t tb_l = kk >= 0 ? (T_start ? T_start[e0 + lane] : T_rp[kk]) : 0;
    const int64_t te_l = kk >= 0 ? T_rp[kk + 1] : 0;
    {  // neighbour indices of the next 32: in flight during this block
      const int64_t en = e0 + 32 + lane;
      kk_n = en < b ? A_col[en] : -1;
      if (NEED_VAL) av_n = en < b ? A_val[en] : 0.0;
    }
    const int len_l = (int)(te_l - tb_l);
    const int rounds_l = (len_l + 127) >> 7;
    int R;
    const int ex_l = warp_excl_scan_i(rounds_l, lane, &R);
    const int cum_l = ex_l + rounds_l;
    const int64_t tbx_l = tb_l - ((int64_t)ex_l << 7);  // round r of this k starts at tbx + 128 r ...
    const int lenx_l = len_l + (ex_l << 7);              // ... and holds the entries below lenx - 128 r
    auto load = [&](int r, Buf& B) {
      const int q = __ffs(__ballot_sync(FULL, cum_l > r)) - 1;  // the first k whose rounds end beyond r owns round r
      // CONSEC: a lane takes 4 consecutive entries of the round (its columns are neighbours), else entries 32 apart
      constexpr int LS = CONSEC ? 4 : 1, US = CONSEC ? 1 : 32;
      const int64_t first = __shfl_sync(FULL, tbx_l, q) + ((int64_t)r << 7) + LS * lane;
      const int left = __shfl_sync(FULL, lenx_l, q) - (r << 7) - LS * lane;  // entries from this lane's first one on
      B.q = q;
      const int32_t* __restrict__ cp = T_col + first;
      const double* __restrict__ vp = T_val + first;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        B.j[u] = US * u < left ? cp[US * u] : -1;
        if (NEED_VAL) B.v[u] = US * u < left ? vp[US * u] : 0.0;
      }
    };
    auto process = [&](const Buf& B) {
      const double aik = NEED_VAL ? __shfl_sync(FULL, av, B.q) : 0.0;
      fn(aik, B.j, B.v);
      if (ORDERED) __syncwarp();
    };
    Buf b0, b1;
    if (0 < R) load(0, b0);
    for (int r = 0; r < R; r += 2) {
      if (r + 1 < R) load(r + 1, b1);
      process(b0);
      if (r + 1 >= R) break;
      if (r + 2 < R) load(r + 2, b0);
      process(b1);
    }
  }
}

// Upper triangle only (A A with A symmetric): of row k the product for row i needs the columns j >= i.  One binary
// search per entry (i, k) of A, all in parallel, finds where they start, so that the walks neither load nor test the
// rest (half of all entries, and rows longer than 128 entries mostly fit one round again).
__global__ void __launch_bounds__(256) k_first_upper(int64_t n, const int64_t* __restrict__ rp,
                                                     const int32_t* __restrict__ col, int64_t* __restrict__ start) {
  const int lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (i >= n) return;
  for (int64_t e = rp[i] + lane; e < rp[i + 1]; e += 32) {
    const int k = col[e];
    int64_t lo = rp[k], hi = rp[k + 1];
    while (lo < hi) {
      const int64_t mid = (lo + hi) >> 1;
      if (col[mid] < i) lo = mid + 1; else hi = mid;
    }
    start[e] = lo;
  }
}

// MODE 0: distinct candidate columns per row (sizes the accumulator); 1: count kept entries; 2: fill (columns + values);
// 3: one pass for the LAST power, whose values are not needed: kept columns go to a scratch row of candidate capacity
//    (offsets out_rp from MODE 0's counts) and cnt[i] = number kept.
// 4: symbolic product (Eq.(8) with eps = 0: "paths of length two"): emits every candidate column at out_rp.
template <int MODE>
__global__ void k_spgemm_threshold(int64_t n, int W, int cap, int upper_only, const int64_t* __restrict__ A_rp,
                                   const int32_t* __restrict__ A_col, const double* __restrict__ A_val,
                                   const int64_t* __restrict__ T_rp, const int32_t* __restrict__ T_col,
                                   const double* __restrict__ T_val, double tau, int32_t* __restrict__ cnt,
                                   const int64_t* __restrict__ out_rp, int32_t* __restrict__ out_col,
                                   double* __restrict__ out_val, uint32_t* __restrict__ bm_io,
                                   const int64_t* __restrict__ T_start) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, w_in_blk = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const size_t per_warp = (size_t)W * 8 + ((MODE == 0 || MODE == 4) ? 0 : (size_t)cap * 8);
  unsigned char* base = smem_raw + per_warp * w_in_blk;
  double* acc = reinterpret_cast<double*>(base);  // cap doubles (first: keeps 8-byte alignment)
  uint32_t* bm = reinterpret_cast<uint32_t*>(base + ((MODE == 0 || MODE == 4) ? 0 : (size_t)cap * 8));
  uint32_t* rk = bm + W;

  for (int64_t i = (int64_t)blockIdx.x * nw + w_in_blk; i < n; i += (int64_t)gridDim.x * nw) {
    const int64_t a = A_rp[i], b = A_rp[i + 1];
    // pass 1: mark candidate columns
    // upper_only: the product is A A with A symmetric, so (A A)_ij == (A A)_ji bit for bit (k ascending, the two
    // factors of every product commute) and only the columns j >= i are formed; S u S^T restores the rest
    const int jmin = upper_only ? (int)i : 0;
    // bm_io: MODE 0 (the sizing pass) leaves its candidate bitmaps there and the later modes of the same product
    // read them back (W coalesced words per row) instead of walking the products a second time
    const bool reload = MODE != 0 && bm_io != nullptr;
    if (reload) {
      for (int w = lane; w < W; w += 32) bm[w] = bm_io[(size_t)i * W + w];
    } else {
    for (int w = lane; w < W; w += 32) bm[w] = 0u;
    __syncwarp();
    // The columns of a T row are sorted, so the entries of one round hit few bitmap words and their atomics serialise
    // (ncu: 79 % of the shared-memory wavefronts of the sizing pass were conflicts).  Here a lane holds 4 CONSECUTIVE
    // entries and merges those that share a word before it issues an atomic.
    walk_products<false, false, true>(lane, a, b, A_col, A_val, T_rp, T_col, T_val, T_start,
                                      [&](double, const int (&j)[4], const double (&)[4]) {
      int cw = -1;
      unsigned cb = 0u;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const bool ok = j[u] >= jmin;  // an empty slot is -1 < jmin
        const int w = ok ? (j[u] >> 5) : -1;
        const unsigned bit = ok ? (1u << (j[u] & 31)) : 0u;
        if (w != cw) {
          if (cw >= 0) atomicOr(&bm[cw], cb);
          cw = w;
          cb = bit;
        } else {
          cb |= bit;
        }
      }
      if (cw >= 0) atomicOr(&bm[cw], cb);
    });
    }
    __syncwarp();
    if (MODE == 0 && bm_io != nullptr)
      for (int w = lane; w < W; w += 32) bm_io[(size_t)i * W + w] = bm[w];
    // compact slot index: rk[w] = number of candidates in words < w
    int running = 0;
    for (int w0 = 0; w0 < W; w0 += 32) {
      const int w = w0 + lane;
      const int c = w < W ? __popc(bm[w]) : 0;
      int tot;
      const int ex = warp_excl_scan_i(c, lane, &tot);
      if (w < W) rk[w] = running + ex;
      running += tot;
    }
    if constexpr (MODE == 0) {
      if (lane == 0) cnt[i] = running;
      __syncwarp();
    } else if constexpr (MODE == 4) {
      const int64_t ob4 = out_rp[i];
      for (int w = lane; w < W; w += 32) {
        uint32_t bits = bm[w];
        int pos = (int)rk[w];
        while (bits) {
          const int bpos = __ffs(bits) - 1;
          bits &= bits - 1;
          out_col[ob4 + pos++] = w * 32 + bpos;
        }
      }
      __syncwarp();
    } else {
    for (int s = lane; s < running; s += 32) acc[s] = 0.0;
    __syncwarp();
    // pass 2: accumulate, k ascending, multiply and add separately rounded
    // branch free, the four entries of a lane as independent chains (the columns of one T row are distinct, so
    // their slots are): entries that do not count (empty, or j < jmin) go to the spare slot cap - 1
    walk_products<true, true, false>(lane, a, b, A_col, A_val, T_rp, T_col, T_val, T_start,
                              [&](double aik, const int (&j)[4], const double (&t)[4]) {
      int slot[4];
      double o[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const bool ok = j[u] >= jmin;
        const int jj = ok ? j[u] : 0;
        const uint32_t word = bm[jj >> 5];
        const int sl = rk[jj >> 5] + __popc(word & ((1u << (jj & 31)) - 1u));
        slot[u] = ok ? sl : cap - 1;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) o[u] = acc[slot[u]];
#pragma unroll
      for (int u = 0; u < 4; ++u) acc[slot[u]] = __dadd_rn(o[u], __dmul_rn(aik, t[u]));
    });
    // emit kept entries in ascending column order
    int kept = 0;
    const int64_t ob = (MODE == 2 || MODE == 3) ? out_rp[i] : 0;
    for (int w0 = 0; w0 < W; w0 += 32) {
      const int w = w0 + lane;
      uint32_t bits = w < W ? bm[w] : 0u;
      const int s0 = w < W ? (int)rk[w] : 0;
      int mine = 0;
      {
        uint32_t t = bits;
        int idx = 0;
        while (t) {
          t &= t - 1;
          if (fabs(acc[s0 + idx]) >= tau) ++mine;
          ++idx;
        }
      }
      int tot;
      const int ex = warp_excl_scan_i(mine, lane, &tot);
      if (MODE == 2 || MODE == 3) {
        int pos = kept + ex, idx = 0;
        while (bits) {
          const int bpos = __ffs(bits) - 1;
          bits &= bits - 1;
          const double v = acc[s0 + idx];
          ++idx;
          if (fabs(v) >= tau) {
            out_col[ob + pos] = w * 32 + bpos;
            if (MODE == 2) out_val[ob + pos] = v;
            ++pos;
          }
        }
      }
      kept += tot;
    }
    if ((MODE == 1 || MODE == 3) && lane == 0) cnt[i] = kept;
    __syncwarp();
    }  // numeric modes
  }
}

// ---------------------------------------------------------------- row-wise union of two patterns (+ self loops)
template <bool FILL>
__global__ void k_union_rows(int64_t n, int W, const int64_t* __restrict__ P_rp, const int32_t* __restrict__ P_col,
                             const double* __restrict__ P_val /* null: pattern only */, double p_tau,
                             const int64_t* __restrict__ Q_rp, const int32_t* __restrict__ Q_col,
                             const int32_t* __restrict__ Q_len /* null: compact CSR */, int add_diag,
                             int32_t* __restrict__ cnt, const int64_t* __restrict__ out_rp,
                             int32_t* __restrict__ out_col) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, w_in_blk = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t* bm = reinterpret_cast<uint32_t*>(smem_raw) + (size_t)W * w_in_blk;
  for (int64_t i = (int64_t)blockIdx.x * nw + w_in_blk; i < n; i += (int64_t)gridDim.x * nw) {
    for (int w = lane; w < W; w += 32) bm[w] = 0u;
    __syncwarp();
    for (int64_t e = P_rp[i] + lane; e < P_rp[i + 1]; e += 32) {
      const int j = P_col[e];
      if ((unsigned)j < (uint64_t)n && (!P_val || fabs(P_val[e]) >= p_tau)) atomicOr(&bm[j >> 5], 1u << (j & 31));
    }
    if (Q_rp) {
      const int64_t qb = Q_rp[i], qe = Q_len ? qb + Q_len[i] : Q_rp[i + 1];
      for (int64_t e = qb + lane; e < qe; e += 32) {
        const int j = Q_col[e];
        if ((unsigned)j < (uint64_t)n) atomicOr(&bm[j >> 5], 1u << (j & 31));
      }
    }
    if (add_diag && lane == 0) atomicOr(&bm[i >> 5], 1u << (i & 31));
    __syncwarp();
    int total = 0;
    const int64_t ob = FILL ? out_rp[i] : 0;
    for (int w0 = 0; w0 < W; w0 += 32) {
      const int w = w0 + lane;
      uint32_t bits = w < W ? bm[w] : 0u;
      int tot;
      const int ex = warp_excl_scan_i(__popc(bits), lane, &tot);
      if (FILL) {
        int pos = total + ex;
        while (bits) {
          const int bpos = __ffs(bits) - 1;
          bits &= bits - 1;
          out_col[ob + pos++] = w * 32 + bpos;
        }
      }
      total += tot;
    }
    if (!FILL && lane == 0) cnt[i] = total;
    __syncwarp();
  }
}

// ---------------------------------------------------------------- transpose of a pattern (rows left unsorted)
__global__ void k_transpose_count(int64_t n, const int64_t* __restrict__ rp, const int32_t* __restrict__ col,
                                  int32_t* __restrict__ cnt) {
  const int lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (i >= n) return;
  for (int64_t e = rp[i] + lane; e < rp[i + 1]; e += 32) atomicAdd(&cnt[col[e]], 1);
}
__global__ void k_transpose_fill(int64_t n, const int64_t* __restrict__ rp, const int32_t* __restrict__ col,
                                 const int64_t* __restrict__ t_rp, int32_t* __restrict__ cursor,
                                 int32_t* __restrict__ t_col) {
  const int lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (i >= n) return;
  for (int64_t e = rp[i] + lane; e < rp[i + 1]; e += 32) {
    const int j = col[e];
    const int pos = atomicAdd(&cursor[j], 1);
    t_col[t_rp[j] + pos] = (int32_t)i;
  }
}

// ---------------------------------------------------------------- optional symmetry check of H
__global__ void k_check_symmetric(int64_t n, const int64_t* __restrict__ rp, const int32_t* __restrict__ col,
                                  const double* __restrict__ val, int32_t* __restrict__ flag) {
  const int lane = threadIdx.x & 31;
  const int64_t i = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (i >= n) return;
  for (int64_t e = rp[i] + lane; e < rp[i + 1]; e += 32) {
    const int j = col[e];
    const double v = val[e];
    if (j < 0 || j >= n) { atomicOr(flag, 2); continue; }
    int64_t lo = rp[j], hi = rp[j + 1];
    while (lo < hi) {
      const int64_t mid = (lo + hi) >> 1;
      if (col[mid] < i) lo = mid + 1; else hi = mid;
    }
    bool ok = lo < rp[j + 1] && col[lo] == i;
    if (ok) {
      // exact equality: with the default power 2 only the upper triangle of floor(A A)_tau is formed, which is the whole
      // product only if A is symmetric bit for bit (an entry within rounding of tau could otherwise differ from its mirror)
      ok = val[lo] == v;
    } else {
      ok = (v == 0.0);  // an explicitly stored zero needs no partner
    }
    if (!ok) atomicOr(flag, 1);
  }
}

int pick_warps(size_t per_warp, int max_warps) {
  const size_t budget = 200 * 1024;
  int nw = (int)(budget / (per_warp ? per_warp : 1));
  if (nw > max_warps) nw = max_warps;
  return nw;
}

struct Pattern {  // device CSR (pattern, optionally with values) owned by DevBufs
  DevBuf rp, col, val;
  int64_t nnz = 0;
};

// row counts -> row pointers.  ub < 0: the total comes back to the host (one synchronisation); ub >= 0: a known upper
// bound of the total - the caller sizes its arrays with it and nothing comes back (*nnz = ub; the exact total is rp[n])
int count_to_rowptr(DevBuf& cnt, int64_t n, DevBuf& rp, int64_t* nnz, cudaStream_t s, int64_t ub = -1);

// row-wise unions on the device: out = [I u] filter(P) u Q
struct Unioner {
  int64_t n = 0;
  int W = 0, uw = 0, ugrid = 0;
  size_t bm_bytes = 0;
  cudaStream_t s = nullptr;
  DevBuf ucnt;  // row counts of the union being sized
  int init(int64_t n_, cudaStream_t s_) {
    n = n_;
    s = s_;
    W = (int)((n + 31) / 32);
    bm_bytes = (size_t)W * 4;
    const int sm_count = gbe_sm_count();  // of the current device
    uw = pick_warps(bm_bytes, 8);
    if (uw < 1) return GBE_EINVAL;  // n too large for a shared-memory bitmap
    GBE_CUDA(cudaFuncSetAttribute(k_union_rows<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bm_bytes * uw)));
    GBE_CUDA(cudaFuncSetAttribute(k_union_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bm_bytes * uw)));
    ugrid = (int)std::min<int64_t>((n + uw - 1) / uw, (int64_t)sm_count * 8);
    return ucnt.alloc((size_t)n * 4);
  }
  int run(const int64_t* p_rp, const int32_t* p_col, const double* p_val, double p_tau, const int64_t* q_rp,
          const int32_t* q_col, const int32_t* q_len, int diag, Pattern& out, int64_t ub = -1) {
    k_union_rows<false><<<ugrid, uw * 32, bm_bytes * uw, s>>>(n, W, p_rp, p_col, p_val, p_tau, q_rp, q_col, q_len, diag,
                                                              ucnt.as<int32_t>(), nullptr, nullptr);
    GBE_LAUNCHED();
    GBE_TRY(count_to_rowptr(ucnt, n, out.rp, &out.nnz, s, ub));
    GBE_TRY(out.col.alloc((size_t)out.nnz * 4));
    k_union_rows<true><<<ugrid, uw * 32, bm_bytes * uw, s>>>(n, W, p_rp, p_col, p_val, p_tau, q_rp, q_col, q_len, diag,
                                                             nullptr, out.rp.as<int64_t>(), out.col.as<int32_t>());
    GBE_LAUNCHED();
    return GBE_OK;
  }
};

// S = P u P^T (P's rows need not be sorted on input; S's are ascending).  P.nnz may be an upper bound.  S is sized
// EXACTLY (one synchronisation): it is the one array of the build that outlives it, and sized by the bound 2 nnz(P) it was
// a block of tens of MB that cycled through the stream-ordered pool on every build - with the host running ahead of the
// device (back-to-back builds of an MD loop) the pool then stalled for 0.1 - 0.9 s at a time
int symmetrise(Pattern& P, Unioner& U, DevBuf& cnt, Pattern& S) {
  const int64_t n = U.n;
  cudaStream_t s = U.s;
  const int rows_grid = (int)((n + 7) / 8);
  Pattern PT;
  GBE_CUDA(cudaMemsetAsync(cnt.p, 0, (size_t)n * 4, s));
  k_transpose_count<<<rows_grid, 256, 0, s>>>(n, P.rp.as<int64_t>(), P.col.as<int32_t>(), cnt.as<int32_t>());
  GBE_LAUNCHED();
  GBE_TRY(count_to_rowptr(cnt, n, PT.rp, &PT.nnz, s, P.nnz));  // a transpose has as many entries
  GBE_TRY(PT.col.alloc((size_t)PT.nnz * 4));
  GBE_CUDA(cudaMemsetAsync(cnt.p, 0, (size_t)n * 4, s));
  k_transpose_fill<<<rows_grid, 256, 0, s>>>(n, P.rp.as<int64_t>(), P.col.as<int32_t>(), PT.rp.as<int64_t>(),
                                             cnt.as<int32_t>(), PT.col.as<int32_t>());
  GBE_LAUNCHED();
  GBE_TRY(U.run(P.rp.as<int64_t>(), P.col.as<int32_t>(), nullptr, 0.0, PT.rp.as<int64_t>(), PT.col.as<int32_t>(), nullptr,
                0, S));
  return GBE_OK;
}

int count_to_rowptr(DevBuf& cnt, int64_t n, DevBuf& rp, int64_t* nnz, cudaStream_t s, int64_t ub) {
  GBE_TRY(rp.alloc((size_t)(n + 1) * 8));
  GBE_TRY(gbe_exclusive_scan_i32_to_i64(cnt.as<int32_t>(), rp.as<int64_t>(), n, s));
  if (ub >= 0) {
    *nnz = ub;
    return GBE_OK;
  }
  GBE_CUDA(cudaMemcpyAsync(nnz, rp.as<int64_t>() + n, 8, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  return GBE_OK;
}

}  // namespace

// Outputs sized by upper bounds are kept below this many bytes; beyond it the exact sizes are fetched (more
// synchronisations, less memory)
static const size_t UB_BYTES_MAX = (size_t)4 << 30;

int gbe_build_pattern(const gbe_csr_view& H, const gbe_state* st, double tau, int power, int check_sym,
                      cudaStream_t s, int64_t** S_row_ptr, int32_t** S_col, int64_t* nnz_S) {
  const int64_t n = H.n;
  const int W = (int)((n + 31) / 32);
  const int rows_grid = (int)((n + 7) / 8);
  const int sm_count = gbe_sm_count();  // of the current device

  if (check_sym) {
    DevBuf flag;
    GBE_TRY(flag.alloc(4));
    GBE_CUDA(cudaMemsetAsync(flag.p, 0, 4, s));
    k_check_symmetric<<<rows_grid, 256, 0, s>>>(n, H.row_ptr, H.col_idx, H.val, flag.as<int32_t>());
    GBE_LAUNCHED();
    int32_t f = 0;
    GBE_CUDA(cudaMemcpyAsync(&f, flag.p, 4, cudaMemcpyDeviceToHost, s));
    GBE_CUDA(cudaStreamSynchronize(s));
    if (f & 2) return GBE_EINVAL;
    if (f) return GBE_ENOTSYM;
  }
  DevBuf cnt;
  GBE_TRY(cnt.alloc((size_t)n * 4));

  // A = floor(X0)_tau, explicit diagonal
  Pattern A;
  k_materialise_A<false><<<rows_grid, 256, 0, s>>>(n, H.row_ptr, H.col_idx, H.val, st, tau, cnt.as<int32_t>(), nullptr,
                                                   nullptr, nullptr);
  GBE_LAUNCHED();
  GBE_TRY(count_to_rowptr(cnt, n, A.rp, &A.nnz, s, H.nnz + n));  // at most the stored entries + the missing diagonals
  GBE_TRY(A.col.alloc((size_t)A.nnz * 4));
  GBE_TRY(A.val.alloc((size_t)A.nnz * 8));
  k_materialise_A<true><<<rows_grid, 256, 0, s>>>(n, H.row_ptr, H.col_idx, H.val, st, tau, nullptr, A.rp.as<int64_t>(),
                                                  A.col.as<int32_t>(), A.val.as<double>());
  GBE_LAUNCHED();
  // pattern accumulator P = I u pat(A)
  Unioner U;
  GBE_TRY(U.init(n, s));
  DevBuf& ucnt = U.ucnt;
  (void)ucnt;
  auto do_union = [&](const int64_t* p_rp, const int32_t* p_col, const int64_t* q_rp, const int32_t* q_col,
                      const int32_t* q_len, int diag, Pattern& out, int64_t ub = -1) -> int {
    return U.run(p_rp, p_col, nullptr, 0.0, q_rp, q_col, q_len, diag, out, ub);
  };

  // (with the default power 2 the union with the second power below takes I and pat(A) directly: one union less)
  Pattern P;
  const bool P_built = power != 2;
  if (P_built) GBE_TRY(do_union(A.rp.as<int64_t>(), A.col.as<int32_t>(), nullptr, nullptr, nullptr, 1, P, A.nnz + n));
  // thresholded powers
  Pattern Tprev;  // T^(k-1) with values; T^(1) aliases A
  const int64_t* T_rp = A.rp.as<int64_t>();
  const int32_t* T_col = A.col.as<int32_t>();
  const double* T_val = A.val.as<double>();
  // candidate bitmaps of the sizing pass, kept for the numeric passes of the same product (n * W words: only while
  // that is a small part of the device memory - beyond it the numeric passes walk the products again)
  DevBuf bmsave;
  const size_t BM_SAVE_MAX = g_bm_save_max;
  if ((size_t)n * W * 4 <= BM_SAVE_MAX && power >= 2 && bmsave.alloc((size_t)n * W * 4) != GBE_OK) {
    (void)cudaGetLastError();  // no room for the bitmaps: not an error, the numeric passes walk the products again
    bmsave.p = nullptr;
  }
  uint32_t* const bm_io = bmsave.as<uint32_t>();
  for (int k = 2; k <= power; ++k) {
    // A A with symmetric A is symmetric bit for bit: when it is the LAST power only its upper triangle is formed
    const int upper_only = (k == 2 && power == 2) ? 1 : 0;
    // upper triangle only: where the columns j >= i start in every row k of every entry (i, k)
    DevBuf tstart;
    const int64_t* t_start = nullptr;
    if (upper_only) {
      GBE_TRY(tstart.alloc((size_t)A.nnz * 8));
      k_first_upper<<<rows_grid, 256, 0, s>>>(n, A.rp.as<int64_t>(), A.col.as<int32_t>(), tstart.as<int64_t>());
      GBE_LAUNCHED();
      t_start = tstart.as<int64_t>();
    }
    // symbolic: accumulator capacity
    {
      const size_t per_warp = (size_t)W * 8;
      const int nw = pick_warps(per_warp, 16);
      if (nw < 1) return GBE_EINVAL;
      GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
      const int grid = (int)std::min<int64_t>((n + nw - 1) / nw, (int64_t)sm_count * 8);
      k_spgemm_threshold<0><<<grid, nw * 32, per_warp * nw, s>>>(n, W, 0, upper_only, A.rp.as<int64_t>(),
                                                                 A.col.as<int32_t>(), A.val.as<double>(), T_rp, T_col, T_val, tau,
                                                                 cnt.as<int32_t>(), nullptr, nullptr, nullptr, bm_io, t_start);
      GBE_LAUNCHED();
    }
    // one scan gives the accumulator capacity (the largest candidate count) and the scratch-row offsets of the last
    // power (the running sum): 16 bytes come back to the host, one synchronisation
    Pattern Tc;  // scratch: rp = offsets by candidate count, col = kept columns, cnt = kept per row
    int64_t total_max[2] = {0, 0};
    GBE_TRY(Tc.rp.alloc((size_t)(n + 2) * 8));
    GBE_TRY(gbe_exclusive_scan_i32_to_i64_max(cnt.as<int32_t>(), Tc.rp.as<int64_t>(), n, s));
    GBE_CUDA(cudaMemcpyAsync(total_max, Tc.rp.as<int64_t>() + n, 16, cudaMemcpyDeviceToHost, s));
    GBE_CUDA(cudaStreamSynchronize(s));
    const int64_t total_cand = total_max[0];
    int cap = std::max<int>(1, (int)total_max[1]);
    cap = ((cap + 1) & ~1) + 2;  // + the spare slot that takes the entries that do not count
    const size_t per_warp = (size_t)W * 8 + (size_t)cap * 8;
    const int nw = pick_warps(per_warp, 16);
    if (nw < 1) return GBE_EINVAL;
    GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
    GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
    const int grid = (int)std::min<int64_t>((n + nw - 1) / nw, (int64_t)sm_count * 8);
    if (k == power) {
      // last power: only its pattern enters S - one numeric pass into scratch rows of candidate capacity
      GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
      GBE_TRY(Tc.col.alloc((size_t)total_cand * 4));
      k_spgemm_threshold<3><<<grid, nw * 32, per_warp * nw, s>>>(n, W, cap, upper_only, A.rp.as<int64_t>(),
                                                                 A.col.as<int32_t>(), A.val.as<double>(), T_rp, T_col, T_val, tau,
                                                                 cnt.as<int32_t>(), Tc.rp.as<int64_t>(),
                                                                 Tc.col.as<int32_t>(), nullptr, bm_io, t_start);
      GBE_LAUNCHED();
      // P u kept(T^(k)) has at most nnz(P) + candidates entries: sized by that bound while it is small, no count comes back
      Pattern Pn;
      const int64_t ub_base = (P_built ? P.nnz : A.nnz + n) + total_cand;
      const int64_t ub = (size_t)ub_base * 8 <= UB_BYTES_MAX ? ub_base : -1;
      if (P_built)
        GBE_TRY(do_union(P.rp.as<int64_t>(), P.col.as<int32_t>(), Tc.rp.as<int64_t>(), Tc.col.as<int32_t>(),
                         cnt.as<int32_t>(), 0, Pn, ub));
      else
        GBE_TRY(do_union(A.rp.as<int64_t>(), A.col.as<int32_t>(), Tc.rp.as<int64_t>(), Tc.col.as<int32_t>(),
                         cnt.as<int32_t>(), 1, Pn, ub));
      // (no synchronisation here: the scratch buffers are released in stream order)
      std::swap(P.rp.p, Pn.rp.p);
      std::swap(P.col.p, Pn.col.p);
      P.nnz = Pn.nnz;
      break;
    }
    Pattern Tn;
    k_spgemm_threshold<1><<<grid, nw * 32, per_warp * nw, s>>>(n, W, cap, 0, A.rp.as<int64_t>(), A.col.as<int32_t>(),
                                                               A.val.as<double>(), T_rp, T_col, T_val, tau,
                                                               cnt.as<int32_t>(), nullptr, nullptr, nullptr, bm_io, nullptr);
    GBE_LAUNCHED();
    GBE_TRY(count_to_rowptr(cnt, n, Tn.rp, &Tn.nnz, s));
    GBE_TRY(Tn.col.alloc((size_t)Tn.nnz * 4));
    GBE_TRY(Tn.val.alloc((size_t)Tn.nnz * 8));
    k_spgemm_threshold<2><<<grid, nw * 32, per_warp * nw, s>>>(n, W, cap, 0, A.rp.as<int64_t>(), A.col.as<int32_t>(),
                                                               A.val.as<double>(), T_rp, T_col, T_val, tau, nullptr,
                                                               Tn.rp.as<int64_t>(), Tn.col.as<int32_t>(),
                                                               Tn.val.as<double>(), bm_io, nullptr);
    GBE_LAUNCHED();
    Pattern Pn;
    GBE_TRY(do_union(P.rp.as<int64_t>(), P.col.as<int32_t>(), Tn.rp.as<int64_t>(), Tn.col.as<int32_t>(), nullptr, 0, Pn));
    GBE_CUDA(cudaStreamSynchronize(s));
    std::swap(P.rp.p, Pn.rp.p);
    std::swap(P.col.p, Pn.col.p);
    P.nnz = Pn.nnz;
    std::swap(Tprev.rp.p, Tn.rp.p);
    std::swap(Tprev.col.p, Tn.col.p);
    std::swap(Tprev.val.p, Tn.val.p);
    Tprev.nnz = Tn.nnz;
    T_rp = Tprev.rp.as<int64_t>();
    T_col = Tprev.col.as<int32_t>();
    T_val = Tprev.val.as<double>();
    // Tn (now holding the previous T) and Pn are released here, after the sync above
  }
  // S = P u P^T
  Pattern S;
  GBE_TRY(symmetrise(P, U, cnt, S));
  *nnz_S = S.nnz;
  *S_row_ptr = reinterpret_cast<int64_t*>(S.rp.release());
  *S_col = reinterpret_cast<int32_t*>(S.col.release());
  return GBE_OK;
}

// ---------------------------------------------------------------- Eq.(8): graph for the next MD step
//     S_tau(t) <- floor( ( floor(D(t - dt))_tau + H(t) )^2 )_eps,  used symbolically with eps = 0:
//     M = I u pat(|D_ij| >= tau) u pat(H(t)),   S = pat(M M) ("paths of length two"),  then S u S^T.
// D is the assembled, non-symmetric P_tau of the previous step on the pattern (D_rp, D_col).
int gbe_build_pattern_eq8(const gbe_csr_view& H, const int64_t* D_rp, const int32_t* D_col, const double* D_val, double tau,
                          cudaStream_t s, int64_t** S_row_ptr, int32_t** S_col, int64_t* nnz_S, int64_t nnz_D) {
  const int64_t n = H.n;
  const int W = (int)((n + 31) / 32);
  const int sm_count = gbe_sm_count();  // of the current device
  Unioner U;
  GBE_TRY(U.init(n, s));
  DevBuf cnt;
  GBE_TRY(cnt.alloc((size_t)n * 4));
  Pattern M;
  GBE_TRY(U.run(D_rp, D_col, D_val, tau, H.row_ptr, H.col_idx, nullptr, 1, M, nnz_D + H.nnz + n));
  // symbolic square: count the candidates of every row, then emit them
  const size_t per_warp = (size_t)W * 8;
  const int nw = pick_warps(per_warp, 16);
  if (nw < 1) return GBE_EINVAL;
  GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
  GBE_CUDA(cudaFuncSetAttribute(k_spgemm_threshold<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
  const int grid = (int)std::min<int64_t>((n + nw - 1) / nw, (int64_t)sm_count * 8);
  DevBuf bmsave;  // candidate bitmaps of the counting pass, read back by the emitting pass
  if ((size_t)n * W * 4 <= g_bm_save_max && bmsave.alloc((size_t)n * W * 4) != GBE_OK) {
    (void)cudaGetLastError();  // no room: the emitting pass walks the products again
    bmsave.p = nullptr;
  }
  uint32_t* const bm_io = bmsave.as<uint32_t>();
  k_spgemm_threshold<0><<<grid, nw * 32, per_warp * nw, s>>>(n, W, 0, 0, M.rp.as<int64_t>(), M.col.as<int32_t>(), nullptr,
                                                             M.rp.as<int64_t>(), M.col.as<int32_t>(), nullptr, 0.0,
                                                             cnt.as<int32_t>(), nullptr, nullptr, nullptr, bm_io, nullptr);
  GBE_LAUNCHED();
  Pattern P;
  GBE_TRY(count_to_rowptr(cnt, n, P.rp, &P.nnz, s));
  GBE_TRY(P.col.alloc((size_t)P.nnz * 4));
  k_spgemm_threshold<4><<<grid, nw * 32, per_warp * nw, s>>>(n, W, 0, 0, M.rp.as<int64_t>(), M.col.as<int32_t>(), nullptr,
                                                             M.rp.as<int64_t>(), M.col.as<int32_t>(), nullptr, 0.0, nullptr,
                                                             P.rp.as<int64_t>(), P.col.as<int32_t>(), nullptr, bm_io, nullptr);
  GBE_LAUNCHED();
  Pattern S;
  GBE_TRY(symmetrise(P, U, cnt, S));
  *nnz_S = S.nnz;
  *S_row_ptr = reinterpret_cast<int64_t*>(S.rp.release());
  *S_col = reinterpret_cast<int32_t*>(S.col.release());
  return GBE_OK;
}
