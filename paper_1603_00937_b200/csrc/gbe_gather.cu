// Step 3 - gather / pack (row 3).
//
//     x_p = X0[s_p, s_p],  X0 = (eps_max I - H)/(eps_max - eps_min)                         (A-2)
// the FULL principal submatrix: every stored H entry with both indices in s_p; zero elsewhere; the diagonal
// gets (eps_max - H_kk)/delta even when H_kk is not stored (A-12).  Output: row-major FP64 blocks,
// ld_p = m_p rounded up to 16 doubles (rows are 128-byte aligned), pad columns zero.
//
// One CTA handles `gather_rows` consecutive rows of one community.  The global -> local index translation is a
// pair of bitmaps (core, halo) over the n vertices with popcount-prefix ranks in shared memory: O(1) per
// stored entry, no search.  Each warp builds one output row in shared memory (zero fill + scattered entries)
// and streams it out with 128-bit stores, so every output byte is written exactly once, fully coalesced.
// The epilogue accumulates the traces of X_0 and X_0^2 over the core rows (t1, t2 of iteration 0):
// (X^2)_ii = sum_c X_ic^2 for symmetric X.
// DIRECT variant (large systems: the bitmaps of ~1e5 vertices plus row buffers of ~2,400 doubles leave one CTA per SM):
// no row buffer - the warp zero-fills the output row in global memory with 128-bit stores and then stores the stored
// entries straight to it (L2 merges the two before the line leaves for DRAM), so the CTA needs the bitmaps only and
// three CTAs fit an SM.  The traces are then summed over the stored entries as they are placed.
// Bound: HBM - writes 8 m_p^2 B per community, reads 12 B per stored entry of every gathered H row.
#include "gbe_internal.cuh"

namespace {

template <bool DIRECT>
__global__ void __launch_bounds__(256, 3) k_gather(int W, int ldmax, int rows_per_cta, const int2* __restrict__ gitems,
                                                const int64_t* __restrict__ H_rp, const int32_t* __restrict__ H_col,
                                                const double* __restrict__ H_val, int64_t n,
                                                const int64_t* __restrict__ sub_ptr, const int32_t* __restrict__ sub_idx,
                                                const int32_t* __restrict__ ncore_arr,
                                                const int64_t* __restrict__ dense_off, const gbe_state* __restrict__ st,
                                                double* __restrict__ X, double* __restrict__ partials) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint32_t* coreb = reinterpret_cast<uint32_t*>(smem_raw);
  uint32_t* halob = coreb + W;
  uint32_t* corerk = halob + W;
  uint32_t* halork = corerk + W;
  int* scratch = reinterpret_cast<int*>(halork + W);                      // 2 * 257 ints
  double* red = reinterpret_cast<double*>(scratch + 516);                  // 16 doubles (8-byte aligned: 4W*4 + 2064)
  double* rowbuf = red + 16;                                               // nwarps * ldmax doubles
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, nw = blockDim.x >> 5;
  const int2 it = gitems[blockIdx.x];
  const int p = it.x, r0 = it.y;
  const int64_t sb = sub_ptr[p];
  const int m = (int)(sub_ptr[p + 1] - sb);
  const int nc = ncore_arr[p];
  const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  // degenerate bounds (eps_max == eps_min, A-12: H is a multiple of I): the status travels with gbe_read_log; the values are
  // kept finite with delta = 1 (X0 = 0) so that a call without a log still writes a defined D
  const double eps_max = st->eps_max, delta = st->degenerate ? 1.0 : st->eps_max - st->eps_min;
  const double inv_delta = 1.0 / delta;
  // x / delta as a reciprocal multiply plus one residual correction: the correctly rounded quotient except in rare
  // half-ulp cases, at a tenth of the instructions of the IEEE division sequence (the row loop is issue bound)
  auto div_delta = [&](double x) {
    const double q = x * inv_delta;
    return fma(fma(-q, delta, x), inv_delta, q);
  };

  // bitmaps of the community's core and halo vertices
  for (int w = t; w < 2 * W; w += blockDim.x) coreb[w] = 0u;
  __syncthreads();
  for (int r = t; r < m; r += blockDim.x) {
    const int v = sub_idx[sb + r];
    atomicOr(r < nc ? &coreb[v >> 5] : &halob[v >> 5], 1u << (v & 31));
  }
  __syncthreads();
  // ranks: exclusive popcount prefix per word (both bitmaps at once)
  {
    const int nt = blockDim.x, chunk = (W + nt - 1) / nt;
    const int b = min(W, t * chunk), e = min(W, b + chunk);
    int c0 = 0, c1 = 0;
    for (int w = b; w < e; ++w) { c0 += __popc(coreb[w]); c1 += __popc(halob[w]); }
    scratch[t] = c0;
    scratch[258 + t] = c1;
    __syncthreads();
    for (int which = wid; which < 2; which += nw) {  // one warp each scans the per-thread counts of the core and the halo bitmap
      int* sc = scratch + 258 * which;
      int run = 0;
      for (int k0 = 0; k0 < nt; k0 += 32) {
        const int v = k0 + lane < nt ? sc[k0 + lane] : 0;
        int tot;
        const int ex = warp_excl_scan_i(v, lane, &tot);
        if (k0 + lane < nt) sc[k0 + lane] = run + ex;
        run += tot;
      }
    }
    __syncthreads();
    c0 = scratch[t];
    c1 = scratch[258 + t];
    for (int w = b; w < e; ++w) {
      corerk[w] = c0; c0 += __popc(coreb[w]);
      halork[w] = c1; c1 += __popc(halob[w]);
    }
  }
  __syncthreads();

  double* buf = DIRECT ? nullptr : rowbuf + (size_t)wid * ldmax;
  double* Xp = X + dense_off[p];
  double s1 = 0.0, s2 = 0.0;
  const int rend = min(m, r0 + rows_per_cta);
  // The row loop is latency bound (sub_idx -> H row pointers -> H entries are dependent loads), so it is software
  // pipelined: the vertex of the row after next, the row pointers of the next row and the first 128 entries of the
  // next row are in flight while the current row is scattered into shared memory and streamed out.
  auto fetch = [&](int64_t base, int64_t end, int (&j)[4], double (&v)[4]) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int64_t e = base + lane + 32 * u;
      j[u] = e < end ? H_col[e] : -1;
      v[u] = e < end ? H_val[e] : 0.0;
    }
  };
  double* out = nullptr;     // DIRECT: the output row being built
  double q = 0.0, dg = 0.0;  // DIRECT: this lane's sum of squares of the row, and the stored diagonal if it placed it
  bool dseen = false;
  auto place = [&](int k, const int (&j)[4], const double (&v)[4]) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int col = j[u];
      if (col < 0 || (int64_t)col >= n) continue;
      const uint32_t bit = 1u << (col & 31), wj = col >> 5;
      int c = -1;
      const uint32_t cw = coreb[wj];
      if (cw & bit) {
        c = corerk[wj] + __popc(cw & (bit - 1u));
      } else {
        const uint32_t hw = halob[wj];
        if (hw & bit) c = nc + halork[wj] + __popc(hw & (bit - 1u));
      }
      if (c >= 0) {
        const double x = div_delta((col == k ? eps_max : 0.0) - v[u]);
        if (DIRECT) {
          out[c] = x;
          q += x * x;
          if (col == k) { dseen = true; dg = x; }
        } else {
          buf[c] = x;
        }
      }
    }
  };
  int r = r0 + wid;
  int k0 = r < rend ? sub_idx[sb + r] : 0;
  int k1 = r + nw < rend ? sub_idx[sb + r + nw] : 0;
  int64_t a0 = 0, b0 = 0, a1 = 0, b1 = 0;
  int cj[4], nj[4];
  double cv[4], nv[4];
  if (r < rend) {
    a0 = H_rp[k0];
    b0 = H_rp[k0 + 1];
    fetch(a0, b0, cj, cv);
  }
  for (; r < rend; r += nw) {
    const bool has1 = r + nw < rend;
    const int k2 = r + 2 * nw < rend ? sub_idx[sb + r + 2 * nw] : 0;
    if (has1) {
      a1 = H_rp[k1];
      b1 = H_rp[k1 + 1];
    }
    double* const zrow = DIRECT ? Xp + (size_t)r * ld : buf;
    for (int c = lane * 2; c < ld; c += 64) *reinterpret_cast<double2*>(zrow + c) = make_double2(0.0, 0.0);
    __syncwarp();  // orders the zero fill before the entries other lanes store into the same row
    if (DIRECT) {
      out = zrow;
      q = 0.0;
      dseen = false;
    } else {
      if (lane == 0) buf[r] = div_delta(eps_max - 0.0);  // a stored diagonal overwrites this below
      __syncwarp();
    }
    for (int64_t base = a0; base < b0; base += 128) {
      if (base + 128 < b0) fetch(base + 128, b0, nj, nv);        // rest of a long row
      else if (has1) fetch(a1, b1, nj, nv);                      // first entries of the next row
      place(k0, cj, cv);
#pragma unroll
      for (int u = 0; u < 4; ++u) { cj[u] = nj[u]; cv[u] = nv[u]; }
    }
    if (a0 >= b0 && has1) fetch(a1, b1, cj, cv);                 // empty row: nothing was prefetched above
    if (DIRECT) {
      if (!__any_sync(0xffffffffu, dseen) && lane == 0) {  // H_kk is not stored: it is zero (A-12)
        dg = div_delta(eps_max - 0.0);
        out[r] = dg;
        q += dg * dg;
        dseen = true;
      }
      if (r < nc) {  // warp-uniform
        s2 += q;
        if (dseen) s1 += dg;
      }
    } else {
      __syncwarp();
      double* orow = Xp + (size_t)r * ld;
      double qq = 0.0;
      for (int c = lane * 2; c < ld; c += 64) {
        const double2 v = *reinterpret_cast<const double2*>(buf + c);
        *reinterpret_cast<double2*>(orow + c) = v;
        qq += v.x * v.x + v.y * v.y;
      }
      if (r < nc) {  // warp-uniform
        s2 += qq;
        if (lane == 0) s1 += buf[r];
      }
      __syncwarp();
    }
    k0 = k1; k1 = k2; a0 = a1; b0 = b1;
  }
  s1 = warp_sum(s1);
  s2 = warp_sum(s2);
  if (lane == 0) { red[wid] = s1; red[8 + wid] = s2; }
  __syncthreads();
  if (t == 0) {
    double a1 = 0.0, a2 = 0.0;
    for (int w = 0; w < nw; ++w) { a1 += red[w]; a2 += red[8 + w]; }
    partials[2 * (size_t)blockIdx.x] = a1;
    partials[2 * (size_t)blockIdx.x + 1] = a2;
  }
}

}  // namespace

// item0, n_it: a sub-range of the work items (one wave of communities, gbe_density_preset in a bounded workspace);
// n_it < 0: all of them
int gbe_launch_gather(const gbe_csr_view& H, const gbe_graph* g, const gbe_state* st, double* X, double* partials,
                      cudaStream_t s, int item0, int n_it) {
  if (n_it < 0) { item0 = 0; n_it = g->n_gitems; }
  if (n_it == 0) return GBE_OK;
  const int2* const gitems = g->gitems + item0;
  partials += 2 * (size_t)item0;
  const int W = (int)((g->n + 31) / 32);
  const int ldmax = (g->max_m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  const size_t fixed = (size_t)4 * W * 4 + 516 * 4 + 16 * 8;
  const size_t budget = 220 * 1024;
  // staged: one row buffer per warp in shared memory; direct: none.  Auto: staged while three CTAs of eight warps still
  // fit an SM with their row buffers (measured: 82 % of the copy bandwidth on the 24,576-orbital box), else direct.
  const size_t staged8 = fixed + (size_t)8 * ldmax * 8;
  bool direct = g->gather_path == 2 || (g->gather_path == 0 && 3 * (staged8 + 1024) > 227 * 1024);
  if (!direct && fixed + (size_t)ldmax * 8 > budget) direct = true;  // not even one row buffer fits
  if (fixed > budget) return GBE_EINVAL;
  if (direct) {
    GBE_CUDA(cudaFuncSetAttribute(k_gather<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fixed));
    GBE_CUDA(cudaFuncSetAttribute(k_gather<true>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    k_gather<true><<<n_it, 256, fixed, s>>>(W, ldmax, g->gather_rows, gitems, H.row_ptr, H.col_idx, H.val, g->n,
                                                   g->sub_ptr, g->sub_idx, g->ncore, g->dense_off, st, X, partials);
  } else {
    const int nw = (int)std::min<size_t>(8, (budget - fixed) / ((size_t)ldmax * 8));
    const size_t smem = fixed + (size_t)nw * ldmax * 8;
    GBE_CUDA(cudaFuncSetAttribute(k_gather<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    GBE_CUDA(cudaFuncSetAttribute(k_gather<false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    k_gather<false><<<n_it, nw * 32, smem, s>>>(W, ldmax, g->gather_rows, gitems, H.row_ptr, H.col_idx, H.val,
                                                       g->n, g->sub_ptr, g->sub_idx, g->ncore, g->dense_off, st, X, partials);
  }
  GBE_LAUNCHED();
  return GBE_OK;
}
