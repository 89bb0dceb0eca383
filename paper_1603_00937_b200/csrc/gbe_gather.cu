// Step 3 - gather / pack (row 3).
//
//     x_p = X0[s_p, s_p],  X0 = (eps_max I - H)/(eps_max - eps_min)                         (A-2)
// the FULL principal submatrix: every stored H entry with both indices in s_p; zero elsewhere; the diagonal
// gets (eps_max - H_kk)/delta even when H_kk is not stored (A-12).  Output: row-major FP64 blocks,
// ld_p = m_p rounded up to 16 doubles (rows are 128-byte aligned), pad columns zero.
//
// One CTA handles `gather_rows` consecutive rows of one community.  The global -> local index translation is a
// pair of bitmaps (core, halo) over the n vertices with popcount-prefix ranks in shared memory, one 16-byte entry
// {core word, halo word, core rank, nc + halo rank} per 32 vertices: one LDS.128 and no branch per stored entry, no
// search.  Each warp builds one output row in shared memory (zero fill + scattered entries) and hands it to the
// copy engine as ONE bulk store (cp.async.bulk shared -> global, UBLKCP), so every output byte is written exactly once,
// in whole lines, and the warp issues no per-element store; the buffer is reused when the engine has read it.
// The epilogue accumulates the traces of X_0 and X_0^2 over the core rows (t1, t2 of iteration 0):
// (X^2)_ii = sum_c X_ic^2 for symmetric X.
// DIRECT variant (large systems: the bitmaps of ~1e5 vertices plus row buffers of ~2,400 doubles leave one CTA per SM):
// no row buffer - the warp zero-fills the output row in global memory with 128-bit stores and then stores the stored
// entries straight to it (L2 merges the two before the line leaves for DRAM), so the CTA needs the bitmaps only and
// three CTAs fit an SM.  The traces are then summed over the stored entries as they are placed.
// Bound: HBM - writes 8 m_p^2 B per community, reads 12 B per stored entry of every gathered H row.
#include "gbe_internal.cuh"

namespace {

// bulk store of one finished row, shared -> global, by the copy engine (sizes and addresses are multiples of 16 bytes);
// the generic-proxy stores that built the row are fenced before the engine (async proxy) reads them
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bulk_store_row(double* dst, const double* src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst),
               "r"((uint32_t)__cvta_generic_to_shared(src_smem)), "r"(bytes)
               : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
// until the engine has READ the source of every bulk store this thread issued (the buffer may be written again)
__device__ __forceinline__ void bulk_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }

template <bool DIRECT>
__global__ void __launch_bounds__(256, 3) k_gather(int W, int ldmax, int rows_per_cta, const gbe_gitem* __restrict__ gitems,
                                                const int64_t* __restrict__ H_rp, const int32_t* __restrict__ H_col,
                                                const double* __restrict__ H_val, int64_t n,
                                                const int32_t* __restrict__ sub_idx, const gbe_state* __restrict__ st,
                                                double* __restrict__ X, double* __restrict__ partials) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint4* tab = reinterpret_cast<uint4*>(smem_raw);                        // W x {core word, halo word, core rank, nc + halo rank}
  int* scratch = reinterpret_cast<int*>(tab + W);                         // 2 * 257 ints
  double* red = reinterpret_cast<double*>(scratch + 516);                  // 16 doubles (8-byte aligned: 4W*4 + 2064)
  double* rowbuf = red + 16;                                               // nwarps * ldmax doubles
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, nw = blockDim.x >> 5;
  // the work item carries the community's sizes and offsets: two 16-byte loads, then sub_idx - no chain through p
  const int4 ia = reinterpret_cast<const int4*>(gitems)[2 * (size_t)blockIdx.x];            // p, r0, m, nc
  const longlong2 ib = reinterpret_cast<const longlong2*>(gitems)[2 * (size_t)blockIdx.x + 1];  // sb, dense_off
  const int r0 = ia.y, m = ia.z, nc = ia.w;
  const int64_t sb = ib.x;
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
  // (this thread's first two vertices are requested before the table is cleared: their latency hides behind it)
  const int l0 = t, l1 = t + (int)blockDim.x;
  const int v0 = l0 < m ? sub_idx[sb + l0] : 0;
  const int v1 = l1 < m ? sub_idx[sb + l1] : 0;
  for (int w = t; w < W; w += blockDim.x) tab[w] = make_uint4(0u, 0u, 0u, 0u);
  __syncthreads();
  if (l0 < m) atomicOr(l0 < nc ? &tab[v0 >> 5].x : &tab[v0 >> 5].y, 1u << (v0 & 31));
  if (l1 < m) atomicOr(l1 < nc ? &tab[v1 >> 5].x : &tab[v1 >> 5].y, 1u << (v1 & 31));
  for (int l = t + 2 * (int)blockDim.x; l < m; l += blockDim.x) {
    const int v = sub_idx[sb + l];
    atomicOr(l < nc ? &tab[v >> 5].x : &tab[v >> 5].y, 1u << (v & 31));
  }
  __syncthreads();
  // ranks: exclusive popcount prefix per word (both bitmaps at once)
  {
    const int nt = blockDim.x, chunk = (W + nt - 1) / nt;
    const int b = min(W, t * chunk), e = min(W, b + chunk);
    int c0 = 0, c1 = 0;
    for (int w = b; w < e; ++w) { c0 += __popc(tab[w].x); c1 += __popc(tab[w].y); }
    scratch[t] = c0;
    scratch[258 + t] = c1;
    __syncthreads();
    for (int which = wid; which < 2; which += nw) {  // one warp each scans the per-thread counts of the core and the halo bitmap
      int* sc = scratch + 258 * which;
      int run = 0;
      for (int i0 = 0; i0 < nt; i0 += 32) {
        const int v = i0 + lane < nt ? sc[i0 + lane] : 0;
        int tot;
        const int ex = warp_excl_scan_i(v, lane, &tot);
        if (i0 + lane < nt) sc[i0 + lane] = run + ex;
        run += tot;
      }
    }
    __syncthreads();
    c0 = scratch[t];
    c1 = nc + scratch[258 + t];
    for (int w = b; w < e; ++w) {
      const uint4 e4 = tab[w];
      tab[w] = make_uint4(e4.x, e4.y, (uint32_t)c0, (uint32_t)c1);
      c0 += __popc(e4.x);
      c1 += __popc(e4.y);
    }
  }
  __syncthreads();

  double* buf = DIRECT ? nullptr : rowbuf + (size_t)wid * ldmax;
  double* Xp = X + ib.y;
  double s1 = 0.0, s2 = 0.0;
  // The row loop is latency bound (sub_idx -> H row pointers -> H entries are dependent loads), so it is software
  // pipelined: the vertex of the row after next and the row pointers of the next row are in flight while the current
  // row is scattered into shared memory; the first 256 entries of the next row (GS slots of 32 per lane: a whole row for
  // all but the longest) are requested into the SAME registers as soon as the current row's have been placed, and land
  // while this row is handed to the copy engine and the buffer turns over.
  const int rend = min(m, r0 + rows_per_cta);
  // (entries base + lane + 32 u of a row of cnt entries; cnt <= 0: nothing)
  constexpr int GS = 8;
  auto fetch = [&](int64_t base, int cnt, int (&j)[GS], double (&v)[GS]) {
    const int32_t* __restrict__ pc = H_col + base + lane;
    const double* __restrict__ pv = H_val + base + lane;
#pragma unroll
    for (int u = 0; u < GS; ++u) {
      const bool ok = lane + 32 * u < cnt;
      j[u] = ok ? pc[32 * u] : -1;
      v[u] = ok ? pv[32 * u] : 0.0;
    }
  };
  const uint32_t nlim = (uint32_t)(n < (int64_t)INT32_MAX ? n : (int64_t)INT32_MAX);  // column indices are int32
  double* out = nullptr;     // DIRECT: the output row being built
  double q = 0.0, dg = 0.0;  // DIRECT: this lane's sum of squares of the row, and the stored diagonal if it placed it
  bool dseen = false;
  auto place = [&](int k, const int (&j)[GS], const double (&v)[GS]) {
#pragma unroll
    for (int u = 0; u < GS; ++u) {
      const int col = j[u];
      const bool inr = (uint32_t)col < nlim;  // (an empty slot holds -1)
      const uint4 e4 = tab[inr ? col >> 5 : 0];
      const uint32_t bit = 1u << (col & 31);
      const bool isc = (e4.x & bit) != 0u;  // core and halo are disjoint
      const uint32_t wsel = isc ? e4.x : e4.y;
      const int c = (int)(isc ? e4.z : e4.w) + __popc(wsel & (bit - 1u));
      if (inr && (wsel & bit) != 0u) {
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
  int64_t a0 = 0, a1 = 0;  // first entry and length of the current and of the next row of H
  int n0 = 0, n1 = 0;
  int cj[GS];
  double cv[GS];
  if (r < rend) {
    a0 = H_rp[k0];
    n0 = (int)(H_rp[k0 + 1] - a0);
    fetch(a0, n0, cj, cv);
  }
  for (; r < rend; r += nw) {
    const bool has1 = r + nw < rend;
    const int k2 = r + 2 * nw < rend ? sub_idx[sb + r + 2 * nw] : 0;
    if (has1) {
      a1 = H_rp[k1];
      n1 = (int)(H_rp[k1 + 1] - a1);
    }
    double* const zrow = DIRECT ? Xp + (size_t)r * ld : buf;
    if (!DIRECT) {  // the engine has read the previous row out of the buffer
      if (lane == 0) bulk_store_wait_read();
      __syncwarp();
    }
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
    for (int off = 0; off < n0; off += 32 * GS) {
      place(k0, cj, cv);
      if (off + 32 * GS < n0) fetch(a0 + off + 32 * GS, n0 - off - 32 * GS, cj, cv);  // rest of a very long row
    }
    if (has1) fetch(a1, n1, cj, cv);  // the next row's entries: in flight until the buffer has turned over
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
      if (r < nc) {  // warp-uniform: a core row, whose diagonal and squares enter t1 and t2 of iteration 0
        double qq = 0.0;
        for (int c = lane * 2; c < ld; c += 64) {
          const double2 v = *reinterpret_cast<const double2*>(buf + c);
          qq += v.x * v.x + v.y * v.y;
        }
        s2 += qq;
        if (lane == 0) s1 += buf[r];
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) bulk_store_row(orow, buf, (uint32_t)ld * 8u);
    }
    k0 = k1; k1 = k2; a0 = a1; n0 = n1;
  }
  if (!DIRECT && lane == 0) bulk_store_wait_read();  // the buffers live as long as the CTA
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
  const gbe_gitem* const gitems = g->gitems + item0;
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
                                                   g->sub_idx, st, X, partials);
  } else {
    const int nw = (int)std::min<size_t>(8, (budget - fixed) / ((size_t)ldmax * 8));
    const size_t smem = fixed + (size_t)nw * ldmax * 8;
    GBE_CUDA(cudaFuncSetAttribute(k_gather<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    GBE_CUDA(cudaFuncSetAttribute(k_gather<false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
    k_gather<false><<<n_it, nw * 32, smem, s>>>(W, ldmax, g->gather_rows, gitems, H.row_ptr, H.col_idx, H.val,
                                                       g->n, g->sub_idx, st, X, partials);
  }
  GBE_LAUNCHED();
  return GBE_OK;
}
