// Step 2 - halo discovery (row 2).
//
// For community p with core C_p = {i : part[i] = p} (obs. (vi) P:L65):
//     s_p = C_p u { k : (k, i) in S_tau, i in C_p }                       (Fig.1)
// local order: core vertices ascending, then halo vertices ascending.  Also built here, once per graph:
//   - the padded batched dense layout (ld_p = m_p rounded up to 16 doubles, element offsets),
//   - the pattern S' of D (A-9): row k holds the core vertices of every community whose subgraph contains k,
//   - the scatter map: for dense row (p, r) the offset in D.val of the run of its ncore_p core columns
//     (contiguous when every core is an index range; otherwise a per-entry map),
//   - the X^2 tile work list (largest communities first) and the gather work list.
// All set work uses a bitmap over the n vertices in shared memory; walking it emits ascending indices.
// Bound: integer/latency; runs once per graph.
#include <algorithm>
#include <numeric>

#include <cmath>

#include "gbe_internal.cuh"

namespace {


__device__ __forceinline__ int part_of(const int32_t* part, int64_t i, int64_t blk) {
  return part ? part[i] : (int)(i / blk);
}

__global__ void k_core_count(int64_t n, const int32_t* __restrict__ part, int64_t blk, int n_part,
                             int32_t* __restrict__ cnt, int32_t* __restrict__ flag) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int p = part_of(part, i, blk);
  if (p < 0 || p >= n_part) { atomicOr(flag, 1); return; }
  atomicAdd(&cnt[p], 1);
}
__global__ void k_core_fill(int64_t n, const int32_t* __restrict__ part, int64_t blk, int n_part,
                            const int64_t* __restrict__ core_ptr, int32_t* __restrict__ cursor,
                            int32_t* __restrict__ core_tmp) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int p = part_of(part, i, blk);
  if (p < 0 || p >= n_part) return;  // flagged by k_core_count; the host looks at the flag at its next synchronisation
  const int pos = atomicAdd(&cursor[p], 1);
  core_tmp[core_ptr[p] + pos] = (int32_t)i;  // order fixed later by the bitmap walk
}

// block-wide: emit the set bits of (bm[w] for w < W) in ascending order to out[], returns the count
__device__ int block_emit_bits(const uint32_t* bm, int W, int32_t* out, int* scratch /* blockDim.x + 1 */) {
  const int t = threadIdx.x, nt = blockDim.x;
  const int chunk = (W + nt - 1) / nt;
  const int b = min(W, t * chunk), e = min(W, b + chunk);
  int c = 0;
  for (int w = b; w < e; ++w) c += __popc(bm[w]);
  scratch[t] = c;
  __syncthreads();
  if (t == 0) {
    int run = 0;
    for (int k = 0; k < nt; ++k) { const int v = scratch[k]; scratch[k] = run; run += v; }
    scratch[nt] = run;
  }
  __syncthreads();
  if (out) {
    int pos = scratch[t];
    for (int w = b; w < e; ++w) {
      uint32_t bits = bm[w];
      while (bits) {
        const int bp = __ffs(bits) - 1;
        bits &= bits - 1;
        out[pos++] = w * 32 + bp;
      }
    }
  }
  const int total = scratch[nt];
  __syncthreads();
  return total;
}

template <bool FILL>
__global__ void __launch_bounds__(256) k_halo(int W, const int64_t* __restrict__ core_ptr,
                                              const int32_t* __restrict__ core_tmp, const int64_t* __restrict__ S_rp,
                                              const int32_t* __restrict__ S_col, int32_t* __restrict__ msize,
                                              int32_t* __restrict__ ncore, const int64_t* __restrict__ sub_ptr,
                                              int32_t* __restrict__ sub_idx, int32_t* __restrict__ row_part) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  uint32_t* coreb = reinterpret_cast<uint32_t*>(smem_raw);
  uint32_t* allb = coreb + W;
  int* scratch = reinterpret_cast<int*>(allb + W);
  const int p = blockIdx.x, t = threadIdx.x, lane = t & 31, wid = t >> 5;
  for (int w = t; w < 2 * W; w += 256) coreb[w] = 0u;
  __syncthreads();
  const int64_t cb = core_ptr[p], ce = core_ptr[p + 1];
  for (int64_t c = cb + wid; c < ce; c += 8) {  // warp per core vertex, lanes along its S row
    const int i = core_tmp[c];
    if (lane == 0) atomicOr(&coreb[i >> 5], 1u << (i & 31));
    for (int64_t e = S_rp[i] + lane; e < S_rp[i + 1]; e += 32) {
      const int k = S_col[e];
      atomicOr(&allb[k >> 5], 1u << (k & 31));
    }
  }
  __syncthreads();
  for (int w = t; w < W; w += 256) allb[w] &= ~coreb[w];  // halo = neighbours that are not core
  __syncthreads();
  const int64_t ob = FILL ? sub_ptr[p] : 0;
  const int nc = block_emit_bits(coreb, W, FILL ? sub_idx + ob : nullptr, scratch);
  const int nh = block_emit_bits(allb, W, FILL ? sub_idx + ob + nc : nullptr, scratch);
  if (FILL) {
    for (int r = t; r < nc + nh; r += 256) row_part[ob + r] = p;
  } else if (t == 0) {
    msize[p] = nc + nh;
    ncore[p] = nc;
  }
}

// counts for the pattern of D and the membership lists
__global__ void k_member_count(int64_t sum_m, const int32_t* __restrict__ sub_idx, const int32_t* __restrict__ row_part,
                               const int32_t* __restrict__ ncore, int32_t* __restrict__ cntD, int32_t* __restrict__ mcnt) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= sum_m) return;
  const int k = sub_idx[q];
  atomicAdd(&cntD[k], ncore[row_part[q]]);
  atomicAdd(&mcnt[k], 1);
}
__global__ void k_member_fill(int64_t sum_m, const int32_t* __restrict__ sub_idx, const int64_t* __restrict__ memb_ptr,
                              int32_t* __restrict__ cursor, int64_t* __restrict__ memb) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= sum_m) return;
  const int k = sub_idx[q];
  const int pos = atomicAdd(&cursor[k], 1);
  memb[memb_ptr[k] + pos] = q;
}
// per dense row q: where it starts in a dense buffer and how many core columns it carries (read by the scatter)
__global__ void k_row_meta(int64_t sum_m, const int32_t* __restrict__ row_part, const int64_t* __restrict__ sub_ptr,
                           const int32_t* __restrict__ ncore, const int64_t* __restrict__ dense_off,
                           int64_t* __restrict__ row_src, int32_t* __restrict__ row_nc) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= sum_m) return;
  const int p = row_part[q];
  const int64_t sb = sub_ptr[p];
  const int64_t m = sub_ptr[p + 1] - sb;
  const int64_t ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  row_src[q] = dense_off[p] + (q - sb) * ld;
  row_nc[q] = ncore[p];
}
// The X^2 work lists (gbe_tile_item), written on the device from one small descriptor per community (the host sorts the
// communities by size and takes two prefix sums; spelling out ~2e4 items on the host cost 0.4 ms per build): block b
// writes the tiles (ti <= tj) of community desc[b].p, ti outer, tj inner, at items[desc[b].off ...]; those with a core row
// (ti * tile < ncore: the first Tc tile rows, i.e. the first tiles of the community's run) also at last[desc[b].loff ...],
// and their position there is the index of their trace partial (pidx; -1 for the others).
struct gbe_tile_desc { int32_t p, m, nc, ld, off, loff; int64_t dense_off; };
__global__ void k_tile_items(const gbe_tile_desc* __restrict__ desc, int tile, gbe_tile_item* __restrict__ items,
                             gbe_tile_item* __restrict__ last) {
  const gbe_tile_desc d = desc[blockIdx.x];
  const int T = (d.m + tile - 1) / tile;
  const int n_t = T * (T + 1) / 2;
  for (int k = threadIdx.x; k < n_t; k += blockDim.x) {
    // k = ti * T - ti (ti - 1) / 2 + (tj - ti): the largest ti whose first index is <= k (T <= 2^15: fp32 start, fixed up)
    int ti = (int)(((float)(2 * T + 1) - sqrtf((float)(2 * T + 1) * (float)(2 * T + 1) - 8.0f * (float)k)) * 0.5f);
    ti = min(max(ti, 0), T - 1);
    while (ti > 0 && ti * T - ti * (ti - 1) / 2 > k) --ti;
    while (ti + 1 < T && (ti + 1) * T - (ti + 1) * ti / 2 <= k) ++ti;
    const int tj = ti + (k - (ti * T - ti * (ti - 1) / 2));
    const bool core_row = ti * tile < d.nc;
    gbe_tile_item it;
    it.pidx = core_row ? d.loff + k : -1;
    it.tij = ti | (tj << 16);
    it.p = d.p;
    it.m = d.m;
    it.nc = d.nc;
    it.ld = d.ld;
    it.dense_off = d.dense_off;
    items[d.off + k] = it;
    if (core_row) last[d.loff + k] = it;
  }
}

__global__ void k_row_ncore(int64_t sum_m, const int32_t* __restrict__ row_part, const int32_t* __restrict__ ncore,
                            int32_t* __restrict__ out) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q < sum_m) out[q] = ncore[row_part[q]];
}

// warp per row k of D: columns = union of the cores of the communities containing k, ascending; scatter offsets.
// MODE 0: D_col + scat_base + contiguity flag; MODE 1: per-entry scat_pos.
template <int MODE>
__global__ void k_d_pattern(int64_t n, int W, const int64_t* __restrict__ memb_ptr, const int64_t* __restrict__ memb,
                            const int32_t* __restrict__ row_part, const int64_t* __restrict__ sub_ptr,
                            const int32_t* __restrict__ sub_idx, const int32_t* __restrict__ ncore,
                            const int64_t* __restrict__ D_rp, int32_t* __restrict__ D_col,
                            int64_t* __restrict__ scat_base, int32_t* __restrict__ noncontig,
                            const int64_t* __restrict__ scat_ofs, int64_t* __restrict__ scat_pos) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, w_in_blk = threadIdx.x >> 5, nw = blockDim.x >> 5;
  uint32_t* bm = reinterpret_cast<uint32_t*>(smem_raw) + (size_t)2 * W * w_in_blk;
  uint32_t* rk = bm + W;
  for (int64_t k = (int64_t)blockIdx.x * nw + w_in_blk; k < n; k += (int64_t)gridDim.x * nw) {
    for (int w = lane; w < W; w += 32) bm[w] = 0u;
    __syncwarp();
    const int64_t mb = memb_ptr[k], me = memb_ptr[k + 1];
    // the communities that contain row k: their metadata is fetched by the lanes side by side (one chain of
    // dependent loads per 32 members instead of one per member) and handed round by shuffle
    for (int64_t x0 = mb; x0 < me; x0 += 32) {
      const int64_t xl = x0 + lane;
      int64_t sb_l = 0;
      int nc_l = 0;
      if (xl < me) {
        const int p = row_part[memb[xl]];
        sb_l = sub_ptr[p];
        nc_l = ncore[p];
      }
      const int cnt = (int)min((int64_t)32, me - x0);
      for (int y = 0; y < cnt; ++y) {
        const int64_t sb = __shfl_sync(0xffffffffu, sb_l, y);
        const int nc = __shfl_sync(0xffffffffu, nc_l, y);
        for (int c = lane; c < nc; c += 32) { const int i = sub_idx[sb + c]; atomicOr(&bm[i >> 5], 1u << (i & 31)); }
      }
    }
    __syncwarp();
    int running = 0;
    const int64_t ob = D_rp[k];
    for (int w0 = 0; w0 < W; w0 += 32) {
      const int w = w0 + lane;
      uint32_t bits = w < W ? bm[w] : 0u;
      int tot;
      const int ex = warp_excl_scan_i(__popc(bits), lane, &tot);
      if (w < W) rk[w] = running + ex;
      if (MODE == 0) {
        int pos = running + ex;
        while (bits) {
          const int bp = __ffs(bits) - 1;
          bits &= bits - 1;
          D_col[ob + pos++] = w * 32 + bp;
        }
      }
      running += tot;
    }
    __syncwarp();
    for (int64_t x0 = mb; x0 < me; x0 += 32) {
      const int64_t xl = x0 + lane;
      int64_t q_l = 0, sb_l = 0, so_l = 0;
      int nc_l = 0, first_l = 0;
      if (xl < me) {
        q_l = memb[xl];
        const int p = row_part[q_l];
        sb_l = sub_ptr[p];
        nc_l = ncore[p];
        first_l = sub_idx[sb_l];
        if (MODE == 1) so_l = scat_ofs[q_l];
      }
      const int cnt = (int)min((int64_t)32, me - x0);
      for (int y = 0; y < cnt; ++y) {
        const int64_t q = __shfl_sync(0xffffffffu, q_l, y);
        const int64_t sb = __shfl_sync(0xffffffffu, sb_l, y);
        const int nc = __shfl_sync(0xffffffffu, nc_l, y);
        const int first = __shfl_sync(0xffffffffu, first_l, y);
        const int64_t so = MODE == 1 ? __shfl_sync(0xffffffffu, so_l, y) : 0;
        const int pos0 = rk[first >> 5] + __popc(bm[first >> 5] & ((1u << (first & 31)) - 1u));
        if (MODE == 0 && lane == 0) scat_base[q] = ob + pos0;
        for (int c = lane; c < nc; c += 32) {
          const int i = sub_idx[sb + c];
          const int pos = rk[i >> 5] + __popc(bm[i >> 5] & ((1u << (i & 31)) - 1u));
          if (MODE == 0) {
            if (pos != pos0 + c) atomicOr(noncontig, 1);
          } else {
            scat_pos[so + c] = ob + pos;
          }
        }
      }
    }
    __syncwarp();
  }
}

template <typename T>
int upload(const std::vector<T>& h, T** d, cudaStream_t s) {
  GBE_TRY(gbe_dev_alloc((void**)d, std::max<size_t>(16, h.size() * sizeof(T))));
  if (!h.empty()) GBE_CUDA(cudaMemcpyAsync(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, s));
  return GBE_OK;
}
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

int gbe_build_subgraphs(gbe_graph* g, const int32_t* part, cudaStream_t s, const double* bounds) {
  const int64_t n = g->n;
  const int n_part = g->n_part;
  const int W = (int)((n + 31) / 32);
  const int64_t blk = (n + n_part - 1) / n_part;
  const int sm_count = gbe_sm_count();  // of the current device
  const int tgrid = (int)((n + 255) / 256);

  // ---- cores
  DevBuf cnt, flag, core_tmp, cursor;
  GBE_TRY(cnt.alloc((size_t)std::max<int64_t>(n_part, n) * 4));
  GBE_TRY(flag.alloc(4));
  GBE_CUDA(cudaMemsetAsync(cnt.p, 0, (size_t)n_part * 4, s));
  GBE_CUDA(cudaMemsetAsync(flag.p, 0, 4, s));
  k_core_count<<<tgrid, 256, 0, s>>>(n, part, blk, n_part, cnt.as<int32_t>(), flag.as<int32_t>());
  GBE_LAUNCHED();
  int32_t hflag = 0, hflag_stack = 0;
  int32_t* const pin = gbe_pinned_words();
  int32_t* const core_flag = pin ? pin : &hflag_stack;  // fetched now, looked at after the next synchronisation
  *core_flag = 0;
  GBE_CUDA(cudaMemcpyAsync(core_flag, flag.p, 4, cudaMemcpyDeviceToHost, s));
  DevBuf core_ptr;
  GBE_TRY(core_ptr.alloc((size_t)(n_part + 1) * 8));
  GBE_TRY(gbe_exclusive_scan_i32_to_i64(cnt.as<int32_t>(), core_ptr.as<int64_t>(), n_part, s));
  GBE_TRY(core_tmp.alloc((size_t)n * 4));
  GBE_TRY(cursor.alloc((size_t)std::max<int64_t>(n_part, n) * 4));
  GBE_CUDA(cudaMemsetAsync(cursor.p, 0, (size_t)n_part * 4, s));
  k_core_fill<<<tgrid, 256, 0, s>>>(n, part, blk, n_part, core_ptr.as<int64_t>(), cursor.as<int32_t>(), core_tmp.as<int32_t>());
  GBE_LAUNCHED();
  // ---- halo: count, then fill
  const size_t halo_smem = (size_t)2 * W * 4 + 257 * 4;
  if (halo_smem > 220 * 1024) return GBE_EINVAL;  // n too large for the shared-memory bitmaps
  GBE_CUDA(cudaFuncSetAttribute(k_halo<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)halo_smem));
  GBE_CUDA(cudaFuncSetAttribute(k_halo<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)halo_smem));
  GBE_TRY(gbe_dev_alloc((void**)&g->msize, (size_t)n_part * 4));
  GBE_TRY(gbe_dev_alloc((void**)&g->ncore, (size_t)n_part * 4));
  k_halo<false><<<n_part, 256, halo_smem, s>>>(W, core_ptr.as<int64_t>(), core_tmp.as<int32_t>(), g->S_row_ptr, g->S_col,
                                               g->msize, g->ncore, nullptr, nullptr, nullptr);
  GBE_LAUNCHED();
  g->h_m.resize(n_part);
  g->h_ncore.resize(n_part);
  GBE_CUDA(cudaMemcpyAsync(g->h_m.data(), g->msize, (size_t)n_part * 4, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaMemcpyAsync(g->h_ncore.data(), g->ncore, (size_t)n_part * 4, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  if (*core_flag) return GBE_EINVAL;  // partition id out of range (k_core_count)
  if (bounds && (!(bounds[1] > bounds[0]) || !std::isfinite(bounds[0]) || !std::isfinite(bounds[1]))) return GBE_EDEGENERATE;
  // ---- host: layout, work lists
  std::vector<int64_t> h_sub_ptr(n_part + 1, 0);
  g->h_dense_off.assign(n_part + 1, 0);
  g->max_m = 0;
  g->max_ncore = 0;
  g->ncore_all_even = 1;
  g->nnz_D = 0;
  g->flops_per_iter = 0;
  g->sym_flops_per_iter = 0;
  for (int p = 0; p < n_part; ++p) {
    const int64_t m = g->h_m[p];
    const int64_t ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    h_sub_ptr[p + 1] = h_sub_ptr[p] + m;
    g->h_dense_off[p + 1] = g->h_dense_off[p] + m * ld;
    g->max_m = std::max<int32_t>(g->max_m, (int32_t)m);
    g->max_ncore = std::max<int32_t>(g->max_ncore, g->h_ncore[p]);
    if (g->h_ncore[p] & 1) g->ncore_all_even = 0;
    g->nnz_D += m * g->h_ncore[p];
    g->flops_per_iter += 2.0 * (double)m * (double)m * (double)m;
    g->sym_flops_per_iter += (double)m * (double)m * (double)(m + 1);  // m (m + 1) / 2 entries of 2 m flop each
  }
  g->sum_m = h_sub_ptr[n_part];
  g->dense_elems = g->h_dense_off[n_part];
  GBE_TRY(upload(h_sub_ptr, &g->sub_ptr, s));
  GBE_TRY(upload(g->h_dense_off, &g->dense_off, s));

  // ---- fill sub_idx / row_part
  GBE_TRY(gbe_dev_alloc((void**)&g->sub_idx, std::max<size_t>(16, (size_t)g->sum_m * 4)));
  GBE_TRY(gbe_dev_alloc((void**)&g->row_part, std::max<size_t>(16, (size_t)g->sum_m * 4)));
  k_halo<true><<<n_part, 256, halo_smem, s>>>(W, core_ptr.as<int64_t>(), core_tmp.as<int32_t>(), g->S_row_ptr, g->S_col,
                                              nullptr, nullptr, g->sub_ptr, g->sub_idx, g->row_part);
  GBE_LAUNCHED();
  // ---- pattern of D and scatter map
  const int64_t sum_m = g->sum_m;
  const int qgrid = (int)std::max<int64_t>(1, (sum_m + 255) / 256);
  GBE_TRY(gbe_dev_alloc((void**)&g->row_src, std::max<size_t>(16, (size_t)sum_m * 8)));
  GBE_TRY(gbe_dev_alloc((void**)&g->row_nc, std::max<size_t>(16, (size_t)sum_m * 4)));
  k_row_meta<<<qgrid, 256, 0, s>>>(sum_m, g->row_part, g->sub_ptr, g->ncore, g->dense_off, g->row_src, g->row_nc);
  GBE_LAUNCHED();
  DevBuf mcnt, memb_ptr, memb;
  GBE_TRY(mcnt.alloc((size_t)n * 4));
  GBE_CUDA(cudaMemsetAsync(cnt.p, 0, (size_t)n * 4, s));
  GBE_CUDA(cudaMemsetAsync(mcnt.p, 0, (size_t)n * 4, s));
  k_member_count<<<qgrid, 256, 0, s>>>(sum_m, g->sub_idx, g->row_part, g->ncore, cnt.as<int32_t>(), mcnt.as<int32_t>());
  GBE_LAUNCHED();
  GBE_TRY(gbe_dev_alloc((void**)&g->D_row_ptr, (size_t)(n + 1) * 8));
  GBE_TRY(gbe_exclusive_scan_i32_to_i64(cnt.as<int32_t>(), g->D_row_ptr, n, s));
  GBE_TRY(memb_ptr.alloc((size_t)(n + 1) * 8));
  GBE_TRY(gbe_exclusive_scan_i32_to_i64(mcnt.as<int32_t>(), memb_ptr.as<int64_t>(), n, s));
  GBE_TRY(memb.alloc(std::max<size_t>(16, (size_t)sum_m * 8)));
  GBE_CUDA(cudaMemsetAsync(cursor.p, 0, (size_t)n * 4, s));
  k_member_fill<<<qgrid, 256, 0, s>>>(sum_m, g->sub_idx, memb_ptr.as<int64_t>(), cursor.as<int32_t>(), memb.as<int64_t>());
  GBE_LAUNCHED();
  GBE_TRY(gbe_dev_alloc((void**)&g->D_col, std::max<size_t>(16, (size_t)g->nnz_D * 4)));
  GBE_TRY(gbe_dev_alloc((void**)&g->scat_base, std::max<size_t>(16, (size_t)sum_m * 8)));
  const size_t per_warp = (size_t)2 * W * 4;
  int nw = (int)std::min<size_t>(8, (200 * 1024) / per_warp);
  if (nw < 1) return GBE_EINVAL;
  GBE_CUDA(cudaFuncSetAttribute(k_d_pattern<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
  GBE_CUDA(cudaFuncSetAttribute(k_d_pattern<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * nw)));
  const int dgrid = (int)std::min<int64_t>((n + nw - 1) / nw, (int64_t)sm_count * 8);
  GBE_CUDA(cudaMemsetAsync(flag.p, 0, 4, s));
  k_d_pattern<0><<<dgrid, nw * 32, per_warp * nw, s>>>(n, W, memb_ptr.as<int64_t>(), memb.as<int64_t>(), g->row_part,
                                                       g->sub_ptr, g->sub_idx, g->ncore, g->D_row_ptr, g->D_col,
                                                       g->scat_base, flag.as<int32_t>(), nullptr, nullptr);
  GBE_LAUNCHED();
  // ---- host: work lists, bins, tensor maps, workspace layout - while the device fills sub_idx and the pattern of D (the
  //      kernels above need the sizes and offsets only; a timeline of the build showed the device idle for 0.5 ms here
  //      when the lists were built first).  Their uploads queue up behind k_d_pattern.
  // X^2 tile list: communities by decreasing m (longest work first), the tiles of one community adjacent
  // so that its panels are reused from L2 by the CTAs that run together.
  {
    std::vector<int32_t> order(n_part);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return g->h_m[a] > g->h_m[b]; });
    g->pk_max_m = gbe_packed_max_m();
    // the lists themselves are written on the device (k_tile_items) from one descriptor per community
    std::vector<gbe_tile_desc> desc, desc_h;  // _h: the communities the packed kernel does not take
    desc.reserve(n_part);
    const int tile = g->tile;
    int64_t n_all = 0, n_last = 0, n_all_h = 0, n_last_h = 0;
    g->exec_flops_per_iter = g->exec_flops_last_iter = g->flops_last_iter = 0;
    for (int p : order) {
      const int m = g->h_m[p], nc = g->h_ncore[p];
      const int64_t T = (m + tile - 1) / tile;
      const int64_t ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
      const int64_t Tc = std::min<int64_t>(T, (nc + tile - 1) / tile);  // tile rows with a core row (ti * tile < ncore)
      const int64_t n_t = T * (T + 1) / 2, n_c = Tc * T - Tc * (Tc - 1) / 2;
      if (n_t > 0) {
        desc.push_back({p, m, nc, (int32_t)ld, (int32_t)n_all, (int32_t)n_last, g->h_dense_off[p]});
        if (m > g->pk_max_m) desc_h.push_back({p, m, nc, (int32_t)ld, (int32_t)n_all_h, (int32_t)n_last_h, g->h_dense_off[p]});
      }
      n_all += n_t;
      n_last += n_c;
      if (m > g->pk_max_m) { n_all_h += n_t; n_last_h += n_c; }
      // executed DMMA work: 8x8 sub-tiles (bi <= bj) with rows < m, columns < ld, each 2*8*8*ld flop
      const double R = (double)((m + 7) / 8), C = (double)(ld / 8);
      g->exec_flops_per_iter += (R * C - R * (R - 1) / 2) * 128.0 * (double)ld;
      // last iteration: the same count restricted to the row blocks of the tiles with a core row
      const double Rc = std::min(R, (double)(Tc * (tile / 8)));
      g->exec_flops_last_iter += (Rc * C - Rc * (Rc - 1) / 2) * 128.0 * (double)ld;
      g->flops_last_iter += 2.0 * (double)m * (double)m * (double)nc;
    }
    if (n_all > INT32_MAX) return GBE_EINVAL;  // the work lists are indexed with 32 bits
    auto make_lists = [&](const std::vector<gbe_tile_desc>& d, int64_t na, int64_t nl, gbe_tile_item** it,
                          gbe_tile_item** la) -> int {
      GBE_TRY(gbe_dev_alloc((void**)it, std::max<size_t>(16, (size_t)na * sizeof(gbe_tile_item))));
      GBE_TRY(gbe_dev_alloc((void**)la, std::max<size_t>(16, (size_t)nl * sizeof(gbe_tile_item))));
      if (d.empty()) return GBE_OK;
      DevBuf dd;
      GBE_TRY(dd.alloc(d.size() * sizeof(gbe_tile_desc)));
      GBE_CUDA(cudaMemcpyAsync(dd.p, d.data(), d.size() * sizeof(gbe_tile_desc), cudaMemcpyHostToDevice, s));
      k_tile_items<<<(unsigned)d.size(), 128, 0, s>>>(dd.as<gbe_tile_desc>(), tile, *it, *la);
      GBE_LAUNCHED();
      return GBE_OK;  // (dd is released in stream order; the copy of a few KB from pageable memory is staged at once)
    };
    g->n_items_h = (int32_t)n_all_h;
    g->n_items_last_h = (int32_t)n_last_h;
    if (n_all_h > 0 && n_all_h < n_all)  // only a mixed graph needs the second pair of lists
      GBE_TRY(make_lists(desc_h, n_all_h, n_last_h, &g->items_h, &g->items_last_h));
    g->n_items = (int32_t)n_all;
    g->n_items_last = (int32_t)n_last;
    GBE_TRY(make_lists(desc, n_all, n_last, &g->items, &g->items_last));
  }
  {
    // rows per gather CTA: every CTA first builds the community's index bitmaps over the n vertices (O(n / 32) words), so
    // large systems amortise that over more rows
    g->gather_rows = n <= 32768 ? 64 : (n <= 131072 ? 256 : 512);
    static thread_local std::vector<gbe_gitem> gi;
    gi.clear();
    for (int p = 0; p < n_part; ++p)
      for (int r0 = 0; r0 < g->h_m[p]; r0 += g->gather_rows)
        gi.push_back(gbe_gitem{p, r0, g->h_m[p], g->h_ncore[p], h_sub_ptr[p], g->h_dense_off[p]});
    g->n_gitems = (int32_t)gi.size();
    GBE_TRY(upload(gi, &g->gitems, s));
  }
  GBE_TRY(gbe_build_packed(g, s));  // bins of the small communities (gbe_small.cu)
  GBE_TRY(gbe_x2_build_tmaps(g, s));  // tensor maps of the tiled kernel's panels (gbe_x2.cu); needs dense_off on the device
  // the resident kernel double-buffers n_part pairs; the packed path writes one pair per bin behind the tiled kernel's
  // (a mixed graph alternates between two sets of tile + bin pairs: the lazy decision, gbe_api.cu)
  g->n_partials = std::max(std::max(std::max(g->n_items, g->n_gitems), 2 * n_part), 2 * (g->n_items_last_h + g->n_pk_ctas));
  // wave mode (gbe_plan_waves): the gather of a later wave must not touch the final pairs of an earlier one
  g->n_partials = std::max(g->n_partials, g->n_items_last + g->n_gitems);
  GBE_TRY(gbe_resident_capacity(g, &g->resident_fits, &g->resident_coresident, &g->resident_cluster));

  // workspace layout
  size_t off = align_up(sizeof(gbe_state), 256);
  g->ws_bounds = off;
  off += align_up(2 * 1024 * sizeof(double), 256);
  g->ws_partials = off;
  off += align_up((size_t)std::max(1, g->n_partials) * 2 * sizeof(double), 256);
  g->ws_x0 = off;
  off += align_up((size_t)g->dense_elems * 8, 256);
  g->ws_x1 = off;
  off += align_up((size_t)g->dense_elems * 8, 256);
  g->ws_bytes = off;
  {  // smallest workspace of gbe_density_preset without traces: two buffers that hold the largest community
    int64_t big = 0;
    for (int p = 0; p < n_part; ++p) big = std::max<int64_t>(big, g->h_dense_off[p + 1] - g->h_dense_off[p]);
    g->ws_bytes_wave_min = g->ws_x0 + 2 * align_up((size_t)big * 8, 256);
  }
  g->ws_x2 = off;
  off += align_up((size_t)g->dense_elems * 8, 256);
  g->ws_x3 = off;
  off += align_up((size_t)g->dense_elems * 8, 256);
  g->ws_bytes_fermi = off;
  GBE_CUDA(cudaMemcpyAsync(&hflag, flag.p, 4, cudaMemcpyDeviceToHost, s));  // (to pageable memory: blocks the host - kept last)
  GBE_CUDA(cudaStreamSynchronize(s));  // the last synchronisation of a build (the general scatter map below needs one more)
  g->contiguous = hflag ? 0 : 1;
  if (!g->contiguous) {
    DevBuf rn, scat_ofs;
    GBE_TRY(rn.alloc(std::max<size_t>(16, (size_t)sum_m * 4)));
    k_row_ncore<<<qgrid, 256, 0, s>>>(sum_m, g->row_part, g->ncore, rn.as<int32_t>());
    GBE_LAUNCHED();
    GBE_TRY(scat_ofs.alloc((size_t)(sum_m + 1) * 8));
    GBE_TRY(gbe_exclusive_scan_i32_to_i64(rn.as<int32_t>(), scat_ofs.as<int64_t>(), sum_m, s));
    GBE_TRY(gbe_dev_alloc((void**)&g->scat_pos, std::max<size_t>(16, (size_t)g->nnz_D * 8)));
    k_d_pattern<1><<<dgrid, nw * 32, per_warp * nw, s>>>(n, W, memb_ptr.as<int64_t>(), memb.as<int64_t>(), g->row_part,
                                                         g->sub_ptr, g->sub_idx, g->ncore, g->D_row_ptr, nullptr, nullptr,
                                                         nullptr, scat_ofs.as<int64_t>(), g->scat_pos);
    GBE_LAUNCHED();
    GBE_CUDA(cudaStreamSynchronize(s));
    g->scat_ofs = reinterpret_cast<int64_t*>(scat_ofs.release());
  }
  return GBE_OK;
}

// ----------------------------------------------------------------------------------------------------------------------
// Waves of communities for a pre-determined SP2 sequence in a BOUNDED workspace (with the sequence fixed beforehand
// every expansion runs "without exchange of information during or between the matrix multiplications", so nothing couples
// the communities and gather -> SP2 loop -> scatter can be done for a few of them at a time).  A wave is a range of
// consecutive communities [p0, p1): contiguous in the dense layout (its buffers are the full-size ones shifted by the
// wave's first offset), in the gather work list and in the dense rows the scatter walks; only the X^2 tile lists, which
// are ordered by size, are re-cut per wave (same order and same trace slots as the whole-batch lists).
// cap_elems: doubles ONE dense buffer of a wave may hold.  The plan is cached in the graph for the cap it was made for.
int gbe_plan_waves(const gbe_graph* g, size_t cap_elems, cudaStream_t s) {
  if (g->waves_cap == cap_elems && !g->waves.empty()) return GBE_OK;
  const int n_part = g->n_part;
  std::vector<gbe_wave> waves;
  std::vector<int32_t> wave_of(n_part, 0);
  {
    gbe_wave w = {};
    int64_t row = 0;
    int gi = 0;
    w.base_elems = 0;
    for (int p = 0; p < n_part; ++p) {
      const int64_t m = g->h_m[p];
      const int64_t e = g->h_dense_off[p + 1] - g->h_dense_off[p];
      if ((size_t)e > cap_elems) return GBE_ENOMEM;
      if (w.p1 > w.p0 && (size_t)(w.elems + e) > cap_elems) {  // close the wave, open the next at p
        waves.push_back(w);
        gbe_wave nw = {};
        nw.p0 = nw.p1 = p;
        nw.base_elems = g->h_dense_off[p];
        nw.row0 = row;
        nw.gi0 = gi;
        w = nw;
      }
      wave_of[p] = (int32_t)waves.size();
      w.p1 = p + 1;
      w.elems += e;
      w.n_rows += m;
      const int ng = (int)((m + g->gather_rows - 1) / g->gather_rows);
      w.gi_n += ng;
      row += m;
      gi += ng;
    }
    waves.push_back(w);
  }
  // tile lists: the whole-batch order (communities by decreasing m, stable) and its trace slots, cut by wave
  std::vector<int32_t> order(n_part);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return g->h_m[a] > g->h_m[b]; });
  std::vector<std::vector<gbe_tile_item>> it(waves.size()), la(waves.size());
  const int tile = g->tile;
  int32_t slot = 0;
  for (int p : order) {
    const int T = (g->h_m[p] + tile - 1) / tile;
    const int64_t ld = (g->h_m[p] + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    const int wv = wave_of[p];
    for (int ti = 0; ti < T; ++ti)
      for (int tj = ti; tj < T; ++tj) {
        const bool core_row = ti * tile < g->h_ncore[p];
        const gbe_tile_item item = {core_row ? slot : -1, ti | (tj << 16), p, g->h_m[p], g->h_ncore[p], (int32_t)ld,
                                    g->h_dense_off[p]};
        it[wv].push_back(item);
        if (core_row) { la[wv].push_back(item); ++slot; }
      }
  }
  std::vector<gbe_tile_item> all_it, all_la;
  for (size_t k = 0; k < waves.size(); ++k) {
    waves[k].it_first = (int32_t)all_it.size();
    waves[k].it_n = (int32_t)it[k].size();
    waves[k].last_first = (int32_t)all_la.size();
    waves[k].last_n = (int32_t)la[k].size();
    all_it.insert(all_it.end(), it[k].begin(), it[k].end());
    all_la.insert(all_la.end(), la[k].begin(), la[k].end());
  }
  gbe_set_alloc_stream(s);
  if (g->items_w) gbe_dev_free(g->items_w);
  if (g->items_last_w) gbe_dev_free(g->items_last_w);
  g->items_w = g->items_last_w = nullptr;
  GBE_TRY(upload(all_it, &g->items_w, s));
  GBE_TRY(upload(all_la, &g->items_last_w, s));
  g->waves = std::move(waves);
  g->waves_cap = cap_elems;
  return GBE_OK;
}
