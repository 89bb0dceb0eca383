// Step 4 (+ 5) for SMALL subgraphs, any number of them: one SP2 iteration per launch, whole matrices in shared memory.
//
//     Y_p = X_p X_p;  X_p <- Y_p  or  2 X_p - Y_p   for every community p with m_p <= 160
//
// The cost law of the paper (more partitions -> smaller core+halo size m) puts a whole regime of the method at
// m ~ 30 - 180 with hundreds to thousands of communities (BASELINE.json configs[4], tau = 1e-3).  There a 64 x 64 tile of
// the tiled kernel (gbe_x2.cu) is mostly mask, and the resident kernel (gbe_resident.cu) cannot run: its grid barrier
// needs all communities co-resident.  Here:
//   - a CTA owns a BIN of 1..16 communities for one iteration.  The bins are packed once per graph on the host (longest
//     processing time first onto k x SM-count bins, k waves), bounded by shared memory, by the accumulator registers
//     (16 warps x 4 work units) and by a cost cap, so that a launch is a whole number of equally heavy waves;
//   - every X_p of the bin is copied to shared memory once (cp.async, row stride ld_p + 4: conflict-free 64-bit
//     fragment loads) - the batch is read exactly once per iteration, and for these sizes it lives in L2;
//   - Y = X X^T on FP64 tensor cores (mma.sync.m8n8k4.f64): a work unit is one 8-row block x up to four 8-column blocks
//     on or above the diagonal; the host deals the units of the whole bin to the 16 warps by cost (at most 4 each),
//     accumulators stay in registers until every warp has finished reading X, then X is overwritten in place
//     (direct + mirrored store), exactly as in the resident kernel;
//   - the core-row traces of the NEW X (t1 = sum X_ii, t2 = sum_c X_ic^2 = Tr_core X^2 for symmetric X) are summed per
//     bin in a fixed order and the new X is streamed out with 128-bit stores;
//   - step 5 fused: the bin that publishes its partial LAST (one ticket per bin; the fence orders 16 bytes, not the bulk
//     stores, which come after it) sums all partials of the iteration in a fixed order and takes the branch decision
//     exactly as k_trace_branch does - one launch per SP2 iteration instead of two.  Which CTA is last does not change
//     the order of the sum: results are reproducible bit for bit.
// Communities with m_p > 160 of the same graph go through the tiled kernel in the same iteration (launched first; its
// partials sit in front of the bins' and enter the same sum).
// Bound: FP64 tensor pipe for m >~ 60; below that the copy in and out of shared memory (L2 latency).
#include <algorithm>
#include <numeric>
#include <queue>

#include "gbe_internal.cuh"

namespace {

constexpr int PK_WARPS = 16;
constexpr int PK_THREADS = PK_WARPS * 32;
constexpr int PK_MAXU = GBE_PK_MAXU;  // work units per warp
constexpr int PK_UCOLS = 4;           // 8-column blocks per unit
constexpr uint16_t PK_NONE = 0xFFFFu;

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;");
  asm volatile("cp.async.wait_group 0;" ::: "memory");
}

template <int NB>
__device__ __forceinline__ void pk_unit_mma(double (&acc)[PK_UCOLS][2], const double* __restrict__ pa,
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

// unit code: slot (4 bits) | row block bi (5) | first column block as (bj - bi) / 4 (3) | blocks - 1 (2)
__host__ __device__ inline uint16_t pk_encode(int slot, int bi, int bj, int nb) {
  return (uint16_t)(slot | (bi << 4) | (((bj - bi) >> 2) << 9) | ((nb - 1) << 12));
}

// fused == 1: the last bin to publish its partial reduces all n_partials pairs and takes the decision of step 5
__global__ void __launch_bounds__(PK_THREADS, 1)
    k_sp2_packed(const gbe_pk_cta* __restrict__ ctas, const gbe_pk_slot* __restrict__ slots, gbe_state* st,
                 const double* __restrict__ Xin, double* __restrict__ Xout, double* __restrict__ partials,
                 int partial_base, int n_partials, int iter, int last, int fused) {
  extern __shared__ __align__(16) double xs[];
  __shared__ gbe_pk_slot sl[GBE_PK_MAX_SLOTS];
  __shared__ double red[2 * PK_WARPS];
  __shared__ int is_last;

  if (st->stop) return;  // idempotency stop already fired (A-7): X is final
  const int branch = st->preset ? (int)st->br[iter] : st->branch;

  const int t = threadIdx.x, lane = t & 31, wid = t >> 5, g = lane >> 2, q = lane & 3;
  const gbe_pk_cta& me = ctas[blockIdx.x];
  const int n_slots = me.n_slots;
  if (t < n_slots * 8) reinterpret_cast<int*>(sl)[t] = reinterpret_cast<const int*>(slots + me.first_slot)[t];
  uint16_t ucode[PK_MAXU];
#pragma unroll
  for (int u = 0; u < PK_MAXU; ++u) ucode[u] = me.units[wid][u];
  __syncthreads();

  // ---- X_n of every community of the bin -> shared memory; rows [m, 8R) are zero (they stay zero under both updates)
  for (int s = 0; s < n_slots; ++s) {
    const int m = sl[s].m, ld = sl[s].ld, stride = ld + 4, h = ld >> 1;
    const double* __restrict__ src = Xin + sl[s].dense_off;
    double* dst = xs + sl[s].soff;
    for (int i = t; i < m * h; i += PK_THREADS) {
      const int r = i / h, c2 = i - r * h;
      cp_async16(dst + (size_t)r * stride + 2 * c2, src + 2 * (size_t)i);
    }
    for (int i = m * stride + t; i < 8 * sl[s].R * stride; i += PK_THREADS) dst[i] = 0.0;
  }
  cp_async_wait_all();
  __syncthreads();

  // ---- Y = X X^T: this warp's units, accumulators in registers
  double acc[PK_MAXU][PK_UCOLS][2];
#pragma unroll
  for (int u = 0; u < PK_MAXU; ++u)
#pragma unroll
    for (int j = 0; j < PK_UCOLS; ++j) acc[u][j][0] = acc[u][j][1] = 0.0;
#pragma unroll
  for (int u = 0; u < PK_MAXU; ++u) {
    if (ucode[u] == PK_NONE) continue;
    const int s = ucode[u] & 15, bi = (ucode[u] >> 4) & 31, bj = bi + 4 * ((ucode[u] >> 9) & 7), nb = 1 + ((ucode[u] >> 12) & 3);
    // the last iteration needs the core rows and (through the mirror) the core columns only (Eq.(6))
    if (last && bi * 8 >= sl[s].nc) continue;
    const int ld = sl[s].ld, stride = ld + 4;
    const double* pa = xs + sl[s].soff + (size_t)(bi * 8 + g) * stride + q;
    const double* pb = xs + sl[s].soff + (size_t)(bj * 8 + g) * stride + q;
    switch (nb) {
      case 4: pk_unit_mma<4>(acc[u], pa, pb, ld, stride); break;
      case 3: pk_unit_mma<3>(acc[u], pa, pb, ld, stride); break;
      case 2: pk_unit_mma<2>(acc[u], pa, pb, ld, stride); break;
      default: pk_unit_mma<1>(acc[u], pa, pb, ld, stride); break;
    }
  }
  __syncthreads();  // every warp is done reading X_n

  // ---- X_{n+1} = Y or 2 X_n - Y in place: only this lane touches (r, c), (r, c + 1) and their mirror images
#pragma unroll
  for (int u = 0; u < PK_MAXU; ++u) {
    if (ucode[u] == PK_NONE) continue;
    const int s = ucode[u] & 15, bi = (ucode[u] >> 4) & 31, bj = bi + 4 * ((ucode[u] >> 9) & 7), nb = 1 + ((ucode[u] >> 12) & 3);
    if (last && bi * 8 >= sl[s].nc) continue;
    const int stride = sl[s].ld + 4;
    double* x0 = xs + sl[s].soff;
    const int r = bi * 8 + g;
#pragma unroll
    for (int j = 0; j < PK_UCOLS; ++j) {
      if (j < nb) {
        const int c = (bj + j) * 8 + 2 * q;
        double* xr = x0 + (size_t)r * stride + c;
        double v0 = acc[u][j][0], v1 = acc[u][j][1];
        if (branch) {
          const double2 x = *reinterpret_cast<const double2*>(xr);
          v0 = 2.0 * x.x - v0;
          v1 = 2.0 * x.y - v1;
        }
        *reinterpret_cast<double2*>(xr) = make_double2(v0, v1);
        if (bj + j != bi) {  // off-diagonal block: mirror (the diagonal block is computed whole)
          x0[(size_t)c * stride + r] = v0;
          x0[(size_t)(c + 1) * stride + r] = v1;
        }
      }
    }
  }
  __syncthreads();

  // ---- core-row traces of X_{n+1}, summed over the bin in a fixed order
  {
    double s1 = 0.0, s2 = 0.0;
    for (int s = 0; s < n_slots; ++s) {
      const int nc = sl[s].nc, ld = sl[s].ld, stride = ld + 4;
      const double* x0 = xs + sl[s].soff;
      for (int i = wid; i < nc; i += PK_WARPS) {
        const double* __restrict__ row = x0 + (size_t)i * stride;
        for (int c = lane; c < ld; c += 32) {
          const double x = row[c];
          s2 += x * x;
          if (c == i) s1 += x;
        }
      }
    }
    s1 = warp_sum(s1);
    s2 = warp_sum(s2);
    if (lane == 0) { red[wid] = s1; red[PK_WARPS + wid] = s2; }
    __syncthreads();
    if (wid == 0) {
      const double a = warp_sum(lane < PK_WARPS ? red[lane] : 0.0);
      const double b = warp_sum(lane < PK_WARPS ? red[PK_WARPS + lane] : 0.0);
      if (lane == 0) {
        double* out = partials + 2 * (size_t)(partial_base + blockIdx.x);
        out[0] = a;
        out[1] = b;
        int lastflag = 0;
        if (fused) {
          __threadfence();  // the pair is visible before the ticket is taken
          lastflag = atomicAdd(&st->ticket, 1u) == gridDim.x - 1;
        }
        is_last = lastflag;
      }
    }
    __syncthreads();
  }

  // ---- step 5, by the bin that arrived last: all partials of this iteration (tiled kernel's and bins') in a fixed order
  if (fused && is_last) {
    __threadfence();
    double a1 = 0.0, a2 = 0.0;
    const double2* __restrict__ p2 = reinterpret_cast<const double2*>(partials);
    for (int i = t; i < n_partials; i += PK_THREADS) {
      const double2 v = __ldcg(p2 + i);
      a1 += v.x;
      a2 += v.y;
    }
    a1 = warp_sum(a1);
    a2 = warp_sum(a2);
    __syncthreads();  // red is free again
    if (lane == 0) { red[wid] = a1; red[PK_WARPS + wid] = a2; }
    __syncthreads();
    if (wid == 0) {
      a1 = warp_sum(lane < PK_WARPS ? red[lane] : 0.0);
      a2 = warp_sum(lane < PK_WARPS ? red[PK_WARPS + lane] : 0.0);
      if (lane == 0) {
        st->ticket = 0;
        gbe_trace_decide(st, a1, a2);
      }
    }
  }

  // ---- X_{n+1} -> the other dense buffer
  for (int s = 0; s < n_slots; ++s) {
    const int m = sl[s].m, ld = sl[s].ld, stride = ld + 4, h = ld >> 1;
    double2* __restrict__ dst = reinterpret_cast<double2*>(Xout + sl[s].dense_off);
    const double* x0 = xs + sl[s].soff;
    for (int i = t; i < m * h; i += PK_THREADS) {
      const int r = i / h, c2 = i - r * h;
      dst[i] = *reinterpret_cast<const double2*>(x0 + (size_t)r * stride + 2 * c2);
    }
  }
}

struct Unit { int slot, bi, bj, nb, cost; };

inline int units_of(int R) {
  int n = 0;
  for (int bi = 0; bi < R; ++bi) n += (R - bi + PK_UCOLS - 1) / PK_UCOLS;
  return n;
}
inline int64_t dmma_of(int m, int ld) {  // DMMA instructions of one X X^T: 8 x 8 blocks on or above the diagonal x ld / 4
  const int64_t R = (m + 7) / 8;
  return R * (R + 1) / 2 * (ld / 4);
}
inline size_t smem_doubles_of(int m, int ld) { return (size_t)((m + 7) / 8 * 8) * (ld + 4); }

template <typename T>
int upload(const std::vector<T>& h, T** d, cudaStream_t s) {
  GBE_TRY(gbe_dev_alloc((void**)d, std::max<size_t>(16, h.size() * sizeof(T))));
  if (!h.empty()) GBE_CUDA(cudaMemcpyAsync(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, s));
  return GBE_OK;
}
}  // namespace

// Packs the communities with 0 < m_p <= GBE_PK_MAX_M into bins (host; once per graph) and uploads the work description.
int gbe_build_packed(gbe_graph* g, cudaStream_t s) {
  g->n_pk_ctas = 0;
  g->pk_smem_bytes = 0;
  g->pk_n_small = 0;
  int dev = 0, smem_max = 0;
  GBE_CUDA(cudaGetDevice(&dev));
  GBE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  const int sms = gbe_sm_count();
  const size_t smem_cap = (size_t)std::max(0, smem_max - 4096) / sizeof(double);  // doubles; static shared memory aside
  std::vector<int> small;
  int64_t total = 0, biggest = 0;
  for (int p = 0; p < g->n_part; ++p) {
    const int m = g->h_m[p];
    if (m <= 0 || m > GBE_PK_MAX_M) continue;
    const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    if (smem_doubles_of(m, ld) > smem_cap || units_of((m + 7) / 8) > PK_WARPS * PK_MAXU) continue;
    small.push_back(p);
    total += dmma_of(m, ld);
    biggest = std::max(biggest, dmma_of(m, ld));
  }
  g->pk_n_small = (int32_t)small.size();
  if (small.empty()) return GBE_OK;
  auto cost = [&](int p) { return dmma_of(g->h_m[p], (g->h_m[p] + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN); };
  std::stable_sort(small.begin(), small.end(), [&](int a, int b) { return cost(a) > cost(b); });

  // k waves of `sms` bins: a bin should carry a few microseconds of tensor work (~3,000 DMMA = 6 us on one SM) so that the
  // copy in and out of shared memory is amortised, but never more than one wave's share
  const int64_t per_sm = (total + sms - 1) / sms;
  const int waves = (int)std::max<int64_t>(1, (per_sm + 1500) / 3000);
  const int n_bins_target = (int)std::min<int64_t>((int64_t)small.size(), (int64_t)waves * sms);
  struct Bin { int64_t load = 0; size_t smem = 0; int units = 0; std::vector<int> ps; };
  std::vector<Bin> bins(n_bins_target);
  using QE = std::pair<int64_t, int>;  // (load, bin): least loaded first, ties by index
  std::priority_queue<QE, std::vector<QE>, std::greater<QE>> pq;
  for (int b = 0; b < n_bins_target; ++b) pq.push({0, b});
  for (int p : small) {
    const int m = g->h_m[p], ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    const size_t need = smem_doubles_of(m, ld);
    const int nu = units_of((m + 7) / 8);
    // the least loaded bins first; a bin without room (registers, shared memory, slots) is set aside for this item
    std::vector<QE> aside;
    int chosen = -1;
    for (int tries = 0; tries < 8 && !pq.empty(); ++tries) {
      const QE e = pq.top();
      pq.pop();
      Bin& b = bins[e.second];
      if (b.units + nu <= PK_WARPS * PK_MAXU && b.smem + need <= smem_cap && (int)b.ps.size() < GBE_PK_MAX_SLOTS) {
        chosen = e.second;
        break;
      }
      aside.push_back(e);
    }
    for (const QE& e : aside) pq.push(e);
    if (chosen < 0) {
      bins.emplace_back();
      chosen = (int)bins.size() - 1;
    }
    Bin& b = bins[chosen];
    b.ps.push_back(p);
    b.units += nu;
    b.smem += need;
    b.load += cost(p);
    pq.push({b.load, chosen});
  }
  // heavy bins first in launch order
  std::vector<int> border(bins.size());
  std::iota(border.begin(), border.end(), 0);
  std::stable_sort(border.begin(), border.end(), [&](int a, int b) { return bins[a].load > bins[b].load; });

  std::vector<gbe_pk_cta> h_ctas;
  std::vector<gbe_pk_slot> h_slots;
  size_t smem_need = 0;
  for (int bi_ : border) {
    const Bin& b = bins[bi_];
    if (b.ps.empty()) continue;
    gbe_pk_cta c;
    c.first_slot = (int32_t)h_slots.size();
    c.n_slots = (int32_t)b.ps.size();
    for (int w = 0; w < PK_WARPS; ++w)
      for (int u = 0; u < PK_MAXU; ++u) c.units[w][u] = PK_NONE;
    std::vector<Unit> units;
    size_t soff = 0;
    for (int k = 0; k < (int)b.ps.size(); ++k) {
      const int p = b.ps[k], m = g->h_m[p], ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN, R = (m + 7) / 8;
      h_slots.push_back({p, m, g->h_ncore[p], ld, (int32_t)soff, R, g->h_dense_off[p]});
      soff += smem_doubles_of(m, ld);
      for (int bi = 0; bi < R; ++bi)
        for (int bj = bi; bj < R; bj += PK_UCOLS) {
          const int nb = std::min(PK_UCOLS, R - bj);
          units.push_back({k, bi, bj, nb, nb * (ld / 4)});
        }
    }
    c.smem_doubles = (int32_t)soff;
    smem_need = std::max(smem_need, soff * sizeof(double));
    // the units of the bin onto the 16 warps: longest first, always to the least loaded warp with a free slot
    std::stable_sort(units.begin(), units.end(), [](const Unit& a, const Unit& b) { return a.cost > b.cost; });
    int wload[PK_WARPS] = {0}, wcnt[PK_WARPS] = {0};
    for (const Unit& un : units) {
      int best = -1;
      for (int w = 0; w < PK_WARPS; ++w)
        if (wcnt[w] < PK_MAXU && (best < 0 || wload[w] < wload[best])) best = w;
      if (best < 0) return GBE_EINVAL;  // cannot happen: units <= 16 x 4 per bin
      c.units[best][wcnt[best]++] = pk_encode(un.slot, un.bi, un.bj, un.nb);
      wload[best] += un.cost;
    }
    h_ctas.push_back(c);
  }
  g->n_pk_ctas = (int32_t)h_ctas.size();
  g->pk_smem_bytes = smem_need;
  GBE_TRY(upload(h_ctas, &g->pk_ctas, s));
  GBE_TRY(upload(h_slots, &g->pk_slots, s));
  return GBE_OK;
}

// One SP2 iteration of the packed communities.  partial_base: index of the first bin's pair in `partials` (the pairs of the
// tiled kernel, if it runs in the same iteration, sit in front); n_partials: all pairs of the iteration.
int gbe_launch_sp2_packed(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials,
                          int partial_base, int n_partials, int iter, bool last, bool fused, cudaStream_t s) {
  if (g->n_pk_ctas == 0) return GBE_OK;
  static gbe_device_once configured;
  if (configured.first()) {
    int dev = 0, smem_max = 0;
    GBE_CUDA(cudaGetDevice(&dev));
    GBE_CUDA(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    GBE_CUDA(cudaFuncSetAttribute(k_sp2_packed, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - 4096));
  }
  k_sp2_packed<<<g->n_pk_ctas, PK_THREADS, g->pk_smem_bytes, s>>>(g->pk_ctas, g->pk_slots, st, Xin, Xout, partials,
                                                                 partial_base, n_partials, iter, last ? 1 : 0,
                                                                 fused ? 1 : 0);
  GBE_LAUNCHED();
  return GBE_OK;
}
