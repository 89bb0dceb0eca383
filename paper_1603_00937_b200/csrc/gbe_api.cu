// The C ABI of include/gbe.h: argument checks, the graph handle, workspace carving and the launch sequence.
// Every step of the path runs in the kernels of gbe_{bounds,graph,halo,gather,x2,trace,scatter}.cu.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "gbe_internal.cuh"

std::atomic<uint64_t> g_gbe_launches{0};
// communities up to this size go to the packed kernel (gbe_small.cu); 116: the largest whose X fits half an SM's shared
// memory, so that two bins share an SM
static std::atomic<int32_t> g_pk_max_m{GBE_PK_MAX_M};
int gbe_packed_max_m() { return g_pk_max_m.load(); }

namespace {
thread_local char g_cuda_err[512] = "";

// Optional per-launch timing (gbe_density_timed): one event pair around every launcher call.
enum Phase { PH_BOUNDS = 0, PH_GATHER, PH_X2, PH_TRACE, PH_SCATTER, PH_X2_LAST, PH_COUNT };
struct Timer {
  struct Rec { int phase, launches; cudaEvent_t e0, e1; };
  std::vector<Rec> recs;
  cudaStream_t s;
  explicit Timer(cudaStream_t st) : s(st) {}
  ~Timer() { for (auto& r : recs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); } }
};
template <typename F>
int timed(Timer* tm, int phase, int launches, F&& fn) {
  if (!tm) return fn();
  Timer::Rec r{phase, launches, nullptr, nullptr};
  GBE_CUDA(cudaEventCreate(&r.e0));
  GBE_CUDA(cudaEventCreate(&r.e1));
  tm->recs.push_back(r);
  GBE_CUDA(cudaEventRecord(r.e0, tm->s));
  const int rc = fn();
  GBE_CUDA(cudaEventRecord(r.e1, tm->s));
  return rc;
}

// mode 0: branch chosen on the device every iteration; 1: preset sequence, traces logged every iteration;
// 2: preset sequence, no per-iteration trace kernel (the final X is in buffer iters & 1)
__global__ void k_init_state(gbe_state* st, double n_occ, double idem_tol, int iters, int mode, int inplace) {
  st->inplace = inplace;
  st->n_occ = n_occ;
  st->idem_tol = idem_tol;
  st->iters = iters;
  st->iter = mode == 2 ? iters : 0;
  st->branch = 0;
  st->stop = 0;
  st->iters_done = mode == 2 ? iters : 0;
  st->preset = mode != 0;
  st->bar = 0;
  st->ticket = 0;
}

struct WS {
  gbe_state* st;
  double *blo, *bhi, *partials, *X0, *X1;
};
int carve(const gbe_graph* g, void* workspace, size_t bytes, WS* w) {
  if (!workspace) return GBE_EINVAL;
  if (bytes < g->ws_bytes) return GBE_ENOMEM;
  if (reinterpret_cast<uintptr_t>(workspace) % 256) return GBE_EINVAL;
  unsigned char* b = static_cast<unsigned char*>(workspace);
  w->st = reinterpret_cast<gbe_state*>(b);
  w->blo = reinterpret_cast<double*>(b + g->ws_bounds);
  w->bhi = w->blo + 1024;
  w->partials = reinterpret_cast<double*>(b + g->ws_partials);
  w->X0 = reinterpret_cast<double*>(b + g->ws_x0);
  w->X1 = reinterpret_cast<double*>(b + g->ws_x1);
  return GBE_OK;
}
int check_csr(const gbe_csr_view* H) {
  if (!H || !H->row_ptr || H->n <= 0 || H->nnz < 0 || H->n > INT32_MAX) return GBE_EINVAL;
  if (H->nnz > 0 && (!H->col_idx || !H->val)) return GBE_EINVAL;
  return GBE_OK;
}
}  // namespace

void gbe_set_cuda_error(cudaError_t e, const char* what, int line) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (%s) at %s, line %d", cudaGetErrorString(e), cudaGetErrorName(e), what,
           line);
}

extern "C" {

const char* gbe_last_cuda_error(void) { return g_cuda_err; }
const char* gbe_version(void) { return "gbe 0.1 (sm_100a)"; }

const char* gbe_strerror(int status) {
  switch (status) {
    case GBE_OK: return "ok";
    case GBE_EINVAL: return "invalid argument";
    case GBE_ENOTSYM: return "H is not symmetric";
    case GBE_EDEGENERATE: return "degenerate spectral bounds (eps_max == eps_min)";
    case GBE_EMISMATCH: return "H does not match the graph";
    case GBE_ENOMEM: return "workspace too small or allocation failed";
    case GBE_ECUDA: return g_cuda_err[0] ? g_cuda_err : "CUDA error";
    case GBE_ELIMIT: return "problem larger than the fixed limit of this entry point (n > GBE_STATIC_MAX_N)";
    default: return "unknown status";
  }
}

void gbe_free_graph(gbe_graph* g) {
  if (!g) return;
  void* ptrs[] = {g->S_row_ptr, g->S_col,     g->sub_ptr,  g->sub_idx,  g->ncore,    g->msize, g->dense_off, g->D_row_ptr,
                  g->D_col,     g->scat_base, g->scat_pos, g->scat_ofs, g->row_part, g->items, g->items_last, g->items_h, g->items_last_h, g->pk[0].ctas, g->pk[0].codes, g->pk[0].rows, g->gitems, g->row_src, g->row_nc, g->H_rp, g->H_ci, g->H_va, g->tmaps, g->items_w, g->items_last_w};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  delete g;
}

static int build_graph_impl(const gbe_csr_view* H, const gbe_graph_opts* opts, const int32_t* part, int32_t n_part,
                            void* cuda_stream, gbe_graph** out, const gbe_graph* prev, const double* D_prev) {
  if (!out) return GBE_EINVAL;
  *out = nullptr;
  GBE_TRY(check_csr(H));
  if (!opts || !(opts->tau >= 0.0) || std::isnan(opts->tau)) return GBE_EINVAL;
  const int power = opts->power == 0 ? 2 : opts->power;
  if (power < 1 || power > GBE_MAX_POWER) return GBE_EINVAL;
  if (n_part < 1 || n_part > H->n) return GBE_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_set_alloc_stream(s);

  gbe_graph* g = new (std::nothrow) gbe_graph();
  if (!g) return GBE_ENOMEM;
  g->n = H->n;
  g->n_part = n_part;
  g->tau = opts->tau;
  g->power = power;
  g->tile = 64;
  struct Guard {
    gbe_graph* g;
    ~Guard() { if (g) gbe_free_graph(g); }
  } guard{g};

  // step 0: bounds of the H given here; they travel to pinned host words and are looked at after the first
  // synchronisation of the build (a build has four: accumulator capacity of the product; nnz(S); subgraph sizes; end)
  DevBuf st, bl;
  GBE_TRY(st.alloc(sizeof(gbe_state)));
  GBE_TRY(bl.alloc(2 * 1024 * sizeof(double)));
  GBE_TRY(gbe_launch_bounds(*H, bl.as<double>(), bl.as<double>() + 1024, 1024, st.as<gbe_state>(), s));
  double stack_b[2] = {0.0, 0.0};
  int32_t* const pin = gbe_pinned_words();
  double* const b = pin ? reinterpret_cast<double*>(pin + 8) : stack_b;
  GBE_CUDA(cudaMemcpyAsync(b, st.p, 2 * sizeof(double), cudaMemcpyDeviceToHost, s));
  if (!pin) GBE_CUDA(cudaStreamSynchronize(s));

  // step 1: S_tau - from H and its thresholded powers (A-1), or by Eq.(8) from the previous D and this H
  if (prev)
    GBE_TRY(gbe_build_pattern_eq8(*H, prev->D_row_ptr, prev->D_col, D_prev, g->tau, s, &g->S_row_ptr, &g->S_col, &g->nnz_S,
                                  prev->nnz_D));
  else
    GBE_TRY(gbe_build_pattern(*H, st.as<gbe_state>(), g->tau, power, opts->check_symmetry, s, &g->S_row_ptr, &g->S_col,
                              &g->nnz_S));
  // step 2: subgraphs, layout, pattern of D, work lists (synchronises; checks the bounds)
  GBE_TRY(gbe_build_subgraphs(g, part, s, b));
  g->eps_min = b[0];
  g->eps_max = b[1];
  guard.g = nullptr;
  *out = g;
  return GBE_OK;
}

int gbe_build_graph(const gbe_csr_view* H, const gbe_graph_opts* opts, const int32_t* part, int32_t n_part,
                    void* cuda_stream, gbe_graph** out) {
  return build_graph_impl(H, opts, part, n_part, cuda_stream, out, nullptr, nullptr);
}

int gbe_update_graph(const gbe_graph* prev, const double* D_prev, const gbe_csr_view* H, const gbe_graph_opts* opts,
                     const int32_t* part, int32_t n_part, void* cuda_stream, gbe_graph** out) {
  if (!prev || (!D_prev && prev->nnz_D > 0)) return GBE_EINVAL;
  if (H && H->n != prev->n) return GBE_EMISMATCH;
  return build_graph_impl(H, opts, part, n_part, cuda_stream, out, prev, D_prev);
}

static int choose_sp2(const gbe_graph* g, int mode);

int gbe_graph_get_info(const gbe_graph* g, gbe_graph_info* o) {
  if (!g || !o) return GBE_EINVAL;
  memset(o, 0, sizeof(*o));
  o->n = g->n;
  o->nnz_S = g->nnz_S;
  o->n_part = g->n_part;
  o->sum_m = g->sum_m;
  o->max_m = g->max_m;
  o->nnz_D = g->nnz_D;
  o->dense_elems = g->dense_elems;
  o->n_tiles = g->n_items;
  o->sp2_flops_per_iter = g->flops_per_iter;
  o->sp2_exec_flops_per_iter = g->exec_flops_per_iter;
  o->sp2_sym_flops_per_iter = g->sym_flops_per_iter;
  o->n_tiles_last = g->n_items_last;
  o->sp2_flops_last_iter = g->flops_last_iter;
  o->sp2_exec_flops_last_iter = g->exec_flops_last_iter;
  o->eps_min = g->eps_min;
  o->eps_max = g->eps_max;
  o->contiguous_cores = g->contiguous;
  o->tile = g->tile;
  o->workspace_bytes = g->ws_bytes;
  o->workspace_bytes_fermi = g->ws_bytes_fermi;
  o->resident_sp2 = choose_sp2(g, 0) == 2 ? 1 : 0;
  o->sp2_path_chosen = choose_sp2(g, 0);
  o->n_small = g->pk_n_small;
  o->n_bins = g->n_pk_ctas;
  o->workspace_bytes_preset_min = g->ws_bytes_wave_min;
  o->x2_tma = g->tmaps ? 1 : 0;
  o->resident_fits = g->resident_fits;
  o->resident_cluster = g->resident_cluster;
  return GBE_OK;
}

int gbe_graph_export(const gbe_graph* g, void* cuda_stream, int64_t* S_row_ptr, int32_t* S_col, int64_t* sub_ptr,
                     int32_t* sub_idx, int32_t* ncore, int64_t* D_row_ptr, int32_t* D_col) {
  if (!g) return GBE_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  auto cp = [&](void* dst, const void* src, size_t bytes) -> int {
    if (dst && bytes) GBE_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, s));
    return GBE_OK;
  };
  GBE_TRY(cp(S_row_ptr, g->S_row_ptr, (size_t)(g->n + 1) * 8));
  GBE_TRY(cp(S_col, g->S_col, (size_t)g->nnz_S * 4));
  GBE_TRY(cp(sub_ptr, g->sub_ptr, (size_t)(g->n_part + 1) * 8));
  GBE_TRY(cp(sub_idx, g->sub_idx, (size_t)g->sum_m * 4));
  GBE_TRY(cp(ncore, g->ncore, (size_t)g->n_part * 4));
  GBE_TRY(cp(D_row_ptr, g->D_row_ptr, (size_t)(g->n + 1) * 8));
  GBE_TRY(cp(D_col, g->D_col, (size_t)g->nnz_D * 4));
  return GBE_OK;
}

static int do_gather(const gbe_csr_view* H, const gbe_graph* g, void* workspace, size_t workspace_bytes,
                     void* cuda_stream, Timer* tm) {
  if (!g) return GBE_EINVAL;
  GBE_TRY(check_csr(H));
  if (H->n != g->n) return GBE_EMISMATCH;
  WS w;
  GBE_TRY(carve(g, workspace, workspace_bytes, &w));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  GBE_TRY(timed(tm, PH_BOUNDS, 2, [&] { return gbe_launch_bounds(*H, w.blo, w.bhi, 1024, w.st, s); }));
  GBE_TRY(timed(tm, PH_GATHER, g->n_gitems ? 1 : 0,
                [&] { return gbe_launch_gather(*H, g, w.st, w.X0, w.partials, s); }));
  return GBE_OK;
}
int gbe_gather(const gbe_csr_view* H, const gbe_graph* g, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  return do_gather(H, g, workspace, workspace_bytes, cuda_stream, nullptr);
}

// Which kernels run steps 4-5 (1 tiled, 2 resident, 3 packed + tiled for the large communities); mode as in k_init_state.
// The resident kernel needs the largest community in shared memory and, unless the sequence is preset and no trace is
// logged (no exchange between CTAs), all communities co-resident (cooperative launch).  The packed kernel takes the
// communities with m <= GBE_PK_MAX_M, any number of them.
static int choose_sp2(const gbe_graph* g, int mode) {
  if (g->n_items == 0 || g->sp2_path == 1) return 1;
  const bool can_res = g->resident_fits && (mode == 2 || g->n_part <= g->resident_coresident);
  const bool can_pk = g->n_pk_ctas > 0;
  if (g->sp2_path == 2) return can_res ? 2 : 1;
  if (g->sp2_path == 3) return can_pk ? 3 : 1;
  // auto.  Resident: one launch for the whole loop - wins whenever the communities are small enough that one SM per
  // community keeps up with the tiled kernels spreading the tiles over all SMs (measured, profiles/r02_small_systems.md:
  // always up to m = 128; at m = 160 from about 50 communities on - 64: 1.09 against 1.24 ms, 32: 1.08 against 0.97 ms).
  if (can_res && (g->max_m <= 128 || g->n_part >= g->resident_coresident / 3)) return 2;
  // Packed: every community fits shared memory and there are enough of them to occupy the device (measured, DESIGN.md 6:
  // a graph that also needs the tiled kernel for some communities pays a second, poorly filled launch per iteration and
  // is not faster than the tiled kernels alone).
  if (can_pk && g->n_pk_ctas >= gbe_sm_count() / 2 && g->n_items_h == 0) return 3;
  // Mixed graph, nearly everything packed: the tiled launch for the few larger communities (at most two tiles per SM)
  // runs next to the last wave of bins (do_sp2); measured on tau = 1e-3 x 512 communities (504 packed, 8 tiled).  Not
  // for a pre-set sequence without traces, which has no decision to synchronise on and keeps the serial pair of launches.
  if (can_pk && mode != 2 && g->n_pk_ctas >= gbe_sm_count() && g->n_items_h > 0 && g->n_items_h <= 2 * gbe_sm_count()) return 3;
  return 1;
}

int gbe_graph_set_sp2_path(gbe_graph* g, int32_t path) {
  if (!g || path < 0 || path > 3) return GBE_EINVAL;
  if (path == 2 && !g->resident_fits) return GBE_EINVAL;
  g->sp2_path = path;
  return GBE_OK;
}

int gbe_graph_set_gather_path(gbe_graph* g, int32_t path) {
  if (!g || path < 0 || path > 2) return GBE_EINVAL;
  g->gather_path = path;
  return GBE_OK;
}

int gbe_graph_set_scatter_path(gbe_graph* g, int32_t path) {
  if (!g || path < 0 || path > 1) return GBE_EINVAL;
  g->scatter_path = path;
  return GBE_OK;
}

static int do_sp2(const gbe_graph* g, double n_occ, int32_t iters, double idem_tol, void* workspace,
                  size_t workspace_bytes, void* cuda_stream, Timer* tm, const uint8_t* preset = nullptr,
                  bool trace_each = true) {
  if (!g) return GBE_EINVAL;
  if (!(n_occ >= 0.0) || n_occ > (double)g->n || iters < 0 || iters > GBE_MAX_ITERS || std::isnan(idem_tol))
    return GBE_EINVAL;
  WS w;
  GBE_TRY(carve(g, workspace, workspace_bytes, &w));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int mode = !preset ? 0 : (trace_each ? 1 : 2);
  int path = choose_sp2(g, mode);
  if (path == 2) {
    const int inplace = 0;
    // small communities: the whole loop in one kernel, X_p resident in shared memory (gbe_resident.cu)
    GBE_TRY(timed(tm, PH_TRACE, 1, [&]() -> int {
      k_init_state<<<1, 1, 0, s>>>(w.st, n_occ, idem_tol, iters, mode, inplace);
      GBE_LAUNCHED();
      if (preset && iters > 0)
        GBE_CUDA(cudaMemcpyAsync(w.st->br, preset, (size_t)iters, cudaMemcpyHostToDevice, s));
      return GBE_OK;
    }));
    const int rc = timed(tm, PH_X2, 1, [&] { return gbe_launch_sp2_resident(g, w.st, w.X0, w.X1, w.partials, mode, s); });
    if (rc != GBE_RESIDENT_UNAVAILABLE) {
      GBE_TRY(rc);
      if (mode == 2)
        GBE_TRY(timed(tm, PH_TRACE, 1, [&] { return gbe_launch_trace_branch(w.st, w.partials, g->n_part, s); }));
      return GBE_OK;
    }
    // the grid does not fit the device at this moment (shared device): the kernels without a grid barrier take over
    path = g->n_pk_ctas > 0 && g->n_items_h == 0 ? 3 : 1;
  }
  // Packed kernel with EVERY community packed: a bin has all of its X_p in shared memory before it stores anything, so
  // X is updated in place in buffer 0 (half the footprint in L2)
  const int inplace = path == 3 && g->n_items_h == 0;
  if (iters > 0 && (path == 1 || g->n_items_h > 0)) GBE_TRY(gbe_x2_prepare(g, w.X0, w.X1, s));  // tensor maps -> this workspace
  // traces of X_0 (partials written by the gather), branch of iteration 0
  GBE_TRY(timed(tm, PH_TRACE, mode == 2 ? 1 : 2, [&]() -> int {
    k_init_state<<<1, 1, 0, s>>>(w.st, n_occ, idem_tol, iters, mode, inplace);
    GBE_LAUNCHED();
    if (preset && iters > 0)
      GBE_CUDA(cudaMemcpyAsync(w.st->br, preset, (size_t)iters, cudaMemcpyHostToDevice, s));
    if (mode == 2) return GBE_OK;
    return gbe_launch_trace_branch(w.st, w.partials, g->n_gitems, s);
  }));
  for (int it = 0; it < iters; ++it) {
    const double* in = (it & 1) && !inplace ? w.X1 : w.X0;
    double* outp = (it & 1) || inplace ? w.X0 : w.X1;
    // Iteration iters - 1 is the last one whether or not the idempotency stop fires before it (then it is a no-op):
    // only the core rows and columns of its result are read again (trace, scatter), so it runs the core tiles only.
    const bool last = it == iters - 1;
    if (path == 3 && inplace && mode != 2 && 2 * g->n_pk_ctas <= g->n_partials) {  // (always: n_partials >= 2 n_part)
      // every community packed: one launch per iteration and NO step-5 tail - the bins of launch it + 1 sum the pairs of
      // launch it themselves (lazy decision, gbe_small.cu); the pairs alternate between two halves of `partials`
      const int nb = g->n_pk_ctas;
      GBE_TRY(timed(tm, last ? PH_X2_LAST : PH_X2, 1, [&]() -> int {
        return gbe_launch_sp2_packed(g, w.st, in, outp, w.partials, (it & 1) * nb, nb, it, last, 2, ((it - 1) & 1) * nb,
                                     it > 0 ? nb : 0, s);
      }));
      if (last)  // t1, t2 of the final X and the last log entry
        GBE_TRY(timed(tm, PH_TRACE, 1, [&] { return gbe_launch_trace_branch(w.st, w.partials + 2 * (size_t)((it & 1) * nb), nb, s); }));
      continue;
    }
    if (path == 3 && g->n_items_h > 0 && mode != 2 && 2 * (g->n_items_last_h + g->n_pk_ctas) <= g->n_partials) {
      // MIXED graph, lazy decision over both kinds of pairs.  The packed launch goes first; the tiled launch for the few
      // larger communities follows as its programmatic dependent: it becomes resident when the last bins have started -
      // on the SMs the last, partly filled wave of bins leaves free - waits at its top for the branch of the iteration
      // (published by bin 0: fence + state.iter) and at its end for the packed launch to complete, so that the packed
      // launch of the next iteration, which waits for the tiled launch only, finds both done.  Pairs: [tiles | bins],
      // alternating between two halves of `partials`.
      const int nh = g->n_items_last_h, nb = g->n_pk_ctas, np = nh + nb;
      const int base = (it & 1) * np, prev = ((it - 1) & 1) * np;
      const int pdl = gbe_pdl_enabled() ? GBE_PDL_TOP : GBE_PDL_NONE;
      GBE_TRY(timed(tm, last ? PH_X2_LAST : PH_X2, 2, [&]() -> int {
        GBE_TRY(gbe_launch_sp2_packed(g, w.st, in, outp, w.partials, base + nh, np, it, last, 2, prev, it > 0 ? np : 0, s));
        return gbe_launch_x2(g, w.st, in, outp, w.partials + 2 * (size_t)base, it, last, true, it & 1, s, pdl, true);
      }));
      if (last)
        GBE_TRY(timed(tm, PH_TRACE, 1, [&] { return gbe_launch_trace_branch(w.st, w.partials + 2 * (size_t)base, np, s); }));
      continue;
    }
    if (path == 3) {
      // (pre-set sequence without traces, or no room for two sets of pairs) small communities: bins in shared memory, one
      // launch per iteration, step 5 taken by the bin that arrives last (gbe_small.cu); the larger communities of the
      // same graph go through the tiled kernel first
      const int n_pairs = g->n_items_last_h + g->n_pk_ctas;
      GBE_TRY(timed(tm, last ? PH_X2_LAST : PH_X2, (g->n_items_h ? 1 : 0) + 1, [&]() -> int {
        GBE_TRY(gbe_launch_x2(g, w.st, in, outp, w.partials, it, last, true, it & 1, s));
        return gbe_launch_sp2_packed(g, w.st, in, outp, w.partials, g->n_items_last_h, n_pairs, it, last, mode != 2 ? 1 : 0,
                                     0, 0, s);
      }));
      continue;
    }
    const int n_part_it = g->n_items_last;  // one packed partial per tile with a core row, in every iteration
    // programmatic dependent launch: k_trace_branch is resident and waiting when the X^2 launch ends, and lets the next
    // X^2 launch go the moment its decision is visible (GBE_PDL_EARLY: that launch never waits).  Without traces an X^2
    // launch follows an X^2 launch and would have to wait at its top: measured slower than plain stream order on small
    // systems (its CTAs become resident next to the running ones and only wait), no gain on large ones - not used.
    const int pdl = gbe_pdl_enabled() && mode != 2 ? GBE_PDL_EARLY : GBE_PDL_NONE;
    GBE_TRY(timed(tm, last ? PH_X2_LAST : PH_X2, g->n_items ? 1 : 0,
                  [&] { return gbe_launch_x2(g, w.st, in, outp, w.partials, it, last, false, it & 1, s, pdl); }));
    if (mode != 2)
      GBE_TRY(timed(tm, PH_TRACE, 1, [&] { return gbe_launch_trace_branch(w.st, w.partials, n_part_it, s, pdl ? GBE_PDL_TOP : GBE_PDL_NONE); }));
  }
  if (mode == 2) {  // one trace kernel at the end: t1, t2 of the final X for the log (written at index iters)
    const int n_pairs = iters == 0 ? g->n_gitems : (path == 3 ? g->n_items_last_h + g->n_pk_ctas : g->n_items_last);
    GBE_TRY(timed(tm, PH_TRACE, 1, [&] { return gbe_launch_trace_branch(w.st, w.partials, n_pairs, s); }));
  }
  return GBE_OK;
}
int gbe_sp2(const gbe_graph* g, double n_occ, int32_t iters, double idem_tol, void* workspace, size_t workspace_bytes,
            void* cuda_stream) {
  return do_sp2(g, n_occ, iters, idem_tol, workspace, workspace_bytes, cuda_stream, nullptr);
}

static int do_scatter(const gbe_graph* g, void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val,
                      Timer* tm) {
  if (!g || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  WS w;
  GBE_TRY(carve(g, workspace, workspace_bytes, &w));
  return timed(tm, PH_SCATTER, g->sum_m ? 1 : 0, [&] {
    return gbe_launch_scatter(g, w.st, w.X0, w.X1, D_val, static_cast<cudaStream_t>(cuda_stream));
  });
}
int gbe_scatter(const gbe_graph* g, void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val) {
  return do_scatter(g, workspace, workspace_bytes, cuda_stream, D_val, nullptr);
}

static int read_log_at(const gbe_graph* g, const void* workspace, void* cuda_stream, gbe_sp2_log* log);
int gbe_read_log(const gbe_graph* g, const void* workspace, size_t workspace_bytes, void* cuda_stream, gbe_sp2_log* log) {
  if (!g || !log) return GBE_EINVAL;
  WS w;
  GBE_TRY(carve(g, const_cast<void*>(workspace), workspace_bytes, &w));
  return read_log_at(g, workspace, cuda_stream, log);
}
// the state sits at the start of the workspace whatever its size
static int read_log_at(const gbe_graph* g, const void* workspace, void* cuda_stream, gbe_sp2_log* log) {
  (void)g;
  WS w;
  w.st = reinterpret_cast<gbe_state*>(const_cast<void*>(workspace));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_state hs_small;  // only the header is needed first
  GBE_CUDA(cudaMemcpyAsync(&hs_small, w.st, offsetof(gbe_state, t1), cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  if (hs_small.degenerate) return GBE_EDEGENERATE;
  const int k = hs_small.iters_done;
  log->iters_done = k;
  if (log->t1) GBE_CUDA(cudaMemcpyAsync(log->t1, w.st->t1, (size_t)(k + 1) * 8, cudaMemcpyDeviceToHost, s));
  if (log->t2) GBE_CUDA(cudaMemcpyAsync(log->t2, w.st->t2, (size_t)(k + 1) * 8, cudaMemcpyDeviceToHost, s));
  if (log->branch && k > 0) GBE_CUDA(cudaMemcpyAsync(log->branch, w.st->br, (size_t)k, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  return GBE_OK;
}

static int do_density(const gbe_csr_view* H, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                      void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val, gbe_sp2_log* log,
                      Timer* tm) {
  if (!g || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  if (!(n_occ >= 0.0) || n_occ > (double)g->n || iters < 0 || iters > GBE_MAX_ITERS || std::isnan(idem_tol))
    return GBE_EINVAL;
  GBE_TRY(do_gather(H, g, workspace, workspace_bytes, cuda_stream, tm));
  GBE_TRY(do_sp2(g, n_occ, iters, idem_tol, workspace, workspace_bytes, cuda_stream, tm));
  GBE_TRY(do_scatter(g, workspace, workspace_bytes, cuda_stream, D_val, tm));
  if (log) GBE_TRY(gbe_read_log(g, workspace, workspace_bytes, cuda_stream, log));
  return GBE_OK;
}
int gbe_density(const gbe_csr_view* H, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val, gbe_sp2_log* log) {
  return do_density(H, g, n_occ, iters, idem_tol, workspace, workspace_bytes, cuda_stream, D_val, log, nullptr);
}

int gbe_density_timed(const gbe_csr_view* H, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                      void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val, gbe_sp2_log* log,
                      gbe_phase_times* times) {
  if (!times) return GBE_EINVAL;
  memset(times, 0, sizeof(*times));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  Timer tm(s);
  GBE_TRY(do_density(H, g, n_occ, iters, idem_tol, workspace, workspace_bytes, cuda_stream, D_val, log, &tm));
  GBE_CUDA(cudaStreamSynchronize(s));
  float* ms[PH_COUNT] = {&times->bounds_ms, &times->gather_ms,  &times->x2_ms,
                         &times->trace_ms,  &times->scatter_ms, &times->x2_last_ms};
  int32_t* nl[PH_COUNT] = {&times->bounds_launches, &times->gather_launches,  &times->x2_launches,
                           &times->trace_launches,  &times->scatter_launches, &times->x2_last_launches};
  for (auto& r : tm.recs) {
    float t = 0.f;
    GBE_CUDA(cudaEventElapsedTime(&t, r.e0, r.e1));
    *ms[r.phase] += t;
    *nl[r.phase] += r.launches;
  }
  if (!tm.recs.empty()) GBE_CUDA(cudaEventElapsedTime(&times->total_ms, tm.recs.front().e0, tm.recs.back().e1));
  return GBE_OK;
}

// gbe_density_preset without traces in a workspace that holds only part of the batch: waves of communities (gbe_plan_waves)
static int density_preset_waves(const gbe_csr_view* H, const gbe_graph* g, const uint8_t* branch, int32_t iters,
                                void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val) {
  GBE_TRY(check_csr(H));
  if (H->n != g->n) return GBE_EMISMATCH;
  if (reinterpret_cast<uintptr_t>(workspace) % 256) return GBE_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  unsigned char* b = static_cast<unsigned char*>(workspace);
  gbe_state* st = reinterpret_cast<gbe_state*>(b);
  double* blo = reinterpret_cast<double*>(b + g->ws_bounds);
  double* partials = reinterpret_cast<double*>(b + g->ws_partials);
  const size_t cap_elems = ((workspace_bytes - g->ws_x0) / 2 / 256 * 256) / 8;  // doubles per dense buffer of a wave
  double* const B0 = reinterpret_cast<double*>(b + g->ws_x0);
  double* const B1 = B0 + cap_elems;
  GBE_TRY(gbe_plan_waves(g, cap_elems, s));
  GBE_TRY(gbe_launch_bounds(*H, blo, blo + 1024, 1024, st, s));
  k_init_state<<<1, 1, 0, s>>>(st, 0.0, -1.0, iters, 2, 0);
  GBE_LAUNCHED();
  if (iters > 0) GBE_CUDA(cudaMemcpyAsync(st->br, branch, (size_t)iters, cudaMemcpyHostToDevice, s));
  for (const gbe_wave& w : g->waves) {
    // the wave's buffers are the full-size ones shifted by its first offset: every kernel keeps its absolute offsets
    double* const X0 = B0 - w.base_elems;
    double* const X1 = B1 - w.base_elems;
    if (iters > 0) GBE_TRY(gbe_x2_prepare(g, X0, X1, s));
    // (the traces of X_0 the gather leaves are only wanted for iters == 0: else they go behind the slots of the tiles)
    GBE_TRY(gbe_launch_gather(*H, g, st, X0, iters > 0 ? partials + 2 * (size_t)g->n_items_last : partials, s, w.gi0, w.gi_n));
    for (int it = 0; it < iters; ++it) {
      const bool last = it == iters - 1;
      GBE_TRY(gbe_launch_x2_items(g, st, (it & 1) ? X1 : X0, (it & 1) ? X0 : X1, partials, it,
                                  (last ? g->items_last_w + w.last_first : g->items_w + w.it_first),
                                  last ? w.last_n : w.it_n, it & 1, s));
    }
    GBE_TRY(gbe_launch_scatter(g, st, X0, X1, D_val, s, w.row0, w.n_rows));
  }
  // t1, t2 of the final X for the log (index iters): every wave left its pairs in the whole-batch slots
  return gbe_launch_trace_branch(st, partials, iters > 0 ? g->n_items_last : g->n_gitems, s);
}

int gbe_density_preset(const gbe_csr_view* H, const gbe_graph* g, const uint8_t* branch, int32_t iters,
                       int32_t trace_every_iteration, void* workspace, size_t workspace_bytes, void* cuda_stream,
                       double* D_val, gbe_sp2_log* log) {
  if (!g || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  if (iters < 0 || iters > GBE_MAX_ITERS || (iters > 0 && !branch)) return GBE_EINVAL;
  for (int k = 0; k < iters; ++k)
    if (branch[k] > 1) return GBE_EINVAL;
  static const uint8_t none = 0;
  if (!trace_every_iteration && workspace && workspace_bytes < g->ws_bytes && workspace_bytes >= g->ws_bytes_wave_min) {
    GBE_TRY(density_preset_waves(H, g, iters > 0 ? branch : &none, iters, workspace, workspace_bytes, cuda_stream, D_val));
    if (log) GBE_TRY(read_log_at(g, workspace, cuda_stream, log));
    return GBE_OK;
  }
  GBE_TRY(do_gather(H, g, workspace, workspace_bytes, cuda_stream, nullptr));
  GBE_TRY(do_sp2(g, 0.0, iters, -1.0, workspace, workspace_bytes, cuda_stream, nullptr, iters > 0 ? branch : &none,
                 trace_every_iteration != 0));
  GBE_TRY(do_scatter(g, workspace, workspace_bytes, cuda_stream, D_val, nullptr));
  if (log) GBE_TRY(gbe_read_log(g, workspace, workspace_bytes, cuda_stream, log));
  return GBE_OK;
}

int gbe_density_fermi(const gbe_csr_view* H, const gbe_graph* g, double mu, double beta, int32_t order, void* workspace,
                      size_t workspace_bytes, void* cuda_stream, double* D_val, double* n_elec) {
  if (!g || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  if (!(beta > 0.0) || std::isnan(mu) || order < 1 || order > GBE_MAX_ITERS) return GBE_EINVAL;
  if (workspace_bytes < g->ws_bytes_fermi) return GBE_ENOMEM;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  GBE_TRY(do_gather(H, g, workspace, workspace_bytes, cuda_stream, nullptr));  // bounds + X0 into the first buffer
  WS w;
  GBE_TRY(carve(g, workspace, workspace_bytes, &w));
  unsigned char* base = static_cast<unsigned char*>(workspace);
  double* BX = w.X0;
  double* Ta = w.X1;                                             // T_0, then T_2, T_4, ...
  double* Tb = reinterpret_cast<double*>(base + g->ws_x2);       // T_1, then T_3, ...
  double* BD = reinterpret_cast<double*>(base + g->ws_x3);
  GBE_TRY(gbe_launch_cheb_coef(w.st, mu, beta, order, s));
  GBE_TRY(gbe_launch_cheb_init(g, w.st, BX, Ta, Tb, BD, s));
  for (int n = 1; n < order; ++n) {  // T_{n+1} from T_n (B operand) and T_{n-1} (overwritten), coefficient c_{n+1}
    const double* Tn = (n & 1) ? Tb : Ta;
    double* Tio = (n & 1) ? Ta : Tb;
    // the LAST term feeds nothing but D, and D is read at its core columns only: core tiles only (as the last SP2 iteration)
    GBE_TRY(gbe_launch_cheb_step(g, w.st, BX, Tn, Tio, BD, w.st->t1, n + 1, w.partials, s, n == order - 1));
  }
  GBE_TRY(gbe_launch_core_trace(g, BD, w.st, s));
  GBE_TRY(gbe_launch_scatter(g, w.st, BD, BD, D_val, s));
  if (n_elec) {
    GBE_CUDA(cudaMemcpyAsync(n_elec, &w.st->t2[0], 8, cudaMemcpyDeviceToHost, s));
    GBE_CUDA(cudaStreamSynchronize(s));
  }
  return GBE_OK;
}

int gbe_expectation(const gbe_graph* g, const double* D_val, const gbe_csr_view* A, void* cuda_stream, double* out) {
  if (!g || !out || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  GBE_TRY(check_csr(A));
  if (A->n != g->n) return GBE_EMISMATCH;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_set_alloc_stream(s);
  DevBuf rows, res;
  GBE_TRY(rows.alloc((size_t)g->n * 8));
  GBE_TRY(res.alloc(8));
  GBE_TRY(gbe_launch_expectation(g, D_val, *A, rows.as<double>(), res.as<double>(), s));
  GBE_CUDA(cudaMemcpyAsync(out, res.p, 8, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  return GBE_OK;
}

// no allocation, no synchronisation, no gbe_set_alloc_stream (which may touch the pool's attributes): checks + two launches
int gbe_expectation_static(const gbe_graph* g, const double* D_val, const gbe_csr_view* A, void* cuda_stream,
                           double* out_dev) {
  if (!g || !out_dev || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  GBE_TRY(check_csr(A));
  if (A->n != g->n) return GBE_EMISMATCH;
  if (g->n > GBE_STATIC_MAX_N) return GBE_ELIMIT;
  return gbe_launch_expectation_static(g, D_val, *A, out_dev, static_cast<cudaStream_t>(cuda_stream));
}

int gbe_error_norms(const gbe_graph* g, const double* D_val, const double* D_ref, int64_t ld_ref, void* cuda_stream,
                    double* out) {
  if (!g || !out || !D_ref || ld_ref < g->n || (!D_val && g->nnz_D > 0)) return GBE_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_set_alloc_stream(s);
  DevBuf rows, res;
  GBE_TRY(rows.alloc((size_t)g->n * 3 * 8));
  GBE_TRY(res.alloc(3 * 8));
  GBE_TRY(gbe_launch_error_norms(g, D_val, D_ref, ld_ref, rows.as<double>(), res.as<double>(), s));
  GBE_CUDA(cudaMemcpyAsync(out, res.p, 3 * 8, cudaMemcpyDeviceToHost, s));
  GBE_CUDA(cudaStreamSynchronize(s));
  return GBE_OK;
}

int32_t gbe_set_dependent_launch(int32_t on) { return gbe_pdl_set(on != 0); }

int32_t gbe_set_packed_max_m(int32_t m) {
  if (m < 0 || m > GBE_PK_MAX_M) return -1;
  return g_pk_max_m.exchange(m);
}

uint64_t gbe_launch_count(void) { return g_gbe_launches.load(std::memory_order_relaxed); }

int gbe_build_graph_host(const gbe_csr_view* Hh, const gbe_graph_opts* opts, const int32_t* part_host, int32_t n_part,
                         void* cuda_stream, gbe_graph** out) {
  if (!out) return GBE_EINVAL;
  *out = nullptr;
  GBE_TRY(check_csr(Hh));
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_set_alloc_stream(s);
  DevBuf rp, ci, va, pt;
  GBE_TRY(rp.alloc((size_t)(Hh->n + 1) * 8));
  GBE_TRY(ci.alloc((size_t)Hh->nnz * 4));
  GBE_TRY(va.alloc((size_t)Hh->nnz * 8));
  GBE_CUDA(cudaMemcpyAsync(rp.p, Hh->row_ptr, (size_t)(Hh->n + 1) * 8, cudaMemcpyHostToDevice, s));
  if (Hh->nnz) {
    GBE_CUDA(cudaMemcpyAsync(ci.p, Hh->col_idx, (size_t)Hh->nnz * 4, cudaMemcpyHostToDevice, s));
    GBE_CUDA(cudaMemcpyAsync(va.p, Hh->val, (size_t)Hh->nnz * 8, cudaMemcpyHostToDevice, s));
  }
  if (part_host) {
    GBE_TRY(pt.alloc((size_t)Hh->n * 4));
    GBE_CUDA(cudaMemcpyAsync(pt.p, part_host, (size_t)Hh->n * 4, cudaMemcpyHostToDevice, s));
  }
  gbe_csr_view Hd{Hh->n, Hh->nnz, rp.as<int64_t>(), ci.as<int32_t>(), va.as<double>()};
  const int rc = gbe_build_graph(&Hd, opts, part_host ? pt.as<int32_t>() : nullptr, n_part, cuda_stream, out);
  cudaStreamSynchronize(s);  // the staging buffers are freed on return
  if (rc == GBE_OK) {  // the device copy of H stays with the graph: gbe_density_host(H_host = NULL) reuses it
    (*out)->H_n = Hh->n;
    (*out)->H_nnz = Hh->nnz;
    (*out)->H_rp = reinterpret_cast<int64_t*>(rp.release());
    (*out)->H_ci = reinterpret_cast<int32_t*>(ci.release());
    (*out)->H_va = reinterpret_cast<double*>(va.release());
  }
  return rc;
}

int gbe_density_host(const gbe_csr_view* Hh, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                     void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val_host, gbe_sp2_log* log) {
  if (!g || (!D_val_host && g->nnz_D > 0)) return GBE_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  gbe_set_alloc_stream(s);
  DevBuf rp, ci, va, dv;
  GBE_TRY(dv.alloc((size_t)g->nnz_D * 8));
  gbe_csr_view Hd{g->H_n, g->H_nnz, g->H_rp, g->H_ci, g->H_va};
  if (Hh) {
    GBE_TRY(check_csr(Hh));
    if (Hh->n != g->n) return GBE_EMISMATCH;
    GBE_TRY(rp.alloc((size_t)(Hh->n + 1) * 8));
    GBE_TRY(ci.alloc((size_t)Hh->nnz * 4));
    GBE_TRY(va.alloc((size_t)Hh->nnz * 8));
    GBE_CUDA(cudaMemcpyAsync(rp.p, Hh->row_ptr, (size_t)(Hh->n + 1) * 8, cudaMemcpyHostToDevice, s));
    if (Hh->nnz) {
      GBE_CUDA(cudaMemcpyAsync(ci.p, Hh->col_idx, (size_t)Hh->nnz * 4, cudaMemcpyHostToDevice, s));
      GBE_CUDA(cudaMemcpyAsync(va.p, Hh->val, (size_t)Hh->nnz * 8, cudaMemcpyHostToDevice, s));
    }
    Hd = gbe_csr_view{Hh->n, Hh->nnz, rp.as<int64_t>(), ci.as<int32_t>(), va.as<double>()};
  } else if (!g->H_rp) {
    return GBE_EINVAL;  // no H given and the graph was not built by gbe_build_graph_host
  }
  int rc = gbe_density(&Hd, g, n_occ, iters, idem_tol, workspace, workspace_bytes, cuda_stream, dv.as<double>(), log);
  if (rc == GBE_OK && g->nnz_D) {
    cudaError_t e = cudaMemcpyAsync(D_val_host, dv.p, (size_t)g->nnz_D * 8, cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) { gbe_set_cuda_error(e, "cudaMemcpyAsync D", __LINE__); rc = GBE_ECUDA; }
  }
  cudaError_t e = cudaStreamSynchronize(s);  // also keeps the staging buffers alive until the work is done
  if (rc == GBE_OK && e != cudaSuccess) { gbe_set_cuda_error(e, "cudaStreamSynchronize", __LINE__); rc = GBE_ECUDA; }
  return rc;
}

}  // extern "C"
