// Internal declarations shared by the kernels of the hot path (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <vector>

#include "gbe.h"

// ----------------------------------------------------------------------------------------------
// error plumbing
// ----------------------------------------------------------------------------------------------
void gbe_set_cuda_error(cudaError_t e, const char* what, int line);
#define GBE_CUDA(call)                                   \
  do {                                                   \
    cudaError_t e__ = (call);                            \
    if (e__ != cudaSuccess) {                            \
      gbe_set_cuda_error(e__, #call, __LINE__);          \
      return GBE_ECUDA;                                  \
    }                                                    \
  } while (0)
// after every kernel launch: count it (gbe_launch_count) and surface launch errors
extern std::atomic<uint64_t> g_gbe_launches;
#define GBE_LAUNCHED()                                   \
  do {                                                   \
    g_gbe_launches.fetch_add(1, std::memory_order_relaxed); \
    GBE_CUDA(cudaGetLastError());                        \
  } while (0)
#define GBE_TRY(call)          \
  do {                         \
    int s__ = (call);          \
    if (s__ != GBE_OK) return s__; \
  } while (0)

// Device allocations of the library come from the device's default stream-ordered memory pool (cudaMallocAsync) with
// the release threshold lifted, so that the dozens of build-time temporaries cost microseconds instead of a
// cudaMalloc / cudaFree (device synchronisation) each.  The stream is the one of the current API call.
void gbe_set_alloc_stream(cudaStream_t s);
cudaStream_t gbe_alloc_stream();
int gbe_dev_alloc(void** p, size_t bytes);  // on gbe_alloc_stream(); GBE_ENOMEM on failure
void gbe_dev_free(void* p);                 // stream-ordered free on gbe_alloc_stream()

// scoped device allocation for build-time temporaries
struct DevBuf {
  void* p = nullptr;
  DevBuf() = default;
  DevBuf(const DevBuf&) = delete;
  DevBuf& operator=(const DevBuf&) = delete;
  ~DevBuf() { if (p) gbe_dev_free(p); }
  template <typename T> T* as() { return reinterpret_cast<T*>(p); }
  int alloc(size_t bytes) {
    if (p) { gbe_dev_free(p); p = nullptr; }
    return gbe_dev_alloc(&p, bytes ? bytes : 16);
  }
  void* release() { void* q = p; p = nullptr; return q; }
};

// ----------------------------------------------------------------------------------------------
// layout constants
// ----------------------------------------------------------------------------------------------
constexpr int GBE_LD_ALIGN = 16;  // leading dimension of a dense block: m rounded up to 16 doubles (128 B rows)
constexpr int GBE_KC = 16;        // K chunk of the X^2 pipeline (one 128-byte line per row)

// Device-resident state of one gbe_density run: lives at the start of the workspace.
struct gbe_state {
  double eps_min, eps_max;  // Gershgorin bounds of the current H (step 0)
  double n_occ, idem_tol;
  int32_t iters;       // requested iterations
  int32_t iter;        // index n of the X_n the partials currently describe
  int32_t branch;      // branch chosen for iteration `iter` (0: X^2, 1: 2X - X^2)
  int32_t stop;        // 1 once the idempotency stop fired (A-7) or `iters` iterations are done
  int32_t iters_done;  // number of updates applied; the final X lives in buffer iters_done & 1
  int32_t degenerate;  // eps_max == eps_min
  int32_t preset;      // 1: the branch sequence br[] was given by the caller (gbe_density_preset)
  uint32_t bar;        // arrival counter of the resident kernel's grid barrier (reset by k_init_state)
  uint32_t ticket;     // bins of the packed kernel that have published their partial this iteration (gbe_small.cu)
  int32_t inplace;     // 1: the SP2 loop updates X in place in buffer 0 (packed kernel, all communities packed)
  double t1[GBE_MAX_ITERS + 1];
  double t2[GBE_MAX_ITERS + 1];
  uint8_t br[GBE_MAX_ITERS];
};

// packed small communities (gbe_small.cu): one CTA works on a bin of up to GBE_PK_MAX_SLOTS communities per launch
constexpr int GBE_PK_MAX_M = 160;     // largest core + halo size the packed (and the resident) kernel holds in shared memory
constexpr int GBE_PK_MAX_SLOTS = 16;  // communities per bin
struct gbe_pk_slot {  // one community of a bin (40 bytes)
  int32_t p, m, nc, ld;  // community, core + halo size, core size, leading dimension
  int32_t soff;          // offset of its X in the bin's shared memory (doubles)
  int16_t R, pad0_;      // 8-row blocks
  int32_t magic, pad1_;  // floor(2^32 / (ld / 8)) + 1: row of a 16-byte piece of a column quarter by one multiply
  int64_t dense_off;     // element offset of X_p in a dense buffer
};
struct gbe_pk_cta {  // one bin: its communities (its work units sit in the class's code array, [bin][round][warp])
  int32_t n_slots, n_rounds, row0, n_rows;  // n_rounds: longest unit list of a warp; the bin's entries in the row table
  gbe_pk_slot slot[GBE_PK_MAX_SLOTS];
};
struct gbe_pk_row {  // one matrix row of a bin = one TMA bulk copy (16 bytes)
  uint32_t soff;     // byte offset of the row in the bin's shared memory
  uint32_t bytes;    // ld * 8 | slot << 24
  int64_t goff;      // element offset of the row in a dense buffer
};
struct gbe_pk_class {  // the bins of one launch of the packed kernel (device arrays owned by the graph)
  gbe_pk_cta* ctas = nullptr;
  uint16_t* codes = nullptr;
  gbe_pk_row* rows = nullptr;  // all bins, slot 0 of a bin first
  int32_t n_ctas = 0, warps = 0, rounds_max = 0, code_stride = 0;
  size_t smem_bytes = 0;
};

struct gbe_tile_item {  // one X^2 work item: tile (ti, tj), ti <= tj, of community p, with p's layout (32 bytes)
  int32_t pidx, tij, p, m;   // pidx: index of the tile's trace partial (tiles with a core row), else -1; tij = ti | tj << 16;
                             // p: community; m = core + halo size
  int32_t nc, ld;            // core size, leading dimension (m rounded up to 16)
  int64_t dense_off;         // element offset of X_p in a dense buffer
};

struct gbe_wave {  // a range of communities processed together by gbe_density_preset in a bounded workspace (gbe_plan_waves)
  int32_t p0, p1;                  // communities [p0, p1)
  int32_t it_first, it_n;          // its X^2 tiles in items_w
  int32_t last_first, last_n;      // its tiles with a core row in items_last_w
  int32_t gi0, gi_n;               // its gather work items
  int64_t row0, n_rows;            // its dense rows (scatter)
  int64_t base_elems, elems;       // first element and size of its part of a full dense buffer
};

// ----------------------------------------------------------------------------------------------
// the graph handle
// ----------------------------------------------------------------------------------------------
// One work item of the gather (and of the Chebyshev initialisation): rows r0 .. r0 + gather_rows - 1 of community p.  It
// carries what the CTA needs about the community, so that one 32-byte load replaces a chain of dependent ones.
struct __align__(16) gbe_gitem {
  int32_t p, r0, m, nc;     // community, first row, size, core size
  int64_t sb, dense_off;    // offset of the community in sub_idx, and of its block in the dense batch
};

struct gbe_graph {
  int64_t n = 0, nnz_S = 0, sum_m = 0, nnz_D = 0, dense_elems = 0;
  int32_t n_part = 0, max_m = 0, max_ncore = 0, tile = 64;
  double eps_min = 0, eps_max = 0, tau = 0, flops_per_iter = 0, exec_flops_per_iter = 0;
  double flops_last_iter = 0, exec_flops_last_iter = 0;  // the core-tiles-only last iteration
  double sym_flops_per_iter = 0;  // sum m^2 (m + 1): upper triangle incl. diagonal of X_p^2
  int32_t power = 2, contiguous = 1;
  int32_t ncore_all_even = 0;  // every core size is even (the scatter's bulk variant moves 16-byte pieces)
  int32_t scatter_path = 0;    // 0 = the library's choice, 1 = register variant (gbe_graph_set_scatter_path)
  // device arrays (owned)
  int64_t* S_row_ptr = nullptr;  // n+1
  int32_t* S_col = nullptr;      // nnz_S
  int64_t* sub_ptr = nullptr;    // n_part+1
  int32_t* sub_idx = nullptr;    // sum_m: core ascending then halo ascending
  int32_t* ncore = nullptr;      // n_part
  int32_t* msize = nullptr;      // n_part: m_p
  int64_t* dense_off = nullptr;  // n_part+1, element offset of X_p in a dense buffer
  int64_t* D_row_ptr = nullptr;  // n+1
  int32_t* D_col = nullptr;      // nnz_D
  int64_t* scat_base = nullptr;  // sum_m: D.val offset of the run (p, r), contiguous-core case
  int64_t* scat_pos = nullptr;   // nnz_D: D.val offset of (p, r, c), general case (else null)
  int64_t* scat_ofs = nullptr;   // sum_m+1: offset of dense row q in scat_pos (general case)
  int32_t* row_part = nullptr;   // sum_m: community of dense row q
  int64_t* row_src = nullptr;    // sum_m: element offset of dense row q in a dense buffer
  int32_t* row_nc = nullptr;     // sum_m: ncore of the community of dense row q
  // SP2 path: 0 auto, 1 tiled kernels (gbe_x2.cu), 2 resident kernel (gbe_resident.cu), 3 packed kernel for the small
  // communities + tiled kernel for the others (gbe_small.cu); set by gbe_graph_set_sp2_path
  int32_t sp2_path = 0;
  // packed path: bins of communities with m <= GBE_PK_MAX_M, and the tile lists of the OTHER communities
  gbe_pk_class pk[1];
  int32_t n_pk_ctas = 0, pk_n_small = 0, pk_max_m = 0;  // bins; communities in them; threshold of THIS graph
  gbe_tile_item* items_h = nullptr;       // tiles of the communities with m > GBE_PK_MAX_M
  gbe_tile_item* items_last_h = nullptr;  // those with a core row
  int32_t n_items_h = 0, n_items_last_h = 0;
  // gather path: 0 auto, 1 staged (row buffer in shared memory), 2 direct (rows built in global memory); gbe_graph_set_gather_path
  int32_t gather_path = 0;
  int32_t resident_fits = 0, resident_coresident = 0;  // gbe_resident_capacity at build time
  int32_t resident_cluster = 0;  // 1: all communities fit ONE thread-block cluster (<= 16): exchange through DSMEM
  gbe_tile_item* items = nullptr;
  int32_t n_items = 0;
  // the tiles of the LAST SP2 iteration: only those with a core row (row0 < ncore_p); they hold, directly or through
  // the mirrored store, every core row and core column of X_p - all that the trace and the scatter read (Eq.(6))
  gbe_tile_item* items_last = nullptr;
  int32_t n_items_last = 0;
  gbe_gitem* gitems = nullptr;  // gather work items (community, first row, and the community's sizes and offsets)
  int32_t n_gitems = 0, gather_rows = 0;
  // device copy of the H uploaded by gbe_build_graph_host (owned; null for graphs built from device pointers)
  int64_t H_n = 0, H_nnz = 0;
  int64_t* H_rp = nullptr;
  int32_t* H_ci = nullptr;
  double* H_va = nullptr;
  // tensor maps of the X^2 TMA variant (gbe_x2.cu), cached for the pair of dense buffers they were encoded for
  void* tmaps = nullptr;  // 2 n_part CUtensorMap: [buffer][community]; null: no encoder in the driver, cp.async kernel
  // wave plan of gbe_density_preset in a bounded workspace, cached for the capacity it was made for (not thread safe)
  mutable std::vector<gbe_wave> waves;
  mutable size_t waves_cap = 0;
  mutable gbe_tile_item *items_w = nullptr, *items_last_w = nullptr;
  size_t ws_bytes_wave_min = 0;  // state + partials + two buffers of the largest community
  // workspace layout (byte offsets)
  size_t ws_partials = 0, ws_bounds = 0, ws_x0 = 0, ws_x1 = 0, ws_bytes = 0;
  size_t ws_x2 = 0, ws_x3 = 0, ws_bytes_fermi = 0;  // two more dense buffers for the Chebyshev recurrence
  int32_t n_partials = 0;
  // host mirrors
  std::vector<int32_t> h_m, h_ncore;
  std::vector<int64_t> h_dense_off;
};

// ----------------------------------------------------------------------------------------------
// programmatic dependent launch (sm_90+): a kernel launched with the stream-serialisation attribute may become resident
// once every CTA of the previous kernel of the stream has executed griddepcontrol.launch_dependents (or exited); it must
// execute griddepcontrol.wait before it touches anything the previous kernel (or, transitively, an earlier one that the
// previous kernel itself did not wait for) produces.  Without the attribute both instructions are no-ops.
//   GBE_PDL_TOP    the kernel waits at its top, before it reads anything a launch produces (safe behind any kernel):
//                  k_trace_branch, k_sp2_packed
//   GBE_PDL_EARLY  X^2 kernel behind k_trace_branch only: it never waits.  k_trace_branch waits for the previous X^2
//                  launch, decides, fences and only then lets its dependents go, so everything this grid reads is final
//                  when it starts
// ----------------------------------------------------------------------------------------------
enum { GBE_PDL_NONE = 0, GBE_PDL_TOP = 1, GBE_PDL_EARLY = 2 };
bool gbe_pdl_enabled();   // the process-wide switch (gbe_util.cu; gbe_set_dependent_launch, GBE_PDL=0)
int gbe_pdl_set(int on);  // returns the previous setting
#ifdef __CUDACC__
__device__ __forceinline__ void gbe_griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void gbe_griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
// state words another kernel may be writing while this one runs, or has written since this one started: never cached
// in L1, never merged with an earlier read by the compiler
__device__ __forceinline__ int gbe_ld_state(const int32_t* p) {
  int v;
  asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int gbe_ld_acquire(const int32_t* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int gbe_ld_state(const uint8_t* p) {
  int v;
  asm volatile("ld.global.cg.u8 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
template <typename... KArgs, typename... Args>
inline cudaError_t gbe_launch_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl,
                                     Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}
#endif

// ----------------------------------------------------------------------------------------------
// kernel launchers (each file holds one step of DESIGN.md section 1)
// ----------------------------------------------------------------------------------------------
// step 0
int gbe_launch_bounds(const gbe_csr_view& H, double* block_lo, double* block_hi, int max_blocks, gbe_state* st,
                      cudaStream_t s);
// step 1
// S is sized exactly (*nnz_S entries)
int gbe_build_pattern(const gbe_csr_view& H, const gbe_state* st_dev, double tau, int power, int check_sym,
                      cudaStream_t s, int64_t** S_row_ptr, int32_t** S_col, int64_t* nnz_S);
// Eq.(8): S for the next MD step from the previous D and the new H
int gbe_build_pattern_eq8(const gbe_csr_view& H, const int64_t* D_rp, const int32_t* D_col, const double* D_val, double tau,
                          cudaStream_t s, int64_t** S_row_ptr, int32_t** S_col, int64_t* nnz_S, int64_t nnz_D);
// step 2
// bounds: pinned host copy of (eps_min, eps_max) of step 0, in flight on `s`: looked at after the first synchronisation
int gbe_build_subgraphs(gbe_graph* g, const int32_t* part, cudaStream_t s, const double* bounds);
// step 3
int gbe_launch_gather(const gbe_csr_view& H, const gbe_graph* g, const gbe_state* st, double* X, double* partials,
                      cudaStream_t s, int item0 = 0, int n_it = -1);
// step 4
// iter: index n of the update X_n -> X_{n+1} (selects br[n] when the sequence is preset)
// hybrid: only the tiles of the communities the packed kernel does not take (items_h / items_last_h)
// buffer: which dense buffer Xin is (0 or 1: selects the tensor maps)
// pdl: programmatic dependent launch (GBE_PDL_*): the grid may become resident before the previous kernel of the stream
// has finished and synchronises with it in the kernel
// hyb: the launch runs NEXT TO the packed launch of the same iteration (mixed graphs, gbe_api.cu): its CTAs wait at their
// top until that launch has published the branch of the iteration, and at their end until it has completed
int gbe_launch_x2(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                  bool last, bool hybrid, int buffer, cudaStream_t s, int pdl = 0, bool hyb = false);
int gbe_launch_x2_items(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials, int iter,
                        const gbe_tile_item* items, int n_items, int buffer, cudaStream_t s, int pdl = 0, bool hyb = false);
int gbe_plan_waves(const gbe_graph* g, size_t cap_elems, cudaStream_t s);  // gbe_halo.cu
int gbe_x2_build_tmaps(gbe_graph* g, cudaStream_t s);                                        // once per graph
int gbe_x2_prepare(const gbe_graph* g, const double* X0, const double* X1, cudaStream_t s);  // once per density call
// steps 4 + 5 in one kernel for small communities (gbe_resident.cu); mode as in k_init_state
int gbe_resident_capacity(const gbe_graph* g, int* fits, int* coresident, int* cluster);
constexpr int GBE_RESIDENT_UNAVAILABLE = 1;  // internal: the cooperative / cluster launch does not fit the device right now
int gbe_launch_sp2_resident(const gbe_graph* g, gbe_state* st, double* X0, double* X1, double* partials, int mode,
                            cudaStream_t s);
// steps 4 + 5, one iteration per launch, for communities with m <= g->pk_max_m (gbe_small.cu)
int gbe_packed_max_m();  // process-wide default of the threshold (gbe_set_packed_max_m)
int gbe_build_packed(gbe_graph* g, cudaStream_t s);
// fused: 0 no step 5 in the kernel; 1 ticket (last bin decides); 2 lazy (the bins of the NEXT launch sum the lazy_n pairs
// at partials[lazy_base ...] themselves: pass the previous launch's base and count, 0 for the first launch)
int gbe_launch_sp2_packed(const gbe_graph* g, gbe_state* st, const double* Xin, double* Xout, double* partials,
                          int partial_base, int n_partials, int iter, bool last, int fused, int lazy_base, int lazy_n,
                          cudaStream_t s);
// step 5
int gbe_launch_trace_branch(gbe_state* st, const double* partials, int n_partials, cudaStream_t s, int pdl = 0);
// step 6
int gbe_launch_scatter(const gbe_graph* g, const gbe_state* st, const double* X0, const double* X1, double* D_val,
                       cudaStream_t s, int64_t row0 = 0, int64_t n_rows = -1);

// finite-temperature Chebyshev expansion (gbe_fermi.cu; the product of every term is gbe_x2.cu in its second mode)
int gbe_launch_cheb_coef(gbe_state* st, double mu, double beta, int order, cudaStream_t s);
int gbe_launch_cheb_init(const gbe_graph* g, const gbe_state* st, double* BX, double* B0, double* B1, double* BD,
                         cudaStream_t s);
int gbe_launch_cheb_step(const gbe_graph* g, gbe_state* st, const double* Xt, const double* Tn, double* Tio, double* Dacc,
                         const double* coef, int iter, double* partials, cudaStream_t s, bool last = false);
int gbe_launch_core_trace(const gbe_graph* g, const double* BD, gbe_state* st, cudaStream_t s);
// observables (gbe_observe.cu)
int gbe_launch_expectation(const gbe_graph* g, const double* D_val, const gbe_csr_view& A, double* row_sum, double* out,
                           cudaStream_t s);

// the same with the row partials in a static device array of GBE_STATIC_MAX_N doubles: allocates nothing (gbe_observe.cu)
int gbe_launch_expectation_static(const gbe_graph* g, const double* D_val, const gbe_csr_view& A, double* out_dev,
                                  cudaStream_t s);
int gbe_launch_error_norms(const gbe_graph* g, const double* D_val, const double* D_ref, int64_t ld_ref, double* row_out,
                           double* out, cudaStream_t s);

// small device utilities (gbe_util.cu)
int32_t* gbe_pinned_words();  // 64 pinned host words per thread, or null
int gbe_sm_count();           // multiprocessors of the CURRENT device (cached per device)
// one-time set-up per DEVICE (function attributes, pool thresholds): first() is true once per device for this object
struct gbe_device_once {
  std::atomic<uint64_t> mask[4] = {};
  bool first();
};
int gbe_exclusive_scan_i32_to_i64(const int32_t* in, int64_t* out, int64_t n, cudaStream_t s);
int gbe_exclusive_scan_i32_to_i64_max(const int32_t* in, int64_t* out, int64_t n, cudaStream_t s);

// ----------------------------------------------------------------------------------------------
// device helpers
// ----------------------------------------------------------------------------------------------
#ifdef __CUDACC__
// Step 5's decision (A-6, A-7), taken by ONE thread from the global traces t1, t2 of X_k, k = st->iter: the log entry,
// the idempotency stop, the branch of iteration k (preset or chosen).  Shared by k_trace_branch and by the kernels that
// reduce the traces themselves.
// what gbe_trace_decide reads from the state; none of it is written by an X^2 launch, so k_trace_branch loads it BEFORE it
// waits for the launch that writes the partials
struct gbe_decide_in {
  double n_occ, idem_tol;
  int k, iters, preset, brk;
};
__device__ __forceinline__ gbe_decide_in gbe_trace_decide_load(const gbe_state* st) {
  // (loads that bypass L1: the CTA may have become resident, under a programmatic dependent launch, on an SM whose L1
  //  still holds a line of the state from an earlier launch)
  gbe_decide_in d;
  d.n_occ = __ldcg(&st->n_occ);
  d.idem_tol = __ldcg(&st->idem_tol);
  d.k = __ldcg(&st->iter);  // the partials describe X_k
  d.iters = __ldcg(&st->iters);
  d.preset = __ldcg(&st->preset);
  d.brk = d.k < GBE_MAX_ITERS ? (int)__ldcg(&st->br[d.k]) : 0;
  return d;
}
__device__ __forceinline__ void gbe_trace_decide(gbe_state* st, double t1, double t2, const gbe_decide_in& d) {
  const int k = d.k;
  st->t1[k] = t1;
  st->t2[k] = t2;
  st->iters_done = k;
  if (k >= d.iters || (d.idem_tol >= 0.0 && k >= 1 && fabs(t1 - t2) <= d.idem_tol)) {
    st->stop = 1;
  } else {
    const int b = d.preset ? d.brk : ((fabs(t2 - d.n_occ) < fabs(2.0 * t1 - t2 - d.n_occ)) ? 0 : 1);
    st->branch = b;
    st->br[k] = (uint8_t)b;
    __threadfence();
    st->iter = k + 1;
  }
}
__device__ __forceinline__ void gbe_trace_decide(gbe_state* st, double t1, double t2) {
  const double n_occ = st->n_occ;
  const int k = st->iter;  // the partials describe X_k
  st->t1[k] = t1;
  st->t2[k] = t2;
  st->iters_done = k;
  if (k >= st->iters || (st->idem_tol >= 0.0 && k >= 1 && fabs(t1 - t2) <= st->idem_tol)) {
    st->stop = 1;
  } else {
    const int b = st->preset ? (int)st->br[k] : ((fabs(t2 - n_occ) < fabs(2.0 * t1 - t2 - n_occ)) ? 0 : 1);
    st->branch = b;
    st->br[k] = (uint8_t)b;
    __threadfence();   // iter == k + 1 PUBLISHES the branch of iteration k: the tiled kernel of a mixed graph runs next to
    st->iter = k + 1;  // the packed kernel that decides and reads iter with acquire (gbe_x2.cu, hyb)
  }
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int warp_sum_i(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int warp_excl_scan_i(int v, int lane, int* total) {
  int x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  *total = __shfl_sync(0xffffffffu, x, 31);
  return x - v;
}
#endif
