/*
 * gbe.h - C ABI of the B200-native graph-based electronic-structure hot path
 *         (arXiv:1603.00937, "Graph-based linear scaling electronic structure theory").
 *
 * What the library computes (citations: P:Lnn = line nn of the paper text; A-n = reading n in DESIGN.md 3):
 *
 *   P_tau(H): the thresholded matrix polynomial of Eq.(4), evaluated by the partitioned
 *   subgraph expansion of Eq.(6) P:L58-63.  For every community p (obs. (vi) P:L65) the core vertices and
 *   all halo vertices directly connected to them in the data-dependency graph S_tau (Eq.(2) P:L38-40,
 *   Fig.1) induce a dense principal submatrix x[s_p].  The polynomial is the recursive
 *   second-order zero-temperature Fermi-operator expansion ("SP2"):
 *   X <- X^2 or 2X - X^2, the SAME sequence for every subgraph ("the same for each subgraph expansion",
 *   P:L90), chosen on the device from the trace summed over all core diagonals.  The core columns are
 *   collected into the sparse, non-symmetric density matrix D = P_tau(H) (obs. (i) P:L65).
 *
 * Conventions
 *   - All functions return 0 (GBE_OK) or a negative gbe_status.  No exceptions, no aborts, no stdout.
 *   - "device" pointers are CUDA device memory of the current device; "host" pointers are ordinary host
 *     memory.  Inputs are borrowed for the duration of the call (device inputs: until the work enqueued on
 *     `cuda_stream` has finished); the library never frees caller memory.  Outputs and the workspace are
 *     caller-allocated; the only library allocation is the graph handle (freed by gbe_free_graph).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - gbe_build_graph synchronises the stream (it sizes its outputs).  gbe_density and the three phase calls
 *     only enqueue work: no host round trip between SP2 iterations; they return before completion.
 *   - CSR: row_ptr int64 [n+1], col_idx int32 [nnz] ascending within a row, val double [nnz]; 0-based.
 *   - Devices and threads.  Every call works on the CURRENT device of the calling thread (cudaSetDevice); a graph, its
 *     workspace and the buffers passed with it belong to the device that was current when the graph was built.  One-time
 *     set-up (kernel attributes, memory-pool thresholds) is kept per device.  Calls from different host threads are safe as
 *     long as they do not share a graph handle, a workspace or an output buffer; the process-wide knobs
 *     (gbe_set_build_scratch_limit, gbe_set_packed_max_m) are atomic but apply to graphs built afterwards.
 */
#ifndef GBE_H
#define GBE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GBE_OK = 0,
  GBE_EINVAL = -1,      /* null pointer, n <= 0, tau < 0 or NaN, n_occ outside [0,n], iters outside [0,GBE_MAX_ITERS],
                           partition id out of range, power outside [1,GBE_MAX_POWER], n above the supported size
                           (the index maps of steps 1-3 are bitmaps over the n vertices in shared memory: about
                           4e5 orbitals with core+halo sizes up to a few thousand) */
  GBE_ENOTSYM = -2,     /* H is not symmetric (pattern or values); only tested when opts.check_symmetry != 0 */
  GBE_EDEGENERATE = -3, /* eps_max == eps_min: the spectrum cannot be mapped to [0,1] (A-12).  gbe_build_graph returns it;
                           the density calls only enqueue work, so for THEIR H it is reported by gbe_read_log (hence by a
                           call with log != NULL) - without a log they return GBE_OK and D holds the finite values of
                           X0 = (eps_max I - H) / 1 carried through the same updates */
  GBE_EMISMATCH = -4,   /* H.n differs from the graph's n */
  GBE_ENOMEM = -5,      /* workspace too small (required size: gbe_graph_info.workspace_bytes) or allocation failed */
  GBE_ECUDA = -6,       /* a CUDA call failed; text via gbe_strerror / gbe_last_cuda_error */
  GBE_ELIMIT = -7       /* the problem is larger than a fixed limit of the entry point (gbe_expectation_static:
                           n > GBE_STATIC_MAX_N); nothing was launched */
} gbe_status;

#define GBE_MAX_ITERS 1024
#define GBE_MAX_POWER 8

/* Sparse symmetric matrix in CSR (the Hamiltonian H).  DEVICE pointers, borrowed. */
typedef struct {
  int64_t n;
  int64_t nnz;
  const int64_t* row_ptr; /* n+1 */
  const int32_t* col_idx; /* nnz, ascending within a row */
  const double* val;      /* nnz */
} gbe_csr_view;

/* Opaque, library-owned, immutable after gbe_build_graph: S_tau, the communities, their core+halo index
 * lists, the padded batched dense layout, the pattern of D and the scatter map, the tile work list. */
typedef struct gbe_graph gbe_graph;

typedef struct {
  double tau;             /* threshold of Eq.(2), applied to magnitudes (A-3), on the normalised X0 (A-1) */
  int32_t power;          /* highest thresholded power T^(n) entering S_tau (A-1); 0 -> default 2 */
  int32_t check_symmetry; /* != 0: verify H == H^T (pattern and values) and fail with GBE_ENOTSYM otherwise */
} gbe_graph_opts;

typedef struct {
  int64_t n;          /* vertices = orbitals = rows of H */
  int64_t nnz_S;      /* edges of S_tau incl. self loops (directed count) */
  int64_t n_part;     /* communities */
  int64_t sum_m;      /* sum over communities of m_p = core + halo size */
  int64_t max_m;      /* largest m_p */
  int64_t nnz_D;      /* stored entries of D = sum_p m_p * ncore_p */
  int64_t dense_elems;/* doubles in ONE batched dense buffer = sum_p m_p * ld_p (ld_p = m_p rounded up to 16) */
  int64_t n_tiles;    /* X^2 work items per SP2 iteration (upper-triangle tiles over all communities) */
  double sp2_flops_per_iter; /* sum_p 2 m_p^3: algorithmic flops of one SP2 iteration (unpadded, no symmetry) */
  double sp2_exec_flops_per_iter; /* flops the X^2 kernel issues to the FP64 tensor pipe per iteration: the 8 x 8
                                     sub-tiles on or above the diagonal only (X is symmetric), K padded to ld_p */
  int64_t n_tiles_last;      /* work items of the LAST SP2 iteration: the tiles with a core row only (the trace and
                                the scatter read nothing else of the final X_p, Eq.(6)) */
  double sp2_flops_last_iter;      /* sum_p 2 m_p^2 ncore_p: algorithmic flops of the last iteration (core columns) */
  double sp2_exec_flops_last_iter; /* flops issued to the FP64 tensor pipe by the last iteration */
  double eps_min, eps_max;   /* Gershgorin bounds of the H given to gbe_build_graph (A-5) */
  int32_t contiguous_cores;  /* 1: every core is a contiguous index range (fast scatter); 0: per-entry map */
  int32_t tile;              /* edge of the square X^2 tile chosen for this graph */
  size_t workspace_bytes;    /* device workspace gbe_density needs (two dense buffers + state + partials) */
  size_t workspace_bytes_fermi; /* device workspace gbe_density_fermi needs (four dense buffers + state + partials) */
  int32_t resident_sp2;      /* 1: gbe_density will run the SP2 loop of this graph in the shared-memory-resident kernel */
  int32_t resident_fits;     /* 1: the largest community fits that kernel (max_m <= 160); see gbe_graph_set_sp2_path */
  int32_t resident_cluster;  /* 1: all communities fit ONE thread-block cluster (n_part <= 16): the resident kernel then
                                exchanges the traces through distributed shared memory and the cluster barrier */
  int32_t sp2_path_chosen;   /* the kernels gbe_density will run for steps 4-5 of this graph: 1 tiled, 2 resident, 3 packed */
  double sp2_sym_flops_per_iter; /* sum_p m_p^2 (m_p + 1): the flops of one SP2 iteration the METHOD needs when the symmetry
                                    of X_p is used (only the entries on or above the diagonal of X_p^2 are formed; obs. (x)
                                    P:L65) - the numerator of bench.py's roofline fraction */
  int64_t n_small;           /* communities with 0 < m_p <= 160 (gbe_set_packed_max_m): the ones the packed kernel takes */
  int64_t n_bins;            /* CTAs of one packed launch (bins of 1..16 small communities) */
  size_t workspace_bytes_preset_min; /* smallest workspace gbe_density_preset(trace_every_iteration = 0) accepts: it then
                                        works through the communities in waves (see there) */
  int32_t x2_tma;            /* 1: the tiled X^2 kernel of this graph stages its panels by 2-D TMA (tensor maps; long K loops),
                                0: by cp.async (short K loops, or no tensor-map encoder in the driver) */
  int32_t reserved2_;
} gbe_graph_info;

/* SP2 log (host memory, caller-allocated; valid after the stream has been synchronised).
 * t1[k] = sum_p sum_{i<ncore_p} (X_k)_ii, t2[k] = same for X_k^2, k = 0..iters_done;
 * branch[k] = 0 (X <- X^2) or 1 (X <- 2X - X^2), k = 0..iters_done-1 (A-6). */
typedef struct {
  int32_t iters_done;
  uint8_t* branch; /* >= iters entries */
  double* t1;      /* >= iters + 1 entries */
  double* t2;      /* >= iters + 1 entries */
} gbe_sp2_log;

/* Steps 0-2 of the path: Gershgorin bounds of H, the graph
 *     S_tau = I u pat(A) u pat(floor(A A)_tau) [u ... up to `power`], A = floor((eps_max I - H)/(eps_max-eps_min))_tau,
 * symmetrised (reading A-1 of Eq.(2) P:L38-40 / Eq.(8)), then for every community p its subgraph
 *     s_p = C_p u { k : (k,i) in S_tau, i in C_p }            (local order: core ascending, halo ascending)
 * and the pattern S' of D (A-9).
 *   H     device CSR, SYMMETRIC.  With the default power 2 the library forms only the upper triangle of the
 *         thresholded product A A (bit for bit symmetric when A is) and symmetrises the pattern; a non-symmetric H
 *         gives the graph of that upper triangle.  opts.check_symmetry verifies the premise.
 *   part  device int32[n], vertex -> community id in [0, n_part); every vertex lies in exactly one core;
 *         empty communities are allowed.  NULL: contiguous blocks of ceil(n / n_part) rows.
 *         (The paper's partitioner, METIS P:L78, is outside the library.)
 *   out   receives the handle.  Synchronises `cuda_stream`. */
int gbe_build_graph(const gbe_csr_view* H, const gbe_graph_opts* opts, const int32_t* part, int32_t n_part,
                    void* cuda_stream, gbe_graph** out);

/* The graph for the NEXT molecular-dynamics step, Eq.(8) P:L84-88:
 *     S_tau(t) <- floor( ( floor(D(t - dt))_tau + H(t) )^2 )_eps
 * in the symbolic form the paper uses (eps = 0): M = I u pat(|D_ij| >= tau) u pat(H(t)), S = pattern of M M ("paths of
 * length two"), symmetrised.  Steps 0 and 2 (bounds of H(t), halos, pattern of the new D) as gbe_build_graph.
 *   prev    the graph D_prev was computed on (gives D's CSR pattern); not modified, still to be freed by the caller.
 *   D_prev  device double[prev nnz_D]: D(t - dt) as written by gbe_density.
 *   H       device CSR of H(t); opts->tau is the threshold applied to D (the paper uses 1e-4); opts->power is ignored.
 *   part / n_part as gbe_build_graph (may differ from prev's).  Synchronises `cuda_stream`. */
int gbe_update_graph(const gbe_graph* prev, const double* D_prev, const gbe_csr_view* H, const gbe_graph_opts* opts,
                     const int32_t* part, int32_t n_part, void* cuda_stream, gbe_graph** out);

int gbe_graph_get_info(const gbe_graph* g, gbe_graph_info* out);

/* Copies the graph to caller-allocated DEVICE buffers (any may be NULL to skip), sizes from gbe_graph_info:
 * S_row_ptr[n+1], S_col[nnz_S], sub_ptr[n_part+1], sub_idx[sum_m], ncore[n_part], D_row_ptr[n+1], D_col[nnz_D]. */
int gbe_graph_export(const gbe_graph* g, void* cuda_stream, int64_t* S_row_ptr, int32_t* S_col, int64_t* sub_ptr,
                     int32_t* sub_idx, int32_t* ncore, int64_t* D_row_ptr, int32_t* D_col);

/* Which kernels run the SP2 loop (steps 4-5) of this graph.  Three implementations compute the same updates:
 *   tiled    (any size)  one X^2 launch + one trace/branch launch per iteration over the batched dense layout in HBM;
 *   packed   (communities with m_p <= 160 [gbe_set_packed_max_m], any number of them; the cost law P:L78 - more partitions, smaller m)
 *            one launch per iteration: a CTA copies a bin of 1..16 whole matrices to shared memory, squares them on the
 *            FP64 tensor cores, writes them back and leaves one trace pair; the bins of the NEXT launch sum those pairs
 *            (the same fixed order in every bin) and take the branch decision themselves, so there is no separate
 *            trace/branch launch between iterations (one after the last).  Larger communities of the same graph go
 *            through the tiled kernel in the same iteration, launched next to the bins;
 *   resident (max_m <= 160) ONE launch for the whole loop, X_p held in shared memory by one CTA per community; the
 *            global trace (one sequence for all subgraphs) is exchanged through a grid barrier, which needs all
 *            communities co-resident (cooperative launch; one thread-block cluster with the exchange in distributed
 *            shared memory when there are at most 16 communities) - unless the sequence is preset and no trace is logged
 *            (gbe_density_preset with trace_every_iteration = 0), where the CTAs never communicate.
 * path = 0 (default): resident when it applies and all communities fit the device at once; else packed when the graph
 *        has enough small communities to occupy the device and at most a few larger ones; else tiled;
 *        1: always tiled;  2: resident whenever it can run (GBE_EINVAL if max_m is too large; calls for which the
 *        communities are not co-resident still take the tiled kernels);  3: packed whenever the graph has a community
 *        small enough (else tiled).
 * Results of the paths agree to rounding (different summation order of the global trace), each is bitwise
 * reproducible.  Not thread safe against concurrent calls on the same graph. */
int gbe_graph_set_sp2_path(gbe_graph* g, int32_t path);

/* Which kernel packs the dense blocks (step 3).  Two variants compute the same x_p = X0[s_p, s_p]:
 *   staged  each warp builds an output row in a shared-memory row buffer and streams it out once;
 *   direct  the row is zero-filled and the stored entries are stored straight to global memory (no row buffer: for
 *           large systems, where the index bitmaps over the n vertices and row buffers of max_m doubles would leave one
 *           CTA per SM).
 * path = 0 (default): staged while three CTAs with their row buffers fit an SM, else direct; 1: staged; 2: direct.
 * The dense blocks of the two are bit-identical; the traces of X_0 are summed in a different order (agree to rounding). */
int gbe_graph_set_gather_path(gbe_graph* g, int32_t path);

/* Which kernel moves the core columns into D (step 6).  Two variants copy the same runs:
 *   register  a warp moves 8 runs per iteration through registers (any core sizes, any partition vector);
 *   bulk      the copy engine moves the runs global -> shared -> global (cp.async.bulk), 32 per warp in flight; needs
 *             index-range cores of even size and a 16-byte aligned D_val (every run is then a whole number of 16-byte
 *             pieces on both sides).
 * path = 0 (default): bulk where its conditions hold, else register; 1: register.  D is bit-identical. */
int gbe_graph_set_scatter_path(gbe_graph* g, int32_t path);

/* Steps 0 and 3-6: D = P_tau(H) on the pattern fixed by the graph (Eq.(6)).
 *   H         device CSR; values AND pattern may differ from the H the graph was built from (MD use):
 *             H values are looked up at gather time, entries outside a subgraph are simply not gathered.
 *             The Gershgorin bounds are recomputed from this H.
 *   n_occ     target occupation (number of occupied orbitals), 0 <= n_occ <= n.
 *   iters     SP2 iterations (fixed count when idem_tol < 0).  Iteration iters - 1 computes only the tiles of X_p that
 *             hold a core row or core column: nothing else of the final X_p is read (Eq.(6) P:L58-63 keeps the core
 *             columns), so after the call the rest of the dense buffers in the workspace is stale scratch.
 *   idem_tol  >= 0: stop before iteration k >= 1 once |t1[k] - t2[k]| <= idem_tol (A-7); < 0: never stop early.
 *   workspace device memory, >= info.workspace_bytes, 256-byte aligned; contents are scratch.
 *   D_val     device double[nnz_D], CSR order of (D_row_ptr, D_col); entry (k,i) is taken from the expansion of
 *             the community that owns column i.  NOT symmetric (obs. (i) P:L65); not symmetrised.
 *   log       optional host log.  With log != NULL the call SYNCHRONISES the stream (twice: the header of the log sizes the
 *             copy of its arrays) and is therefore not capturable in a CUDA graph; with log == NULL it only enqueues
 *             (gbe_read_log fetches the log of the last run later). */
int gbe_density(const gbe_csr_view* H, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val, gbe_sp2_log* log);

/* The three phases of gbe_density as separate calls (same arguments, same kernels, same stream semantics);
 * gbe_density == gbe_gather; gbe_sp2; gbe_scatter.  They exist so that a caller can time the phases. */
int gbe_gather(const gbe_csr_view* H, const gbe_graph* g, void* workspace, size_t workspace_bytes,
               void* cuda_stream);   /* steps 0, 3: bounds, pack x[s_p] = X0[s_p,s_p], traces of X_0 */
int gbe_sp2(const gbe_graph* g, double n_occ, int32_t iters, double idem_tol, void* workspace,
            size_t workspace_bytes, void* cuda_stream);   /* steps 4-5, `iters` times */
int gbe_scatter(const gbe_graph* g, void* workspace, size_t workspace_bytes, void* cuda_stream,
                double* D_val);       /* step 6 */
int gbe_read_log(const gbe_graph* g, const void* workspace, size_t workspace_bytes, void* cuda_stream,
                 gbe_sp2_log* log);   /* enqueue the device->host copy of the log of the last gbe_sp2 */

/* Same as gbe_density with HOST buffers: H (row_ptr, col_idx, val) and D_val are host pointers; the call
 * copies H to the device, runs the path, copies D back and synchronises the stream before returning.
 * H_host == NULL: use the device copy of H that gbe_build_graph_host left with the graph (one upload for
 * build + density of the same H); GBE_EINVAL if the graph was built from device pointers.
 * `workspace` stays a device buffer of info.workspace_bytes. */
int gbe_density_host(const gbe_csr_view* H_host, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                     void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val_host,
                     gbe_sp2_log* log);

/* gbe_build_graph with HOST buffers: H (row_ptr, col_idx, val) and part (may be NULL) are host pointers; the call
 * copies them to the device and builds the graph.  The device copy of H stays with the graph (freed by
 * gbe_free_graph) so that gbe_density_host(H_host = NULL) can reuse it. */
int gbe_build_graph_host(const gbe_csr_view* H_host, const gbe_graph_opts* opts, const int32_t* part_host,
                         int32_t n_part, void* cuda_stream, gbe_graph** out);

/* Device time of the kernels of one gbe_density run, measured with CUDA events recorded on `cuda_stream` around
 * every launch (milliseconds; *_launches = kernel launches summed into the field before it). */
typedef struct {
  float bounds_ms;  int32_t bounds_launches;   /* step 0 */
  float gather_ms;  int32_t gather_launches;   /* step 3 */
  float x2_ms;      int32_t x2_launches;       /* step 4: the X^2 / 2X - X^2 kernel, one launch per SP2 iteration
                                                  (all but the last iteration) */
  float trace_ms;   int32_t trace_launches;    /* step 5 (+ the state initialisation kernel) */
  float scatter_ms; int32_t scatter_launches;  /* step 6 */
  float total_ms;                              /* first launch to last launch, on the stream */
  float x2_last_ms; int32_t x2_last_launches;  /* step 4, last iteration: the tiles with a core row only */
} gbe_phase_times;

/* gbe_density with the same kernels and the same launch sequence, plus one event pair per launch; synchronises
 * the stream before returning.  For measurement only: the events serialise nothing but cost a few us each. */
int gbe_density_timed(const gbe_csr_view* H, const gbe_graph* g, double n_occ, int32_t iters, double idem_tol,
                      void* workspace, size_t workspace_bytes, void* cuda_stream, double* D_val, gbe_sp2_log* log,
                      gbe_phase_times* times);

/* gbe_density with a PRE-DETERMINED SP2 sequence ("the complete SP2 sequence (the same for each subgraph
 * expansion) ... determined beforehand", e.g. from the previous MD step): iteration k applies X <- X^2 if branch[k] == 0,
 * X <- 2X - X^2 if branch[k] == 1, for every community.  No decision is taken on the device.
 *   branch   HOST array of `iters` bytes, each 0 or 1 (read before the call returns).
 *   trace_every_iteration != 0: the global traces t1[k], t2[k] are still reduced and logged every iteration;
 *                         == 0: no per-iteration reduction kernel at all ("without exchange of information during or
 *                               between the matrix multiplications"); the log then holds only t1, t2 of the
 *                               final X at index `iters` (earlier entries are unspecified) and the given branches.
 * Bounded workspace.  With trace_every_iteration == 0 nothing couples the communities, so the call also accepts a
 * workspace SMALLER than info.workspace_bytes, down to info.workspace_bytes_preset_min (room for the largest community):
 * it then gathers, expands and scatters the communities in waves that fit the workspace given - the same kernels on the
 * same tiles, D bit for bit the same; the memory of the dense batch no longer grows with the system (config 4 of
 * BASELINE.json: 2 x 20 GB at once, or waves in a few GB).
 * Other arguments, stream semantics and D_val as gbe_density. */
int gbe_density_preset(const gbe_csr_view* H, const gbe_graph* g, const uint8_t* branch, int32_t iters,
                       int32_t trace_every_iteration, void* workspace, size_t workspace_bytes, void* cuda_stream,
                       double* D_val, gbe_sp2_log* log);

/* Finite-temperature density matrix by the Chebyshev Fermi-operator expansion, Eq.(7) P:L67-72:
 *     D = [e^{beta (H - mu)} + 1]^{-1}  ~  sum_{n=0}^{order} c_n T_n((H - b)/a)
 * evaluated per community on x[s_p] (Eq.(6)) with the three-term recurrence T_{n+1} = 2 Ht T_n - T_{n-1}
 * (Eq.(5)), one dense product per term; a, b from the Gershgorin bounds of H, c_n by Chebyshev-Gauss
 * quadrature of the Fermi function (2048 nodes), all on the device.  Gather and scatter as gbe_density.
 *   mu, beta   chemical potential and inverse temperature, in the units of H (beta > 0).
 *   order      highest Chebyshev order, 1 <= order <= GBE_MAX_ITERS.
 *   workspace  >= info.workspace_bytes_fermi.
 *   n_elec     optional HOST double: sum over all core diagonals of D (the occupation); if given, the call
 *              synchronises the stream, otherwise it only enqueues. */
int gbe_density_fermi(const gbe_csr_view* H, const gbe_graph* g, double mu, double beta, int32_t order, void* workspace,
                      size_t workspace_bytes, void* cuda_stream, double* D_val, double* n_elec);

/* Expectation value <A> = Tr[D A] = sum_{k,i} D_ki A_ik; with A = H the band energy E_band = Tr[DH].
 *   D_val  device double[nnz_D]: the values gbe_density wrote, on the pattern of `g`.
 *   A      device CSR of dimension n, ascending columns (need not be symmetric, need not share D's pattern).
 *   out    HOST double; the call synchronises the stream.  The reduction order is fixed: reproducible bit for bit. */
int gbe_expectation(const gbe_graph* g, const double* D_val, const gbe_csr_view* A, void* cuda_stream, double* out);

/* gbe_expectation for callers that cannot allocate (code under CUDA-graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same <A> = Tr[D A], same kernels, same fixed reduction order - bit for bit the value
 * gbe_expectation returns - but
 *   - the call allocates NOTHING (no cudaMalloc / cudaMallocAsync / cudaFree, no allocating library routine) and does
 *     not synchronise: it enqueues two kernels on `cuda_stream` and returns;
 *   - its scratch (n per-row partial sums) is a static device array of GBE_STATIC_MAX_N doubles (1 MiB) inside the
 *     library, held by every GPU that loads the library until the process exits.  n > GBE_STATIC_MAX_N: GBE_ELIMIT,
 *     nothing launched (use gbe_expectation);
 *   - out_dev is a DEVICE double[1] of the caller, valid once the stream reaches that point.
 *   g, D_val, A   as for gbe_expectation (device pointers; borrowed for the duration of the enqueued work).
 * All calls on one device share the scratch array: calls that OVERLAP on the GPU (different streams without an ordering
 * between them) race on it and return garbage; calls on one stream, or ordered by events, are safe.  Nothing in it needs
 * clearing between calls (every word read was written by the same call).  The first call on each device looks up the
 * array's device address (cudaGetSymbolAddress, no allocation); make that first call outside a stream capture.
 * Errors: GBE_EINVAL (null g / out_dev / A, null D_val with nnz_D > 0), GBE_EMISMATCH (A.n != n), GBE_ELIMIT, GBE_ECUDA. */
#define GBE_STATIC_MAX_N 131072
int gbe_expectation_static(const gbe_graph* g, const double* D_val, const gbe_csr_view* A, void* cuda_stream,
                           double* out_dev);

/* Error of D against a dense reference matrix, e.g. the exact projector (Fig.2: "the error in the calculated
 * density matrix ... as measured by the Frobenius norm (normalized per atom)"; obs. (ii) P:L65: the error is set by tau).
 *   D_val   device double[nnz_D] on the pattern of `g`.
 *   D_ref   device double, n rows of ld_ref >= n doubles, row-major (entry (k,i) at D_ref[k * ld_ref + i]).
 *   out     HOST double[3]; the call synchronises the stream:
 *           out[0] = max |D_ki - D_ref_ki| over the stored entries of D,
 *           out[1] = sum (D_ki - D_ref_ki)^2 over the stored entries,
 *           out[2] = ||D - D_ref||_F^2 over the full matrix: where D stores nothing it is zero (obs. (iv) P:L65).
 *           Frobenius error per atom = sqrt(out[2]) / n_atoms.  Fixed reduction order: reproducible bit for bit. */
int gbe_error_norms(const gbe_graph* g, const double* D_val, const double* D_ref, int64_t ld_ref, void* cuda_stream,
                    double* out);

/* Number of CUDA kernels this library has launched in this process so far (all threads). */
uint64_t gbe_launch_count(void);

/* Scratch memory the graph builds (gbe_build_graph, gbe_update_graph) may take for the candidate bitmaps of the
 * thresholded product (step 1): the sizing pass leaves one bitmap of n bits per row (n^2 / 8 bytes) for the numeric pass,
 * which otherwise walks all products a_ik t_kj a second time.  Above the limit (default 8 GiB), or when the allocation
 * fails, the second walk is taken; the graph is the same bit for bit.  bytes = 0 switches the bitmaps off.
 * Process-wide; returns the previous limit. */
size_t gbe_set_build_scratch_limit(size_t bytes);

/* Programmatic dependent launch of the SP2 kernels (sm_90+: the next kernel of an iteration becomes resident while the
 * previous one drains and synchronises with it in the kernel).  It changes when kernels start, never what
 * they compute: results are bit for bit the same on and off (tests/test_gpu_parity.py).  On by default; GBE_PDL=0 in the
 * environment at load time, or on = 0 here, switches it off (debugging, profilers that cannot follow programmatic edges).
 * Process-wide; affects calls made from now on; returns the previous setting (0 / 1). */
int32_t gbe_set_dependent_launch(int32_t on);

/* Largest core+halo size m_p the packed SP2 kernel takes in graphs built FROM NOW ON (see gbe_graph_set_sp2_path); larger
 * communities of the same graph run through the tiled kernel.  0 <= m <= 160 (160 = what fits one SM's shared memory,
 * and the default: one bin of up to 16 communities per SM).  Process-wide tuning knob; returns the previous value,
 * -1 if m is out of range. */
int32_t gbe_set_packed_max_m(int32_t m);

void gbe_free_graph(gbe_graph* g);

const char* gbe_strerror(int status);
const char* gbe_last_cuda_error(void); /* text of the most recent failing CUDA call in this thread ("" if none) */
const char* gbe_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GBE_H */
