// Finite-temperature Fermi-operator expansion on the subgraphs.
//
//     D = [e^{beta (H - mu)} + 1]^{-1}  ~  sum_{n=0}^{M} c_n T_n(Ht),   Ht = (H - b)/a in [-1, 1]        (Eq.(7))
// with Chebyshev polynomials T_n, evaluated per community on x[s_p] exactly like the zero-temperature path (Eq.(6)
// P:L58-63): the three-term recurrence T_{n+1} = 2 Ht T_n - T_{n-1} is Eq.(5) P:L51-56 with its alpha_n, one dense
// product per term ("same gather/scatter, three-term recurrence of dense GEMMs instead of SP2").
//   a = (eps_max - eps_min)/2, b = (eps_max + eps_min)/2 from the Gershgorin bounds of the global H (A-5), so the
//   gathered X0 = (eps_max I - H)/(eps_max - eps_min) gives Ht = I - 2 X0.
//   c_n = (2 - delta_n0)/N sum_{k<N} f(cos th_k) cos(n th_k), th_k = pi (k + 1/2)/N (Chebyshev-Gauss quadrature, N = 2048),
//   f(x) = 1/(1 + exp(beta (a x + b - mu))), computed on the device from the device-resident bounds: no host round trip.
// The dense product of every term runs in the X^2 kernel's second mode (gbe_x2.cu, OP = 1).
#include "gbe_internal.cuh"

namespace {
constexpr int CHEB_NQ = 2048;

__global__ void __launch_bounds__(256) k_cheb_coef(gbe_state* st, double mu, double beta, int order) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n > order) return;
  const double a = 0.5 * (st->eps_max - st->eps_min), b = 0.5 * (st->eps_max + st->eps_min);
  double acc = 0.0;
  for (int k = 0; k < CHEB_NQ; ++k) {
    const double th = M_PI * (k + 0.5) / CHEB_NQ;
    const double arg = beta * (a * cos(th) + b - mu);
    double f;
    if (arg > 0.0) {
      const double e = exp(-arg);
      f = e / (1.0 + e);
    } else {
      f = 1.0 / (1.0 + exp(arg));
    }
    acc += f * cos(n * th);
  }
  st->t1[n] = (n == 0 ? 1.0 : 2.0) * acc / CHEB_NQ;  // the coefficient array lives in the (unused) t1 log
}

// From the gathered X0 (in BX): BX <- Ht = I - 2 X0; B0 <- T_0 = I; B1 <- T_1 = Ht; BD <- c_0 I + c_1 Ht.
// One CTA per gather work item (community, 64 rows); pad columns stay zero in all four buffers.
__global__ void __launch_bounds__(256) k_cheb_init(int rows_per_cta, const gbe_gitem* __restrict__ gitems,
                                                   const int64_t* __restrict__ sub_ptr, const int64_t* __restrict__ dense_off,
                                                   const gbe_state* __restrict__ st, double* __restrict__ BX,
                                                   double* __restrict__ B0, double* __restrict__ B1, double* __restrict__ BD) {
  const int p = gitems[blockIdx.x].p, r0 = gitems[blockIdx.x].r0;
  const int m = (int)(sub_ptr[p + 1] - sub_ptr[p]);
  const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
  const int64_t off = dense_off[p];
  const double c0 = st->t1[0], c1 = st->t1[1];
  const int rend = min(m, r0 + rows_per_cta);
  const int nel = (rend - r0) * ld;
  for (int e = threadIdx.x; e < nel; e += blockDim.x) {
    const int r = r0 + e / ld, c = e % ld;
    const int64_t idx = off + (int64_t)r * ld + c;
    const double id = (r == c) ? 1.0 : 0.0;
    const double xt = c < m ? id - 2.0 * BX[idx] : 0.0;
    BX[idx] = xt;
    B0[idx] = id;
    B1[idx] = xt;
    BD[idx] = c0 * id + c1 * xt;
  }
}

// occupation: sum over all communities of the core diagonal of D (fixed order: one CTA, strided partial sums, tree)
__global__ void __launch_bounds__(1024) k_core_trace(int n_part, const int64_t* __restrict__ sub_ptr,
                                                     const int32_t* __restrict__ ncore, const int64_t* __restrict__ dense_off,
                                                     const double* __restrict__ BD, gbe_state* st) {
  __shared__ double sh[1024];
  const int t = threadIdx.x;
  double a = 0.0;
  for (int p = 0; p < n_part; ++p) {
    const int m = (int)(sub_ptr[p + 1] - sub_ptr[p]);
    const int ld = (m + GBE_LD_ALIGN - 1) / GBE_LD_ALIGN * GBE_LD_ALIGN;
    const double* D = BD + dense_off[p];
    for (int i = t; i < ncore[p]; i += 1024) a += D[(int64_t)i * ld + i];
  }
  sh[t] = a;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (t < o) sh[t] += sh[t + o];
    __syncthreads();
  }
  if (t == 0) {
    st->t2[0] = sh[0];
    st->iters_done = 0;  // the scatter reads buffer (iters_done & 1): the caller passes BD for both
    st->inplace = 0;
  }
}
}  // namespace

int gbe_launch_cheb_coef(gbe_state* st, double mu, double beta, int order, cudaStream_t s) {
  k_cheb_coef<<<(order + 256) / 256, 256, 0, s>>>(st, mu, beta, order);
  GBE_LAUNCHED();
  return GBE_OK;
}
int gbe_launch_cheb_init(const gbe_graph* g, const gbe_state* st, double* BX, double* B0, double* B1, double* BD,
                         cudaStream_t s) {
  if (g->n_gitems == 0) return GBE_OK;
  k_cheb_init<<<g->n_gitems, 256, 0, s>>>(g->gather_rows, g->gitems, g->sub_ptr, g->dense_off, st, BX, B0, B1, BD);
  GBE_LAUNCHED();
  return GBE_OK;
}
int gbe_launch_core_trace(const gbe_graph* g, const double* BD, gbe_state* st, cudaStream_t s) {
  k_core_trace<<<1, 1024, 0, s>>>(g->n_part, g->sub_ptr, g->ncore, g->dense_off, BD, st);
  GBE_LAUNCHED();
  return GBE_OK;
}
