// Single-RHS Oktay-Kronfeld Dirac apply, Eq. (2.2), on the reduced W storage formats
// OK_W_BLOCK (the 260 non-zero colour blocks) and OK_W_DS (D and S once per term); SURVEY.md 8(f) item 1.
// Same operator and same spinor layout as ok_apply.cu; only the bytes of W that are streamed change:
//   31 104 B/site (dense)  ->  18 720 B (OK_W_BLOCK)  ->  9 504 B (OK_W_DS), fp32.
//
// lane <-> site (blocks of 32 sites), CTA = 2 warps: warp a owns spin row a of the upper AND of the lower spin
// half, i.e. output rows 3a..3a+2 and 6+3a..6+3a+2, because both halves use the same rows of D and S:
//   out_u += UL[a,:] psi_u + UR[a,:] psi_l        out_l += LL[a,:] psi_u + LR[a,:] psi_l
// with UL = LR = D, UR = S, LL = +-S for OK_W_DS.  W goes global -> registers with streaming 8/16-byte loads
// (one complex per lane, 256/512 contiguous bytes per warp load); the zero pattern of every term is a
// compile-time template argument, terms of equal pattern share one loop body.
#include "ok_internal.cuh"
#include "ok_sparse.cuh"

namespace okd {

__constant__ int8_t c_soff[kTerms][4];
__constant__ int c_srun[3][kTerms][2][4];   // [format - 1][term][a][m] -> first complex unit of the run
static bool g_sparse_ready = false;

namespace {

template <typename real> struct SV;
template <> struct SV<float> { using cx = float2; using vec = float4; static constexpr int NC = 6; };
template <> struct SV<double> { using cx = double2; using vec = double2; static constexpr int NC = 12; };

__device__ __forceinline__ int wraps(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

// the spin column a non-zero block j of row a sits in
template <int MASK> __device__ __forceinline__ int spin_col(int a, int j) {
  return MASK == kMaskFull ? j : (MASK == kMaskDiag ? a : 1 - a);
}
template <int MASK> struct NB { static constexpr int v = MASK == kMaskFull ? 2 : (MASK == 0 ? 0 : 1); };

// acc[cr] += sign * sum_{j,cc} w[cr][j][cc] * s[3 * spin_col(a, j) + cc]     (s = one spin half of the neighbour spinor)
template <typename real, int MASK, typename cx>
__device__ __forceinline__ void rows_times(real (&acc)[3][2], const cx (&w)[3][2][3], const cx* s, int a, real sign) {
#pragma unroll
  for (int j = 0; j < NB<MASK>::v; ++j) {
    const int b = spin_col<MASK>(a, j);
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      // b is warp-uniform but a runtime value: select the spinor component without dynamic register indexing
      const cx sv = b ? s[3 + cc] : s[cc];
      const real sr = sign * sv.x, si = sign * sv.y;
#pragma unroll
      for (int cr = 0; cr < 3; ++cr) {
        acc[cr][0] = fma(w[cr][j][cc].x, sr, acc[cr][0]);
        acc[cr][0] = fma(-w[cr][j][cc].y, si, acc[cr][0]);
        acc[cr][1] = fma(w[cr][j][cc].x, si, acc[cr][1]);
        acc[cr][1] = fma(w[cr][j][cc].y, sr, acc[cr][1]);
      }
    }
  }
}

// STREAM: evict-first loads (W is read once); OK_W_CONJ reads every stored matrix twice (own site, neighbour's partner
// term) and wants the second read served by L2, so it loads with the default policy
template <int MASK, bool STREAM = true, typename cx>
__device__ __forceinline__ void load_rows(cx (&w)[3][2][3], const cx* run) {
  constexpr int nb = NB<MASK>::v;
#pragma unroll
  for (int cr = 0; cr < 3; ++cr)
#pragma unroll
    for (int j = 0; j < nb; ++j)
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) {
        const cx* q = run + (size_t)((cr * nb + j) * 3 + cc) * kBlock;
        w[cr][j][cc] = STREAM ? __ldcs(q) : __ldg(q);
      }
}

// OK_W_CONJ, opposite-direction term: rows a of M^dag from the partner's matrix M at the neighbour site,
//   (M^dag)[a,cr][b,cc] = conj(M[b,cc][a,cr]) ; M[b,.][a,.] sits in the run of spin row b at (cc * nb + jj) * 3 + cr
template <int MASK, typename cx>
__device__ __forceinline__ void load_rows_conj(cx (&w)[3][2][3], const cx* Wn, const int (*runs)[4], int m, int a) {
  constexpr int nb = NB<MASK>::v;
  const int jj = MASK == kMaskFull ? a : 0;
#pragma unroll
  for (int j = 0; j < nb; ++j) {
    const cx* run = Wn + (size_t)runs[spin_col<MASK>(a, j)][m] * kBlock;
#pragma unroll
    for (int cr = 0; cr < 3; ++cr)
#pragma unroll
      for (int cc = 0; cc < 3; ++cc) {
        cx v = __ldg(run + (size_t)((cc * nb + jj) * 3 + cr) * kBlock);
        v.y = -v.y;
        w[cr][j][cc] = v;
      }
  }
}

}  // namespace

namespace {

template <typename real>
struct SiteCtx {
  int x, y, z, t, lane, a;
  Geom g;
};

// one stencil term whose zero pattern is (MD, UL, LR, MS) and whose LL = -S when NEG
template <typename real, int FMT, int MD, int UL, int LR, int MS, int NEG, int CONJ = 0>
__device__ __forceinline__ void term_body(int term, const SiteCtx<real>& c, const typename SV<real>::cx* __restrict__ W0, const typename SV<real>::cx* __restrict__ Wb,
                                          const typename SV<real>::vec* __restrict__ psi, real (&acc_u)[3][2], real (&acc_l)[3][2]) {
  using cx = typename SV<real>::cx;
  using vec = typename SV<real>::vec;
  constexpr int NC = SV<real>::NC;
  const int xx = wraps(c.x + c_soff[term][0], c.g.L[0]);
  const int yy = wraps(c.y + c_soff[term][1], c.g.L[1]);
  const int zz = wraps(c.z + c_soff[term][2], c.g.L[2]);
  const int tt = wraps(c.t + c_soff[term][3], c.g.L[3]);
  const int nn = xx + c.g.L[0] * (yy + c.g.L[1] * (zz + c.g.L[2] * tt));
  const vec* sp = psi + (size_t)(nn >> 5) * NC * kBlock + (nn & 31);
  cx s[12];
  if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int u = 0; u < 6; ++u) {
      const float4 v = __ldg(sp + u * kBlock);
      s[2 * u] = make_float2(v.x, v.y);
      s[2 * u + 1] = make_float2(v.z, v.w);
    }
  } else {
#pragma unroll
    for (int u = 0; u < 12; ++u) s[u] = __ldg(sp + u * kBlock);
  }
  const int* ro = c_srun[FMT - 1][term][c.a];
  cx w[3][2][3];
  if constexpr (CONJ) {
    // W_term(x) = [[D^dag, -S^dag], [-S^dag, D^dag]] of the partner term at the neighbour site nn (the site psi comes from too)
    const cx* Wn = W0 + (size_t)(nn >> 5) * sparse_site_units(FMT) * kBlock + (nn & 31);
    const int (*runs)[4] = c_srun[FMT - 1][term];
    cx wd[3][2][3];
    if constexpr (MD != 0) load_rows_conj<MD>(wd, Wn, runs, 0, c.a);
    load_rows_conj<MS>(w, Wn, runs, 1, c.a);
    if constexpr (MD != 0) {
      if constexpr (UL) rows_times<real, MD>(acc_u, wd, s, c.a, real(1));
      if constexpr (LR) rows_times<real, MD>(acc_l, wd, s + 6, c.a, real(1));
    }
    rows_times<real, MS>(acc_u, w, s + 6, c.a, real(-1));
    rows_times<real, MS>(acc_l, w, s, c.a, real(-1));
  } else if constexpr (FMT != OK_W_BLOCK) {
    cx wd[3][2][3];
    constexpr bool ST = FMT != OK_W_CONJ;
    if constexpr (MD != 0) load_rows<MD, ST>(wd, Wb + (size_t)ro[0] * kBlock);   // both runs in flight before the first use
    load_rows<MS, ST>(w, Wb + (size_t)ro[1] * kBlock);
    if constexpr (MD != 0) {
      if constexpr (UL) rows_times<real, MD>(acc_u, wd, s, c.a, real(1));
      if constexpr (LR) rows_times<real, MD>(acc_l, wd, s + 6, c.a, real(1));
    }
    rows_times<real, MS>(acc_u, w, s + 6, c.a, real(1));
    rows_times<real, MS>(acc_l, w, s, c.a, NEG ? real(-1) : real(1));
  } else {
    if constexpr (MD != 0 && UL) {
      load_rows<MD>(w, Wb + (size_t)ro[0] * kBlock);
      rows_times<real, MD>(acc_u, w, s, c.a, real(1));
    }
    load_rows<MS>(w, Wb + (size_t)ro[1] * kBlock);
    rows_times<real, MS>(acc_u, w, s + 6, c.a, real(1));
    load_rows<MS>(w, Wb + (size_t)ro[2] * kBlock);
    rows_times<real, MS>(acc_l, w, s, c.a, real(1));
    if constexpr (MD != 0 && LR) {
      load_rows<MD>(w, Wb + (size_t)ro[3] * kBlock);
      rows_times<real, MD>(acc_l, w, s + 6, c.a, real(1));
    }
  }
}

}  // namespace

template <typename real, int FMT, bool DOT>
__global__ void __launch_bounds__(64)
apply_sparse_kernel(const typename SV<real>::cx* __restrict__ W, const typename SV<real>::vec* __restrict__ psi,
                    typename SV<real>::vec* __restrict__ out, Geom g, const typename SV<real>::vec* __restrict__ dot_a,
                    double* __restrict__ partials) {
  using cx = typename SV<real>::cx;
  constexpr int NC = SV<real>::NC;
  SiteCtx<real> c;
  c.lane = threadIdx.x & 31;
  c.a = threadIdx.x >> 5;
  c.g = g;
  const int blk = blockIdx.x;
  int n = blk * kBlock + c.lane;
  const bool padded = n >= g.V;   // padded lane of the last block: its own W is zero, but OK_W_CONJ also reads a neighbour's
  if (padded) n = 0;
  c.x = n % g.L[0];
  int q = n / g.L[0];
  c.y = q % g.L[1];
  q /= g.L[1];
  c.z = q % g.L[2];
  c.t = q / g.L[2];

  real acc_u[3][2], acc_l[3][2];
#pragma unroll
  for (int r = 0; r < 3; ++r) acc_u[r][0] = acc_u[r][1] = acc_l[r][0] = acc_l[r][1] = real(0);

  const cx* Wb = W + (size_t)blk * sparse_site_units(FMT) * kBlock + c.lane;

  // term classes (ok_sparse.cuh: term_desc): the loops run over terms of one zero pattern; OK_W_CONJ takes the even
  // (opposite-direction) terms from the partner matrix of the neighbour site
  constexpr int CJ = FMT == OK_W_CONJ ? 1 : 0;
#define OK_TERM(MD, UL, LR, MS, NEG, o) term_body<real, FMT, MD, UL, LR, MS, NEG, 0>(o, c, W, Wb, psi, acc_u, acc_l)
#define OK_TERM_PAIR(MD, UL, LR, MS, o)                                                                      \
  if (CJ && !((o) & 1)) term_body<real, FMT, MD, UL, LR, MS, 0, CJ>(o, c, W, Wb, psi, acc_u, acc_l);        \
  else term_body<real, FMT, MD, UL, LR, MS, 0, 0>(o, c, W, Wb, psi, acc_u, acc_l)
  OK_TERM(kMaskFull, 1, 1, kMaskFull, 1, 0);
#pragma unroll 1
  for (int o = 1; o <= 6; ++o) { OK_TERM_PAIR(kMaskFull, 1, 1, kMaskFull, o); }
  OK_TERM(kMaskDiag, 0, 1, kMaskFull, 0, 7);
  term_body<real, FMT, kMaskDiag, 1, 0, kMaskFull, 0, CJ>(8, c, W, Wb, psi, acc_u, acc_l);
#pragma unroll 1
  for (int o = 9; o <= 12; ++o) { OK_TERM_PAIR(kMaskDiag, 1, 1, kMaskOff, o); }
#pragma unroll 1
  for (int o = 13; o <= 14; ++o) { OK_TERM_PAIR(kMaskDiag, 1, 1, kMaskDiag, o); }
#pragma unroll 1
  for (int o = 15; o <= 18; ++o) { OK_TERM_PAIR(0, 0, 0, kMaskOff, o); }
#pragma unroll 1
  for (int o = 19; o <= 26; ++o) { OK_TERM_PAIR(0, 0, 0, kMaskFull, o); }
#undef OK_TERM
#undef OK_TERM_PAIR

  if (padded) {
#pragma unroll
    for (int r = 0; r < 3; ++r) acc_u[r][0] = acc_u[r][1] = acc_l[r][0] = acc_l[r][1] = real(0);
  }
  // store: row -> (unit, sub) of the internal spinor layout
  real* ob = reinterpret_cast<real*>(out + (size_t)blk * NC * kBlock);
  constexpr int RPU = 12 / NC;   // rows (components) per 16-byte unit: 2 (fp32) or 1 (fp64)
  auto dst_of = [&](real* base, int row) { return base + ((size_t)(row / RPU) * kBlock + c.lane) * (2 * RPU) + 2 * (row % RPU); };
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      const int row = 6 * h + 3 * c.a + r;
      const real vr = h ? acc_l[r][0] : acc_u[r][0], vi = h ? acc_l[r][1] : acc_u[r][1];
      real* dst = dst_of(ob, row);
      if constexpr (sizeof(real) == 4)
        *reinterpret_cast<float2*>(dst) = make_float2(vr, vi);
      else
        *reinterpret_cast<double2*>(dst) = make_double2(vr, vi);
    }

  if constexpr (DOT) {
    // partials[blk] = ( Re<a,out>, Im<a,out>, ||out||^2 ), fp64, fixed summation order
    real* ab = const_cast<real*>(reinterpret_cast<const real*>(dot_a + (size_t)blk * NC * kBlock));
    double d0 = 0.0, d1 = 0.0, d2 = 0.0;
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int r = 0; r < 3; ++r) {
        const int row = 6 * h + 3 * c.a + r;
        const real* src = dst_of(ab, row);
        const double ar = (double)src[0], ai = (double)src[1];
        const double vr = (double)(h ? acc_l[r][0] : acc_u[r][0]), vi = (double)(h ? acc_l[r][1] : acc_u[r][1]);
        d0 += ar * vr + ai * vi;
        d1 += ar * vi - ai * vr;
        d2 += vr * vr + vi * vi;
      }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) {
      d0 += __shfl_xor_sync(0xffffffffu, d0, m);
      d1 += __shfl_xor_sync(0xffffffffu, d1, m);
      d2 += __shfl_xor_sync(0xffffffffu, d2, m);
    }
    __shared__ double red[2][3];
    if (c.lane == 0) { red[c.a][0] = d0; red[c.a][1] = d1; red[c.a][2] = d2; }
    __syncthreads();
    if (threadIdx.x == 0) {
      partials[(size_t)blk * 3 + 0] = red[0][0] + red[1][0];
      partials[(size_t)blk * 3 + 1] = red[0][1] + red[1][1];
      partials[(size_t)blk * 3 + 2] = red[0][2] + red[1][2];
    }
  }
}

template <typename real, int FMT>
static int launch_sparse(const Geom& g, const void* W, const void* psi, void* out, double* partials, const void* dot_a) {
  using cx = typename SV<real>::cx;
  using vec = typename SV<real>::vec;
  if (partials)
    apply_sparse_kernel<real, FMT, true><<<g.nblk, 64, 0, ctx().stream>>>(static_cast<const cx*>(W), static_cast<const vec*>(psi),
                                                                       static_cast<vec*>(out), g, static_cast<const vec*>(dot_a), partials);
  else
    apply_sparse_kernel<real, FMT, false><<<g.nblk, 64, 0, ctx().stream>>>(static_cast<const cx*>(W), static_cast<const vec*>(psi),
                                                                        static_cast<vec*>(out), g, nullptr, nullptr);
  OK_LAUNCHED("apply_sparse_kernel");
  return OK_SUCCESS;
}

int launch_apply_sparse(const ok_params* p, const void* W, const void* psi, void* out, double* partials, const void* dot_a) {
  if (p->nrhs != 1 || p->storage < OK_W_BLOCK || p->storage > OK_W_CONJ) return OK_EINVAL;
  if (!g_sparse_ready) {
    static int h_run[3][kTerms][2][4];
    for (int f = 0; f < 3; ++f) sparse_fill_runs(f + 1, h_run[f]);
    OK_CUDA(cudaMemcpyToSymbol(c_srun, h_run, sizeof(h_run)));
    OK_CUDA(cudaMemcpyToSymbol(c_soff, kOffsets, sizeof(kOffsets)));
    g_sparse_ready = true;
  }
  Geom g = make_geom(p);
  const bool f64 = p->precision == OK_FP64;
  switch (p->storage) {
    case OK_W_BLOCK: return f64 ? launch_sparse<double, OK_W_BLOCK>(g, W, psi, out, partials, dot_a) : launch_sparse<float, OK_W_BLOCK>(g, W, psi, out, partials, dot_a);
    case OK_W_DS: return f64 ? launch_sparse<double, OK_W_DS>(g, W, psi, out, partials, dot_a) : launch_sparse<float, OK_W_DS>(g, W, psi, out, partials, dot_a);
    default: return f64 ? launch_sparse<double, OK_W_CONJ>(g, W, psi, out, partials, dot_a) : launch_sparse<float, OK_W_CONJ>(g, W, psi, out, partials, dot_a);
  }
}

}  // namespace okd
