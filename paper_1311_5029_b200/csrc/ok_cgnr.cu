// Conjugate gradient on the normal equations M^dag M x = M^dag b ("M^dag M preconditioning": future work
// in the paper): a second solver on the same Dirac apply, any W storage format.
// M^dag = Gamma_5 M Gamma_5 (gamma_5-hermiticity of the OK action, oracle pin P4), gamma_5 = [[0,-i],[i,0]] x 1_colour in
// the basis of DESIGN.md R-GAMMA, so M^dag v costs one apply plus two sign/swap passes over the spinor.
//
//   x = 0; r = b; z = M^dag r; p = z
//   loop:  w = M p ; alpha = <z,z>/<w,w> ; x += alpha p ; r -= alpha w ; stop on ||r|| <= tol ||b|| (true-residual check,
//          restart from it when it fails) ; z' = M^dag r ; beta = <z',z'>/<z,z> ; p = z' + beta p
// Reductions in fp64 with a fixed order (per-CTA tree, lattice-determined grid, single-CTA final sum): bit-reproducible.
#include <math.h>

#include "ok_internal.cuh"

namespace okd {

namespace {

constexpr int kCgThreads = 256;
constexpr int kCgPerCta = 8 * kBlock * 12;   // complex numbers per CTA
constexpr double kCgTiny = 1e-300;

template <typename real> struct CC;
template <> struct CC<float> { using type = float2; };
template <> struct CC<double> { using type = double2; };

struct CgScal {
  double zz, ww, rr, bnorm2, alpha, beta;
  int breakdown, pad;
};

// flat complex index -> is the component in the upper spin half?  (fp64: [blk][c 12][site 32]; fp32: [blk][u 6][site 32][2])
template <typename real> __device__ __forceinline__ bool upper_half(long long i) {
  return sizeof(real) == 8 ? ((i >> 5) % 12) < 6 : ((i >> 6) % 6) < 3;
}
// (gamma_5 v)_upper = -i v_lower ; (gamma_5 v)_lower = +i v_upper ; the partner component sits 192 complex away in both layouts
template <typename real, typename c2> __device__ __forceinline__ c2 g5_at(const c2* __restrict__ v, long long i) {
  c2 o;
  if (upper_half<real>(i)) { const c2 q = v[i + 192]; o.x = q.y; o.y = -q.x; }
  else { const c2 q = v[i - 192]; o.x = -q.y; o.y = q.x; }
  return o;
}

__device__ __forceinline__ void cta_sum_store(double d, double* __restrict__ partials) {
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) d += __shfl_xor_sync(0xffffffffu, d, m);
  __shared__ double red[kCgThreads / 32];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = d;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kCgThreads / 32; ++w) s += red[w];
    partials[blockIdx.x] = s;
  }
}

#define OK_CG_LOOP(i)                                                          \
  const long long e0__ = (long long)blockIdx.x * kCgPerCta;                    \
  long long e1__ = e0__ + kCgPerCta;                                           \
  if (e1__ > n) e1__ = n;                                                      \
  for (long long i = e0__ + threadIdx.x; i < e1__; i += kCgThreads)

enum CgMode { CG_COPY = 0, CG_G5 = 1, CG_RESID = 2 };

// out = in (COPY) | gamma_5 in (G5) | b - in (RESID) ; partial ||out||^2 ; ZERO: also x = 0
template <typename real, int MODE, bool ZERO>
__global__ void __launch_bounds__(kCgThreads)
cg_map_norm(const typename CC<real>::type* __restrict__ in, const typename CC<real>::type* __restrict__ b,
            typename CC<real>::type* __restrict__ out, typename CC<real>::type* __restrict__ x, long long n, double* __restrict__ partials) {
  using c2 = typename CC<real>::type;
  double d = 0.0;
  OK_CG_LOOP(i) {
    c2 v;
    if (MODE == CG_G5) v = g5_at<real>(in, i);
    else if (MODE == CG_RESID) { const c2 bv = b[i], tv = in[i]; v.x = (real)((double)bv.x - (double)tv.x); v.y = (real)((double)bv.y - (double)tv.y); }
    else v = in[i];
    if (out) out[i] = v;
    if (ZERO) { c2 z; z.x = z.y = real(0); x[i] = z; }
    d += (double)v.x * v.x + (double)v.y * v.y;
  }
  cta_sum_store(d, partials);
}

// x += alpha p ; r -= alpha w ; partial ||r||^2
template <typename real>
__global__ void __launch_bounds__(kCgThreads)
cg_xr(typename CC<real>::type* __restrict__ x, typename CC<real>::type* __restrict__ r, const typename CC<real>::type* __restrict__ p,
      const typename CC<real>::type* __restrict__ w, long long n, const CgScal* __restrict__ sc, double* __restrict__ partials) {
  using c2 = typename CC<real>::type;
  const double a = sc->alpha;
  double d = 0.0;
  OK_CG_LOOP(i) {
    const c2 xv = x[i], rv = r[i], pv = p[i], wv = w[i];
    c2 xo, ro;
    xo.x = (real)((double)xv.x + a * pv.x);
    xo.y = (real)((double)xv.y + a * pv.y);
    ro.x = (real)((double)rv.x - a * wv.x);
    ro.y = (real)((double)rv.y - a * wv.y);
    x[i] = xo;
    r[i] = ro;
    d += (double)ro.x * ro.x + (double)ro.y * ro.y;
  }
  cta_sum_store(d, partials);
}

// p = z + beta p   (FIRST: p = z)
template <typename real, bool FIRST>
__global__ void __launch_bounds__(kCgThreads)
cg_p(typename CC<real>::type* __restrict__ p, const typename CC<real>::type* __restrict__ z, long long n, const CgScal* __restrict__ sc) {
  using c2 = typename CC<real>::type;
  const double be = FIRST ? 0.0 : sc->beta;
  OK_CG_LOOP(i) {
    const c2 zv = z[i];
    c2 o = zv;
    if (!FIRST) { const c2 pv = p[i]; o.x = (real)((double)zv.x + be * pv.x); o.y = (real)((double)zv.y + be * pv.y); }
    p[i] = o;
  }
}

enum CgStage { CS_B = 0, CS_Z0 = 1, CS_W = 2, CS_R = 3, CS_Z = 4, CS_RTRUE = 5 };

template <int STAGE>
__global__ void __launch_bounds__(kCgThreads) cg_finalize(const double* __restrict__ partials, int count, CgScal* sc) {
  __shared__ double red[kCgThreads];
  double s = 0.0;
  for (int i = threadIdx.x; i < count; i += kCgThreads) s += partials[i];
  red[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x != 0) return;
  double a = 0.0;
  for (int k = 0; k < kCgThreads; ++k) a += red[k];
  if (STAGE == CS_B) { sc->bnorm2 = a; sc->rr = a; sc->breakdown = 0; }
  else if (STAGE == CS_Z0) { sc->zz = a; }
  else if (STAGE == CS_W) {
    sc->ww = a;
    if (!(a >= kCgTiny) || !(sc->zz >= kCgTiny) || isinf(a)) sc->breakdown = 1;
    sc->alpha = sc->zz / a;
  } else if (STAGE == CS_R || STAGE == CS_RTRUE) { sc->rr = a; }
  else if (STAGE == CS_Z) { sc->beta = a / sc->zz; sc->zz = a; }
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

template <typename real>
int cg_solve(const ok_params* p, const void* W, const void* src, void* xout, double tol, int maxit, int* iters, double* resid) {
  using c2 = typename CC<real>::type;
  Geom g = make_geom(p);
  cudaStream_t st = ctx().stream;
  const long long n = (long long)g.nblk * kBlock * 12;
  const int ncta = (int)((n + kCgPerCta - 1) / kCgPerCta);
  const size_t vb = align_up((size_t)n * sizeof(c2), 256);
  char* w8 = static_cast<char*>(ctx().work);
  c2* r = reinterpret_cast<c2*>(w8);
  c2* z = reinterpret_cast<c2*>(w8 + vb);
  c2* pp = reinterpret_cast<c2*>(w8 + 2 * vb);
  c2* w = reinterpret_cast<c2*>(w8 + 3 * vb);
  c2* t1 = reinterpret_cast<c2*>(w8 + 4 * vb);
  double* partials = reinterpret_cast<double*>(w8 + 5 * vb);
  CgScal* sc = reinterpret_cast<CgScal*>(w8 + 5 * vb + align_up((size_t)ncta * sizeof(double), 256));
  const c2* b = static_cast<const c2*>(src);
  c2* x = static_cast<c2*>(xout);
  int rc;
#define OK_TRY(e) do { if ((rc = (e))) return rc; } while (0)
  auto fin = [&](int stage) -> int {
    switch (stage) {
      case CS_B: cg_finalize<CS_B><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
      case CS_Z0: cg_finalize<CS_Z0><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
      case CS_W: cg_finalize<CS_W><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
      case CS_R: cg_finalize<CS_R><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
      case CS_Z: cg_finalize<CS_Z><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
      default: cg_finalize<CS_RTRUE><<<1, kCgThreads, 0, st>>>(partials, ncta, sc); break;
    }
    OK_LAUNCHED("cg_finalize");
    return OK_SUCCESS;
  };
  auto fetch = [&](CgScal* h) -> int {
    OK_CUDA(cudaMemcpyAsync(h, sc, sizeof(CgScal), cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaStreamSynchronize(st));
    return OK_SUCCESS;
  };
  // z = M^dag r = g5 M g5 r ; partial ||z||^2 left in `partials`
  auto mdag_r = [&]() -> int {
    cg_map_norm<real, CG_G5, false><<<ncta, kCgThreads, 0, st>>>(r, nullptr, t1, nullptr, n, partials);
    OK_LAUNCHED("cg_map_norm");
    OK_TRY(launch_apply(p, W, t1, w, nullptr, nullptr, nullptr));
    cg_map_norm<real, CG_G5, false><<<ncta, kCgThreads, 0, st>>>(w, nullptr, z, nullptr, n, partials);
    OK_LAUNCHED("cg_map_norm");
    return OK_SUCCESS;
  };
  auto true_residual = [&](CgScal* h) -> int {   // r = b - M x ; rr
    OK_TRY(launch_apply(p, W, x, w, nullptr, nullptr, nullptr));
    cg_map_norm<real, CG_RESID, false><<<ncta, kCgThreads, 0, st>>>(w, b, r, nullptr, n, partials);
    OK_LAUNCHED("cg_map_norm");
    OK_TRY(fin(CS_RTRUE));
    return fetch(h);
  };

  CgScal h;
  OK_CUDA(cudaMemsetAsync(sc, 0, sizeof(CgScal), st));
  cg_map_norm<real, CG_COPY, true><<<ncta, kCgThreads, 0, st>>>(b, nullptr, r, x, n, partials);   // r = b, x = 0, ||b||^2
  OK_LAUNCHED("cg_map_norm");
  OK_TRY(fin(CS_B));
  OK_TRY(fetch(&h));
  const double bnorm2 = h.bnorm2;
  if (isnan(bnorm2)) return OK_EBREAKDOWN;
  if (bnorm2 == 0.0) { *iters = 0; *resid = 0.0; return OK_SUCCESS; }
  const double target = tol * tol * bnorm2;
  OK_TRY(mdag_r());
  OK_TRY(fin(CS_Z0));
  cg_p<real, true><<<ncta, kCgThreads, 0, st>>>(pp, z, n, sc);
  OK_LAUNCHED("cg_p");
  int it = 0, status = OK_EMAXIT;
  while (it < maxit) {
    ++it;
    OK_TRY(launch_apply(p, W, pp, w, nullptr, nullptr, nullptr));
    cg_map_norm<real, CG_COPY, false><<<ncta, kCgThreads, 0, st>>>(w, nullptr, nullptr, nullptr, n, partials);
    OK_LAUNCHED("cg_map_norm");
    OK_TRY(fin(CS_W));
    cg_xr<real><<<ncta, kCgThreads, 0, st>>>(x, r, pp, w, n, sc, partials);
    OK_LAUNCHED("cg_xr");
    OK_TRY(fin(CS_R));
    OK_TRY(fetch(&h));
    if (h.breakdown || isnan(h.rr)) { status = OK_EBREAKDOWN; break; }
    if (h.rr <= target) {
      OK_TRY(true_residual(&h));
      if (h.rr <= target) { status = OK_SUCCESS; break; }
      OK_TRY(mdag_r());            // restart from the true residual
      OK_TRY(fin(CS_Z0));
      cg_p<real, true><<<ncta, kCgThreads, 0, st>>>(pp, z, n, sc);
      OK_LAUNCHED("cg_p");
      continue;
    }
    OK_TRY(mdag_r());
    OK_TRY(fin(CS_Z));
    cg_p<real, false><<<ncta, kCgThreads, 0, st>>>(pp, z, n, sc);
    OK_LAUNCHED("cg_p");
  }
  if (status != OK_SUCCESS) OK_TRY(true_residual(&h));
  *iters = it;
  *resid = sqrt(h.rr / bnorm2);
#undef OK_TRY
  return status;
}

}  // namespace

int run_cgnr(const ok_params* p, const void* W, const void* src, void* x, double tol, int maxit, int* iters, double* resid) {
  if (p->nrhs != 1) return OK_EINVAL;
  return p->precision == OK_FP64 ? cg_solve<double>(p, W, src, x, tol, maxit, iters, resid)
                                 : cg_solve<float>(p, W, src, x, tol, maxit, iters, resid);
}

}  // namespace okd
