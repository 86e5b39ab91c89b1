// Mixed-precision inversion ("We perform a mixed precision inversion by calling the QOPQDP inverter or
// Dirac operation module in single or double precision, as appropriate"; DESIGN.md R-MIXED):
// defect correction around the fp32 BiCGStab with BOTH precalculation-matrix sets resident in HBM (the 1.5 GB GTX480
// of the paper had to wipe and re-copy them at every precision change).
//
//     x = 0 ; r = b                                                  fp64
//     repeat:  stop when ||r|| <= tol ||b||
//              e  = BiCGStab_fp32( W32, r / ||r|| rounded to fp32, inner_tol )      ok_bicgstab.cu, fp32 W
//              x += ||r|| e ;  r = b - M x                                          fp64 apply with W64
//
// Vector kernels here: residual + norm (fixed-order fp64 reduction), fp64 -> fp32 scaled copy, fp64 += scale * fp32.
// Internal spinor layouts (ok.h): fp64 [block][c 12][site 32][complex], fp32 [block][u 6][site 32][2 complex].
#include <math.h>

#include "ok_internal.cuh"

namespace okd {

namespace {

constexpr int kMxThreads = 256;
constexpr int kMxPerCta = 8 * kBlock * 12;   // complex numbers per CTA (8 site blocks): lattice-determined grid

struct MixScal {
  double rr;      // ||r||^2
  double rn;      // ||r||
  double inv_rn;  // 1 / ||r||  (0 when r = 0)
};

__device__ __forceinline__ long long idx32_of(long long i64) {   // fp64 flat complex index -> fp32 flat complex index
  const long long site = i64 & 31, bc = i64 >> 5;
  const long long comp = bc % 12, blk = bc / 12;
  return ((blk * 6 + (comp >> 1)) * 32 + site) * 2 + (comp & 1);
}

// r = b - t (t == nullptr: r = b) ; partials[cta] = sum |r|^2 in a fixed order
__global__ void __launch_bounds__(kMxThreads)
mx_residual(const double2* __restrict__ b, const double2* __restrict__ t, double2* __restrict__ r, long long n, double* __restrict__ partials) {
  const long long e0 = (long long)blockIdx.x * kMxPerCta;
  long long e1 = e0 + kMxPerCta;
  if (e1 > n) e1 = n;
  double d = 0.0;
  for (long long i = e0 + threadIdx.x; i < e1; i += kMxThreads) {
    double2 v = b[i];
    if (t) { const double2 tv = t[i]; v.x -= tv.x; v.y -= tv.y; }
    r[i] = v;
    d += v.x * v.x + v.y * v.y;
  }
#pragma unroll
  for (int m = 16; m > 0; m >>= 1) d += __shfl_xor_sync(0xffffffffu, d, m);
  __shared__ double red[kMxThreads / 32];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = d;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < kMxThreads / 32; ++w) s += red[w];
    partials[blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(kMxThreads) mx_finalize(const double* __restrict__ partials, int count, MixScal* sc) {
  __shared__ double red[kMxThreads];
  double s = 0.0;
  for (int i = threadIdx.x; i < count; i += kMxThreads) s += partials[i];
  red[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0;
    for (int k = 0; k < kMxThreads; ++k) a += red[k];
    sc->rr = a;
    sc->rn = sqrt(a);
    sc->inv_rn = a > 0.0 ? 1.0 / sqrt(a) : 0.0;
  }
}

// lo = (float)(r * inv_rn)
__global__ void __launch_bounds__(kMxThreads)
mx_down(const double2* __restrict__ r, float2* __restrict__ lo, long long n, const MixScal* __restrict__ sc) {
  const long long i = (long long)blockIdx.x * kMxThreads + threadIdx.x;
  if (i >= n) return;
  const double s = sc->inv_rn;
  const double2 v = r[i];
  lo[idx32_of(i)] = make_float2((float)(v.x * s), (float)(v.y * s));
}

// x += rn * e
__global__ void __launch_bounds__(kMxThreads)
mx_up(double2* __restrict__ x, const float2* __restrict__ e, long long n, const MixScal* __restrict__ sc) {
  const long long i = (long long)blockIdx.x * kMxThreads + threadIdx.x;
  if (i >= n) return;
  const double s = sc->rn;
  const float2 ev = e[idx32_of(i)];
  double2 v = x[i];
  v.x += s * (double)ev.x;
  v.y += s * (double)ev.y;
  x[i] = v;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

size_t mixed_work_bytes(const ok_params* p) {
  ok_params p32 = *p, p64 = *p;
  p32.precision = OK_FP32;
  p64.precision = OK_FP64;
  p32.nrhs = p64.nrhs = 1;
  Geom g = make_geom(p);
  const size_t n = (size_t)g.nblk * kBlock * 12;
  const size_t ncta = (n + kMxPerCta - 1) / kMxPerCta;
  return align_up(bicgstab_work_bytes(&p32), 256) + 2 * align_up(n * sizeof(double2), 256) + 2 * align_up(n * sizeof(float2), 256) +
         align_up(ncta * sizeof(double), 256) + 256;
}

int run_bicgstab_mixed(const ok_params* p64, const void* W64, const ok_params* p32, const void* W32, const void* src, void* xout,
                       double tol, double inner_tol, int maxit, int max_outer, int* iters, int* outer_out, double* resid) {
  Geom g = make_geom(p64);
  cudaStream_t st = ctx().stream;
  const long long n = (long long)g.nblk * kBlock * 12;
  const int ncta = (int)((n + kMxPerCta - 1) / kMxPerCta);
  const unsigned egrid = (unsigned)((n + kMxThreads - 1) / kMxThreads);
  char* w = static_cast<char*>(ctx().work) + align_up(bicgstab_work_bytes(p32), 256);
  const size_t v64 = align_up((size_t)n * sizeof(double2), 256), v32 = align_up((size_t)n * sizeof(float2), 256);
  double2* r = reinterpret_cast<double2*>(w);
  double2* t = reinterpret_cast<double2*>(w + v64);
  float2* lo = reinterpret_cast<float2*>(w + 2 * v64);
  float2* e = reinterpret_cast<float2*>(w + 2 * v64 + v32);
  double* partials = reinterpret_cast<double*>(w + 2 * v64 + 2 * v32);
  MixScal* sc = reinterpret_cast<MixScal*>(w + 2 * v64 + 2 * v32 + align_up((size_t)ncta * sizeof(double), 256));
  const double2* b = static_cast<const double2*>(src);
  double2* x = static_cast<double2*>(xout);

  auto residual = [&](const double2* tt, double* rr) -> int {
    mx_residual<<<ncta, kMxThreads, 0, st>>>(b, tt, r, n, partials);
    OK_LAUNCHED("mx_residual");
    mx_finalize<<<1, kMxThreads, 0, st>>>(partials, ncta, sc);
    OK_LAUNCHED("mx_finalize");
    MixScal h;
    OK_CUDA(cudaMemcpyAsync(&h, sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaStreamSynchronize(st));
    *rr = h.rr;
    return OK_SUCCESS;
  };

  int rc;
  OK_CUDA(cudaMemsetAsync(x, 0, (size_t)n * sizeof(double2), st));
  double rr = 0.0;
  if ((rc = residual(nullptr, &rr))) return rc;
  const double bnorm2 = rr;
  int total = 0, outer = 0, status = OK_EMAXIT;
  if (isnan(bnorm2)) return OK_EBREAKDOWN;
  if (bnorm2 == 0.0) {
    *iters = 0; *outer_out = 0; *resid = 0.0;
    return OK_SUCCESS;
  }
  for (;;) {
    if (rr <= tol * tol * bnorm2) { status = OK_SUCCESS; break; }
    if (outer >= max_outer || total >= maxit) break;
    if (isnan(rr)) { status = OK_EBREAKDOWN; break; }
    mx_down<<<egrid, kMxThreads, 0, st>>>(r, lo, n, sc);
    OK_LAUNCHED("mx_down");
    int it = 0;
    double ires = 0.0;
    rc = run_bicgstab(p32, W32, lo, e, inner_tol, maxit - total, &it, &ires);
    total += it;
    ++outer;
    if (rc != OK_SUCCESS && rc != OK_EMAXIT) { status = rc; break; }
    // the inner solve used the front of the workspace only; sc (behind it) still holds ||r||
    mx_up<<<egrid, kMxThreads, 0, st>>>(x, e, n, sc);
    OK_LAUNCHED("mx_up");
    if ((rc = launch_apply(p64, W64, x, t, nullptr, nullptr, nullptr))) return rc;
    if ((rc = residual(t, &rr))) return rc;
  }
  *iters = total;
  *outer_out = outer;
  *resid = sqrt(rr / bnorm2);
  return status;
}

}  // namespace okd
