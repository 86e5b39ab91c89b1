// BiCGStab for 12 right-hand sides solved together (BASELINE.json configs[3]): the same
// textbook recurrence as ok_bicgstab.cu (DESIGN.md R-SOLVER), run column by column on shared vectors.
// Every column j has its own rho, alpha, omega, beta; a column whose recursive residual meets the
// tolerance gets the true-residual check and is then frozen (alpha = omega = beta = 0, its vectors stop
// changing) or restarted from its true residual; the others continue.  All applies are the 12-RHS
// tensor-core apply (ok_apply_mrhs.cu), one W stream for the 12 columns.
//
// Vector layout: per-site records of 36 units of 32 B = (re[4], im[4]) of components 4 c4 .. 4 c4 + 3
// for one column (ok_internal.cuh, mrhs_vec_index): unit q = 12 c4 + j, column j = q % 12.
// A thread keeps q (hence j) fixed and strides over sites, so per-column reductions need no atomics:
// thread -> smem -> fixed-order sum per (column, quantity) -> one partial per CTA -> single-CTA final.
//
// The two vectors the operator is applied to, p and s, are ALSO written in the tensor-core operand form (split fp16,
// ok_internal.cuh) by the kernels that update them, so the apply never converts or scans its input.  Their per-column
// power-of-two scales come from norm bounds that are known before the update runs (||x||_2 >= max |x_i|):
//   ||s|| <= ||r|| + |alpha| ||v||          ||p'|| <= ||r'|| + |beta| (||p|| + |omega| ||v||)
// with ||v||^2 from the apply's epilogue and ||p||^2 reduced by the p update itself.  <rhat,v>, ||v||^2, <s,t>, ||t||^2 come
// out of the apply's epilogue (ok_apply_mrhs.cu), so an iteration is 2 applies + 3 vector kernels.
#include <math.h>

#include "ok_internal.cuh"

namespace okd {

namespace {

constexpr int kN = 12;
constexpr int kThreads = 288;          // 8 site slots x 36 units
constexpr int kSitesPerCta = 128;      // 16 strides of 8 sites
constexpr double kTinyM = 1e-300;

struct ScalM {
  double rho[kN][2], alpha[kN][2], omega[kN][2], beta[kN][2];
  double rr[kN], bnorm2[kN];
  double vv[kN], pp[kN];   // ||v||^2 of the last apply of p, ||p||^2 after the last p update
  float sscale[kN], pscale[kN], xscale[kN];   // power-of-two scales of the operand records of s, p (and x for the true residual)
  int breakdown[kN];
  int active[kN];     // written by the host: 1 = iterating, 0 = frozen
  int restart[kN];    // written by the host before k_residual: 1 = take r = rhat = p = true residual
};

struct V8 {
  float4 re, im;
};
__device__ __forceinline__ V8 ld8(const float* p) {
  V8 v;
  v.re = *reinterpret_cast<const float4*>(p);
  v.im = *reinterpret_cast<const float4*>(p + 4);
  return v;
}
__device__ __forceinline__ void st8(float* p, const V8& v) {
  *reinterpret_cast<float4*>(p) = v.re;
  *reinterpret_cast<float4*>(p + 4) = v.im;
}
#define OK_FOR4(k) for (int k = 0; k < 4; ++k)
__device__ __forceinline__ float& f4(float4& v, int k) { return reinterpret_cast<float*>(&v)[k]; }
__device__ __forceinline__ const float& f4(const float4& v, int k) { return reinterpret_cast<const float*>(&v)[k]; }

__device__ __forceinline__ bool badm(double re, double im) {
  const double a = fabs(re) + fabs(im);
  return !(a >= kTinyM) || isinf(a);
}

// sum the NQ per-thread quantities over the 24 threads that share a column; thread (j, q) of the first
// 12*NQ threads writes partials[cta][j*3 + q] (3 slots per column are always reserved)
template <int NQ>
__device__ __forceinline__ void column_reduce(const double (&d)[NQ], int unit, double* __restrict__ out) {
  __shared__ double red[kThreads][NQ];
#pragma unroll
  for (int q = 0; q < NQ; ++q) red[threadIdx.x][q] = d[q];
  __syncthreads();
  if (threadIdx.x < kN * NQ) {
    const int j = threadIdx.x / NQ, q = threadIdx.x % NQ;
    double s = 0.0;
    for (int slot = 0; slot < 8; ++slot)
      for (int c4 = 0; c4 < 3; ++c4) s += red[slot * 36 + c4 * 12 + j][q];
    out[j * 3 + q] = s;
  }
}

#define OK_MRHS_LOOP(site)                                                      \
  const int unit = threadIdx.x % 36, slot = threadIdx.x / 36;                   \
  const int j = unit % 12;                                                      \
  const long long s0__ = (long long)blockIdx.x * kSitesPerCta;                  \
  long long s1__ = s0__ + kSitesPerCta;                                         \
  if (s1__ > V) s1__ = V;                                                       \
  for (long long site = s0__ + slot; site < s1__; site += 8)

#define OK_AT(ptr, site) ((ptr) + (site) * kMrhsVecSiteFloats + unit * 8)

__global__ void __launch_bounds__(kThreads)
m_init(const float* __restrict__ b, float* __restrict__ x, float* __restrict__ r, float* __restrict__ rhat, float* __restrict__ p,
       long long V, double* __restrict__ partials) {
  double d[1] = {0.0};
  OK_MRHS_LOOP(site) {
    const V8 v = ld8(OK_AT(b, site));
    V8 z;
    z.re = z.im = make_float4(0.f, 0.f, 0.f, 0.f);
    st8(OK_AT(x, site), z);
    st8(OK_AT(r, site), v);
    st8(OK_AT(rhat, site), v);
    st8(OK_AT(p, site), v);
    OK_FOR4(k) d[0] += (double)f4(v.re, k) * f4(v.re, k) + (double)f4(v.im, k) * f4(v.im, k);
  }
  (void)j;
  column_reduce<1>(d, unit, partials + (size_t)blockIdx.x * 36);
}

__global__ void __launch_bounds__(kThreads)
m_s_update(const float* __restrict__ r, const float* __restrict__ v, float* __restrict__ s, __half* __restrict__ s_op, long long V,
           const ScalM* __restrict__ sc) {
  OK_MRHS_LOOP(site) {
    const double ar = sc->alpha[j][0], ai = sc->alpha[j][1];
    const float S = sc->sscale[j];
    const V8 rv = ld8(OK_AT(r, site)), vv = ld8(OK_AT(v, site));
    V8 o;
    OK_FOR4(k) {
      f4(o.re, k) = (float)((double)f4(rv.re, k) - (ar * f4(vv.re, k) - ai * f4(vv.im, k)));
      f4(o.im, k) = (float)((double)f4(rv.im, k) - (ar * f4(vv.im, k) + ai * f4(vv.re, k)));
    }
    st8(OK_AT(s, site), o);
    mrhs_store_operand(s_op + site * kMrhsOpSiteHalves, unit / 12, j, o.re, o.im, S);
  }
}

// x += alpha p + omega s ; r = s - omega t ; partials ( ||r||^2, Re<rhat,r>, Im<rhat,r> )
__global__ void __launch_bounds__(kThreads)
m_xr_update(float* __restrict__ x, const float* __restrict__ p, const float* __restrict__ s, const float* __restrict__ t,
            float* __restrict__ r, const float* __restrict__ rhat, long long V, const ScalM* __restrict__ sc,
            double* __restrict__ partials) {
  double d[3] = {0.0, 0.0, 0.0};
  OK_MRHS_LOOP(site) {
    const double ar = sc->alpha[j][0], ai = sc->alpha[j][1], wr = sc->omega[j][0], wi = sc->omega[j][1];
    const V8 xv = ld8(OK_AT(x, site)), pv = ld8(OK_AT(p, site)), sv = ld8(OK_AT(s, site)), tv = ld8(OK_AT(t, site)),
             hv = ld8(OK_AT(rhat, site));
    V8 xo, ro;
    OK_FOR4(k) {
      const double pr = f4(pv.re, k), pi = f4(pv.im, k), sr = f4(sv.re, k), si = f4(sv.im, k), tr = f4(tv.re, k), ti = f4(tv.im, k);
      f4(xo.re, k) = (float)((double)f4(xv.re, k) + (ar * pr - ai * pi) + (wr * sr - wi * si));
      f4(xo.im, k) = (float)((double)f4(xv.im, k) + (ar * pi + ai * pr) + (wr * si + wi * sr));
      const float rr = (float)(sr - (wr * tr - wi * ti)), ri = (float)(si - (wr * ti + wi * tr));
      f4(ro.re, k) = rr;
      f4(ro.im, k) = ri;
      const double hr = f4(hv.re, k), hi = f4(hv.im, k);
      d[0] += (double)rr * rr + (double)ri * ri;
      d[1] += hr * rr + hi * ri;
      d[2] += hr * ri - hi * rr;
    }
    st8(OK_AT(x, site), xo);
    st8(OK_AT(r, site), ro);
  }
  column_reduce<3>(d, unit, partials + (size_t)blockIdx.x * 36);
}

// p = r + beta (p - omega v), its operand records, and the partial ||p||^2 per column (slot 0 of the 3)
__global__ void __launch_bounds__(kThreads)
m_p_update(float* __restrict__ p, __half* __restrict__ p_op, const float* __restrict__ r, const float* __restrict__ v, long long V,
           const ScalM* __restrict__ sc, double* __restrict__ partials) {
  double d[1] = {0.0};
  OK_MRHS_LOOP(site) {
    const double br = sc->beta[j][0], bi = sc->beta[j][1], wr = sc->omega[j][0], wi = sc->omega[j][1];
    const float S = sc->pscale[j];
    const V8 pv = ld8(OK_AT(p, site)), rv = ld8(OK_AT(r, site)), vv = ld8(OK_AT(v, site));
    V8 o;
    OK_FOR4(k) {
      const double qr = (double)f4(pv.re, k) - (wr * f4(vv.re, k) - wi * f4(vv.im, k));
      const double qi = (double)f4(pv.im, k) - (wr * f4(vv.im, k) + wi * f4(vv.re, k));
      f4(o.re, k) = (float)((double)f4(rv.re, k) + (br * qr - bi * qi));
      f4(o.im, k) = (float)((double)f4(rv.im, k) + (br * qi + bi * qr));
      d[0] += (double)f4(o.re, k) * f4(o.re, k) + (double)f4(o.im, k) * f4(o.im, k);
    }
    st8(OK_AT(p, site), o);
    mrhs_store_operand(p_op + site * kMrhsOpSiteHalves, unit / 12, j, o.re, o.im, S);
  }
  column_reduce<1>(d, unit, partials + (size_t)blockIdx.x * 36);
}

// true residual b - Mx: columns flagged restart take r = rhat = p = it; partial ||b - Mx||^2 for every column
__global__ void __launch_bounds__(kThreads)
m_residual(const float* __restrict__ b, const float* __restrict__ Mx, float* __restrict__ r, float* __restrict__ rhat,
           float* __restrict__ p, long long V, const ScalM* __restrict__ sc, double* __restrict__ partials) {
  double d[1] = {0.0};
  OK_MRHS_LOOP(site) {
    const V8 bv = ld8(OK_AT(b, site)), mv = ld8(OK_AT(Mx, site));
    V8 o;
    OK_FOR4(k) {
      f4(o.re, k) = (float)((double)f4(bv.re, k) - (double)f4(mv.re, k));
      f4(o.im, k) = (float)((double)f4(bv.im, k) - (double)f4(mv.im, k));
      d[0] += (double)f4(o.re, k) * f4(o.re, k) + (double)f4(o.im, k) * f4(o.im, k);
    }
    if (sc->restart[j]) {
      st8(OK_AT(r, site), o);
      st8(OK_AT(rhat, site), o);
      st8(OK_AT(p, site), o);
    }
  }
  column_reduce<1>(d, unit, partials + (size_t)blockIdx.x * 36);
}

enum StageM { MF_INIT = 0, MF_V = 1, MF_T = 2, MF_XR = 3, MF_RES = 4, MF_P = 5 };

// single CTA: fixed-order sum of the per-CTA partials (36 doubles each), then the per-column scalars
template <int STAGE>
__global__ void __launch_bounds__(kThreads) m_finalize(const double* __restrict__ partials, int count, ScalM* sc, double* __restrict__ res_out) {
  __shared__ double red[8][36];
  __shared__ double tot[36];
  const int q = threadIdx.x % 36, slot = threadIdx.x / 36;
  double s = 0.0;
  for (int i = slot; i < count; i += 8) s += partials[(size_t)i * 36 + q];
  red[slot][q] = s;
  __syncthreads();
  if (threadIdx.x < 36) {
    double a = 0.0;
    for (int k = 0; k < 8; ++k) a += red[k][threadIdx.x];
    tot[threadIdx.x] = a;
  }
  __syncthreads();
  if (threadIdx.x >= kN) return;
  const int j = threadIdx.x;
  const double t0 = tot[3 * j], t1 = tot[3 * j + 1], t2 = tot[3 * j + 2];
  const bool on = sc->active[j] != 0;
  if (STAGE == MF_INIT) {         // p = r = b
    sc->bnorm2[j] = t0; sc->rr[j] = t0;
    sc->rho[j][0] = t0; sc->rho[j][1] = 0.0;
    sc->breakdown[j] = 0;
    sc->pp[j] = t0;
    sc->pscale[j] = mrhs_scale_from_bound((float)sqrt(t0));
  } else if (STAGE == MF_RES) {   // t0 = ||b - Mx||^2 ; restart columns also reset rho and take p = r = b - Mx
    res_out[j] = t0;
    if (sc->restart[j]) {
      sc->rr[j] = t0; sc->rho[j][0] = t0; sc->rho[j][1] = 0.0; sc->breakdown[j] = 0;
      sc->pp[j] = t0;
      sc->pscale[j] = mrhs_scale_from_bound((float)sqrt(t0));
    }
  } else if (STAGE == MF_P) {     // t0 = ||p||^2 after the p update
    sc->pp[j] = t0;
  } else if (STAGE == MF_V) {     // (Re<rhat,v>, Im<rhat,v>, ||v||^2)
    sc->vv[j] = t2;
    if (!on) {                    // frozen column: s = r
      sc->alpha[j][0] = sc->alpha[j][1] = 0.0;
      sc->sscale[j] = mrhs_scale_from_bound((float)sqrt(sc->rr[j]));
      return;
    }
    if (badm(t0, t1) || badm(sc->rho[j][0], sc->rho[j][1])) sc->breakdown[j] |= 1;
    const double den = t0 * t0 + t1 * t1;
    sc->alpha[j][0] = (sc->rho[j][0] * t0 + sc->rho[j][1] * t1) / den;
    sc->alpha[j][1] = (sc->rho[j][1] * t0 - sc->rho[j][0] * t1) / den;
    // ||s|| = ||r - alpha v|| <= ||r|| + |alpha| ||v||  >= max |s_i|: the scale of s's operand records
    sc->sscale[j] = mrhs_scale_from_bound((float)(sqrt(sc->rr[j]) + hypot(sc->alpha[j][0], sc->alpha[j][1]) * sqrt(t2)));
  } else if (STAGE == MF_T) {     // (Re<s,t>, Im<s,t>, ||t||^2) ; <t,s> = conj<s,t>
    if (!on) { sc->omega[j][0] = sc->omega[j][1] = 0.0; return; }
    if (badm(t2, 0.0)) sc->breakdown[j] |= 2;
    sc->omega[j][0] = t0 / t2;
    sc->omega[j][1] = -t1 / t2;
  } else if (STAGE == MF_XR) {    // (||r||^2, Re<rhat,r>, Im<rhat,r>)
    if (!on) {                    // frozen column: p = r
      sc->beta[j][0] = sc->beta[j][1] = 0.0;
      sc->pscale[j] = mrhs_scale_from_bound((float)sqrt(sc->rr[j]));
      return;
    }
    sc->rr[j] = t0;
    if (badm(sc->omega[j][0], sc->omega[j][1]) || badm(t1, t2)) sc->breakdown[j] |= 4;
    const double r0 = sc->rho[j][0], r1 = sc->rho[j][1];
    double den = r0 * r0 + r1 * r1;
    const double q0 = (t1 * r0 + t2 * r1) / den, q1 = (t2 * r0 - t1 * r1) / den;
    const double w0 = sc->omega[j][0], w1 = sc->omega[j][1];
    den = w0 * w0 + w1 * w1;
    const double a0 = (sc->alpha[j][0] * w0 + sc->alpha[j][1] * w1) / den, a1 = (sc->alpha[j][1] * w0 - sc->alpha[j][0] * w1) / den;
    sc->beta[j][0] = q0 * a0 - q1 * a1;
    sc->beta[j][1] = q0 * a1 + q1 * a0;
    sc->rho[j][0] = t1; sc->rho[j][1] = t2;
    // ||p'|| = ||r' + beta (p - omega v)|| <= ||r'|| + |beta| (||p|| + |omega| ||v||)
    sc->pscale[j] = mrhs_scale_from_bound((float)(sqrt(t0) + hypot(sc->beta[j][0], sc->beta[j][1]) * (sqrt(sc->pp[j]) + hypot(w0, w1) * sqrt(sc->vv[j]))));
  }
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

size_t bicgstab_mrhs_work_bytes(const ok_params* p) {
  Geom g = make_geom(p);
  const size_t vb = align_up((size_t)g.V * kMrhsVecSiteFloats * sizeof(float), 256);
  size_t ncta = ((size_t)g.V + kSitesPerCta - 1) / kSitesPerCta;
  if (ncta < 1024) ncta = 1024;   // also holds the apply's partial rows (one per persistent CTA)
  return 8 * vb + align_up(ncta * 36 * sizeof(double), 256) + align_up(sizeof(ScalM), 256) + 256;
}

// src, xout: nrhs = 12 spinor fields (header + fp32 records + operand records, ok_internal.cuh)
int run_bicgstab_mrhs(const ok_params* p, const void* W, const void* src, void* xout, double tol, int maxit, int* iters,
                      double* resid) {
  Geom g = make_geom(p);
  cudaStream_t st = ctx().stream;
  const long long V = g.V;
  const size_t vb = align_up((size_t)g.V * kMrhsVecSiteFloats * sizeof(float), 256);
  const int ncta = (int)((V + kSitesPerCta - 1) / kSitesPerCta);
  size_t prow = (size_t)ncta < 1024 ? 1024 : (size_t)ncta;
  char* w = static_cast<char*>(ctx().work);
  float* r = reinterpret_cast<float*>(w + 0 * vb);
  float* rhat = reinterpret_cast<float*>(w + 1 * vb);
  float* pp = reinterpret_cast<float*>(w + 2 * vb);
  float* v = reinterpret_cast<float*>(w + 3 * vb);
  float* s = reinterpret_cast<float*>(w + 4 * vb);
  float* t = reinterpret_cast<float*>(w + 5 * vb);
  __half* p_op = reinterpret_cast<__half*>(w + 6 * vb);
  __half* s_op = reinterpret_cast<__half*>(w + 7 * vb);
  double* partials = reinterpret_cast<double*>(w + 8 * vb);
  char* after = w + 8 * vb + align_up(prow * 36 * sizeof(double), 256);
  ScalM* sc = reinterpret_cast<ScalM*>(after);
  double* res_dev = reinterpret_cast<double*>(after + align_up(sizeof(ScalM), 256));   // 12 doubles (inside the +256 tail)
  const float* b = mrhs_f32(src);
  float* x = mrhs_f32(xout);
  MrhsVecHeader* xhdr = static_cast<MrhsVecHeader*>(xout);

  struct HostBuf { ScalM sc; double res[kN]; };
  static HostBuf* h = nullptr;   // pinned host mirror
  static cudaEvent_t ev = nullptr;
  if (!h) OK_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&h), sizeof(HostBuf), cudaHostAllocDefault));
  if (!ev) OK_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
  int rc;
#define OK_TRY(e) do { if ((rc = (e))) return rc; } while (0)
  auto fetch = [&]() -> int {
    OK_CUDA(cudaMemcpyAsync(&h->sc, sc, sizeof(ScalM), cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaMemcpyAsync(h->res, res_dev, sizeof(double) * kN, cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaEventRecord(ev, st));
    return OK_SUCCESS;
  };
  auto wait = [&]() -> int {
    OK_CUDA(cudaEventSynchronize(ev));
    return OK_SUCCESS;
  };
  int active[kN], restart[kN], it_conv[kN];
  auto push_flags = [&]() -> int {   // host -> device: active / restart masks (pageable source is copied before return)
    OK_CUDA(cudaMemcpyAsync(reinterpret_cast<char*>(sc) + offsetof(ScalM, active), active, sizeof(active), cudaMemcpyHostToDevice, st));
    OK_CUDA(cudaMemcpyAsync(reinterpret_cast<char*>(sc) + offsetof(ScalM, restart), restart, sizeof(restart), cudaMemcpyHostToDevice, st));
    return OK_SUCCESS;
  };
  for (int j = 0; j < kN; ++j) { active[j] = 1; restart[j] = 0; it_conv[j] = 0; }
  OK_CUDA(cudaMemsetAsync(sc, 0, sizeof(ScalM), st));
  OK_CUDA(cudaMemsetAsync(res_dev, 0, sizeof(double) * kN, st));
  OK_CUDA(cudaMemsetAsync(xhdr, 0, kMrhsVecHeaderBytes, st));   // x's operand records are stale from here on
  OK_TRY(push_flags());

  m_init<<<ncta, kThreads, 0, st>>>(b, x, r, rhat, pp, V, partials);
  OK_LAUNCHED("m_init");
  m_finalize<MF_INIT><<<1, kThreads, 0, st>>>(partials, ncta, sc, res_dev);
  OK_LAUNCHED("m_finalize");
  OK_TRY(mrhs_write_operand(p, pp, p_op, sc->pscale));   // p = b in operand form
  OK_TRY(fetch());
  OK_TRY(wait());
  double bnorm2[kN], target[kN], true_rr[kN];
  int nactive = 0;
  for (int j = 0; j < kN; ++j) {
    bnorm2[j] = h->sc.bnorm2[j];
    if (isnan(bnorm2[j])) return OK_EBREAKDOWN;
    target[j] = tol * tol * bnorm2[j];
    true_rr[j] = bnorm2[j];
    if (!(bnorm2[j] > 0.0)) { active[j] = 0; true_rr[j] = 0.0; }   // zero column: x_j = 0
    nactive += active[j];
  }
  OK_TRY(push_flags());

  auto true_residual = [&]() -> int {   // t = M x ; ||b - t||^2 per column ; flagged columns restart
    OK_TRY(push_flags());
    OK_CUDA(cudaMemsetAsync(&xhdr->valid, 0, sizeof(unsigned), st));
    OK_TRY(mrhs_ensure_operand(p, xout));   // x in operand form (column maxima + split: two passes over x, only here)
    OK_TRY(launch_apply_mrhs(p, W, mrhs_op(xout, g.V), xhdr->scale, t, nullptr, nullptr, nullptr, nullptr));
    m_residual<<<ncta, kThreads, 0, st>>>(b, t, r, rhat, pp, V, sc, partials);
    OK_LAUNCHED("m_residual");
    m_finalize<MF_RES><<<1, kThreads, 0, st>>>(partials, ncta, sc, res_dev);
    OK_LAUNCHED("m_finalize");
    bool any = false;
    for (int j = 0; j < kN; ++j) any = any || restart[j];
    if (any) OK_TRY(mrhs_write_operand(p, pp, p_op, sc->pscale));   // restarted columns: p = true residual
    OK_TRY(fetch());
    OK_TRY(wait());
    return OK_SUCCESS;
  };

  int status = OK_SUCCESS;
  int it = 0, na = 0;
  while (nactive > 0 && it < maxit) {
    ++it;
    OK_TRY(launch_apply_mrhs(p, W, p_op, sc->pscale, v, nullptr, rhat, partials, &na));   // v = M p ; <rhat,v>, ||v||^2
    m_finalize<MF_V><<<1, kThreads, 0, st>>>(partials, na, sc, res_dev);
    OK_LAUNCHED("m_finalize");
    m_s_update<<<ncta, kThreads, 0, st>>>(r, v, s, s_op, V, sc);
    OK_LAUNCHED("m_s_update");
    OK_TRY(launch_apply_mrhs(p, W, s_op, sc->sscale, t, nullptr, s, partials, &na));      // t = M s ; <s,t>, ||t||^2
    m_finalize<MF_T><<<1, kThreads, 0, st>>>(partials, na, sc, res_dev);
    OK_LAUNCHED("m_finalize");
    m_xr_update<<<ncta, kThreads, 0, st>>>(x, pp, s, t, r, rhat, V, sc, partials);
    OK_LAUNCHED("m_xr_update");
    m_finalize<MF_XR><<<1, kThreads, 0, st>>>(partials, ncta, sc, res_dev);
    OK_LAUNCHED("m_finalize");
    OK_TRY(fetch());
    m_p_update<<<ncta, kThreads, 0, st>>>(pp, p_op, r, v, V, sc, partials);
    OK_LAUNCHED("m_p_update");
    m_finalize<MF_P><<<1, kThreads, 0, st>>>(partials, ncta, sc, res_dev);
    OK_LAUNCHED("m_finalize");
    OK_TRY(wait());
    bool check = false, broke = false;
    for (int j = 0; j < kN; ++j) {
      restart[j] = 0;
      if (!active[j]) continue;
      it_conv[j] = it;
      if (h->sc.breakdown[j] & 3) { broke = true; continue; }
      if (h->sc.rr[j] <= target[j]) { restart[j] = 1; check = true; continue; }
      if ((h->sc.breakdown[j] & 4) || isnan(h->sc.rr[j])) broke = true;
    }
    if (broke) { status = OK_EBREAKDOWN; break; }
    if (check) {
      // candidates are flagged `restart`: if their true residual passes they are frozen (their restarted
      // r = rhat = p is then never used), otherwise they continue from the true residual
      OK_TRY(true_residual());
      for (int j = 0; j < kN; ++j) {
        if (!restart[j]) continue;
        true_rr[j] = h->res[j];
        if (h->res[j] <= target[j]) { active[j] = 0; --nactive; }
        restart[j] = 0;
      }
      OK_TRY(push_flags());
    }
  }
  if (status == OK_SUCCESS && nactive > 0) status = OK_EMAXIT;
  // Report the true residual of every column at exit.  After a clean finish every column was frozen right after its own
  // true-residual check and has not changed since, so those values stand; otherwise recompute them all.
  if (status != OK_SUCCESS) {
    for (int j = 0; j < kN; ++j) restart[j] = 0;
    OK_TRY(true_residual());
    for (int j = 0; j < kN; ++j) true_rr[j] = h->res[j];
  }
  double worst = 0.0;
  int itmax = 0;
  for (int j = 0; j < kN; ++j) {
    if (bnorm2[j] > 0.0) worst = fmax(worst, sqrt(true_rr[j] / bnorm2[j]));
    if (it_conv[j] > itmax) itmax = it_conv[j];
  }
  *iters = itmax;
  *resid = worst;
#undef OK_TRY
  return status;
}

}  // namespace okd
