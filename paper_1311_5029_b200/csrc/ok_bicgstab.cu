// BiCGStab ("bi-stabilized CG") around the precalculated-W apply: fused vector
// update + reduction kernels (the paper's "Common Module", Table 1c) and the
// host driver.  Algorithm = textbook van der Vorst, unpreconditioned, x0 = 0, rhat = b
// (DESIGN.md R-SOLVER):
//   v = M p; alpha = rho/<rhat,v>; s = r - alpha v; t = M s; omega = <t,s>/<t,t>;
//   x += alpha p + omega s; r = s - omega t; [converged? -> true-residual check / restart]
//   rho' = <rhat,r>; beta = (rho'/rho)(alpha/omega); p = r + beta (p - omega v).
//
// Determinism: every reduction is (thread: fixed-order fp64 sum) -> (warp: xor-shuffle tree) ->
// (CTA: fixed-order sum over warps) -> one fp64 partial per CTA; the number of CTAs depends on
// the lattice only; a single-CTA kernel then sums the partials in a fixed order and computes
// the BiCGStab scalars on the device.  No floating-point atomics anywhere.
// <rhat,v>, <t,s>, <t,t> are produced by the apply kernel's epilogue (no extra pass over v, t).
// Vector arithmetic is done in fp64 registers and rounded once to the storage precision.
#include <math.h>

#include "ok_internal.cuh"

namespace okd {

constexpr int kVecThreads = 256;
constexpr int kBlocksPerCta = 8;   // site blocks per CTA in the vector kernels (lattice-determined grid)
constexpr double kTiny = 1e-300;

struct Scal {
  double rho[2], alpha[2], omega[2], beta[2];
  double rr, bnorm2, tt;
  int breakdown;   // bit 0: rho/<rhat,v> ; bit 1: <t,t> ; bit 2: omega / rho'
  int pad;
};

__device__ __forceinline__ bool bad(double re, double im) {
  double a = fabs(re) + fabs(im);
  return !(a >= kTiny) || isinf(a);
}

// ---- block reduction of NQ fp64 quantities, fixed order; result valid in thread 0 -----------
template <int NQ>
__device__ __forceinline__ void block_reduce(double (&d)[NQ], double* out) {
  __shared__ double red[kVecThreads / 32][NQ];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < NQ; ++q)
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) d[q] += __shfl_xor_sync(0xffffffffu, d[q], m);
  if (lane == 0)
#pragma unroll
    for (int q = 0; q < NQ; ++q) red[w][q] = d[q];
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      double s = 0.0;
      for (int k = 0; k < kVecThreads / 32; ++k) s += red[k][q];
      out[q] = s;
    }
  }
}

// Element loop of the vector kernels: CTA b owns complex elements [b*E, (b+1)*E), E = 8*32*12.
#define OK_VEC_LOOP(i)                                                             \
  const long long e0__ = (long long)blockIdx.x * (kBlocksPerCta * kBlock * 12);    \
  long long e1__ = e0__ + kBlocksPerCta * kBlock * 12;                             \
  if (e1__ > ncomplex) e1__ = ncomplex;                                            \
  for (long long i = e0__ + threadIdx.x; i < e1__; i += kVecThreads)

template <typename real> struct C2;
template <> struct C2<float> { using type = float2; };
template <> struct C2<double> { using type = double2; };

template <typename real>
__global__ void __launch_bounds__(kVecThreads)
k_init(const typename C2<real>::type* __restrict__ b, typename C2<real>::type* __restrict__ x,
       typename C2<real>::type* __restrict__ r, typename C2<real>::type* __restrict__ rhat,
       typename C2<real>::type* __restrict__ p, long long ncomplex, double* __restrict__ partials) {
  using c2 = typename C2<real>::type;
  double d[1] = {0.0};
  OK_VEC_LOOP(i) {
    c2 v = b[i];
    c2 z; z.x = 0; z.y = 0;
    x[i] = z; r[i] = v; rhat[i] = v; p[i] = v;
    d[0] += (double)v.x * v.x + (double)v.y * v.y;
  }
  block_reduce<1>(d, partials + (size_t)blockIdx.x * 3);
}

template <typename real>
__global__ void __launch_bounds__(kVecThreads)
k_s_update(const typename C2<real>::type* __restrict__ r, const typename C2<real>::type* __restrict__ v,
           typename C2<real>::type* __restrict__ s, long long ncomplex, const Scal* __restrict__ sc) {
  using c2 = typename C2<real>::type;
  const double ar = sc->alpha[0], ai = sc->alpha[1];
  OK_VEC_LOOP(i) {
    c2 rv = r[i], vv = v[i];
    c2 o;
    o.x = (real)((double)rv.x - (ar * vv.x - ai * vv.y));
    o.y = (real)((double)rv.y - (ar * vv.y + ai * vv.x));
    s[i] = o;
  }
}

// x += alpha p + omega s ; r = s - omega t ; partials: ||r||^2, <rhat, r>
template <typename real>
__global__ void __launch_bounds__(kVecThreads)
k_xr_update(typename C2<real>::type* __restrict__ x, const typename C2<real>::type* __restrict__ p,
            const typename C2<real>::type* __restrict__ s, const typename C2<real>::type* __restrict__ t,
            typename C2<real>::type* __restrict__ r, const typename C2<real>::type* __restrict__ rhat,
            long long ncomplex, const Scal* __restrict__ sc, double* __restrict__ partials) {
  using c2 = typename C2<real>::type;
  const double ar = sc->alpha[0], ai = sc->alpha[1], wr = sc->omega[0], wi = sc->omega[1];
  double d[3] = {0.0, 0.0, 0.0};
  OK_VEC_LOOP(i) {
    c2 xv = x[i], pv = p[i], sv = s[i], tv = t[i], hv = rhat[i];
    c2 xo, ro;
    xo.x = (real)((double)xv.x + (ar * pv.x - ai * pv.y) + (wr * sv.x - wi * sv.y));
    xo.y = (real)((double)xv.y + (ar * pv.y + ai * pv.x) + (wr * sv.y + wi * sv.x));
    ro.x = (real)((double)sv.x - (wr * tv.x - wi * tv.y));
    ro.y = (real)((double)sv.y - (wr * tv.y + wi * tv.x));
    x[i] = xo;
    r[i] = ro;
    d[0] += (double)ro.x * ro.x + (double)ro.y * ro.y;
    d[1] += (double)hv.x * ro.x + (double)hv.y * ro.y;   // Re conj(rhat) r
    d[2] += (double)hv.x * ro.y - (double)hv.y * ro.x;   // Im conj(rhat) r
  }
  block_reduce<3>(d, partials + (size_t)blockIdx.x * 3);
}

template <typename real>
__global__ void __launch_bounds__(kVecThreads)
k_p_update(typename C2<real>::type* __restrict__ p, const typename C2<real>::type* __restrict__ r,
           const typename C2<real>::type* __restrict__ v, long long ncomplex, const Scal* __restrict__ sc) {
  using c2 = typename C2<real>::type;
  const double br = sc->beta[0], bi = sc->beta[1], wr = sc->omega[0], wi = sc->omega[1];
  OK_VEC_LOOP(i) {
    c2 pv = p[i], rv = r[i], vv = v[i];
    const double qr = (double)pv.x - (wr * vv.x - wi * vv.y);
    const double qi = (double)pv.y - (wr * vv.y + wi * vv.x);
    c2 o;
    o.x = (real)((double)rv.x + (br * qr - bi * qi));
    o.y = (real)((double)rv.y + (br * qi + bi * qr));
    p[i] = o;
  }
}

// r = b - Mx ; optionally rhat = p = r (restart) ; partial ||r||^2
template <typename real>
__global__ void __launch_bounds__(kVecThreads)
k_residual(const typename C2<real>::type* __restrict__ b, const typename C2<real>::type* __restrict__ Mx,
           typename C2<real>::type* __restrict__ r, typename C2<real>::type* __restrict__ rhat,
           typename C2<real>::type* __restrict__ p, long long ncomplex, double* __restrict__ partials) {
  using c2 = typename C2<real>::type;
  double d[1] = {0.0};
  OK_VEC_LOOP(i) {
    c2 bv = b[i], mv = Mx[i];
    c2 o;
    o.x = (real)((double)bv.x - (double)mv.x);
    o.y = (real)((double)bv.y - (double)mv.y);
    r[i] = o; rhat[i] = o; p[i] = o;
    d[0] += (double)o.x * o.x + (double)o.y * o.y;
  }
  block_reduce<1>(d, partials + (size_t)blockIdx.x * 3);
}

// ---- single-CTA finalisers: sum `count` partial triples in fixed order, update the scalars ---
enum Stage { FIN_INIT = 0, FIN_V = 1, FIN_T = 2, FIN_XR = 3, FIN_RES = 4 };

// the BiCGStab scalars from the three totals of a reduction stage (one thread)
template <int STAGE>
__device__ __forceinline__ void update_scalars(const double (&tot)[3], Scal* sc) {
  if (STAGE == FIN_INIT) {
    sc->bnorm2 = tot[0]; sc->rr = tot[0];
    sc->rho[0] = tot[0]; sc->rho[1] = 0.0;
    sc->breakdown = 0;
  } else if (STAGE == FIN_RES) {   // after a true-residual recomputation (restart state)
    sc->rr = tot[0];
    sc->rho[0] = tot[0]; sc->rho[1] = 0.0;
    sc->breakdown = 0;
  } else if (STAGE == FIN_V) {     // apply epilogue gave (Re<rhat,v>, Im<rhat,v>, ||v||^2)
    const double vr = tot[0], vi = tot[1];
    int bd = (bad(vr, vi) || bad(sc->rho[0], sc->rho[1])) ? 1 : 0;
    const double den = vr * vr + vi * vi;
    sc->alpha[0] = (sc->rho[0] * vr + sc->rho[1] * vi) / den;
    sc->alpha[1] = (sc->rho[1] * vr - sc->rho[0] * vi) / den;
    sc->breakdown |= bd;
  } else if (STAGE == FIN_T) {     // (Re<s,t>, Im<s,t>, ||t||^2);  <t,s> = conj<s,t>
    const double tt = tot[2];
    sc->tt = tt;
    if (bad(tt, 0.0)) sc->breakdown |= 2;
    sc->omega[0] = tot[0] / tt;
    sc->omega[1] = -tot[1] / tt;
  } else if (STAGE == FIN_XR) {    // (||r||^2, Re<rhat,r>, Im<rhat,r>)
    sc->rr = tot[0];
    const double nr = tot[1], ni = tot[2];
    if (bad(sc->omega[0], sc->omega[1]) || bad(nr, ni)) sc->breakdown |= 4;
    // beta = (rho'/rho) (alpha/omega)
    const double r0 = sc->rho[0], r1 = sc->rho[1];
    double den = r0 * r0 + r1 * r1;
    const double q0 = (nr * r0 + ni * r1) / den, q1 = (ni * r0 - nr * r1) / den;
    const double w0 = sc->omega[0], w1 = sc->omega[1];
    den = w0 * w0 + w1 * w1;
    const double a0 = (sc->alpha[0] * w0 + sc->alpha[1] * w1) / den, a1 = (sc->alpha[1] * w0 - sc->alpha[0] * w1) / den;
    sc->beta[0] = q0 * a0 - q1 * a1;
    sc->beta[1] = q0 * a1 + q1 * a0;
    sc->rho[0] = nr; sc->rho[1] = ni;
  }
}

template <int STAGE>
__global__ void __launch_bounds__(kVecThreads) k_finalize(const double* __restrict__ partials, int count, Scal* sc) {
  // thread-serial sum in a fixed order; the loads of 8 consecutive strides are issued together (latency, not order, changes)
  constexpr bool kThree = STAGE == FIN_V || STAGE == FIN_T || STAGE == FIN_XR;
  double d[3] = {0.0, 0.0, 0.0};
  int i = threadIdx.x;
  for (; i + 7 * kVecThreads < count; i += 8 * kVecThreads) {
    double v[8][3];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const double* q = partials + (size_t)(i + u * kVecThreads) * 3;
      v[u][0] = q[0];
      v[u][1] = kThree ? q[1] : 0.0;
      v[u][2] = kThree ? q[2] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) { d[0] += v[u][0]; d[1] += v[u][1]; d[2] += v[u][2]; }
  }
  for (; i < count; i += kVecThreads) {
    d[0] += partials[(size_t)i * 3 + 0];
    if (kThree) {
      d[1] += partials[(size_t)i * 3 + 1];
      d[2] += partials[(size_t)i * 3 + 2];
    }
  }
  __shared__ double tot[3];
  block_reduce<3>(d, tot);
  if (threadIdx.x != 0) return;
  update_scalars<STAGE>(tot, sc);
}

// -------------------------------------------------------------------------------------------
static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

size_t bicgstab_work_bytes(const ok_params* p) {
  if (p->nrhs != 1) return 0;
  Geom g = make_geom(p);
  size_t vb = align_up((size_t)g.nblk * kBlock * 24 * real_bytes(p), 256);
  size_t parts = align_up((size_t)g.nblk * 3 * sizeof(double), 256);
  return 6 * vb + parts + 256;
}

template <typename real>
static int solve(const ok_params* p, const void* W, const void* src, void* xout, double tol, int maxit, int* iters,
                 double* resid) {
  using c2 = typename C2<real>::type;
  Geom g = make_geom(p);
  cudaStream_t st = ctx().stream;
  const long long ncomplex = (long long)g.nblk * kBlock * 12;
  const size_t vb = align_up((size_t)ncomplex * 2 * sizeof(real), 256);
  char* w = static_cast<char*>(ctx().work);
  c2* r = reinterpret_cast<c2*>(w + 0 * vb);
  c2* rhat = reinterpret_cast<c2*>(w + 1 * vb);
  c2* pp = reinterpret_cast<c2*>(w + 2 * vb);
  c2* v = reinterpret_cast<c2*>(w + 3 * vb);
  c2* s = reinterpret_cast<c2*>(w + 4 * vb);
  c2* t = reinterpret_cast<c2*>(w + 5 * vb);
  double* partials = reinterpret_cast<double*>(w + 6 * vb);
  Scal* sc = reinterpret_cast<Scal*>(w + 6 * vb + align_up((size_t)g.nblk * 3 * sizeof(double), 256));
  const c2* b = static_cast<const c2*>(src);
  c2* x = static_cast<c2*>(xout);
  const int ngrp = (g.nblk + kBlocksPerCta - 1) / kBlocksPerCta;

  static Scal* h = nullptr;   // pinned host mirror of the scalars (host memory, allocated once)
  static cudaEvent_t ev = nullptr;
  if (!h) OK_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&h), sizeof(Scal), cudaHostAllocDefault));
  if (!ev) OK_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));

  auto fetch = [&]() -> int {   // scalars -> host; later kernels may already be queued behind it
    OK_CUDA(cudaMemcpyAsync(h, sc, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaEventRecord(ev, st));
    return OK_SUCCESS;
  };
  auto wait = [&]() -> int {
    OK_CUDA(cudaEventSynchronize(ev));
    return OK_SUCCESS;
  };
  int rc;
#define OK_TRY(e) do { if ((rc = (e))) return rc; } while (0)

  k_init<real><<<ngrp, kVecThreads, 0, st>>>(b, x, r, rhat, pp, ncomplex, partials);
  OK_LAUNCHED("k_init");
  k_finalize<FIN_INIT><<<1, kVecThreads, 0, st>>>(partials, ngrp, sc);
  OK_LAUNCHED("k_finalize");
  OK_TRY(fetch());
  OK_TRY(wait());
  const double bnorm2 = h->bnorm2;
  *iters = 0;
  if (!(bnorm2 > 0.0)) {   // b = 0 -> x = 0
    *resid = 0.0;
    return isnan(bnorm2) ? OK_EBREAKDOWN : OK_SUCCESS;
  }
  const double target = tol * tol * bnorm2;

  auto true_residual = [&]() -> int {   // r = rhat = p = b - M x ; rr, rho reset ; host gets rr
    OK_TRY(launch_apply(p, W, x, t, nullptr, nullptr, nullptr));
    k_residual<real><<<ngrp, kVecThreads, 0, st>>>(b, t, r, rhat, pp, ncomplex, partials);
    OK_LAUNCHED("k_residual");
    k_finalize<FIN_RES><<<1, kVecThreads, 0, st>>>(partials, ngrp, sc);
    OK_LAUNCHED("k_finalize");
    OK_TRY(fetch());
    OK_TRY(wait());
    return OK_SUCCESS;
  };

  int status = OK_EMAXIT;
  int it = 0;
  while (it < maxit) {
    ++it;
    OK_TRY(launch_apply(p, W, pp, v, partials, rhat, nullptr));   // v = M p, partials <- <rhat,v>
    k_finalize<FIN_V><<<1, kVecThreads, 0, st>>>(partials, g.nblk, sc);
    OK_LAUNCHED("k_finalize");
    k_s_update<real><<<ngrp, kVecThreads, 0, st>>>(r, v, s, ncomplex, sc);
    OK_LAUNCHED("k_s_update");
    OK_TRY(launch_apply(p, W, s, t, partials, s, nullptr));       // t = M s, partials <- <s,t>, <t,t>
    k_finalize<FIN_T><<<1, kVecThreads, 0, st>>>(partials, g.nblk, sc);
    OK_LAUNCHED("k_finalize");
    k_xr_update<real><<<ngrp, kVecThreads, 0, st>>>(x, pp, s, t, r, rhat, ncomplex, sc, partials);
    OK_LAUNCHED("k_xr_update");
    k_finalize<FIN_XR><<<1, kVecThreads, 0, st>>>(partials, ngrp, sc);
    OK_LAUNCHED("k_finalize");
    OK_TRY(fetch());
    // the p update does not need the host: queue it behind the read-back so the GPU stays busy
    k_p_update<real><<<ngrp, kVecThreads, 0, st>>>(pp, r, v, ncomplex, sc);
    OK_LAUNCHED("k_p_update");
    OK_TRY(wait());
    if (h->breakdown & 3) { status = OK_EBREAKDOWN; break; }
    if (h->rr <= target) {
      OK_TRY(true_residual());
      if (h->rr <= target) { status = OK_SUCCESS; break; }
      continue;   // restarted from the true residual
    }
    if ((h->breakdown & 4) || isnan(h->rr)) { status = OK_EBREAKDOWN; break; }
  }
  if (status != OK_SUCCESS) OK_TRY(true_residual());   // report the true residual in every case
  *iters = it;
  *resid = sqrt(h->rr / bnorm2);
#undef OK_TRY
  return status;
}

int run_bicgstab(const ok_params* p, const void* W, const void* src, void* x, double tol, int maxit, int* iters,
                 double* resid) {
  if (p->nrhs != 1) return OK_EINVAL;
  if (p->precision == OK_FP64) return solve<double>(p, W, src, x, tol, maxit, iters, resid);
  return solve<float>(p, W, src, x, tol, maxit, iters, resid);
}

// =====================================================================================================
// t-slab decomposition: the same BiCGStab over a lattice cut along T into slabs.
// "In the temporal direction, only the nearest neighbors are involved" and "off-node communications are
// necessary only for the outermost boundary surfaces": W is slab-local, a slab's fields carry one halo
// time slice below and above (ok.h); an apply reads its t-neighbours' boundary slices in place where they belong to a slab
// of this process (fused halo loads, apply_direct_kernel<.., PEER>) and from the halo slices filled by the caller's
// `exchange` at the two outer faces of the process.  Reductions:
// per-CTA partials (as above) -> one fixed-order total per SLAB -> (all-gather over processes) -> sum over all slabs in
// global slab order -> scalars.  The result therefore depends on the number of slabs, not on how they are dealt to
// processes; every process computes identical scalars.
template <bool THREE>
__global__ void __launch_bounds__(kVecThreads)
k_slab_sum(const double* __restrict__ partials, const int* __restrict__ first, const int* __restrict__ count, double* __restrict__ slabtot) {
  const double* q = partials + (size_t)first[blockIdx.x] * 3;
  const int n = count[blockIdx.x];
  double d[3] = {0.0, 0.0, 0.0};
  for (int i = threadIdx.x; i < n; i += kVecThreads) {
    d[0] += q[(size_t)i * 3 + 0];
    if (THREE) {
      d[1] += q[(size_t)i * 3 + 1];
      d[2] += q[(size_t)i * 3 + 2];
    }
  }
  block_reduce<3>(d, slabtot + (size_t)blockIdx.x * 3);
}

template <int STAGE>
__global__ void k_slab_scalars(const double* __restrict__ slabtot, int nslab_all, Scal* sc) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double tot[3] = {0.0, 0.0, 0.0};
  for (int i = 0; i < nslab_all; ++i) {   // global slab order
    tot[0] += slabtot[(size_t)i * 3 + 0];
    tot[1] += slabtot[(size_t)i * 3 + 1];
    tot[2] += slabtot[(size_t)i * 3 + 2];
  }
  update_scalars<STAGE>(tot, sc);
}

size_t bicgstab_slab_work_bytes(const ok_params* p) {   // per slab; p: the slab's own lattice
  if (p->nrhs != 1) return 0;
  Geom g = make_geom(p);
  const size_t slice = (size_t)p->dims[0] * p->dims[1] * p->dims[2];
  const size_t vb = align_up(((size_t)g.V + 2 * slice) * 24 * real_bytes(p), 256);
  return 6 * vb + align_up((size_t)g.nblk * 3 * sizeof(double), 256);
}
size_t bicgstab_slab_shared_bytes(int nslab, int nranks) {   // once per solve
  return align_up((size_t)nslab * 3 * sizeof(int), 256) + align_up((size_t)nslab * 3 * sizeof(double), 256) +
         align_up((size_t)nslab * (size_t)nranks * 3 * sizeof(double), 256) + 256;
}

template <typename real>
static int solve_slabs(int nslab, const ok_params* const* ps, const void* const* Ws, const void* const* srcs, void* const* xs, double tol,
                       int maxit, const ok_comm* comm, int* iters, double* resid) {
  using c2 = typename C2<real>::type;
  cudaStream_t st = ctx().stream;
  const int nranks = comm ? comm->nranks : 1;
  struct Slab {
    const ok_params* p;
    const void* W;
    Geom g;
    long long halo, ncomplex;   // complex elements of one time slice; of the interior
    size_t slice_bytes;
    int ngrp, pfirst;
    c2 *r, *rhat, *pp, *v, *s, *t, *x;   // extended fields (base pointers)
    const c2* b;
  };
  Slab sl[64];
  if (nslab < 1 || nslab > 64) return OK_EINVAL;
  char* w = static_cast<char*>(ctx().work);
  size_t need = 0;
  int nblk_all = 0;
  for (int i = 0; i < nslab; ++i) {
    Slab& a = sl[i];
    a.p = ps[i];
    a.W = Ws[i];
    a.g = make_geom(ps[i]);
    a.halo = (long long)ps[i]->dims[0] * ps[i]->dims[1] * ps[i]->dims[2] * 12;
    a.ncomplex = (long long)a.g.V * 12;
    a.slice_bytes = (size_t)a.halo * 2 * sizeof(real);
    a.ngrp = (a.g.nblk + kBlocksPerCta - 1) / kBlocksPerCta;
    a.pfirst = nblk_all;
    nblk_all += a.g.nblk;
    const size_t vb = align_up((size_t)(a.ncomplex + 2 * a.halo) * 2 * sizeof(real), 256);
    c2** f[6] = {&a.r, &a.rhat, &a.pp, &a.v, &a.s, &a.t};
    for (int k = 0; k < 6; ++k) {
      *f[k] = reinterpret_cast<c2*>(w + need);
      need += vb;
    }
    a.x = static_cast<c2*>(xs[i]);
    a.b = static_cast<const c2*>(srcs[i]);
    if (i > 0 && (ps[i]->dims[0] != ps[0]->dims[0] || ps[i]->dims[1] != ps[0]->dims[1] || ps[i]->dims[2] != ps[0]->dims[2])) return OK_EINVAL;
  }
  double* partials = reinterpret_cast<double*>(w + need);
  need += align_up((size_t)nblk_all * 3 * sizeof(double), 256);
  int* d_first = reinterpret_cast<int*>(w + need);          // [nslab] first partial triple of a slab
  int* d_cnt_apply = d_first + nslab;                       // [nslab] triples written by the apply (one per 32-site block)
  int* d_cnt_vec = d_first + 2 * nslab;                     // [nslab] triples written by a vector kernel (one per CTA)
  need += align_up((size_t)nslab * 3 * sizeof(int), 256);
  double* slabtot = reinterpret_cast<double*>(w + need);    // [nslab][3]
  need += align_up((size_t)nslab * 3 * sizeof(double), 256);
  double* gathered = reinterpret_cast<double*>(w + need);   // [nranks][nslab][3]
  need += align_up((size_t)nslab * nranks * 3 * sizeof(double), 256);
  Scal* sc = reinterpret_cast<Scal*>(w + need);
  need += 256;
  if (!ctx().work || ctx().work_bytes < need) return OK_EWORKSPACE;
  {
    int hbuf[3 * 64];
    for (int i = 0; i < nslab; ++i) {
      hbuf[i] = sl[i].pfirst;
      hbuf[nslab + i] = sl[i].g.nblk;
      hbuf[2 * nslab + i] = sl[i].ngrp;
    }
    OK_CUDA(cudaMemcpyAsync(d_first, hbuf, (size_t)nslab * 3 * sizeof(int), cudaMemcpyHostToDevice, st));   // pageable source: copied before return
  }

  static Scal* h = nullptr;
  static cudaEvent_t ev = nullptr;
  if (!h) OK_CUDA(cudaHostAlloc(reinterpret_cast<void**>(&h), sizeof(Scal), cudaHostAllocDefault));
  if (!ev) OK_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
  int rc;
#define OK_TRY(e) do { if ((rc = (e))) return rc; } while (0)
  auto fetch = [&]() -> int {
    OK_CUDA(cudaMemcpyAsync(h, sc, sizeof(Scal), cudaMemcpyDeviceToHost, st));
    OK_CUDA(cudaEventRecord(ev, st));
    return OK_SUCCESS;
  };
  auto wait = [&]() -> int {
    OK_CUDA(cudaEventSynchronize(ev));
    return OK_SUCCESS;
  };
  // one reduction stage: slab totals -> all slabs of all processes in global order -> scalars
  auto finalize = [&](int stage, bool from_apply) -> int {
    const bool three = stage == FIN_V || stage == FIN_T || stage == FIN_XR;
    const int* cnt = from_apply ? d_cnt_apply : d_cnt_vec;
    if (three) k_slab_sum<true><<<nslab, kVecThreads, 0, st>>>(partials, d_first, cnt, slabtot);
    else k_slab_sum<false><<<nslab, kVecThreads, 0, st>>>(partials, d_first, cnt, slabtot);
    OK_LAUNCHED("k_slab_sum");
    const double* all = slabtot;
    if (comm && comm->allgather) {
      if (comm->allgather(comm->user, slabtot, gathered, 3 * nslab)) return OK_ECOMM;
      all = gathered;
    }
    const int n = nslab * nranks;
    switch (stage) {
      case FIN_INIT: k_slab_scalars<FIN_INIT><<<1, 32, 0, st>>>(all, n, sc); break;
      case FIN_V: k_slab_scalars<FIN_V><<<1, 32, 0, st>>>(all, n, sc); break;
      case FIN_T: k_slab_scalars<FIN_T><<<1, 32, 0, st>>>(all, n, sc); break;
      case FIN_XR: k_slab_scalars<FIN_XR><<<1, 32, 0, st>>>(all, n, sc); break;
      default: k_slab_scalars<FIN_RES><<<1, 32, 0, st>>>(all, n, sc); break;
    }
    OK_LAUNCHED("k_slab_scalars");
    return OK_SUCCESS;
  };
  // The t-faces of one field of every slab.  Slabs of this process read each other's boundary slices in place (the apply's
  // PEER loads, ok_slab_dirac_apply_peer): nothing is copied for them.  Only the two outer faces of the process arrive through
  // the caller's `exchange`, into the lower halo slice of the first slab and the upper halo slice of the last one; without
  // comm the process holds the whole T extent and the periodic closure is one more in-place read (the boundary condition
  // sits in W).  lo[i] / hi[i]: where slab i finds psi(x - t) of its first slice and psi(x + t) of its last one.
  const char* face_lo[64];
  const char* face_hi[64];
  auto faces = [&](c2* Slab::*field) -> int {
    auto lo_halo = [&](Slab& a) { return reinterpret_cast<char*>(a.*field); };
    auto first_slice = [&](Slab& a) { return reinterpret_cast<char*>(a.*field) + a.slice_bytes; };
    auto last_slice = [&](Slab& a) { return reinterpret_cast<char*>(a.*field) + (size_t)a.p->dims[3] * a.slice_bytes; };
    auto hi_halo = [&](Slab& a) { return reinterpret_cast<char*>(a.*field) + (size_t)(a.p->dims[3] + 1) * a.slice_bytes; };
    const size_t nb = sl[0].slice_bytes;
    for (int i = 0; i < nslab; ++i) {
      face_lo[i] = i > 0 ? last_slice(sl[i - 1]) : nullptr;
      face_hi[i] = i + 1 < nslab ? first_slice(sl[i + 1]) : nullptr;
    }
    Slab &a0 = sl[0], &a1 = sl[nslab - 1];
    const ok_slab_peers* pr = slab_peers();
    if (comm && comm->exchange && pr) {
      // peer access (ok_slab_set_peers): the outer faces too are read in place, from the neighbour processes' memory.  Every
      // process has the same workspace layout (equal slabs, the same number per process), so the lower neighbour's last slab
      // keeps its field where this process's last slab keeps its own, and x is the caller's buffer named in the peers.
      if (pr->barrier(pr->user)) return OK_ECOMM;
      auto remote = [&](const void* peer_work, const void* peer_x, const char* mine, const Slab& a) -> const char* {
        const char* wb = static_cast<const char*>(ctx().work);
        if (mine >= wb && mine < wb + ctx().work_bytes) return static_cast<const char*>(peer_work) + (mine - wb);
        return static_cast<const char*>(peer_x) + (mine - reinterpret_cast<const char*>(a.x));
      };
      face_lo[0] = remote(pr->lo_work, pr->lo_x, last_slice(a1), a1);
      face_hi[nslab - 1] = remote(pr->hi_work, pr->hi_x, first_slice(a0), a0);
    } else if (comm && comm->exchange) {
      if (comm->exchange(comm->user, first_slice(a0), last_slice(a1), lo_halo(a0), hi_halo(a1), nb)) return OK_ECOMM;
      face_lo[0] = lo_halo(a0);
      face_hi[nslab - 1] = hi_halo(a1);
    } else {
      face_lo[0] = last_slice(a1);
      face_hi[nslab - 1] = first_slice(a0);
    }
    return OK_SUCCESS;
  };
#define OK_INT(a, f) ((a).f + (a).halo)   /* interior of an extended field */
  for (int i = 0; i < nslab; ++i) {
    Slab& a = sl[i];
    k_init<real><<<a.ngrp, kVecThreads, 0, st>>>(OK_INT(a, b), OK_INT(a, x), OK_INT(a, r), OK_INT(a, rhat), OK_INT(a, pp), a.ncomplex,
                                               partials + (size_t)a.pfirst * 3);
    OK_LAUNCHED("k_init");
  }
  OK_TRY(finalize(FIN_INIT, false));
  OK_TRY(fetch());
  OK_TRY(wait());
  const double bnorm2 = h->bnorm2;
  *iters = 0;
  if (!(bnorm2 > 0.0)) {
    *resid = 0.0;
    return isnan(bnorm2) ? OK_EBREAKDOWN : OK_SUCCESS;
  }
  const double target = tol * tol * bnorm2;
  auto apply_all = [&](c2* Slab::*in, c2* Slab::*out, c2* Slab::*dot) -> int {
    OK_TRY(faces(in));
    for (int i = 0; i < nslab; ++i) {
      Slab& a = sl[i];
      OK_TRY(launch_apply_slab(a.p, a.W, a.*in, a.*out, dot ? partials + (size_t)a.pfirst * 3 : nullptr, dot ? a.*dot : nullptr,
                               face_lo[i], face_hi[i]));
    }
    return OK_SUCCESS;
  };
  auto true_residual = [&]() -> int {
    OK_TRY(apply_all(&Slab::x, &Slab::t, nullptr));
    for (int i = 0; i < nslab; ++i) {
      Slab& a = sl[i];
      k_residual<real><<<a.ngrp, kVecThreads, 0, st>>>(OK_INT(a, b), OK_INT(a, t), OK_INT(a, r), OK_INT(a, rhat), OK_INT(a, pp), a.ncomplex,
                                                     partials + (size_t)a.pfirst * 3);
      OK_LAUNCHED("k_residual");
    }
    OK_TRY(finalize(FIN_RES, false));
    OK_TRY(fetch());
    OK_TRY(wait());
    return OK_SUCCESS;
  };
  int status = OK_EMAXIT;
  int it = 0;
  while (it < maxit) {
    ++it;
    OK_TRY(apply_all(&Slab::pp, &Slab::v, &Slab::rhat));   // v = M p, <rhat,v>
    OK_TRY(finalize(FIN_V, true));
    for (int i = 0; i < nslab; ++i) {
      Slab& a = sl[i];
      k_s_update<real><<<a.ngrp, kVecThreads, 0, st>>>(OK_INT(a, r), OK_INT(a, v), OK_INT(a, s), a.ncomplex, sc);
      OK_LAUNCHED("k_s_update");
    }
    OK_TRY(apply_all(&Slab::s, &Slab::t, &Slab::s));       // t = M s, <s,t>, <t,t>
    OK_TRY(finalize(FIN_T, true));
    for (int i = 0; i < nslab; ++i) {
      Slab& a = sl[i];
      k_xr_update<real><<<a.ngrp, kVecThreads, 0, st>>>(OK_INT(a, x), OK_INT(a, pp), OK_INT(a, s), OK_INT(a, t), OK_INT(a, r), OK_INT(a, rhat),
                                                      a.ncomplex, sc, partials + (size_t)a.pfirst * 3);
      OK_LAUNCHED("k_xr_update");
    }
    OK_TRY(finalize(FIN_XR, false));
    OK_TRY(fetch());
    for (int i = 0; i < nslab; ++i) {
      Slab& a = sl[i];
      k_p_update<real><<<a.ngrp, kVecThreads, 0, st>>>(OK_INT(a, pp), OK_INT(a, r), OK_INT(a, v), a.ncomplex, sc);
      OK_LAUNCHED("k_p_update");
    }
    OK_TRY(wait());
    if (h->breakdown & 3) { status = OK_EBREAKDOWN; break; }
    if (h->rr <= target) {
      OK_TRY(true_residual());
      if (h->rr <= target) { status = OK_SUCCESS; break; }
      continue;
    }
    if ((h->breakdown & 4) || isnan(h->rr)) { status = OK_EBREAKDOWN; break; }
  }
  if (status != OK_SUCCESS) OK_TRY(true_residual());
  *iters = it;
  *resid = sqrt(h->rr / bnorm2);
#undef OK_INT
#undef OK_TRY
  return status;
}

int run_bicgstab_slabs(int nslab, const ok_params* const* ps, const void* const* Ws, const void* const* srcs, void* const* xs, double tol,
                       int maxit, const ok_comm* comm, int* iters, double* resid) {
  if (ps[0]->precision == OK_FP64) return solve_slabs<double>(nslab, ps, Ws, srcs, xs, tol, maxit, comm, iters, resid);
  return solve_slabs<float>(nslab, ps, Ws, srcs, xs, tol, maxit, comm, iters, resid);
}

}  // namespace okd
