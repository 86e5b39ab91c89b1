// Layout conversion kernels: canonical (ok.h) <-> site-blocked SoA internal layouts.
// One thread moves one 16-byte unit; the internal side is always the coalesced one.
#include "ok_internal.cuh"

namespace okd {

// Spinor.  Internal unit index u = (block*NC + c)*32 + s ; canonical unit index = n*NC + c,
// NC = units per site (fp32: 6 pairs of components, fp64: 12 components; nrhs=12: see below).
template <typename vec_t>
__global__ void pack_spinor_kernel(const vec_t* __restrict__ canon, vec_t* __restrict__ packed, int V, int nblk,
                                   int NC, bool unpack) {
  long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nblk * NC * kBlock;
  if (u >= total) return;
  int s = (int)(u % kBlock);
  int c = (int)((u / kBlock) % NC);
  int b = (int)(u / ((long long)kBlock * NC));
  int n = b * kBlock + s;
  if (unpack) {
    if (n < V) const_cast<vec_t*>(canon)[(long long)n * NC + c] = packed[u];
  } else {
    vec_t z = {};
    packed[u] = (n < V) ? canon[(long long)n * NC + c] : z;
  }
}

// nrhs = 12, fp32: canonical [n][comp][rhs] complex -> internal [block][comp][site][rhs] complex.
// Unit = float4 = two consecutive rhs; per (site, comp) there are 6 units.
__global__ void pack_spinor_mrhs_kernel(const float4* __restrict__ canon, float4* __restrict__ packed, int V,
                                        int nblk, bool unpack) {
  long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nblk * 12 * kBlock * 6;
  if (u >= total) return;
  int q = (int)(u % 6);
  int s = (int)((u / 6) % kBlock);
  int comp = (int)((u / (6 * kBlock)) % 12);
  int b = (int)(u / (6LL * kBlock * 12));
  int n = b * kBlock + s;
  long long cu = ((long long)n * 12 + comp) * 6 + q;
  if (unpack) {
    if (n < V) const_cast<float4*>(canon)[cu] = packed[u];
  } else {
    packed[u] = (n < V) ? canon[cu] : make_float4(0.f, 0.f, 0.f, 0.f);
  }
}

int launch_pack_spinor(const ok_params* p, const void* canon, void* packed, bool unpack) {
  Geom g = make_geom(p);
  const int T = 256;
  if (p->nrhs == 12) {
    long long total = (long long)g.nblk * 12 * kBlock * 6;
    pack_spinor_mrhs_kernel<<<(unsigned)((total + T - 1) / T), T, 0, ctx().stream>>>(
        static_cast<const float4*>(canon), static_cast<float4*>(packed), g.V, g.nblk, unpack);
    OK_LAUNCHED("pack_spinor_mrhs_kernel");
    return OK_SUCCESS;
  }
  int NC = p->precision == OK_FP64 ? 12 : 6;
  long long total = (long long)g.nblk * NC * kBlock;
  unsigned grid = (unsigned)((total + T - 1) / T);
  if (p->precision == OK_FP64)
    pack_spinor_kernel<double2><<<grid, T, 0, ctx().stream>>>(static_cast<const double2*>(canon),
                                                             static_cast<double2*>(packed), g.V, g.nblk, NC, unpack);
  else
    pack_spinor_kernel<float4><<<grid, T, 0, ctx().stream>>>(static_cast<const float4*>(canon),
                                                            static_cast<float4*>(packed), g.V, g.nblk, NC, unpack);
  OK_LAUNCHED("pack_spinor_kernel");
  return OK_SUCCESS;
}

// W.  Internal unit u = ((((b*27 + t)*12 + r)*NC + c)*32 + s ; canonical unit = ((n*27 + t)*12 + r)*NC + c.
template <typename vec_t>
__global__ void pack_W_kernel(const vec_t* __restrict__ canon, vec_t* __restrict__ packed, int V, long long total,
                              int NC, bool unpack) {
  long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= total) return;
  int s = (int)(u % kBlock);
  long long v = u / kBlock;
  int c = (int)(v % NC);
  v /= NC;
  int r = (int)(v % 12);
  v /= 12;
  int t = (int)(v % kTerms);
  int b = (int)(v / kTerms);
  int n = b * kBlock + s;
  long long cu = (((long long)n * kTerms + t) * 12 + r) * NC + c;
  if (unpack) {
    if (n < V) const_cast<vec_t*>(canon)[cu] = packed[u];
  } else {
    vec_t z = {};
    packed[u] = (n < V) ? canon[cu] : z;
  }
}

int launch_pack_W(const ok_params* p, const void* canon, void* Wp, bool unpack) {
  Geom g = make_geom(p);
  int NC = p->precision == OK_FP64 ? 12 : 6;
  long long total = (long long)g.nblk * kTerms * 12 * NC * kBlock;
  const int T = 256;
  unsigned grid = (unsigned)((total + T - 1) / T);
  if (p->precision == OK_FP64)
    pack_W_kernel<double2><<<grid, T, 0, ctx().stream>>>(static_cast<const double2*>(canon),
                                                        static_cast<double2*>(Wp), g.V, total, NC, unpack);
  else
    pack_W_kernel<float4><<<grid, T, 0, ctx().stream>>>(static_cast<const float4*>(canon), static_cast<float4*>(Wp),
                                                       g.V, total, NC, unpack);
  OK_LAUNCHED("pack_W_kernel");
  return OK_SUCCESS;
}

}  // namespace okd
