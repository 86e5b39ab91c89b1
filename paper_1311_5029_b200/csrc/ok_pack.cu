// Layout conversion kernels: canonical (ok.h) <-> site-blocked SoA internal layouts.
// One thread moves one 16-byte unit; the internal side is always the coalesced one.
#include "ok_internal.cuh"
#include "ok_sparse.cuh"

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

// nrhs = 12, fp32: canonical [n][comp][rhs][re,im] <-> the fp32 per-site records of the field (ok_internal.cuh,
// mrhs_vec_index).  One thread per complex number.  Packing then also writes the operand records (mrhs_ensure_operand).
__global__ void pack_spinor_mrhs_kernel(const float2* __restrict__ canon, float* __restrict__ packed, int V, bool unpack) {
  long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= (long long)V * 144) return;
  const int rhs = (int)(u % 12), comp = (int)((u / 12) % 12);
  const long long n = u / 144;
  float* rec = packed + n * kMrhsVecSiteFloats;
  const int ir = mrhs_vec_index(comp, rhs, 0), ii = mrhs_vec_index(comp, rhs, 1);
  if (unpack) {
    const_cast<float2*>(canon)[u] = make_float2(rec[ir], rec[ii]);
  } else {
    const float2 v = canon[u];
    rec[ir] = v.x;
    rec[ii] = v.y;
  }
}

// nrhs = 12 W: canonical [n][27][12][12][re,im] (fp32) <-> per-site split-fp16 B-operand tiles
// (ok_internal.cuh: mrhs_W_index, mrhs_split).  Packing keeps 22 significant bits of every real
// (|x - unpack(pack(x))| <= 2^-22 |x| for 2^-14 <= |x| <= 65504); the zero pad is written when packing.
__global__ void pack_W_mrhs_kernel(const float2* __restrict__ canon, __half* __restrict__ packed, int V, bool unpack) {
  constexpr int kPer = kTerms * 144 + 192;
  long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= (long long)V * kPer) return;
  const int e = (int)(u % kPer);
  const long long n = u / kPer;
  __half* tile = packed + n * kMrhsWSiteHalves;
  if (e >= kTerms * 144) {   // the 192 zero pad halves of the last stage
    if (!unpack) tile[mrhs_W_pad_index(e - kTerms * 144)] = __float2half_rn(0.f);
    return;
  }
  const int col = e % 12, row = (e / 12) % 12, term = e / 144;
  const int rh = mrhs_W_index(term, row, col, 0, 0), rl = mrhs_W_index(term, row, col, 0, 1);
  const int ih = mrhs_W_index(term, row, col, 1, 0), il = mrhs_W_index(term, row, col, 1, 1);
  const long long cu = n * (kTerms * 144) + e;
  if (unpack) {
    const_cast<float2*>(canon)[cu] = make_float2(mrhs_join(tile[rh], tile[rl]), mrhs_join(tile[ih], tile[il]));
  } else {
    const float2 v = canon[cu];
    mrhs_split(v.x, &tile[rh], &tile[rl]);
    mrhs_split(v.y, &tile[ih], &tile[il]);
  }
}

int launch_pack_spinor(const ok_params* p, const void* canon, void* packed, bool unpack) {
  Geom g = make_geom(p);
  const int T = 256;
  if (p->nrhs == 12) {
    long long total = (long long)g.V * 144;
    if (!unpack) OK_CUDA(cudaMemsetAsync(packed, 0, kMrhsVecHeaderBytes, ctx().stream));   // header: operand records not valid yet
    pack_spinor_mrhs_kernel<<<(unsigned)((total + T - 1) / T), T, 0, ctx().stream>>>(
        static_cast<const float2*>(canon), mrhs_f32(packed), g.V, unpack);
    OK_LAUNCHED("pack_spinor_mrhs_kernel");
    return unpack ? OK_SUCCESS : mrhs_ensure_operand(p, packed);
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

// Reduced formats (ok_sparse.cuh): canonical [n][27][12][12] <-> [block][unit][site 32][complex].  One thread per canonical
// element of a (padded) site.  Packing drops what the format does not keep (structural zeros; for OK_W_DS the implied
// quadrants LR, LL); unpacking rebuilds the full matrices (zeros, copies, LL = -S of W^0).
__constant__ int c_prun[3][kTerms][2][4];
__constant__ int8_t c_pkoff[kTerms][4];
static bool g_prun_ready = false;

template <typename cx>
__global__ void pack_W_sparse_kernel(const cx* __restrict__ canon, cx* __restrict__ packed, int V, int nblk, int fmt, bool unpack, Geom g) {
  const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long total = (long long)nblk * kBlock * kTerms * 144;
  if (e >= total) return;
  const int col = (int)(e % 12), row = (int)((e / 12) % 12), term = (int)((e / 144) % kTerms);
  const long long n = e / (144 * kTerms);
  const SparseRef r = sparse_ref(fmt, term, row, col, c_prun[fmt - 1]);
  long long ns = n;   // site that holds the stored value
  if (r.shift >= 0 && n < V) {   // OK_W_CONJ: the positive matrix of the neighbour site x + offset[term]
    int xc[4], q = (int)n;
    for (int dd = 0; dd < 3; ++dd) { xc[dd] = q % g.L[dd]; q /= g.L[dd]; }
    xc[3] = q;
    for (int dd = 0; dd < 4; ++dd) xc[dd] = (xc[dd] + c_pkoff[r.shift][dd] + g.L[dd]) % g.L[dd];
    ns = xc[0] + g.L[0] * (xc[1] + g.L[1] * (xc[2] + (long long)g.L[2] * xc[3]));
  }
  cx* dst = r.unit < 0 ? nullptr : packed + ((size_t)(ns >> 5) * sparse_site_units_rt(fmt) + r.unit) * kBlock + (ns & 31);
  if (unpack) {
    if (n >= V) return;
    cx v = {};
    if (dst) { v = *dst; v.x *= r.sign; v.y *= r.conj ? -r.sign : r.sign; }
    const_cast<cx*>(canon)[e] = v;
  } else if (dst && r.stored) {
    cx v = {};
    if (n < V) v = canon[e];
    *dst = v;
  }
}

static int launch_pack_W_sparse(const ok_params* p, const void* canon, void* Wp, bool unpack) {
  if (!g_prun_ready) {
    static int h[3][kTerms][2][4];
    for (int f = 0; f < 3; ++f) sparse_fill_runs(f + 1, h[f]);
    OK_CUDA(cudaMemcpyToSymbol(c_prun, h, sizeof(h)));
    OK_CUDA(cudaMemcpyToSymbol(c_pkoff, kOffsets, sizeof(kOffsets)));
    g_prun_ready = true;
  }
  Geom g = make_geom(p);
  const long long total = (long long)g.nblk * kBlock * kTerms * 144;
  const unsigned grid = (unsigned)((total + 255) / 256);
  if (p->precision == OK_FP64)
    pack_W_sparse_kernel<double2><<<grid, 256, 0, ctx().stream>>>(static_cast<const double2*>(canon), static_cast<double2*>(Wp), g.V, g.nblk, p->storage, unpack, g);
  else
    pack_W_sparse_kernel<float2><<<grid, 256, 0, ctx().stream>>>(static_cast<const float2*>(canon), static_cast<float2*>(Wp), g.V, g.nblk, p->storage, unpack, g);
  OK_LAUNCHED("pack_W_sparse_kernel");
  return OK_SUCCESS;
}

int launch_pack_W(const ok_params* p, const void* canon, void* Wp, bool unpack) {
  Geom g = make_geom(p);
  if (p->nrhs == 1 && p->storage != OK_W_DENSE) return launch_pack_W_sparse(p, canon, Wp, unpack);
  if (p->nrhs == 12) {
    long long tot = (long long)g.V * (kTerms * 144 + 192);
    pack_W_mrhs_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, ctx().stream>>>(static_cast<const float2*>(canon),
                                                                                static_cast<__half*>(Wp), g.V, unpack);
    OK_LAUNCHED("pack_W_mrhs_kernel");
    return OK_SUCCESS;
  }
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
