// Single-RHS Oktay-Kronfeld Dirac apply, Eq. (2.2):
//   out(x) = sum_{term=0..26} W_term(x) psi(x + offset_term)      (coordinates modulo dims)
//
// HBM-bound: 31 104 B (fp32) of W per site are read exactly once, against 96 B of psi and
// 96 B of out.  Layout (ok.h): W [block][term][row][c][site 32][16 B]; lane <-> site, so every
// warp-wide W load is one contiguous 512-B line and a (block, term) tile is contiguous.
//
// Variant "direct" (this file): CTA = 12/RPT warps, warp g owns output rows g*RPT..g*RPT+RPT-1
// of the CTA's 32 sites.  W goes global -> registers with streaming (evict-first) 16-B loads;
// the neighbour spinor is gathered through L1/L2 (psi is L2 resident); complex 12x12 matvec in
// registers; optional fused reduction epilogue for BiCGStab (<a,out>, ||out||^2 per CTA, fixed order).
#include "ok_internal.cuh"

namespace okd {

__constant__ int8_t c_off[kTerms][4];
static bool g_off_uploaded = false;

static int upload_offsets() {
  if (g_off_uploaded) return OK_SUCCESS;
  OK_CUDA(cudaMemcpyToSymbol(c_off, kOffsets, sizeof(kOffsets)));
  g_off_uploaded = true;
  return OK_SUCCESS;
}

template <typename real> struct Vec;
template <> struct Vec<float> { using type = float4; static constexpr int NC = 6; };
template <> struct Vec<double> { using type = double2; static constexpr int NC = 12; };

// acc[0..1] (re, im) += (row of W restricted to this unit) * (spinor unit)
__device__ __forceinline__ void cmac(float (&a)[2], const float4& w, const float4& s) {
  a[0] = fmaf(w.x, s.x, a[0]); a[0] = fmaf(-w.y, s.y, a[0]);
  a[0] = fmaf(w.z, s.z, a[0]); a[0] = fmaf(-w.w, s.w, a[0]);
  a[1] = fmaf(w.x, s.y, a[1]); a[1] = fmaf(w.y, s.x, a[1]);
  a[1] = fmaf(w.z, s.w, a[1]); a[1] = fmaf(w.w, s.z, a[1]);
}
__device__ __forceinline__ void cmac(double (&a)[2], const double2& w, const double2& s) {
  a[0] = fma(w.x, s.x, a[0]); a[0] = fma(-w.y, s.y, a[0]);
  a[1] = fma(w.x, s.y, a[1]); a[1] = fma(w.y, s.x, a[1]);
}

__device__ __forceinline__ int wrap(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

// PEER (t-slab only, ok_slab_dirac_apply_peer): the two halo time slices of the extended field are not read from psi but from
// lo_peer / hi_peer -- the t-neighbours' own boundary slices, wherever they live (another slab's field on this GPU, or a
// neighbour GPU's memory mapped through NVLink peer access): the halo exchange is the apply's own loads, no copy, no staging.
template <typename real, int RPT, bool DOT, bool PEER = false>
__global__ void __launch_bounds__(32 * (12 / RPT))
apply_direct_kernel(const typename Vec<real>::type* __restrict__ W, const typename Vec<real>::type* __restrict__ psi,
                    typename Vec<real>::type* __restrict__ out, Geom g, int vblk0,
                    const typename Vec<real>::type* __restrict__ dot_a, double* __restrict__ partials,
                    const typename Vec<real>::type* __restrict__ lo_peer = nullptr,
                    const typename Vec<real>::type* __restrict__ hi_peer = nullptr) {
  using vec_t = typename Vec<real>::type;
  constexpr int NC = Vec<real>::NC;
  constexpr int NW = 12 / RPT;
  const int lane = threadIdx.x & 31;
  const int rg = threadIdx.x >> 5;
  // blk: 32-site block of W (and of the partial sums); vblk: the same sites' block in the spinor fields, whose lattice is g.
  // Whole lattice: vblk0 = 0.  t-slab (ok_slab_dirac_apply): the fields carry one halo time slice below and above the slab,
  // g is that extended lattice and vblk0 the blocks of one slice, so the +-t neighbours of the boundary slices are the halos.
  const int blk = blockIdx.x, vblk = blk + vblk0;
  int n = vblk * kBlock + lane;
  if (n >= g.V) n = 0;   // padded lane: W is zero there, the result is zero
  const int x = n % g.L[0];
  int q = n / g.L[0];
  const int y = q % g.L[1];
  q /= g.L[1];
  const int z = q % g.L[2];
  const int t = q / g.L[2];

  real acc[RPT][2];
#pragma unroll
  for (int r = 0; r < RPT; ++r) acc[r][0] = acc[r][1] = real(0);

  const vec_t* Wp = W + ((size_t)blk * kTerms * 12 + rg * RPT) * NC * kBlock + lane;

#pragma unroll 1
  for (int o = 0; o < kTerms; ++o) {
    const int xx = wrap(x + c_off[o][0], g.L[0]);
    const int yy = wrap(y + c_off[o][1], g.L[1]);
    const int zz = wrap(z + c_off[o][2], g.L[2]);
    const int tt = wrap(t + c_off[o][3], g.L[3]);
    const int nn = xx + g.L[0] * (yy + g.L[1] * (zz + g.L[2] * tt));
    const vec_t* sp = psi + (size_t)(nn >> 5) * NC * kBlock + (nn & 31);
    if constexpr (PEER) {   // a time slice is a whole number of blocks (vblk0), so tt is uniform over the warp
      if (tt == 0) sp = lo_peer + (size_t)(nn >> 5) * NC * kBlock + (nn & 31);
      else if (tt == g.L[3] - 1) sp = hi_peer + (size_t)((nn >> 5) - (g.L[3] - 1) * vblk0) * NC * kBlock + (nn & 31);
    }
    vec_t w[RPT][NC];
#pragma unroll
    for (int r = 0; r < RPT; ++r)
#pragma unroll
      for (int c = 0; c < NC; ++c) w[r][c] = __ldcs(Wp + ((size_t)o * 12 + r) * NC * kBlock + c * kBlock);
    vec_t s[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) s[c] = __ldg(sp + c * kBlock);
#pragma unroll
    for (int r = 0; r < RPT; ++r)
#pragma unroll
      for (int c = 0; c < NC; ++c) cmac(acc[r], w[r][c], s[c]);
  }

  // store: row -> (unit c, sub) of the internal spinor layout
  real* ob = reinterpret_cast<real*>(out + (size_t)vblk * NC * kBlock);
  constexpr int RPU = 12 / NC;   // rows (components) per 16-byte unit: 2 (fp32) or 1 (fp64)
#pragma unroll
  for (int r = 0; r < RPT; ++r) {
    const int row = rg * RPT + r;
    const int c = row / RPU, sub = row % RPU;
    real* dst = ob + ((size_t)c * kBlock + lane) * (2 * RPU) + 2 * sub;
    if constexpr (sizeof(real) == 4)
      *reinterpret_cast<float2*>(dst) = make_float2(acc[r][0], acc[r][1]);
    else
      *reinterpret_cast<double2*>(dst) = make_double2(acc[r][0], acc[r][1]);
  }

  if constexpr (DOT) {
    // partials[blk] = ( Re<a,out>, Im<a,out>, ||out||^2 ), fp64, fixed summation order
    const real* ab = reinterpret_cast<const real*>(dot_a + (size_t)vblk * NC * kBlock);
    double d0 = 0.0, d1 = 0.0, d2 = 0.0;
#pragma unroll
    for (int r = 0; r < RPT; ++r) {
      const int row = rg * RPT + r;
      const int c = row / RPU, sub = row % RPU;
      const real* src = ab + ((size_t)c * kBlock + lane) * (2 * RPU) + 2 * sub;
      const double ar = (double)src[0], ai = (double)src[1];
      const double vr = (double)acc[r][0], vi = (double)acc[r][1];
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
    __shared__ double red[NW][3];
    if (lane == 0) { red[rg][0] = d0; red[rg][1] = d1; red[rg][2] = d2; }
    __syncthreads();
    if (threadIdx.x == 0) {
      double s0 = 0.0, s1 = 0.0, s2 = 0.0;
#pragma unroll
      for (int w2 = 0; w2 < NW; ++w2) { s0 += red[w2][0]; s1 += red[w2][1]; s2 += red[w2][2]; }
      partials[(size_t)blk * 3 + 0] = s0;
      partials[(size_t)blk * 3 + 1] = s1;
      partials[(size_t)blk * 3 + 2] = s2;
    }
  }
}

template <typename real, int RPT>
static int launch_direct(const Geom& g, const void* W, const void* psi, void* out, double* partials,
                         const void* dot_a, int nblk = -1, int vblk0 = 0, const void* lo_peer = nullptr, const void* hi_peer = nullptr) {
  using vec_t = typename Vec<real>::type;
  dim3 grid(nblk < 0 ? g.nblk : nblk), block(32 * (12 / RPT));
  if (lo_peer && hi_peer) {
    if (partials)
      apply_direct_kernel<real, RPT, true, true><<<grid, block, 0, ctx().stream>>>(
          static_cast<const vec_t*>(W), static_cast<const vec_t*>(psi), static_cast<vec_t*>(out), g, vblk0,
          static_cast<const vec_t*>(dot_a), partials, static_cast<const vec_t*>(lo_peer), static_cast<const vec_t*>(hi_peer));
    else
      apply_direct_kernel<real, RPT, false, true><<<grid, block, 0, ctx().stream>>>(
          static_cast<const vec_t*>(W), static_cast<const vec_t*>(psi), static_cast<vec_t*>(out), g, vblk0, nullptr, nullptr,
          static_cast<const vec_t*>(lo_peer), static_cast<const vec_t*>(hi_peer));
    OK_LAUNCHED("apply_direct_kernel (peer halos)");
    return OK_SUCCESS;
  }
  if (partials)
    apply_direct_kernel<real, RPT, true><<<grid, block, 0, ctx().stream>>>(
        static_cast<const vec_t*>(W), static_cast<const vec_t*>(psi), static_cast<vec_t*>(out), g, vblk0,
        static_cast<const vec_t*>(dot_a), partials);
  else
    apply_direct_kernel<real, RPT, false><<<grid, block, 0, ctx().stream>>>(
        static_cast<const vec_t*>(W), static_cast<const vec_t*>(psi), static_cast<vec_t*>(out), g, vblk0, nullptr, nullptr);
  OK_LAUNCHED("apply_direct_kernel");
  return OK_SUCCESS;
}

constexpr int kRowsPerWarp = 3;   // 4 warps per CTA, 40 registers: the measured optimum (profiles/r01_apply.md)
constexpr int kSmallLatticeBlocks = 4 * 148;   // below four CTAs per SM: 12 warps per CTA

int launch_apply(const ok_params* p, const void* W, const void* psi, void* out, double* partials,
                 const void* dot_a, const void* /*unused*/) {
  if (p->nrhs != 1) return OK_EINVAL;   // multi-RHS apply: ok_apply_mrhs.cu
  if (p->storage == OK_W_PAULI) return launch_apply_pauli(p, W, psi, out, partials, dot_a);     // ok_pauli.cu
  if (p->storage != OK_W_DENSE) return launch_apply_sparse(p, W, psi, out, partials, dot_a);   // ok_apply_sparse.cu
  int st = upload_offsets();
  if (st) return st;
  Geom g = make_geom(p);
  // Small lattices (BASELINE configs[0], [1]): one CTA per 32-site block leaves most SMs with one or two CTAs, too few W
  // loads in flight to fill the HBM pipe.  There a CTA uses 12 warps of one output row each instead of 4 warps of three
  // (same arithmetic and summation order per row, hence the same bits).
  if (g.nblk < kSmallLatticeBlocks) {
    if (p->precision == OK_FP64) return launch_direct<double, 1>(g, W, psi, out, partials, dot_a);
    return launch_direct<float, 1>(g, W, psi, out, partials, dot_a);
  }
  if (p->precision == OK_FP64) return launch_direct<double, kRowsPerWarp>(g, W, psi, out, partials, dot_a);
  return launch_direct<float, kRowsPerWarp>(g, W, psi, out, partials, dot_a);
}

// Eq. (2.2) for the 32-site blocks [blk0, blk0 + nblk) of the whole lattice only (ok_dirac_apply_host pipelines the apply over
// chunks of time slices behind the host -> device copy); Wp = W's payload of the whole lattice.
int launch_apply_range(const ok_params* p, const void* Wp, const void* psi, void* out, int blk0, int nblk) {
  if (p->nrhs != 1 || p->storage != OK_W_DENSE) return OK_EINVAL;
  int st = upload_offsets();
  if (st) return st;
  const Geom g = make_geom(p);
  const size_t wblock = (size_t)kTerms * 144 * 2 * real_bytes(p) * kBlock;   // bytes of W per 32-site block
  const char* Wb = static_cast<const char*>(Wp) + (size_t)blk0 * wblock;
  if (p->precision == OK_FP64) return launch_direct<double, kRowsPerWarp>(g, Wb, psi, out, nullptr, nullptr, nblk, blk0);
  return launch_direct<float, kRowsPerWarp>(g, Wb, psi, out, nullptr, nullptr, nblk, blk0);
}

// t-slab apply (ok_slab.cu): p = the slab's own lattice (Lx, Ly, Lz, Tloc) whose W this is; psi, out, dot_a are fields of the
// extended lattice (Lx, Ly, Lz, Tloc + 2) in the internal layout, i.e. [lower halo slice][Tloc slices][upper halo slice].
// lo_peer / hi_peer (both or neither): the neighbours' boundary slices, read in place of psi_ext's halo slices.
int launch_apply_slab(const ok_params* p, const void* W, const void* psi_ext, void* out_ext, double* partials, const void* dot_a_ext,
                      const void* lo_peer, const void* hi_peer) {
  if ((lo_peer == nullptr) != (hi_peer == nullptr)) return OK_EINVAL;
  if (p->nrhs != 1 || p->storage != OK_W_DENSE) return OK_EINVAL;
  int st = upload_offsets();
  if (st) return st;
  const Geom g = make_geom(p);
  const int slice = p->dims[0] * p->dims[1] * p->dims[2];
  if (slice % kBlock) return OK_EINVAL;
  Geom ge = g;
  ge.L[3] = g.L[3] + 2;
  ge.V = g.V + 2 * slice;
  ge.nblk = ge.V / kBlock;
  if (p->precision == OK_FP64)
    return launch_direct<double, kRowsPerWarp>(ge, W, psi_ext, out_ext, partials, dot_a_ext, g.nblk, slice / kBlock, lo_peer, hi_peer);
  return launch_direct<float, kRowsPerWarp>(ge, W, psi_ext, out_ext, partials, dot_a_ext, g.nblk, slice / kBlock, lo_peer, hi_peer);
}

}  // namespace okd
