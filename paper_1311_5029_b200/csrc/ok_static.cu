// ok_dirac_apply_dot_static (ok.h): the Dirac apply with BiCGStab's fused reductions for callers that may not allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc -- and have no workspace to lend.
//   out = M psi (Eq. 2.2),  result = ( Re<a,out>, Im<a,out>, ||out||^2 )   (the dots of PAPER.md:114's solver)
// The apply kernels' reduction epilogue writes one row of three fp64 partial sums per 32-site block into scratch memory; here
// that scratch is the file-scope array g_static_partials below instead of the caller's workspace:
//   OK_STATIC_MAX_SITES = 2 097 152 sites (32^3 x 64, the largest BASELINE config) -> 65 536 rows x 24 B = 1.5 MiB,
// held by every GPU that loads the library until the process exits.
// In host code the array's name is a host-side stand-in, not a device address: the launchers get the address from
// cudaGetSymbolAddress, once per device with that device current; the reducing kernel below names the array directly.
// Shared by all calls: two calls whose kernels overlap on the GPU (different streams) race on it.  Nothing has to start at
// zero -- a call's apply overwrites rows [0, nblk) before its reduction reads exactly those rows; older contents beyond
// them are never read.
#include "ok_internal.cuh"

namespace okd {

constexpr int kStaticMaxBlocks = OK_STATIC_MAX_SITES / kBlock;
static __device__ __align__(256) double g_static_partials[(size_t)kStaticMaxBlocks * 3];

constexpr int kStaticThreads = 256;

// One CTA, thread-serial sums in a fixed order (bit-reproducible), then a fixed-order tree: result[0..2].
__global__ void __launch_bounds__(kStaticThreads) static_reduce_kernel(int count, double* __restrict__ result) {
  double d[3] = {0.0, 0.0, 0.0};
  for (int i = threadIdx.x; i < count; i += kStaticThreads) {
    const double* q = g_static_partials + (size_t)i * 3;
    d[0] += q[0];
    d[1] += q[1];
    d[2] += q[2];
  }
  __shared__ double red[kStaticThreads / 32][3];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < 3; ++q)
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) d[q] += __shfl_xor_sync(0xffffffffu, d[q], m);
  if (lane == 0) { red[w][0] = d[0]; red[w][1] = d[1]; red[w][2] = d[2]; }
  __syncthreads();
  if (threadIdx.x < 3) {
    double s = 0.0;
    for (int k = 0; k < kStaticThreads / 32; ++k) s += red[k][threadIdx.x];
    result[threadIdx.x] = s;
  }
}

static char g_static_err[256] = "no error";

// device address of g_static_partials on the bound device (resolved once per device, with that device current)
static int static_partials_ptr(double** out) {
  constexpr int kMaxDev = 64;
  static double* ptr[kMaxDev] = {};
  int dev = -1;
  OK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return OK_EINVAL;
  if (!ptr[dev]) {
    double* q = nullptr;
    OK_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&q), g_static_partials));
    if (!q) return OK_ECUDA;
    ptr[dev] = q;
  }
  *out = ptr[dev];
  return OK_SUCCESS;
}

}  // namespace okd

using namespace okd;

extern "C" {

size_t ok_static_max_sites(void) { return OK_STATIC_MAX_SITES; }

const char* ok_static_strerror(void) { return g_static_err; }

int ok_dirac_apply_dot_static(const void* W, const void* psi, const void* a, void* out, double* result) {
  if (!aligned16(psi) || !aligned16(out) || !aligned16(a) || !result || psi == out || a == out) {
    snprintf(g_static_err, sizeof(g_static_err), "ok_dirac_apply_dot_static: null or misaligned pointer, or out aliases psi / a");
    return OK_EINVAL;
  }
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) {
    snprintf(g_static_err, sizeof(g_static_err), "ok_dirac_apply_dot_static: W is not a buffer written by ok_precalc_W / ok_pack_W");
    return st;
  }
  if (p.nrhs != 1 || p.reserved_ == OK_SLAB) {
    snprintf(g_static_err, sizeof(g_static_err), "ok_dirac_apply_dot_static: nrhs = 1 and a whole lattice only");
    return OK_EINVAL;
  }
  const Geom g = make_geom(&p);
  if ((long long)g.nblk > (long long)kStaticMaxBlocks) {
    snprintf(g_static_err, sizeof(g_static_err),
             "ok_dirac_apply_dot_static: %d sites exceed the static scratch array (OK_STATIC_MAX_SITES = %d); use ok_bicgstab's "
             "workspace path for larger lattices",
             g.V, (int)OK_STATIC_MAX_SITES);
    return OK_EINVAL;
  }
  double* partials = nullptr;
  if ((st = static_partials_ptr(&partials))) {
    snprintf(g_static_err, sizeof(g_static_err), "ok_dirac_apply_dot_static: cudaGetSymbolAddress failed: %s", ok_strerror(st));
    return st;
  }
  if ((st = launch_apply(&p, W_payload(W), psi, out, partials, a, nullptr))) return st;
  static_reduce_kernel<<<1, kStaticThreads, 0, ctx().stream>>>(g.nblk, result);
  OK_LAUNCHED("static_reduce_kernel");
  return OK_SUCCESS;
}

}  // extern "C"
