// C-ABI entry points of libokdirac (include/ok.h): argument checks, sizes, handle table.
// Every step of the hot path runs in the CUDA kernels of the other translation units.
#include <iterator>
#include <mutex>
#include <stdlib.h>
#include <string.h>
#include <unordered_map>

#include "ok_internal.cuh"
#include "ok_sparse.cuh"

namespace okd {

const int8_t kOffsets[kTerms][4] = {
    {0, 0, 0, 0},
    {1, 0, 0, 0},  {-1, 0, 0, 0}, {0, 1, 0, 0},  {0, -1, 0, 0}, {0, 0, 1, 0},  {0, 0, -1, 0},
    {0, 0, 0, 1},  {0, 0, 0, -1},
    {2, 0, 0, 0},  {-2, 0, 0, 0}, {0, 2, 0, 0},  {0, -2, 0, 0}, {0, 0, 2, 0},  {0, 0, -2, 0},
    {1, 1, 0, 0},  {-1, -1, 0, 0}, {1, -1, 0, 0}, {-1, 1, 0, 0},
    {1, 0, 1, 0},  {-1, 0, -1, 0}, {1, 0, -1, 0}, {-1, 0, 1, 0},
    {0, 1, 1, 0},  {0, -1, -1, 0}, {0, 1, -1, 0}, {0, -1, 1, 0}};

Ctx& ctx() {
  static Ctx c;
  static bool init = [] {
    const char* e = getenv("OK_SYNC_CHECK");
    c.sync_check = e && e[0] == '1';
    return true;
  }();
  (void)init;
  return c;
}

int bind_device() {
  int dev = -1;
  OK_CUDA(cudaGetDevice(&dev));
  if (ctx().device < 0) ctx().device = dev;
  if (ctx().device != dev) {
    snprintf(ctx().err, sizeof(ctx().err), "libokdirac is bound to CUDA device %d; this call arrived on device %d", ctx().device, dev);
    return OK_EINVAL;
  }
  return OK_SUCCESS;
}

int fail_cuda(cudaError_t e, const char* where) {
  snprintf(ctx().err, sizeof(ctx().err), "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), where);
  return OK_ECUDA;
}

static uint32_t layout_id(const ok_params* p) {
  if (p->nrhs == 12) return kLayoutMrhs;
  return p->storage == OK_W_BLOCK ? kLayoutBlock : p->storage == OK_W_DS ? kLayoutDS : p->storage == OK_W_CONJ ? kLayoutConj :
         p->storage == OK_W_PAULI ? kLayoutPauli : kLayoutDense;
}

bool valid_params(const ok_params* p) {
  if (!p) return false;
  long long V = 1;
  for (int d = 0; d < 4; ++d) {
    if (p->dims[d] < 2 || p->dims[d] > 4096) return false;
    if (p->bc[d] != 1 && p->bc[d] != -1) return false;
    V *= p->dims[d];
  }
  if (V > (1LL << 30)) return false;
  if (p->precision != OK_FP32 && p->precision != OK_FP64) return false;
  if (p->nrhs != 1 && p->nrhs != 12) return false;
  if (p->nrhs == 12 && p->precision != OK_FP32) return false;
  if (p->storage < OK_W_DENSE || p->storage > OK_W_PAULI) return false;
  if (p->nrhs == 12 && p->storage != OK_W_DENSE) return false;
  if (!(p->kappa > 0.0) || !(p->u0 > 0.0)) return false;
  return true;
}

Geom make_geom(const ok_params* p) {
  Geom g;
  g.V = 1;
  for (int d = 0; d < 4; ++d) {
    g.L[d] = p->dims[d];
    g.V *= p->dims[d];
  }
  g.nblk = (g.V + kBlock - 1) / kBlock;
  return g;
}

static std::mutex g_mu;
static std::unordered_map<const void*, ok_params> g_table;

int remember_W(const void* W, const ok_params* p) {
  std::lock_guard<std::mutex> lk(g_mu);
  // a W written here invalidates every record whose bytes it overwrites (a buffer handed out again by a caching
  // allocator without ok_forget_W, or a W carved out of a larger arena)
  const uintptr_t lo = reinterpret_cast<uintptr_t>(W), hi = lo + ok_W_bytes(p);
  for (auto it = g_table.begin(); it != g_table.end();) {
    const uintptr_t a = reinterpret_cast<uintptr_t>(it->first), b = a + ok_W_bytes(&it->second);
    it = (a < hi && lo < b) ? g_table.erase(it) : std::next(it);
  }
  g_table[W] = *p;
  return OK_SUCCESS;
}

int refresh_W(const void* W, ok_params* p) {
  if (!aligned16(W)) return OK_EINVAL;
  WHeader h;
  OK_CUDA(cudaMemcpyAsync(&h, W, sizeof(h), cudaMemcpyDeviceToHost, ctx().stream));
  OK_CUDA(cudaStreamSynchronize(ctx().stream));
  if (h.magic != kMagic || !valid_params(&h.p) || h.layout != layout_id(&h.p)) {
    std::lock_guard<std::mutex> lk(g_mu);
    g_table.erase(W);
    return OK_EINVAL;
  }
  remember_W(W, &h.p);
  *p = h.p;
  return OK_SUCCESS;
}

int lookup_W(const void* W, ok_params* p) {
  if (!aligned16(W)) return OK_EINVAL;
  int st = bind_device();
  if (st) return st;
  {
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_table.find(W);
    if (it != g_table.end()) {
      *p = it->second;
      return OK_SUCCESS;
    }
  }
  return refresh_W(W, p);
}

static int write_header(void* W, const ok_params* p) {
  // Staged through a static pinned-free host copy: cudaMemcpyAsync from pageable memory copies
  // the source before returning, so a stack object is safe here.
  char buf[OK_W_HEADER_BYTES];
  memset(buf, 0, sizeof(buf));
  WHeader h;
  h.magic = kMagic;
  h.layout = layout_id(p);
  h.p = *p;
  memcpy(buf, &h, sizeof(h));
  OK_CUDA(cudaMemcpyAsync(W, buf, sizeof(buf), cudaMemcpyHostToDevice, ctx().stream));
  return remember_W(W, p);
}

static ok_slab_peers g_peers;
static bool g_have_peers = false;
const ok_slab_peers* slab_peers() { return g_have_peers ? &g_peers : nullptr; }

}  // namespace okd

using namespace okd;

extern "C" {

size_t ok_vec_bytes(const ok_params* p) {
  if (!valid_params(p)) return 0;
  Geom g = make_geom(p);
  if (p->nrhs == 12)   // header + fp32 records + tensor-core operand records (ok_internal.cuh)
    return (kMrhsVecHeaderBytes + (size_t)g.V * (kMrhsVecSiteFloats * 4 + kMrhsOpSiteHalves * 2) + 255) / 256 * 256;
  return (size_t)g.nblk * kBlock * 12 * 2 * real_bytes(p);
}

size_t ok_W_bytes(const ok_params* p) {
  if (!valid_params(p)) return 0;
  Geom g = make_geom(p);
  if (p->nrhs == 12) return OK_W_HEADER_BYTES + (size_t)g.V * kMrhsWSiteBytes;
  if (p->storage == OK_W_PAULI) return OK_W_HEADER_BYTES + (size_t)g.nblk * kBlock * (OK_W_PAULI_MATS * 9) * 2 * real_bytes(p);
  if (p->storage != OK_W_DENSE)
    return OK_W_HEADER_BYTES + (size_t)g.nblk * kBlock * sparse_site_units_rt(p->storage) * 2 * real_bytes(p);
  return OK_W_HEADER_BYTES + (size_t)g.nblk * kBlock * kTerms * 144 * 2 * real_bytes(p);
}

size_t ok_work_bytes(const ok_params* p) {
  if (!valid_params(p)) return 0;
  size_t a = precalc_work_bytes(p), b = p->nrhs == 12 ? bicgstab_mrhs_work_bytes(p) : bicgstab_work_bytes(p);
  size_t host_io = 2 * ok_vec_bytes(p) + 2 * ok_vec_bytes(p);   // ok_dirac_apply_host staging
  size_t m = a > b ? a : b;
  return (m > host_io ? m : host_io) + 4096;
}

int ok_set_stream(void* s) {
  ctx().stream = static_cast<cudaStream_t>(s);
  return OK_SUCCESS;
}

int ok_set_workspace(void* dev, size_t bytes) {
  if (dev && (reinterpret_cast<uintptr_t>(dev) & 255)) return OK_EINVAL;
  ctx().work = dev;
  ctx().work_bytes = dev ? bytes : 0;
  return OK_SUCCESS;
}

uint64_t ok_launch_count(void) { return ctx().launches; }

int ok_pack_spinor(const ok_params* p, const void* canon, void* packed) {
  if (!valid_params(p) || !aligned16(canon) || !aligned16(packed)) return OK_EINVAL;
  if (int st = bind_device()) return st;
  return launch_pack_spinor(p, canon, packed, false);
}

int ok_unpack_spinor(const ok_params* p, const void* packed, void* canon) {
  if (!valid_params(p) || !aligned16(canon) || !aligned16(packed)) return OK_EINVAL;
  if (int st = bind_device()) return st;
  return launch_pack_spinor(p, canon, const_cast<void*>(packed), true);
}

int ok_pack_W(const ok_params* p, const void* canon, void* W) {
  if (!valid_params(p) || !aligned16(canon) || !aligned16(W)) return OK_EINVAL;
  if (p->storage == OK_W_PAULI) return OK_EINVAL;   // only ok_precalc_W writes this format (ok.h)
  int st = bind_device();
  if (st) return st;
  st = write_header(W, p);
  if (st) return st;
  return launch_pack_W(p, canon, W_payload(W), false);
}

int ok_unpack_W(const void* W, void* canon) {
  ok_params p;
  if (!aligned16(canon)) return OK_EINVAL;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (p.storage == OK_W_PAULI) return launch_unpack_pauli(&p, W_payload(W), canon);
  return launch_pack_W(&p, canon, const_cast<char*>(W_payload(W)), true);
}

int ok_forget_W(const void* W) {
  std::lock_guard<std::mutex> lk(g_mu);
  g_table.erase(W);
  return OK_SUCCESS;
}

int ok_W_params(const void* W, ok_params* p) {
  if (!p) return OK_EINVAL;
  int st = bind_device();
  if (st) return st;
  return refresh_W(W, p);   // always from the device header, so a W refilled behind the library's back is seen
}

int ok_precalc_W(const void* links, const ok_params* p, void* W) {
  if (!valid_params(p) || !aligned16(links) || !aligned16(W)) return OK_EINVAL;
  if (!ctx().work || ctx().work_bytes < precalc_work_bytes(p)) return OK_EWORKSPACE;
  int st = bind_device();
  if (st) return st;
  st = write_header(W, p);
  if (st) return st;
  return launch_precalc(p, links, W_payload(W), ctx().work);
}

int ok_dirac_apply(const void* W, const void* psi, void* out) {
  if (!aligned16(psi) || !aligned16(out) || psi == out) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (p.reserved_ == OK_SLAB) return OK_EINVAL;   // a t-slab is open in t: ok_slab_dirac_apply
  if (p.nrhs == 12) return mrhs_apply_vec(&p, W_payload(W), const_cast<void*>(psi), out);
  return launch_apply(&p, W_payload(W), psi, out, nullptr, nullptr, nullptr);
}

// Host-buffer apply, pipelined: the lattice is cut into chunks of time slices; chunk c is applied as soon as chunks c - 1, c,
// c + 1 have landed (the stencil reaches one slice in t) while later chunks are still crossing PCIe, and its
// result starts back to the host while the next chunk is computed.  Three streams: copies in, the caller's stream for
// pack / apply / unpack, copies out.  Copy order n-1, 0, 1, ..., n-2 so that chunk 0 (which needs the last chunk through the
// periodic closure) can start after three chunks.  The applies (with their unpack) alternate between two more library-owned
// streams, so that the ramp-down of one chunk's launch overlaps the next chunk's ramp-up (16 short launches otherwise lose
// a tail each).  The paper's GPU code pays these copies in sequence on every call (96.6 % of its
// overhead); here they hide behind the W stream.
static int apply_host_pipelined(const ok_params& p, const void* W, const char* psi_host, char* out_host, char* canon_in, char* packed_in,
                                char* packed_out, char* canon_out) {
  constexpr int kMaxChunks = 16;
  static cudaStream_t s_in = nullptr, s_out = nullptr, s_ap[2] = {nullptr, nullptr};
  static cudaEvent_t ev_start = nullptr, ev_end = nullptr, ev_in[kMaxChunks], ev_done[kMaxChunks], ev_packed[kMaxChunks];
  if (!s_in) {
    OK_CUDA(cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking));
    OK_CUDA(cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking));
    OK_CUDA(cudaStreamCreateWithFlags(&s_ap[0], cudaStreamNonBlocking));
    OK_CUDA(cudaStreamCreateWithFlags(&s_ap[1], cudaStreamNonBlocking));
    OK_CUDA(cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming));
    OK_CUDA(cudaEventCreateWithFlags(&ev_end, cudaEventDisableTiming));
    for (int c = 0; c < kMaxChunks; ++c) {
      OK_CUDA(cudaEventCreateWithFlags(&ev_in[c], cudaEventDisableTiming));
      OK_CUDA(cudaEventCreateWithFlags(&ev_done[c], cudaEventDisableTiming));
      OK_CUDA(cudaEventCreateWithFlags(&ev_packed[c], cudaEventDisableTiming));
    }
  }
  cudaStream_t st = ctx().stream;
  const int T = p.dims[3], n = T >= 2 * kMaxChunks ? kMaxChunks : (T >= 16 ? 8 : 4);
  const size_t slice_sites = (size_t)p.dims[0] * p.dims[1] * p.dims[2];
  const size_t sb = slice_sites * 12 * 2 * real_bytes(&p);          // bytes of a time slice, canonical and internal alike
  int t0[kMaxChunks + 1];
  for (int c = 0; c <= n; ++c) t0[c] = (int)((long long)c * T / n);
  if (n == kMaxChunks && T >= 64) {
    // small chunks at both ends, large ones in the middle: the first apply starts after three short copies (chunks n-1, 0, 1)
    // and only a short result is still on its way back when the last apply ends; in between the copies run ahead of the applies
    static const int w[kMaxChunks] = {1, 1, 2, 4, 6, 6, 6, 6, 6, 6, 6, 6, 4, 2, 1, 1};   // sum 64
    int acc = 0;
    for (int c = 0; c < n; ++c) {
      t0[c] = (int)((long long)acc * T / 64);
      acc += w[c];
    }
    t0[n] = T;
  }
  OK_CUDA(cudaEventRecord(ev_start, st));
  OK_CUDA(cudaStreamWaitEvent(s_in, ev_start, 0));
  OK_CUDA(cudaStreamWaitEvent(s_out, ev_start, 0));
  for (int k = 0; k < n; ++k) {
    const int c = (k + n - 1) % n;   // n-1, 0, 1, ..., n-2
    const size_t off = (size_t)t0[c] * sb;
    OK_CUDA(cudaMemcpyAsync(canon_in + off, psi_host + off, (size_t)(t0[c + 1] - t0[c]) * sb, cudaMemcpyHostToDevice, s_in));
    OK_CUDA(cudaEventRecord(ev_in[c], s_in));
  }
  int rc = OK_SUCCESS;
  auto chunk_params = [&](int c) {
    ok_params q = p;
    q.dims[3] = t0[c + 1] - t0[c];
    return q;
  };
  int last_packed = -1;   // the packs run in issue order on st, so the latest one's event covers all of them
  auto pack = [&](int c) -> int {
    OK_CUDA(cudaStreamWaitEvent(st, ev_in[c], 0));
    const ok_params q = chunk_params(c);
    const size_t off = (size_t)t0[c] * sb;
    int r = launch_pack_spinor(&q, canon_in + off, packed_in + off, false);
    if (r) return r;
    OK_CUDA(cudaEventRecord(ev_packed[c], st));
    last_packed = c;
    return OK_SUCCESS;
  };
  auto apply = [&](int c) -> int {   // issued right after the last pack it needs
    const ok_params q = chunk_params(c);
    const size_t off = (size_t)t0[c] * sb;
    const int blk0 = (int)(t0[c] * slice_sites / kBlock), nblk = (int)((t0[c + 1] - t0[c]) * slice_sites / kBlock);
    cudaStream_t sa = s_ap[c & 1];
    OK_CUDA(cudaStreamWaitEvent(sa, ev_packed[last_packed], 0));
    ctx().stream = sa;
    int r = launch_apply_range(&p, W_payload(W), packed_in, packed_out, blk0, nblk);
    if (!r) r = launch_pack_spinor(&q, canon_out + off, packed_out + off, true);
    ctx().stream = st;
    if (r) return r;
    OK_CUDA(cudaEventRecord(ev_done[c], sa));
    OK_CUDA(cudaStreamWaitEvent(s_out, ev_done[c], 0));
    OK_CUDA(cudaMemcpyAsync(out_host + off, canon_out + off, (size_t)(t0[c + 1] - t0[c]) * sb, cudaMemcpyDeviceToHost, s_out));
    return OK_SUCCESS;
  };
#define OK_STEP(e) do { if ((rc = (e))) return rc; } while (0)
  OK_STEP(pack(n - 1)); OK_STEP(pack(0)); OK_STEP(pack(1));
  OK_STEP(apply(0));
  for (int c = 2; c <= n - 2; ++c) { OK_STEP(pack(c)); OK_STEP(apply(c - 1)); }
  OK_STEP(apply(n - 2));
  OK_STEP(apply(n - 1));
#undef OK_STEP
  OK_CUDA(cudaEventRecord(ev_end, s_out));
  OK_CUDA(cudaStreamWaitEvent(st, ev_end, 0));
  OK_CUDA(cudaStreamSynchronize(st));
  return OK_SUCCESS;
}

int ok_dirac_apply_host(const void* W, const void* psi_host, void* out_host) {
  if (!psi_host || !out_host) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (p.reserved_ == OK_SLAB) return OK_EINVAL;
  size_t vb = ok_vec_bytes(&p);
  Geom g = make_geom(&p);
  size_t cb = (size_t)g.V * 12 * 2 * real_bytes(&p) * p.nrhs;   // canonical bytes (no padding)
  if (!ctx().work || ctx().work_bytes < 4 * vb) return OK_EWORKSPACE;
  char* w = static_cast<char*>(ctx().work);
  char *canon_in = w, *packed_in = w + vb, *packed_out = w + 2 * vb, *canon_out = w + 3 * vb;
  // (small fields: the two dozen extra launches and event waits of the pipeline cost more than the copies it hides)
  if (p.nrhs == 1 && p.storage == OK_W_DENSE && p.dims[3] >= 8 && ((long long)p.dims[0] * p.dims[1] * p.dims[2]) % kBlock == 0 &&
      (cb >= ((size_t)8 << 20) || getenv("OK_HOST_PIPELINE")))
    return apply_host_pipelined(p, W, static_cast<const char*>(psi_host), static_cast<char*>(out_host), canon_in, packed_in, packed_out,
                                canon_out);
  OK_CUDA(cudaMemcpyAsync(canon_in, psi_host, cb, cudaMemcpyHostToDevice, ctx().stream));
  if ((st = launch_pack_spinor(&p, canon_in, packed_in, false))) return st;
  st = p.nrhs == 12 ? mrhs_apply_vec(&p, W_payload(W), packed_in, packed_out)
                    : launch_apply(&p, W_payload(W), packed_in, packed_out, nullptr, nullptr, nullptr);
  if (st) return st;
  if ((st = launch_pack_spinor(&p, canon_out, packed_out, true))) return st;
  OK_CUDA(cudaMemcpyAsync(out_host, canon_out, cb, cudaMemcpyDeviceToHost, ctx().stream));
  OK_CUDA(cudaStreamSynchronize(ctx().stream));
  return OK_SUCCESS;
}

int ok_bicgstab(const void* W, const void* src, void* x, double tol, int maxit, int* iters, double* resid) {
  if (!aligned16(src) || !aligned16(x) || src == x || !iters || !resid || !(tol > 0.0) || maxit < 1) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (p.reserved_ == OK_SLAB) return OK_EINVAL;   // ok_slab_bicgstab
  if (p.nrhs == 12) {
    if (!ctx().work || ctx().work_bytes < bicgstab_mrhs_work_bytes(&p)) return OK_EWORKSPACE;
    return run_bicgstab_mrhs(&p, W_payload(W), src, x, tol, maxit, iters, resid);
  }
  if (!ctx().work || ctx().work_bytes < bicgstab_work_bytes(&p)) return OK_EWORKSPACE;
  return run_bicgstab(&p, W_payload(W), src, x, tol, maxit, iters, resid);
}

int ok_cgnr(const void* W, const void* src, void* x, double tol, int maxit, int* iters, double* resid) {
  if (!aligned16(src) || !aligned16(x) || src == x || !iters || !resid || !(tol > 0.0) || maxit < 1) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (p.nrhs != 1 || p.reserved_ == OK_SLAB) return OK_EINVAL;
  if (!ctx().work || ctx().work_bytes < bicgstab_work_bytes(&p)) return OK_EWORKSPACE;
  return run_cgnr(&p, W_payload(W), src, x, tol, maxit, iters, resid);
}

size_t ok_mixed_work_bytes(const ok_params* p) {
  if (!valid_params(p) || p->nrhs != 1) return 0;
  return mixed_work_bytes(p) + 4096;
}

int ok_bicgstab_mixed(const void* W64, const void* W32, const void* src, void* x, double tol, double inner_tol, int maxit,
                      int max_outer, int* iters, int* outer, double* resid) {
  if (!aligned16(src) || !aligned16(x) || src == x || !iters || !outer || !resid || !(tol > 0.0) || !(inner_tol > 0.0) || !(inner_tol < 1.0) ||
      maxit < 1 || max_outer < 1)
    return OK_EINVAL;
  ok_params p64, p32;
  int st = lookup_W(W64, &p64);
  if (st) return st;
  if ((st = lookup_W(W32, &p32))) return st;
  if (p64.precision != OK_FP64 || p32.precision != OK_FP32 || p64.nrhs != 1 || p32.nrhs != 1 || p64.reserved_ || p32.reserved_) return OK_EINVAL;
  for (int d = 0; d < 4; ++d)
    if (p64.dims[d] != p32.dims[d]) return OK_EINVAL;
  if (!ctx().work || ctx().work_bytes < mixed_work_bytes(&p64)) return OK_EWORKSPACE;
  return run_bicgstab_mixed(&p64, W_payload(W64), &p32, W_payload(W32), src, x, tol, inner_tol, maxit, max_outer, iters, outer, resid);
}

// ---- t-slab decomposition ---------------------------------------------------------------------------------------
static bool valid_slab(const ok_params* p) {
  return valid_params(p) && p->reserved_ == OK_SLAB && p->nrhs == 1 && p->storage == OK_W_DENSE &&
         ((long long)p->dims[0] * p->dims[1] * p->dims[2]) % kBlock == 0;
}

size_t ok_slab_slice_bytes(const ok_params* p) {
  if (!valid_slab(p)) return 0;
  return (size_t)p->dims[0] * p->dims[1] * p->dims[2] * 12 * 2 * real_bytes(p);
}

size_t ok_slab_vec_bytes(const ok_params* p) { return valid_slab(p) ? (size_t)(p->dims[3] + 2) * ok_slab_slice_bytes(p) : 0; }

static ok_params slab_link_lattice(const ok_params* p) {   // the lattice the slab's link window lives on
  ok_params e = *p;
  e.dims[3] = p->dims[3] + 2 * OK_SLAB_LINK_HALO;
  e.reserved_ = 0;
  return e;
}

size_t ok_slab_work_bytes(const ok_params* p, int nslab, int nranks) {
  if (!valid_slab(p) || nslab < 1 || nranks < 1) return 0;
  const ok_params e = slab_link_lattice(p);
  const size_t a = precalc_work_bytes(&e), b = (size_t)nslab * bicgstab_slab_work_bytes(p) + bicgstab_slab_shared_bytes(nslab, nranks);
  return (a > b ? a : b) + 4096;
}

int ok_slab_precalc_W(const void* links_ext, const ok_params* p, int T, int t0, void* W) {
  if (!valid_slab(p) || !aligned16(links_ext) || !aligned16(W)) return OK_EINVAL;
  const int Tloc = p->dims[3], H = OK_SLAB_LINK_HALO;
  if (T < Tloc + 2 * H || t0 < 0 || t0 >= T) return OK_EINVAL;
  const ok_params e = slab_link_lattice(p);
  if (!ctx().work || ctx().work_bytes < precalc_work_bytes(&e)) return OK_EWORKSPACE;
  int st = bind_device();
  if (st) return st;
  if ((st = write_header(W, p))) return st;
  // window slice k holds global t = t0 - H + k (mod T): where is T - 1 ?
  int k = ((T - 1) - (t0 - H)) % T;
  if (k < 0) k += T;
  const int tfold = k < Tloc + 2 * H ? k : -1;
  const int slice_blocks = p->dims[0] * p->dims[1] * p->dims[2] / kBlock;
  return launch_precalc_window(&e, links_ext, W_payload(W), ctx().work, tfold, H * slice_blocks, Tloc * slice_blocks);
}

int ok_slab_dirac_apply(const void* W, const void* psi, void* out) {
  if (!aligned16(psi) || !aligned16(out) || psi == out) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (!valid_slab(&p)) return OK_EINVAL;
  return launch_apply_slab(&p, W_payload(W), psi, out, nullptr, nullptr);
}

int ok_slab_set_peers(const ok_slab_peers* peers) {
  if (!peers) {
    g_have_peers = false;
    return OK_SUCCESS;
  }
  if (!peers->lo_work || !peers->hi_work || !peers->lo_x || !peers->hi_x || !peers->barrier) return OK_EINVAL;
  g_peers = *peers;
  g_have_peers = true;
  return OK_SUCCESS;
}

int ok_slab_dirac_apply_peer(const void* W, const void* psi, const void* lo_slice, const void* hi_slice, void* out) {
  if (!aligned16(psi) || !aligned16(out) || !aligned16(lo_slice) || !aligned16(hi_slice) || psi == out) return OK_EINVAL;
  ok_params p;
  int st = lookup_W(W, &p);
  if (st) return st;
  if (!valid_slab(&p)) return OK_EINVAL;
  return launch_apply_slab(&p, W_payload(W), psi, out, nullptr, nullptr, lo_slice, hi_slice);
}

int ok_slab_bicgstab(int nslab, const void* const* W, const void* const* src, void* const* x, double tol, int maxit, const ok_comm* comm,
                     int* iters, double* resid) {
  if (nslab < 1 || nslab > 64 || !W || !src || !x || !iters || !resid || !(tol > 0.0) || maxit < 1) return OK_EINVAL;
  if (comm && (comm->nranks < 1 || comm->rank < 0 || comm->rank >= comm->nranks)) return OK_EINVAL;
  static ok_params ps[64];
  const ok_params* pp[64];
  const void* payload[64];
  for (int i = 0; i < nslab; ++i) {
    if (!aligned16(src[i]) || !aligned16(x[i]) || src[i] == x[i]) return OK_EINVAL;
    int st = lookup_W(W[i], &ps[i]);
    if (st) return st;
    if (!valid_slab(&ps[i]) || ps[i].precision != ps[0].precision) return OK_EINVAL;
    pp[i] = &ps[i];
    payload[i] = W_payload(W[i]);
  }
  return run_bicgstab_slabs(nslab, pp, payload, src, x, tol, maxit, comm, iters, resid);
}

int ok_W_unit_index(int storage, int term, int row, int col, int* info) {
  if (storage < OK_W_BLOCK || storage > OK_W_CONJ || term < 0 || term >= kTerms || row < 0 || row >= 12 || col < 0 || col >= 12) return -2;
  const SparseRef r = sparse_ref(storage, term, row, col);
  if (info) { info[0] = r.unit >= 0 ? r.stored : 0; info[1] = r.sign; info[2] = r.conj; info[3] = r.shift; }
  return r.unit;
}

const char* ok_strerror(int status) {
  switch (status) {
    case OK_SUCCESS: return "success";
    case OK_EINVAL: return "invalid argument (dims, precision, nrhs, null/misaligned pointer, or unknown W buffer)";
    case OK_ECUDA: return ctx().err;
    case OK_EBREAKDOWN: return "BiCGStab breakdown";
    case OK_EMAXIT: return "BiCGStab: maximum iterations reached without convergence";
    case OK_EWORKSPACE: return "workspace missing or too small (see ok_work_bytes / ok_set_workspace)";
    case OK_ECOMM: return "an ok_comm callback reported a failure";
    default: return "unknown status";
  }
}

const char* ok_version(void) { return "okdirac 0.1 (sm_100a)"; }

}  // extern "C"
