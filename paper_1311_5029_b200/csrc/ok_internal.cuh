// Internal declarations shared by the translation units of libokdirac (not part of the ABI).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "ok.h"

namespace okd {

constexpr int kBlock = OK_SITE_BLOCK;   // sites per block (= warp width: lane <-> site)
constexpr int kTerms = OK_NTERMS;
constexpr uint32_t kMagic = 0x4F4B5731u;   // "OKW1"
constexpr uint32_t kLayoutDense = 1;       // [block][term][row][c][site][16 B]
constexpr uint32_t kLayoutBlock = 4;       // OK_W_BLOCK: [block][unit 2340][site][complex]   (ok_sparse.cuh)
constexpr uint32_t kLayoutConj = 6;        // OK_W_CONJ:  [block][unit 630][site][complex]
constexpr uint32_t kLayoutDS = 5;          // OK_W_DS:    [block][unit 1188][site][complex]
constexpr uint32_t kLayoutPauli = 7;       // OK_W_PAULI: [block][37 x 9 units][site][complex]   (ok_pauli.cu)
constexpr uint32_t kLayoutMrhs = 3;        // nrhs = 12: per-site tcgen05 operand tiles, split fp16 (ok_apply_mrhs.cu)

// ---- nrhs = 12 (tensor-core) layouts, fp32 fields (ok_apply_mrhs.cu) -------------------------------
// The per-site contraction Out[12 x 12] = sum_term W_term[12 x 12] Psi(x + o_term)[12 x 12] (complex) is run
// real-split on tcgen05 kind::f16 as  D[n][w] = sum_k A[n][k] B[w][k]  with
//   A (M side, tensor memory)  = Psi^T : row n = 2 rhs + part (part 0 = Re, 1 = Im), K = (term, component)
//   B (N side, shared memory)  = W     : row w = 8 (row/4) + 2 (row%4) + part,       K = (term, column)
// and every fp32 number carried as two fp16 pieces  x = hi + lo / 2048  (hi = rn(x), lo = rn((x - hi) 2048)),
// 22 significant bits, stacked as extra rows on both sides.
//
// K order: 7 stages of 48 k (4 stencil terms each; the last stage has 3 terms + 12 zero pad k).
//   stage c < 6 : k = 16 (comp/4) + 4 (term%4) + comp%4
//   stage 6     : s = 3 (term - 24) + comp/4 ;  k = 16 (s/4) + 4 (s%4) + comp%4   (k = 36..47 are pad)
// This is the order in which a spinor producer thread (row n, cp = lane%4) holds its three 16-byte loads.
//
// W tile (per site, fp16, 31 488 B): the UMMA canonical K-major no-swizzle layout of B,
//   [stage 7][k chunk k/8 : 6][row group w48/8 : 6][w48 % 8][k % 8],   w48 = 24 hl + w  (hl 0 = hi, 1 = lo)
// (core matrix = 8 rows x 16 B; SBO = 128 B between row groups, LBO = 768 B between k chunks); the all-pad
// k chunk 5 of stage 6 is not stored.  One contiguous tile = one bulk copy into shared memory.
constexpr int kMrhsStages = 7;
constexpr int kMrhsStageK = 48;
constexpr int kMrhsStageHalves = 48 * kMrhsStageK;                           // 2304 (4608 B)
constexpr int kMrhsWSiteHalves = kMrhsStages * kMrhsStageHalves - 6 * 64;    // 15 744
constexpr int kMrhsWSiteBytes = 2 * kMrhsWSiteHalves;                        // 31 488
constexpr float kMrhsLoScale = 2048.f;                                       // lo pieces are stored x 2^11
__host__ __device__ inline int mrhs_k(int term, int comp, int* stage) {
  const int c = term >> 2;
  *stage = c;
  if (c < 6) return 16 * (comp >> 2) + 4 * (term & 3) + (comp & 3);
  const int s = 3 * (term - 24) + (comp >> 2);
  return 16 * (s >> 2) + 4 * (s & 3) + (comp & 3);
}
__host__ __device__ inline int mrhs_W_row(int row, int part) { return 8 * (row >> 2) + 2 * (row & 3) + part; }
__host__ __device__ inline int mrhs_W_half_index(int stage, int k, int w48) {
  return stage * kMrhsStageHalves + (k >> 3) * 384 + (w48 >> 3) * 64 + (w48 & 7) * 8 + (k & 7);
}
__host__ __device__ inline int mrhs_W_index(int term, int row, int col, int part, int hl) {
  int stage;
  const int k = mrhs_k(term, col, &stage);
  return mrhs_W_half_index(stage, k, 24 * hl + mrhs_W_row(row, part));
}
__host__ __device__ inline int mrhs_W_pad_index(int q) {   // q = 0..191: zero pad halves (k = 36..39 of stage 6, 48 rows)
  return mrhs_W_half_index(6, 36 + (q & 3), q >> 2);
}
__host__ __device__ inline void mrhs_split(float x, __half* hi, __half* lo) {
  const __half h = __float2half_rn(x);
  *hi = h;
  *lo = __float2half_rn((x - __half2float(h)) * kMrhsLoScale);
}
__host__ __device__ inline float mrhs_join(__half hi, __half lo) { return __half2float(hi) + __half2float(lo) * (1.f / kMrhsLoScale); }
// nrhs = 12 spinor field (ok_vec_bytes): [header 256 B][fp32 records V x 1152 B][operand records V x 1152 B].
//   fp32 record (the field itself): [component/4 : 3][n = 2 rhs + part : 24][component%4]
//   operand record (what the tensor-core apply reads; valid only when header.valid != 0): the same numbers scaled per
//   right-hand side by a power of two S_j (header.scale) and split into two fp16 pieces, x S_j = hi + lo / 2048, stored
//   [q = n/12 : 2][g = component/4 : 3][slot : 24][component%4] halves.  A producer warp of TMEM lane quarter q reads 8 B per
//   lane with lane <-> slot (one LDG.64 = 192 contiguous bytes) and stores them with tcgen05.st.32x32b, so `slot` is the TMEM
//   lane order of the A rows: lanes 0-7 hi of n%12 = 0..7, 8-15 their lo, 16-19 hi of n%12 = 8..11, 24-27 their lo (the
//   epilogue's tcgen05.ld.16x256b finds hi and lo of one row 8 lanes apart).
//   Writers of an operand record: ok_pack_spinor, the BiCGStab update kernels (p, s) and mrhs_ensure_operand (fp32 ->
//   operand on demand); ok_dirac_apply writes only the fp32 records of `out` and clears out's header.valid.
constexpr int kMrhsVecSiteFloats = 288;
constexpr int kMrhsVecHeaderBytes = 256;
constexpr int kMrhsOpSiteHalves = 576;
struct MrhsVecHeader {
  float scale[12];        // S_j (power of two) of the operand records
  unsigned maxbits[12];   // scratch of mrhs_ensure_operand: bit pattern of max |psi_j|
  unsigned valid;         // operand records match the fp32 records
  unsigned done;          // scratch: CTAs of the split pass that have finished
};
static_assert(sizeof(MrhsVecHeader) <= kMrhsVecHeaderBytes, "header too large");
__host__ __device__ inline int mrhs_vec_index(int comp, int rhs, int part) {
  return ((comp >> 2) * 24 + 2 * rhs + part) * 4 + (comp & 3);
}
__host__ __device__ inline int mrhs_op_slot(int nl, int hl) { return nl < 8 ? nl + 8 * hl : 16 + (nl - 8) + 4 * hl; }
__host__ __device__ inline int mrhs_op_index(int comp, int rhs, int part, int hl) {
  const int n = 2 * rhs + part;
  return (((n / 12) * 3 + (comp >> 2)) * 24 + mrhs_op_slot(n % 12, hl)) * 4 + (comp & 3);
}
inline float* mrhs_f32(void* vec) { return reinterpret_cast<float*>(static_cast<char*>(vec) + kMrhsVecHeaderBytes); }
inline const float* mrhs_f32(const void* vec) { return reinterpret_cast<const float*>(static_cast<const char*>(vec) + kMrhsVecHeaderBytes); }
inline __half* mrhs_op(void* vec, int V) {
  return reinterpret_cast<__half*>(static_cast<char*>(vec) + kMrhsVecHeaderBytes + (size_t)V * kMrhsVecSiteFloats * 4);
}
inline const __half* mrhs_op(const void* vec, int V) { return mrhs_op(const_cast<void*>(vec), V); }
// power-of-two scale for an operand record from an upper bound B >= max |x| of the column: B S <= 2^15 (fp16 max 65504)
__host__ __device__ inline float mrhs_scale_from_bound(float B) {
  if (!(B > 0.f) || !(B < 3.0e38f)) return 1.f;
  unsigned bits;
#ifdef __CUDA_ARCH__
  bits = __float_as_uint(B);
#else
  memcpy(&bits, &B, 4);
#endif
  int e = (int)(bits >> 23);           // B in [2^(e-127), 2^(e-126))
  int f = 268 - e;                     // biased exponent of S = 2^(141 - e): B S in [2^14, 2^15)
  f = f > 227 ? 227 : (f < 1 ? 1 : f);
  bits = (unsigned)f << 23;
  float S;
#ifdef __CUDA_ARCH__
  S = __uint_as_float(bits);
#else
  memcpy(&S, &bits, 4);
#endif
  return S;
}
// x -> (hi, lo) pieces of x S, saturating at the fp16 range
__device__ __forceinline__ void mrhs_split_scaled(float x, float S, __half* hi, __half* lo) {
  float y = x * S;
  y = fminf(fmaxf(y, -65504.f), 65504.f);
  const __half h = __float2half_rn(y);
  *hi = h;
  *lo = __float2half_rn((y - __half2float(h)) * kMrhsLoScale);
}

// OK_W_PAULI (ok_pauli.cu): where element e (row-major 3x3) of a stored matrix sits for the site at `lane` of a 32-site block, in
// complex units from the matrix's base ((block * OK_W_PAULI_MATS + m) * 288).  The elements of a site are kept in PAIRS, so that
// a lane moves 16 bytes at a time in fp32 (one cp.async / LDS.128 per pair instead of two 8-byte ones): [pair e/2 : 4][site][2],
// then element 8 as [site].
__host__ __device__ inline int pauli_elem_index(int e, int lane) { return e < 8 ? (e >> 1) * 64 + lane * 2 + (e & 1) : 256 + lane; }

struct Geom {
  int L[4];
  int V;      // sites
  int nblk;   // ceil(V / 32)
};

struct WHeader {         // first OK_W_HEADER_BYTES of a W buffer (device) and its host mirror
  uint32_t magic;
  uint32_t layout;
  ok_params p;
};
static_assert(sizeof(WHeader) <= OK_W_HEADER_BYTES, "header too large");

struct Ctx {
  cudaStream_t stream = nullptr;
  void* work = nullptr;
  size_t work_bytes = 0;
  uint64_t launches = 0;
  int device = -1;          // ordinal bound at the first compute call (one device per process, ok.h)
  bool sync_check = false;  // OK_SYNC_CHECK=1: synchronise after every launch so an asynchronous fault names its kernel
  char err[512] = "no error";
};
Ctx& ctx();
// Binds the library to the current CUDA device at the first call; OK_EINVAL if a later call arrives on another
// device (the __constant__ tables and cached attributes are per device and are initialised once).
int bind_device();

int fail_cuda(cudaError_t e, const char* where);

#define OK_CUDA(call)                                         \
  do {                                                        \
    cudaError_t e__ = (call);                                 \
    if (e__ != cudaSuccess) return okd::fail_cuda(e__, #call); \
  } while (0)

#define OK_LAUNCHED(name)                                         \
  do {                                                            \
    okd::ctx().launches++;                                        \
    cudaError_t e__ = cudaGetLastError();                         \
    if (e__ == cudaSuccess && okd::ctx().sync_check) e__ = cudaStreamSynchronize(okd::ctx().stream); \
    if (e__ != cudaSuccess) return okd::fail_cuda(e__, name);     \
  } while (0)

bool valid_params(const ok_params* p);
Geom make_geom(const ok_params* p);
inline size_t real_bytes(const ok_params* p) { return p->precision == OK_FP64 ? 8 : 4; }
inline bool aligned16(const void* q) { return q && (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

// W handle table: header mirror keyed by device pointer (filled by pack/precalc, or by one
// synchronous header read the first time an unknown pointer is seen).
int remember_W(const void* W, const ok_params* p);   // also drops every record whose byte range overlaps [W, W + ok_W_bytes(p))
int refresh_W(const void* W, ok_params* p);          // always reads the device header (synchronises) and refreshes the record
int lookup_W(const void* W, ok_params* p);
inline const char* W_payload(const void* W) { return static_cast<const char*>(W) + OK_W_HEADER_BYTES; }
inline char* W_payload(void* W) { return static_cast<char*>(W) + OK_W_HEADER_BYTES; }

// One thread per (site, unit = 12 c4 + rhs): the unit's 8 floats (re[4], im[4] of components 4 c4 ..) become two 16-byte
// stores: [re hi4 | im hi4] at slot (n%12, hi) and [re lo4 | im lo4] at slot (n%12, lo), n = 2 rhs.
__device__ __forceinline__ void mrhs_store_operand(__half* __restrict__ rec, int c4, int rhs, const float4& re, const float4& im, float S) {
  __half h[16];
  mrhs_split_scaled(re.x, S, &h[0], &h[8]);  mrhs_split_scaled(re.y, S, &h[1], &h[9]);
  mrhs_split_scaled(re.z, S, &h[2], &h[10]); mrhs_split_scaled(re.w, S, &h[3], &h[11]);
  mrhs_split_scaled(im.x, S, &h[4], &h[12]); mrhs_split_scaled(im.y, S, &h[5], &h[13]);
  mrhs_split_scaled(im.z, S, &h[6], &h[14]); mrhs_split_scaled(im.w, S, &h[7], &h[15]);
  const int n = 2 * rhs, q = n / 12, nl = n % 12;
  __half* base = rec + ((q * 3 + c4) * 24) * 4;
  *reinterpret_cast<uint4*>(base + mrhs_op_slot(nl, 0) * 4) = *reinterpret_cast<const uint4*>(&h[0]);
  *reinterpret_cast<uint4*>(base + mrhs_op_slot(nl, 1) * 4) = *reinterpret_cast<const uint4*>(&h[8]);
}

// Stencil offsets in the term order of ok.h (host copy; device copies live in each TU).
extern const int8_t kOffsets[kTerms][4];

// ---- launchers (each enqueues on ctx().stream and returns an ok_status) -------------------
int launch_pack_spinor(const ok_params* p, const void* canon, void* packed, bool unpack);
int launch_pack_W(const ok_params* p, const void* canon, void* Wpayload, bool unpack);
int launch_apply(const ok_params* p, const void* Wpayload, const void* psi, void* out,
                 double* dot_partials /* nullable */, const void* dot_a, const void* dot_b);
int launch_precalc(const ok_params* p, const void* links, void* Wpayload, void* work);
int launch_precalc_window(const ok_params* p, const void* links, void* Wpayload, void* work, int tfold, int win_blk0, int win_nblk);
// t-slab decomposition (ok.h): p = the slab's own lattice
int launch_apply_range(const ok_params* p, const void* Wpayload, const void* psi, void* out, int blk0, int nblk);
int launch_apply_slab(const ok_params* p, const void* Wpayload, const void* psi_ext, void* out_ext, double* partials, const void* dot_a_ext,
                      const void* lo_peer = nullptr, const void* hi_peer = nullptr);
size_t bicgstab_slab_work_bytes(const ok_params* p);
size_t bicgstab_slab_shared_bytes(int nslab, int nranks);
int run_bicgstab_slabs(int nslab, const ok_params* const* ps, const void* const* Wpayloads, const void* const* srcs, void* const* xs,
                       double tol, int maxit, const ok_comm* comm, int* iters, double* resid);
const ok_slab_peers* slab_peers();   // what ok_slab_set_peers stored (nullptr: none)
int launch_apply_pauli(const ok_params* p, const void* Wpayload, const void* psi, void* out, double* dot_partials, const void* dot_a);
int launch_unpack_pauli(const ok_params* p, const void* Wpayload, void* canon);
int launch_apply_sparse(const ok_params* p, const void* Wpayload, const void* psi, void* out, double* dot_partials, const void* dot_a);
size_t precalc_work_bytes(const ok_params* p);
int run_bicgstab(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit,
                 int* iters, double* resid);
size_t bicgstab_work_bytes(const ok_params* p);
// CG on the normal equations (ok_cgnr.cu); workspace: bicgstab_work_bytes
int run_cgnr(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit, int* iters, double* resid);
// mixed precision (ok_mixed.cu)
size_t mixed_work_bytes(const ok_params* p);
int run_bicgstab_mixed(const ok_params* p64, const void* W64payload, const ok_params* p32, const void* W32payload, const void* src, void* x,
                       double tol, double inner_tol, int maxit, int max_outer, int* iters, int* outer, double* resid);
// nrhs = 12
// psi_op: operand records; psi_scale: 12 floats (device); out: fp32 records.  dot_a (fp32 records, nullable) with partials
// (gridDim rows of 36 doubles: per column Re<a,out>, Im<a,out>, ||out||^2; *npartials = rows written) fuses the reductions
// BiCGStab needs into the epilogue.  out_hdr (nullable): header whose `valid` is cleared.
int launch_apply_mrhs(const ok_params* p, const void* Wpayload, const __half* psi_op, const float* psi_scale, float* out,
                      MrhsVecHeader* out_hdr, const float* dot_a, double* partials, int* npartials);
// fp32 records -> operand records of the same vector, only if header.valid == 0 (two small kernels that return at once
// otherwise); sets header.scale and header.valid
int mrhs_ensure_operand(const ok_params* p, void* vec);
// operand records from fp32 records with given per-column scales (device pointer to 12 floats)
int mrhs_write_operand(const ok_params* p, const float* f32, __half* op, const float* scale);
int mrhs_apply_vec(const ok_params* p, const void* Wpayload, void* psi_vec, void* out_vec);   // ok_dirac_apply for nrhs = 12
int mrhs_max_apply_ctas();
int run_bicgstab_mrhs(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit,
                      int* iters, double* resid);
size_t bicgstab_mrhs_work_bytes(const ok_params* p);

}  // namespace okd
