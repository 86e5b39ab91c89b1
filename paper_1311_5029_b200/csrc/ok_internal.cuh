// Internal declarations shared by the translation units of libokdirac (not part of the ABI).
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "ok.h"

namespace okd {

constexpr int kBlock = OK_SITE_BLOCK;   // sites per block (= warp width: lane <-> site)
constexpr int kTerms = OK_NTERMS;
constexpr uint32_t kMagic = 0x4F4B5731u;   // "OKW1"
constexpr uint32_t kLayoutDense = 1;       // [block][term][row][c][site][16 B]
constexpr uint32_t kLayoutBlock = 4;       // OK_W_BLOCK: [block][unit 2340][site][complex]   (ok_sparse.cuh)
constexpr uint32_t kLayoutConj = 6;        // OK_W_CONJ:  [block][unit 630][site][complex]
constexpr uint32_t kLayoutDS = 5;          // OK_W_DS:    [block][unit 1188][site][complex]
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
// spinor record (per site, fp32, 1152 B): [component/4 : 3][n = 2 rhs + part : 24][component%4]
constexpr int kMrhsVecSiteFloats = 288;
__host__ __device__ inline int mrhs_vec_index(int comp, int rhs, int part) {
  return ((comp >> 2) * 24 + 2 * rhs + part) * 4 + (comp & 3);
}

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
  int apply_variant = 0;
  uint64_t launches = 0;
  char err[512] = "no error";
};
Ctx& ctx();

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
    if (e__ != cudaSuccess) return okd::fail_cuda(e__, name);     \
  } while (0)

bool valid_params(const ok_params* p);
Geom make_geom(const ok_params* p);
inline size_t real_bytes(const ok_params* p) { return p->precision == OK_FP64 ? 8 : 4; }
inline bool aligned16(const void* q) { return q && (reinterpret_cast<uintptr_t>(q) & 15) == 0; }

// W handle table: header mirror keyed by device pointer (filled by pack/precalc, or by one
// synchronous header read the first time an unknown pointer is seen).
int remember_W(const void* W, const ok_params* p);
int lookup_W(const void* W, ok_params* p);
inline const char* W_payload(const void* W) { return static_cast<const char*>(W) + OK_W_HEADER_BYTES; }
inline char* W_payload(void* W) { return static_cast<char*>(W) + OK_W_HEADER_BYTES; }

// Stencil offsets in the term order of ok.h (host copy; device copies live in each TU).
extern const int8_t kOffsets[kTerms][4];

// ---- launchers (each enqueues on ctx().stream and returns an ok_status) -------------------
int launch_pack_spinor(const ok_params* p, const void* canon, void* packed, bool unpack);
int launch_pack_W(const ok_params* p, const void* canon, void* Wpayload, bool unpack);
int launch_apply(const ok_params* p, const void* Wpayload, const void* psi, void* out,
                 double* dot_partials /* nullable */, const void* dot_a, const void* dot_b);
int launch_precalc(const ok_params* p, const void* links, void* Wpayload, void* work);
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
int launch_apply_mrhs(const ok_params* p, const void* Wpayload, const void* psi, void* out);
int run_bicgstab_mrhs(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit,
                      int* iters, double* resid);
size_t bicgstab_mrhs_work_bytes(const ok_params* p);

}  // namespace okd
