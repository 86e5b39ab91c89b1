// Internal declarations shared by the translation units of libokdirac (not part of the ABI).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "ok.h"

namespace okd {

constexpr int kBlock = OK_SITE_BLOCK;   // sites per block (= warp width: lane <-> site)
constexpr int kTerms = OK_NTERMS;
constexpr uint32_t kMagic = 0x4F4B5731u;   // "OKW1"
constexpr uint32_t kLayoutDense = 1;       // [block][term][row][c][site][16 B]
constexpr uint32_t kLayoutMrhs = 2;        // nrhs = 12: per-site tcgen05 A-operand tiles (ok_apply_mrhs.cu)

// ---- nrhs = 12 (tensor-core) layouts, fp32 only -------------------------------------------------
// W: per site the real-split A operand [W_r ; W_i] (24 row-parts x K = 324), cut along K into 7 chunks of
// 4 stencil terms (48 k; the last chunk holds 3 terms + 4 zero pad k = 40).  Inside a chunk the 24
// row-parts are ordered for the four TMEM lane quarters of ok_apply_mrhs.cu: rp = 6*(row/3) + 2*(row%3)
// + part (part 0 = Re, 1 = Im), each a contiguous run of 48 (40) floats.  Inside a run the k order is
// permuted so that the 16 B a thread loads are exactly the 4 values it stores with tcgen05.st.16x256b:
// float m = 16 J + 4 cp + 2 h + e  <->  TMEM column (= k in chunk) c = 16 J + 8 h + 2 cp + e
// (columns 32..39 of the last chunk are stored in natural order).  31 488 B per site.
constexpr int kMrhsChunkTerms = 4;
constexpr int kMrhsChunks = 7;
constexpr int kMrhsChunkK = 48;
constexpr int kMrhsLastK = 40;
constexpr int kMrhsChunkFloats = 24 * kMrhsChunkK;                          // 1152
constexpr int kMrhsWSiteFloats = 6 * kMrhsChunkFloats + 24 * kMrhsLastK;    // 7872
__host__ __device__ inline int mrhs_W_perm(int c) {   // column in chunk -> float position in the run
  return (c & ~15) | (((c >> 1) & 3) << 2) | (((c >> 3) & 1) << 1) | (c & 1);
}
__host__ __device__ inline int mrhs_W_rowpart(int row, int part) { return 6 * (row / 3) + 2 * (row % 3) + part; }
__host__ __device__ inline int mrhs_W_index(int term, int row, int col, int part) {
  const int chunk = term >> 2, c = (term & 3) * 12 + col, rp = mrhs_W_rowpart(row, part);
  if (chunk < 6) return chunk * kMrhsChunkFloats + rp * kMrhsChunkK + mrhs_W_perm(c);
  return 6 * kMrhsChunkFloats + rp * kMrhsLastK + (c < 32 ? mrhs_W_perm(c) : c);
}
__host__ __device__ inline int mrhs_W_pad_index(int q) {   // q = 0..95: the zero pad floats (k = 36..39 of the last chunk)
  return 6 * kMrhsChunkFloats + (q >> 2) * kMrhsLastK + 36 + (q & 3);
}
// spinor: per site the B operand [Psi_r , Psi_i] (24 x 12) as 9 core matrices:
// [n group n/8 = 0..2][k chunk c/4 = 0..2][n%8][c%4], n = 2*rhs + part, c = component.  1152 B per site.
constexpr int kMrhsVecSiteFloats = 288;
__host__ __device__ inline int mrhs_vec_index(int comp, int rhs, int part) {
  const int n = 2 * rhs + part;
  return ((n >> 3) * 3 + (comp >> 2)) * 32 + (n & 7) * 4 + (comp & 3);
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
size_t precalc_work_bytes(const ok_params* p);
int run_bicgstab(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit,
                 int* iters, double* resid);
size_t bicgstab_work_bytes(const ok_params* p);
// nrhs = 12
int launch_apply_mrhs(const ok_params* p, const void* Wpayload, const void* psi, void* out);
int run_bicgstab_mrhs(const ok_params* p, const void* Wpayload, const void* src, void* x, double tol, int maxit,
                      int* iters, double* resid);
size_t bicgstab_mrhs_work_bytes(const ok_params* p);

}  // namespace okd
