// 12-right-hand-side Oktay-Kronfeld Dirac apply on the 5th-generation tensor cores:
//   Out(x)[12 x 12] = sum_{term} W_term(x)[12 x 12] Psi(x + offset_term)[12 x 12]        PAPER.md:53-55, Eq. (2.2)
// i.e. per site a complex 12 x 324 by 324 x 12 contraction, a different W at every site.
//
// Real split: A = [W_r ; W_i] (24 x 324), B = [Psi_r , Psi_i] (324 x 24)  ->  P = A B (24 x 24),
//   Out_r = P_rr - P_ii,  Out_i = P_ri + P_ir   (epilogue).
// Precision: tcgen05 kind::tf32 truncates fp32 operands to 10 mantissa bits (measured on B200), far
// above the 2e-5 tolerance, so each operand is split a = hi + lo with hi = trunc_tf32(a) (what the
// tensor core sees when fed the raw fp32 word) and lo = a - hi (exact in fp32).  hi and lo are STACKED in
// the M and N dimensions of one accumulator:  [A_hi ; A_lo] (48 x K) times [B_hi , B_lo] (K x 48)
// gives all four products from ONE series of 41 MMAs (M = 64, N = 48, K = 8) instead of three series;
// the epilogue adds the four quadrants.  Error: lo operands truncated again, ~2^-20 relative.
//
// CTA = 128 threads, a run of consecutive sites, several CTAs per SM.  Per site, 7 pipeline stages of
// 4 stencil terms (K = 48; the last has 3 terms + a zero pad chunk, K = 40), double-buffered in smem:
//   fill:  all threads stream the W tile chunks (global, evict-first) and gather the neighbour
//          spinor records (L2), split hi/lo in registers, store both into the UMMA canonical
//          K-major no-swizzle layout (core matrix = 8 rows x 16 B; LBO = 128 B, SBO = 1536 B);
//   mma:   one thread issues 6 (5) tcgen05.mma into the 64-lane x 48-column fp32 accumulator in TMEM
//          and commits to the stage's mbarrier (which frees the buffer);
//   epilogue (per site): warps 0-2 read their 16 accumulator lanes with tcgen05.ld, fold hi/lo
//          columns, exchange through smem, combine re/im and write the output record.
// Layouts of W and of the spinor records: ok_internal.cuh (kLayoutMrhs).
#include "ok_internal.cuh"

namespace okd {

__constant__ int8_t c_moff[kTerms][4];
static bool g_moff_uploaded = false;

namespace {

constexpr int kStageChunks = 12;                    // k-chunks (4 k each) per stage = 4 terms
constexpr int kSBO = kStageChunks * 128;            // 1536 B between 8-row groups
constexpr int kLBO = 128;                           // between the two k-chunks of one MMA
constexpr int kAStage = 6 * kSBO;                   // rows 0..47 (hi 24 + lo 24); rows 48..63 read garbage from B
constexpr int kBStage = 6 * kSBO;                   // n 0..47
constexpr int kStage = kAStage + kBStage;           // 18 432 B
constexpr int kStagesPerSite = 7;
constexpr int kSmemT = 48 * 24 * 4;                 // epilogue exchange
constexpr int kSmemBytes = 2 * kStage + kSmemT;     // 41 472 B
constexpr int kTmemCols = 64;
constexpr uint32_t kIdesc = (1u << 4) /*D f32*/ | (2u << 7) /*A tf32*/ | (2u << 10) /*B tf32*/ | ((48u >> 3) << 17) | ((64u >> 4) << 24);

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {   // K-major, no swizzle, version 1
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(kLBO >> 4) << 16) | ((uint64_t)(kSBO >> 4) << 32) | ((uint64_t)1 << 46);
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}

__device__ __forceinline__ float4 tf32_lo(const float4& v) {   // v - trunc_tf32(v), exact
  float4 r;
  r.x = v.x - __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u);
  r.y = v.y - __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u);
  r.z = v.z - __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u);
  r.w = v.w - __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u);
  return r;
}

__device__ __forceinline__ int wrapc(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

}  // namespace

__global__ void __launch_bounds__(128, 5)
apply_mrhs_kernel(const float4* __restrict__ W, const float4* __restrict__ psi, float4* __restrict__ out, Geom g,
                  int sites_per_cta) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint32_t s_tmem;
  __shared__ __align__(8) uint64_t s_bar[3];   // [0],[1]: stage buffer free ; [2]: site accumulator complete
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  float* sT = reinterpret_cast<float*>(smem + 2 * kStage);

  if (tid == 0) {
    for (int i = 0; i < 3; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&s_bar[i])));
    asm volatile("fence.mbarrier_init.release.cluster;");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem = s_tmem;
  const uint32_t bar_free[2] = {smem_u32(&s_bar[0]), smem_u32(&s_bar[1])};
  const uint32_t bar_done = smem_u32(&s_bar[2]);

  const int site0 = blockIdx.x * sites_per_cta;
  const int nsite = min(sites_per_cta, g.V - site0);
  uint32_t it = 0;
  for (int ls = 0; ls < nsite; ++ls) {
    const int n = site0 + ls;
    const int x = n % g.L[0];
    int q = n / g.L[0];
    const int y = q % g.L[1];
    q /= g.L[1];
    const int z = q % g.L[2];
    const int t = q / g.L[2];
    const float4* Wsite = W + (size_t)n * (kMrhsWSiteFloats / 4);

    for (int s = 0; s < kStagesPerSite; ++s, ++it) {
      const uint32_t buf = it & 1u;
      mbar_wait(bar_free[buf], ((it >> 1) & 1u) ^ 1u);   // MMAs that read this buffer two stages ago are done
      uint8_t* sA = smem + buf * kStage;
      uint8_t* sB = sA + kAStage;
      const int nch = (s < 6) ? kStageChunks : 10;       // last stage: 9 chunks + the zero pad chunk
      // ---- A: 3 row groups x nch chunks x 8 rows, 16-B units; global order == smem order
      for (int u = tid; u < 3 * nch * 8; u += 128) {
        const int rg = u / (nch * 8), w = u - rg * (nch * 8);
        const float4 v = __ldcs(Wsite + (rg * kMrhsChunks + s * kStageChunks) * 8 + w);
        *reinterpret_cast<float4*>(sA + rg * kSBO + w * 16) = v;
        *reinterpret_cast<float4*>(sA + (3 + rg) * kSBO + w * 16) = tf32_lo(v);
      }
      // ---- B: 4 (3) neighbour records of 72 units: [n group 3][chunk 3][row 8]
      const int nterm = (s < 6) ? 4 : 3;
      for (int u = tid; u < nterm * 72; u += 128) {
        const int tl = u / 72, r = u - tl * 72;
        const int ng = r / 24, w = r - ng * 24;
        const int o = 4 * s + tl;
        const int xx = wrapc(x + c_moff[o][0], g.L[0]);
        const int yy = wrapc(y + c_moff[o][1], g.L[1]);
        const int zz = wrapc(z + c_moff[o][2], g.L[2]);
        const int tt = wrapc(t + c_moff[o][3], g.L[3]);
        const int nn = xx + g.L[0] * (yy + g.L[1] * (zz + g.L[2] * tt));
        const float4 v = __ldg(psi + (size_t)nn * (kMrhsVecSiteFloats / 4) + r);
        uint8_t* dst = sB + ng * kSBO + (tl * 24 + w) * 16;
        *reinterpret_cast<float4*>(dst) = v;
        *reinterpret_cast<float4*>(dst + 3 * kSBO) = tf32_lo(v);
      }
      if (s == 6 && tid < 48) {   // zero pad chunk (stage chunk 9) of the 6 n groups
        const int ng6 = tid >> 3, row = tid & 7;
        *reinterpret_cast<float4*>(sB + ng6 * kSBO + (9 * 8 + row) * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy stores -> visible to the tensor core
      __syncthreads();
      if (tid == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        const uint32_t a0 = smem_u32(sA), b0 = smem_u32(sB);
        const int nmma = nch >> 1;
        for (int j = 0; j < nmma; ++j) {
          const uint64_t da = umma_desc(a0 + j * 256), db = umma_desc(b0 + j * 256);
          const uint32_t acc = (s > 0 || j > 0) ? 1u : 0u, zero = 0u;
          asm volatile(
              "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
              "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, {%5, %5, %5, %5}, p;\n\t}\n" ::"r"(tmem),
              "l"(da), "l"(db), "r"(kIdesc), "r"(acc), "r"(zero)
              : "memory");
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar_free[buf]) : "memory");
        if (s == kStagesPerSite - 1)
          asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar_done) : "memory");
      }
    }

    // ---- epilogue of this site
    mbar_wait(bar_done, (uint32_t)ls & 1u);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (warp < 3) {   // accumulator row i lives in lane (i % 16) + 32 (i / 16): warp w holds rows 16w .. 16w+15
      uint32_t d[48];
      const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16);
#pragma unroll
      for (int c = 0; c < 48; c += 16)
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
            : "=r"(d[c + 0]), "=r"(d[c + 1]), "=r"(d[c + 2]), "=r"(d[c + 3]), "=r"(d[c + 4]), "=r"(d[c + 5]), "=r"(d[c + 6]),
              "=r"(d[c + 7]), "=r"(d[c + 8]), "=r"(d[c + 9]), "=r"(d[c + 10]), "=r"(d[c + 11]), "=r"(d[c + 12]), "=r"(d[c + 13]),
              "=r"(d[c + 14]), "=r"(d[c + 15])
            : "r"(taddr + c));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (lane < 16) {
        float* dstT = sT + (warp * 16 + lane) * 24;
#pragma unroll
        for (int c = 0; c < 24; ++c) dstT[c] = __uint_as_float(d[c]) + __uint_as_float(d[24 + c]);   // B_hi + B_lo columns
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (tid < 72) {   // one 16-B output unit: (n group, chunk c4, rhs-in-group p, part), components 4 c4 .. 4 c4 + 3
      const int row8 = tid & 7, c4 = (tid >> 3) % 3, ng = tid / 24;
      const int p = row8 >> 1, part = row8 & 1;
      const int col_same = 8 * ng + 2 * p + part, col_other = 8 * ng + 2 * p + (1 - part);
      float o[4];
#pragma unroll
      for (int ci = 0; ci < 4; ++ci) {
        const int r = 4 * c4 + ci;
        // S[m][n] = T[m][n] + T[24 + m][n]  (A_hi + A_lo rows); rows m < 12: W_r, m >= 12: W_i
        const float s_r_same = sT[r * 24 + col_same] + sT[(24 + r) * 24 + col_same];
        const float s_i_other = sT[(12 + r) * 24 + col_other] + sT[(36 + r) * 24 + col_other];
        // re: W_r Psi_r - W_i Psi_i ; im: W_r Psi_i + W_i Psi_r
        o[ci] = part == 0 ? s_r_same - s_i_other : s_r_same + s_i_other;
      }
      out[(size_t)n * (kMrhsVecSiteFloats / 4) + tid] = make_float4(o[0], o[1], o[2], o[3]);
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols));
}

int launch_apply_mrhs(const ok_params* p, const void* W, const void* psi, void* out) {
  if (p->nrhs != 12 || p->precision != OK_FP32) return OK_EINVAL;
  if (!g_moff_uploaded) {
    OK_CUDA(cudaMemcpyToSymbol(c_moff, kOffsets, sizeof(kOffsets)));
    g_moff_uploaded = true;
  }
  Geom g = make_geom(p);
  const int spc = 16;
  const int grid = (g.V + spc - 1) / spc;
  apply_mrhs_kernel<<<grid, 128, kSmemBytes, ctx().stream>>>(static_cast<const float4*>(W), static_cast<const float4*>(psi),
                                                           static_cast<float4*>(out), g, spc);
  OK_LAUNCHED("apply_mrhs_kernel");
  return OK_SUCCESS;
}

}  // namespace okd
