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
// gives all four products from ONE series of 41 MMAs (M = 64, N = 48, K = 8); the epilogue adds the
// four quadrants.  Error: lo operands truncated again, ~2^-21 relative.
//
// One persistent CTA per SM, 20 specialised warps, sites dealt round-robin (site = blockIdx.x + k gridDim.x,
// so the CTAs sweep the lattice together and the gathered spinor records stay in L2).  The K dimension of a
// site is cut into 7 chunks of 4 stencil terms (48 k; the last chunk 36 + 4 zero k), pipelined through an
// 8-stage ring that spans site boundaries:
//   A operand (W)   lives in TENSOR MEMORY: 8 warps (two per TMEM lane quarter) stream the W chunk from HBM
//                   (evict-first 16-B loads, 3 chunks of prefetch in registers), form lo = w - trunc(w) and
//                   write hi and lo rows with tcgen05.st.16x256b (a thread's 4 registers are rows g, g+8 =
//                   hi, lo of one W row-part).  W never touches shared memory.
//   B operand (Psi) lives in shared memory: 6 warps gather the 4 neighbour records of the chunk from L2,
//                   split hi/lo and store both halves in the UMMA canonical K-major no-swizzle layout
//                   (core matrix = 8 rows x 16 B; LBO = 128 B, SBO = 1536 B).
//   MMA             one thread issues 6 (5) tcgen05.mma (A from TMEM, B from smem) per chunk into one of two
//                   64-lane x 48-column fp32 accumulators and commits to the stage's mbarrier.
//   epilogue        4 warps (one per lane quarter) read the accumulator with tcgen05.ld.16x256b, fold the
//                   hi/lo rows and columns, combine re/im and write the 1152-B output record through smem.
//   index           1 warp computes the 27 neighbour site indices of upcoming sites into a small smem ring.
// Layouts of W and of the spinor records: ok_internal.cuh (kLayoutMrhs).
#include "ok_internal.cuh"

namespace okd {

__constant__ int8_t c_moff[kTerms][4];
static bool g_moff_uploaded = false;

namespace {

constexpr int kStages = 8;                          // chunk ring (A slot in TMEM + B tile in smem)
constexpr int kSBO = 12 * 128;                      // 1536 B between 8-row groups of the B tile
constexpr int kLBO = 128;                           // between the two k-chunks (4 k each) of one MMA
constexpr int kBStage = 6 * kSBO;                   // n = 0..47 (hi 24 + lo 24): 9216 B
constexpr int kACols = kMrhsChunkK;                 // 48 TMEM columns per A slot
constexpr int kDCol0 = kStages * kACols;            // 384: accumulator 0; accumulator 1 at +64
constexpr int kTmemCols = 512;
constexpr int kNbrRing = 4;
constexpr int kAPrefetch = 3;                       // W chunks in flight per A warp (registers)

constexpr int kWarpMma = 0, kWarpB0 = 1, kWarpA = 4, kWarpEpi = 12, kWarpB1 = 16, kWarpIdx = 19;
constexpr int kWarps = 20, kThreads = kWarps * 32;

constexpr int kSmemB = kStages * kBStage;           // 73 728
constexpr int kSmemOut = 2 * kMrhsVecSiteFloats * 4;
constexpr int kSmemNbr = kNbrRing * 32 * 4;
constexpr int kSmemBytes = kSmemB + kSmemOut + kSmemNbr;

constexpr uint32_t kIdesc = (1u << 4) /*D f32*/ | (2u << 7) /*A tf32*/ | (2u << 10) /*B tf32*/ | ((48u >> 3) << 17) | ((64u >> 4) << 24);

struct Bars {
  uint64_t full[kStages], empty[kStages], dfull[2], dempty[2], nfull[kNbrRing], nempty[kNbrRing];
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {   // K-major, no swizzle, version 1
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(kLBO >> 4) << 16) | ((uint64_t)(kSBO >> 4) << 32) | ((uint64_t)1 << 46);
}

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done)
        : "r"(a), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ float tf32_lo(float v) { return v - __uint_as_float(__float_as_uint(v) & 0xFFFFE000u); }   // exact
__device__ __forceinline__ float4 tf32_lo(const float4& v) { return make_float4(tf32_lo(v.x), tf32_lo(v.y), tf32_lo(v.z), tf32_lo(v.w)); }

// 16 lanes x 8 columns: registers (r0, r1) -> lane t/4, columns 2(t%4), 2(t%4)+1 ; (r2, r3) -> lane t/4 + 8 (measured).
__device__ __forceinline__ void tmem_st_16x256(uint32_t taddr, float r0, float r1, float r2, float r3) {
  asm volatile("tcgen05.st.sync.aligned.16x256b.x1.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "f"(r0), "f"(r1), "f"(r2), "f"(r3) : "memory");
}
__device__ __forceinline__ void tmem_ld_16x256(uint32_t taddr, float& r0, float& r1, float& r2, float& r3) {
  asm volatile("tcgen05.ld.sync.aligned.16x256b.x1.b32 {%0, %1, %2, %3}, [%4];" : "=f"(r0), "=f"(r1), "=f"(r2), "=f"(r3) : "r"(taddr));
}

__device__ __forceinline__ int wrapc(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

struct AChunk {   // one thread's share of a W chunk: one row-part, 12 k values
  float4 v[3];
};

}  // namespace

__global__ void __launch_bounds__(kThreads, 1)
apply_mrhs_kernel(const float* __restrict__ W, const float4* __restrict__ psi, float4* __restrict__ out, Geom g) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint32_t s_tmem;
  __shared__ __align__(8) Bars bars;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint8_t* sB = smem;
  float* sOut = reinterpret_cast<float*>(smem + kSmemB);
  int* sNbr = reinterpret_cast<int*>(smem + kSmemB + kSmemOut);

  if (tid == 0) {
    for (int i = 0; i < kStages; ++i) { mbar_init(&bars.full[i], 7); mbar_init(&bars.empty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&bars.dfull[i], 1); mbar_init(&bars.dempty[i], 4); }
    for (int i = 0; i < kNbrRing; ++i) { mbar_init(&bars.nfull[i], 1); mbar_init(&bars.nempty[i], 6); }
    asm volatile("fence.mbarrier_init.release.cluster;");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  const int nsite = ((int)blockIdx.x < g.V) ? (g.V - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const int total = nsite * kMrhsChunks;   // chunk iterations of this CTA

  if (warp == kWarpMma) {
    // ------------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      for (int k = 0, it = 0; k < nsite; ++k) {
        const int d = k & 1;
        mbar_wait(&bars.dempty[d], (((uint32_t)k >> 1) & 1u) ^ 1u);   // epilogue drained this accumulator
        tc_fence_after();
        const uint32_t dcol = tmem + kDCol0 + 64 * d;
        for (int c = 0; c < kMrhsChunks; ++c, ++it) {
          const int st = it & (kStages - 1);
          mbar_wait(&bars.full[st], ((uint32_t)it / kStages) & 1u);
          tc_fence_after();
          const uint32_t a0 = tmem + st * kACols, b0 = smem_u32(sB + st * kBStage);
          const int nmma = (c < 6) ? 6 : 5;
          for (int j = 0; j < nmma; ++j) {
            const uint64_t db = umma_desc(b0 + j * 256);
            const uint32_t acc = (c > 0 || j > 0) ? 1u : 0u, zero = 0u;
            asm volatile(
                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n\t}\n" ::"r"(dcol),
                "r"(a0 + 8 * j), "l"(db), "r"(kIdesc), "r"(acc), "r"(zero)
                : "memory");
          }
          umma_commit(&bars.empty[st]);                 // frees the A slot and the B tile
          if (c == kMrhsChunks - 1) umma_commit(&bars.dfull[d]);
        }
      }
    }
    __syncwarp();
  } else if (warp >= kWarpA && warp < kWarpA + 8) {
    // ------------------------------------------------------------------ A producers: W (HBM) -> TMEM
    const int q = warp & 3, half = (warp - kWarpA) >> 2;
    const int gq = lane >> 2, cp = lane & 3;
    const bool active = gq < 6;                         // 6 row-parts per quarter; lanes 6,7 (+8) are pad rows
    const int rp = q * 6 + gq;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;

    auto load = [&](int it, AChunk& a) {
      const int k = it / kMrhsChunks, c = it - k * kMrhsChunks;
      const size_t n = (size_t)blockIdx.x + (size_t)k * gridDim.x;
      const float* tile = W + n * kMrhsWSiteFloats;
      if (!active) { a.v[0] = a.v[1] = a.v[2] = make_float4(0.f, 0.f, 0.f, 0.f); return; }
      if (c < 6) {
        const float4* p = reinterpret_cast<const float4*>(tile + c * kMrhsChunkFloats + rp * kMrhsChunkK) + cp;
        a.v[0] = __ldcs(p); a.v[1] = __ldcs(p + 4); a.v[2] = __ldcs(p + 8);
      } else {
        const float* row = tile + 6 * kMrhsChunkFloats + rp * kMrhsLastK;
        const float4* p = reinterpret_cast<const float4*>(row) + cp;
        a.v[0] = __ldcs(p); a.v[1] = __ldcs(p + 4);
        const float2 t2 = __ldcs(reinterpret_cast<const float2*>(row + 32) + cp);
        a.v[2] = make_float4(t2.x, t2.y, 0.f, 0.f);
      }
    };
    auto store = [&](int it, const AChunk& a) {
      const int st = it & (kStages - 1);
      mbar_wait(&bars.empty[st], (((uint32_t)it / kStages) & 1u) ^ 1u);
      tc_fence_after();
      const uint32_t t0 = tmem + lane_base + st * kACols;
#pragma unroll
      for (int J = 0; J < 3; ++J) {
        const float4 hi = a.v[J], lo = tf32_lo(hi);
        tmem_st_16x256(t0 + 16 * J, hi.x, hi.y, lo.x, lo.y);
        tmem_st_16x256(t0 + 16 * J + 8, hi.z, hi.w, lo.z, lo.w);   // last chunk: columns 40..47 are never read
      }
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.full[st]);
    };

    AChunk ring[kAPrefetch];
#pragma unroll
    for (int i = 0; i < kAPrefetch; ++i)
      if (half + 2 * i < total) load(half + 2 * i, ring[i]);
    for (int it = half; it < total; it += 2 * kAPrefetch) {
#pragma unroll
      for (int i = 0; i < kAPrefetch; ++i) {
        const int cur = it + 2 * i;
        if (cur < total) {
          store(cur, ring[i]);
          if (cur + 2 * kAPrefetch < total) load(cur + 2 * kAPrefetch, ring[i]);
        }
      }
    }
  } else if ((warp >= kWarpB0 && warp < kWarpB0 + 3) || (warp >= kWarpB1 && warp < kWarpB1 + 3)) {
    // ------------------------------------------------------------------ B producers: Psi (L2) -> smem
    const int grp = warp >= kWarpB1 ? 1 : 0;
    const int v = (warp - (grp ? kWarpB1 : kWarpB0)) * 32 + lane;   // 0..95; 72 units per record
    const bool active = v < 72;
    const int ng = v / 24, w = v - ng * 24;
    const uint32_t dst0 = (uint32_t)(ng * kSBO + w * 16);

    auto load = [&](int it, float4 (&r)[4]) {
      const int k = it / kMrhsChunks, c = it - k * kMrhsChunks;
      const int slot = k & (kNbrRing - 1);
      if (c < 2) mbar_wait(&bars.nfull[slot], ((uint32_t)k / kNbrRing) & 1u);   // first chunk of site k for this group
#pragma unroll
      for (int rec = 0; rec < 4; ++rec) {
        const int term = 4 * c + rec;
        r[rec] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (active && term < kTerms) {
          const int nn = sNbr[slot * 32 + term];
          r[rec] = __ldg(psi + (size_t)nn * (kMrhsVecSiteFloats / 4) + v);
        }
      }
      if (c >= 5) {   // last chunk of site k for this group: the index slot may be refilled
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars.nempty[slot]);
      }
    };
    auto store = [&](int it, const float4 (&r)[4]) {
      const int st = it & (kStages - 1);
      mbar_wait(&bars.empty[st], (((uint32_t)it / kStages) & 1u) ^ 1u);
      if (active) {
        uint8_t* base = sB + st * kBStage + dst0;
#pragma unroll
        for (int rec = 0; rec < 4; ++rec) {
          *reinterpret_cast<float4*>(base + rec * 384) = r[rec];
          *reinterpret_cast<float4*>(base + rec * 384 + 3 * kSBO) = tf32_lo(r[rec]);
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy stores -> visible to the tensor core
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.full[st]);
    };

    float4 ra[4], rb[4];
    if (grp < total) load(grp, ra);
    for (int it = grp; it < total; it += 4) {
      if (it + 2 < total) load(it + 2, rb);
      store(it, ra);
      if (it + 2 < total) {
        if (it + 4 < total) load(it + 4, ra);
        store(it + 2, rb);
      }
    }
  } else if (warp >= kWarpEpi && warp < kWarpEpi + 4) {
    // ------------------------------------------------------------------ epilogue: TMEM -> out
    const int q = warp & 3;
    const int gq = lane >> 2, cp = lane & 3;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const int et = tid - kWarpEpi * 32;   // 0..127
    for (int k = 0; k < nsite; ++k) {
      const int d = k & 1;
      mbar_wait(&bars.dfull[d], ((uint32_t)k >> 1) & 1u);
      tc_fence_after();
      const uint32_t t0 = tmem + lane_base + kDCol0 + 64 * d;
      float r[6][4];
#pragma unroll
      for (int j = 0; j < 6; ++j) tmem_ld_16x256(t0 + 8 * j, r[j][0], r[j][1], r[j][2], r[j][3]);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.dempty[d]);
      // rows g (hi) + g+8 (lo), columns c (B hi) + c+24 (B lo):  S[j][e], n = 8 j + 2 cp + e = 2 rhs + part_psi
      float S[3][2], O[3][2];
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) S[j][e] = (r[j][e] + r[j][2 + e]) + (r[j + 3][e] + r[j + 3][2 + e]);
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) O[j][e] = __shfl_xor_sync(0xffffffffu, S[j][e], 4);   // partner row-part (Re <-> Im of W)
      // row-part gq = 2 cr + part_w.  part_w = 0 lanes write Out_r = Sr[0] - Si[1]; part_w = 1 lanes write Out_i = Sr[1] + Si[0]
      if (gq < 6) {
        const int part = gq & 1, comp = 3 * q + (gq >> 1);
        float* so = sOut + d * kMrhsVecSiteFloats;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const float val = part == 0 ? S[j][0] - O[j][1] : O[j][1] + S[j][0];
          // out record: n = 2 rhs + part = 8 j + 2 cp + part
          so[(j * 3 + (comp >> 2)) * 32 + (2 * cp + part) * 4 + (comp & 3)] = val;
        }
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (et < kMrhsVecSiteFloats / 4) {
        const size_t n = (size_t)blockIdx.x + (size_t)k * gridDim.x;
        out[n * (kMrhsVecSiteFloats / 4) + et] = reinterpret_cast<const float4*>(sOut + d * kMrhsVecSiteFloats)[et];
      }
    }
  } else if (warp == kWarpIdx) {
    // ------------------------------------------------------------------ neighbour indices
    for (int k = 0; k < nsite; ++k) {
      const int slot = k & (kNbrRing - 1);
      mbar_wait(&bars.nempty[slot], (((uint32_t)k / kNbrRing) & 1u) ^ 1u);
      const int n = (int)blockIdx.x + k * (int)gridDim.x;
      const int x = n % g.L[0];
      int qq = n / g.L[0];
      const int y = qq % g.L[1];
      qq /= g.L[1];
      const int z = qq % g.L[2];
      const int t = qq / g.L[2];
      if (lane < kTerms) {
        const int xx = wrapc(x + c_moff[lane][0], g.L[0]);
        const int yy = wrapc(y + c_moff[lane][1], g.L[1]);
        const int zz = wrapc(z + c_moff[lane][2], g.L[2]);
        const int tt = wrapc(t + c_moff[lane][3], g.L[3]);
        sNbr[slot * 32 + lane] = xx + g.L[0] * (yy + g.L[1] * (zz + g.L[2] * tt));
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.nfull[slot]);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols));
}

int launch_apply_mrhs(const ok_params* p, const void* W, const void* psi, void* out) {
  if (p->nrhs != 12 || p->precision != OK_FP32) return OK_EINVAL;
  static int sm_count = 0;
  if (!g_moff_uploaded) {
    OK_CUDA(cudaMemcpyToSymbol(c_moff, kOffsets, sizeof(kOffsets)));
    int dev = 0;
    OK_CUDA(cudaGetDevice(&dev));
    OK_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    OK_CUDA(cudaFuncSetAttribute(apply_mrhs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    g_moff_uploaded = true;
  }
  Geom g = make_geom(p);
  const int grid = g.V < sm_count ? g.V : sm_count;   // one persistent CTA per SM (it owns all 512 TMEM columns)
  apply_mrhs_kernel<<<grid, kThreads, kSmemBytes, ctx().stream>>>(static_cast<const float*>(W), static_cast<const float4*>(psi),
                                                                 static_cast<float4*>(out), g);
  OK_LAUNCHED("apply_mrhs_kernel");
  return OK_SUCCESS;
}

}  // namespace okd
