// 12-right-hand-side Oktay-Kronfeld Dirac apply on the 5th-generation tensor cores:
//   Out(x)[12 x 12] = sum_{term} W_term(x)[12 x 12] Psi(x + offset_term)[12 x 12]        PAPER.md:53-55, Eq. (2.2)
// i.e. per site a complex 12 x 324 by 324 x 12 contraction, with a different W at every site.
//
// Real split, spinor on the M side:  D[n][w] = sum_k A[n][k] B[w][k],
//   A = Psi^T (n = 2 rhs + part, 24 rows),  B = [W_r ; W_i] (w = (row, part), 24 rows),  K = 324 (+12 pad),
//   Out_r = D(psi_r, W_r) - D(psi_i, W_i),  Out_i = D(psi_i, W_r) + D(psi_r, W_i)             (epilogue).
// Precision: every fp32 operand is carried as two fp16 pieces x = hi + lo / 2048 (22 significant bits; the
// spinor is first scaled per right-hand side by a power of two so that |x| < 2^15).  hi and lo are STACKED
// as rows on both sides, A = [Psi_hi ; Psi_lo], B = [W_hi ; W_lo] (N = 48), so one series of 21
// tcgen05.mma.kind::f16 (K = 16) per site yields all four products; the epilogue folds them with the
// weights 1, 2^-11, 2^-11, 2^-22 in fp32.
//
// BOTH operands are kept pre-split in HBM (4 bytes per real, like fp32; layouts in ok_internal.cuh):
//   W   per-site UMMA tile, HBM -> shared memory by one bulk copy, read by the tensor core; no thread touches it.
//   Psi per-site operand record written by whoever produced the vector (ok_pack_spinor, the BiCGStab update
//       kernels, mrhs_ensure_operand).  The producer warps only MOVE it: 8-byte loads with lane <-> A row (192
//       contiguous bytes per warp load, 2-3 L1 wavefronts) straight into tensor memory with tcgen05.st.32x32b --
//       no conversion arithmetic, no column-maximum pass in the apply.
//
// One persistent CTA per SM, 12 warps; sites are dealt in runs of consecutive x, runs round-robin over the CTAs (all CTAs
// sweep the lattice together, so the gathered records stay in L2).  Per site 7 K-stages of 4 stencil terms (48 k = 24
// TMEM columns):
//   W loader    1 thread: one 31 488-B bulk copy (cp.async.bulk, L2 evict-first) per site into a 4-slot smem ring.
//   Psi gather  3 warps: each of 9 lanes issues one 1152-B bulk copy of the operand record of neighbour t into a 3-slot smem ring
//               (a slot = the 27 records of a site).  No register ever waits on a gathered byte: the gathers of site k + 2
//               are in flight while the tensor core works on site k, however long L2 takes.
//   A movers    4 warps, (TMEM lane quarter q) x (A slot k % 2): when the records have landed AND the tensor core has
//               released the slot: 12 LDS.64 (lane <-> A row, conflict-free) + 3 tcgen05.st.32x32b.x8 per stage.  (The first
//               version of this kernel gathered straight into registers; its fourth stage could only be loaded after the slot
//               was free, which put one L2 round trip per site on the tensor core's critical path: ncu showed the MMA thread
//               waiting 40 % of the time for A.)
//   MMA         1 thread: 3 tcgen05.mma (M = 128: A rows = TMEM lanes; A from tensor memory, B from smem) per stage
//               into one of two 48-column fp32 accumulators; tcgen05.commit frees the A slot / the W slot.
//   epilogue    2 warps (one per lane quarter): tcgen05.ld.16x256b (hi and lo row of an n in one thread), fold the
//               pieces, combine Re/Im with one shuffle, coalesced 128-B stores; optionally the per-column reductions
//               <a, out>, ||out||^2 of BiCGStab in fp64 with a fixed order.
//   index       1 warp: the 27 neighbour site indices of upcoming sites into a small smem ring.
#include "ok_internal.cuh"

namespace okd {

__constant__ int8_t c_moff[kTerms][4];
static bool g_mrhs_ready = false;
static int g_sm_count = 0;

namespace {

constexpr int kASites = 2;                          // A ring (tensor memory): two whole sites
constexpr int kACols = 24;                          // TMEM columns per stage (48 fp16 k)
constexpr int kASiteCols = kMrhsStages * kACols;    // 168
constexpr int kWSlots = 4;                          // W ring (sites)
constexpr int kPsiSlots = 3;                        // ring of gathered operand records (sites)
constexpr int kPsiSlotBytes = kTerms * kMrhsOpSiteHalves * 2;     // 31 104
constexpr int kWSlotBytes = kMrhsStages * kMrhsStageHalves * 2;   // 32 256 (the last 768 B stay zero)
constexpr int kDCol0 = 384;                         // accumulator 0; accumulator 1 at +64 (A uses columns 0..335)
constexpr int kTmemCols = 512;
constexpr int kNbrRing = 8;
constexpr int kSBO = 128, kLBO = 768;

// warp w may touch TMEM lanes 32 (w % 4) ..; the A rows live in quarters 0 and 1
// movers: warps 0, 1 (slot 0) and 4, 5 (slot 1); epilogue: warps 8, 9
// gather: warps 7, 10, 11 (issuing a bulk copy costs a warp ~55 cycles, 27 of them would take the whole site period)
constexpr int kWarpMma = 2, kWarpTma = 3, kWarpIdx = 6, kWarpEpi = 8;
constexpr int kGatherWarps = 3, kGatherTerms = kTerms / kGatherWarps;
constexpr int kWarps = 12, kThreads = kWarps * 32;
static_assert(kGatherWarps * kGatherTerms == kTerms, "gather split");
static_assert(kASites == 2 && kASites * kASiteCols <= kDCol0, "A ring layout");

constexpr int kSmemW = kWSlots * kWSlotBytes;       // 129 024
constexpr int kSmemPsi = kPsiSlots * kPsiSlotBytes; // 93 312
constexpr int kSmemNbr = kNbrRing * 32 * 4;
constexpr int kDotRing = 4;                          // DOT: ring of `dot_a` records (1152 B each), filled by the W loader
constexpr int kDotRecBytes = kMrhsVecSiteFloats * 4;
constexpr int kSmemDot = kDotRing * kDotRecBytes;
constexpr int kSmemBytes = kSmemW + kSmemPsi + kSmemNbr + kSmemDot;

// D f32, A f16, B f16, both K-major, N = 48, M = 128: row r of A and D = TMEM lane r (rows 64..127 are never written or read;
// M = 64 costs the same 24 cycles but uses only the lower 16 lanes of a quarter)
constexpr uint32_t kIdesc = (1u << 4) | (0u << 7) | (0u << 10) | ((48u >> 3) << 17) | ((128u >> 4) << 24);

// Every barrier is waited on, phase after phase, by the same threads: a try_wait by parity cannot tell phase u from phase
// u - 2, so a warp that skipped a phase of a barrier (a slot that other warps fill in between) could pass early.
struct Bars {
  uint64_t afull[kASites], aempty[kASites], wfull[kWSlots], wempty[kWSlots], dfull[2], dempty[2], nfull[kNbrRing], nempty[kNbrRing];
  uint64_t vfull[kDotRing], vempty[kDotRing];   // DOT: the other vector of the reductions, one record per site
  uint64_t pfull[kPsiSlots], pempty[kPsiSlots]; // gathered operand records
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
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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

__device__ __forceinline__ int wrapc(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

__device__ __forceinline__ bool elect_one() {   // one lane of a converged warp
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}\n" : "=r"(pred));
  return pred != 0;
}

// work distribution: runs of `run` consecutive sites, run u -> CTA u % gridDim.x; iterates this CTA's site sequence
struct SiteIter {
  int n, r, run, skip;
  __device__ __forceinline__ explicit SiteIter(int run_) : n((int)blockIdx.x * run_), r(0), run(run_), skip(((int)gridDim.x - 1) * run_) {}
  __device__ __forceinline__ void next() {
    ++n;
    if (++r == run) { r = 0; n += skip; }
  }
};

__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

}  // namespace

// ------------------------------------------------------------------ fp32 records -> operand records
// max |psi| per right-hand side into header.maxbits: block = 4 sites x 72 float4 units; unit u of a record holds row n = u % 24
__global__ void __launch_bounds__(288) mrhs_colmax_kernel(const float4* __restrict__ psi, int V, MrhsVecHeader* __restrict__ hdr) {
  if (hdr->valid) return;
  __shared__ unsigned smax[12];
  if (threadIdx.x < 12) smax[threadIdx.x] = 0u;
  __syncthreads();
  const int unit = threadIdx.x % 72, slot = threadIdx.x / 72;
  const int rhs = (unit % 24) >> 1;
  unsigned m = 0u;
  for (long long s = (long long)blockIdx.x * 4 + slot; s < V; s += (long long)gridDim.x * 4) {
    const float4 v = __ldg(psi + s * 72 + unit);
    m = max(m, __float_as_uint(v.x) & 0x7fffffffu);
    m = max(m, __float_as_uint(v.y) & 0x7fffffffu);
    m = max(m, __float_as_uint(v.z) & 0x7fffffffu);
    m = max(m, __float_as_uint(v.w) & 0x7fffffffu);
  }
  atomicMax(&smax[rhs], m);
  __syncthreads();
  if (threadIdx.x < 12 && smax[threadIdx.x]) atomicMax(&hdr->maxbits[threadIdx.x], smax[threadIdx.x]);
}

// mode 0: scales from header.maxbits (skips if header.valid), the last CTA sets header.scale / valid; mode 1: given scales
template <int MODE>
__global__ void __launch_bounds__(288) mrhs_split_kernel(const float* __restrict__ f32, __half* __restrict__ op, int V,
                                                          MrhsVecHeader* __restrict__ hdr, const float* __restrict__ scale) {
  if (MODE == 0 && hdr->valid) return;
  const int unit = threadIdx.x % 36, slot = threadIdx.x / 36;
  const int rhs = unit % 12, c4 = unit / 12;
  const float S = MODE == 0 ? mrhs_scale_from_bound(__uint_as_float(hdr->maxbits[rhs])) : scale[rhs];
  for (long long s = (long long)blockIdx.x * 8 + slot; s < V; s += (long long)gridDim.x * 8) {
    const float* src = f32 + s * kMrhsVecSiteFloats + unit * 8;
    mrhs_store_operand(op + s * kMrhsOpSiteHalves, c4, rhs, *reinterpret_cast<const float4*>(src), *reinterpret_cast<const float4*>(src + 4), S);
  }
  if (MODE == 0) {
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
      if (atomicAdd(&hdr->done, 1u) + 1u == gridDim.x) {      // last CTA: publish
        for (int j = 0; j < 12; ++j) {
          hdr->scale[j] = mrhs_scale_from_bound(__uint_as_float(hdr->maxbits[j]));
          hdr->maxbits[j] = 0u;
        }
        hdr->done = 0u;
        __threadfence();
        hdr->valid = 1u;
      }
    }
  }
}

template <bool DOT>
__global__ void __launch_bounds__(kThreads, 1)
apply_mrhs_kernel(const uint8_t* __restrict__ W, const uint2* __restrict__ psi_op, const float* __restrict__ psi_scale, float* __restrict__ out,
                  Geom g, int run, MrhsVecHeader* __restrict__ out_hdr, const float* __restrict__ dot_a, double* __restrict__ partials) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint32_t s_tmem;
  __shared__ __align__(8) Bars bars;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint8_t* sW = smem;
  uint8_t* sPsi = smem + kSmemW;
  int* sNbr = reinterpret_cast<int*>(smem + kSmemW + kSmemPsi);
  const float* sDot = reinterpret_cast<const float*>(smem + kSmemW + kSmemPsi + kSmemNbr);

  if (tid == 0) {
    for (int i = 0; i < kASites; ++i) { mbar_init(&bars.aempty[i], 1); mbar_init(&bars.afull[i], 2); }
    for (int i = 0; i < kPsiSlots; ++i) { mbar_init(&bars.pfull[i], kGatherWarps); mbar_init(&bars.pempty[i], 4); }
    for (int i = 0; i < kWSlots; ++i) { mbar_init(&bars.wfull[i], 1); mbar_init(&bars.wempty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&bars.dfull[i], 1); mbar_init(&bars.dempty[i], 2); }
    for (int i = 0; i < kNbrRing; ++i) { mbar_init(&bars.nfull[i], 1); mbar_init(&bars.nempty[i], kGatherWarps); }
    for (int i = 0; i < kDotRing; ++i) { mbar_init(&bars.vfull[i], 1); mbar_init(&bars.vempty[i], 2); }
    asm volatile("fence.mbarrier_init.release.cluster;");
    if (blockIdx.x == 0 && out_hdr) {   // out's operand records no longer match; leave a clean header behind
      out_hdr->valid = 0u;
      out_hdr->done = 0u;
      for (int j = 0; j < 12; ++j) out_hdr->maxbits[j] = 0u;
    }
  }
  // the never-copied tail of every W slot (k chunk 5 of the last stage) must read as zero
  for (int i = tid; i < kWSlots * 48; i += kThreads)
    *reinterpret_cast<float4*>(sW + (i / 48) * kWSlotBytes + kMrhsWSiteBytes + (i % 48) * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = s_tmem;

  int nsite;   // sites of this CTA
  {
    const int nruns = (g.V + run - 1) / run, b = (int)blockIdx.x, G = (int)gridDim.x;
    const int mine = b < nruns ? (nruns - 1 - b) / G + 1 : 0;
    nsite = mine * run;
    if (mine > 0 && (nruns - 1) % G == b) nsite -= nruns * run - g.V;   // this CTA owns the (possibly short) last run
  }

  if (warp == kWarpMma) {
    // ------------------------------------------------------------------ MMA issuer (one elected thread, warp-uniform path)
    if (elect_one()) {
      // One wait per site and resource (a try_wait costs ~90 cycles even when the phase is complete)
      uint32_t wph = 0, dph = 1;
      int ws = 0;
      for (int k = 0; k < nsite; ++k) {
        const int d = k & 1, as = k & (kASites - 1);
        mbar_wait(&bars.dempty[d], dph);          // epilogue drained this accumulator
        dph ^= (uint32_t)d;                       // both accumulators used once -> next phase
        mbar_wait(&bars.wfull[ws], wph);          // W tile landed
        mbar_wait(&bars.afull[as], (uint32_t)(k / kASites) & 1u);   // the site's 7 A stages are in tensor memory
        tc_fence_after();
        const uint32_t dcol = tmem + kDCol0 + 64 * d;
        const uint32_t w0 = smem_u32(sW + ws * kWSlotBytes);
        const uint32_t a0 = tmem + as * kASiteCols;
#pragma unroll
        for (int c = 0; c < kMrhsStages; ++c) {
#pragma unroll
          for (int j = 0; j < 3; ++j) {
            const uint64_t db = umma_desc(w0 + c * (kMrhsStageHalves * 2) + j * (2 * kLBO));
            const uint32_t acc = (c > 0 || j > 0) ? 1u : 0u, zero = 0u;
            asm volatile(
                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n\t}\n" ::"r"(dcol),
                "r"(a0 + c * kACols + 8 * j), "l"(db), "r"(kIdesc), "r"(acc), "r"(zero)
                : "memory");
          }
        }
        umma_commit(&bars.aempty[as]);
        umma_commit(&bars.wempty[ws]);
        umma_commit(&bars.dfull[d]);
        if (++ws == kWSlots) { ws = 0; wph ^= 1u; }
      }
    }
    __syncwarp();
  } else if (warp == kWarpTma) {
    // ------------------------------------------------------------------ W loader: HBM -> smem ring, one bulk copy per site
    if (elect_one()) {
      uint64_t policy;
      asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(policy));
      SiteIter si(run);
      int ws = 0;
      uint32_t eph = 1;
      for (int k = 0; k < nsite; ++k, si.next()) {
        mbar_wait(&bars.wempty[ws], eph);
        mbar_expect_tx(&bars.wfull[ws], kMrhsWSiteBytes);
        const uint8_t* src = W + (size_t)si.n * kMrhsWSiteBytes;
        asm volatile(
            "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                smem_u32(sW + ws * kWSlotBytes)),
            "l"(src), "r"(kMrhsWSiteBytes), "r"(smem_u32(&bars.wfull[ws])), "l"(policy)
            : "memory");
        if (DOT) {   // the site's record of the other vector of the fused reductions -> smem (the epilogue never waits on HBM)
          const int vs = k & (kDotRing - 1);
          mbar_wait(&bars.vempty[vs], ((uint32_t)(k / kDotRing) & 1u) ^ 1u);
          mbar_expect_tx(&bars.vfull[vs], kDotRecBytes);
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                           smem_u32(sDot + vs * kMrhsVecSiteFloats)),
                       "l"(dot_a + (size_t)si.n * kMrhsVecSiteFloats), "r"(kDotRecBytes), "r"(smem_u32(&bars.vfull[vs]))
                       : "memory");
        }
        if (++ws == kWSlots) { ws = 0; eph ^= 1u; }
      }
    }
    __syncwarp();
  } else if (warp == kWarpIdx) {
    // ------------------------------------------------------------------ neighbour indices
    SiteIter si(run);
    int slot = 0;
    uint32_t eph = 1;
    for (int k = 0; k < nsite; ++k, si.next()) {
      mbar_wait(&bars.nempty[slot], eph);
      const int n = si.n;
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
      if (++slot == kNbrRing) { slot = 0; eph ^= 1u; }
    }
  } else if (warp == kWarpEpi || warp == kWarpEpi + 1) {
    // ------------------------------------------------------------------ epilogue: TMEM -> out (+ fused reductions)
    // thread (gq, cp) of half h: rows n%12 = gq + 8h (hi in TMEM lane 16h + gq, lo 8 lanes further), D columns 8i + 2cp + e
    const int q = warp & 3;
    const int gq = lane >> 2, cp = lane & 3;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const int n0 = 12 * q + gq, n1 = 12 * q + 8 + gq;        // n = 2 rhs + part of the two halves (n1 valid for gq < 4)
    const bool on1 = gq < 4;
    const float invS0 = 1.f / psi_scale[n0 >> 1], invS1 = on1 ? 1.f / psi_scale[n1 >> 1] : 0.f;
    const float kLo = 1.f / kMrhsLoScale;
    const float sgn = (gq & 1) ? 1.f : -1.f;
    const int off0 = n0 * 4 + cp, off1 = n1 * 4 + cp, pof0 = (n0 ^ 1) * 4 + cp, pof1 = (n1 ^ 1) * 4 + cp;
    double acc[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    SiteIter si(run);
    uint32_t fph = 0;
    for (int k = 0; k < nsite; ++k, si.next()) {
      const int d = k & 1;
      float a_own[2][3], a_par[2][3];
      if (DOT) {   // the other vector of the reductions: staged in smem by the W loader several sites ahead
        const int vs = k & (kDotRing - 1);
        mbar_wait(&bars.vfull[vs], (uint32_t)(k / kDotRing) & 1u);
        const float* ar = sDot + vs * kMrhsVecSiteFloats;
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          a_own[0][j] = ar[j * 96 + off0];
          a_par[0][j] = ar[j * 96 + pof0];
          a_own[1][j] = on1 ? ar[j * 96 + off1] : 0.f;
          a_par[1][j] = on1 ? ar[j * 96 + pof1] : 0.f;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars.vempty[vs]);
      }
      mbar_wait(&bars.dfull[d], fph);
      fph ^= (uint32_t)d;
      tc_fence_after();
      const uint32_t t0 = tmem + lane_base + kDCol0 + 64 * d;
      float r[2][24];   // r[h][4J + e] = D[hi row][col 8J + 2cp + e], r[h][4J + 2 + e] = D[lo row][same col]
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t th = t0 + ((uint32_t)(16 * h) << 16);
        asm volatile("tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                     : "=f"(r[h][0]), "=f"(r[h][1]), "=f"(r[h][2]), "=f"(r[h][3]), "=f"(r[h][4]), "=f"(r[h][5]), "=f"(r[h][6]), "=f"(r[h][7]),
                       "=f"(r[h][8]), "=f"(r[h][9]), "=f"(r[h][10]), "=f"(r[h][11]), "=f"(r[h][12]), "=f"(r[h][13]), "=f"(r[h][14]), "=f"(r[h][15])
                     : "r"(th));
        asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                     : "=f"(r[h][16]), "=f"(r[h][17]), "=f"(r[h][18]), "=f"(r[h][19]), "=f"(r[h][20]), "=f"(r[h][21]), "=f"(r[h][22]), "=f"(r[h][23])
                     : "r"(th + 32));
      }
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.dempty[d]);
      float* rec = out + (size_t)si.n * kMrhsVecSiteFloats;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        // fold psi lo (second row) and W lo (columns 24..47 = J 3..5):  Sv[j][e] for W row w = 8 j + 2 cp + e = (c = 4 j + cp, part e)
        const float invS = h ? invS1 : invS0;
        float Sv[3][2], O[3];
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const float hi = fmaf(r[h][4 * j + 2 + e], kLo, r[h][4 * j + e]);
            const float lo = fmaf(r[h][4 * (j + 3) + 2 + e], kLo, r[h][4 * (j + 3) + e]);
            Sv[j][e] = fmaf(lo, kLo, hi) * invS;
          }
#pragma unroll
        for (int j = 0; j < 3; ++j) O[j] = __shfl_xor_sync(0xffffffffu, Sv[j][1], 4);   // partner row: Re <-> Im of psi
        // even n (psi_r): Out_r = W_r psi_r - W_i psi_i ; odd n (psi_i): Out_i = W_r psi_i + W_i psi_r
        if (h == 0 || on1) {
          const int off = h ? off1 : off0;
#pragma unroll
          for (int j = 0; j < 3; ++j) {
            const float o = fmaf(sgn, O[j], Sv[j][0]);
            rec[j * 96 + off] = o;
            if (DOT) {   // this thread holds one part (Re for even n, Im for odd n) of out: <a,out> = sum conj(a) out
              const double od = (double)o;
              acc[h][0] += (double)a_own[h][j] * od;            // Re: a_r o_r + a_i o_i
              acc[h][1] += (double)(sgn * a_par[h][j]) * od;    // Im: a_r o_i - a_i o_r
              acc[h][2] += od * od;
            }
          }
        }
      }
    }
    if (DOT) {
      // the 8 lanes (n, n^1) x cp of a right-hand side: fixed-order butterfly, then one partial row per CTA
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          double v = acc[h][c];
          v += shfl_xor_d(v, 1);
          v += shfl_xor_d(v, 2);
          v += shfl_xor_d(v, 4);
          acc[h][c] = v;
        }
      if ((lane & 7) == 0) {
        double* row = partials + (size_t)blockIdx.x * 36;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          row[(n0 >> 1) * 3 + c] = acc[0][c];
          if (on1) row[(n1 >> 1) * 3 + c] = acc[1][c];
        }
      }
    }
  } else if (warp == 7 || warp >= 10) {
    // ------------------------------------------------------------------ Psi gather: 27 neighbour operand records -> smem slot
    const int gw = warp == 7 ? 0 : warp - 9;      // this warp issues the copies of terms 9 gw .. 9 gw + 8
    int ps = 0;
    uint32_t eph = 1;
    for (int k = 0; k < nsite; ++k) {
      const int ns = k & (kNbrRing - 1);
      mbar_wait(&bars.nfull[ns], (uint32_t)(k / kNbrRing) & 1u);
      mbar_wait(&bars.pempty[ps], eph);
      if (lane == 0) mbar_expect_tx(&bars.pfull[ps], kGatherTerms * kMrhsOpSiteHalves * 2);
      __syncwarp();
      if (lane < kGatherTerms) {
        const int term = gw * kGatherTerms + lane;
        const int nb = sNbr[ns * 32 + term];
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                         smem_u32(sPsi + ps * kPsiSlotBytes + term * (kMrhsOpSiteHalves * 2))),
                     "l"(psi_op + (size_t)nb * (kMrhsOpSiteHalves / 4)), "r"(kMrhsOpSiteHalves * 2), "r"(smem_u32(&bars.pfull[ps]))
                     : "memory");
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.nempty[ns]);
      if (++ps == kPsiSlots) { ps = 0; eph ^= 1u; }
    }
  } else if (warp < 6) {
    // ------------------------------------------------------------------ A movers: gathered records (smem) -> tensor memory
    // warp (q, as): A rows of lane quarter q, sites k = as, as + 2, ... of this CTA (A ring slot as).  Per stage 12 LDS.64 (lane
    // <-> A row: 24 consecutive 8-byte words, conflict-free) and 3 tcgen05.st.  Lanes 20-23 and 28-31 own no A row: they
    // re-read a neighbouring lane's row (any finite numbers do; their TMEM lanes are never read), so no lane is predicated off.
    const int q = warp & 3, as = warp >> 2;
    const int slot = lane < 20 ? lane : (lane < 28 ? lane - 4 : lane - 8);
    const uint32_t tbase = tmem + ((uint32_t)(32 * q) << 16) + as * kASiteCols;
    int ps = 0;
    uint32_t pph = 0;
    for (int k = 0; k < nsite; ++k, ps = (ps + 1 == kPsiSlots ? 0 : ps + 1), pph ^= (ps == 0 ? 1u : 0u)) {
      // every mover observes EVERY phase of the record ring and releases every slot (a wait by parity cannot tell phase u from
      // u - 2), also for the sites the other A slot's movers handle
      mbar_wait(&bars.pfull[ps], pph);
      if ((k & 1) != as) {
        if (lane == 0) mbar_arrive(&bars.pempty[ps]);
        continue;
      }
      const uint2* rec = reinterpret_cast<const uint2*>(sPsi + ps * kPsiSlotBytes) + q * 72 + slot;   // + 144 term + 24 g (8-byte units)
      auto load = [&](int c, uint2 (&w)[12]) {   // w[pair]: TMEM columns 2 pair, 2 pair + 1 of stage c
        if (c < 6) {       // pair = 4 g + t4: term 4 c + t4, components 4 g .. 4 g + 3
#pragma unroll
          for (int gg = 0; gg < 3; ++gg)
#pragma unroll
            for (int t4 = 0; t4 < 4; ++t4) w[4 * gg + t4] = rec[(4 * c + t4) * 144 + 24 * gg];
        } else {           // terms 24..26: pair = s = 3 (term - 24) + g, s < 9; pairs 9..11 are the zero pad (W's pad is zero too)
#pragma unroll
          for (int t3 = 0; t3 < 3; ++t3)
#pragma unroll
            for (int gg = 0; gg < 3; ++gg) w[3 * t3 + gg] = rec[(24 + t3) * 144 + 24 * gg];
          w[9] = w[10] = w[11] = make_uint2(0u, 0u);
        }
      };
      auto store = [&](int c, const uint2 (&w)[12]) {
        const uint32_t t0 = tbase + c * kACols;
#pragma unroll
        for (int j = 0; j < 3; ++j)
          asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(t0 + 8 * j), "r"(w[4 * j].x), "r"(w[4 * j].y),
                       "r"(w[4 * j + 1].x), "r"(w[4 * j + 1].y), "r"(w[4 * j + 2].x), "r"(w[4 * j + 2].y), "r"(w[4 * j + 3].x), "r"(w[4 * j + 3].y)
                       : "memory");
      };
      uint2 v[3][12];
      load(0, v[0]); load(1, v[1]); load(2, v[2]);
      // the tensor core has finished the site that used this A slot
      mbar_wait(&bars.aempty[as], ((uint32_t)(k / kASites) & 1u) ^ 1u);
      tc_fence_after();
      store(0, v[0]); load(3, v[0]);
      store(1, v[1]); load(4, v[1]);
      store(2, v[2]); load(5, v[2]);
      store(3, v[0]); load(6, v[0]);
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.pempty[ps]);     // every record byte this warp needs is in registers
      store(4, v[1]); store(5, v[2]); store(6, v[0]);
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.afull[as]);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols));
}

static int mrhs_init() {
  if (g_mrhs_ready) return OK_SUCCESS;
  OK_CUDA(cudaMemcpyToSymbol(c_moff, kOffsets, sizeof(kOffsets)));
  int dev = 0;
  OK_CUDA(cudaGetDevice(&dev));
  OK_CUDA(cudaDeviceGetAttribute(&g_sm_count, cudaDevAttrMultiProcessorCount, dev));
  OK_CUDA(cudaFuncSetAttribute(apply_mrhs_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
  OK_CUDA(cudaFuncSetAttribute(apply_mrhs_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
  g_mrhs_ready = true;
  return OK_SUCCESS;
}

int mrhs_max_apply_ctas() {
  if (mrhs_init()) return 1024;
  return g_sm_count;
}

int launch_apply_mrhs(const ok_params* p, const void* W, const __half* psi_op, const float* psi_scale, float* out, MrhsVecHeader* out_hdr,
                      const float* dot_a, double* partials, int* npartials) {
  if (p->nrhs != 12 || p->precision != OK_FP32) return OK_EINVAL;
  int st = mrhs_init();
  if (st) return st;
  Geom g = make_geom(p);
  const int run = g.L[0] < 8 ? 8 : (g.L[0] > 32 ? 32 : g.L[0]);   // consecutive sites per work unit (an x line when 8 <= Lx <= 32)
  const int nruns = (g.V + run - 1) / run;
  const int grid = nruns < g_sm_count ? nruns : g_sm_count;   // one persistent CTA per SM (it owns all 512 TMEM columns)
  if (dot_a) {
    apply_mrhs_kernel<true><<<grid, kThreads, kSmemBytes, ctx().stream>>>(static_cast<const uint8_t*>(W), reinterpret_cast<const uint2*>(psi_op),
                                                                          psi_scale, out, g, run, out_hdr, dot_a, partials);
    if (npartials) *npartials = grid;
  } else {
    apply_mrhs_kernel<false><<<grid, kThreads, kSmemBytes, ctx().stream>>>(static_cast<const uint8_t*>(W), reinterpret_cast<const uint2*>(psi_op),
                                                                           psi_scale, out, g, run, out_hdr, nullptr, nullptr);
  }
  OK_LAUNCHED("apply_mrhs_kernel");
  return OK_SUCCESS;
}

int mrhs_ensure_operand(const ok_params* p, void* vec) {
  int st = mrhs_init();
  if (st) return st;
  Geom g = make_geom(p);
  MrhsVecHeader* hdr = static_cast<MrhsVecHeader*>(vec);
  const int cgrid = (g.V + 3) / 4 < g_sm_count * 8 ? (g.V + 3) / 4 : g_sm_count * 8;
  mrhs_colmax_kernel<<<cgrid, 288, 0, ctx().stream>>>(reinterpret_cast<const float4*>(mrhs_f32(vec)), g.V, hdr);
  OK_LAUNCHED("mrhs_colmax_kernel");
  const int sgrid = (g.V + 7) / 8 < g_sm_count * 8 ? (g.V + 7) / 8 : g_sm_count * 8;
  mrhs_split_kernel<0><<<sgrid, 288, 0, ctx().stream>>>(mrhs_f32(vec), mrhs_op(vec, g.V), g.V, hdr, nullptr);
  OK_LAUNCHED("mrhs_split_kernel");
  return OK_SUCCESS;
}

int mrhs_write_operand(const ok_params* p, const float* f32, __half* op, const float* scale) {
  int st = mrhs_init();
  if (st) return st;
  Geom g = make_geom(p);
  const int sgrid = (g.V + 7) / 8 < g_sm_count * 8 ? (g.V + 7) / 8 : g_sm_count * 8;
  mrhs_split_kernel<1><<<sgrid, 288, 0, ctx().stream>>>(f32, op, g.V, nullptr, scale);
  OK_LAUNCHED("mrhs_split_kernel");
  return OK_SUCCESS;
}

int mrhs_apply_vec(const ok_params* p, const void* W, void* psi_vec, void* out_vec) {
  Geom g = make_geom(p);
  int st = mrhs_ensure_operand(p, psi_vec);
  if (st) return st;
  const MrhsVecHeader* hin = static_cast<const MrhsVecHeader*>(psi_vec);
  return launch_apply_mrhs(p, W, mrhs_op(psi_vec, g.V), hin->scale, mrhs_f32(out_vec), static_cast<MrhsVecHeader*>(out_vec), nullptr, nullptr,
                           nullptr);
}

}  // namespace okd
