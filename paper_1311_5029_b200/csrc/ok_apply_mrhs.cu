// 12-right-hand-side Oktay-Kronfeld Dirac apply on the 5th-generation tensor cores:
//   Out(x)[12 x 12] = sum_{term} W_term(x)[12 x 12] Psi(x + offset_term)[12 x 12]        PAPER.md:53-55, Eq. (2.2)
// i.e. per site a complex 12 x 324 by 324 x 12 contraction, with a different W at every site.
//
// Real split, spinor on the M side:  D[n][w] = sum_k A[n][k] B[w][k],
//   A = Psi^T (n = 2 rhs + part, 24 rows),  B = [W_r ; W_i] (w = (row, part), 24 rows),  K = 324 (+12 pad),
//   Out_r = D(psi_r, W_r) - D(psi_i, W_i),  Out_i = D(psi_i, W_r) + D(psi_r, W_i)             (epilogue).
// Precision: every fp32 operand is carried as two fp16 pieces x = hi + lo / 2048 (22 significant bits; the
// spinor is first scaled per right-hand side by a power of two so that |x| < 2^15).  hi and lo are STACKED
// as rows on both sides, A = [Psi_hi ; Psi_lo] (48 rows of M = 64), B = [W_hi ; W_lo] (N = 48), so one series
// of 21 tcgen05.mma.kind::f16 (K = 16) per site yields all four products; the epilogue folds them with the
// weights 1, 2^-11, 2^-11, 2^-22 in fp32.  W is stored pre-split in HBM (4 bytes per real, like fp32), so it
// goes HBM -> shared memory -> tensor core with no thread touching it.
//
// One persistent CTA per SM, 20 specialised warps; sites are dealt in runs of consecutive x (L1 reuse of the
// gathered spinor records), runs round-robin over the CTAs (so all CTAs sweep the lattice together and the
// records stay in L2).  Per site 7 K-stages of 4 stencil terms (48 k = 24 TMEM columns):
//   W loader   1 thread: one 31 488-B bulk copy (cp.async.bulk, L2 evict-first) per site into a 4-slot smem ring.
//   A producers 12 warps (4 per TMEM lane quarter, quarter q = rows n = 8q..8q+7): gather the 4 neighbour records
//              of a stage (three 16-B loads per thread, L1/L2), scale, split into fp16 hi/lo and write rows g
//              (hi) and g + 8 (lo) with tcgen05.st.16x256b into a 16-slot ring of 24 TMEM columns.
//   MMA        1 thread: 3 tcgen05.mma (A from tensor memory, B from smem) per stage into one of two
//              64-row x 48-column fp32 accumulators; tcgen05.commit frees the stage / the W slot.
//   epilogue   3 warps (one per lane quarter): tcgen05.ld.16x256b, fold pieces, combine Re/Im, coalesced stores.
//   index      1 warp: the 27 neighbour site indices of upcoming sites into a small smem ring.
// A first small kernel finds max |psi| per right-hand side (the power-of-two scales).
// Layouts of W and of the spinor records: ok_internal.cuh.
#include "ok_internal.cuh"

namespace okd {

__constant__ int8_t c_moff[kTerms][4];
__device__ unsigned g_colmax[12];   // bit patterns of max |psi| per right-hand side (atomicMax on non-negative floats)
static bool g_mrhs_ready = false;

namespace {

constexpr int kG = 4;                               // producer warps per lane quarter
constexpr int kARing = 16;                          // A ring slots
constexpr int kACols = 24;                          // TMEM columns per slot (48 fp16 k)
constexpr int kWSlots = 4;                          // W ring (sites)
constexpr int kWSlotBytes = kMrhsStages * kMrhsStageHalves * 2;   // 32 256 (the last 768 B stay zero)
constexpr int kDCol0 = kARing * kACols;             // 384: accumulator 0; accumulator 1 at +64
constexpr int kTmemCols = 512;
constexpr int kNbrRing = 8;
constexpr int kSBO = 128, kLBO = 768;

constexpr int kWarpMma = 3, kWarpTma = 7, kWarpIdx = 11, kWarpEpi = 4 * kG;   // warps 4i + 3 are free of TMEM lane duty
constexpr int kWarps = 4 * kG + 4, kThreads = kWarps * 32;
static_assert(kG >= 3 && kG <= 7, "producer groups");

constexpr int kSmemW = kWSlots * kWSlotBytes;       // 129 024
constexpr int kSmemNbr = kNbrRing * 32 * 4;
constexpr int kSmemBytes = kSmemW + kSmemNbr;

// D f32, A f16, B f16, both K-major, N = 48, M = 64: row r of A and D sits in TMEM lane 32 (r / 16) + r % 16, i.e. the 16 lanes
// (8 hi + 8 lo rows) each of the three producer quarters fills; M = 128 costs the same 24 cycles but reads 128 lanes
constexpr uint32_t kIdesc = (1u << 4) | (0u << 7) | (0u << 10) | ((48u >> 3) << 17) | ((64u >> 4) << 24);

struct Bars {
  uint64_t afull[kARing], aempty[kARing], wfull[kWSlots], wempty[kWSlots], dfull[2], dempty[2], nfull[kNbrRing], nempty[kNbrRing];
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

__device__ __forceinline__ uint32_t pack_h2(float lo_elem, float hi_elem) {   // low 16 bits = first argument
  const __half2 h = __floats2half2_rn(lo_elem, hi_elem);
  return *reinterpret_cast<const uint32_t*>(&h);
}

// power-of-two scale for one right-hand side from the bit pattern of max |psi|: max * S in [2^14, 2^15)
__device__ __forceinline__ void rhs_scale(unsigned maxbits, float* S, float* invS) {
  int e = (int)(maxbits >> 23);        // biased exponent, max in [2^(e-127), 2^(e-126))
  int f = 268 - e;                     // biased exponent of S = 2^(141 - e)
  f = f > 227 ? 227 : f;
  if (maxbits == 0u) f = 127;
  *S = __uint_as_float((uint32_t)f << 23);
  *invS = __uint_as_float((uint32_t)(254 - f) << 23);
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

}  // namespace

// max |psi| per right-hand side: block = 4 sites x 72 float4 units; unit u of a record holds row n = u % 24
__global__ void __launch_bounds__(288) colmax_kernel(const float4* __restrict__ psi, int V, unsigned* __restrict__ colmax) {
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
  if (threadIdx.x < 12 && smax[threadIdx.x]) atomicMax(&colmax[threadIdx.x], smax[threadIdx.x]);
}

__global__ void __launch_bounds__(kThreads, 1)
apply_mrhs_kernel(const uint8_t* __restrict__ W, const float4* __restrict__ psi, float* __restrict__ out, Geom g, int run,
                  const unsigned* __restrict__ colmax) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ uint32_t s_tmem;
  __shared__ __align__(8) Bars bars;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint8_t* sW = smem;
  int* sNbr = reinterpret_cast<int*>(smem + kSmemW);

  if (tid == 0) {
    for (int i = 0; i < kARing; ++i) { mbar_init(&bars.afull[i], 3); mbar_init(&bars.aempty[i], 1); }
    for (int i = 0; i < kWSlots; ++i) { mbar_init(&bars.wfull[i], 1); mbar_init(&bars.wempty[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&bars.dfull[i], 1); mbar_init(&bars.dempty[i], 3); }
    for (int i = 0; i < kNbrRing; ++i) { mbar_init(&bars.nfull[i], 1); mbar_init(&bars.nempty[i], 3 * kG); }
    asm volatile("fence.mbarrier_init.release.cluster;");
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
  const int total = nsite * kMrhsStages;   // stage iterations of this CTA

  if (warp == kWarpMma) {
    // ------------------------------------------------------------------ MMA issuer (one elected thread, warp-uniform path)
    if (elect_one()) {
      int st = 0;
      uint32_t aph = 0, wph = 0, dph = 1;
      int ws = 0;
      for (int k = 0; k < nsite; ++k) {
        const int d = k & 1;
        mbar_wait(&bars.dempty[d], dph);          // epilogue drained this accumulator
        dph ^= (uint32_t)d;                       // both accumulators used once -> next phase
        mbar_wait(&bars.wfull[ws], wph);          // W tile landed
        tc_fence_after();
        const uint32_t dcol = tmem + kDCol0 + 64 * d;
        const uint32_t w0 = smem_u32(sW + ws * kWSlotBytes);
#pragma unroll
        for (int c = 0; c < kMrhsStages; ++c) {
          mbar_wait(&bars.afull[st], aph);
          tc_fence_after();
          const uint32_t a0 = tmem + st * kACols;
#pragma unroll
          for (int j = 0; j < 3; ++j) {
            const uint64_t db = umma_desc(w0 + c * (kMrhsStageHalves * 2) + j * (2 * kLBO));
            const uint32_t acc = (c > 0 || j > 0) ? 1u : 0u, zero = 0u;
            asm volatile(
                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, {%5, %5, %5, %5}, p;\n\t}\n" ::"r"(dcol),
                "r"(a0 + 8 * j), "l"(db), "r"(kIdesc), "r"(acc), "r"(zero)
                : "memory");
          }
          umma_commit(&bars.aempty[st]);
          if (++st == kARing) { st = 0; aph ^= 1u; }
        }
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
  } else if (warp >= kWarpEpi && warp < kWarpEpi + 3) {
    // ------------------------------------------------------------------ epilogue: TMEM -> out
    const int q = warp & 3;
    const int gq = lane >> 2, cp = lane & 3;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const int nrow = 8 * q + gq;                 // n = 2 rhs + part
    float S, invS;
    rhs_scale(colmax[nrow >> 1], &S, &invS);
    const float kLo = 1.f / kMrhsLoScale;
    const float sgn = (gq & 1) ? 1.f : -1.f;
    float* obase = out + nrow * 4 + cp;
    SiteIter si(run);
    uint32_t fph = 0;
    for (int k = 0; k < nsite; ++k, si.next()) {
      const int d = k & 1;
      mbar_wait(&bars.dfull[d], fph);
      fph ^= (uint32_t)d;
      tc_fence_after();
      const uint32_t t0 = tmem + lane_base + kDCol0 + 64 * d;
      float r[24];   // r[4J + e] = D[row g (psi hi)][col 8J + 2cp + e], r[4J + 2 + e] = D[row g + 8 (psi lo)][same col]
      asm volatile("tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                   : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]),
                     "=f"(r[9]), "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15])
                   : "r"(t0));
      asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                   : "=f"(r[16]), "=f"(r[17]), "=f"(r[18]), "=f"(r[19]), "=f"(r[20]), "=f"(r[21]), "=f"(r[22]), "=f"(r[23])
                   : "r"(t0 + 32));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.dempty[d]);
      // fold psi lo (rows g + 8) and W lo (columns 24..47 = J 3..5):  Sv[j][e] for W row w = 8 j + 2 cp + e = (c = 4 j + cp, part e)
      float Sv[3][2], O[3];
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const float hi = fmaf(r[4 * j + 2 + e], kLo, r[4 * j + e]);
          const float lo = fmaf(r[4 * (j + 3) + 2 + e], kLo, r[4 * (j + 3) + e]);
          Sv[j][e] = fmaf(lo, kLo, hi) * invS;
        }
#pragma unroll
      for (int j = 0; j < 3; ++j) O[j] = __shfl_xor_sync(0xffffffffu, Sv[j][1], 4);   // partner row: Re <-> Im of psi
      // even g (psi_r): Out_r = W_r psi_r - W_i psi_i ; odd g (psi_i): Out_i = W_r psi_i + W_i psi_r
      float* rec = obase + (size_t)si.n * kMrhsVecSiteFloats;
#pragma unroll
      for (int j = 0; j < 3; ++j) rec[j * 96] = fmaf(sgn, O[j], Sv[j][0]);
    }
  } else if ((warp & 3) < 3 && warp < 4 * kG) {
    // ------------------------------------------------------------------ A producers: Psi (L1/L2) -> fp16 hi/lo -> TMEM
    // warp (q, gi) handles the stages it = gi, gi + kG, ... of this CTA's stage sequence (it = 7 k + c) for rows 8q..8q+7
    const int q = warp & 3, gi = warp >> 2;
    const int gq = lane >> 2, cp = lane & 3;
    const int nrow = 8 * q + gq;
    float S, invS;
    rhs_scale(colmax[nrow >> 1], &S, &invS);
    const float S2 = S * kMrhsLoScale;
    const float4* pbase = psi + nrow;                       // + 72 nn + 24 c4
    const uint32_t tbase = tmem + ((uint32_t)(32 * q) << 16);
    const int nmine = total > gi ? (total - gi + kG - 1) / kG : 0;

    // load side state: stage c of the site in index-ring slot lslot
    int lc = gi, lslot = 0;
    uint32_t lph = 0;
    auto load = [&](float4 (&v)[3]) {
      if (lc < kG) mbar_wait(&bars.nfull[lslot], lph);      // this warp's first stage of the site
      const int* nb = sNbr + lslot * 32;
      if (lc < 6) {
        const float4* rec = pbase + (size_t)nb[4 * lc + cp] * (kMrhsVecSiteFloats / 4);
        v[0] = __ldg(rec);
        v[1] = __ldg(rec + 24);
        v[2] = __ldg(rec + 48);
      } else {   // terms 24..26: slot s = 4 j + cp < 9 -> (term 24 + s/3, c4 = s%3)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const int s = 4 * j + cp;
          v[j] = make_float4(0.f, 0.f, 0.f, 0.f);
          if (s < 9) v[j] = __ldg(pbase + (size_t)nb[24 + s / 3] * (kMrhsVecSiteFloats / 4) + (s % 3) * 24);
        }
      }
      if (lc >= kMrhsStages - kG) {                         // this warp's last stage of the site: the index slot may be refilled
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars.nempty[lslot]);
      }
      lc += kG;
      if (lc >= kMrhsStages) {
        lc -= kMrhsStages;
        if (++lslot == kNbrRing) { lslot = 0; lph ^= 1u; }
      }
    };
    // store side state: A ring slot
    int st = gi;
    uint32_t eph = 1;
    auto store = [&](const float4 (&v)[3]) {
      uint32_t h[3][4];   // [j][0,1] = hi pieces of columns 8j + 2cp, +1 ; [j][2,3] = lo pieces
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const __half2 h01 = __floats2half2_rn(v[j].x * S, v[j].y * S), h23 = __floats2half2_rn(v[j].z * S, v[j].w * S);
        const float2 f01 = __half22float2(h01), f23 = __half22float2(h23);
        h[j][0] = *reinterpret_cast<const uint32_t*>(&h01);
        h[j][1] = *reinterpret_cast<const uint32_t*>(&h23);
        h[j][2] = pack_h2(fmaf(-kMrhsLoScale, f01.x, v[j].x * S2), fmaf(-kMrhsLoScale, f01.y, v[j].y * S2));
        h[j][3] = pack_h2(fmaf(-kMrhsLoScale, f23.x, v[j].z * S2), fmaf(-kMrhsLoScale, f23.y, v[j].w * S2));
      }
      mbar_wait(&bars.aempty[st], eph);
      tc_fence_after();
      const uint32_t t0 = tbase + st * kACols;
      asm volatile("tcgen05.st.sync.aligned.16x256b.x2.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(t0), "r"(h[0][0]), "r"(h[0][1]),
                   "r"(h[0][2]), "r"(h[0][3]), "r"(h[1][0]), "r"(h[1][1]), "r"(h[1][2]), "r"(h[1][3])
                   : "memory");
      asm volatile("tcgen05.st.sync.aligned.16x256b.x1.b32 [%0], {%1,%2,%3,%4};" ::"r"(t0 + 16), "r"(h[2][0]), "r"(h[2][1]), "r"(h[2][2]),
                   "r"(h[2][3])
                   : "memory");
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars.afull[st]);
      st += kG;
      if (st >= kARing) { st -= kARing; eph ^= 1u; }
    };

    float4 ra[3], rb[3], rc[3];   // two stages of gathers in flight behind the one being converted
    if (nmine > 0) load(ra);
    if (nmine > 1) load(rb);
    for (int i = 0; i < nmine; i += 3) {
      if (i + 2 < nmine) load(rc);
      store(ra);
      if (i + 1 < nmine) {
        if (i + 3 < nmine) load(ra);
        store(rb);
      }
      if (i + 2 < nmine) {
        if (i + 4 < nmine) load(rb);
        store(rc);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols));
}

int launch_apply_mrhs(const ok_params* p, const void* W, const void* psi, void* out) {
  if (p->nrhs != 12 || p->precision != OK_FP32) return OK_EINVAL;
  static int sm_count = 0;
  static unsigned* colmax = nullptr;
  if (!g_mrhs_ready) {
    OK_CUDA(cudaMemcpyToSymbol(c_moff, kOffsets, sizeof(kOffsets)));
    int dev = 0;
    OK_CUDA(cudaGetDevice(&dev));
    OK_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev));
    OK_CUDA(cudaFuncSetAttribute(apply_mrhs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    OK_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&colmax), g_colmax));
    g_mrhs_ready = true;
  }
  Geom g = make_geom(p);
  cudaStream_t st = ctx().stream;
  OK_CUDA(cudaMemsetAsync(colmax, 0, sizeof(unsigned) * 12, st));
  const int cgrid = (g.V + 3) / 4 < sm_count * 8 ? (g.V + 3) / 4 : sm_count * 8;
  colmax_kernel<<<cgrid, 288, 0, st>>>(static_cast<const float4*>(psi), g.V, colmax);
  OK_LAUNCHED("colmax_kernel");
  const int run = g.L[0] < 8 ? 8 : (g.L[0] > 32 ? 32 : g.L[0]);   // consecutive sites per work unit (an x line when 8 <= Lx <= 32)
  const int nruns = (g.V + run - 1) / run;
  const int grid = nruns < sm_count ? nruns : sm_count;   // one persistent CTA per SM (it owns all 512 TMEM columns)
  apply_mrhs_kernel<<<grid, kThreads, kSmemBytes, st>>>(static_cast<const uint8_t*>(W), static_cast<const float4*>(psi),
                                                        static_cast<float*>(out), g, run, colmax);
  OK_LAUNCHED("apply_mrhs_kernel");
  return OK_SUCCESS;
}

}  // namespace okd
