// OK_W_PAULI: the paper's strongest compression of the precalculation matrices ("compress the 432 color
// blocks into 50"), SURVEY.md 8(f) item 2.  Every 6x6 block of Eqs. (2.6)-(2.12) is a Pauli sum  sum_k sigma_k (x) C_k  of 3x3
// colour matrices; counting the non-vanishing components block by block gives
//   W^0: 3 + 3    W^+_4: 1 + 3    W^+_i: 3 + 4 (x3)    W^{++}_ii: 1 + 1 (x3)    W^{++}_ij, W^{+-}_ij: 0 + 2 (x6)    = 49
// colour blocks for W^0 and the 13 positive-direction matrices (the opposite-direction ones follow from Eqs. 2.3, 2.10).
// Where two components of a term are the same matrix up to a constant of the action (D.C_0 = d1 U and S.C_i = a1 U of a hop;
// D = (c4/u0) P and S = ((c1+2c2)/2u0) sigma_i P of W_ii; the two sigma components of a pair term) it is stored once, so a
// site holds 37 colour matrices = 333 complex = 2 664 B in fp32 (dense: 31 104 B; OK_W_CONJ: 5 040 B).
//
// Stored matrices, index m (layout [block 32 sites][m][element pairs 4][site][2 complex], then [element 8][site]; pauli_elem_index):
//   0..2  i d0 B_m           3..5  s0 E_m             (Eq. 2.6; D^0, S^0 components sigma_m)
//   6     U_4                7..9  T_m = (cEE/2u0^4)(U_4 E_m(x+t) - E_m(x) U_4)                              (Eq. 2.7)
//   10+6i U_i   +1 S.C_0   +2 S.C_k   +3 S.C_l   +4 D.C_k   +5 D.C_l      (Eq. 2.8; i = 0..2, cyclic (i,k,l); hop_blocks_kernel)
//   28+i  P_ii = U_i(x) U_i(x+i)                                                                             (Eq. 2.9)
//   31+2q P_ij = U_i(x)U_j(x+i) + U_j(x)U_i(x+j)     32+2q  P_i-j = U_i(x)U_j(x-j+i)^dag + U_j(x-j)^dag U_i(x-j)   (2.11, 2.12)
// The boundary-condition signs are inside the links, as everywhere.
//
// Apply: out(x) = mass psi(x) + sum over 68 "uses" of a stored matrix: (matrix m at the neighbour site of stencil term t, or its
// adjoint for an opposite-direction term, Eqs. 2.3/2.10) times the four colour vectors of psi(x + offset_t), placed into the
// output by one or two Pauli placements  coef * sigma_k  in the diagonal (D) or off-diagonal (S) spin blocks.  The uses are a
// constexpr table written straight from the equations (make_uses below); the apply kernels are specialised on every entry
// at compile time (no table reads, no runtime flags, constant offsets), ok_unpack_W walks the same table at run time.
// 19.6 kflop per 2 856 B per site: this format is bound by the fp32 pipes, not by HBM.
#include "ok_internal.cuh"

namespace okd {

namespace {

constexpr int kPauliMats = OK_W_PAULI_MATS;   // 37
constexpr int kMaxUses = 80;
#ifndef OK_PAULI_MINB
#define OK_PAULI_MINB 4
#endif
#ifndef OK_PAULI_PARTS
#define OK_PAULI_PARTS 2
#endif
constexpr int kPauliParts = OK_PAULI_PARTS;   // launches per apply (see apply_pauli_part_kernel)
enum Coef { C_ONE = 0, C_MINUS, C_D1, C_A1, C_MA1, C_DII, C_SII, C_MSII, C_SIJ, C_MSIJ, C_COUNT };

// (plain ints: the kernel reads the table from constant memory every iteration, byte fields cost a PRMT each)
struct Placement {
  int kind;    // 0: D (diagonal spin blocks), 1: S (off-diagonal), -1: none
  int sigma;   // 0 = 1, 1..3 = sigma_x, sigma_y, sigma_z
  int coef;    // Coef
  int flags;   // D: bit 0 = upper-left block present, bit 1 = lower-right ; S: bit 2 = the lower-left block carries a minus
};
struct Use {
  int m, term, adj, np;
  Placement pl[2];
};
struct UseTable {
  int n;
  int first[kPauliParts + 1];   // part q (one launch) handles uses first[q] .. first[q+1]-1: whole terms, so the neighbour spinor is loaded once per term
  Use u[kMaxUses];
};

__constant__ UseTable c_uses;
__constant__ int8_t c_poff2[kTerms][4];
static bool g_pauli_ready = false;

constexpr Placement Dp(int sigma, int coef, int ul = 1, int lr = 1) { return Placement{0, sigma, coef, ul | (lr << 1)}; }
constexpr Placement Sp(int sigma, int coef, int llneg = 0) { return Placement{1, sigma, coef, llneg << 2}; }
constexpr Placement kNoPlacement{-1, 0, 0, 0};

constexpr void add_use(UseTable& t, int m, int term, int adj, Placement a, Placement b = kNoPlacement) {
  Use& u = t.u[t.n++];
  u.m = m; u.term = term; u.adj = adj; u.np = b.kind >= 0 ? 2 : 1;
  u.pl[0] = a;
  u.pl[1] = b;
}

// The 68 uses, term by term, from Eqs. (2.6)-(2.12) and the conjugation relations (2.3), (2.10):
// the opposite-direction matrix is [[D^dag, -S^dag], [-S^dag, D^dag]] of the blocks at the neighbour site.
// constexpr: the apply kernel is specialised on every entry at compile time; ok_unpack_W reads the same table at run time.
constexpr UseTable make_uses() {
  UseTable t{};
  t.n = 0;
  int start_of_term[kTerms + 1] = {};
  // term 0: W^0 = [[D0, S0], [-S0, D0]] + mass
  start_of_term[0] = t.n;
  for (int m = 0; m < 3; ++m) add_use(t, m, 0, 0, Dp(m + 1, C_ONE));
  for (int m = 0; m < 3; ++m) add_use(t, 3 + m, 0, 0, Sp(m + 1, C_ONE, 1));
  // terms 1..6: one-link hops +-i
  for (int i = 0; i < 3; ++i) {
    const int b = 10 + 6 * i, k = (i + 1) % 3, l = (i + 2) % 3;
    for (int neg = 0; neg < 2; ++neg) {
      const int term = 1 + 2 * i + neg;
      start_of_term[term] = t.n;
      add_use(t, b, term, neg, Dp(0, C_D1), Sp(i + 1, neg ? C_MA1 : C_A1));
      add_use(t, b + 1, term, neg, Sp(0, neg ? C_MINUS : C_ONE));
      add_use(t, b + 2, term, neg, Sp(k + 1, neg ? C_MINUS : C_ONE));
      add_use(t, b + 3, term, neg, Sp(l + 1, neg ? C_MINUS : C_ONE));
      add_use(t, b + 4, term, neg, Dp(k + 1, C_ONE));
      add_use(t, b + 5, term, neg, Dp(l + 1, C_ONE));
    }
  }
  // terms 7, 8: temporal hop; D = -U_4 sits in the lower-right block for +t and in the upper-left one for -t
  for (int neg = 0; neg < 2; ++neg) {
    start_of_term[7 + neg] = t.n;
    add_use(t, 6, 7 + neg, neg, Dp(0, C_MINUS, neg ? 1 : 0, neg ? 0 : 1));
    for (int m = 0; m < 3; ++m) add_use(t, 7 + m, 7 + neg, neg, Sp(m + 1, neg ? C_MINUS : C_ONE));
  }
  // terms 9..14: +-2i
  for (int i = 0; i < 3; ++i)
    for (int neg = 0; neg < 2; ++neg) {
      start_of_term[9 + 2 * i + neg] = t.n;
      add_use(t, 28 + i, 9 + 2 * i + neg, neg, Dp(0, C_DII), Sp(i + 1, neg ? C_MSII : C_SII));
    }
  // terms 15..26: pairs (x,y), (x,z), (y,z): +i+j, -i-j, +i-j, -i+j
  for (int q = 0; q < 3; ++q) {
    const int i = q == 2 ? 1 : 0, j = q == 0 ? 1 : 2;
    for (int w = 0; w < 4; ++w) {
      const int term = 15 + 4 * q + w, neg = w & 1, minus = w >= 2 ? 1 : 0;
      start_of_term[term] = t.n;
      const int ci = neg ? C_MSIJ : C_SIJ, cj = (neg != minus) ? C_MSIJ : C_SIJ;
      add_use(t, 31 + 2 * q + minus, term, neg, Sp(i + 1, ci), Sp(j + 1, cj));
    }
  }
  start_of_term[kTerms] = t.n;
  // the parts: whole terms each, as even as the term boundaries allow
  t.first[0] = 0;
  t.first[kPauliParts] = t.n;
  int term = 0;
  for (int w = 1; w < kPauliParts; ++w) {
    while (term < kTerms && start_of_term[term] < (t.n * w + kPauliParts / 2) / kPauliParts) ++term;
    t.first[w] = start_of_term[term];
  }
  return t;
}
constexpr UseTable kUses = make_uses();
static_assert(kUses.n == 68, "68 matrix uses per site");
// stencil offsets, term order of ok.h (compile-time copy of kOffsets; pauli_init checks the two agree)
constexpr int kOffC[kTerms][4] = {
    {0, 0, 0, 0},
    {1, 0, 0, 0},  {-1, 0, 0, 0}, {0, 1, 0, 0},  {0, -1, 0, 0}, {0, 0, 1, 0},  {0, 0, -1, 0},
    {0, 0, 0, 1},  {0, 0, 0, -1},
    {2, 0, 0, 0},  {-2, 0, 0, 0}, {0, 2, 0, 0},  {0, -2, 0, 0}, {0, 0, 2, 0},  {0, 0, -2, 0},
    {1, 1, 0, 0},  {-1, -1, 0, 0}, {1, -1, 0, 0}, {-1, 1, 0, 0},
    {1, 0, 1, 0},  {-1, 0, -1, 0}, {1, 0, -1, 0}, {-1, 0, 1, 0},
    {0, 1, 1, 0},  {0, -1, -1, 0}, {0, 1, -1, 0}, {0, -1, 1, 0}};

template <typename real> struct PV;
template <> struct PV<float> { using cx = float2; using vec = float4; static constexpr int NC = 6; };
template <> struct PV<double> { using cx = double2; using vec = double2; static constexpr int NC = 12; };

struct PauliArgs {
  Geom g;
  double coef[C_COUNT];
  double mass;
};
__constant__ float c_coef32[C_COUNT];
__constant__ double c_coef64[C_COUNT];
template <typename real> __device__ __forceinline__ real coef_of(int id);
template <> __device__ __forceinline__ float coef_of<float>(int id) { return c_coef32[id]; }
template <> __device__ __forceinline__ double coef_of<double>(int id) { return c_coef64[id]; }

__device__ __forceinline__ int wrapp(int x, int L) {
  x += (x < 0) ? L : 0;
  x -= (x >= L) ? L : 0;
  return x;
}

// v * f(sigma, al), f = sigma[al][src]: 1 (sigma_0, sigma_x), -/+ i (sigma_y: al = 0 / 1), +/- 1 (sigma_z)
template <typename cx, typename real>
__device__ __forceinline__ cx pauli_factor(cx v, int sigma, int al, real c) {
  if (sigma == 2) v = al == 0 ? cx{v.y, -v.x} : cx{-v.y, v.x};
  if (sigma == 3 && al == 1) c = -c;
  return cx{c * v.x, c * v.y};
}

// ---- the apply, specialised at compile time on every entry of kUses (no table reads, no runtime flags, constant offsets)
template <typename real>
struct PState {
  using cx = typename PV<real>::cx;
  using vec = typename PV<real>::vec;
  cx acc[12];
  cx phi[12];
  uint32_t ring16, ring8;   // fp32 only: shared-memory addresses of this lane's 16-byte and 8-byte columns of the warp's matrix ring (see use_ct)
  const cx* W;
  const vec* psi;
  int n, x, y, z, t;
  int L0, L1, L2, L3;
};

template <int BASE, int SIGMA, typename cx, typename real>
__device__ __forceinline__ void place_ct(cx (&acc)[12], const cx (&tv)[2][3], real c) {
#pragma unroll
  for (int ca = 0; ca < 3; ++ca) {
    if constexpr (sizeof(real) == 4) {   // packed: (Re, Im) of one output component per FFMA2
      if constexpr (SIGMA == 0 || SIGMA == 3) {
        const float c1 = SIGMA == 3 ? -c : c;
        acc[BASE + ca] = __ffma2_rn(make_float2(c, c), tv[0][ca], acc[BASE + ca]);
        acc[BASE + 3 + ca] = __ffma2_rn(make_float2(c1, c1), tv[1][ca], acc[BASE + 3 + ca]);
      } else if constexpr (SIGMA == 1) {
        acc[BASE + ca] = __ffma2_rn(make_float2(c, c), tv[1][ca], acc[BASE + ca]);
        acc[BASE + 3 + ca] = __ffma2_rn(make_float2(c, c), tv[0][ca], acc[BASE + 3 + ca]);
      } else {                            // sigma_y: -i v below the diagonal, +i v above: (v.y, -v.x) and (-v.y, v.x)
        acc[BASE + ca] = __ffma2_rn(make_float2(c, -c), make_float2(tv[1][ca].y, tv[1][ca].x), acc[BASE + ca]);
        acc[BASE + 3 + ca] = __ffma2_rn(make_float2(-c, c), make_float2(tv[0][ca].y, tv[0][ca].x), acc[BASE + 3 + ca]);
      }
    } else if constexpr (SIGMA == 0 || SIGMA == 3) {
      const real c1 = SIGMA == 3 ? -c : c;
      acc[BASE + ca].x = fma(c, tv[0][ca].x, acc[BASE + ca].x);
      acc[BASE + ca].y = fma(c, tv[0][ca].y, acc[BASE + ca].y);
      acc[BASE + 3 + ca].x = fma(c1, tv[1][ca].x, acc[BASE + 3 + ca].x);
      acc[BASE + 3 + ca].y = fma(c1, tv[1][ca].y, acc[BASE + 3 + ca].y);
    } else if constexpr (SIGMA == 1) {
      acc[BASE + ca].x = fma(c, tv[1][ca].x, acc[BASE + ca].x);
      acc[BASE + ca].y = fma(c, tv[1][ca].y, acc[BASE + ca].y);
      acc[BASE + 3 + ca].x = fma(c, tv[0][ca].x, acc[BASE + 3 + ca].x);
      acc[BASE + 3 + ca].y = fma(c, tv[0][ca].y, acc[BASE + 3 + ca].y);
    } else {
      acc[BASE + ca].x = fma(c, tv[1][ca].y, acc[BASE + ca].x);
      acc[BASE + ca].y = fma(-c, tv[1][ca].x, acc[BASE + ca].y);
      acc[BASE + 3 + ca].x = fma(-c, tv[0][ca].y, acc[BASE + 3 + ca].x);
      acc[BASE + 3 + ca].y = fma(c, tv[0][ca].x, acc[BASE + 3 + ca].y);
    }
  }
}

template <typename real, int U, int PI, int H>
__device__ __forceinline__ void placement_ct(PState<real>& st, const typename PV<real>::cx (&tv)[2][3]) {
  constexpr Placement pl = kUses.u[U].pl[PI];
  if constexpr (pl.kind == 0) {                 // D: output half = input half, if that diagonal block is present
    if constexpr (((pl.flags >> H) & 1) != 0) place_ct<6 * H, pl.sigma>(st.acc, tv, coef_of<real>(pl.coef));
  } else if constexpr (pl.kind == 1) {          // S: the other half; the lower-left block of W^0 is negated
    constexpr int TH = 1 - H;
    const real c = coef_of<real>(pl.coef);
    place_ct<6 * TH, pl.sigma>(st.acc, tv, (TH == 1 && (pl.flags & 4)) ? -c : c);
  }
}

// site index of x + offset(term T)
template <typename real, int T>
__device__ __forceinline__ int neighbour_ct(const PState<real>& st) {
  if constexpr (T == 0) return st.n;
  const int xx = wrapp(st.x + kOffC[T][0], st.L0), yy = wrapp(st.y + kOffC[T][1], st.L1);
  const int zz = wrapp(st.z + kOffC[T][2], st.L2), tt = wrapp(st.t + kOffC[T][3], st.L3);
  return xx + st.L0 * (yy + st.L1 * (zz + st.L2 * tt));
}
// where use U's stored matrix lives (own site, or the neighbour's for an opposite-direction term): the matrix's base in its
// 32-site block and the site's lane there; element e at base[pauli_elem_index(e, lane)] (ok_internal.cuh)
template <typename real, int U>
__device__ __forceinline__ const typename PV<real>::cx* matrix_base_ct(const PState<real>& st, int* lane) {
  constexpr Use u = kUses.u[U];
  const int nm = u.adj ? neighbour_ct<real, u.term>(st) : st.n;
  *lane = nm & 31;
  return st.W + ((size_t)(nm >> 5) * kPauliMats + u.m) * (9 * kBlock);
}
// fp32: the matrices reach the FMAs through a per-warp ring in shared memory filled by asynchronous copies (cp.async, SASS
// LDGSTS; four of 16 bytes -- an element pair -- and one of 8 per matrix and lane): with packed FMAs a use is ~150 issue slots,
// too short to hide an L2 / HBM round trip behind the four warps of a scheduler, and registers cannot hold several uses in
// flight.  Every lane copies and later reads only its own site's elements, so no barrier is needed: cp.async.wait_group
// orders a lane's reads after its own copies.
#ifndef OK_PAULI_RING
#define OK_PAULI_RING 4
#endif
constexpr int kRingDepth = OK_PAULI_RING;             // uses in flight per warp
constexpr int kRingSlotBytes = 9 * kBlock * 8;        // one 3x3 complex fp32 matrix for 32 sites: [pair 4][lane][16 B], [lane][8 B]
template <int U>
__device__ __forceinline__ void ring_issue_ct(const PState<float>& st, int slot) {
  int ln;
  const float2* p = matrix_base_ct<float, U>(st, &ln);
#pragma unroll
  for (int q = 0; q < 4; ++q)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(st.ring16 + slot * kRingSlotBytes + q * (kBlock * 16)), "l"(p + q * 64 + ln * 2)
                 : "memory");
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(st.ring8 + slot * kRingSlotBytes), "l"(p + 256 + ln) : "memory");
}

template <int U, int UEND, int D>
__device__ __forceinline__ void ring_prologue_ct(const PState<float>& st) {   // the first kRingDepth uses of the range: D = slot
  if constexpr (D < kRingDepth) {
    if constexpr (U < UEND) ring_issue_ct<U>(st, D);
    asm volatile("cp.async.commit_group;" ::: "memory");
    ring_prologue_ct<U + 1, UEND, D + 1>(st);
  }
}

// one use; FIRST: first use of this warp's range (a new term starts there by construction); UEND: end of the range
template <typename real, int U, int UBEG, int UEND, bool MASS>
__device__ __forceinline__ void use_ct(PState<real>& st, real mass) {
  constexpr bool FIRST = U == UBEG;
  using cx = typename PV<real>::cx;
  using vec = typename PV<real>::vec;
  constexpr int NC = PV<real>::NC;
  constexpr Use u = kUses.u[U];
  constexpr bool newterm = FIRST || kUses.u[U > 0 ? U - 1 : 0].term != u.term;
  cx C[9];
  if constexpr (sizeof(real) == 4) {
    if constexpr (FIRST) ring_prologue_ct<U, UEND, 0>(st);
    asm volatile("cp.async.wait_group %0;" ::"n"(kRingDepth - 1) : "memory");
    constexpr int slot = (U - UBEG) % kRingDepth;
#pragma unroll
    for (int q = 0; q < 4; ++q)
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                   : "=f"(C[2 * q].x), "=f"(C[2 * q].y), "=f"(C[2 * q + 1].x), "=f"(C[2 * q + 1].y)
                   : "r"(st.ring16 + slot * kRingSlotBytes + q * (kBlock * 16))
                   : "memory");
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(C[8].x), "=f"(C[8].y) : "r"(st.ring8 + slot * kRingSlotBytes) : "memory");
  } else {
    int ln;
    const cx* p = matrix_base_ct<real, U>(st, &ln);
#pragma unroll
    for (int e = 0; e < 9; ++e) C[e] = __ldg(p + pauli_elem_index(e, ln));
  }
  if constexpr (newterm) {
    constexpr int T = u.term;
    const int nn = neighbour_ct<real, T>(st);
    const vec* sp = st.psi + (size_t)(nn >> 5) * NC * kBlock + (nn & 31);
    if constexpr (sizeof(real) == 4) {
#pragma unroll
      for (int c = 0; c < 6; ++c) {
        const float4 v = __ldg(sp + c * kBlock);
        st.phi[2 * c] = cx{v.x, v.y};
        st.phi[2 * c + 1] = cx{v.z, v.w};
      }
    } else {
#pragma unroll
      for (int c = 0; c < 12; ++c) st.phi[c] = __ldg(sp + c * kBlock);
    }
    if constexpr (MASS && T == 0) {
#pragma unroll
      for (int r = 0; r < 12; ++r) { st.acc[r].x += mass * st.phi[r].x; st.acc[r].y += mass * st.phi[r].y; }
    }
  }
  if constexpr (sizeof(real) == 4) {
    // fp32: packed FMAs (fma.rn.f32x2, SASS FFMA2: two fp32 FMAs per issue slot on sm_100; one operand may be a broadcast scalar,
    // the other may be read with its halves swapped).  With w = C[ca][cb] (or C[cb][ca] for the adjoint) and v = (v.x, v.y):
    //   A += w.x (v.x, v.y) ,  B += w.y (v.y, v.x)   and   w v = A + (-B.x, B.y) ,  conj(w) v = A + (B.x, -B.y)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      cx tv[2][3];
#pragma unroll
      for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int ca = 0; ca < 3; ++ca) {
          float2 A = make_float2(0.f, 0.f), B = make_float2(0.f, 0.f);
#pragma unroll
          for (int cb = 0; cb < 3; ++cb) {
            const cx w = u.adj != 0 ? C[3 * cb + ca] : C[3 * ca + cb];
            const cx v = st.phi[3 * (2 * h + s) + cb];
            A = __ffma2_rn(make_float2(w.x, w.x), v, A);
            B = __ffma2_rn(make_float2(w.y, w.y), make_float2(v.y, v.x), B);
          }
          tv[s][ca] = __ffma2_rn(B, u.adj != 0 ? make_float2(1.f, -1.f) : make_float2(-1.f, 1.f), A);
        }
      if (h == 0) { placement_ct<real, U, 0, 0>(st, tv); placement_ct<real, U, 1, 0>(st, tv); }
      else { placement_ct<real, U, 0, 1>(st, tv); placement_ct<real, U, 1, 1>(st, tv); }
    }
    // this use's slot is free (its values are in registers and consumed): refill it kRingDepth uses ahead
    if constexpr (U + kRingDepth < UEND) ring_issue_ct<U + kRingDepth>(st, (U - UBEG) % kRingDepth);
    asm volatile("cp.async.commit_group;" ::: "memory");
  } else {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    cx tv[2][3];
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
      for (int ca = 0; ca < 3; ++ca) {
        real re = 0, im = 0;
#pragma unroll
        for (int cb = 0; cb < 3; ++cb) {
          const cx v = st.phi[3 * (2 * h + s) + cb];
          if constexpr (u.adj != 0) {
            const cx w = C[3 * cb + ca];
            re = fma(w.x, v.x, re); re = fma(w.y, v.y, re);
            im = fma(w.x, v.y, im); im = fma(-w.y, v.x, im);
          } else {
            const cx w = C[3 * ca + cb];
            re = fma(w.x, v.x, re); re = fma(-w.y, v.y, re);
            im = fma(w.x, v.y, im); im = fma(w.y, v.x, im);
          }
        }
        tv[s][ca] = cx{re, im};
      }
    if (h == 0) { placement_ct<real, U, 0, 0>(st, tv); placement_ct<real, U, 1, 0>(st, tv); }
    else { placement_ct<real, U, 0, 1>(st, tv); placement_ct<real, U, 1, 1>(st, tv); }
  }
  }   // fp64
}

template <typename real, int U, int UBEG, int UEND, bool MASS>
__device__ __forceinline__ void run_uses(PState<real>& st, real mass) {
  if constexpr (U < UEND) {
    use_ct<real, U, UBEG, UEND, MASS>(st, mass);
    run_uses<real, U + 1, UBEG, UEND, MASS>(st, mass);
  }
}

// kPauliParts launches per apply, each with its share of the uses: the straight-line code of all 68 specialised uses (about
// 13 k instructions) does not fit the instruction cache -- as ONE kernel it runs at 1.0 ms, slower than the table-driven loop
// it replaced (0.72 ms) -- while halves do: 0.40 ms with 2 parts (3: 0.47, 4: 0.49, 6: 0.59, 8: 0.62 ms; 20^3x64 fp32).  Part 0
// writes out (with the mass term), the later parts add to it, the last one also does the fused BiCGStab reductions; launches
// on one stream are ordered, so the sum has a fixed order.  lane <-> site, one warp per 32-site block, four blocks per CTA.
template <typename real, int PART, bool DOT>
__global__ void __launch_bounds__(128, sizeof(real) == 4 ? OK_PAULI_MINB : 1)
apply_pauli_part_kernel(const typename PV<real>::cx* __restrict__ W, const typename PV<real>::vec* __restrict__ psi,
                        typename PV<real>::vec* __restrict__ out, PauliArgs a, const typename PV<real>::vec* __restrict__ dot_a,
                        double* __restrict__ partials) {
  using cx = typename PV<real>::cx;
  using vec = typename PV<real>::vec;
  constexpr int NC = PV<real>::NC;
  const int lane = threadIdx.x & 31;
  const int blk = blockIdx.x * 4 + (threadIdx.x >> 5);
  if (blk >= a.g.nblk) return;
  int n = blk * kBlock + lane;
  const bool live = n < a.g.V;
  if (!live) n = 0;
  PState<real> st;
  st.n = n;
  st.L0 = a.g.L[0]; st.L1 = a.g.L[1]; st.L2 = a.g.L[2]; st.L3 = a.g.L[3];
  st.x = n % st.L0;
  int q = n / st.L0;
  st.y = q % st.L1;
  q /= st.L1;
  st.z = q % st.L2;
  st.t = q / st.L2;
  st.W = W; st.psi = psi;
  if constexpr (sizeof(real) == 4) {
    extern __shared__ __align__(16) uint8_t pauli_ring[];
    const uint32_t wring = (uint32_t)__cvta_generic_to_shared(pauli_ring) + (threadIdx.x >> 5) * (kRingDepth * kRingSlotBytes);
    st.ring16 = wring + lane * 16;
    st.ring8 = wring + 4 * (kBlock * 16) + lane * 8;
  }
  vec* ob = out + (size_t)blk * NC * kBlock + lane;
  if constexpr (PART == 0) {
#pragma unroll
    for (int r = 0; r < 12; ++r) st.acc[r] = cx{0, 0};
  } else if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      const float4 v = ob[c * kBlock];
      st.acc[2 * c] = cx{v.x, v.y};
      st.acc[2 * c + 1] = cx{v.z, v.w};
    }
  } else {
#pragma unroll
    for (int c = 0; c < 12; ++c) st.acc[c] = ob[c * kBlock];
  }
  run_uses<real, kUses.first[PART], kUses.first[PART], kUses.first[PART + 1], PART == 0>(st, (real)a.mass);
  if (!live) {
#pragma unroll
    for (int r = 0; r < 12; ++r) st.acc[r] = cx{0, 0};
  }
  if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int c = 0; c < 6; ++c) ob[c * kBlock] = make_float4(st.acc[2 * c].x, st.acc[2 * c].y, st.acc[2 * c + 1].x, st.acc[2 * c + 1].y);
  } else {
#pragma unroll
    for (int c = 0; c < 12; ++c) ob[c * kBlock] = st.acc[c];
  }
  if constexpr (DOT && PART == kPauliParts - 1) {
    const vec* ab = dot_a + (size_t)blk * NC * kBlock + lane;
    double d0 = 0.0, d1 = 0.0, d2 = 0.0;
#pragma unroll
    for (int r = 0; r < 12; ++r) {
      double ar, ai;
      if constexpr (sizeof(real) == 4) {
        const float4 v = ab[(r >> 1) * kBlock];
        ar = (r & 1) ? v.z : v.x;
        ai = (r & 1) ? v.w : v.y;
      } else {
        const double2 v = ab[r * kBlock];
        ar = v.x; ai = v.y;
      }
      const double vr = (double)st.acc[r].x, vi = (double)st.acc[r].y;
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
    if (lane == 0) {
      partials[(size_t)blk * 3 + 0] = d0;
      partials[(size_t)blk * 3 + 1] = d1;
      partials[(size_t)blk * 3 + 2] = d2;
    }
  }
}

// OK_W_PAULI -> canonical W[n][27][12][12] (ok_unpack_W): the same table, the placements written out as matrix entries
template <typename real>
__global__ void __launch_bounds__(128) unpack_pauli_kernel(const typename PV<real>::cx* __restrict__ W, typename PV<real>::cx* __restrict__ canon,
                                                           PauliArgs a) {
  using cx = typename PV<real>::cx;
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= (long long)a.g.V * kTerms) return;
  const int n = (int)(id / kTerms), term = (int)(id % kTerms);
  cx M[144];
  for (int e = 0; e < 144; ++e) M[e] = cx{0, 0};
  if (term == 0)
    for (int r = 0; r < 12; ++r) M[13 * r].x = (real)a.mass;
  int q = n / a.g.L[0];
  const int x = n % a.g.L[0], y = q % a.g.L[1];
  q /= a.g.L[1];
  const int z = q % a.g.L[2], t = q / a.g.L[2];
  for (int ui = 0; ui < c_uses.n; ++ui) {
    const Use u = c_uses.u[ui];
    if (u.term != term) continue;
    int nm = n;
    if (u.adj) {
      const int xx = wrapp(x + c_poff2[term][0], a.g.L[0]), yy = wrapp(y + c_poff2[term][1], a.g.L[1]);
      const int zz = wrapp(z + c_poff2[term][2], a.g.L[2]), tt = wrapp(t + c_poff2[term][3], a.g.L[3]);
      nm = xx + a.g.L[0] * (yy + a.g.L[1] * (zz + a.g.L[2] * tt));
    }
    const cx* cp = W + ((size_t)(nm >> 5) * kPauliMats + u.m) * (9 * kBlock);
    cx C[9];
    for (int ca = 0; ca < 3; ++ca)
      for (int cb = 0; cb < 3; ++cb) {
        cx v = cp[pauli_elem_index(u.adj ? 3 * cb + ca : 3 * ca + cb, nm & 31)];
        if (u.adj) v.y = -v.y;
        C[3 * ca + cb] = v;
      }
    for (int pi = 0; pi < u.np; ++pi) {
      const Placement pl = u.pl[pi];
      for (int th = 0; th < 2; ++th) {        // output spin half
        const int h = pl.kind == 0 ? th : 1 - th;   // input spin half
        real c = (real)a.coef[pl.coef];
        if (pl.kind == 0 && !((pl.flags >> h) & 1)) continue;
        if (pl.kind == 1 && th == 1 && (pl.flags & 4)) c = -c;
        const bool swap = pl.sigma == 1 || pl.sigma == 2;
        for (int al = 0; al < 2; ++al) {
          const int be = swap ? 1 - al : al;
          for (int ca = 0; ca < 3; ++ca)
            for (int cb = 0; cb < 3; ++cb) {
              const cx f = pauli_factor<cx, real>(C[3 * ca + cb], pl.sigma, al, c);
              cx& d = M[(6 * th + 3 * al + ca) * 12 + 6 * h + 3 * be + cb];
              d.x += f.x; d.y += f.y;
            }
        }
      }
    }
  }
  cx* dst = canon + (size_t)id * 144;
  for (int e = 0; e < 144; ++e) dst[e] = M[e];
}

int pauli_init() {
  if (g_pauli_ready) return OK_SUCCESS;
  for (int t = 0; t < kTerms; ++t)
    for (int d = 0; d < 4; ++d)
      if (kOffC[t][d] != kOffsets[t][d]) return OK_EINVAL;   // the compile-time copy of the stencil offsets must match ok.h's
  static const UseTable h_uses = kUses;
  OK_CUDA(cudaMemcpyToSymbol(c_uses, &h_uses, sizeof(UseTable)));
  OK_CUDA(cudaMemcpyToSymbol(c_poff2, kOffsets, sizeof(kOffsets)));
  g_pauli_ready = true;
  return OK_SUCCESS;
}

PauliArgs make_args(const ok_params* p) {
  PauliArgs a;
  a.g = make_geom(p);
  const double u0 = p->u0;
  const double a1 = 0.5 * (p->zeta - 2.0 * p->c1 - 12.0 * p->c2), d1 = -0.5 * (p->rs * p->zeta + 8.0 * p->c4);
  const double dii = p->c4 / u0, sii = (p->c1 + 2.0 * p->c2) / (2.0 * u0), sij = p->c2 / (2.0 * u0);
  a.coef[C_ONE] = 1.0; a.coef[C_MINUS] = -1.0;
  a.coef[C_D1] = d1; a.coef[C_A1] = a1; a.coef[C_MA1] = -a1;
  a.coef[C_DII] = dii; a.coef[C_SII] = sii; a.coef[C_MSII] = -sii;
  a.coef[C_SIJ] = sij; a.coef[C_MSIJ] = -sij;
  a.mass = u0 / (2.0 * p->kappa);
  return a;
}

template <typename real, int PART>
int launch_parts(unsigned grid, cudaStream_t st, const typename PV<real>::cx* W, const typename PV<real>::vec* psi, typename PV<real>::vec* out,
                 const PauliArgs& a, const typename PV<real>::vec* dot_a, double* partials) {
  if constexpr (PART < kPauliParts) {
    constexpr size_t smem = sizeof(real) == 4 ? 4 * kRingDepth * kRingSlotBytes : 0;   // 4 warps x ring (36 864 B: below the 48 KB default)
    if (PART == kPauliParts - 1 && partials) apply_pauli_part_kernel<real, PART, true><<<grid, 128, smem, st>>>(W, psi, out, a, dot_a, partials);
    else apply_pauli_part_kernel<real, PART, false><<<grid, 128, smem, st>>>(W, psi, out, a, nullptr, nullptr);
    OK_LAUNCHED("apply_pauli_part_kernel");
    return launch_parts<real, PART + 1>(grid, st, W, psi, out, a, dot_a, partials);
  }
  return OK_SUCCESS;
}

template <typename real>
int launch_pauli(const ok_params* p, const void* W, const void* psi, void* out, double* partials, const void* dot_a) {
  using cx = typename PV<real>::cx;
  using vec = typename PV<real>::vec;
  const PauliArgs a = make_args(p);
  static double last[C_COUNT + 1];   // the constants of the action of the last launch (one device, one thread per process: ok.h)
  static bool have = false;
  bool same = have;
  for (int k = 0; k < C_COUNT && same; ++k) same = last[k] == a.coef[k];
  if (!same) {
    float c32[C_COUNT];
    for (int k = 0; k < C_COUNT; ++k) { c32[k] = (float)a.coef[k]; last[k] = a.coef[k]; }
    OK_CUDA(cudaMemcpyToSymbolAsync(c_coef32, c32, sizeof(c32), 0, cudaMemcpyHostToDevice, ctx().stream));
    OK_CUDA(cudaMemcpyToSymbolAsync(c_coef64, a.coef, sizeof(a.coef), 0, cudaMemcpyHostToDevice, ctx().stream));
    have = true;
  }
  const cx* Wc = static_cast<const cx*>(W);
  const vec* ps = static_cast<const vec*>(psi);
  vec* o = static_cast<vec*>(out);
  const vec* da = static_cast<const vec*>(dot_a);
  const unsigned grid = (unsigned)((a.g.nblk + 3) / 4);
  cudaStream_t st = ctx().stream;
  return launch_parts<real, 0>(grid, st, Wc, ps, o, a, da, partials);
}

}  // namespace

int launch_apply_pauli(const ok_params* p, const void* W, const void* psi, void* out, double* partials, const void* dot_a) {
  if (p->nrhs != 1 || p->storage != OK_W_PAULI) return OK_EINVAL;
  if (int st = pauli_init()) return st;
  return p->precision == OK_FP64 ? launch_pauli<double>(p, W, psi, out, partials, dot_a) : launch_pauli<float>(p, W, psi, out, partials, dot_a);
}

int launch_unpack_pauli(const ok_params* p, const void* W, void* canon) {
  if (int st = pauli_init()) return st;
  const PauliArgs a = make_args(p);
  const long long total = (long long)a.g.V * kTerms;
  const unsigned grid = (unsigned)((total + 127) / 128);
  if (p->precision == OK_FP64)
    unpack_pauli_kernel<double><<<grid, 128, 0, ctx().stream>>>(static_cast<const double2*>(W), static_cast<double2*>(canon), a);
  else
    unpack_pauli_kernel<float><<<grid, 128, 0, ctx().stream>>>(static_cast<const float2*>(W), static_cast<float2*>(canon), a);
  OK_LAUNCHED("unpack_pauli_kernel");
  return OK_SUCCESS;
}

}  // namespace okd
