// W precalculation: the 27 "precalculation matrices" of Eq. (2.2) from
// SU(3) links, Eqs. (2.6)-(2.9), (2.11), (2.12) for the 14 positive matrices and the conjugation
// relations (2.3), (2.10) for the 13 negative ones.  One-time cost, bound by the W write.
//
// Arithmetic is fp64 throughout; W is rounded once to the storage precision.
//
// Representation: every 6x6 block of the paper is a Pauli combination  sum_{k=0..3} sigma_k (x) C_k
// (sigma_0 = 1) of four 3x3 colour matrices C_k.  The kernel computes the C_k ("P4") of the
// diagonal block A and of the off-diagonal block B of a term, from which the 12x12 entries follow:
//   (a,a')=(0,0): C0+C3   (1,1): C0-C3   (0,1): C1 - i C2   (1,0): C1 + i C2 .
// With B_k, E_k the clover fields (DESIGN.md R-F), U = U_i(x), cyclic (i,k,l), Eq. (2.8) reduces to
//   S^+_i: C0 = i cs (U B_i(x+i) + B_i(x) U), C_i = (zeta-2c1-12c2)/2 U,
//          C_k = cs (U B_l(x+i) - B_l(x) U),  C_l = -cs (U B_k(x+i) - B_k(x) U),   cs = c3/(2 u0^4)
//   D^+_i: C0 = -(rs zeta+8c4)/2 U, C_i = 0,
//          C_k =  i cg G_l + i c5/u0^4 (U B_k(x+i) + B_k(x) U),
//          C_l = -i cg G_k + i c5/u0^4 (U B_l(x+i) + B_l(x) U),   cg = (c5/4)(u0^-2 - u0^-4),
//   G_m = U_m(x)U_i(x+m)U_m(x+i)^dag - U_m(x-m)^dag U_i(x-m) U_m(x-m+i)   (staples).
// Negative matrices are NOT read from another site's W: the positive blocks are recomputed at
// the shifted site and conjugated, so the kernel has no inter-site dependency.
// Boundary conditions: U_mu(x) is multiplied by bc[mu] on the last slice of axis mu at load
// time (DESIGN.md R-BC); closed loops are unaffected, every hop across the boundary gets one sign.
#include "ok_internal.cuh"
#include "ok_sparse.cuh"

namespace okd {

struct cm3 {
  double2 e[9];
};

struct PrecalcArgs {
  Geom g;
  int bc[4];
  int Vpad;
  int mrhs;                    // 1: write the nrhs = 12 tensor-core tile layout (ok_internal.cuh)
  int storage;                 // OK_W_DENSE / OK_W_BLOCK / OK_W_DS (ok_sparse.cuh)
  int pair;                    // 1: the thread of a positive-direction term also writes the opposite term of the neighbour site
  int posonly;                 // 1: grid over W^0 and the 13 positive-direction terms only (pair, or OK_W_CONJ)
  int blk0;                    // first 32-site block of this launch (t-slab: the first interior block of the extended link window)
  int tfold;                   // time slice whose U_4 carries bc[3] (L[3] - 1 on a whole lattice; t-slab: where global T - 1 sits, or -1)
  double mass;                 // u0 / (2 kappa)
  double d0, s0;               // D^0, S^0 prefactors (Eq. 2.6)
  double s4;                   // c_EE / (2 u0^4)      (Eq. 2.7)
  double a1, cs, d1, cg, c5u;  // Eq. (2.8)
  double dii, sii;             // c4/u0, (c1+2c2)/(2u0) (Eq. 2.9)
  double sij;                  // c2/(2u0)             (Eqs. 2.11, 2.12)
};

__constant__ int8_t c_poff[kTerms][4];
__constant__ int c_qrun[3][kTerms][2][4];   // run offsets of the reduced formats (ok_sparse.cuh)
static bool g_poff_uploaded = false;

// ------------------------------------------------------------------------- complex 3x3 algebra
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }   // a * conj(b)
__device__ __forceinline__ double2 cconjmul(double2 a, double2 b) { return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }  // conj(a) * b

__device__ __forceinline__ cm3 zero3() {
  cm3 r;
#pragma unroll
  for (int i = 0; i < 9; ++i) r.e[i] = make_double2(0.0, 0.0);
  return r;
}
// s += a b, s += a conj(b), s += conj(a) b: four DFMA each (written out so that no product is rounded on its own and added later:
// the clover and hop-block kernels are bound by the fp64 pipe)
__device__ __forceinline__ void cmac(double2& s, double2 a, double2 b) {
  s.x = fma(a.x, b.x, s.x); s.x = fma(-a.y, b.y, s.x);
  s.y = fma(a.x, b.y, s.y); s.y = fma(a.y, b.x, s.y);
}
__device__ __forceinline__ void cmacc(double2& s, double2 a, double2 b) {   // a * conj(b)
  s.x = fma(a.x, b.x, s.x); s.x = fma(a.y, b.y, s.x);
  s.y = fma(a.y, b.x, s.y); s.y = fma(-a.x, b.y, s.y);
}
__device__ __forceinline__ void cconjmac(double2& s, double2 a, double2 b) {   // conj(a) * b
  s.x = fma(a.x, b.x, s.x); s.x = fma(a.y, b.y, s.x);
  s.y = fma(a.x, b.y, s.y); s.y = fma(-a.y, b.x, s.y);
}
__device__ cm3 mul(const cm3& A, const cm3& B) {   // A B
  cm3 r;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double2 s = cmul(A.e[3 * i], B.e[j]);
#pragma unroll
      for (int k = 1; k < 3; ++k) cmac(s, A.e[3 * i + k], B.e[3 * k + j]);
      r.e[3 * i + j] = s;
    }
  return r;
}
__device__ cm3 mul_nd(const cm3& A, const cm3& B) {   // A B^dag
  cm3 r;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double2 s = cmulc(A.e[3 * i], B.e[3 * j]);
#pragma unroll
      for (int k = 1; k < 3; ++k) cmacc(s, A.e[3 * i + k], B.e[3 * j + k]);
      r.e[3 * i + j] = s;
    }
  return r;
}
__device__ cm3 mul_dn(const cm3& A, const cm3& B) {   // A^dag B
  cm3 r;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double2 s = cconjmul(A.e[i], B.e[j]);
#pragma unroll
      for (int k = 1; k < 3; ++k) cconjmac(s, A.e[3 * k + i], B.e[3 * k + j]);
      r.e[3 * i + j] = s;
    }
  return r;
}
__device__ __forceinline__ cm3 adj(const cm3& A) {
  cm3 r;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) r.e[3 * i + j] = make_double2(A.e[3 * j + i].x, -A.e[3 * j + i].y);
  return r;
}
// r += (cr + i ci) * A
__device__ __forceinline__ void axpy(cm3& r, double cr, double ci, const cm3& A) {
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    r.e[i].x = fma(cr, A.e[i].x, r.e[i].x); r.e[i].x = fma(-ci, A.e[i].y, r.e[i].x);
    r.e[i].y = fma(cr, A.e[i].y, r.e[i].y); r.e[i].y = fma(ci, A.e[i].x, r.e[i].y);
  }
}

// ------------------------------------------------------------------------- geometry
struct Site {
  int c[4];
};
__device__ __forceinline__ Site site_of(int n, const Geom& g) {
  Site s;
  s.c[0] = n % g.L[0]; n /= g.L[0];
  s.c[1] = n % g.L[1]; n /= g.L[1];
  s.c[2] = n % g.L[2];
  s.c[3] = n / g.L[2];
  return s;
}
__device__ __forceinline__ int index_of(const Site& s, const Geom& g) {
  return s.c[0] + g.L[0] * (s.c[1] + g.L[1] * (s.c[2] + g.L[2] * s.c[3]));
}
__device__ __forceinline__ Site shift(Site s, int mu, int d, const Geom& g) {   // |d| <= L
  int v = s.c[mu] + d;
  v += (v < 0) ? g.L[mu] : 0;
  v -= (v >= g.L[mu]) ? g.L[mu] : 0;
  s.c[mu] = v;
  return s;
}

// U_mu(x) with the boundary-condition sign folded in.
// `links` inside the kernels is the TRANSPOSED copy made by transpose_links_kernel: element e of U_mu(n) at
// [(9 mu + e) Vpad + n], so that with lane <-> site a warp-wide load is one contiguous 512-byte line (the canonical
// [n][mu][3][3] layout has 576 bytes between lanes: ncu showed the field-strength and hop kernels L1-throughput bound on it).
__device__ __forceinline__ cm3 ldU(const double2* __restrict__ links, const Site& s, int mu, const PrecalcArgs& a) {
  const double2* p = links + (size_t)(9 * mu) * a.Vpad + index_of(s, a.g);
  const double sg = (a.bc[mu] < 0 && s.c[mu] == (mu == 3 ? a.tfold : a.g.L[mu] - 1)) ? -1.0 : 1.0;
  cm3 r;
#pragma unroll
  for (int i = 0; i < 9; ++i) {
    double2 v = __ldg(p + (size_t)i * a.Vpad);
    r.e[i] = make_double2(sg * v.x, sg * v.y);
  }
  return r;
}
// Scratch colour-matrix fields (clover fields, hop blocks) are kept the same way: matrix k, element e of site n at
// [(9 k + e) Vpad + n] double2 (a `cm3*` advanced by k Vpad still points at matrix k).
__device__ __forceinline__ cm3 ldF(const cm3* __restrict__ FS, int k, const Site& s, const PrecalcArgs& a) {
  const double2* p = reinterpret_cast<const double2*>(FS) + (size_t)(9 * k) * a.Vpad + index_of(s, a.g);
  cm3 r;
#pragma unroll
  for (int i = 0; i < 9; ++i) r.e[i] = __ldg(p + (size_t)i * a.Vpad);
  return r;
}
__device__ __forceinline__ void stF(cm3* __restrict__ FS, int k, int n, const cm3& F, const PrecalcArgs& a) {
  double2* p = reinterpret_cast<double2*>(FS) + (size_t)(9 * k) * a.Vpad + n;
#pragma unroll
  for (int i = 0; i < 9; ++i) p[(size_t)i * a.Vpad] = F.e[i];
}
__global__ void __launch_bounds__(256) transpose_links_kernel(const double2* __restrict__ canon, double2* __restrict__ T, PrecalcArgs a) {
  const long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // one 16-byte element; the transposed side is coalesced
  if (u >= (long long)36 * a.g.V) return;
  const int n = (int)(u % a.g.V), q = (int)(u / a.g.V);
  T[(size_t)q * a.Vpad + n] = __ldg(canon + (size_t)n * 36 + q);
}

// ------------------------------------------------------------------------- step a1: clover F
// FS[k][n]: k = 0..2 -> B_1,B_2,B_3 = F_23, F_31, F_12 ; k = 3..5 -> E_i = F_4i   (anti-Hermitian,
// F = (Q - Q^dag)/8, Q = sum of the four leaves starting and ending at x, no trace subtraction).
__global__ void __launch_bounds__(128, 3) field_strength_kernel(const double2* __restrict__ links, cm3* __restrict__ FS, PrecalcArgs a) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y;
  if (n >= a.g.V) return;
  int mu, nu;
  if (k < 3) { mu = (k + 1) % 3; nu = (k + 2) % 3; } else { mu = 3; nu = k - 3; }
  const Site x = site_of(n, a.g);
  const Site xpm = shift(x, mu, 1, a.g), xpn = shift(x, nu, 1, a.g);
  const Site xmm = shift(x, mu, -1, a.g), xmn = shift(x, nu, -1, a.g);
  const Site xmmpn = shift(xmm, nu, 1, a.g), xmmmn = shift(xmm, nu, -1, a.g), xpmmn = shift(xpm, nu, -1, a.g);
  cm3 Q, T;
  // U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
  T = mul(ldU(links, x, mu, a), ldU(links, xpm, nu, a));
  T = mul_nd(T, ldU(links, xpn, mu, a));
  Q = mul_nd(T, ldU(links, x, nu, a));
  // U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
  T = mul_nd(ldU(links, x, nu, a), ldU(links, xmmpn, mu, a));
  T = mul_nd(T, ldU(links, xmm, nu, a));
  T = mul(T, ldU(links, xmm, mu, a));
  axpy(Q, 1.0, 0.0, T);
  // U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
  T = mul_dn(ldU(links, xmm, mu, a), adj(ldU(links, xmmmn, nu, a)));
  T = mul(T, ldU(links, xmmmn, mu, a));
  T = mul(T, ldU(links, xmn, nu, a));
  axpy(Q, 1.0, 0.0, T);
  // U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
  T = mul_dn(ldU(links, xmn, nu, a), ldU(links, xmn, mu, a));
  T = mul(T, ldU(links, xpmmn, nu, a));
  T = mul_nd(T, ldU(links, x, mu, a));
  axpy(Q, 1.0, 0.0, T);
  cm3 F;
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      F.e[3 * i + j].x = (Q.e[3 * i + j].x - Q.e[3 * j + i].x) * 0.125;
      F.e[3 * i + j].y = (Q.e[3 * i + j].y + Q.e[3 * j + i].y) * 0.125;
    }
  stF(FS, k, n, F, a);
}

// ------------------------------------------------------------------------- step a1b: colour matrices of the one-link hops
// The Pauli components of W^+_i that need link-times-field products or staples (Eq. 2.8, see the header comment), computed
// once per (site, direction) by three threads -- one per B component entering the products -- instead of inside the thread
// that later writes the 2 x 144 entries of W^+_i(x) and W^-_i(x + i).  HB[(5 i + q)][n], cyclic (i, k, l):
//   q = 0: S.C_0 =  i cs (U B_i(x+i) + B_i(x) U)
//   q = 1: S.C_k =    cs (U B_l(x+i) - B_l(x) U)            q = 3: D.C_k = i c5/u0^4 (U B_k(x+i) + B_k(x) U) + i cg G_l
//   q = 2: S.C_l =   -cs (U B_k(x+i) - B_k(x) U)            q = 4: D.C_l = i c5/u0^4 (U B_l(x+i) + B_l(x) U) - i cg G_k
// role 0 writes q = 0; role 1 (products with B_k, staples along l) q = 2, 3; role 2 (B_l, staples along k) q = 1, 4.
constexpr int kHopMats = 18;   // 15 of the spatial hops + T_m = (cEE/2u0^4) (U_4 E_m(x+t) - E_m(x) U_4), m = 0..2 (Eq. 2.7)
__global__ void __launch_bounds__(128) hop_blocks_kernel(const double2* __restrict__ links, const cm3* __restrict__ FS, cm3* __restrict__ HB,
                                                         PrecalcArgs a) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= a.g.V) return;
  if (blockIdx.y >= 9) {   // the temporal hop: S^+_4 components
    const int m = blockIdx.y - 9;
    const Site x = site_of(n, a.g);
    const cm3 U = ldU(links, x, 3, a);
    cm3 T = zero3();
    axpy(T, a.s4, 0.0, mul(U, ldF(FS, 3 + m, shift(x, 3, 1, a.g), a)));
    axpy(T, -a.s4, 0.0, mul(ldF(FS, 3 + m, x, a), U));
    stF(HB, 15 + m, n, T, a);
    return;
  }
  const int i = blockIdx.y / 3, role = blockIdx.y % 3;
  const int k = (i + 1) % 3, l = (i + 2) % 3;
  const int m = role == 0 ? i : (role == 1 ? k : l);       // the B component of this thread's products
  const Site x = site_of(n, a.g);
  const Site xp = shift(x, i, 1, a.g);
  const cm3 U = ldU(links, x, i, a);
  const cm3 P = mul(U, ldF(FS, m, xp, a)), Q = mul(ldF(FS, m, x, a), U);
  if (role == 0) {
    cm3 R = zero3();
    axpy(R, 0.0, a.cs, P);
    axpy(R, 0.0, a.cs, Q);
    stF(HB, 5 * i, n, R, a);
    return;
  }
  cm3 Sd = zero3(), Dd = zero3();
  const double sg = role == 1 ? -1.0 : 1.0;                 // role 1: S.C_l = -cs Dif_k ; role 2: S.C_k = +cs Dif_l
  axpy(Sd, sg * a.cs, 0.0, P);
  axpy(Sd, -sg * a.cs, 0.0, Q);
  axpy(Dd, 0.0, a.c5u, P);
  axpy(Dd, 0.0, a.c5u, Q);
  if (a.cg != 0.0) {
    const int sd = role == 1 ? l : k;                       // staple direction; role 1: + i cg G_l, role 2: - i cg G_k
    const double gs = role == 1 ? 1.0 : -1.0;
    cm3 G = mul(ldU(links, x, sd, a), ldU(links, shift(x, sd, 1, a.g), i, a));   // up: U_m(x) U_i(x+m) U_m(x+i)^dag
    G = mul_nd(G, ldU(links, xp, sd, a));
    axpy(Dd, 0.0, gs * a.cg, G);
    const Site xm = shift(x, sd, -1, a.g);                                        // down: U_m(x-m)^dag U_i(x-m) U_m(x-m+i)
    G = mul_dn(ldU(links, xm, sd, a), ldU(links, xm, i, a));
    G = mul(G, ldU(links, shift(xm, i, 1, a.g), sd, a));
    axpy(Dd, 0.0, -gs * a.cg, G);
  }
  stF(HB, 5 * i + (role == 1 ? 2 : 1), n, Sd, a);
  stF(HB, 5 * i + (role == 1 ? 3 : 4), n, Dd, a);
}

// ------------------------------------------------------------------------- step a2: W assembly
struct P4 {
  cm3 c[4];
};

// Positive blocks of the term family at site x.  A = diagonal block, B = off-diagonal block.
//   fam 0: W^0 (Eq. 2.6)   fam 1: W^+_4 (2.7)   fam 2: W^+_i (2.8)   fam 3: W^++_ii (2.9)
//   fam 4: W^++_ij (2.11)  fam 5: W^+-_ij (2.12)
template <int fam, int i, int j>
__device__ __forceinline__ void positive_blocks(const Site& x, const double2* __restrict__ links,
                                                const cm3* __restrict__ FS, const PrecalcArgs& a, P4& A, P4& B) {
#pragma unroll
  for (int k = 0; k < 4; ++k) { A.c[k] = zero3(); B.c[k] = zero3(); }
  if constexpr (fam == 0) {
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      axpy(A.c[m + 1], 0.0, a.d0, ldF(FS, m, x, a));       // D^0 = d0 * i sum sigma_m B_m
      axpy(B.c[m + 1], a.s0, 0.0, ldF(FS, 3 + m, x, a));   // S^0 = s0 * sum sigma_m E_m
    }
  } else if constexpr (fam == 1) {
    const cm3 U = ldU(links, x, 3, a);
    const Site xp = shift(x, 3, 1, a.g);
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      axpy(B.c[m + 1], a.s4, 0.0, mul(U, ldF(FS, 3 + m, xp, a)));
      axpy(B.c[m + 1], -a.s4, 0.0, mul(ldF(FS, 3 + m, x, a), U));
    }
    axpy(A.c[0], -1.0, 0.0, U);
  } else if constexpr (fam == 2) {
    constexpr int k = (i + 1) % 3, l = (i + 2) % 3;
    const cm3 U = ldU(links, x, i, a);
    const cm3* HB = FS + (size_t)(6 + 5 * i) * a.Vpad;      // hop_blocks_kernel (the scratch follows the six clover fields)
    axpy(B.c[i + 1], a.a1, 0.0, U);
    axpy(A.c[0], a.d1, 0.0, U);
    B.c[0] = ldF(HB, 0, x, a);
    B.c[k + 1] = ldF(HB, 1, x, a);
    B.c[l + 1] = ldF(HB, 2, x, a);
    A.c[k + 1] = ldF(HB, 3, x, a);
    A.c[l + 1] = ldF(HB, 4, x, a);
  } else if constexpr (fam == 3) {
    const cm3 P = mul(ldU(links, x, i, a), ldU(links, shift(x, i, 1, a.g), i, a));
    axpy(A.c[0], a.dii, 0.0, P);
    axpy(B.c[i + 1], a.sii, 0.0, P);
  } else if constexpr (fam == 4) {
    cm3 P = mul(ldU(links, x, i, a), ldU(links, shift(x, i, 1, a.g), j, a));
    axpy(P, 1.0, 0.0, mul(ldU(links, x, j, a), ldU(links, shift(x, j, 1, a.g), i, a)));
    axpy(B.c[i + 1], a.sij, 0.0, P);
    axpy(B.c[j + 1], a.sij, 0.0, P);
  } else {
    const Site xmj = shift(x, j, -1, a.g);
    cm3 P = mul_nd(ldU(links, x, i, a), ldU(links, shift(xmj, i, 1, a.g), j, a));
    axpy(P, 1.0, 0.0, mul_dn(ldU(links, xmj, j, a), ldU(links, xmj, i, a)));
    axpy(B.c[i + 1], a.sij, 0.0, P);
    axpy(B.c[j + 1], -a.sij, 0.0, P);
  }
}

// entry (alpha', a ; beta', b) of sum_k sigma_k (x) C_k
__device__ __forceinline__ double2 pauli_entry(const P4& P, int al, int be, int ab) {
  const double2 c0 = P.c[0].e[ab], c1 = P.c[1].e[ab], c2 = P.c[2].e[ab], c3 = P.c[3].e[ab];
  if (al == be) return al == 0 ? make_double2(c0.x + c3.x, c0.y + c3.y) : make_double2(c0.x - c3.x, c0.y - c3.y);
  // (0,1): c1 - i c2 ; (1,0): c1 + i c2
  return al == 0 ? make_double2(c1.x + c2.y, c1.y - c2.x) : make_double2(c1.x - c2.y, c1.y + c2.x);
}

template <typename real> struct WUnit;
template <> struct WUnit<float> { using type = float4; using cx = float2; static constexpr int NC = 6; };
template <> struct WUnit<double> { using type = double2; using cx = double2; static constexpr int NC = 12; };

// One (site, term) with the family and directions as template arguments: Pauli components that vanish for the family are
// never materialised, so the per-term register footprint stays far below the 8 colour matrices of the generic form.
template <typename real, int fam, int i, int j>
__device__ __noinline__ void assemble_term(const double2* __restrict__ links, const cm3* __restrict__ FS,
                                              typename WUnit<real>::type* __restrict__ W, typename WUnit<real>::type* __restrict__ Wt,
                                              const PrecalcArgs& a, int term, bool neg, int n, int blk, int lane) {
  using unit_t = typename WUnit<real>::type;
  constexpr int NC = WUnit<real>::NC;
  Site x = site_of(n, a.g);
  if (neg) {   // positive blocks at x - offset(term_positive) = x + offset(term)
    for (int mu = 0; mu < 4; ++mu) x = shift(x, mu, c_poff[term][mu], a.g);
  }
  P4 A, B;
  positive_blocks<fam, i, j>(x, links, FS, a, A, B);
  auto conjugate = [&]() {   // Eqs. (2.3), (2.10): A -> A^dag, B -> -B^dag
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      A.c[k] = adj(A.c[k]);
      cm3 t = adj(B.c[k]);
#pragma unroll
      for (int q = 0; q < 9; ++q) B.c[k].e[q] = make_double2(-t.e[q].x, -t.e[q].y);
    }
  };
  if (neg) conjugate();
  // writes W_term (built from the current A, B) of the site that sits at (blk, lane) of the output buffer
  auto emit = [&](int term, bool neg, unit_t* Wt, int blk, int lane) {
  // block pattern: UL, LR use A (or 0); UR uses B; LL uses +-B
  const bool ulA = !(fam == 4 || fam == 5) && !(fam == 1 && !neg);
  const bool lrA = !(fam == 4 || fam == 5) && !(fam == 1 && neg);
  const double llsgn = (fam == 0) ? -1.0 : 1.0;
  const double mass = (fam == 0) ? a.mass : 0.0;

#pragma unroll
  for (int r = 0; r < 12; ++r) {
    const int alpha = r / 3, ca = r % 3, bi = alpha >> 1, al = alpha & 1;
    double2 row[12];
#pragma unroll
    for (int col = 0; col < 12; ++col) {
      const int beta = col / 3, cb = col % 3, bj = beta >> 1, be = beta & 1;
      double2 v = make_double2(0.0, 0.0);
      if (bi == bj) {
        if (bi == 0 ? ulA : lrA) v = pauli_entry(A, al, be, 3 * ca + cb);
        if (r == col) v.x += mass;
      } else {
        v = pauli_entry(B, al, be, 3 * ca + cb);
        if (bi == 1) { v.x *= llsgn; v.y *= llsgn; }
      }
      row[col] = v;
    }
    if (a.storage != OK_W_DENSE) {   // reduced formats: keep only what the format stores (rounded once, like the dense W)
      using cx = typename WUnit<real>::cx;
      cx* Ws = reinterpret_cast<cx*>(W) + (size_t)blk * sparse_site_units_rt(a.storage) * kBlock + lane;
      const TermDesc d = term_desc(term);
      const int hr = r / 6, sa = (r % 6) / 3, cr = r % 3;
#pragma unroll
      for (int hc = 0; hc < 2; ++hc) {
        const int quad = 2 * hr + hc;
        const bool diag = hr == hc;
        if (diag && !(quad == 0 ? d.ul : d.lr)) continue;
        int m = quad;
        if (a.storage != OK_W_BLOCK) {
          if (!(diag ? (quad == 0 || !d.ul) : quad == 1)) continue;   // LR = D and LL = +-S are implied
          m = diag ? 0 : 1;
        }
        const int mr = mask_row(diag ? d.maskD : d.maskS, sa), nb = popc2(mr);
        cx* run = Ws + (size_t)(c_qrun[a.storage - 1][term][sa][m] + cr * nb * 3) * kBlock;
#pragma unroll
        for (int b = 0; b < 2; ++b) {
          if (!((mr >> b) & 1)) continue;
          const int bc = (b == 1 && (mr & 1)) ? 1 : 0;
#pragma unroll
          for (int cc = 0; cc < 3; ++cc) {
            cx v;
            v.x = (real)row[6 * hc + 3 * b + cc].x;
            v.y = (real)row[6 * hc + 3 * b + cc].y;
            run[(size_t)(bc * 3 + cc) * kBlock] = v;
          }
        }
      }
      continue;
    }
    unit_t* dst = Wt + (size_t)r * NC * kBlock;
    if constexpr (sizeof(real) == 4) {
#pragma unroll
      for (int c = 0; c < 6; ++c)
        dst[(size_t)c * kBlock] = make_float4((float)row[2 * c].x, (float)row[2 * c].y, (float)row[2 * c + 1].x, (float)row[2 * c + 1].y);
    } else {
#pragma unroll
      for (int c = 0; c < 12; ++c) dst[(size_t)c * kBlock] = row[c];
    }
  }
  };   // emit
  emit(term, neg, Wt, blk, lane);
  if (a.pair && fam != 0 && !neg) {
    // the opposite-direction matrix of the site x + offset(term) is the conjugate of this one: W^-_o(y) from W^+_o(y - o)
    Site y = x;
    for (int mu = 0; mu < 4; ++mu) y = shift(y, mu, c_poff[term][mu], a.g);
    const int n2 = index_of(y, a.g), blk2 = n2 >> 5, lane2 = n2 & 31;
    conjugate();
    emit(term + 1, true, W + ((size_t)blk2 * kTerms + term + 1) * 12 * NC * kBlock + lane2, blk2, lane2);
  }
}


// CLS splits the 27 terms into four launches so that every launch carries only the registers its families need:
//   0: W^0, W^+-_4 (terms 0, 7, 8)   1: W^+-_i (1..6, the heavy one)   2: W^{++/--}_ii (9..14)   3: the 12 pair terms (15..26)
template <typename real, int CLS>
#ifndef OK_CLS1_MINB
#define OK_CLS1_MINB 4
#endif
__global__ void __launch_bounds__(32 * 3, CLS == 1 ? OK_CLS1_MINB : 4) assemble_W_kernel(const double2* __restrict__ links, const cm3* __restrict__ FS,
                                                                           typename WUnit<real>::type* __restrict__ W, PrecalcArgs a) {
  using unit_t = typename WUnit<real>::type;
  constexpr int NC = WUnit<real>::NC;
  const int lane = threadIdx.x;
  const int idx = blockIdx.y * 3 + threadIdx.y;
  // a.posonly: the grid covers W^0 and the positive-direction terms only (their threads write or imply the opposite ones)
  int term;
  if (a.posonly) {
    term = CLS == 0 ? (idx == 0 ? 0 : 7) : CLS == 1 ? 1 + 2 * idx : CLS == 2 ? 9 + 2 * idx : 15 + 2 * idx;
    if (CLS == 0 && idx > 1) return;
  } else {
    term = CLS == 0 ? (idx == 0 ? 0 : 6 + idx) : CLS == 1 ? 1 + idx : CLS == 2 ? 9 + idx : 15 + idx;
  }
  const int blk = blockIdx.x;                        // block inside the output buffer
  const int n = (blk + a.blk0) * kBlock + lane;      // lattice site
  unit_t* Wt = W + ((size_t)blk * kTerms + term) * 12 * NC * kBlock + lane;
  if (a.storage == OK_W_CONJ && term_is_neg(term)) return;   // rebuilt at apply time from term - 1 of the neighbour site
  if (a.pair && term_is_neg(term)) return;                   // written by the thread of term - 1 of the neighbour site
  const int nzero = (a.pair && term > 0) ? 2 : 1;            // padded site: this term (and its partner) are zero
  if (n >= a.g.V && a.storage != OK_W_DENSE) {   // padded site, reduced format: zero the units the terms keep
    using cx = typename WUnit<real>::cx;
    cx* Ws = reinterpret_cast<cx*>(W) + (size_t)blk * sparse_site_units_rt(a.storage) * kBlock + lane;
    for (int tz = term; tz < term + nzero; ++tz)
      for (int r = 0; r < 12; ++r)
        for (int col = 0; col < 12; ++col) {
          const SparseRef ref = sparse_ref(a.storage, tz, r, col, c_qrun[a.storage - 1]);
          if (ref.unit >= 0 && ref.stored) Ws[(size_t)ref.unit * kBlock] = cx{};
        }
    return;
  }
  if (n >= a.g.V) {   // padded site: zeros
    unit_t z = {};
    for (int u = 0; u < 12 * NC * nzero; ++u) Wt[(size_t)u * kBlock] = z;
    return;
  }
  // term -> family, directions, sign of the hop (term order of ok.h)
#define OK_ASM(F, I_, J_, NEG) assemble_term<real, F, I_, J_>(links, FS, W, Wt, a, term, NEG, n, blk, lane)
  if constexpr (CLS == 0) {
    if (term == 0) OK_ASM(0, 0, 0, false); else OK_ASM(1, 0, 0, term == 8);
  } else if constexpr (CLS == 1) {
    const bool ng = (term & 1) == 0;
    if (term <= 2) OK_ASM(2, 0, 0, ng); else if (term <= 4) OK_ASM(2, 1, 0, ng); else OK_ASM(2, 2, 0, ng);
  } else if constexpr (CLS == 2) {
    const bool ng = (term & 1) == 0;
    if (term <= 10) OK_ASM(3, 0, 0, ng); else if (term <= 12) OK_ASM(3, 1, 0, ng); else OK_ASM(3, 2, 0, ng);
  } else {
    {
      const int q = (term - 15) >> 2, w = (term - 15) & 3;   // pair (x,y), (x,z), (y,z) ; (++, --, +-, -+)
      const bool ng = (w & 1) != 0;
      if (w < 2) {
        if (q == 0) OK_ASM(4, 0, 1, ng); else if (q == 1) OK_ASM(4, 0, 2, ng); else OK_ASM(4, 1, 2, ng);
      } else {
        if (q == 0) OK_ASM(5, 0, 1, ng); else if (q == 1) OK_ASM(5, 0, 2, ng); else OK_ASM(5, 1, 2, ng);
      }
    }
  }
#undef OK_ASM
}

// ------------------------------------------------------------------------- step a2, W^0, W^+-_i, W^+-_4 (dense layout)
// Terms 0..8: every 6x6 block is a Pauli sum  sum_k sigma_k (x) C_k  whose colour matrices C_k are, up to a constant, one of the
// scratch fields (clover fields, hop blocks) or a link.  One thread per (site, term); a rolled loop over the colour row reads
// row ca of each C_k (for the opposite-direction terms: column ca of the matrices at x + offset, conjugated, Eqs. 2.3 / 2.10)
// straight from the transposed scratch -- 3 contiguous-line loads per matrix -- and writes the four spin rows (alpha, ca) of
// W.  No matrix is held in registers across rows (the templated path spilled 2.5-3 KB per thread on the seven matrices of a
// one-link hop), every thread writes its own site only.  fp64 throughout, rounded once.
// what a thread of W^0, W^+-_i or W^+-_4 needs besides the colour row: family, directions, signs, and where its colour matrices live
struct PauliTerm {
  int fam, i, k, l;           // fam 0: W^0, 1: W^+-_4, 2: W^+-_i ; hop direction i, cyclic (i, k, l)
  bool neg, ulA, lrA;
  double usg, llsgn, mass;
  const double2* F;           // scratch fields at the site of the positive blocks: matrix m, element e at F[(9 m + e) Vpad]
  const double2* Ul;          // the hop's link there
};
__device__ __forceinline__ PauliTerm pauli_term_of(int term, int n, const double2* __restrict__ links, const cm3* __restrict__ FS,
                                                   const PrecalcArgs& a) {
  PauliTerm c;
  c.fam = term == 0 ? 0 : (term >= 7 ? 1 : 2);
  c.i = c.fam == 2 ? (term - 1) >> 1 : 3;           // hop direction
  c.neg = c.fam == 0 ? false : (c.fam == 1 ? term == 8 : ((term - 1) & 1) != 0);
  Site x = site_of(n, a.g);
  if (c.neg)
    for (int mu = 0; mu < 4; ++mu) x = shift(x, mu, c_poff[term][mu], a.g);
  const int ns = index_of(x, a.g);
  c.F = reinterpret_cast<const double2*>(FS) + ns;
  c.usg = (c.fam != 0 && a.bc[c.i] < 0 && x.c[c.i] == (c.i == 3 ? a.tfold : a.g.L[c.i] - 1)) ? -1.0 : 1.0;
  c.Ul = links + (size_t)(9 * (c.fam == 0 ? 0 : c.i)) * a.Vpad + ns;
  c.k = c.fam == 2 ? (c.i + 1) % 3 : 1;
  c.l = c.fam == 2 ? (c.i + 2) % 3 : 2;
  c.ulA = c.fam == 1 ? c.neg : true;
  c.lrA = c.fam == 1 ? !c.neg : true;
  c.llsgn = c.fam == 0 ? -1.0 : 1.0;
  c.mass = c.fam == 0 ? a.mass : 0.0;
  return c;
}
// Colour row ca of the term as the 24 complex numbers its four spin rows (alpha, ca) are made of: with the Pauli components
// C_0..C_3 of a 6x6 block (header comment), combo 0: C0 + C3 (al = be = 0), 1: C0 - C3 (al = be = 1), 2: C1 - i C2 (al, be = 0, 1),
// 3: C1 + i C2 (1, 0); Dv[combo][cb] for the diagonal blocks (the mass term of W^0 included), Sv[combo][cb] for the off-diagonal ones.
__device__ __forceinline__ void pauli_term_tables(const PauliTerm& t, int ca, const PrecalcArgs& a, double2 (&Dv)[4][3], double2 (&Sv)[4][3]) {
  const int fam = t.fam, i = t.i, k = t.k;
  const bool neg = t.neg;
  const double usg = t.usg;
  const double2* F = t.F;
  const double2* Ul = t.Ul;
  auto at = [&](const double2* base, int kmat, int e) { return __ldg(base + (size_t)(9 * kmat + e) * a.Vpad); };
#pragma unroll
  for (int cb = 0; cb < 3; ++cb) {
    const int e = neg ? 3 * cb + ca : 3 * ca + cb;       // the adjoint reads the transposed element
    const double2 z = make_double2(0.0, 0.0);
    double2 a0 = z, a1 = z, a2 = z, a3 = z, b0 = z, b1 = z, b2 = z, b3 = z;
    if (fam == 0) {          // D^0 = i d0 sum sigma_m B_m ; S^0 = s0 sum sigma_m E_m     (Eq. 2.6)
      const double2 f0 = at(F, 0, e), f1 = at(F, 1, e), f2 = at(F, 2, e);
      a1 = make_double2(-a.d0 * f0.y, a.d0 * f0.x); a2 = make_double2(-a.d0 * f1.y, a.d0 * f1.x); a3 = make_double2(-a.d0 * f2.y, a.d0 * f2.x);
      const double2 g0 = at(F, 3, e), g1 = at(F, 4, e), g2 = at(F, 5, e);
      b1 = make_double2(a.s0 * g0.x, a.s0 * g0.y); b2 = make_double2(a.s0 * g1.x, a.s0 * g1.y); b3 = make_double2(a.s0 * g2.x, a.s0 * g2.y);
    } else if (fam == 1) {   // D^+_4 = -U_4 ; S^+_4 = sum sigma_m T_m                        (Eq. 2.7)
      const double2 u = __ldg(Ul + (size_t)e * a.Vpad);
      a0 = make_double2(-usg * u.x, -usg * u.y);
      b1 = at(F, 6 + 15, e); b2 = at(F, 6 + 16, e); b3 = at(F, 6 + 17, e);
    } else {                 // Eq. (2.8): hop_blocks_kernel's q = 0..4 of direction i, and U_i itself
      const double2 u = __ldg(Ul + (size_t)e * a.Vpad);
      const int hb = 6 + 5 * i;
      const double2 vi_b = make_double2(a.a1 * usg * u.x, a.a1 * usg * u.y);                     // S.C_i = a1 U
      const double2 vk_b = at(F, hb + 1, e), vl_b = at(F, hb + 2, e), vk_a = at(F, hb + 3, e), vl_a = at(F, hb + 4, e);
      a0 = make_double2(a.d1 * usg * u.x, a.d1 * usg * u.y);                                     // D.C_0 = d1 U
      b0 = at(F, hb, e);
      // direction d carries the i-, k- or l-component
      a1 = i == 0 ? z : (k == 0 ? vk_a : vl_a); b1 = i == 0 ? vi_b : (k == 0 ? vk_b : vl_b);
      a2 = i == 1 ? z : (k == 1 ? vk_a : vl_a); b2 = i == 1 ? vi_b : (k == 1 ? vk_b : vl_b);
      a3 = i == 2 ? z : (k == 2 ? vk_a : vl_a); b3 = i == 2 ? vi_b : (k == 2 ? vk_b : vl_b);
    }
    if (neg) {               // A -> A^dag, B -> -B^dag (the element was read transposed)
      a0.y = -a0.y; a1.y = -a1.y; a2.y = -a2.y; a3.y = -a3.y;
      b0.x = -b0.x; b1.x = -b1.x; b2.x = -b2.x; b3.x = -b3.x;
    }
    const double m = ca == cb ? t.mass : 0.0;
    Dv[0][cb] = make_double2(a0.x + a3.x + m, a0.y + a3.y);
    Dv[1][cb] = make_double2(a0.x - a3.x + m, a0.y - a3.y);
    Dv[2][cb] = make_double2(a1.x + a2.y, a1.y - a2.x);
    Dv[3][cb] = make_double2(a1.x - a2.y, a1.y + a2.x);
    Sv[0][cb] = make_double2(b0.x + b3.x, b0.y + b3.y);
    Sv[1][cb] = make_double2(b0.x - b3.x, b0.y - b3.y);
    Sv[2][cb] = make_double2(b1.x + b2.y, b1.y - b2.x);
    Sv[3][cb] = make_double2(b1.x - b2.y, b1.y + b2.x);
  }
}
// the four spin rows (alpha, ca), alpha = 0..3: emit(alpha, row[12]) with row[3 beta + cb]
template <class Emit>
__device__ __forceinline__ void pauli_term_rows(const PauliTerm& t, int ca, const PrecalcArgs& a, Emit&& emit) {
  double2 Dv[4][3], Sv[4][3];
  pauli_term_tables(t, ca, a, Dv, Sv);
#pragma unroll
  for (int alpha = 0; alpha < 4; ++alpha) {
    const int bi = alpha >> 1, al = alpha & 1;
    double2 row[12];
#pragma unroll
    for (int beta = 0; beta < 4; ++beta) {
      const int bj = beta >> 1, be = beta & 1;
      const int combo = al == be ? al : (al == 0 ? 2 : 3);
#pragma unroll
      for (int cb = 0; cb < 3; ++cb) {
        double2 v;
        if (bi == bj) {
          v = (bi == 0 ? t.ulA : t.lrA) ? Dv[combo][cb] : make_double2(0.0, 0.0);
        } else {
          v = Sv[combo][cb];
          if (bi == 1) { v.x *= t.llsgn; v.y *= t.llsgn; }
        }
        row[3 * beta + cb] = v;
      }
    }
    emit(alpha, row);
  }
}

// one row of 12 complex numbers -> the dense layout (rounded once to the storage precision)
template <typename real>
__device__ __forceinline__ void store_dense_row(typename WUnit<real>::type* __restrict__ dst, const double2 (&row)[12]) {
  if constexpr (sizeof(real) == 4) {
#pragma unroll
    for (int c = 0; c < 6; ++c)
      dst[(size_t)c * kBlock] = make_float4((float)row[2 * c].x, (float)row[2 * c].y, (float)row[2 * c + 1].x, (float)row[2 * c + 1].y);
  } else {
#pragma unroll
    for (int c = 0; c < 12; ++c) dst[(size_t)c * kBlock] = row[c];
  }
}

template <typename real>
__global__ void __launch_bounds__(32 * 3) pauli_terms_kernel(const double2* __restrict__ links, const cm3* __restrict__ FS,
                                                             typename WUnit<real>::type* __restrict__ W, PrecalcArgs a) {
  using unit_t = typename WUnit<real>::type;
  constexpr int NC = WUnit<real>::NC;
  const int lane = threadIdx.x;
  const int term = blockIdx.y * 3 + threadIdx.y;          // 0..8
  const int blk = blockIdx.x;
  const int n = (blk + a.blk0) * kBlock + lane;
  unit_t* Wt = W + ((size_t)blk * kTerms + term) * 12 * NC * kBlock + lane;
  if (n >= a.g.V) {
    unit_t z = {};
    for (int u = 0; u < 12 * NC; ++u) Wt[(size_t)u * kBlock] = z;
    return;
  }
  const PauliTerm t = pauli_term_of(term, n, links, FS, a);
#pragma unroll 1
  for (int ca = 0; ca < 3; ++ca)
    pauli_term_rows(t, ca, a, [&](int alpha, const double2 (&row)[12]) { store_dense_row<real>(Wt + (size_t)(3 * alpha + ca) * NC * kBlock, row); });
}

// ------------------------------------------------------------------------- step a2, the 18 two-link terms (dense layout)
// W^{++}_ii, W^{++}_ij, W^{+-}_ij and their conjugates (Eqs. 2.9-2.12; terms 9..26, two thirds of W's bytes) are Kronecker
// products  W = K (x) P  of a 4x4 spin matrix K and ONE 3x3 colour matrix:
//   P_ii = U_i(x) U_i(x+i)                                    D = (c4/u0) 1 (x) P ,       S = ((c1+2c2)/2u0) sigma_i (x) P      (2.9)
//   P_ij = U_i(x) U_j(x+i) + U_j(x) U_i(x+j)                  D = 0 ,                     S = (c2/2u0) (sigma_i + sigma_j) (x) P  (2.11)
//   P_i-j = U_i(x) U_j(x-j+i)^dag + U_j(x-j)^dag U_i(x-j)     D = 0 ,                     S = (c2/2u0) (sigma_i - sigma_j) (x) P  (2.12)
// W = [[D, S], [S, D]]; the opposite-direction matrix is [[D^dag, -S^dag], [-S^dag, D^dag]] of the blocks at x + offset (2.3, 2.10):
// same K with the sign of S flipped, P -> P^dag.  One thread per (site, term) writes its own site only (coalesced, sector
// aligned), one rolled loop over the spin row keeps the code small: the templated assembly path spends most of its time waiting
// for instructions (profiles/r02_precalc.md).  fp64 throughout, rounded once.
// the colour matrix of a two-link term at site x: fam 3 P_ii, fam 4 P_ij, fam 5 P_i-j (see above)
__device__ __forceinline__ cm3 two_link_P(const double2* __restrict__ links, const Site& x, int fam, int i, int j, const PrecalcArgs& a) {
  cm3 P;
  if (fam == 3) {
    P = mul(ldU(links, x, i, a), ldU(links, shift(x, i, 1, a.g), i, a));
  } else if (fam == 4) {
    P = mul(ldU(links, x, i, a), ldU(links, shift(x, i, 1, a.g), j, a));
    axpy(P, 1.0, 0.0, mul(ldU(links, x, j, a), ldU(links, shift(x, j, 1, a.g), i, a)));
  } else {
    const Site xmj = shift(x, j, -1, a.g);
    P = mul_nd(ldU(links, x, i, a), ldU(links, shift(xmj, i, 1, a.g), j, a));
    axpy(P, 1.0, 0.0, mul_dn(ldU(links, xmj, j, a), ldU(links, xmj, i, a)));
  }
  return P;
}

// OK_W_PAULI (ok_pauli.cu has the list of the 37 stored matrices): thread = (site, matrix); everything but the two-link
// products is a scaled copy of a scratch field or a link
template <typename real>
__global__ void __launch_bounds__(32 * 4) pauli_store_kernel(const double2* __restrict__ links, const cm3* __restrict__ FS,
                                                             typename WUnit<real>::cx* __restrict__ W, PrecalcArgs a) {
  using cx = typename WUnit<real>::cx;
  const int lane = threadIdx.x, m = blockIdx.y * 4 + threadIdx.y;
  if (m >= OK_W_PAULI_MATS) return;
  const int blk = blockIdx.x, n = (blk + a.blk0) * kBlock + lane;
  cx* dst = W + ((size_t)blk * OK_W_PAULI_MATS + m) * (9 * kBlock);   // + pauli_elem_index(e, lane)
  cm3 C = zero3();
  if (n < a.g.V) {
    const Site x = site_of(n, a.g);
    if (m < 3) axpy(C, 0.0, a.d0, ldF(FS, m, x, a));
    else if (m < 6) axpy(C, a.s0, 0.0, ldF(FS, m, x, a));
    else if (m == 6) C = ldU(links, x, 3, a);
    else if (m < 10) C = ldF(FS, 6 + 15 + (m - 7), x, a);
    else if (m < 28) {
      const int i = (m - 10) / 6, r = (m - 10) % 6;
      C = r == 0 ? ldU(links, x, i, a) : ldF(FS, 6 + 5 * i + (r - 1), x, a);
    } else if (m < 31) C = two_link_P(links, x, 3, m - 28, 0, a);
    else {
      const int q = (m - 31) >> 1;
      C = two_link_P(links, x, ((m - 31) & 1) ? 5 : 4, q == 2 ? 1 : 0, q == 0 ? 1 : 2, a);
    }
  }
#pragma unroll
  for (int e = 0; e < 9; ++e) {
    cx v;
    v.x = (real)C.e[e].x;
    v.y = (real)C.e[e].y;
    dst[pauli_elem_index(e, lane)] = v;
  }
}

// term 9..26 -> family, directions, sign and the spin coefficients of K (term order of ok.h)
struct KronTerm {
  int fam, i, j;
  bool neg;
  double kD, sk[3];   // D = kD 1 ; S = s1 sigma_1 + s2 sigma_2 + s3 sigma_3 (real coefficients)
};
__device__ __forceinline__ KronTerm kron_term_of(int term, const PrecalcArgs& a) {
  KronTerm t;
  t.j = 0;
  if (term < 15) {
    t.fam = 3; t.i = (term - 9) >> 1; t.neg = ((term - 9) & 1) != 0;
  } else {
    const int q = (term - 15) >> 2, w = (term - 15) & 3;
    t.i = q == 2 ? 1 : 0;
    t.j = q == 0 ? 1 : 2;
    t.fam = w < 2 ? 4 : 5;
    t.neg = (w & 1) != 0;
  }
  t.kD = t.fam == 3 ? a.dii : 0.0;
  t.sk[0] = t.sk[1] = t.sk[2] = 0.0;
  const double sgn = t.neg ? -1.0 : 1.0;
  if (t.fam == 3) {
#pragma unroll
    for (int d = 0; d < 3; ++d) t.sk[d] = d == t.i ? sgn * a.sii : 0.0;
  } else {
#pragma unroll
    for (int d = 0; d < 3; ++d) t.sk[d] = d == t.i ? sgn * a.sij : (d == t.j ? sgn * (t.fam == 4 ? a.sij : -a.sij) : 0.0);
  }
  return t;
}
// spin row alpha of K = [[D, S], [S, D]], S2[al][be] = [[s3, s1 - i s2], [s1 + i s2, -s3]]: K[beta], beta = 2 bj + be
__device__ __forceinline__ void kron_K_row(const KronTerm& t, int alpha, double2 (&K)[4]) {
  const int bi = alpha >> 1, al = alpha & 1;
#pragma unroll
  for (int beta = 0; beta < 4; ++beta) {
    const int bj = beta >> 1, be = beta & 1;
    double2 v;
    if (bi == bj) {
      v = make_double2(al == be ? t.kD : 0.0, 0.0);
    } else if (al == be) {
      v = make_double2(al == 0 ? t.sk[2] : -t.sk[2], 0.0);
    } else {
      v = make_double2(t.sk[0], al == 0 ? -t.sk[1] : t.sk[1]);
    }
    K[beta] = v;
  }
}

template <typename real>
__global__ void __launch_bounds__(32 * 3) kron_terms_kernel(const double2* __restrict__ links, typename WUnit<real>::type* __restrict__ W,
                                                            PrecalcArgs a) {
  using unit_t = typename WUnit<real>::type;
  constexpr int NC = WUnit<real>::NC;
  const int lane = threadIdx.x;
  const int term = 9 + blockIdx.y * 3 + threadIdx.y;
  const int blk = blockIdx.x;
  const int n = (blk + a.blk0) * kBlock + lane;
  unit_t* Wt = W + ((size_t)blk * kTerms + term) * 12 * NC * kBlock + lane;
  if (n >= a.g.V) {   // padded site: zeros
    unit_t z = {};
    for (int u = 0; u < 12 * NC; ++u) Wt[(size_t)u * kBlock] = z;
    return;
  }
  const KronTerm t = kron_term_of(term, a);
  Site x = site_of(n, a.g);
  if (t.neg)   // the positive blocks live at x + offset(term)
    for (int mu = 0; mu < 4; ++mu) x = shift(x, mu, c_poff[term][mu], a.g);
  cm3 P = two_link_P(links, x, t.fam, t.i, t.j, a);
  if (t.neg) P = adj(P);
#pragma unroll 1
  for (int alpha = 0; alpha < 4; ++alpha) {
    double2 K[4];
    kron_K_row(t, alpha, K);
#pragma unroll
    for (int ca = 0; ca < 3; ++ca) {
      double2 row[12];
#pragma unroll
      for (int beta = 0; beta < 4; ++beta)
#pragma unroll
        for (int cb = 0; cb < 3; ++cb) row[3 * beta + cb] = cmul(K[beta], P.e[3 * ca + cb]);
      store_dense_row<real>(Wt + (size_t)(3 * alpha + ca) * NC * kBlock, row);
    }
  }
}

// ------------------------------------------------------------------------- 12-RHS tile writer
// The 12-RHS W tile of a site (ok_internal.cuh) interleaves the four terms of a K stage inside 16-byte core-matrix rows, so a
// (site, term) thread would write 8-byte pieces 31 KB apart.  mrhs_tiles_kernel computes the entries where they are needed
// instead: one CTA = one 32-site block x one HALF stage (two stencil terms = the even or the odd 768-byte k chunks of the
// stage: 3 x 768 B per site), one thread per (site, term, colour row ca).  A thread forms its four spin rows (alpha, ca) --
// terms 0..8 by pauli_term_rows, terms 9..26 as K (x) (row ca of P) -- rounds them once to fp32 exactly as the dense layout
// does, splits every number into its two fp16 pieces and puts them into the site's tile image in shared memory (74 KB, two
// CTAs per SM); the CTA then writes the images with coalesced 16-byte stores.  The last stage (three terms, 5 k chunks, its
// K order differs) is done by two CTAs of 16 sites x 3 terms.  No dense intermediate, no workspace beyond the scratch fields.
struct LinkRef {
  const double2* p;   // element e at p[e Vpad]
  double sg;          // boundary sign
  bool dag;
};
__device__ __forceinline__ LinkRef link_ref(const double2* __restrict__ links, const Site& s, int mu, bool dag, const PrecalcArgs& a) {
  LinkRef L;
  L.p = links + (size_t)(9 * mu) * a.Vpad + index_of(s, a.g);
  L.sg = (a.bc[mu] < 0 && s.c[mu] == (mu == 3 ? a.tfold : a.g.L[mu] - 1)) ? -1.0 : 1.0;
  L.dag = dag;
  return L;
}
__device__ __forceinline__ double2 link_el(const LinkRef& L, int r, int c, int Vpad) {   // element (r, c) of U or U^dag
  const double2 v = __ldg(L.p + (size_t)(L.dag ? 3 * c + r : 3 * r + c) * Vpad);
  return make_double2(L.sg * v.x, L.dag ? -L.sg * v.y : L.sg * v.y);
}
// out[t] += (X Y)[ca][t]  (tr = false)   or   (X Y)[t][ca]  (tr = true: the caller conjugates, row ca of (X Y)^dag)
__device__ __forceinline__ void acc_prod_line(double2 (&out)[3], const LinkRef& X, const LinkRef& Y, bool tr, int ca, int Vpad) {
  double2 v[3];
#pragma unroll
  for (int m = 0; m < 3; ++m) v[m] = tr ? link_el(Y, m, ca, Vpad) : link_el(X, ca, m, Vpad);
#pragma unroll
  for (int t = 0; t < 3; ++t)
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      const double2 b = tr ? link_el(X, t, m, Vpad) : link_el(Y, m, t, Vpad);
      cmac(out[t], v[m], b);
    }
}
// row ca of the colour matrix of a two-link term (two_link_P at x, or its adjoint for an opposite-direction term)
__device__ __forceinline__ void two_link_P_row(const double2* __restrict__ links, const Site& x, const KronTerm& t, int ca, const PrecalcArgs& a,
                                               double2 (&P)[3]) {
  const int i = t.i, j = t.j;
#pragma unroll
  for (int c = 0; c < 3; ++c) P[c] = make_double2(0.0, 0.0);
  if (t.fam == 3) {
    acc_prod_line(P, link_ref(links, x, i, false, a), link_ref(links, shift(x, i, 1, a.g), i, false, a), t.neg, ca, a.Vpad);
  } else if (t.fam == 4) {
    acc_prod_line(P, link_ref(links, x, i, false, a), link_ref(links, shift(x, i, 1, a.g), j, false, a), t.neg, ca, a.Vpad);
    acc_prod_line(P, link_ref(links, x, j, false, a), link_ref(links, shift(x, j, 1, a.g), i, false, a), t.neg, ca, a.Vpad);
  } else {
    const Site xmj = shift(x, j, -1, a.g);
    acc_prod_line(P, link_ref(links, x, i, false, a), link_ref(links, shift(xmj, i, 1, a.g), j, true, a), t.neg, ca, a.Vpad);
    acc_prod_line(P, link_ref(links, xmj, j, true, a), link_ref(links, xmj, i, false, a), t.neg, ca, a.Vpad);
  }
  if (t.neg) {
#pragma unroll
    for (int c = 0; c < 3; ++c) P[c].y = -P[c].y;
  }
}

// the 24 complex numbers of pauli_term_tables as fp16 pieces: [0 = D, 1 = S][combo][cb] -> (Re, Im) as __half2
struct HalfTab {
  uint32_t hi[2][4][3], lo[2][4][3];
};
// one complex number, rounded once to fp32 (as the dense layout stores it), then split as mrhs_split does
__device__ __forceinline__ void split_cx(const double2& v, uint32_t& hi, uint32_t& lo) {
  const float fx = (float)v.x, fy = (float)v.y;
  const __half2 h = __floats2half2_rn(fx, fy);
  const float2 b = __half22float2(h);
  const __half2 l = __floats2half2_rn((fx - b.x) * kMrhsLoScale, (fy - b.y) * kMrhsLoScale);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

constexpr int kTilesThreads = 192;                               // 32 sites x 2 terms x 3 colour rows
constexpr int kTilesHalfBytes = 3 * 768;                         // a half stage of one site: its 3 k chunks
constexpr int kTilesLastBytes = 5 * 768;                         // stage 6 of one site (the all-pad k chunk 5 is not stored)
constexpr int kTilesSmem = kBlock * (kTilesHalfBytes + 16);      // 74 240 (>= 16 x (3840 + 16)); + 16: odd multiple of 16 B between sites

// LAST = false: grid (blocks, 12 half stages), CTA = 32 sites x 2 terms.  LAST = true: grid (blocks, 2), CTA = 16 sites x the 3 terms of stage 6.
template <bool LAST>
__global__ void __launch_bounds__(kTilesThreads, 2) mrhs_tiles_kernel(const double2* __restrict__ links, const cm3* __restrict__ FS,
                                                                       __half* __restrict__ tiles, PrecalcArgs a) {
  extern __shared__ __align__(16) uint8_t sm[];
  const int tid = threadIdx.x, blk = blockIdx.x, h = blockIdx.y;
  constexpr int nsite = LAST ? 16 : 32, nterm = LAST ? 3 : 2;
  constexpr int stride = (LAST ? kTilesLastBytes : kTilesHalfBytes) + 16;
  const int stage = LAST ? 6 : h >> 1;
  const int s = tid & (nsite - 1), item = tid / nsite;          // item = 3 tl + ca
  const int site0 = blk * kBlock + (LAST ? h * 16 : 0);
  if (LAST) {   // the pad k = 36..39 of the last stage (the second slot of every row of k chunk 4) is zero; no thread below writes it
    for (int q = tid; q < nsite * 48; q += kTilesThreads) {
      const int zs = q / 48, row = q - 48 * zs;
      reinterpret_cast<uint2*>(sm + zs * stride)[4 * 96 + 2 * row + (1 ^ ((zs >> 3) & 1))] = make_uint2(0u, 0u);
    }
  }
  const int n = site0 + s;
  if (item < 3 * nterm && n < a.g.V) {
    const int tl = item / 3, ca = item - 3 * tl;
    const int term = LAST ? 24 + tl : 4 * stage + 2 * (h & 1) + tl;
    HalfTab T;
    uint32_t mUL = 0xffffffffu, mLR = 0xffffffffu, sLL = 0u;   // zero / sign masks of the UL, LR, LL blocks
    if (term < 9) {
      const PauliTerm t = pauli_term_of(term, n, links, FS, a);
      double2 Dv[4][3], Sv[4][3];
      pauli_term_tables(t, ca, a, Dv, Sv);
#pragma unroll
      for (int c = 0; c < 4; ++c)
#pragma unroll
        for (int cb = 0; cb < 3; ++cb) {
          split_cx(Dv[c][cb], T.hi[0][c][cb], T.lo[0][c][cb]);
          split_cx(Sv[c][cb], T.hi[1][c][cb], T.lo[1][c][cb]);
        }
      mUL = t.ulA ? 0xffffffffu : 0u;
      mLR = t.lrA ? 0xffffffffu : 0u;
      sLL = t.llsgn < 0.0 ? 0x80008000u : 0u;
    } else {   // W = K (x) P: D = kD 1 (x) P, S = (s1 sigma_1 + s2 sigma_2 + s3 sigma_3) (x) P
      const KronTerm t = kron_term_of(term, a);
      Site x = site_of(n, a.g);
      if (t.neg)
        for (int mu = 0; mu < 4; ++mu) x = shift(x, mu, c_poff[term][mu], a.g);
      double2 P[3];
      two_link_P_row(links, x, t, ca, a, P);
#pragma unroll
      for (int cb = 0; cb < 3; ++cb) {
        split_cx(make_double2(t.kD * P[cb].x, t.kD * P[cb].y), T.hi[0][0][cb], T.lo[0][0][cb]);
        T.hi[0][1][cb] = T.hi[0][0][cb]; T.lo[0][1][cb] = T.lo[0][0][cb];
        T.hi[0][2][cb] = T.hi[0][3][cb] = T.lo[0][2][cb] = T.lo[0][3][cb] = 0u;
        split_cx(make_double2(t.sk[2] * P[cb].x, t.sk[2] * P[cb].y), T.hi[1][0][cb], T.lo[1][0][cb]);
        T.hi[1][1][cb] = T.hi[1][0][cb] ^ 0x80008000u; T.lo[1][1][cb] = T.lo[1][0][cb] ^ 0x80008000u;
        split_cx(cmul(make_double2(t.sk[0], -t.sk[1]), P[cb]), T.hi[1][2][cb], T.lo[1][2][cb]);
        split_cx(cmul(make_double2(t.sk[0], t.sk[1]), P[cb]), T.hi[1][3][cb], T.lo[1][3][cb]);
      }
    }
    // The image of a site in 8-byte slots: [k chunk][row group w48/8 : 6][w48 % 8][k % 8 / 4]; a slot holds columns 4g .. 4g + 3 of
    // one term.  Sites 8 apart share their banks: the odd ones among them swap the two slots of every 16 bytes.
    uint2* mine = reinterpret_cast<uint2*>(sm + s * stride);
    const int swz = (s >> 3) & 1;
    int gslot[3];
#pragma unroll
    for (int g = 0; g < 3; ++g) {
      if (LAST) { const int sq = 3 * tl + g; gslot[g] = (2 * (sq >> 2) + ((sq & 3) >> 1)) * 96 + ((sq & 1) ^ swz); }
      else gslot[g] = g * 96 + (tl ^ swz);
    }
#pragma unroll
    for (int alpha = 0; alpha < 4; ++alpha) {
      const int r = 3 * alpha + ca, bi = alpha >> 1, al = alpha & 1;
      uint2* rowp = mine + (r >> 2) * 16 + (r & 3) * 4;   // B rows w = 8 (r / 4) + 2 (r % 4) + part (hi) and w + 24 (lo)
#pragma unroll
      for (int g = 0; g < 3; ++g) {
        uint2* dst = rowp + gslot[g];
#pragma unroll
        for (int hl = 0; hl < 2; ++hl)
#pragma unroll
          for (int part = 0; part < 2; ++part) {
            uint32_t w[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {   // columns 4 g + 2 e and the next
              const int c0 = 4 * g + 2 * e, c1 = c0 + 1;
              const int be0 = c0 / 3, cb0 = c0 % 3, be1 = c1 / 3, cb1 = c1 % 3;
              const int bj = be0 >> 1;      // = be1 >> 1: a column pair never straddles the spin blocks
              const int ds = bi == bj ? 0 : 1;
              const int k0 = al == (be0 & 1) ? al : (al == 0 ? 2 : 3), k1 = al == (be1 & 1) ? al : (al == 0 ? 2 : 3);
              const uint32_t v0 = hl ? T.lo[ds][k0][cb0] : T.hi[ds][k0][cb0], v1 = hl ? T.lo[ds][k1][cb1] : T.hi[ds][k1][cb1];
              uint32_t v = __byte_perm(v0, v1, part ? 0x7632 : 0x5410);
              if (ds == 0) v &= bi == 0 ? mUL : mLR;
              else if (bi == 1) v ^= sLL;
              w[e] = v;
            }
            dst[hl * 48 + part * 2] = make_uint2(w[0], w[1]);
          }
      }
    }
  }
  __syncthreads();
  // images -> tiles in 768-byte pieces (48 x 16 B): thread = (16-byte unit u of a piece, site ss = pp, pp + 4, ...); half stage: the
  // 3 pieces are the even or the odd k chunks of the stage, last stage: 5 contiguous pieces
  constexpr int npiece = LAST ? 5 : 3;
  const int u = tid % 48, pp = tid / 48;
  const uint8_t* src = sm + pp * stride + u * 16;
  uint8_t* dstg = reinterpret_cast<uint8_t*>(tiles) + ((size_t)(site0 + pp) * kMrhsWSiteHalves + (size_t)stage * kMrhsStageHalves) * 2 +
                  (LAST ? 0 : (h & 1) * 768) + u * 16;
#pragma unroll 2
  for (int ss = pp; ss < nsite; ss += 4, src += 4 * stride, dstg += (size_t)4 * kMrhsWSiteBytes) {
    if (site0 + ss >= a.g.V) break;
    const bool swp = (ss >> 3) & 1;
#pragma unroll
    for (int g = 0; g < npiece; ++g) {
      uint4 v = *reinterpret_cast<const uint4*>(src + g * 768);
      if (swp) { uint32_t t0 = v.x; v.x = v.z; v.z = t0; t0 = v.y; v.y = v.w; v.w = t0; }
      *reinterpret_cast<uint4*>(dstg + g * (LAST ? 768 : 1536)) = v;
    }
  }
}

size_t precalc_work_bytes(const ok_params* p) {
  Geom g = make_geom(p);
  return (size_t)(6 + kHopMats + 4) * g.nblk * kBlock * sizeof(cm3);
}

int launch_precalc(const ok_params* p, const void* links, void* Wp, void* work) {
  return launch_precalc_window(p, links, Wp, work, p->dims[3] - 1, 0, -1);
}

// p: the lattice the LINKS live on.  win_nblk < 0: W of the whole lattice.  Otherwise (t-slab, ok_slab.cu): W of the
// 32-site blocks [win_blk0, win_blk0 + win_nblk) only, written compactly to Wp, every term assembled by its own thread
// (the partner site of the pairing trick may lie outside the window); nrhs = 1, OK_W_DENSE.
int launch_precalc_window(const ok_params* p, const void* links, void* Wp, void* work, int tfold, int win_blk0, int win_nblk) {
  if (!g_poff_uploaded) {
    OK_CUDA(cudaMemcpyToSymbol(c_poff, kOffsets, sizeof(kOffsets)));
    static int h[3][kTerms][2][4];
    for (int f = 0; f < 3; ++f) sparse_fill_runs(f + 1, h[f]);
    OK_CUDA(cudaMemcpyToSymbol(c_qrun, h, sizeof(h)));
    g_poff_uploaded = true;
  }
  PrecalcArgs a;
  a.g = make_geom(p);
  for (int d = 0; d < 4; ++d) a.bc[d] = p->bc[d];
  a.Vpad = a.g.nblk * kBlock;
  a.mrhs = p->nrhs == 12;
  a.storage = p->storage;
  a.pair = (p->nrhs == 1 && p->storage != OK_W_CONJ && win_nblk < 0) ? 1 : 0;   // chunks / windows: the partner site may be outside
  a.tfold = tfold;
  a.posonly = (a.pair || p->storage == OK_W_CONJ) ? 1 : 0;
  const double u0 = p->u0, u2 = u0 * u0, u3 = u2 * u0, u4 = u2 * u2;
  a.mass = u0 / (2.0 * p->kappa);
  a.d0 = -(p->cB * p->zeta + 16.0 * p->c5) / (2.0 * u3);
  a.s0 = -(p->cE * p->zeta) / (2.0 * u3);
  a.s4 = p->cEE / (2.0 * u4);
  a.a1 = 0.5 * (p->zeta - 2.0 * p->c1 - 12.0 * p->c2);
  a.cs = p->c3 / (2.0 * u4);
  a.d1 = -0.5 * (p->rs * p->zeta + 8.0 * p->c4);
  a.cg = 0.25 * p->c5 * (1.0 / u2 - 1.0 / u4);
  a.c5u = p->c5 / u4;
  a.dii = p->c4 / u0;
  a.sii = (p->c1 + 2.0 * p->c2) / (2.0 * u0);
  a.sij = p->c2 / (2.0 * u0);
  cm3* FS = static_cast<cm3*>(work);
  cudaStream_t st = ctx().stream;
  // scratch: [6 clover fields][15 hop blocks][the 4 links, transposed]
  double2* linksT = reinterpret_cast<double2*>(FS + (size_t)(6 + kHopMats) * a.Vpad);
  transpose_links_kernel<<<(unsigned)(((long long)36 * a.g.V + 255) / 256), 256, 0, st>>>(static_cast<const double2*>(links), linksT, a);
  OK_LAUNCHED("transpose_links_kernel");
  links = linksT;
  field_strength_kernel<<<dim3((a.g.V + 127) / 128, 6), 128, 0, st>>>(static_cast<const double2*>(links), FS, a);
  OK_LAUNCHED("field_strength_kernel");
  hop_blocks_kernel<<<dim3((a.g.V + 127) / 128, 12), 128, 0, st>>>(static_cast<const double2*>(links), FS, FS + (size_t)6 * a.Vpad, a);
  OK_LAUNCHED("hop_blocks_kernel");
  const dim3 block(32, 3);
  const double2* lk = static_cast<const double2*>(links);
#define OK_ASM_LAUNCH(CLS, NY, NB, OUT)                                                                                     \
  do {                                                                                                                      \
    if (p->precision == OK_FP64) assemble_W_kernel<double, CLS><<<dim3(NB, NY), block, 0, st>>>(lk, FS, static_cast<double2*>(OUT), a); \
    else assemble_W_kernel<float, CLS><<<dim3(NB, NY), block, 0, st>>>(lk, FS, static_cast<float4*>(OUT), a);               \
    OK_LAUNCHED("assemble_W_kernel");                                                                                       \
  } while (0)
#define OK_PAULI_LAUNCH(NB, OUT)                                                                                            \
  do {                                                                                                                      \
    if (p->precision == OK_FP64) pauli_terms_kernel<double><<<dim3(NB, 3), block, 0, st>>>(lk, FS, static_cast<double2*>(OUT), a); \
    else pauli_terms_kernel<float><<<dim3(NB, 3), block, 0, st>>>(lk, FS, static_cast<float4*>(OUT), a);                    \
    OK_LAUNCHED("pauli_terms_kernel");                                                                                      \
  } while (0)
#define OK_KRON_LAUNCH(NB, OUT)                                                                                             \
  do {                                                                                                                      \
    if (p->precision == OK_FP64) kron_terms_kernel<double><<<dim3(NB, 6), block, 0, st>>>(lk, static_cast<double2*>(OUT), a); \
    else kron_terms_kernel<float><<<dim3(NB, 6), block, 0, st>>>(lk, static_cast<float4*>(OUT), a);                         \
    OK_LAUNCHED("kron_terms_kernel");                                                                                       \
  } while (0)
  a.blk0 = 0;
  if (a.mrhs) {   // the split-fp16 tiles straight from the scratch fields and links
    static bool attr_set = false;
    if (!attr_set) {
      OK_CUDA(cudaFuncSetAttribute(mrhs_tiles_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTilesSmem));
      OK_CUDA(cudaFuncSetAttribute(mrhs_tiles_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kTilesSmem));
      attr_set = true;
    }
    mrhs_tiles_kernel<false><<<dim3(a.g.nblk, 12), kTilesThreads, kTilesSmem, st>>>(lk, FS, static_cast<__half*>(Wp), a);
    OK_LAUNCHED("mrhs_tiles_kernel");
    mrhs_tiles_kernel<true><<<dim3(a.g.nblk, 2), kTilesThreads, kTilesSmem, st>>>(lk, FS, static_cast<__half*>(Wp), a);
    OK_LAUNCHED("mrhs_tiles_kernel");
    return OK_SUCCESS;
  }
  const int nb = win_nblk < 0 ? a.g.nblk : win_nblk;
  a.blk0 = win_nblk < 0 ? 0 : win_blk0;
  if (p->storage == OK_W_PAULI) {
    const dim3 pgrid(nb, (OK_W_PAULI_MATS + 3) / 4), pblock(32, 4);
    if (p->precision == OK_FP64) pauli_store_kernel<double><<<pgrid, pblock, 0, st>>>(lk, FS, static_cast<double2*>(Wp), a);
    else pauli_store_kernel<float><<<pgrid, pblock, 0, st>>>(lk, FS, static_cast<float2*>(Wp), a);
    OK_LAUNCHED("pauli_store_kernel");
    return OK_SUCCESS;
  }
  if (p->storage == OK_W_DENSE) {
    OK_PAULI_LAUNCH(nb, Wp);
    OK_KRON_LAUNCH(nb, Wp);
  } else {
    OK_ASM_LAUNCH(1, (a.posonly ? 1 : 2), nb, Wp);   // the heavy class first
    OK_ASM_LAUNCH(0, 1, nb, Wp);
    OK_ASM_LAUNCH(2, (a.posonly ? 1 : 2), nb, Wp);
    OK_ASM_LAUNCH(3, (a.posonly ? 2 : 4), nb, Wp);
  }
#undef OK_ASM_LAUNCH
#undef OK_KRON_LAUNCH
#undef OK_PAULI_LAUNCH
  return OK_SUCCESS;
}

}  // namespace okd
