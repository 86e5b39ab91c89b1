// Structure of the 27 precalculation matrices and the two reduced W storage formats.
//
// Every W of Eqs. (2.6)-(2.12), (2.3), (2.10) is a 2 x 2 arrangement of 6 x 6 blocks over
// upper/lower spin, [[UL, UR], [LL, LR]], each 6 x 6 = 2 x 2 spin x 3 x 3 colour, of the form
//     UL, LR in {0, D}      UR = S      LL = +S  (LL = -S for the on-site term W^0, Eq. 2.6)
// and D, S have fixed zero patterns in their 2 x 2 spin structure (sigma_3 and 1 are diagonal, sigma_1,
// sigma_2 off-diagonal).  172 of the 432 colour blocks of a site vanish identically.
//   OK_W_BLOCK : the 260 non-zero colour blocks, every quadrant stored on its own (any matrix with the
//                zero pattern is representable)                      ->  2340 complex / site, 18 720 B fp32
//   OK_W_DS    : D and S stored once per term (UL = LR = D, LL = +-S are implied by the equations)
//                                                                    ->  1188 complex / site,  9 504 B fp32
//   OK_W_CONJ  : OK_W_DS for W^0 and the 13 positive-direction terms only; an opposite-direction matrix is
//                taken from the positive one of the neighbour site, Eqs. (2.3), (2.10):
//                    W^-_o(x) = [[D^dag, -S^dag], [-S^dag, D^dag]] of W^+_o(x - o)   (UL/LR presence swapped for +-t)
//                                                                    ->   630 complex / site,  5 040 B fp32
// Device layout of both: [block of 32 sites][unit][site 32][complex], unit order
//     [term 27][a = spin row inside the 6 x 6 : 2][stored matrix m][colour row 3][non-zero spin column][colour column 3]
// so that the warp that owns spin row a reads one contiguous run per term.
#pragma once

#include "ok_internal.cuh"

namespace okd {

struct TermDesc {
  int maskD;    // 2 x 2 spin-block mask of D: bit (2 a + b); 0 = the term has no diagonal quadrant
  int ul, lr;   // quadrant UL / LR holds D
  int maskS;    // mask of S (UR and LL)
  int negLL;    // LL = -S
};

constexpr int kMaskFull = 0xF, kMaskDiag = 0x9, kMaskOff = 0x6;

__host__ __device__ constexpr TermDesc term_desc(int term) {
  if (term == 0) return {kMaskFull, 1, 1, kMaskFull, 1};                    // W^0      Eq. (2.6)
  if (term <= 6) return {kMaskFull, 1, 1, kMaskFull, 0};                    // W^+-_i   Eqs. (2.8), (2.10)
  if (term == 7) return {kMaskDiag, 0, 1, kMaskFull, 0};                    // W^+_4 = [[0,S],[S,-U]]   Eq. (2.7)
  if (term == 8) return {kMaskDiag, 1, 0, kMaskFull, 0};                    // W^-_4 = [[-U^dag,-S^dag],[-S^dag,0]]
  if (term <= 14) return {kMaskDiag, 1, 1, (term - 9) / 2 == 2 ? kMaskDiag : kMaskOff, 0};   // W^{++}_ii: S ~ sigma_i   Eq. (2.9)
  return {0, 0, 0, (term - 15) / 4 == 0 ? kMaskOff : kMaskFull, 0};         // pairs: S ~ sigma_i +- sigma_j   Eqs. (2.11), (2.12)
}

__host__ __device__ constexpr int mask_row(int mask, int a) { return (mask >> (2 * a)) & 3; }
__host__ __device__ constexpr int popc2(int m) { return (m & 1) + ((m >> 1) & 1); }

// term order of ok.h: every even term > 0 is the opposite direction of the odd term before it
__host__ __device__ constexpr bool term_is_neg(int term) { return term > 0 && (term & 1) == 0; }

// stored matrices of a term: OK_W_BLOCK m = 0..3 -> UL, UR, LL, LR ; OK_W_DS / OK_W_CONJ m = 0, 1 -> D, S
__host__ __device__ constexpr int sparse_nmat(int fmt) { return fmt == OK_W_BLOCK ? 4 : 2; }
__host__ __device__ constexpr int sparse_mat_mask(int fmt, int term, int m) {
  const TermDesc d = term_desc(term);
  if (fmt == OK_W_CONJ && term_is_neg(term)) return 0;   // rebuilt from term - 1 of the neighbour site
  if (fmt != OK_W_BLOCK) return m == 0 ? ((d.ul || d.lr) ? d.maskD : 0) : d.maskS;
  return m == 0 ? (d.ul ? d.maskD : 0) : m == 3 ? (d.lr ? d.maskD : 0) : d.maskS;
}
// complex units a (term, spin row a, matrix m) run holds: 3 colour rows x non-zero spin columns x 3 colour columns
__host__ __device__ constexpr int sparse_run_units(int fmt, int term, int a, int m) {
  return 9 * popc2(mask_row(sparse_mat_mask(fmt, term, m), a));
}
__host__ __device__ constexpr int sparse_run_offset(int fmt, int term, int a, int m) {
  int off = 0;
  for (int t = 0; t <= term; ++t)
    for (int aa = 0; aa < 2; ++aa)
      for (int mm = 0; mm < sparse_nmat(fmt); ++mm) {
        if (t == term && aa == a && mm == m) return off;
        off += sparse_run_units(fmt, t, aa, mm);
      }
  return off;
}
__host__ __device__ constexpr int sparse_site_units(int fmt) { return sparse_run_offset(fmt, kTerms - 1, 1, sparse_nmat(fmt) - 1) + sparse_run_units(fmt, kTerms - 1, 1, sparse_nmat(fmt) - 1); }
__host__ __device__ constexpr int sparse_site_units_rt(int fmt) { return fmt == OK_W_BLOCK ? 2340 : fmt == OK_W_DS ? 1188 : 630; }   // runtime format
static_assert(sparse_site_units(OK_W_BLOCK) == 260 * 9, "260 non-zero colour blocks (PAPER.md:63: 432 - 172)");
static_assert(sparse_site_units(OK_W_DS) == 132 * 9, "D, S once per term");
static_assert(sparse_site_units(OK_W_CONJ) == 70 * 9, "D, S of W^0 and of the 13 positive-direction terms");
static_assert(sparse_site_units_rt(OK_W_BLOCK) == sparse_site_units(OK_W_BLOCK) && sparse_site_units_rt(OK_W_DS) == sparse_site_units(OK_W_DS) &&
              sparse_site_units_rt(OK_W_CONJ) == sparse_site_units(OK_W_CONJ), "runtime table");

// Where element (row, col) of W_term lives: unit index inside the site (or -1 when it is not stored), and for
// OK_W_DS whether it is stored (stored = 1) or implied by another quadrant (stored = 0, sign = +-1 of the copy).
struct SparseRef {
  int unit;     // -1: structurally zero
  int stored;   // this quadrant is the one kept in memory
  int sign;     // value = sign * stored value (LL of W^0; off-diagonal quadrants of a conjugated term)
  int conj;     // value = sign * conj(stored value)                         (OK_W_CONJ, opposite-direction terms)
  int shift;    // >= 0: the stored value lives at the site x + offset[shift] (OK_W_CONJ, opposite-direction terms)
};
// `runs` = table [term][a][m] of sparse_run_offset for the format (nullptr: computed on the fly, slow)
__host__ __device__ inline SparseRef sparse_ref(int fmt, int term, int row, int col, const int (*runs)[2][4] = nullptr) {
  const TermDesc d = term_desc(term);
  const int hr = row / 6, a = (row % 6) / 3, cr = row % 3, hc = col / 6, b = (col % 6) / 3, cc = col % 3;
  const int quad = 2 * hr + hc;   // 0 UL, 1 UR, 2 LL, 3 LR
  SparseRef r = {-1, 1, 1, 0, -1};
  const bool diag = quad == 0 || quad == 3;
  if (diag && !(quad == 0 ? d.ul : d.lr)) return r;
  const int mask = diag ? d.maskD : d.maskS;
  const int mr = mask_row(mask, a);
  if (!((mr >> b) & 1)) return r;
  if (fmt == OK_W_CONJ && term_is_neg(term)) {
    // element [a,cr][b,cc] of D^dag (resp. -S^dag) = conj of element [b,cc][a,cr] of the positive term's D (resp. -S)
    const int m2 = diag ? 0 : 1, mrb = mask_row(mask, b), nbb = popc2(mrb), jj = (a == 1 && (mrb & 1)) ? 1 : 0;
    r.stored = 0;
    r.sign = diag ? 1 : -1;
    r.conj = 1;
    r.shift = term;
    r.unit = (runs ? runs[term - 1][b][m2] : sparse_run_offset(fmt, term - 1, b, m2)) + (cc * nbb + jj) * 3 + cr;
    return r;
  }
  int m = quad;
  if (fmt != OK_W_BLOCK) {
    m = diag ? 0 : 1;
    // the kept copy: D from UL when present (else LR), S from UR
    r.stored = diag ? ((quad == 0) || !d.ul) : (quad == 1);
    r.sign = (quad == 2 && d.negLL) ? -1 : 1;
  }
  const int nb = popc2(mr), bc = (b == 1 && (mr & 1)) ? 1 : 0;
  r.unit = (runs ? runs[term][a][m] : sparse_run_offset(fmt, term, a, m)) + (cr * nb + bc) * 3 + cc;
  return r;
}

// host helper: fills table[term][a][m] for a format
inline void sparse_fill_runs(int fmt, int (*table)[2][4]) {
  for (int t = 0; t < kTerms; ++t)
    for (int a = 0; a < 2; ++a)
      for (int m = 0; m < 4; ++m) {
        const int ts = (fmt == OK_W_CONJ && term_is_neg(t)) ? t - 1 : t;   // a conjugated term reads the runs of its partner
        table[t][a][m] = m < sparse_nmat(fmt) ? sparse_run_offset(fmt, ts, a, m) : 0;
      }
}

}  // namespace okd
