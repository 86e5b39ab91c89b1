/* ok.h -- C-ABI of libokdirac: the precalculated-W Oktay-Kronfeld Dirac apply, the W
 * precalculation and BiCGStab, on one NVIDIA B200 (sm_100a).
 *
 * Reference: arXiv:1311.5029, Sec. 2.  Problem statement:
 *   - Eq. (2.1): solve  sum_{y,beta,b} M^{alpha beta,ab}_{xy} psi^{beta b}_y = xi^{alpha a}_x ;
 *   - Eq. (2.2): M psi is a 27-term stencil, each term a per-site 12x12 complex spin-colour
 *     matrix W ("precalculation matrix") times the 12-spinor at x + offset;
 *   - "The W matrices remain the same for all CG iterations. We precalculate and reuse them."
 * Hence the three calls: ok_precalc_W (links -> W), ok_dirac_apply (W, psi -> M psi),
 * ok_bicgstab (W, xi -> psi; "bi-stabilized CG").
 *
 * General rules
 *   - Every data pointer is a DEVICE pointer (cudaMalloc'ed / torch CUDA tensor), 16-byte
 *     aligned, unless the argument is documented as HOST.  `ok_params*`, `iters`, `resid`
 *     are HOST pointers.
 *   - The caller owns every buffer.  The library allocates no persistent device memory and
 *     frees nothing; scratch comes from the buffer given to ok_set_workspace (one exception: the
 *     fixed 1.5 MiB static array behind ok_dirac_apply_dot_static, see there).
 *   - All work is enqueued on the stream given to ok_set_stream (default: the legacy default
 *     stream).  Calls are asynchronous except ok_bicgstab, ok_*_host and the first use of a W
 *     buffer the library has not seen (one 1 KiB header read), which synchronise that stream.
 *   - Return value: 0 (OK_SUCCESS) or a negative ok_status.  No exceptions, no aborts.
 *   - There is no CPU fallback: without a CUDA device every compute call returns OK_ECUDA.
 *   - One device and one calling thread per process (the model is one process per GPU): the stream, the workspace,
 *     the W handle table and a few device-side scratch symbols are process-wide state, not per-call arguments.
 *     The library binds to the CUDA device that is current at its first compute call; a later call on another
 *     device returns OK_EINVAL (its constant tables live on the bound device only).
 *   - Errors of a kernel that faults while running surface at the next synchronising call.  With the environment
 *     variable OK_SYNC_CHECK=1 every launch is followed by a stream synchronisation, so OK_ECUDA names the kernel
 *     that faulted (debugging aid; serialises the stream).
 *
 * Canonical (external) layouts, complex numbers interleaved (re, im):
 *   site index   n = x + Lx*(y + Ly*(z + Lz*t)),  dims = {Lx, Ly, Lz, T};  V = Lx*Ly*Lz*T
 *   links        double  U[n][mu][a][b][2]   mu = 0,1,2 (x,y,z), 3 (t); U_mu(x) joins x to x+mu;
 *                always fp64 (the precalculation computes in fp64 and rounds W once)
 *   spinor       real    psi[n][3*alpha+a][2]            (alpha = spin 0..3, a = colour 0..2)
 *   multi-RHS    real    psi[n][3*alpha+a][rhs][2]       (nrhs = 12)
 *   W            real    W[n][term][3*alpha+a][3*beta+b][2]   term order below
 *   `real` is float for OK_FP32 and double for OK_FP64.
 *
 * Stencil term order (Eq. 2.2), offsets in lattice units (dx,dy,dz,dt):
 *   0: 0 | 1,2: +x,-x | 3,4: +y,-y | 5,6: +z,-z | 7,8: +t,-t | 9,10: +2x,-2x | 11,12: +2y,-2y |
 *   13,14: +2z,-2z | then for (i,j) = (x,y),(x,z),(y,z): +i+j, -i-j, +i-j, -i+j  (15..26).
 *   out(x) = sum_term W_term(x) psi(x + offset_term), coordinates modulo dims.  Boundary
 *   conditions (bc) are folded into W by ok_precalc_W; ok_dirac_apply is purely periodic.
 *
 * Internal (device) layouts -- what psi/out/src/x/W of the three main calls hold.  Sites are
 * grouped in blocks of 32 consecutive site indices (the last block zero-padded):
 *   spinor  [block][c][site_in_block][16 bytes]   fp32: c = 0..5, (re,im) of components 2c, 2c+1
 *                                                 fp64: c = 0..11, (re,im) of component c
 *   W       1024-byte header, then [block][term][row 0..11][c][site_in_block][16 bytes]
 *           with c pairing the COLUMNS of W exactly as the spinor pairs components.
 *   OK_W_BLOCK / OK_W_DS: header, then [block][unit][site_in_block][complex]; the unit order is the list of
 *           stored colour-block rows in csrc/ok_sparse.cuh.  ok_pack_W drops what the format does not keep
 *           (OK_W_DS keeps UL (else LR) as D and UR as S); ok_unpack_W rebuilds the full 12 x 12 matrices.
 *   OK_W_PAULI: header, then per block and stored colour matrix m = 0..36 (csrc/ok_pauli.cu) 288 complex numbers: the row-major
 *           3 x 3 elements in pairs, [pair e/2 : 4][site_in_block][2], then element 8 as [site_in_block] (a lane moves 16 bytes).
 *   nrhs=12 (fp32, OK_W_DENSE only): spinor = 256-byte header, then per-site fp32 records [component/4][2*rhs+part][component%4]
 *           (1152 B, the field), then per-site tensor-core operand records (1152 B: the same numbers scaled per right-hand
 *           side by a power of two and split into two fp16 pieces).  The operand records are what ok_dirac_apply reads; they
 *           are written by ok_pack_spinor and by the solver for its own vectors, and rebuilt on demand (two passes over the
 *           field) when ok_dirac_apply is given a field whose header says they are stale, e.g. the `out` of an earlier
 *           apply.  Never write such a buffer except through this library.
 *           W = per-site split-fp16 tensor-core tiles (31 488 B), see csrc/ok_internal.cuh.
 *   Use ok_pack_ and ok_unpack_ to convert; the sizes are given by ok_vec_bytes and ok_W_bytes.
 */
#ifndef OK_H_
#define OK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define OK_FP32 0
#define OK_FP64 1

/* W storage formats (ok_params.storage).  All three hold the same operator, Eq. (2.2); the reduced ones
 * exploit the fixed structure of the 27 matrices, W = [[UL,UR],[LL,LR]] over upper/lower spin with
 * UL, LR in {0, D}, UR = S, LL = +-S (Eqs. 2.6-2.12) and fixed zero colour blocks
 * (172 of the 432 per site).  nrhs = 12 supports OK_W_DENSE only. */
#define OK_W_DENSE 0        /* 27 x 12 x 12 complex per site: 31 104 B (fp32)                              */
#define OK_W_BLOCK 1        /* the 260 non-zero colour blocks, each quadrant on its own: 18 720 B (fp32)   */
#define OK_W_DS 2           /* D and S once per term (132 colour blocks): 9 504 B (fp32)                   */
#define OK_W_CONJ 3         /* OK_W_DS for W^0 and the 13 positive-direction terms only (70 colour blocks,  */
                            /* 5 040 B fp32); the opposite-direction matrices are rebuilt from the          */
                            /* neighbour site by the conjugation relations, Eqs. (2.3), (2.10) */

#define OK_W_PAULI 4        /* the Pauli components of D and S of W^0 and the 13 positive-direction terms: the paper's "50 colour  */
                            /* blocks" (49 by the structure of Eqs. 2.6-2.12, 37 stored matrices = 2 664 B fp32   */
                            /* once components that coincide up to a constant of the action are merged; csrc/ok_pauli.cu).        */
                            /* Written by ok_precalc_W only (ok_pack_W returns OK_EINVAL: a general W has no such form);          */
                            /* ok_unpack_W rebuilds the 27 dense matrices.  The apply is bound by the fp32 pipes, not by HBM.     */
#define OK_W_PAULI_MATS 37

#define OK_NTERMS 27
#define OK_SITE_BLOCK 32
#define OK_W_HEADER_BYTES 1024

typedef enum ok_status {
  OK_SUCCESS = 0,
  OK_EINVAL = -1,      /* bad dims / precision / nrhs / null or misaligned pointer / unknown W   */
  OK_ECUDA = -2,       /* CUDA runtime or launch error; text via ok_strerror(OK_ECUDA)           */
  OK_EBREAKDOWN = -3,  /* BiCGStab breakdown: |rho|, |<rhat,v>|, <t,t> or |omega| < 1e-300 / NaN */
  OK_EMAXIT = -4,      /* BiCGStab did not converge in maxit iterations (x, iters, resid valid)   */
  OK_EWORKSPACE = -5,  /* workspace missing or smaller than ok_work_bytes                        */
  OK_ECOMM = -6        /* a caller-supplied ok_comm callback returned non-zero                   */
} ok_status;

typedef struct ok_params {
  int32_t dims[4];    /* Lx, Ly, Lz, T; each >= 2                                              */
  int32_t precision;  /* OK_FP32 / OK_FP64: storage and arithmetic of W and spinors            */
  int32_t bc[4];      /* +1 periodic, -1 antiperiodic (fermion field); paper: {+1,+1,+1,-1}    */
  int32_t nrhs;       /* 1, or 12 for the multi-right-hand-side mode (fp32 only)               */
  double kappa, u0;   /* hopping parameter, tadpole factor (Eq. 2.6)                           */
  double zeta, rs;    /* Eqs. (2.6)-(2.8)                                                      */
  double cB, cE, cEE, c1, c2, c3, c4, c5;
  int32_t storage;    /* OK_W_DENSE / OK_W_BLOCK / OK_W_DS / OK_W_CONJ / OK_W_PAULI: how W is held in device memory */
  int32_t reserved_;  /* 0; OK_SLAB (1) in the parameters of a t-slab (see ok_slab_*): dims[3] is then the slab's    */
                      /* own extent Tloc and the lattice is open in t (its t-neighbours arrive as halo slices)       */
} ok_params;

/* ---- sizes (pure host arithmetic; 0 on invalid params) ---------------------------------- */
size_t ok_W_bytes(const ok_params* p);    /* device bytes of W incl. header and block padding   */
size_t ok_vec_bytes(const ok_params* p);  /* device bytes of one spinor field, internal layout  */
size_t ok_work_bytes(const ok_params* p); /* workspace needed by ok_precalc_W, ok_bicgstab, ok_*_host */

/* ---- execution context ------------------------------------------------------------------ */
int ok_set_stream(void* cuda_stream);             /* cudaStream_t as void*; NULL = default stream */
int ok_set_workspace(void* dev, size_t bytes);    /* DEVICE scratch, caller-owned, 256-B aligned  */

/* ---- layout conversion (device -> device, asynchronous) --------------------------------- */
int ok_pack_spinor(const ok_params* p, const void* canon, void* packed);
int ok_unpack_spinor(const ok_params* p, const void* packed, void* canon);
/* canonical W [n][27][12][12] (precision of p) <-> internal W; ok_pack_W also writes the header.
 * Lets a caller inject precalculation matrices computed elsewhere, or inspect them. */
int ok_pack_W(const ok_params* p, const void* canon_W, void* W);
int ok_unpack_W(const void* W, void* canon_W);

/* ---- the hot path ------------------------------------------------------------------------ */

/* Precalculation, PAPER.md:59, 89-107 (Eqs. 2.6-2.12, 2.3, 2.10): builds the 27 matrices per
 * site from SU(3) links (canonical layout, fp64) and writes them, with the header, into W
 * (ok_W_bytes).  Arithmetic in fp64; W rounded once to p->precision.  Needs the workspace. */
int ok_precalc_W(const void* links, const ok_params* params, void* W);

/* Dirac apply, PAPER.md:53-55 (Eq. 2.2): out = M psi.  psi, out: internal spinor layout,
 * out must not alias psi.  Dimensions/precision are taken from W's header.
 * nrhs = 12: psi's operand records are brought up to date first if its header marks them stale (the buffer behind the
 * const pointer is written in that case); out gets fp32 records only. */
int ok_dirac_apply(const void* W, const void* psi, void* out);

/* BiCGStab: solves M x = src (x0 = 0; x on entry ignored), unpreconditioned,
 * reductions and scalars in fp64 with a fixed summation order (bit-reproducible).  Stops when
 * the recursive residual satisfies ||r|| <= tol ||src|| AND the recomputed true residual does
 * too (otherwise restarts from the true residual).  *iters = BiCGStab iterations (2 applies
 * each); *resid = true relative residual ||src - M x|| / ||src|| at exit.  nrhs = 12: every
 * column has its own scalars; converged columns are frozen; *iters = max over columns and
 * *resid = max over columns.  iters/resid: HOST pointers.  Needs the workspace. */
int ok_bicgstab(const void* W, const void* src, void* x, double tol, int maxit, int* iters, double* resid);

/* CG on the normal equations M^dag M x = M^dag src ("M^dag M preconditioning"), with
 * M^dag = Gamma_5 M Gamma_5: a second solver on the same apply, nrhs = 1, any precision and W storage format.
 * Same conventions as ok_bicgstab (x0 = 0, fp64 fixed-order reductions, stop on ||r|| <= tol ||src|| confirmed by the
 * true residual); *iters = CG iterations (2 applies each).  Needs the workspace (ok_work_bytes). */
int ok_cgnr(const void* W, const void* src, void* x, double tol, int maxit, int* iters, double* resid);

/* Mixed-precision inversion, PAPER.md:114 ("We perform a mixed precision inversion by calling the ... inverter or
 * Dirac operation module in single or double precision, as appropriate"): defect correction around the fp32
 * BiCGStab with both sets of precalculation matrices resident,
 *     x = 0, r = src;  repeat { stop if ||r|| <= tol ||src|| ;  e = ok_bicgstab(W32, r/||r|| in fp32, inner_tol) ;
 *                               x += ||r|| e ;  r = src - M x with W64 }.
 * W64: fp64 W, W32: fp32 W of the same lattice (any storage format each); src, x: fp64 internal spinor layout.
 * maxit bounds the total number of fp32 BiCGStab iterations, max_outer the corrections.  *iters = total inner
 * iterations, *outer = corrections done, *resid = fp64 true relative residual.  iters/outer/resid: HOST pointers.
 * Needs a workspace of ok_mixed_work_bytes(p) bytes (p: the parameters of either W).  Synchronises the stream. */
size_t ok_mixed_work_bytes(const ok_params* p);
int ok_bicgstab_mixed(const void* W64, const void* W32, const void* src, void* x, double tol, double inner_tol,
                      int maxit, int max_outer, int* iters, int* outer, double* resid);

/* Same apply with HOST spinors in the canonical layout (precision of W): copies psi to the
 * device, packs, applies, unpacks and copies back, synchronising the stream.  W stays
 * device-resident across calls (the paper keeps the precalculation matrices on the GPU and
 * copies the fermion field every call).  Needs the workspace.
 * nrhs = 1, OK_W_DENSE, T >= 8, Lx*Ly*Lz a multiple of 32 and a field of at least 8 MiB (or OK_HOST_PIPELINE set in the
 * environment, for tests): the call is pipelined over chunks of time slices on two
 * library-owned copy streams beside the caller's stream (the stencil reaches one slice in t), so the copies
 * hide behind the W stream; pinned host buffers are needed for that overlap (pageable ones still work, serially). */
int ok_dirac_apply_host(const void* W, const void* psi_host, void* out_host);

/* ---- t-slab decomposition ------------------------------------------------------------------
 * The path shards along T: "In the temporal direction, only the nearest neighbors are involved", "off-node
 * communications are necessary only for the outermost boundary surfaces" (the paper itself runs on 4 nodes,
 * PAPER.md:120).  The lattice (Lx, Ly, Lz, T) is cut into slabs of Tloc consecutive time slices, slab s owning global
 * t = t0 .. t0 + Tloc - 1.  W is slab-local and never communicated; per apply one time slice of the spinor (Lx Ly Lz * 96 B
 * in fp32: 768 KB at 20^3) travels each way between t-neighbours, and a BiCGStab iteration adds four all-gathers of three
 * doubles per slab.  One process may hold several slabs (that is also how the decomposition is verified on one GPU).
 *
 * Slab parameters: an ok_params with dims = {Lx, Ly, Lz, Tloc}, reserved_ = OK_SLAB, nrhs = 1, storage = OK_W_DENSE,
 * Lx*Ly*Lz a multiple of 32 (a time slice is then a whole number of 32-site blocks), Tloc >= 2, Tloc + 4 <= T.
 * Slab fields ("extended" internal layout, ok_slab_vec_bytes): [lower halo slice][Tloc slices][upper halo slice], each slice
 * ok_slab_slice_bytes long; the middle part IS an ordinary internal-layout field of the (Lx, Ly, Lz, Tloc) lattice, so
 * ok_pack_spinor / ok_unpack_spinor with (base + ok_slab_slice_bytes) convert it.  The library fills the halos itself inside
 * ok_slab_bicgstab; for ok_slab_dirac_apply the caller puts the neighbours' boundary slices there. */
#define OK_SLAB 1
#define OK_SLAB_LINK_HALO 2   /* time slices of links a slab's W needs beyond its own, below and above */

/* Communication between processes, supplied by the caller (torch.distributed in the Python binding: plumbing only).
 * Both callbacks receive DEVICE pointers, must order their transfers after the work already enqueued on the library's
 * stream and before work enqueued on it afterwards, and return 0 on success.  NULL callbacks / NULL ok_comm: the process
 * holds the whole T extent. */
typedef struct ok_comm {
  int32_t rank, nranks;     /* consecutive groups of slabs live on consecutive ranks; every rank holds the same number */
  /* send_lo (this process's first time slice) goes to rank - 1, which receives it in ITS recv_hi; send_hi (the last
   * slice) goes to rank + 1's recv_lo; ranks are cyclic.  `bytes` each. */
  int (*exchange)(void* user, const void* send_lo, const void* send_hi, void* recv_lo, void* recv_hi, size_t bytes);
  /* recv[r * n + i] = send[i] of rank r, for all ranks, n doubles each */
  int (*allgather)(void* user, const double* send, double* recv, int n);
  void* user;
} ok_comm;

size_t ok_slab_slice_bytes(const ok_params* slab);   /* bytes of one time slice of a field, internal layout            */
size_t ok_slab_vec_bytes(const ok_params* slab);     /* (Tloc + 2) slices                                              */
/* workspace: ok_slab_precalc_W needs ok_slab_work_bytes(slab, 1, 1); ok_slab_bicgstab over nslab equal slabs in one process
 * of nranks needs ok_slab_work_bytes(slab, nslab, nranks) */
size_t ok_slab_work_bytes(const ok_params* slab, int nslab, int nranks);

/* Precalculation of one slab's W (same matrices, Eqs. 2.6-2.12, as ok_precalc_W gives for these sites on the whole lattice).
 * links_ext: canonical fp64 links [n][mu][3][3] of the Tloc + 2*OK_SLAB_LINK_HALO global time slices
 * t0 - 2 .. t0 + Tloc + 1 (modulo T), n = x + Lx (y + Ly (z + Lz k)), k = 0 .. Tloc + 3.  The antiperiodic sign of
 * slab->bc[3] is applied to U_4 of global slice T - 1 wherever it falls in that window.  W: ok_W_bytes(slab). */
int ok_slab_precalc_W(const void* links_ext, const ok_params* slab, int T_global, int t0, void* W);

/* Eq. (2.2) on one slab: out(x) for the slab's sites; psi_ext must hold the two halo slices.  out_ext's halos are not written. */
int ok_slab_dirac_apply(const void* W, const void* psi_ext, void* out_ext);

/* The same apply with the halo exchange fused into it (only the two outermost time slices of a node's
 * sub-lattice involve its neighbours): the halo slices of psi_ext are NOT read; wherever Eq. (2.2) reaches across the lower /
 * upper t-face the kernel loads psi(x -+ t) straight from lo_slice / hi_slice -- the lower neighbour's LAST own time slice and
 * the upper neighbour's FIRST own time slice, internal layout, ok_slab_slice_bytes each.  Any address this GPU can load from
 * will do: another slab's field in the same process (its ext base + Tloc slices, resp. + 1 slice), or a buffer in a
 * neighbour GPU's memory opened through CUDA peer access / IPC, in which case the neighbour's slice crosses NVLink once, as
 * the 512-byte lines the warps ask for, with no copy kernel, staging buffer or collective in front of the apply.  The caller
 * orders the call after the neighbours have finished writing those slices (same stream, an event, or a barrier between the
 * processes) and keeps them unchanged until the apply has completed.  Bit-identical to ok_slab_dirac_apply on filled halos. */
int ok_slab_dirac_apply_peer(const void* W, const void* psi_ext, const void* lo_slice, const void* hi_slice, void* out_ext);

/* BiCGStab (as ok_bicgstab) over the nslab slabs this process holds, in t order (W[s], src_ext[s], x_ext[s] of slab s);
 * with comm, over nslab * comm->nranks slabs in all.  Every reduction is summed per slab and then over the slabs in global
 * order, so the iteration is bit-reproducible and independent of how the slabs are dealt to processes.  *iters, *resid as
 * ok_bicgstab, identical on every process.  Pointer arrays, iters, resid: HOST.
 * Between slabs of one process the applies read each other's boundary slices in place (as ok_slab_dirac_apply_peer does); only
 * the two outer faces of a process go through comm->exchange into halo slices. */
int ok_slab_bicgstab(int nslab, const void* const* W, const void* const* src_ext, void* const* x_ext, double tol, int maxit,
                     const ok_comm* comm, int* iters, double* resid);

/* Peer access for ok_slab_bicgstab (optional).  With peers set, a process's two OUTER t-faces are read in place as well: its
 * applies load the neighbour processes' boundary slices straight from their memory (NVLink peer access / CUDA IPC mappings), and
 * comm->exchange is not called; barrier() takes its place before every apply.  Requirements: every process holds the same number
 * of equal slabs and has given ok_set_workspace a buffer of the same size (the solver's vectors then sit at the same offsets
 * everywhere); lo_work / hi_work = the lower / upper neighbour's workspace base as mapped into THIS process; lo_x = x_ext of the
 * lower neighbour's LAST slab, hi_x = x_ext of the upper neighbour's FIRST slab, mapped likewise; barrier(user) returns 0 once
 * all work enqueued so far on every process's library stream is complete (or ordered before whatever the streams run next).
 * The neighbours never overwrite a slice while it may still be read: every apply is followed by an all-gather of its
 * reductions.  NULL clears the setting.  Results are bit-identical to the exchange path. */
typedef struct ok_slab_peers {
  const void *lo_work, *hi_work, *lo_x, *hi_x;
  int (*barrier)(void* user);
  void* user;
} ok_slab_peers;
int ok_slab_set_peers(const ok_slab_peers* peers);

/* ---- an entry point that allocates nothing ------------------------------------------------ */
/* For callers that cannot call cudaMalloc and have no workspace to lend (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid allocation): the Dirac apply of Eq. (2.2) together with the three
 * reductions BiCGStab takes from it,
 *     out = M psi ,   result[0..2] = ( Re<a,out>, Im<a,out>, ||out||^2 ) ,   <a,b> = sum conj(a) b ,
 * fp64 sums in a fixed order (bit-reproducible).  W, psi, a, out as in ok_dirac_apply (nrhs = 1, any precision and W storage
 * format; out must alias neither psi nor a); result: DEVICE, 3 doubles, written by the call (asynchronously, on the library's stream).
 * The per-block partial sums live in a static __device__ array inside the library instead of the workspace: 1.5 MiB
 * (65 536 rows of 3 doubles) on every GPU that loads the library, for lattices of up to OK_STATIC_MAX_SITES sites.  Larger
 * lattices are rejected with OK_EINVAL and a message in ok_static_strerror().  The call uses neither the workspace nor
 * cudaMalloc / cudaFree nor any allocating library routine.  Every call shares the one array: calls whose kernels overlap on the GPU
 * (two streams) race on it; calls on one stream are safe, nothing in the array has to be cleared between them.
 * The first use of a W buffer the library has not seen reads its 1 KiB header synchronously (General rules). */
#define OK_STATIC_MAX_SITES 2097152   /* 32^3 x 64 */
int ok_dirac_apply_dot_static(const void* W, const void* psi, const void* a, void* out, double* result);
size_t ok_static_max_sites(void);          /* = OK_STATIC_MAX_SITES */
const char* ok_static_strerror(void);      /* text of the last error ok_dirac_apply_dot_static returned */

/* ---- diagnostics -------------------------------------------------------------------------- */
/* Read the parameters stored in W's header back into *p (HOST).  Always reads the 1 KiB device header (synchronises the
 * stream) and refreshes the library's host-side record of W from it. */
int ok_W_params(const void* W, ok_params* p);
/* Drop the library's host-side record of W (the header mirror that lets the three main calls run
 * without a params argument and without reading the device).  Call it before freeing the buffer or
 * reusing its memory for anything else; a later W written there by ok_precalc_W / ok_pack_W is
 * recorded again.  Unknown pointers are ignored.  Returns OK_SUCCESS.
 * Hazard this guards against: the record, not the device header, decides which kernels run.  ok_precalc_W / ok_pack_W
 * drop every record whose byte range overlaps the W they write, so reusing memory THROUGH the library is safe; a W
 * buffer overwritten by a plain device copy (say a checkpoint restore with other dims or storage) must be followed by
 * ok_forget_W or ok_W_params, which re-reads the header. */
int ok_forget_W(const void* W);
/* Layout query for the reduced storage formats (pure host arithmetic, no device needed): where element (row, col) of
 * W_term is kept.  Returns the complex-unit index inside a site's OK_W_BLOCK / OK_W_DS / OK_W_CONJ record
 * ([block][unit][site 32][complex]), or -1 when the element is structurally zero, or -2 on bad arguments.  info[0] = 1 if
 * this element is the stored copy (0: implied by another quadrant / by the neighbour site), info[1] = sign (+1/-1) and
 * info[2] = 1 if the value is the complex conjugate of the stored number, info[3] = term whose offset leads to the site
 * holding it (-1: the same site).  info: HOST, 4 ints, may be NULL. */
int ok_W_unit_index(int storage, int term, int row, int col, int* info);
/* Number of kernels the library has launched since load (for launch accounting in benches). */
uint64_t ok_launch_count(void);
const char* ok_strerror(int status);
const char* ok_version(void);

#ifdef __cplusplus
}
#endif
#endif /* OK_H_ */
