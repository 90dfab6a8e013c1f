/*
 * tm.h -- C-ABI boundary of the B200-native even-odd preconditioned Wilson twisted-mass dslash
 * (hot path of arXiv 1311.4462; citations are PAPER.md:<line> + section / equation).
 *
 * Operator (Eq. 2.1; readings C1-C3), hopping-parameter normalisation:
 *     M = 2 kappa D = R - kappa D_hop,     R = 1 + i a gamma5 tau3 + b tau1,  a = 2 kappa mu,  b = 2 kappa epsilon
 *     (D_hop psi)(x) = sum_mu  eta+ (1 - gamma_mu) U_mu(x) psi(x+mu) + eta- (1 + gamma_mu) U_mu(x-mu)^dag psi(x-mu)
 * periodic in space; in time the wrapped hop is multiplied by t_boundary (-1 = antiperiodic).
 * gamma matrices: gamma_4-diagonal "non-relativistic" basis (C5):
 *     gamma_k = [[0, i sigma_k], [-i sigma_k, 0]],  gamma_4 = diag(1,1,-1,-1),  gamma_5 = [[0,1],[1,0]].
 *
 * Everything runs on ONE GPU (sm_100a); there is no CPU fallback.  All functions return TM_OK (0) or a
 * negative tm_status; they never throw, abort or print.  tm_last_error() gives a thread-local message.
 *
 * HOST canonical order (always double, complex = (re, im), C-contiguous; never retained after return):
 *     spinor, full lattice : [flavor (n_flavor)][lex site (V)][spin 4][color 3][2]
 *     spinor, one parity   : [flavor (n_flavor)][cb  site (V/2)][spin 4][color 3][2]
 *     gauge                : [mu 0..3 = x,y,z,t][lex site (V)][row 3][col 3][2]  = U_mu(x), the link x -> x+mu,
 *                            pure SU(3), no boundary phase folded in
 *     lex = x1 + X (x2 + Y (x3 + Z x4)),  parity = (x1+x2+x3+x4) & 1 (0 = even),  cb = lex / 2.
 * DEVICE layout is private to the library: checkerboarded SoA in 128-bit chunks.
 */
#ifndef TM_H
#define TM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TM_OK = 0,
    TM_ERR_ARG = -1,          /* NULL handle / pointer, bad enum value                                   */
    TM_ERR_DIMS = -2,         /* an extent is odd or < 4 (the checkerboard needs even extents; at extent 2
                                 the forward and backward neighbours coincide)                           */
    TM_ERR_MISMATCH = -3,     /* operands differ in context, precision or flavor count; gauge precision
                                 differs from the fields'; params.twist_flavor disagrees with n_flavor   */
    TM_ERR_ALIAS = -4,        /* out aliases in (neighbour reads make in-place application impossible)   */
    TM_ERR_PARAM = -5,        /* |1 + a^2 - b^2| < 1e-12: R has no inverse; or epsilon != 0 with a single
                                 flavor; or t_boundary not +-1                                           */
    TM_ERR_NOMEM = -6,
    TM_ERR_CUDA = -7,         /* a CUDA call failed; tm_last_error() holds cudaGetErrorString            */
    TM_ERR_UNSUPPORTED = -8   /* tm_mat_pc(TM_MATPC_SYM, dagger=1): needs the D R^-1 ordering */
} tm_status;

typedef enum { TM_DOUBLE = 8, TM_SINGLE = 4, TM_HALF = 2 } tm_precision;
/* TM_HALF: 16-bit fixed point, one float norm per (site, flavor): q = rint(v * 32767 / max|v|)
 * (Table 1 "half"; format per DESIGN.md reading C9); arithmetic in fp32.              */

typedef enum { TM_RECON_18 = 18, TM_RECON_12 = 12, TM_RECON_8 = 8 } tm_recon;
/* TM_RECON_12: rows 0 and 1 stored, row 2 = conj(row0 x row1) rebuilt in the kernel.
 * TM_RECON_8 : "8 ... parameter reconstruct" (Table 1 rows "8").  Stored per link: U01, U02, U10
 *   (complex) and arg(U00)/pi, arg(U20)/pi; the kernel rebuilds |U00|, |U20| from the unit norm of row 0 and
 *   column 0, U11 and U12 from <row0,row1> = 0 and U20 = conj(U01 U12 - U02 U11), then row 2 as for 12-real
 *   (chart: DESIGN.md reading C11).  The chart divides by N = |U01|^2 + |U02|^2: rounding errors grow like
 *   eps / N and a link with N < 1e-10 (e.g. the unit matrix) makes tm_gauge_load return TM_ERR_PARAM.    */

typedef enum { TM_EVEN = 0, TM_ODD = 1 } tm_parity;

typedef enum {                       /* the fused kernels of PAPER.md:68 (section 2.1); p = output parity */
    TM_TWIST_INV_DSLASH = 0,         /* A      : out_p = R^-1 D_hop in                                   */
    TM_TWIST_INV_DSLASH_XPAY = 1,    /* A-xpay : out_p = x_p - kappa^2 R^-1 D_hop in                     */
    TM_DSLASH_TWIST_XPAY = 2,        /* B      : out_p = R x_p - kappa^2 D_hop in                        */
    TM_RECONSTRUCT = 3,              /* REC    : out_p = R^-1 (x_p + kappa D_hop in)     (Eq. 2.4)       */
    /* the same hopping kernels with no twist (R = 1): the pieces of M^_sym^dag and of the right-hand sides */
    TM_DSLASH_XPAY = 4,              /*          out_p = x_p - kappa^2 D_hop in                          */
    TM_DSLASH_AXPY = 5,              /*          out_p = x_p + kappa D_hop in                            */
    /* the fused "D R^-1" forms: the inverse twist is applied to the 8 neighbour INPUT sites in registers before the spin
     * projection ("all local operators ... merged into dslash kernels"; the right-hand sides
     * b_e + kappa D_eo R_oo^-1 b_o, and the exact adjoint of Eq. 2.3's operator).  gamma5 mixes the spin halves and tau1 the
     * flavors, so these kernels read the whole neighbour site on the time hops too (one spinor of traffic more per site
     * than kernel A, two fewer than a separate twist pass).                                                          */
    TM_TWIST_INV_DSLASH_TWIST_INV = 6, /*        out_p = R^-1 D_hop R^-1 in                                */
    TM_RECONSTRUCT_TWIST_INV = 7,    /*          out_p = R^-1 (x_p + kappa D_hop R^-1 in)                  */
    TM_DSLASH_TWIST_INV_AXPY = 8     /*          out_p = x_p + kappa D_hop R^-1 in                         */
} tm_kernel_type;
/* dagger != 0: D_hop -> D_hop^dag (projectors swapped) and R -> R^dag (a -> -a), order kept.            */

typedef enum { TM_MATPC_ASYM = 0 /* LHS of Eq. 2.2 */, TM_MATPC_SYM = 1 /* LHS of Eq. 2.3 */ } tm_matpc;

typedef struct {
    double kappa, mu, epsilon;   /* bare mu-bar, epsilon-bar                          */
    int twist_flavor;            /* +1 / -1: one flavor, tau3 -> +-1, epsilon must be 0 (QUDA_TWIST_PLUS /
                                    MINUS); 0: non-degenerate doublet (n_flavor = 2)     */
    int t_boundary;              /* -1 antiperiodic in time, +1 periodic                                 */
} tm_params;

typedef struct tm_ctx tm_ctx;       /* lattice geometry + device + stream                                 */
typedef struct tm_field tm_field;   /* ONE single-parity spinor field (V/2 sites, n_flavor flavors)       */
typedef struct tm_gauge tm_gauge;   /* all 4V links, both parities                                        */

/* ---- context ------------------------------------------------------------------------------------- */
/* dims: host pointer to {X, Y, Z, T}. Selects cuda_device for the calling thread. */
int tm_init(const int dims[4], int cuda_device, tm_ctx **ctx);
/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 * All later compute calls on this context are enqueued there. */
int tm_set_stream(tm_ctx *ctx, void *cuda_stream);
int tm_sync(tm_ctx *ctx);           /* cudaStreamSynchronize; surfaces asynchronous faults */
void tm_finalize(tm_ctx *ctx);      /* does not free fields / gauges created from it */

/* ---- fields (a1 of DESIGN.md: checkerboarded SoA layouts) ------------------------------------------
 * A field is one parity of a spinor -- the operands of the even-odd preconditioned operators of PAPER.md:56-66 (Eq. 2.2-2.4
 * act on psi_e / psi_o) --, with n_flavor = 1 for the degenerate doublet (epsilon = 0 in Eq. 2.1: the flavors
 * decouple) or 2 for the non-degenerate one ("one has to apply the dslash on both flavors"), in one of the three
 * storage precisions of Table 1. */
size_t tm_field_bytes(const tm_ctx *ctx, tm_precision prec, int n_flavor);   /* 0 on bad arguments */
/* ext_dev_ptr == NULL: the library allocates (and frees in tm_field_free).  Otherwise ext_dev_ptr is DEVICE
 * memory of at least tm_field_bytes() bytes, 256-byte aligned, BORROWED (e.g. a torch tensor's storage). */
int tm_field_alloc(tm_ctx *ctx, tm_precision prec, int n_flavor, void *ext_dev_ptr, size_t ext_bytes,
                   tm_field **f);
void tm_field_free(tm_field *f);
void *tm_field_device_ptr(const tm_field *f);
/* host_full: HOST pointer, full-lattice canonical spinor; only the sites of `parity` are read / written.
 * Both calls synchronise the context stream. */
int tm_field_upload(tm_field *f, tm_parity parity, const double *host_full);
int tm_field_download(const tm_field *f, tm_parity parity, double *host_full);
/* host_cb: HOST pointer, single-parity canonical spinor [n_flavor][V/2][4][3][2] in cb order of `parity`.
 * (The cb order does not depend on the parity; the argument is kept for symmetry and validated.) */
int tm_field_upload_cb(tm_field *f, tm_parity parity, const double *host_cb);
int tm_field_download_cb(const tm_field *f, tm_parity parity, double *host_cb);
/* Asynchronous forms (host_cb: HOST pointer to PINNED memory, same layout as above).  They return at once: the copies run on
 * two private streams (one per direction, each with its own device staging buffer) and are ordered against the kernels of
 * the context stream by events -- an upload's pack kernel waits for the kernels already queued (they may still read the
 * field), kernels queued afterwards wait for it; a download unpacks after the kernels already queued, kernels queued
 * afterwards wait for the unpack (not for the copy).  So the H2D copy of the next input, the kernels and the D2H copy of the
 * previous result overlap.  The host buffers must stay valid, and a downloaded buffer is complete, only after tm_sync().
 * Consecutive transfers in the same direction run in issue order.                                                        */
int tm_field_upload_cb_async(tm_field *f, tm_parity parity, const double *host_cb);
int tm_field_download_cb_async(const tm_field *f, tm_parity parity, double *host_cb);
/* The same with the host array in SINGLE precision (same index order, float instead of double): half the bytes over PCIe for
 * fields whose device precision is single or half anyway (the conversion to the field's format happens in the pack kernel on
 * the device; a double field takes float input too, with float accuracy). */
int tm_field_upload_cb_async_f32(tm_field *f, tm_parity parity, const float *host_cb);
int tm_field_download_cb_async_f32(const tm_field *f, tm_parity parity, float *host_cb);

/* ---- host spin basis (SURVEY.md section 8f "minor": chiral <-> non-relativistic rotation in the pack kernels) ---- */
/* The kernels work in the non-relativistic basis of PAPER.md:52 (gamma_4 diagonal; reading C5), which is also
 * the default basis of host spinors.  With another host basis the pack / unpack kernels of tm_field_upload* /
 * tm_field_download* rotate the spin index: psi_device = S psi_host on upload, psi_host = S^dag psi_device on download,
 * where S is unitary with  gamma^host_mu = S^dag gamma^nonrel_mu S.  The setting belongs to the context and applies to
 * every later upload / download; fields already on the device are not touched.
 *   TM_BASIS_NONREL : S = 1 (default; `custom` ignored)
 *   TM_BASIS_CHIRAL : S = (1/sqrt 2) [[1, 1], [1, -1]] in 2x2 spin blocks, i.e. the chiral basis with
 *                     gamma_k = [[0, -i s_k], [i s_k, 0]], gamma_4 = [[0, 1], [1, 0]], gamma_5 = diag(1, 1, -1, -1)
 *                     (reading C12; `custom` ignored)
 *   TM_BASIS_CUSTOM : `custom` = HOST pointer to S as 32 doubles, row-major [4][4][re, im]; copied; must be unitary to
 *                     1e-12 (else TM_ERR_ARG)                                                                       */
typedef enum { TM_BASIS_NONREL = 0, TM_BASIS_CHIRAL = 1, TM_BASIS_CUSTOM = 2 } tm_basis;
int tm_set_host_basis(tm_ctx *ctx, tm_basis basis, const double *custom);

/* ---- gauge (a1, a4) -------------------------------------------------------------------------------- */
/* The gauge links U_mu(x) of the Wilson term D_W (Eq. 2.1; "re-use the gauge field"), stored per parity in the precision of the kernels
 * that read them and in one of the compressed forms of PAPER.md:97 ("12 or 8 parameter reconstruct"; 18 = uncompressed).
 * host_links: HOST pointer, canonical gauge field; copied (may be freed on return). */
int tm_gauge_load(tm_ctx *ctx, const double *host_links, tm_precision prec, tm_recon recon, tm_gauge **g);
void tm_gauge_free(tm_gauge *g);

/* ---- the hot path ---------------------------------------------------------------------------------- */
/* One fused kernel launch (rows a2-a9 of DESIGN.md).  out: field on `parity`; in: field on the
 * opposite parity; x: field on `parity` (NULL allowed only for TM_TWIST_INV_DSLASH).  out must not alias in
 * (TM_ERR_ALIAS); out may alias x.  `prec` must equal the operands' precision (TM_ERR_MISMATCH).
 * Asynchronous: enqueues on the context stream and returns. */
int tm_dslash_apply(tm_field *out, const tm_field *in, const tm_field *x, const tm_gauge *g,
                    const tm_params *p, tm_parity parity, int dagger, tm_kernel_type kt, tm_precision prec);

/* LHS of Eq. 2.2 (ASYM: out_e = (R_ee - kappa^2 D_eo R_oo^-1 D_oe) in_e) or Eq. 2.3 (SYM:
 * out_e = (1 - kappa^2 R_ee^-1 D_eo R_oo^-1 D_oe) in_e): two launches, tmp_o is the odd
 * intermediate R_oo^-1 D_oe in_e.  dagger: the exact adjoint.  ASYM: the same two launches with the daggered
 * kernels.  SYM: M^_sym^dag = 1 - kappa^2 D^dag_eo R^dag^-1_oo D^dag_oe R^dag^-1_ee (C7) = the fused
 * TM_TWIST_INV_DSLASH_TWIST_INV^dag kernel (R^dag^-1 D^dag R^dag^-1) and the plain xpay kernel: two launches as well
 * (half-precision doublets: the local twist into out_e first, three launches; out_e must not alias in_e, TM_ERR_ALIAS).
 * Asynchronous. */
int tm_mat_pc(tm_field *out_e, const tm_field *in_e, tm_field *tmp_o, const tm_gauge *g, const tm_params *p,
              tm_matpc type, int dagger);

/* The local twist alone, site by site on one parity field ("local operators"):
 * out = R in (inverse = 0) or R^-1 in (inverse = 1); dagger != 0: R -> R^dag (a -> -a).  out may be in itself
 * (in place) but must not partially overlap it.  TM_ERR_PARAM if R is singular.  Asynchronous. */
int tm_twist_apply(tm_field *out, const tm_field *in, const tm_params *p, int inverse, int dagger);

/* Right-hand side of Eq. 2.2 (ASYM: rhs_e = b_e + kappa D_eo R_oo^-1 b_o) or Eq. 2.3 (SYM: rhs_e = R_ee^-1 (b_e +
 * kappa D_eo R_oo^-1 b_o)), PAPER.md:60-64 in the reading C4 of DESIGN.md.  One launch of the fused D R^-1 kernel
 * (TM_DSLASH_TWIST_INV_AXPY / TM_RECONSTRUCT_TWIST_INV); half-precision doublets, for which the fused kernel measured
 * slower, take the local twist into tmp_o and the plain kernel instead (two launches).  tmp_o is scratch: a valid field that does
 * not alias b_e, b_o or rhs_e (TM_ERR_ALIAS); rhs_e may alias b_e.  Asynchronous. */
int tm_prepare_rhs(tm_field *rhs_e, const tm_field *b_e, const tm_field *b_o, tm_field *tmp_o, const tm_gauge *g,
                   const tm_params *p, tm_matpc type);

/* Eq. 2.4 (reading C4): psi_o = R_oo^-1 (b_o + kappa D_oe psi_e).  psi_o may alias b_o. */
int tm_reconstruct_odd(tm_field *psi_o, const tm_field *psi_e, const tm_field *b_o, const tm_gauge *g,
                       const tm_params *p);

/* ---- vector operations and the mixed-precision CG --- */
/* z = a x + b y on single-parity fields (y may be NULL: z = a x).  z may be x or y itself.  Precisions may differ in
 * these combinations: all equal; z double, x single / half, y double; z single / half, x double, y NULL or like z
 * (anything else: TM_ERR_UNSUPPORTED).  Half operands are dequantised / requantised site by site.  Asynchronous. */
int tm_field_axpby(tm_field *z, double a, const tm_field *x, double b, const tm_field *y);
/* *result (HOST) = Re <x, y> = sum over sites, flavors, spin, color of re x re y + im x im y, accumulated in double in
 * a fixed order (deterministic).  x = y gives |x|^2.  Synchronises the context stream. */
int tm_field_redot(const tm_field *x, const tm_field *y, double *result);
/* The same sum for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): *dev_result (DEVICE pointer to one double, the caller's) = Re <x, y>.  Calls no cudaMalloc / cudaFree and no
 * allocating library routine, copies nothing to the host and does not synchronise: two launches on the context stream.  Its
 * scratch (per-block partial sums) is a fixed 512 KiB __device__ array inside the library, held by every GPU that loads the
 * library until the process exits, hence the limit: fields of more than TM_NOALLOC_MAX_SITES sites per parity ->
 * TM_ERR_UNSUPPORTED (use tm_field_redot).  Same arithmetic and summation order as tm_field_redot: identical result.  Every call
 * on a device shares the array: calls that OVERLAP on the GPU (two contexts / streams on one device, two host threads) race
 * and return garbage; calls on one context are ordered by its stream.  The first call on a device looks up the array's
 * device address (cudaGetSymbolAddress: make one call before starting a capture).  With tm_set_allreduce the hook is applied
 * to *dev_result. */
#define TM_NOALLOC_MAX_SITES 8388608L     /* 65536 partial sums x 128 sites; 48^3 x 96 has 5 308 416 sites per parity */
int tm_field_redot_noalloc(const tm_field *x, const tm_field *y, double *dev_result);

/* Multi-GPU reductions: after tm_set_allreduce(ctx, fn, user) every sum the library forms (tm_field_redot, the scalars of
 * tm_invert_cg) is passed through fn(dev_sums, n, cuda_stream, user): dev_sums is a DEVICE array of n doubles holding this
 * rank's partial sums; fn must replace them by the sums over all ranks, ordered on `cuda_stream` (e.g. ncclAllReduce, or
 * torch.distributed.all_reduce on a tensor that aliases the memory), and return 0.  fn = NULL: single GPU (default). */
typedef int (*tm_allreduce_fn)(double *dev_sums, int n, void *cuda_stream, void *user);
int tm_set_allreduce(tm_ctx *ctx, tm_allreduce_fn fn, void *user);

/* The operator of the solver: by default tm_mat_pc on the context's lattice.  A distributed caller supplies its own
 * application of M (dagger = 0) / M^dag (dagger = 1) with the face exchange inside (paper_1311_4462_b200.sharded.Slab.mat_pc);
 * it must enqueue on the context stream and return 0. */
typedef int (*tm_cg_op_fn)(tm_field *out_e, const tm_field *in_e, tm_field *tmp_o, const tm_gauge *g, const tm_params *p,
                           tm_matpc type, int dagger, void *user);
typedef struct {
    double tol;                    /* stop when |b - A x| / |b| <= tol, the residual formed in double                 */
    int max_iter;                  /* cap on the number of CG iterations                                              */
    tm_precision sloppy_precision; /* precision of the CG iteration (TM_DOUBLE: plain double CG)                      */
    double delta;                  /* reliable update (true residual in double, solution accumulated in double) whenever
                                      the iterated residual has dropped by this factor since the last one
                                      (0 < delta < 1; e.g. 0.1 for single, 0.3 for half)                               */
    tm_cg_op_fn op;                /* NULL: tm_mat_pc                                                                  */
    void *op_user;
} tm_cg_params;
typedef struct {
    int iterations;                /* CG iterations (applications of A = M^dag M in the sloppy precision)             */
    int restarts;                  /* reliable updates (double-precision residual computations)                        */
    double residual;               /* last true relative residual |b - A x| / |b|                                      */
    int converged;                 /* 1 if residual <= tol                                                            */
} tm_cg_info;
/* ---- domain decomposition in y, z and t ---------------------------------
 * One sub-lattice X x Y_loc x Z_loc x T_loc of the global lattice per context (per GPU), a process grid over the directions
 * mu = 1 (y), 2 (z), 3 (t) in any combination; the local extents even, so local and global site parities agree.  x is never
 * cut (the checkerboard index lives on it).  PAPER.md:72: the packing routines "take into account the fifth flavor dimension
 * when gathering boundary-spinor sites in non-temporal lattice directions": a face of a non-temporal direction is a STRIDED
 * set of sites of the tiled layout, gathered per flavor.  One distributed dslash =
 *   for every cut direction: tm_halo_pack(in, dir)  ->  the two face buffers reach the neighbouring sub-lattices (either the
 *   buffers ARE the neighbours' receive buffers, mapped with CUDA IPC / peer access, and the pack kernel's stores are the
 *   transfer, signalled by the flags below; or the caller moves them: NCCL send / recv, paper_1311_4462_b200.sharded)
 *   ->  tm_dslash_apply with tm_set_open_dirs(ctx, mask) (the kernels give the hops that leave the sub-lattice in a cut
 *   direction the weight 0)  ->  for every cut direction: tm_halo_apply(out, dir),
 * after which `out` equals the single-lattice result on this sub-lattice (tests/test_gpu_sharded.py against the oracle on
 * the global lattice).  The exchange can overlap the interior kernel; tm_halo_apply follows both on the context stream.
 * Face buffers are DEVICE memory owned by the caller, tm_halo_bytes(dir) each: [n_flavor][V_loc / (2 L_dir)][12 reals] of
 * double (fp64 fields) or float (fp32 and half fields); site j of a face = checkerboard order of the face's sites
 * (x fastest, then the uncut coordinates in increasing order), the same on both sides of the cut.
 *   dev_to_prev  : spin-projected half-spinors ((1 -+ gamma_dir) psi, 12 reals per site AND FLAVOR) of the FIRST slice
 *                  x_dir = 0, for the previous sub-lattice's forward hops
 *   dev_to_next  : U_dir^dag times the projected half-spinors of the LAST slice, for the next one's backward hops (the link
 *                  lives with the sender)
 *   dev_from_prev = the previous sub-lattice's dev_to_next, dev_from_next = the next one's dev_to_prev
 *   sign_prev / sign_next : +1, or for dir = 3 the time boundary condition (-1 antiperiodic) where that face is the global
 *                  boundary (TM_ERR_ARG for -1 in a spatial direction: space is periodic)
 *   flags (all may be NULL = no signalling): DEVICE pointers to 32-bit unsigned words.  tm_halo_pack stores `epoch` to
 *   *dev_flag_prev and *dev_flag_next (system-scope release) after every face element has been written; tm_halo_apply
 *   spins until *dev_wait_prev >= epoch and *dev_wait_next >= epoch (system-scope acquire) before it reads the faces.  With
 *   peer-mapped receive buffers the sender's flag_prev / flag_next are words in the NEIGHBOURS' memory next to the buffers.
 *   Epochs must increase by one per exchange and direction; two receive-buffer sets used alternately (epoch & 1) make the
 *   scheme race-free for nearest-neighbour exchanges (paper_1311_4462_b200/sharded.py: PeerRing).
 * `out_parity`, `dagger`, `kt` are those of the tm_dslash_apply call being completed; every kernel type is supported
 * (the fused epilogues are affine in the hopping sum), and the directions' completions commute.
 * tm_set_open_dirs: mask bit mu (1 << mu) for mu = 1, 2, 3; TM_ERR_ARG for other bits.  tm_set_open_time(ctx, on) =
 * tm_set_open_dirs(ctx, on ? 8 : 0).                                                                                  */
int tm_set_open_dirs(tm_ctx *ctx, int mask);
int tm_set_open_time(tm_ctx *ctx, int on);
size_t tm_halo_bytes(const tm_ctx *ctx, tm_precision prec, int n_flavor, int dir);
int tm_halo_pack(const tm_field *in, const tm_gauge *g, tm_parity out_parity, int dagger, int dir, void *dev_to_prev, void *dev_to_next,
                 unsigned *dev_flag_prev, unsigned *dev_flag_next, unsigned epoch);
int tm_halo_apply(tm_field *out, const void *dev_from_prev, const void *dev_from_next, const tm_gauge *g, const tm_params *p,
                  tm_parity out_parity, int dagger, tm_kernel_type kt, int dir, int sign_prev, int sign_next,
                  const unsigned *dev_wait_prev, const unsigned *dev_wait_next, unsigned epoch);

/* Mixed-precision conjugate gradient on the normal equations of the even-odd preconditioned operator (the paper's
 * "double-single" / "double-half" CG) with RELIABLE UPDATES: solves
 *     M^dag M x_e = b_e ,   M = the LHS of Eq. 2.2 (ASYM) or Eq. 2.3 (SYM),
 * starting from x_e = 0 (the content of x_e on entry is ignored).  One CG recurrence runs in sloppy_precision; whenever
 * its residual has dropped by `delta` the partial solution is added to x_e in double, the true residual b - A x is formed
 * in double and replaces the iterated one, and the recurrence continues with the same search direction (no restart).
 * x_e, b_e and g_precise are double; g_sloppy is the same gauge field loaded in sloppy_precision (ignored, may be NULL,
 * when that is TM_DOUBLE).  The work fields live on the context and are reused by later solves (tm_cg_release frees
 * them; tm_finalize does too); nothing is allocated in a solve after the first.  The scalars of the recurrence stay on the
 * device; the host looks at them one iteration late (no stream synchronisation per iteration).  Returns TM_OK also when
 * max_iter was reached or the true residual stagnated (see info->converged); TM_ERR_PARAM on breakdown (<p, A p> <= 0). */
int tm_invert_cg(tm_field *x_e, const tm_field *b_e, const tm_gauge *g_precise, const tm_gauge *g_sloppy,
                 const tm_params *p, tm_matpc type, const tm_cg_params *cp, tm_cg_info *info);
void tm_cg_release(tm_ctx *ctx);

/* ---- diagnostics ----------------------------------------------------------------------------------- */
const char *tm_last_error(void);       /* thread-local, never NULL */
/* Number of dslash kernel launches issued through this context so far (bench.py's gpu_launches). */
long tm_launch_count(const tm_ctx *ctx);
/* Name of the kernel variant the last tm_dslash_apply on this context dispatched to (static string). */
const char *tm_last_kernel_name(const tm_ctx *ctx);
/* Per-launch device timing (bench.py's roofline leg): while enabled, every dslash launch is bracketed by CUDA
 * events on the context stream.  tm_timing_read synchronises, writes up to max_records (kernel name, milliseconds)
 * pairs in launch order into the HOST arrays names / ms, stores the number written in *n, and clears the log.
 * on = 1: an event pair around every launch (start, launch, stop).  on = 2: ONE event between consecutive launches -- a launch's
 * interval runs from its predecessor's stop event to its own, so the intervals tile the stream without gaps (whatever else the
 * caller enqueues between two dslash launches is charged to the later one) and cost half the event records; the first launch
 * after enabling or reading records its own start.  on = 0: off, the log is dropped. */
int tm_timing_enable(tm_ctx *ctx, int on);
int tm_timing_read(tm_ctx *ctx, int max_records, const char **names, float *ms, int *n);
/* Force a code path: 0 = automatic (default), 1 = generic direct-load kernels only.  For tests / profiling. */
int tm_set_path(tm_ctx *ctx, int path);
/* Performance knobs (never change results).  key is a HOST C string:
 *   "prefetch_blocks": L2 prefetch distance of the dslash kernels in thread blocks, 0 = off, -1 = library
 *   default (chosen per precision and flavor count);
 *   "stage_links": 1 = the 8 links of a site are copied to shared memory with cp.async before the hops, 0 = direct
 *   loads, -1 = library default;   "block_threads": 32 / 64 / 128 sites per thread block, 0 = library default;
 *   "z_chunks": the thread blocks walk the lattice in n chunks of Z / n z-planes (all time slices of a chunk first) so that
 *   the input spinor's reuse window fits the L2; -1 = library default (from the size of three time slices);
 *   "pdl": 1 (default) = the fused kernels are launched with the programmatic-stream-serialization attribute (each waits with
 *   griddepcontrol.wait for its predecessor before touching a field; hides the launch gap, 1 % of a 20-launch step), 0 = plain launches;
 *   "tile_kernel": half precision, 18- / 12-real links: 0 = thread-per-site kernels only, 1 or -1 (default) = the warp-per-tile
 *   kernel wherever the geometry fits (X/2 in {4, 8, 16}, Y a multiple of 64/X); both give bit-identical results.
 *   Unknown key or bad value -> TM_ERR_ARG. */
int tm_set_tuning(tm_ctx *ctx, const char *key, int value);

#ifdef __cplusplus
}
#endif
#endif /* TM_H */
