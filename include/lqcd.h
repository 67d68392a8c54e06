/* lqcd.h -- C ABI of the B200-native Wilson-clover library (liblqcd_b200.so).
 *
 * The library computes what the solvers of arXiv:1109.2935 ("Scaling Lattice QCD beyond
 * 100 GPUs", Babich et al., SC11) spend their time in.  Citations are lines of the paper
 * text plus section / equation; "R<n>" are the readings listed in DESIGN.md
 * for points on which the paper is silent.
 *
 *   problem           M x = b                                    PAPER.md:88-92  Sec. 2.1 Eq. 1
 *   operator          M = A(kappa) - kappa D,  A = 1 + kappa T   PAPER.md:98-108 Sec. 2.2 Eq. 2 (R1-R4)
 *   even-odd          Mhat = A_pp - kappa^2 D A^-1 D             PAPER.md:128    Sec. 3.1     (R6)
 *   solvers           mixed-precision BiCGstab, CGNR, CGNE
 *                     GCR-DD (Algorithm 1) + additive Schwarz/MR PAPER.md:146, :248-292 Sec. 8.1
 *   improved staggered D, M^dag M + sigma, multi-shift CG         PAPER.md:114-134, :296 (lqcd_staggered_*)
 *
 * Conventions
 *   - Unless a function says "host", every field pointer is a DEVICE pointer owned by the
 *     caller (e.g. a PyTorch tensor).  The library never frees or reallocates caller memory.
 *     The library owns the context, its packed gauge / clover copies and solver workspace;
 *     lqcd_destroy frees them.
 *   - `stream` is a cudaStream_t passed as void* (0 = legacy default stream).  Calls are
 *     stream-ordered and asynchronous, except lqcd_invert and the *_host calls, which
 *     synchronise the stream before returning.
 *   - Every function returns 0 (LQCD_OK) or a negative error code; nothing is printed, no
 *     exception crosses the ABI, nothing aborts.  lqcd_last_error gives the text.
 *   - A context is used from one host thread at a time.
 *
 * Canonical (external) layouts, C-contiguous complex128 (interleaved re, im):
 *   gauge   U[mu][t][z][y][x][row][col]  mu = 0:x 1:y 2:z 3:t.  U_mu(x) multiplies psi(x+mu)
 *           in Eq. 2.  Links carry NO boundary signs.
 *   spinor  psi[t][z][y][x][spin][colour]   DeGrand-Rossi chiral gamma basis (R2):
 *           gamma5 = diag(1,1,-1,-1).
 * Packed (internal) layouts are private: even-odd checkerboarded structure-of-arrays, one
 * parity per field; their size is queried with lqcd_field_bytes.  A packed field of one
 * precision is only meaningful to calls with the same `prec`.
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx;

/* error codes */
#define LQCD_OK          0
#define LQCD_EINVAL     (-1)   /* bad argument: null pointer, odd extent, bad enum, block not dividing dims */
#define LQCD_ESTATE     (-2)   /* call order: dslash before load_gauge, matpc before build_clover, c_sw mismatch */
#define LQCD_ENOMEM     (-3)
#define LQCD_ECUDA      (-4)   /* a CUDA call failed; text in lqcd_last_error */
#define LQCD_ENOCONV    (-5)   /* max_iter reached */
#define LQCD_EBREAKDOWN (-6)   /* BiCGstab rho/omega breakdown or NaN */

/* storage precisions.  HALF = int16 fixed point with one fp32 norm per site
 * (PAPER.md:164 (c): "custom 16-bit fixed-point storage format"; R9); arithmetic in fp32. */
#define LQCD_PREC_DOUBLE 0
#define LQCD_PREC_SINGLE 1
#define LQCD_PREC_HALF   2

/* gauge-link compression (PAPER.md:164 (a): 18 -> 12 or 8 reals per link) */
#define LQCD_RECON_18 18
#define LQCD_RECON_12 12
#define LQCD_RECON_8   8

#define LQCD_SOLVER_BICGSTAB 0
#define LQCD_SOLVER_GCR_DD   1
#define LQCD_SOLVER_CGNR     2   /* CG on Mhat^dag Mhat x = Mhat^dag bhat, mixed precision, reliable updates */
#define LQCD_SOLVER_CGNE     3   /* Craig's method: CG on Mhat Mhat^dag y = bhat, x = Mhat^dag y */

#define LQCD_MATPC_ASYMMETRIC 0
#define LQCD_MATPC_SYMMETRIC  1

#define LQCD_SCHWARZ_ADDITIVE       0
#define LQCD_SCHWARZ_MULTIPLICATIVE 1

#define LQCD_FIELD_SPINOR_PARITY 0
#define LQCD_FIELD_STAGGERED_PARITY 1   /* 3-component colour vectors of one parity (fp64 / fp32 only) */

/* Create a context for a lattice dims = (X,Y,Z,T), all even and >= 2, with per-direction
 * boundary condition boundary[mu] = +1 periodic / -1 antiperiodic (R5).  `device` is the
 * CUDA device ordinal.  Host pointers. */
int lqcd_create(lqcd_ctx** ctx, const int dims[4], const int boundary[4], int device);
int lqcd_destroy(lqcd_ctx* ctx);
const char* lqcd_last_error(const lqcd_ctx* ctx);
/* Solver and host-pipeline workspace is cached in the context between calls (allocating ~1 GB per solve costs
 * milliseconds); this frees the cache (lqcd_destroy does it too).  Synchronises the device. */
int lqcd_release_workspace(lqcd_ctx* ctx);

/* Load the gauge field (canonical layout, device pointer, 4*V*9 complex128).  Packs the
 * checkerboarded fp64 / recon-18 copy immediately; other precision x compression copies are
 * derived from it on first use.  Invalidates a previously built clover term. */
int lqcd_load_gauge(lqcd_ctx* ctx, const void* U_canonical, void* stream);

/* Build the clover term T_x = c_sw * sum_{mu<nu} (i sigma_munu) (x) F_munu(x) with the
 * four-leaf field strength (fn.1 :138; R4), kappa-independent, stored as
 * two Hermitian 6x6 chiral blocks = 72 reals per site. */
int lqcd_build_clover(lqcd_ctx* ctx, double c_sw, void* stream);

/* Bytes of one packed field of `kind` in precision `prec`. */
size_t lqcd_field_bytes(const lqcd_ctx* ctx, int kind, int prec);

/* canonical (full lattice, complex128) <-> packed (one parity, `prec`).  pack reads only the
 * sites of `parity`; unpack writes only those sites and leaves the others untouched. */
int lqcd_pack_spinor(lqcd_ctx* ctx, void* packed, const void* canonical, int parity, int prec, void* stream);
int lqcd_unpack_spinor(lqcd_ctx* ctx, void* canonical, const void* packed, int parity, int prec, void* stream);

/* out_p = D_{p,pbar} in_pbar : the hopping term of Eq. 2, no kappa, no
 * clover; `in` is a packed field of parity 1-parity_out, `out` of parity parity_out;
 * dagger != 0 applies D^dagger.  Nominal 1320 flop per output site.  out must not alias in. */
int lqcd_dslash(lqcd_ctx* ctx, void* out, const void* in, int parity_out, int dagger,
                int prec, int recon, void* stream);

/* out = A in (inverse == 0) or A^-1 in, A = 1 + kappa T on sites of `parity`.  504 flop/site. */
int lqcd_clover(lqcd_ctx* ctx, void* out, const void* in, int parity, int inverse,
                double kappa, int prec, void* stream);

/* out = Mhat in on `parity` (R6): two fused launches
 *   tmp = A^-1_{pbar pbar} D_{pbar p} in ;  out = A_pp in - kappa^2 D_{p pbar} tmp.
 * 3696 flop per site.  out must not alias in. */
int lqcd_matpc(lqcd_ctx* ctx, void* out, const void* in, int parity, int dagger,
               double kappa, int prec, int recon, void* stream);

/* Symmetric even-odd form (SURVEY.md 8(c).5 "Optional"; same Schur complement, reference [11] of the
 * paper, left-multiplied by A_pp^-1):  out = Mhat_s in,  Mhat_s = 1 - kappa^2 A_pp^-1 D A_pbar^-1 D = A_pp^-1 Mhat;
 * dagger != 0 applies Mhat_s^dag = 1 - kappa^2 D^dag A^-1 D^dag A^-1.  Same bytes and flops as lqcd_matpc. */
int lqcd_matpc_sym(lqcd_ctx* ctx, void* out, const void* in, int parity, int dagger,
                   double kappa, int prec, int recon, void* stream);

/* Multi-right-hand-side forms (not in the paper): the same operators applied
 * to nrhs (1..LQCD_MAX_RHS) packed fields that share the gauge field, in one launch per Dslash.
 * `in` and `out` hold the nrhs packed fields of precision `prec` back to back (field r starts at
 * r * lqcd_field_bytes).  A link is loaded, decoded and reconstructed once per CTA for 4
 * right-hand sides: 2/3 of the compulsory bytes of a single-source fp32/recon-12 Dslash are links.
 * Same results as nrhs single calls (same arithmetic per site).  Errors as lqcd_dslash, plus
 * LQCD_EINVAL for nrhs out of range. */
#define LQCD_MAX_RHS 64
int lqcd_dslash_mrhs(lqcd_ctx* ctx, void* out, const void* in, int nrhs, int parity_out, int dagger,
                     int prec, int recon, void* stream);
int lqcd_matpc_mrhs(lqcd_ctx* ctx, void* out, const void* in, int nrhs, int parity, int dagger,
                    double kappa, int prec, int recon, void* stream);

/* Schwarz preconditioner K (R7): out = K in on `parity`, n_mr
 * minimum-residual steps on the Dirichlet-cut Mhat_D with one alpha per block.  in/out are
 * packed fields (natural layout) of precision `prec_io`; the MR iteration itself runs in
 * `prec` on block-major copies. */
int lqcd_schwarz(lqcd_ctx* ctx, void* out, const void* in, int parity, double kappa,
                 const int block[4], int n_mr, double omega_mr, int prec, int recon,
                 int prec_io, void* stream);

/* Multiplicative Schwarz (SAP: section 4, ref. [20]; named as the alternative to the additive form in
 * PAPER.md:146; reading R16): blocks coloured (bx+by+bz+bt) mod 2, n_cycle cycles, in each cycle for colour 0 then 1:
 * n_mr MR steps on the blocks of that colour applied to the current residual, out += y, residual -= Mhat y with the
 * FULL operator (precision prec_io, links recon_io).  Needs an even number of blocks in x (LQCD_EINVAL otherwise).
 * in / out: packed fields of precision prec_io, natural layout; the block solves run in `prec` / `recon`. */
int lqcd_schwarz_sap(lqcd_ctx* ctx, void* out, const void* in, int parity, double kappa,
                     const int block[4], int n_mr, double omega_mr, int n_cycle, int prec, int recon,
                     int prec_io, int recon_io, void* stream);

/* Blocks per launch group for later lqcd_schwarz calls on this context (lqcd_invert takes it from
 * lqcd_invert_params::schwarz_group); 0 = all blocks per launch.  LQCD_EINVAL if negative. */
int lqcd_set_schwarz_group(lqcd_ctx* ctx, int blocks_per_group);

/* Overlapping Schwarz domains for later lqcd_schwarz calls on this context (lqcd_invert takes the value from
 * lqcd_invert_params::schwarz_overlap).  PAPER.md:146 ("blocks which may or may not overlap ... a tunable parameter"),
 * :338; reading R18: restricted additive Schwarz -- the domain of a block is its box grown by `overlap` sites
 * on both sides of every partitioned direction (through the lattice's periodic wrap), the MR steps run on the domain
 * with Dirichlet boundaries, and the result is kept on the block's own box.  0 = non-overlapping (default, the paper's
 * runs).  LQCD_EINVAL at the next Schwarz call if a grown domain would reach around the lattice (block + 2 overlap >=
 * extent) or if overlap x number of partitioned directions is odd; the multiplicative variant takes no overlap.  The
 * block-major copies of links, clover blocks and work vectors grow by the volume ratio of grown domain to block. */
int lqcd_set_schwarz_overlap(lqcd_ctx* ctx, int overlap);

typedef struct {
  double kappa;
  double c_sw;            /* must equal the value given to lqcd_build_clover */
  double tol;             /* stop on ||b - M x|| <= tol * ||b||  (full system) */
  double delta;           /* BiCGstab: reliable-update trigger; GCR: early restart (Alg. 1) */
  int    max_iter;
  int    solver;          /* LQCD_SOLVER_* */
  int    prec_outer, prec_sloppy, prec_precond;
  int    recon_outer, recon_sloppy, recon_precond;
  int    parity;          /* parity on which the Schur system is solved */
  int    gcr_kmax;        /* restart length (16) */
  int    schwarz_block[4];/* e.g. 12,12,12,24; extents even, dividing dims */
  int    mr_steps;        /* 10 */
  double mr_omega;        /* 1.0 */
  int    use_initial_guess;
  int    precondition;    /* GCR: 1 = Schwarz/MR preconditioner, 0 = plain GCR */
  int    matpc_type;      /* LQCD_MATPC_ASYMMETRIC (default, R6) or LQCD_MATPC_SYMMETRIC: the Krylov iteration runs on
                             Mhat_s x_p = A_pp^-1 bhat; the stopping test stays ||b - M x|| <= tol ||b|| (fp64, at
                             reliable updates).  BiCGstab, CGNR and CGNE only. */
  int    schwarz_group;   /* GCR-DD: blocks per launch group of the preconditioner; all mr_steps run on one group before
                             the next is touched, so that a group sized to the L2 (about 5 blocks of 12^3x24 in half) keeps
                             its links, clover blocks and vectors on chip.  0 = all blocks
                             in one launch per step.  Results do not depend on it (blocks are independent). */
  int    schwarz_type;    /* LQCD_SCHWARZ_ADDITIVE (default) or LQCD_SCHWARZ_MULTIPLICATIVE (lqcd_schwarz_sap) */
  int    sap_cycles;      /* multiplicative: cycles over the two colours per preconditioner application (0 -> 1) */
  int    history_len;     /* capacity of residual_history in doubles (0 = none) */
  double* residual_history; /* optional HOST buffer (caller-owned): entry k = iterated residual norm / ||b|| after
                             iteration k+1 of the low-precision iteration (BiCGstab, CGNR, CGNE) or after outer iteration
                             k+1 (GCR); lqcd_invert_result::history_count entries are written.  Reported, never
                             asserted (convergence history is "parity unpinned"). */
  int    schwarz_overlap; /* GCR-DD, additive: sites by which every Schwarz domain is grown on both sides of each partitioned
                             direction (lqcd_set_schwarz_overlap; 0 = the paper's non-overlapping blocks) */
} lqcd_invert_params;

typedef struct {
  int    status;          /* LQCD_OK, LQCD_ENOCONV, LQCD_EBREAKDOWN */
  int    iterations;      /* BiCGstab / CGNR iterations, GCR outer iterations */
  int    restarts;        /* reliable updates (BiCGstab) or restarts (GCR) */
  int    matpc_sloppy, matpc_outer, matpc_precond;   /* operator applications by precision */
  double true_residual;   /* ||bhat - Mhat x_p|| / ||b|| in fp64 = ||b - M x|| / ||b|| */
  double iterated_residual;
  double seconds;         /* device time of the whole call (CUDA events) */
  double gflop;           /* nominal flops executed (operators 3696/site + BLAS-1) / 1e9 */
  int    history_count;   /* entries written to lqcd_invert_params::residual_history */
} lqcd_invert_result;

/* Solve M x = b on the full lattice (Eq. 1): source preparation, parity solve of the Schur
 * system, reconstruction of the other parity.  x and b are canonical full-lattice DEVICE
 * arrays.  Synchronises `stream`. */
int lqcd_invert(lqcd_ctx* ctx, void* x_canonical, const void* b_canonical,
                const lqcd_invert_params* params, lqcd_invert_result* result, void* stream);

/* Batched solve of M x_r = b_r for nrhs (1..LQCD_MAX_RHS) sources sharing the gauge field: nrhs mixed-
 * precision BiCGstab recurrences in lockstep on the multi-right-hand-side operators (SURVEY.md 8(f)
 * NEXT-4; not in the paper).  x_canonical / b_canonical: nrhs canonical full-lattice DEVICE arrays back
 * to back; result[r] describes source r (seconds and gflop are those of the whole batch).  Every
 * source is iterated to its own ||b_r - M x_r|| <= tol ||b_r||.  params: solver must be
 * LQCD_SOLVER_BICGSTAB, matpc_type LQCD_MATPC_ASYMMETRIC.  Returns LQCD_OK, or LQCD_ENOCONV /
 * LQCD_EBREAKDOWN if at least one source ended that way (see result[r].status).  Synchronises `stream`. */
int lqcd_invert_mrhs(lqcd_ctx* ctx, void* x_canonical, const void* b_canonical, int nrhs,
                     const lqcd_invert_params* params, lqcd_invert_result* result, void* stream);

/* ---- improved staggered (asqtad) path: PAPER.md:114-122 Sec. 2.3 Eq. 3, :130-134 Eq. 4, :296 Sec. 8.2;
 * SURVEY.md 8(f) NEXT-3; readings R13-R15 of DESIGN.md ------------------------------------------------
 *   (D chi)(x) = sum_mu eta_mu(x) [ fat_mu(x) chi(x+mu) - fat_mu(x-mu)^dag chi(x-mu)
 *                                 + lng_mu(x) chi(x+3mu) - lng_mu(x-3mu)^dag chi(x-3mu) ],   M = -D/2 + m,
 *   eta_x = 1, eta_y = (-1)^x, eta_z = (-1)^(x+y), eta_t = (-1)^(x+y+z); boundary sign on hops that wrap.
 * Canonical layouts (device, complex128): fat / lng [mu][t][z][y][x][3][3], general 3x3 (the fat links
 * are not unitary; path coefficients are part of the links; NO phases, NO boundary signs);
 * colour vectors chi[t][z][y][x][3].  Packed fields: lqcd_field_bytes(LQCD_FIELD_STAGGERED_PARITY),
 * precisions LQCD_PREC_DOUBLE and LQCD_PREC_SINGLE (half is "not amenable", PAPER.md:298 fn. 3).
 * Every extent must be >= 4 (three-hop term).  Errors as for the Wilson-clover calls. */
/* long_scale != 0 declares every long link to be long_scale x SU(3) (the three-link Naik term of asqtad is
 * c3 x a product of three SU(3) links): the library verifies it (LQCD_EINVAL otherwise) and stores 12 reals per
 * long link, third row = conj(row0 x row1) / long_scale (PAPER.md:164 (a)); long_scale = 0: general 3x3, 18 reals. */
int lqcd_load_staggered_links(lqcd_ctx* ctx, const void* fat_canonical, const void* lng_canonical, double long_scale,
                              void* stream);
int lqcd_pack_staggered(lqcd_ctx* ctx, void* packed, const void* canonical, int parity, int prec, void* stream);
int lqcd_unpack_staggered(lqcd_ctx* ctx, void* canonical, const void* packed, int parity, int prec, void* stream);
/* out_p = D_{p,pbar} in_pbar: 16 hops, 1146 flop per site.  out must not alias in. */
int lqcd_staggered_dslash(lqcd_ctx* ctx, void* out, const void* in, int parity_out, int prec, void* stream);
/* out = (M^dag M + sigma) in on `parity` = (m^2 + sigma) in - D_{p,pbar} D_{pbar,p} in / 4: two launches. */
int lqcd_staggered_mdagm(lqcd_ctx* ctx, void* out, const void* in, int parity, double mass, double sigma,
                         int prec, void* stream);

/* Solve (M^dag M + sigma_i) x_i = b on `parity` for nshift (1..32) shifts 0 <= sigma_0 < sigma_1 < ... (Eq. 4,
 * PAPER.md:130-134) with the paper's strategy: a pure single-precision multi-shift CG for all
 * shifts at once, then sequential mixed-precision CG (fp64 outer with reliable updates, fp32 inner) refining
 * every x_i until ||b - (M^dag M + sigma_i) x_i|| <= tol ||b|| in fp64.  b_canonical: chi-shaped DEVICE array
 * (only the sites of `parity` are read); x_canonical: nshift such arrays back to back (sites of the other
 * parity are set to zero).  result[i]: iterations / restarts / matpc_sloppy / matpc_outer of shift i's
 * refinement, true_residual; result[0].matpc_precond = iterations of the multi-shift phase; seconds and gflop
 * are those of the whole call.  max_iter bounds each phase.  multishift_prec: LQCD_PREC_SINGLE = the paper's
 * strategy; LQCD_PREC_DOUBLE = the multi-shift phase itself in fp64 down to tol (what PAPER.md:294-296 rules out
 * for memory and fp64 rate on 2011 GPUs; on B200 it is the faster of the two); the refinement
 * then only confirms.  Synchronises `stream`. */
int lqcd_staggered_multishift(lqcd_ctx* ctx, void* x_canonical, const void* b_canonical, int parity, double mass,
                              const double* sigma, int nshift, double tol, int max_iter, int multishift_prec,
                              lqcd_invert_result* result, void* stream);

/* ---- host-buffer entry points (end-to-end path: host<->device copies inside the call) ---- */
/* out_host/in_host: canonical full-lattice complex128 HOST arrays (pinned for full PCIe speed;
 * pageable works), owned by the caller, not overlapping.
 * out = D in on both parities (op == 0) or out_p = Mhat in_p on `parity`, rest zero (op == 1),
 * computed in (prec, recon).  The call pipelines host->device copy, pack, operator, unpack and
 * device->host copy over slabs of time slices on two internal copy streams plus `stream`
 * (staging buffers are cached in the context); it starts after the work already queued on
 * `stream` and returns after everything, including the copy back, has completed.
 * Errors: LQCD_EINVAL (null pointer, bad op/parity/prec/recon), LQCD_ESTATE (no gauge / clover),
 * LQCD_ENOMEM, LQCD_ECUDA. */
int lqcd_apply_host(lqcd_ctx* ctx, void* out_host, const void* in_host, int op, int parity, int dagger,
                    double kappa, int prec, int recon, void* stream);
/* The same call with complex64 canonical HOST arrays (half the PCIe bytes; the path is PCIe-bound): for fp32 and
 * half-precision compute only (prec == LQCD_PREC_DOUBLE -> LQCD_EINVAL), whose storage holds no more digits. */
int lqcd_apply_host_c64(lqcd_ctx* ctx, void* out_host, const void* in_host, int op, int parity, int dagger,
                        double kappa, int prec, int recon, void* stream);
int lqcd_invert_host(lqcd_ctx* ctx, void* x_host, const void* b_host,
                     const lqcd_invert_params* params, lqcd_invert_result* result, void* stream);

/* ---- fused BLAS-1 on packed fields, exported for tests and the bench ---- */
/* y += a*x ; returns ||y||^2 in *norm2_host after a stream sync (host pointer). */
int lqcd_axpy_norm(lqcd_ctx* ctx, double a, const void* x, void* y, int prec, double* norm2_host, void* stream);
/* <x,y> = sum conj(x) y -> dot_host[0..1] (re, im). */
int lqcd_cdot(lqcd_ctx* ctx, const void* x, const void* y, int prec, double* dot_host, void* stream);

/* <x,y> and ||y||^2 WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (stream capture into a CUDA
 * graph, serving loops, harnesses that forbid it).  Same sums as lqcd_cdot (the reductions of the
 * Krylov solvers).  x, y: packed parity fields of precision prec (DEVICE).  out_device: 3 doubles in DEVICE memory
 * owned by the caller, written on `stream`: re <x,y>, im <x,y>, ||y||^2; no copy to the host and no stream sync.
 * The per-CTA partial sums live in a 768 KiB file-scope __device__ array of the library (held by every GPU that
 * loads it until the process exits), which bounds the field: at most 2^23 = 8,388,608 sites per parity field, else
 * LQCD_EINVAL with the limit in lqcd_last_error.  The call issues two kernel launches and no cudaMalloc / cudaFree /
 * memcpy / event; the first call on a device also looks up the array's address (cudaGetSymbolAddress; make that call
 * outside stream capture).  All calls on a device share the array: calls ordered on one stream are safe, calls that
 * overlap on the GPU (two streams, two threads) race.  Sums are added in a fixed order (bit-reproducible). */
int lqcd_cdot_static(lqcd_ctx* ctx, const void* x, const void* y, int prec, double* out_device, void* stream);

/* number of kernel launches issued by this context since creation (bench: gpu_launches) */
long long lqcd_launch_count(const lqcd_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
