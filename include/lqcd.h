/*
 * lqcd.h -- C ABI of the B200-native Wilson dslash library (liblqcd.so).
 *
 * The hot path of "LatticeQCD using OpenCL" (arXiv:1112.5280): the Wilson hopping
 * operator ("the non-diagonal part of the Dirac matrix ('dslash')", sec. 3),
 * in full and even-odd preconditioned form (Fig. 5 caption), and the
 * fermion matrix M built on it ("M is the fermion matrix", sec. 4).
 * The paper prints no formula; the definition is the textbook Wilson form fixed in
 * SURVEY.md sec. 8(c) / Appendix A and restated in DESIGN.md:
 *
 *   (H psi)(x) = sum_{mu=0..3} [ (1 - gamma_mu) U_mu(x)         psi(x + mu^)
 *                              + (1 + gamma_mu) U_mu(x - mu^)^+  psi(x - mu^) ]
 *   M_full = 1 - kappa H ;   M_eo = 1 - kappa^2 H_eo H_oe  on even sites
 *   psi(x + L_mu mu^) = bc_mu psi(x),  |bc_mu| = 1   (phase applied at the crossing hop only)
 *
 * mu = 0,1,2,3 = x,y,z,t; parity p(x) = (x+y+z+t) & 1; chiral gamma basis of DESIGN.md.
 *
 * General rules for every entry point
 *   - Pointers named *_dev are CUDA device pointers, *_host are host pointers.  The caller
 *     (PyTorch) allocates and frees every buffer; the library allocates no field memory and
 *     keeps no pointer after a call returns.  lqcd_ctx is host memory owned by the library.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     entry points only enqueue work and return; they never synchronise.  The *_host entry points
 *     and the CG solvers synchronise `stream` before returning (their results live in host memory).
 *   - Native device fields (spinors, links, workspaces) are accessed with 256-bit words and must be 32-byte
 *     aligned for every precision; canonical device buffers 16-byte aligned; the solver and host-path
 *     workspaces 256-byte aligned.  A misaligned pointer returns LQCD_EALIGN before anything is launched.
 *   - The stencil is not in-place safe: `out` overlapping `in` / `workspace` gives LQCD_EALIAS.
 *   - Errors are return codes only: nothing throws, aborts or prints.
 *
 * Layouts (element type = float for precision 32, double for precision 64)
 *   canonical (interchange; complex interleaved re,im; C-contiguous; what torch.complex64/128 holds)
 *     full spinor  [T][Z][Y][X][spin 4][colour 3]
 *     half spinor  [V/2][spin 4][colour 3]  -- the sites of one parity in increasing
 *                  lexicographic order lex = x + X(y + Y(z + Z t)), i.e. indexed by cb = lex >> 1
 *     links        [mu 4][T][Z][Y][X][row 3][col 3],  (U psi)_a = sum_b U[a][b] psi_b,  U_mu(x) at x
 *   native (what the hot path reads/writes; array of structures of arrays, checkerboarded, warp tiles)
 *     Sites of one parity are numbered by cb and grouped in tiles of 32 consecutive cb;
 *     ntiles = ceil(V/2 / 32), the last tile is padded (padding is never read or written).
 *     real component r = 6 spin + 2 colour + reim (spinor, 24) or 6 row + 2 col + reim (link,
 *     first `recon` reals of 18).  W = 32 bytes / sizeof(element) reals per 256-bit spinor word.
 *     half spinor  word q = r / W, lane = r % W  at element ((cb/32 * 24/W + q) * 32 + cb%32) * W + lane
 *     full spinor  [even half | odd half], each of lqcd_spinor_bytes(ctx, 1) bytes
 *     precision 16: a half spinor is 3 16-byte words of 8 halfs per site, [tile][word 3][32], holding v / n(x),
 *                  n(x) = max |component|, followed by the fp32 norms n(x), float[32 ntiles]; links are 3 8-byte words
 *                  of 4 halfs, [parity][tile][hop 8][word 3][32] (52 bytes per spinor site, 24 per link)
 *     links        gathered by output site: [parity p of x][tile][hop k 8][word][32][lane], hop k = 2 mu holds
 *                  U_mu(x), k = 2 mu + 1 holds U_mu(x - mu^) (stored as is; the kernel takes the adjoint).
 *                  Words of 4 floats (precision 32 recon 12, 3 words), 2 floats (precision 32 recon 18, 9 words),
 *                  4 doubles (precision 64 recon 12, 3 words) or 2 doubles (precision 64 recon 18, 9 words); recon 8: 2
                  words of 4 reals (Re U01, Im U01, Re U02, Im U02 | Re U10, Im U10, arg U00 / pi, arg U20 / pi).
                  Every link is stored twice (capacity for contiguity: all
 *                  8 links of a warp's 32 sites form one contiguous block); one application of
 *                  lqcd_dslash_eo still reads 8 links per output site exactly once.
 */
#ifndef LQCD_H
#define LQCD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx; /* opaque: geometry + constants, host memory */

typedef enum {
    LQCD_OK = 0,
    LQCD_EINVAL = 1,       /* null pointer, bad extent / parity / precision / recon, |bc| != 1 */
    LQCD_EALIGN = 2,       /* a device pointer is misaligned: native 32 B, canonical 16 B, big workspaces 256 B */
    LQCD_EALIAS = 3,       /* out overlaps in or workspace */
    LQCD_EUNSUPPORTED = 4, /* combination not compiled in */
    LQCD_ECUDA = 5,        /* CUDA runtime / launch error */
    LQCD_ETOOBIG = 6       /* lqcd_apply_M_eo_static only: the lattice needs more than LQCD_STATIC_SCRATCH_BYTES */
} lqcd_status;

typedef struct {
    int dims[4];      /* X,Y,Z,T (mu = 0..3); each even and >= 4 (reading A17) */
    int precision;    /* 64 or 32: storage and arithmetic type of all fields; 16: fields stored as IEEE half
                         (spinors normalised per site, with an fp32 norm), fp32 arithmetic, recon 12 only;
                         canonical buffers are complex64; the CG iterates in fp32 on 16-bit operator fields */
    int recon;        /* 18, 12 or 8: stored reals per link; 12 = two rows, third rebuilt in
                         registers as conj(row0 x row1) ("RECONSTRUCT TWELVE"); 8 = the minimal
                         parametrisation of ref. [3]: U01, U02, U10 and the phases of U00, U20,
                         the rest rebuilt in registers from unitarity and det = 1 (precision 32 / 64 only).
                         Singular where |U00| = 1: unit links cannot be stored with recon 8, and a link loses
                         digits like eps / min(|U00|, sqrt(1 - |U00|^2), |U20|) -- see lqcd_gauge_recon8_margin.
                         lqcd_pack_gauge refuses a field with a link whose margin is below 64 eps (LQCD_EUNSUPPORTED) */
    double bc_re[4];  /* boundary phase bc_mu = bc_re + i bc_im, |bc_mu| = 1 within 1e-12; */
    double bc_im[4];  /* periodic (1,0), antiperiodic (-1,0), any U(1) phase allowed        */
    int link_precision; /* 0: links stored like the spinors.  16 with precision 32 and recon 12: fp32 spinors,
                           links stored as 12 IEEE halfs (24 instead of 48 bytes per link; the link stream is 2/3 of
                           the traffic) -- meant for the inner solver of lqcd_cg_solve_tm_mixed */
} lqcd_params;

#define LQCD_PARITY_EVEN 0
#define LQCD_PARITY_ODD 1
#define LQCD_PARITY_BOTH (-1)

/* Validate p, copy it; *ctx is set on LQCD_OK only. */
lqcd_status lqcd_create(lqcd_ctx** ctx, const lqcd_params* p);
lqcd_status lqcd_destroy(lqcd_ctx* ctx); /* NULL is a no-op */

/* Sizes in bytes of native buffers for this ctx (0 if ctx is NULL). */
size_t lqcd_spinor_bytes(const lqcd_ctx* ctx, int half); /* half != 0: one parity; 0: full [even|odd] */
size_t lqcd_gauge_bytes(const lqcd_ctx* ctx);            /* native links, 2*8*recon*32*ntiles elements */
size_t lqcd_workspace_bytes(const lqcd_ctx* ctx);        /* lqcd_apply_M(eo=1): one native half spinor */
size_t lqcd_host_workspace_bytes(const lqcd_ctx* ctx);   /* device scratch of lqcd_dslash_eo_host */

/* canonical <-> native conversion kernels (layout only, no arithmetic; not on the timed path).
 * All pointers are device pointers; asynchronous on `stream`.
 * parity = LQCD_PARITY_EVEN/ODD: canonical half spinor <-> native half spinor;
 * parity = LQCD_PARITY_BOTH:     canonical full spinor <-> native full spinor [even|odd]. */
/* recon 8 only: lqcd_pack_gauge / lqcd_pack_gauge_slab also check every link against the encoding's singular set (unit
 * links, |U00| = 1, U00 = 0 or U20 = 0: the decoder would divide by zero and the dslash would return NaN) and, for that,
 * synchronise `stream` before returning: LQCD_EUNSUPPORTED if a link's margin (lqcd_gauge_recon8_margin) is below
 * 64 eps of the precision, or is NaN; the native buffer is then not usable.  Store such a field with recon 12. */
lqcd_status lqcd_pack_gauge(const lqcd_ctx* ctx, void* native_dev, const void* canonical_dev, void* stream);
lqcd_status lqcd_pack_spinor(const lqcd_ctx* ctx, void* native_dev, const void* canonical_dev, int parity,
                             void* stream);
lqcd_status lqcd_unpack_spinor(const lqcd_ctx* ctx, void* canonical_dev, const void* native_dev, int parity,
                               void* stream);

/* min over all links of min(|U00|, sqrt(|U01|^2 + |U02|^2), |U20|) for a canonical link field on the device: the
 * moduli the 8-real decoder obtains from differences and divides by.  0 means the field cannot be stored with
 * recon 8 (e.g. unit links); otherwise the worst link is accurate to about eps / margin.  scratch_dev: 8 bytes of
 * device memory, 8-byte aligned.  Synchronises `stream`; *margin_host is host memory. */
lqcd_status lqcd_gauge_recon8_margin(const lqcd_ctx* ctx, const void* canonical_dev, void* scratch_dev,
                                     double* margin_host, void* stream);

/* ---- hot path: device pointers, native layout ---- */

/* out = H in on all sites; in/out native full spinors.  One launch. */
lqcd_status lqcd_dslash_full(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                             void* stream);

/* out_p = H_{p,1-p} in_{1-p}: in is a native half spinor of parity 1-out_parity, out one of parity
 * out_parity (0: H_eo, odd in -> even out; 1: H_oe).  One launch.  No kappa (pure H, so the
 * 1320 flop/site convention is exact; reading A7). */
lqcd_status lqcd_dslash_eo(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                           int out_parity, void* stream);

/* ---- time-slab decomposition over several GPUs (next row f3; the paper's multi-device story is host-mediated,
 * PAPER.md:71, :103; T slabs, projected half-spinor faces between ring neighbours) ----
 * A rank owns T_loc consecutive global time slices (T_loc even, so local and global parities agree) as a local lattice
 * X,Y,Z,T_loc: a ctx created with those extents, then lqcd_set_time_slab.  One application of H on a slab:
 *   1. lqcd_slab_push_faces   projects the first and the last time slice of `in` to half spinors (12 reals per site:
 *                             (1 - gamma_t) psi for the rank below, (1 + gamma_t) psi for the rank above) and stores
 *                             them into dst_down / dst_up -- the NEIGHBOURS' halo buffers mapped over NVLink peer memory
 *                             (the transfer is the kernel's own stores), or local send buffers for ncclSend/ncclRecv
 *   2. lqcd_dslash_eo_range   on the interior slices [1, T_loc - 1): needs no halo, overlaps the transfer
 *   3. lqcd_dslash_eo_slab    on slices 0 and T_loc - 1: the t hops that leave the slab read halo_from_up / halo_from_down
 * Ordering between 1 (on the neighbour) and 3: either by the caller (stream events after a collective / P2P receive:
 * pass NULL flags), or on the device: push_faces publishes `epoch` with a system-scope release into the neighbours'
 * flags (8-byte counters in peer memory) after its stores, and the slab kernel spins (system-scope acquire, bounded to
 * ~10 s, then traps) until its own two flags have reached `epoch`.  Use a fresh, increasing epoch per application.
 * Halo buffer (lqcd_halo_bytes): [face tile][word][32] 16-byte words, 3 (precision 32) / 6 (precision 64) per site,
 * face site = checkerboard index within the time slice.  Precision 32 / 64 and every recon; not precision 16.
 * lqcd_set_time_slab moves the t boundary phase from the local wrap to where the global boundary cuts the slab: the
 * forward hop from slice t_cross_fwd and the backward hop from slice t_cross_bwd carry bc_t / conj(bc_t); -1 = none; a
 * whole lattice has (T - 1, 0).  lqcd_pack_gauge_slab packs the local links; the backward t link of the first slice,
 * U_t(x - t^), belongs to the rank below and is read from tlinks_below_dev, a canonical [Z][Y][X][3][3] array. */
lqcd_status lqcd_set_time_slab(lqcd_ctx* ctx, int t_cross_fwd, int t_cross_bwd);
lqcd_status lqcd_pack_gauge_slab(const lqcd_ctx* ctx, void* native_dev, const void* canonical_dev,
                                 const void* tlinks_below_dev, void* stream);
size_t lqcd_halo_bytes(const lqcd_ctx* ctx); /* one face; 0: no slab path for this ctx */
lqcd_status lqcd_slab_push_faces(const lqcd_ctx* ctx, const void* in_dev, void* dst_up_dev, void* dst_down_dev,
                                 void* flag_up_dev, void* flag_down_dev, unsigned long long epoch, void* stream);
lqcd_status lqcd_dslash_eo_range(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                                 int out_parity, int t_begin, int t_end, void* stream);
lqcd_status lqcd_dslash_eo_slab(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                                const void* halo_from_up_dev, const void* halo_from_down_dev, const void* wait_up_dev,
                                const void* wait_down_dev, unsigned long long epoch, int out_parity, int t_begin,
                                int t_end, void* stream);

/* eo = 0: out = in - kappa H in, native full spinors, one launch, workspace unused (may be NULL).
 * eo = 1: out_e = in_e - kappa^2 H_eo H_oe in_e, native even half spinors; two launches;
 *         workspace_dev holds the intermediate odd half spinor (lqcd_workspace_bytes). */
lqcd_status lqcd_apply_M(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                         double kappa, int eo, void* workspace_dev, void* stream);

/* ---- the even-odd fermion matrix for callers that cannot allocate device memory ----
 * lqcd_apply_M(eo = 1) needs a workspace, and by the rules above the caller provides it.  Some callers cannot: this
 * library is a plain C ABI, and a C or Fortran HMC driver that links it is typically handed three device pointers (links,
 * source, destination) by a host application whose own pool owns all of HBM -- it has no CUDA runtime binding to call
 * cudaMalloc with, and if it had one the call would fail (nothing is left outside the pool) or stall the device (cudaMalloc
 * and cudaFree synchronise).  The same holds for code that runs where allocation is forbidden by contract, such as the
 * inner loop of a solver that promised its caller a fixed memory footprint.
 *
 * For them: out_e = in_e - kappa^2 H_eo H_oe in_e exactly as lqcd_apply_M(ctx, out, gauge, in, kappa, 1, workspace, stream)
 * computes it (same two launches, same arithmetic, bit-identical result), with the intermediate odd half spinor kept in
 * an array inside the library image instead of a caller's workspace.  The call itself allocates and frees nothing, on the
 * host or on the device, and calls no library routine that does.
 *   Limit.     The array is LQCD_STATIC_SCRATCH_BYTES (16 MiB) and exists once per GPU: every GPU on which this library
 *              is used gives up that much memory from the moment the module is loaded until the process exits, called or
 *              not.  A lattice fits when lqcd_workspace_bytes(ctx) <= lqcd_static_scratch_bytes(): up to 16^3 x 32 in
 *              precision 64, 16^3 x 64 in precision 32.  A larger one returns LQCD_ETOOBIG before anything is launched;
 *              use lqcd_apply_M with a workspace of your own then.
 *   First call. The first call on each device looks up where that device keeps the array (cudaGetSymbolAddress, which
 *              may also make the runtime load the module); later calls on that device reuse the answer.  Make that first
 *              call with the device current, outside any stream capture, before the phase of your program in which
 *              allocation is off limits.
 *   Sharing.   All calls on one GPU -- from any context, thread or stream -- use the same array.  It needs no clearing:
 *              the first launch overwrites every site before the second reads it, so whatever an earlier call left there is
 *              harmless.  But two calls whose kernels can overlap on the GPU (different streams, different host threads
 *              without ordering between them) race on the intermediate field and both results are garbage; order them
 *              on one stream or with events.  The contents after a call are unspecified.
 * Pointers, alignment, aliasing and error codes as for lqcd_apply_M; in, out: native even half spinors. */
#define LQCD_STATIC_SCRATCH_BYTES ((size_t)16 << 20)
size_t lqcd_static_scratch_bytes(void);
lqcd_status lqcd_apply_M_eo_static(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                                   double kappa, void* stream);

/* Twisted-mass Wilson fermion matrix for one flavour ("N_f = 2 twisted-mass Wilson fermions",
 * "even-odd preconditioning"; the other flavour is mu -> -mu; reading F1):
 * eo = 0: out = (1 + 2 i kappa mu gamma_5) in - kappa H in, native full spinors, one launch.
 * eo = 1: out_e = (1 + 2 i kappa mu gamma_5) in_e - kappa^2 H_eo (1 + 2 i kappa mu gamma_5)^-1 H_oe in_e, the Schur
 *         complement on the even sites; native even half spinors; two launches; workspace as for lqcd_apply_M.
 * The site-diagonal term and its inverse are applied in the epilogues of the dslash launches (gamma_5 is
 * diagonal in the chiral basis), so the traffic is that of lqcd_apply_M.  mu = 0 gives lqcd_apply_M. */
lqcd_status lqcd_apply_M_tm(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                            double kappa, double mu, int eo, void* workspace_dev, void* stream);

/* Q(mu) = gamma_5 Mhat_tm(mu) on the even sites (even-odd form of lqcd_apply_M_tm with a final gamma_5):
 * Q(mu)^+ = Q(-mu), so Mhat(mu)^+ Mhat(mu) = Q(-mu) Q(mu).  Native even half spinors, two launches. */
lqcd_status lqcd_apply_Q_tm(const lqcd_ctx* ctx, void* out_dev, const void* gauge_dev, const void* in_dev,
                            double kappa, double mu, void* workspace_dev, void* stream);

/* Conjugate gradient ("the inversion of the fermion matrix"; reading F2): solves
 *     Mhat_tm(mu)^+ Mhat_tm(mu) x = b      on the even sites, x0 = 0,
 * textbook CG, stopping when the recursive residual satisfies |r| <= tol |b| or after maxiter iterations.
 * x_dev, b_dev: native even half spinors (b is not modified; x must not overlap b).  workspace_dev:
 * lqcd_cg_workspace_bytes(ctx) bytes of device scratch, 256-byte aligned.  All vector updates, reductions and
 * scalars (alpha, beta, <r,r>, the convergence flag) stay on the device; the host looks at the flag every 8
 * iterations (every iteration once |r|^2 is within 1000x of the target), and iterations enqueued after convergence
 * leave x untouched.  Reductions are deterministic.
 * The call synchronises `stream` before returning: *iters_out = iterations performed, *relres_out = |r| / |b|
 * of the recursive residual (host pointers, either may be NULL).  Arithmetic in the ctx precision.
 * Precision 16 (16-bit solver, PAPER.md:89 ref. [3]): x_dev and b_dev are 16-bit native half spinors; b is widened to fp32,
 * the iterate x and the residual r are kept in fp32 (their recurrences carry the accuracy), the search direction p, Q p
 * and A p live in the 16-bit format the operator reads and writes; x is rounded to the 16-bit format at the end.  The
 * recursive residual then drifts from the true one at the 1e-3 level: use it as the inner solver of
 * lqcd_cg_solve_tm_mixed, or with tol >= 1e-3. */
size_t lqcd_cg_workspace_bytes(const lqcd_ctx* ctx);
lqcd_status lqcd_cg_solve_tm(const lqcd_ctx* ctx, void* x_dev, const void* gauge_dev, const void* b_dev, double kappa,
                             double mu, double tol, int maxiter, void* workspace_dev, int* iters_out,
                             double* relres_out, void* stream);

/* Mixed-precision CG (fp64 defect correction around the fp32 CG): solves the same equation as lqcd_cg_solve_tm
 * for fp64 fields to fp64 accuracy while doing the iterations in fp32.
 *   x = 0, r = b;  repeat { fp32 CG on A e = (float) r to relative tolerance inner_tol;  x += e;  r = b - A x in fp64 }
 *   until |r| <= tol |b| (r is the TRUE fp64 residual), the total inner iteration count reaches maxiter, or a
 *   correction brings no progress.
 * ctx64 / ctx32: contexts of precision 64 and of precision 32 or 16 with the same extents and boundary phases (each with
 * its own recon; precision 16: the inner iteration keeps x, r in fp32 and p, Q p, A p in 16-bit storage); gauge64_dev / gauge32_dev: the link field packed for each; x_dev, b_dev: fp64 native even half spinors.
 * workspace_dev: lqcd_cg_mixed_workspace_bytes bytes, 256-byte aligned.  Synchronises `stream`.
 * *iters_out = total inner iterations, *outer_out = corrections applied, *relres_out = |b - A x| / |b|. */
size_t lqcd_cg_mixed_workspace_bytes(const lqcd_ctx* ctx64, const lqcd_ctx* ctx32);
lqcd_status lqcd_cg_solve_tm_mixed(const lqcd_ctx* ctx64, const lqcd_ctx* ctx32, void* x_dev, const void* gauge64_dev,
                                   const void* gauge32_dev, const void* b_dev, double kappa, double mu, double tol,
                                   double inner_tol, int maxiter, void* workspace_dev, int* iters_out, int* outer_out,
                                   double* relres_out, void* stream);

/* End-to-end path for host-resident data: canonical host buffers in, canonical host buffers out.
 * For each of the n items: copy in_host[i] (canonical half spinor of parity 1 - out_parity[i]) to the device,
 * pack, lqcd_dslash_eo, unpack, copy the canonical half spinor of parity out_parity[i] to out_host[i].
 * Items are pipelined over three device slots and three streams (upload / kernels on `stream` / download; the two
 * copy streams and the events are created at a context's first host-path call and released by lqcd_destroy), so
 * both PCIe directions and the kernels overlap.  Host-path calls on one context are serialised.  gauge_host: canonical links, uploaded and packed first; NULL
 * reuses the links packed into workspace_dev by an earlier call.  workspace_dev: device scratch of
 * lqcd_host_workspace_bytes bytes, 256-byte aligned, owned by the caller.  Host buffers should be pinned
 * (pageable memory works, without overlap).  Work already enqueued on `stream` is ordered before the call; the
 * call synchronises before returning (its results live in host memory).  lqcd_dslash_eo_host is the n = 1 case. */
lqcd_status lqcd_dslash_eo_host_batch(const lqcd_ctx* ctx, int n, void* const* out_host, const void* gauge_host,
                                      const void* const* in_host, const int* out_parity, void* workspace_dev,
                                      void* stream);
lqcd_status lqcd_dslash_eo_host(const lqcd_ctx* ctx, void* out_host, const void* gauge_host,
                                const void* in_host, int out_parity, void* workspace_dev, void* stream);

/* ---- pure-gauge SU(3) heatbath (next row f4; "On the PGT side we need a SU(3) heatbath algorithm [20]",
 * ref. [20] at :156: Creutz, Cabibbo-Marinari, Kennedy-Pendleton; reading F7) ----
 * Wilson action S = beta sum_p (1 - 1/3 Re tr U_p).  The update kernels work on the UPDATE LAYOUT of the link field
 * (precision-64 contexts only; links are periodic and carry no boundary phase): structure of arrays, checkerboarded --
 * the complex128 word w = 3 row + col of U_mu(x), x of parity p and checkerboard index cb, at
 * ((mu 2 + p) 9 + w) 32 ntiles + cb -- lqcd_update_links_bytes bytes, 16-byte aligned; lqcd_pack_update_links /
 * lqcd_unpack_update_links convert from / to the canonical field [mu 4][T][Z][Y][X][3][3] complex128 on the device.
 * lqcd_heatbath_sublattice updates, in place, the links U_mu(x) of one direction mu on the sites of one parity: staple
 * sum, then the SU(2) subgroups (0,1), (0,2), (1,2), each drawn with the Kennedy-Pendleton sampler.  The uniform random
 * numbers are an INPUT: uniforms_dev holds lqcd_heatbath_uniforms(ctx, ntries) doubles in (0, 1], [site cb of the parity]
 * [subgroup 3][4 ntries + 2] (the 4 numbers of attempt t at [4 t, 4 t + 4), then cos(theta) and phi of the direction); a
 * subgroup with none of its ntries (1..64) attempts accepted is left unchanged.  Eight calls (mu = 0..3, parity 0, 1) are
 * a sweep; unpack and lqcd_pack_gauge before the next dslash.  One launch each, asynchronous on `stream`.
 * lqcd_plaquette: the average of 1/3 Re tr U_p over all 6 V plaquettes of a field in the update layout, to host
 * (synchronises `stream`); workspace_dev: lqcd_plaquette_workspace_bytes bytes, 256-byte aligned.  Deterministic. */
size_t lqcd_update_links_bytes(const lqcd_ctx* ctx);
lqcd_status lqcd_pack_update_links(const lqcd_ctx* ctx, void* update_dev, const void* canonical_dev, void* stream);
lqcd_status lqcd_unpack_update_links(const lqcd_ctx* ctx, void* canonical_dev, const void* update_dev, void* stream);
size_t lqcd_heatbath_uniforms(const lqcd_ctx* ctx, int ntries);
lqcd_status lqcd_heatbath_sublattice(const lqcd_ctx* ctx, void* links_update_dev, double beta, int mu, int parity,
                                     const void* uniforms_dev, int ntries, void* stream);
/* Projects every link of a field in the update layout back to SU(3), in place (reading F8): row 0 normalised,
 * row 1 orthogonalised against it and normalised, row 2 = conj(row 0 x row 1).  Every sublattice update multiplies a
 * link by a rounded SU(2) element, so over many sweeps the links drift off the group, and 12- / 8-real storage assumes
 * det = 1 and unitarity exactly: call this every few sweeps and before lqcd_unpack_update_links + lqcd_pack_gauge.
 * A link that already is in SU(3) changes by rounding only.  One launch, asynchronous on `stream`; precision 64. */
lqcd_status lqcd_reunitarise_links(const lqcd_ctx* ctx, void* links_update_dev, void* stream);
size_t lqcd_plaquette_workspace_bytes(const lqcd_ctx* ctx);
lqcd_status lqcd_plaquette(const lqcd_ctx* ctx, const void* links_update_dev, void* workspace_dev, double* plaq_host,
                           void* stream);

/* Which kernel the hot-path entry points of this ctx launch (same arithmetic, same results up to the order of the
 * floating-point accumulation, which is identical: both add the eight hops in the order x+, x-, y+, y-, z+, z-, t+, t-):
 *   LQCD_KERNEL_GATHER  one thread per output site, operands gathered into registers (the default)
 *   LQCD_KERNEL_PIPE    persistent warp-specialised kernel, one CTA per SM: a producer warp stages links and
 *                       neighbour-spinor tiles in a shared-memory ring with TMA bulk copies (cp.async.bulk + mbarrier),
 *                       consumer warps compute from shared memory (north_star (3): "shared-memory or TMA staging of
 *                       neighbour tiles").  Precision 32 / 64 with links of the same precision; otherwise
 *                       LQCD_EUNSUPPORTED.  The time-slab boundary kernel (lqcd_dslash_eo_slab) is always the gather form. */
#define LQCD_KERNEL_GATHER 0
#define LQCD_KERNEL_PIPE 1
#define LQCD_KERNEL_BLOCKED 2 /* the gather kernel with the blocked thread -> site map (4-D boxes of warp tiles per block) */
#define LQCD_KERNEL_LSTAGE 3  /* the gather kernel with the link stream staged through shared memory by the TMA unit
                                 (every warp double-buffers its tile's link blocks with cp.async.bulk); precision 32 / 64 */
lqcd_status lqcd_set_kernel(lqcd_ctx* ctx, int kernel);

/* Host-side self test of the index map's division-free arithmetic: n / d as the kernels compute it (multiply-shift by a
 * reciprocal of the extent d set up in lqcd_create), for 1 <= d and n < 2^30.  tests/test_abi.py compares it with n / d. */
unsigned lqcd_selftest_fastdiv(unsigned d, unsigned n);

/* Number of kernels this library has launched since load (a claim counter for bench.py). */
unsigned long long lqcd_launch_count(void);

const char* lqcd_status_string(lqcd_status s);
const char* lqcd_last_cuda_error(void); /* text of the last CUDA error seen by this thread's calls */

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
