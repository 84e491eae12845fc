/* hisq.h -- C ABI of libhisq: the even-odd HISQ staggered Dslash on multiple right-hand sides and the
 * multi-RHS conjugate gradient on (m^2 - D_eo D_oe) x = b, hand-written CUDA for sm_100a (B200).
 *
 * What is computed (arXiv:2306.01098, cited by line of reference/PAPER.md):
 *
 *   (D phi)(x) = sum_{mu=0..3} [ X_mu(x) phi(x+mu) - X_mu(x-mu)^+ phi(x-mu)
 *                              + W_mu(x) phi(x+3mu) - W_mu(x-3mu)^+ phi(x-3mu) ]
 *
 * X = fat links, W = Naik links, both complex 3x3 with every constant and the staggered phases
 * already folded in by the caller; site coordinates periodic, the colour-vector field
 * periodic in x,y,z and ANTI-periodic in t -- the library applies that sign itself.
 * D only connects sites of opposite parity pi(x) = (x+y+z+t) mod 2, so it splits into D_eo (even
 * outputs from odd inputs) and D_oe.  The solver works on A = m^2 - D_eo D_oe, the even-even block
 * of M^+ M for M = D + m (Eq. (1), :139-141 `applyMdaggM`).
 *
 * Conventions common to all calls
 *   - mu = 0,1,2,3 <-> x,y,z,t; V = Lx*Ly*Lz*Lt; Vh = V/2.  All four extents must be even and >= 4.
 *   - Site index, Eq. (4):  lex = x + Lx*(y + Ly*(z + Lz*t)),  h = lex / 2 (integer),
 *     eo = h + pi(x)*Vh: even sites fill [0,Vh), odd sites [Vh,V).
 *   - CANONICAL link array, Eq. (5): matrix of (x, mu) at slot mu*V + eo(x); each
 *     matrix 9 complex numbers row-major U[a][b], (re, im) interleaved; (U phi)_a = sum_b U_ab phi_b.
 *   - CANONICAL half-lattice field of one parity with n right-hand sides: element (k, h, c) at
 *     ((k*Vh + h)*3 + c) complex, (re, im) interleaved  (k = RHS, c = colour).
 *   - NATIVE half-lattice field (what hisq_dslash / hisq_cg read and write, so that no per-call
 *     repack sits inside the operator): element (k, c, h) at ((k*3 + c)*Vh + h) complex.
 *     hisq_spinor_pack / hisq_spinor_unpack convert.  RHS k is one contiguous block of 3*Vh complex.
 *   - Element type follows `prec`: HISQ_FP32 -> float, HISQ_FP64 and HISQ_MIXED -> double.
 *   - Unless a parameter says HOST, every data pointer is a CUDA DEVICE pointer, 16-byte aligned,
 *     owned by the caller (e.g. a torch tensor's data_ptr()).  The library allocates no device
 *     memory: the caller gives it one workspace (hisq_workspace_bytes / hisq_set_workspace).
 *   - All work is enqueued on the stream given to hisq_set_stream (default: the legacy stream).
 *   - Every function returns 0 on success or a negative HISQ_E* code; nothing throws or aborts.
 *   - A context is not thread-safe; use one per host thread / per GPU.
 */
#ifndef HISQ_H
#define HISQ_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hisq_ctx hisq_ctx; /* opaque; created by hisq_create, freed by hisq_destroy */

enum { HISQ_FP32 = 4, HISQ_FP64 = 8, HISQ_MIXED = 12 }; /* `prec` */
enum { HISQ_EVEN = 0, HISQ_ODD = 1 };                   /* parity of the OUTPUT sites */
enum { HISQ_MAX_NRHS = 16 };

enum {
    HISQ_OK = 0,
    HISQ_EINVAL = -1,       /* bad extent (odd or < 4), nrhs < 1 or > HISQ_MAX_NRHS, bad parity/prec, null
                               or misaligned pointer, in/out aliasing, unknown option                      */
    HISQ_ENOLINKS = -2,     /* hisq_dslash / hisq_cg before hisq_set_links                                 */
    HISQ_ENOWORKSPACE = -3, /* no workspace set, or it is smaller than hisq_workspace_bytes(nrhs)          */
    HISQ_ECUDA = -4,        /* a CUDA call failed; text via hisq_last_error                                */
    HISQ_ENOCONV = -5,      /* max_iter reached; x holds the last iterate, hisq_get_info the residuals     */
    HISQ_EBREAKDOWN = -6,   /* <p, A p> <= 0 or a non-finite scalar appeared in CG; hisq_smear: singular link */
    HISQ_EIO = -7,          /* file cannot be opened / is truncated / fails its checksum or link trace     */
    HISQ_EPEER = -8,        /* multi-rank solve: another rank aborted (its error, or options that differ
                               between the ranks); the mailboxes must be zeroed and re-attached             */
    HISQ_ETOOBIG = -9       /* hisq_norm2_noalloc: more right-hand sides or reals than its static scratch holds */
};

/* Create a context for an Lx x Ly x Lz x Lt lattice on the current CUDA device.
 * prec: HISQ_FP32 (fp32 links, fields, arithmetic), HISQ_FP64, or HISQ_MIXED (fp64 interface; CG runs
 * the fp32 operator inside and an fp64 reliable update outside; hisq_dslash is the fp64 operator). */
int hisq_create(hisq_ctx **h, int Lx, int Ly, int Lz, int Lt, int prec);
int hisq_destroy(hisq_ctx *h);

/* cuda_stream: a cudaStream_t passed as void* (e.g. torch.cuda.current_stream().cuda_stream). */
int hisq_set_stream(hisq_ctx *h, void *cuda_stream);

/* Bytes of device workspace needed for links (internal copy/copies) plus CG temporaries, reduction
 * buffers and host-call staging for up to `nrhs` right-hand sides.  0 if the arguments are invalid. */
size_t hisq_workspace_bytes(const hisq_ctx *h, int nrhs);
/* Hand the library `bytes` of device memory at dev_ptr (256-byte aligned).  The caller keeps ownership
 * and must keep it alive and untouched until hisq_destroy or the next hisq_set_workspace.  Setting a
 * workspace invalidates links set earlier. */
int hisq_set_workspace(hisq_ctx *h, void *dev_ptr, size_t bytes);

/* Copy the two CANONICAL link arrays (each 4*V matrices, Eq. (5)) into the library's own layout: one RECORD per output
 * site holding the 16 links its stencil needs (its own 8 forward links and the 8 links of its backward neighbours x - mu,
 * x - 3 mu, fetched here once), the records of 32 consecutive sites interleaved by 16-byte chunk, so that the Dslash
 * streams its links as contiguous 3.5 - 4.5 KB runs per warp and stencil term (bulk-copy / TMA friendly) and never
 * computes a link address.  Every link is stored twice (once forward, once backward): 2 x 16 x 18 reals per site pair of
 * workspace, the bytes READ per Dslash application stay 16 links per output site.  fp32 and fp64 copies for HISQ_MIXED.
 * Synchronises the stream before returning: the caller may free fat / naik at once.
 * Links carry all coefficients and phases; the library applies none. */
int hisq_set_links(hisq_ctx *h, const void *fat, const void *naik);

/* out = D_eo in (parity = HISQ_EVEN: `out` on even sites, `in` on odd sites) or out = D_oe in
 * (parity = HISQ_ODD), for nrhs fields at once, each link loaded once and applied to all of them
 * (PAPER.md:582-586).  in / out: NATIVE half-lattice fields, must not overlap.  Asynchronous. */
int hisq_dslash(hisq_ctx *h, void *out, const void *in, int parity, int nrhs);

/* out = (mass^2 - D_eo D_oe) in on even sites for nrhs fields: the operator the solvers invert (PAPER.md:139-141
 * `applyMdaggM`), two Dslash launches, the second fused with the m^2 term.  in / out: NATIVE even half-lattice fields,
 * must not overlap; uses the workspace (sized for >= nrhs).  HISQ_MIXED runs it in fp64.  Asynchronous.  Not available on
 * partitioned contexts. */
int hisq_apply_A(hisq_ctx *h, void *out, const void *in, double mass, int nrhs);

/* Solve (mass^2 - D_eo D_oe) x_k = b_k, k < nrhs, on even sites by conjugate gradient with
 * independent alpha_k, beta_k per right-hand side and a shared operator application
 * (PAPER.md:135, :141).  b, x: NATIVE even half-lattice fields; x is overwritten (initial guess 0).
 * Stops when ||r_k|| <= tol * ||b_k|| (2-norm, not squared) for every k, confirmed on the residual
 * recomputed as b - A x in fp64; converged right-hand sides are frozen while the rest continue.
 * HISQ_MIXED: fp32 operator and fp32 r, p, Ap; every `reliable_interval` iterations x is accumulated
 * in fp64 and r replaced by the fp64 true residual, the search direction kept.
 * Returns after the solve has finished (synchronises the stream).  HISQ_ENOCONV / HISQ_EBREAKDOWN as above. */
int hisq_cg(hisq_ctx *h, void *x, const void *b, double mass, double tol, int nrhs);

/* Multi-shift CG (AdvancedMultiShiftCG): solve (mass^2 + shifts[k] - D_eo D_oe) x_k = b for nshift
 * shifts sigma_k >= 0 (HOST array) and ONE right-hand side b, with one operator application per iteration (on the
 * smallest shift; the Krylov space is shift invariant, the other solutions cost extra AXPYs only).
 * b: one NATIVE even half-lattice field; x: nshift NATIVE fields, x_k at offset k*3*Vh complex, overwritten.
 * nshift <= the nrhs the workspace was sized for.  Each shift stops when |zeta_k| ||r|| <= tol ||b|| / 2 (the
 * factor 2 is a margin for the drift of the recursive residual) and is frozen; afterwards the true residuals
 * ||b - (A + sigma_k) x_k|| / ||b|| are recomputed (hisq_get_info) and HISQ_ENOCONV is returned if one exceeds tol.
 * HISQ_FP64 and HISQ_FP32 contexts only (HISQ_MIXED: HISQ_EINVAL). */
int hisq_cg_multishift(hisq_ctx *h, void *x, const void *b, double mass, const double *shifts, int nshift, double tol);

/* Solve the full staggered system  M x = b,  M = D + mass  (Eq. (1)), on BOTH parities for nrhs right-hand
 * sides, by even-odd (Schur complement) preconditioning on top of hisq_cg (the solvers work on
 * M^+ M, whose even-even block is mass^2 - D_eo D_oe):
 *     s_e = mass b_e - D_eo b_o                     one Dslash, the xpay fused into its epilogue
 *     (mass^2 - D_eo D_oe) x_e = s_e                hisq_cg (this context's precision mode, incl. HISQ_MIXED)
 *     x_o = (b_o - D_oe x_e) / mass                 one Dslash + one element-wise kernel
 * b_even, b_odd, x_even, x_odd: NATIVE half-lattice fields (nrhs each), pairwise non-overlapping; x_odd is also used as
 * scratch during the solve.  mass > 0.  Since b - M x = (r_e / mass, 0) with r_e the residual of the even system,
 * the even solve is run to tol * min_k( mass ||b_k|| / ||s_e,k|| ), so that on success every right-hand side has
 * ||b_k - M x_k|| <= tol ||b_k|| over the whole lattice; hisq_get_info then reports that full-lattice ratio.
 * Returns after the solve has finished (synchronises the stream).  Errors as hisq_cg; partitioned contexts:
 * HISQ_EINVAL. */
int hisq_solve_M(hisq_ctx *h, void *x_even, void *x_odd, const void *b_even, const void *b_odd, double mass, double tol,
                 int nrhs);

/* HISQ link smearing ("X and W are smeared gauge fields"; HISQ action):
 * from the thin gauge links U build the two link fields hisq_set_links takes,
 *     V = F7[U]  (fat7: weights 1/8, 1/16, 1/64, 1/384 for the 1-, 3-, 5-, 7-link paths)
 *     W = V (V^+ V)^(-1/2)                              (projection to U(3))
 *     fat  = fat_scale  * eta_mu(x) * F7L[W]            (fat7 with one-link weight 1 plus the Lepage term, weight -1/8)
 *     naik = naik_scale * eta_mu(x) * W_mu(x) W_mu(x+mu) W_mu(x+2mu)
 * eta_mu(x) = 1, (-1)^x, (-1)^(x+y), (-1)^(x+y+z) if fold_phases != 0, else 1.  With fat_scale = 1 and
 * naik_scale = -1/24 the free-field operator is 2 i sum_mu eta_mu (9/8 sin p - 1/24 sin 3p) = 2 i (p + O(p^5)); halve
 * both for the conventionally normalised derivative.  The gauge field is periodic.
 * thin, fat, naik, scratch: CANONICAL link arrays (4*V matrices each, Eq. (5)) in the context's element type, pairwise
 * non-overlapping; scratch: hisq_smear_bytes(h) bytes = two link arrays (on return the SECOND holds W, canonical).  Needs a
 * workspace (one counter).  Intermediate fields are kept structure-of-arrays inside fat / naik / scratch.
 * Synchronises the stream.  HISQ_EBREAKDOWN if a level-1 link is singular (no unitary factor); partitioned contexts:
 * HISQ_EINVAL. */
size_t hisq_smear_bytes(const hisq_ctx *h);
int hisq_smear(hisq_ctx *h, const void *thin, void *fat, void *naik, void *scratch, double fat_scale, double naik_scale,
               int fold_phases);

/* Gauge configurations in the NERSC archive format (PAPER.md:540 lists the formats the paper's code
 * reads: ILDG, MILC, NERSC, openQCD; the other three: hisq_cfg_* below).  HOST functions, no context, no CUDA: text header
 * (DATATYPE = 4D_SU3_GAUGE_3x3 | 4D_SU3_GAUGE, DIMENSION_1..4, FLOATING_POINT = IEEE64BIG | IEEE32BIG | IEEE64LITTLE |
 * IEEE32LITTLE, CHECKSUM, LINK_TRACE, PLAQUETTE) followed by the links in lexicographic site order (x fastest), mu = 0..3
 * per site, row-major matrices; the two-row type is completed with row 2 = conj(row0 x row1).
 * hisq_nersc_info: header only (any output pointer may be NULL; rows = 2 | 3, real_bytes = 4 | 8).
 * hisq_nersc_read: links_host (HOST, `bytes` >= 4*V*9 complex double) receives the CANONICAL link array (Eq. (5)) as
 *   complex double -- copy it to the device (convert for an fp32 context) and pass it to hisq_smear.  Verifies the
 *   32-bit checksum and the link trace of the header: HISQ_EIO if either fails, the file is short or cannot be opened;
 *   HISQ_EINVAL for a malformed header or extents the library does not take (odd or < 4).
 * hisq_nersc_write: the inverse (IEEE64BIG, rows = 2 | 3; `plaquette` goes into the header as given). */
int hisq_nersc_info(const char *path, int *L, int *rows, int *real_bytes, double *link_trace, double *plaquette);
int hisq_nersc_read(const char *path, void *links_host, size_t bytes);
int hisq_nersc_write(const char *path, const void *links_host, const int *L, int rows, double plaquette);

/* The other three formats of PAPER.md:540 -- ILDG (LIME container), MILC (version 5 binary) and openQCD (export_cnfg) --
 * behind one trio of HOST functions (csrc/cfg_io.cpp states each format as it is read).  All deliver / take the CANONICAL
 * link array (Eq. (5)) as complex double on the host.
 * hisq_cfg_info : extents L[4] = (Lx, Ly, Lz, Lt) and the width in bytes of the reals in the file (ILDG 4 | 8, MILC 4,
 *                 openQCD 8); either output pointer may be NULL.
 * hisq_cfg_read : `bytes` >= 4*V*9 complex double.  Integrity: ILDG verifies the SciDAC checksum record when the file has
 *                 one; MILC its two rotating-XOR checksums; openQCD recomputes the average plaquette (its only check).
 *                 HISQ_EIO on a failed check, a short or unreadable file; HISQ_EINVAL for a malformed header, a MILC file
 *                 with a site list (order != 0), or extents the library does not take (odd or < 4).
 * hisq_cfg_write: the inverse; real_bytes selects the file precision (ILDG 4 | 8, MILC 4, openQCD 8, else HISQ_EINVAL). */
enum { HISQ_FMT_ILDG = 1, HISQ_FMT_MILC = 2, HISQ_FMT_OPENQCD = 3 };
int hisq_cfg_info(const char *path, int format, int *L, int *real_bytes);
int hisq_cfg_read(const char *path, int format, void *links_host, size_t bytes);
int hisq_cfg_write(const char *path, int format, const void *links_host, const int *L, int real_bytes);

/* Options: "max_iter" (default 100000), "reliable_interval" (default 100 for HISQ_MIXED, 0 = off for
 * the others), "check_interval" (iterations enqueued between host polls of the convergence flag,
 * default 32), "use_graph" (1: replay one CG iteration as a CUDA graph, default 1),
 * "nrhs_inner" (RHS per thread, 0 = auto),
 * "tile_y", "tile_z" (CTA sweep order blocking in y,z; 0 = auto),
 * "naik_compress" (see hisq_naik_compressed; default 0), "fused_blas" (1: cooperative fused x/r/p update kernel when the
 * fields are small enough to stay in registers across a grid barrier, default 1), "window_mb" (L2 budget of the CTA sweep
 * order, default 20), "dot_fp64" (fp32 operator only: how the scalar products fused into the Dslash epilogue, <p,Ap> and
 * ||b - A x||^2, are accumulated: 1 = every product in fp64, 0 = the 6 products of one site summed in fp32 and widened once,
 * -1 = fp64 for the 1- and 2-RHS kernels (HBM-bound, free) and the per-site fp32 sum for the wider ones; default -1; sums
 * across sites are fp64 in every case), "overlap" (hisq_cg on a partitioned context: compute the slices that read no halo while the halo is
 * in flight; -1 = when at least half of the owned slices qualify (Lt_loc >= 12), 0 never, 1 always; default -1). */
int hisq_set_option(hisq_ctx *h, const char *key, double value);

/* After hisq_cg: iterations done, number of fp64 true-residual recomputations, and per RHS the true
 * relative residual ||b - A x|| / ||b|| (array of nrhs doubles on the HOST; any pointer may be NULL). */
int hisq_get_info(const hisq_ctx *h, int *iterations, int *reliable_updates, double *true_rel_resid);

/* CANONICAL <-> NATIVE half-lattice field conversion (device to device, asynchronous). */
int hisq_spinor_pack(hisq_ctx *h, void *native, const void *canonical, int nrhs);
int hisq_spinor_unpack(hisq_ctx *h, void *canonical, const void *native, int nrhs);

/* End-to-end variants with HOST buffers (pinned or pageable) in the CANONICAL layout: copy in, pack,
 * run, unpack, copy out, synchronise.  Staging lives in the workspace. */
int hisq_dslash_host(hisq_ctx *h, void *out_host, const void *in_host, int parity, int nrhs);
int hisq_cg_host(hisq_ctx *h, void *x_host, const void *b_host, double mass, double tol, int nrhs);

/* Row f3, first step: a lattice partitioned along t over `nranks` processes / GPUs (the paper's sub-lattices with
 * halos; "full" indices with halo Eq. (6)/(7) :467-488).  The context of rank r holds the
 * Lt_global/nranks time slices [r*Lt_loc, (r+1)*Lt_loc) on an EXTENDED local lattice Lx x Ly x Lz x (Lt_loc + 8):
 * local slice 4 + i is global slice r*Lt_loc + i; local slices 0..3 and Lt_loc+4..Lt_loc+7 are halos (depth 4: the Naik
 * term needs 3, 4 keeps local site parity = global site parity).  All layouts of this header apply to the extended
 * lattice (V = Lx*Ly*Lz*(Lt_loc+8)).  Links: the caller provides the links of the extended lattice (at least the
 * interior and the LOWER halo slices must hold the true links; the upper halo is never read).
 * hisq_dslash computes the interior slices only, reads t-neighbours from the halo slices of `in` (which the caller
 * must have filled: hisq_halo_pack -> exchange with the neighbouring ranks -> hisq_halo_unpack), and applies the
 * antiperiodic sign only on the ranks that own the global t boundary.  Halo slices of `out` are left untouched.
 * Lt_loc must be even and >= 4.  hisq_cg on a partitioned context (fp32 or fp64) solves across the ranks once the peer
 * mailboxes are attached (hisq_peer_attach, below; HISQ_EINVAL before): every rank calls it with its slab of b and
 * gets its slab of x (halo slices of x are overwritten); same arithmetic and stopping rule as on one GPU, including
 * the true-residual confirmation b - A x (over all ranks) and the resume if it fails; hisq_get_info reports the
 * global true residuals, identical on every rank.  HISQ_MIXED contexts run the fp32 iteration across the ranks with the
 * fp64 reliable update (halos of x and D_oe x in fp64, one all-reduce) every `reliable_interval` iterations;
 * hisq_cg_multishift (fp32 / fp64 contexts) runs the base system's two halo exchanges and two one-number all-reduces per
 * iteration, every rank getting its slab of all nshift solutions; mailboxes sized for nrhs >= 1 suffice for it.
 * A rank that fails releases the others: they return HISQ_EPEER instead of waiting for ever; every rank must be called
 * with the same arguments and options (checked at the start of the solve, HISQ_EINVAL on all ranks if not). */
int hisq_create_part(hisq_ctx **h, int Lx, int Ly, int Lz, int Lt_global, int prec, int rank, int nranks);
/* A second cut, along z: an nz x nt grid of ranks, rank = rz + nz * rt (the paper's sub-lattices are 4-dimensional,
 * PAPER.md:187-191; two cuts are what lets the 8 GPUs of a node share BASELINE's C5, whose Lt = 24 admits at most 6 ranks
 * along t).  With nz > 1 the extended local lattice is Lx x Ly x (Lz/nz + 8) x (Lt/nt + 8): local plane 4 + j is global
 * plane rz*Lz_loc + j, the 4 planes on each side are halos (3 are read; periodic direction, no sign).  The stencil is
 * axis-aligned, so the two halos are independent: z planes are exchanged for the owned time slices only, no corners.
 * Lz/nz and Lt/nt must be even and >= 4, nz * nt <= 16.  nz = 1 is hisq_create_part.  Everything said there holds;
 * hisq_halo_send / recv move both halos; hisq_cg does not split its Dslashes around the exchange on such a context (every
 * time slice reads the z halo).  hisq_zhalo_bytes / pack / unpack are the z counterparts of hisq_halo_bytes / pack /
 * unpack: buffers [k][c][Lt_loc][3 * (Lx/2) * Ly] complex; 0 / HISQ_EINVAL on a context without a z cut. */
int hisq_create_part2(hisq_ctx **h, int Lx, int Ly, int Lz_global, int Lt_global, int prec, int rank, int nz, int nt);
size_t hisq_zhalo_bytes(const hisq_ctx *h, int nrhs);
int hisq_zhalo_pack(hisq_ctx *h, void *send_lo, void *send_hi, const void *field, int nrhs);
int hisq_zhalo_unpack(hisq_ctx *h, void *field, const void *recv_lo, const void *recv_hi, int nrhs);
/* hisq_dslash restricted to the OWNED time slices [t_first, t_first + t_count) (0 <= t_first, t_first + t_count <= the
 * number of owned slices: Lt_loc on a partitioned context, Lt otherwise); all other slices of `out` are left untouched.
 * The slices [3, Lt_loc - 3) read no halo slice (the stencil reaches 3 sites), so the caller can compute
 * them while the halo exchange of `in` is in flight and the first and last 3 after hisq_halo_unpack: that is how
 * communication hides behind computation.  Errors as hisq_dslash; HISQ_EINVAL for a bad range. */
int hisq_dslash_slices(hisq_ctx *h, void *out, const void *in, int parity, int nrhs, int t_first, int t_count);
/* The first `width` and the last `width` owned slices in ONE launch (all owned slices if 2*width >= their number):
 * with width = 3, what is left to do once the halo has arrived. */
int hisq_dslash_edges(hisq_ctx *h, void *out, const void *in, int parity, int nrhs, int width);
/* Bytes of ONE halo buffer (3 slices, nrhs fields: of the 4 halo slices on a side only the 3 nearest are ever read);
 * 0 for a non-partitioned context. */
size_t hisq_halo_bytes(const hisq_ctx *h, int nrhs);
/* send_lo <- the 3 lowest interior slices (for the previous rank's upper halo), send_hi <- the 3 highest (for the next
 * rank's lower halo); buffers are device memory of hisq_halo_bytes each, layout [k][c][3*S] complex.  Asynchronous. */
int hisq_halo_pack(hisq_ctx *h, void *send_lo, void *send_hi, const void *field, int nrhs);
/* lower halo <- recv_lo (what the previous rank packed as send_hi), upper halo <- recv_hi (the next rank's send_lo). */
int hisq_halo_unpack(hisq_ctx *h, void *field, const void *recv_lo, const void *recv_hi, int nrhs);

/* Halo transport and all-reduce through peer-mapped memory, without a communication library (the exchange of
 * PAPER.md:340-348 done by the packing kernel's own stores over NVLink).  Every rank owns a MAILBOX of
 * hisq_peer_bytes(h, nrhs) bytes of device memory (256-byte aligned, ZEROED by the caller before any other rank
 * attaches) that the other ranks can address: cudaDeviceEnablePeerAccess within a process, a CUDA IPC mapping between
 * processes -- obtaining those pointers is the caller's plumbing.
 * hisq_peer_attach(h, boxes, nboxes, nrhs): boxes[r] = mailbox of rank r as addressable from this device (boxes[own
 * rank] = this rank's), nboxes = nranks of hisq_create_part (<= 16); nrhs = the capacity the mailboxes were sized for.
 * Then, per halo exchange and in this order on every rank:
 *   hisq_halo_send(h, field, nrhs)   packs the 3 lowest / highest owned slices of `field` straight into the
 *                                     t-neighbours' mailboxes; the kernel's last CTA bumps their arrival counters;
 *   hisq_halo_recv(h, field, nrhs)   waits (stream memory operation) until both neighbours' halos have arrived and
 *                                     unpacks its mailbox into the halo slices of `field`.
 * and per all-reduce (sum over ranks of the first nrhs doubles of a CG state array; which = 2 rho, 3 pq, 4 sums as in
 * hisq_cgp_ptr; in place):
 *   hisq_peer_reduce_send(h, which, nrhs)   stores the local values into every rank's mailbox, bumps its counter;
 *   hisq_peer_reduce_recv(h, which, nrhs)   waits until all ranks' values have arrived and adds them in rank order
 *                                            (the same order on every rank: all ranks end up with the same bits).
 * All four are asynchronous on the context's stream.  Signalling = system-scope atomics issued by the sending kernel
 * after fencing its stores; waiting = cuStreamWaitValue32 on the receiver's stream: no kernel spins, and work enqueued
 * between send and recv (the interior slices, hisq_dslash_slices) overlaps the transfer.  Mailboxes hold two slots
 * used in turn.  Every rank must issue the same sequence of calls, sends and recvs strictly alternating (send e,
 * recv e, send e+1, ...; likewise for reduces) -- that order is what makes a slot safe to overwrite two exchanges
 * later without any acknowledgement; a call out of order is refused (HISQ_EINVAL).  HISQ_ECUDA if the driver lacks
 * stream memory operations. */
size_t hisq_peer_bytes(const hisq_ctx *h, int nrhs);
int hisq_peer_attach(hisq_ctx *h, void *const *boxes, int nboxes, int nrhs);
int hisq_halo_send(hisq_ctx *h, const void *field, int nrhs);
int hisq_halo_recv(hisq_ctx *h, void *field, int nrhs);
int hisq_peer_reduce_send(hisq_ctx *h, int which, int nrhs);
int hisq_peer_reduce_recv(hisq_ctx *h, int which, int nrhs);

/* CG on a t-partitioned lattice, phase by phase.  The solver's reductions span all ranks, so the iteration is cut where
 * a cross-rank step is due and the CALLER performs it between the calls (halo exchange of a field through
 * hisq_halo_pack / unpack, all-reduce (sum) of nrhs doubles); paper_2306_01098_b200/partition.py holds the loop.
 *   hisq_cgp_begin(h, x, b, tol, nrhs)   x := 0, r := b (halo slices zeroed), LOCAL ||b_k||^2 -> rho
 *       -> all-reduce rho ->                                      hisq_cgp_phase(h, 0, mass)
 *   per iteration:  hisq_cgp_phase(h, 1, mass)   p = r + beta p                  -> halo exchange of p
 *                   hisq_cgp_phase(h, 2, mass)   t = D_oe p                      -> halo exchange of t
 *                   hisq_cgp_phase(h, 3, mass)   q = mass^2 p - D_eo t, LOCAL Re<p_k,q_k> -> pq      -> all-reduce pq
 *                   hisq_cgp_phase(h, 4, mass)   x += alpha p, r -= alpha q, LOCAL ||r_k||^2 -> sums -> all-reduce sums
 *                   hisq_cgp_phase(h, 5, mass)   beta_k, convergence flags, iteration count
 *   overlapped form: phase 2 = 20 (owned slices [3, Lt_loc-3), needs no halo) + 21 (the first and last 3 slices, after
 *                   the halo of p has arrived); phase 3 = 30 + 31 in the same way with the halo of t.  20/30 are empty
 *                   and 21/31 do everything when Lt_loc <= 6.  pq after 30 + 31 is bit-identical to phase 3's.
 *   hisq_cgp_status: synchronises and reports iterations, done, breakdown, recursive relative residuals (HOST arrays).
 * x, b: NATIVE even fields on the extended lattice (halo slices of b are ignored, those of x are undefined).
 * Same arithmetic and stopping rule as hisq_cg (no final true-residual check).  Works on ordinary contexts too
 * (then no exchange is needed).  hisq_cgp_ptr: device pointers the caller needs: 0 = p, 1 = t (fields),
 * 2 = rho, 3 = pq, 4 = sums (arrays of HISQ_MAX_NRHS doubles, the first nrhs are used). */
int hisq_cgp_begin(hisq_ctx *h, void *x, const void *b, double tol, int nrhs);
int hisq_cgp_phase(hisq_ctx *h, int phase, double mass);
void *hisq_cgp_ptr(hisq_ctx *h, int which);
int hisq_cgp_status(hisq_ctx *h, int *iterations, int *done, int *breakdown, double *rel_resid);

/* Row f2 (the paper's CompressionType).  With option "naik_compress" = 1, the next hisq_set_links
 * stores each Naik link as 14 reals: rows 0, 1 and the complex number d = det(W) / |row0 x row1|^2, from which
 * row 2 = conj(row0 x row1) d is rebuilt in registers.  That is exact for W = c U with c real and U in U(3) (d = det(U)/c):
 * the U(3)-projected Naik links hisq_smear produces as well as real multiples of SU(3) matrices.  The format is used
 * PROVIDED every Naik link passes |row2 - conj(row0 x row1) d| <= tol |row0| (tol 1e-12 fp64, 1e-5 fp32); otherwise the
 * links stay uncompressed.  Returns 1 if the context currently uses the compressed format. */
int hisq_naik_compressed(const hisq_ctx *h);

/* Number of kernels this context has launched since creation (bench.py's gpu_launches). */
long long hisq_launch_count(const hisq_ctx *h);

const char *hisq_strerror(int code);
/* Text of the last CUDA error seen by this context ("" if none). */
const char *hisq_last_error(const hisq_ctx *h);

/* An entry point that allocates NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid allocation): no context, no workspace.  out[k] = ||a_k||^2 = sum_i a[k][i]^2 for
 * nrhs fields of nreal reals each (field k at offset k*nreal reals; element type by prec: HISQ_FP32 float, HISQ_FP64 and
 * HISQ_MIXED double; for a half-lattice field nreal = 6*Vh), accumulated in fp64 in the fixed two-stage order of the CG's own
 * reductions (block partition and order of the solver's ||b_k||^2: the same bits).  field, out: DEVICE pointers (field
 * 16-byte aligned), out receives nrhs doubles; asynchronous on cuda_stream (a cudaStream_t as void*, NULL = legacy stream).
 * The scratch of the reduction (block partial sums, last-block ticket) is a file-scope __device__ array of 2 MiB + 256 B that
 * every GPU loading the library holds until the process exits; its device address is resolved once per device
 * (cudaGetSymbolAddress) on the first call with that device current.  Limits: nrhs <= HISQ_NOALLOC_MAX_NRHS (16) and
 * nreal <= hisq_norm2_noalloc_max_reals() = HISQ_NOALLOC_MAX_COLS * 4096 = 67 108 864 (BASELINE's largest lattice, 96^3 x 24,
 * has 63 700 992 reals per field); beyond either: HISQ_ETOOBIG, nothing is launched.  HISQ_EINVAL for null / misaligned
 * pointers, nreal = 0, nrhs < 1, a bad prec.  Calls no cudaMalloc / cudaFree or allocating library routine.
 * ALL calls on a device share the one array: calls that overlap on the GPU (different streams or host threads without
 * ordering between them) race and return wrong sums; ordered calls are safe (the array keeps the previous call's contents;
 * the partial sums are rewritten before they are read and the ticket is cleared on the stream before every launch). */
enum { HISQ_NOALLOC_MAX_NRHS = 16, HISQ_NOALLOC_MAX_COLS = 16384 };
size_t hisq_norm2_noalloc_max_reals(void);
int hisq_norm2_noalloc(const void *field, int prec, size_t nreal, int nrhs, double *out, void *cuda_stream);

/* Introspection (tests, DESIGN.md tables; no effect on any result).
 * hisq_debug_dslash_regs: registers per thread of the Dslash kernel instantiation for prec (HISQ_FP32 | HISQ_FP64),
 *   nr right-hand sides per thread (1,2,3,4,6,8) and epilogue mode (0 plain, 1 A-apply, 2 residual); -1 if unknown.
 * hisq_debug_tiles: out[0], out[1] = the (tile_y, tile_z) CTA sweep blocking the next Dslash launch with nrhs
 *   right-hand sides would use. */
int hisq_debug_dslash_regs(int prec, int nr, int mode);
int hisq_debug_tiles(hisq_ctx *h, int nrhs, int *out);

#ifdef __cplusplus
}
#endif
#endif /* HISQ_H */
