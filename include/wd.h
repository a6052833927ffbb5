/*
 * wd.h -- C ABI of the B200-native Wilson-Dirac matvec library (libwd.so).
 *
 * The one operation: apply the fine Wilson-Dirac operator of eq. (2.2) of arXiv:0912.2186
 * (section 2) to one or several spinor fields on a periodic 4-D lattice,
 *
 *   (D psi)(x) = (4+m) psi(x)
 *              - 1/2 sum_{mu=1..4} [ (1 - gamma_mu) (x) U_mu(x)        psi(x+mu)     forward hop
 *                                  + (1 + gamma_mu) (x) U_mu(x-mu)^dag psi(x-mu) ]   backward hop
 *
 * gamma_mu in the DeGrand-Rossi basis (reading S2), gamma on spin, U on colour,
 * x +- mu modulo L_mu (periodic, no phase; reading S3).  The "many test vectors, same links"
 * use of the adaptive set-up (eq. (2.6); N_v = 20) is the
 * nrhs > 1 case: out[r] = D in[r] for r < nrhs, one link load shared by all r.
 *
 * Everything is plain C: opaque handles, raw pointers, ints and doubles.  No torch types.
 * Every pointer named *_dev is a CUDA DEVICE pointer owned by the caller (e.g. the data_ptr()
 * of a torch tensor); every pointer named *_host is HOST memory owned by the caller.  The
 * library never frees caller memory and keeps no reference to it after the call returns,
 * except that work enqueued on the stream still reads/writes it until the stream reaches
 * that point: keep buffers alive until you synchronise.
 *
 * Error behaviour: every int-returning function returns WD_OK (0) or a negative wd_status;
 * nothing throws, exits or prints.  wd_last_error() gives a human-readable message for the
 * last failure on the calling thread.  wd_apply does not synchronise the host with the
 * device: launch errors are reported, asynchronous faults surface at the caller's next sync.
 * There is NO CPU fallback anywhere: without a CUDA device every compute entry point
 * returns WD_ERR_CUDA.
 *
 * Threads: a wd_lattice may be shared freely (it is immutable).  A wd_gauge handle owns mutable state -- its stream,
 * tuning, caches built on first use (the parity-ordered links of the red/black entry points, solver workspaces,
 * staging buffers), also behind entry points that take it as `const wd_gauge *` -- so calls on ONE gauge handle must not
 * run concurrently on several host threads; different handles are independent (wd_apply_schur_static excepted: all its
 * calls share one static array).
 *
 * CANONICAL layouts (what callers, tests and the oracle speak; C order, last index fastest):
 *   spinor  psi[rhs][t][z][y][x][spin 0..3][colour 0..2][re,im]      24 reals per site
 *   links   U  [mu 0..3][t][z][y][x][row a][col b][re,im]            18 reals per link
 *           mu = 0,1,2,3 <-> x,y,z,t; dims = {Lx, Ly, Lz, Lt}; U_mu(x) sits on the link
 *           x -> x+mu and (U psi)_a = sum_b U[a][b] psi_b            (readings S5, S6)
 * NATIVE layouts (what wd_apply reads and writes):
 *   spinor  [rhs][block of 32 sites][16-byte vector (float4 / double2)][lane], site = 32*block + lane
 *           = x + Lx*(y + Ly*(z + Lz*t)); the volume is padded to a multiple of 32 sites, so a native
 *           buffer holds wd_spinor_bytes() bytes (>= nrhs*V*24*sizeof(real)); pad sites are never read.
 *   links   private to wd_gauge.
 *   wd_pack_spinor / wd_unpack_spinor convert between the two, so a Krylov loop (100 applies
 *   back to back, BASELINE.json:configs[3]) never repacks.
 */
#ifndef WD_H
#define WD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    WD_OK = 0,
    WD_ERR_NULL = -1,      /* a required pointer is NULL                                   */
    WD_ERR_DIMS = -2,      /* an extent < 1, volume overflow, or dims do not match gauge   */
    WD_ERR_PRECISION = -3, /* precision is not WD_FP32 / WD_FP64 or differs from the gauge */
    WD_ERR_RECON = -4,     /* recon is not WD_RECON_18 / _12 / _8, or the links cannot be stored that way */
    WD_ERR_NRHS = -5,      /* nrhs < 1                                                     */
    WD_ERR_ALIAS = -6,     /* out and in overlap (the stencil is not in-place safe)        */
    WD_ERR_MISMATCH = -7,  /* handle belongs to another lattice / bad kernel selector      */
    WD_ERR_CUDA = -8,      /* a CUDA runtime call or launch failed (see wd_last_error)     */
    WD_ERR_ALLOC = -9      /* host or device allocation failed                             */
} wd_status;

/* WD_FP32 / WD_FP64: arithmetic AND storage type.  WD_FP16: half-precision STORAGE with float32 arithmetic (PAPER.md:159-167,
 * Table 2 row "Half"; reading RH): links as IEEE binary16 reals; spinors as, per site, a float32 scale s = max |component|
 * and the 24 ratios component / s as binary16 (value = s * ratio) -- 52 bytes per site and right-hand side.  With
 * WD_FP16 the CANONICAL buffers of wd_load_gauge / wd_pack_spinor / wd_unpack_spinor are float32; it is accepted by
 * wd_create_lattice .. wd_spinor_bytes, wd_load_gauge, wd_pack_spinor, wd_unpack_spinor, wd_apply and wd_apply_dagger
 * (one-thread-per-site kernel for any extents and nrhs, staged kernel where the lattice can be tiled), and by the
 * red/black family wd_spinor_bytes_parity, wd_pack_spinor_parity, wd_unpack_spinor_parity, wd_apply_hop, wd_apply_schur,
 * wd_apply_schur_dagger (the operator of the paper's "Half" kernel row; the intermediate field of the two launches is a
 * half-storage field too); every other entry point (solvers, transfer and coarse operators) answers WD_ERR_PRECISION. */
typedef enum { WD_FP16 = 16, WD_FP32 = 32, WD_FP64 = 64 } wd_precision;
typedef enum { WD_RECON_18 = 18, WD_RECON_12 = 12, WD_RECON_8 = 8 } wd_recon; /* reals stored per link */

/* Kernel selector for wd_set_kernel (measurement and tests; default WD_KERNEL_AUTO). */
typedef enum {
    WD_KERNEL_AUTO = 0,    /* fastest kernel valid for the lattice                         */
    WD_KERNEL_SITE = 1,    /* one thread per site, neighbours straight from L1/L2, any dims */
    /* 2 was the round-1 tile kernel: superseded by the staged kernel on every measured case, removed */
    WD_KERNEL_STAGE = 3    /* t-marching tile kernel, all global reads staged by cp.async (fp32 and fp64; its multi-RHS
                              member shares the staged links between right-hand sides in fp32) */
} wd_kernel;

typedef struct wd_lattice wd_lattice; /* opaque: extents, volume                           */
typedef struct wd_gauge wd_gauge;     /* opaque: native device copy of the links + stream  */

/*
 * wd_create_lattice -- describe a periodic Lx x Ly x Lz x Lt lattice ("a
 * hypercubic lattice", vector space of dimension 12 L^3 T).  Host-only, needs no GPU.
 * dims[mu] >= 1 (extent 1 and 2 follow reading S4: coincident neighbours both count).
 * On success *lat is a new handle to be released with wd_destroy.
 */
int wd_create_lattice(const int dims[4], wd_lattice **lat);

/* Extents / volume of a lattice handle (host-only helpers). */
int wd_lattice_dims(const wd_lattice *lat, int dims_out[4]);
long long wd_lattice_volume(const wd_lattice *lat);

/*
 * wd_load_gauge -- take the links U_mu(x) of eq. (2.2) ("3x3 (dense) SU(3) color
 * matrices") in CANONICAL 18-real layout from DEVICE memory `links_canonical_dev`
 * (4*V*18 reals of the given precision) and build the library's native copy:
 * reordered to structure-of-arrays and, for recon == WD_RECON_12, compressed to rows 0 and 1
 * of each link, the third row being rebuilt in the kernel as conj(row0 x row1)
 * ("Gauge field stored as 12 ... floats"; reading S7).  recon == WD_RECON_8 ("or 8
 * floats"; reading R8): per link the eight reals (Re a2, Im a2, Re a3, Im a3, Re b1, Im b1, arg(a1)/pi, arg(c1)/pi) of
 * its rows a, b, c -- phases formed in double, rounded once to the working precision; the kernels rebuild the link from
 * |a1|^2 = 1 - |a2|^2 - |a3|^2, |c1|^2 = 1 - |a1|^2 - |b1|^2 and unitarity.  A link with a2 = a3 = 0 (e.g. the unit
 * matrix, hence temporal-gauge links) has no such representation: WD_ERR_RECON (checked; synchronises the stream).
 * Rounding in the rebuilt rows is amplified by 1 / (|a2|^2 + |a3|^2): tolerance in DESIGN.md section 2.
 * The conversion is enqueued on `stream` (a cudaStream_t cast to void*, NULL = default
 * stream), which also becomes the stream wd_apply launches on.  The caller may free
 * `links_canonical_dev` once that stream work has completed.  *gauge is owned by the
 * library (device memory from cudaMalloc) until wd_destroy_gauge.
 */
int wd_load_gauge(const wd_lattice *lat, const void *links_canonical_dev, int precision, int recon,
                  void *stream, wd_gauge **gauge);

/* Stream (cudaStream_t as void*) on which every entry point that takes a wd_gauge launches from now on: wd_apply,
 * wd_apply_dagger, wd_apply_hop / _schur, the solvers, wd_set_temporal_gauge, wd_apply_host (which also uses three
 * private streams, ordered after and before this one).  Work already queued on the previous stream (the link conversion
 * of wd_load_gauge, earlier applies) is ordered BEFORE anything launched on the new stream (event record + wait).
 * wd_pack_spinor / wd_unpack_spinor / the transfer operators take their own stream argument and are NOT tied to the
 * gauge's stream: the caller orders them. */
int wd_set_stream(wd_gauge *gauge, void *stream);

/* Tuning variables of the launchers.  They are read from the environment ONCE, at wd_load_gauge
 * (WD_TILE_SHAPE=ty,tz, WD_TILE_TC, WD_TILE_NCHUNK, WD_TILE_NRB, WD_MRHS_PATCH, WD_STAGE_NO_MRHS, WD_SITE_SLAB_MB,
 * WD_HOST_NO_PIPELINE, WD_MRHS_NO_TAIL, WD_HOST_NSLAB, WD_MRHS_BULK, WD_MRHS_REG, WD_MRHS_RGRP, WD_STAGE_BULK), and stored in the gauge handle; no launch reads the environment.
 * wd_set_tuning changes one of them afterwards: name is the lower-case variable without the WD_ prefix ("tile_ty",
 * "tile_tz", "tile_tc", "tile_nchunk", "tile_nrb", "mrhs_patch", "stage_no_mrhs", "site_slab_mb", "host_no_pipeline",
 * "mrhs_no_tail", "host_nslab", "mrhs_bulk", "mrhs_reg", "mrhs_rgrp", "stage_bulk"); value < 0 restores the default.  WD_ERR_MISMATCH for an unknown name.  Host-only. */
int wd_set_tuning(wd_gauge *gauge, const char *name, int value);

/* Temporal gauge ("temporal gauge fixing", Fig. 4 / Table 2 "GF"): on != 0 declares that the loaded links
 * satisfy U_t(x,t) = 1 for every t < Lt-1 (the last slice carries the Polyakov lines).  The library verifies it
 * (WD_ERR_MISMATCH if some such link differs from 1 by more than 1e-6 / 1e-12; synchronises the stream) and the staged
 * kernels and the red/black kernel (wd_apply_hop, wd_apply_schur*, the solvers) then neither load those links nor
 * multiply by them; the other kernels ignore the flag (same result).
 * The operator is unchanged: D(U^g)(g psi) = g D(U) psi. */
int wd_set_temporal_gauge(wd_gauge *gauge, int on);

/* Force a kernel variant (wd_kernel).  WD_ERR_MISMATCH if it cannot handle the lattice. */
int wd_set_kernel(wd_gauge *gauge, int kernel);

/* The kernel (wd_kernel, > 0) that wd_apply will launch for this gauge and nrhs right-hand sides:
 * the forced one, or what WD_KERNEL_AUTO resolves to.  Host-only query; negative wd_status on error. */
int wd_selected_kernel(const wd_gauge *gauge, int nrhs);

/* Bytes of a NATIVE spinor buffer holding nrhs fields: nrhs * Vpad * 24 * sizeof(real), where
 * Vpad = V rounded up to a multiple of 32 sites.  0 on bad arguments. */
size_t wd_spinor_bytes(const wd_lattice *lat, int nrhs, int precision);

/*
 * wd_pack_spinor / wd_unpack_spinor -- CANONICAL <-> NATIVE spinor layout on the device
 * (pure data movement, no arithmetic), enqueued on `stream`.  The canonical buffer holds nrhs
 * fields of V*24 reals, the native buffer wd_spinor_bytes() bytes; they must not overlap.
 */
int wd_pack_spinor(const wd_lattice *lat, void *native_dev, const void *canonical_dev, int nrhs,
                   int precision, void *stream);
int wd_unpack_spinor(const wd_lattice *lat, void *canonical_dev, const void *native_dev, int nrhs,
                     int precision, void *stream);

/*
 * wd_apply -- out[r] = D(U; mass) in[r], r = 0..nrhs-1: eq. (2.2); all of
 * SURVEY.md section 8(a) steps a1-a7 (neighbour gather with periodic wrap, 12-real link
 * reconstruction, spin projection, SU(3) mat-vec on half spinors, reconstruct-and-accumulate,
 * fused (4+m) diagonal, store) run inside ONE kernel launch on the gauge's stream.
 *   out_native_dev, in_native_dev : DEVICE, NATIVE layout, nrhs fields, 16-byte aligned, no overlap
 *   gauge     : from wd_load_gauge
 *   mass      : m of eq. (2.2); the diagonal coefficient 4+m is formed in double, then rounded
 *               to the working precision; the hopping coefficient is exactly 1/2 (reading S8)
 *   dims      : must equal the lattice the gauge was loaded for (checked, not trusted)
 *   nrhs      : number of right-hand sides (>= 1); links are loaded once per site and
 *               direction for a group of right-hand sides
 *   precision : WD_FP32 / WD_FP64, must equal the gauge's
 * Signature order follows BASELINE.json:north_star.
 */
int wd_apply(void *out_native_dev, const void *in_native_dev, const wd_gauge *gauge, double mass,
             const int dims[4], int nrhs, int precision);

/* wd_apply_dagger -- out[r] = D^dagger in[r] = gamma5 D gamma5 in[r] ("gamma5-Hermiticity"): every
 * projector 1 -+ gamma_mu swapped; same arguments, checks and kernel selection as wd_apply (the staged kernel is
 * templated on the projector sign; several right-hand sides go through its single-RHS member). */
int wd_apply_dagger(void *out_native_dev, const void *in_native_dev, const wd_gauge *gauge, double mass,
                    const int dims[4], int nrhs, int precision);

/*
 * wd_apply_host -- the same operation for callers whose data lives in HOST memory, in
 * CANONICAL layout: copies in_canonical_host to the device, packs, applies D, unpacks, copies
 * the result to out_canonical_host and synchronises the gauge's stream before returning.
 * Fields of at least 8 MB on lattices with Lx*Ly*Lz a multiple of 128 and Lt >= 3 are cut into
 * slabs of whole time slices (16 by default, tuning variable "host_nslab", 3..32) and pipelined
 * over three internal streams (copies in; pack, apply on a range of time slices, unpack; copies
 * out), so the two PCIe directions overlap; other lattices go through one stream.  Both paths
 * give the same bits.  Work already enqueued on the gauge's stream is waited for first.
 * Device staging buffers, streams and events are owned by the gauge handle (created on first use,
 * reused, released by wd_destroy_gauge); not re-entrant for one gauge handle.
 * Pinned host memory gives asynchronous copies; pageable memory works but is slower.
 */
int wd_apply_host(void *out_canonical_host, const void *in_canonical_host, wd_gauge *gauge,
                  double mass, const int dims[4], int nrhs, int precision);

/*
 * ---- red/black (even-odd) blocks: PAPER.md:126 ("red/black preconditioning"), PAPER.md:157 (the paper's GPU
 * kernel is the even-odd matvec); SURVEY.md 8(f) row f1.  Every extent must be even (WD_ERR_DIMS otherwise).
 * Site parity p(x) = (x+y+z+t) mod 2; D = [ (4+m) 1, H_eo ; H_oe, (4+m) 1 ] with H_pq the hopping term of
 * eq. (2.2) from parity q to parity p (factor -1/2 included).  A HALF FIELD holds the V/2 sites of one parity in
 * the blocked native layout over the checkerboard index lex/2; wd_spinor_bytes_parity() is its size.
 * The first red/black call on a gauge handle (wd_apply_hop, wd_apply_schur*, any solver) allocates and fills, on the
 * gauge's stream, a parity-ordered copy of the handle's link records (as large as the native links; WD_ERR_ALLOC if
 * that fails); it is owned by the handle and released by wd_destroy_gauge.
 */
size_t wd_spinor_bytes_parity(const wd_lattice *lat, int nrhs, int precision);

/* CANONICAL full-lattice field (nrhs * V * 24 reals, DEVICE) -> native half field of `parity`, and back
 * (unpack writes only the sites of `parity`; the other sites of the canonical buffer are left untouched). */
int wd_pack_spinor_parity(const wd_lattice *lat, void *native_half_dev, const void *canonical_dev, int nrhs,
                          int precision, int parity, void *stream);
int wd_unpack_spinor_parity(const wd_lattice *lat, void *canonical_dev, const void *native_half_dev, int nrhs,
                            int precision, int parity, void *stream);

/* out_p = H_pq in_q : `out_half_dev` is a half field of parity `parity_out`, `in_half_dev` of the opposite
 * parity; one kernel launch on the gauge's stream.  Buffers 16-byte aligned, no overlap. */
int wd_apply_hop(void *out_half_dev, const void *in_half_dev, const wd_gauge *gauge, const int dims[4], int nrhs,
                 int precision, int parity_out);

/* Even-odd preconditioned operator on `parity`:  out = (4+mass) in - H_pq (4+mass)^-1 H_qp in  (two launches;
 * `tmp_half_dev` is a caller-owned half field that receives H_qp in).  mass != -4. */
int wd_apply_schur(void *out_half_dev, const void *in_half_dev, void *tmp_half_dev, const wd_gauge *gauge, double mass,
                   const int dims[4], int nrhs, int precision, int parity);

/* out = Mhat^dagger in  (= gamma5 Mhat gamma5): same calling convention as wd_apply_schur. */
int wd_apply_schur_dagger(void *out_half_dev, const void *in_half_dev, void *tmp_half_dev, const wd_gauge *gauge,
                          double mass, const int dims[4], int nrhs, int precision, int parity);

/*
 * wd_apply_schur_static -- wd_apply_schur for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): out = Mhat in on `parity`, WD_FP32 or
 * WD_FP64, any link format, two launches on the gauge's stream.  The intermediate half field H_qp in lives in a static
 * device array of WD_STATIC_SCRATCH_BYTES inside the library (every GPU that loads the library holds it until the
 * process exits) and the links are read from the gauge handle's ordinary native links, so the call allocates nothing:
 * no cudaMalloc, cudaFree or allocating library routine, on the first call or any later one (unlike the other
 * red/black entry points, whose first call on a handle allocates a parity-ordered link copy).
 * Limit: nrhs * padded(V/2) * 24 * sizeof(real) <= WD_STATIC_SCRATCH_BYTES (padded = rounded up to 32 sites), e.g. one
 * fp32 right-hand side on 349 504 lattice sites (16^3 x 32 fits 2 in fp32, 1 in fp64); beyond it: WD_ERR_DIMS, nothing
 * launched.  Other errors as wd_apply_schur.  Every call shares the array and it keeps the last call's contents
 * (nothing in it has to start at zero: it is fully written before it is read); calls that overlap on the GPU
 * (different streams, several host threads, several gauge handles) race on it -- serialise them.
 */
#define WD_STATIC_SCRATCH_BYTES (16u << 20)
int wd_apply_schur_static(void *out_half_dev, const void *in_half_dev, const wd_gauge *gauge, double mass,
                          const int dims[4], int nrhs, int precision, int parity);

/*
 * wd_cgnr_schur -- conjugate gradients on the normal equations of the even-odd preconditioned operator
 * ("CG on the normal equations"; CG around the even-odd matvec):
 *     Mhat^dagger Mhat x = Mhat^dagger b,   x_0 = 0,   one right-hand side, half fields of `parity`.
 * tol = 0 runs exactly max_iter iterations with no host synchronisation inside the loop (all scalars stay on the
 * device, reductions are deterministic fp64 sums); hist_host then holds the RECURSIVELY updated residual norms.
 * tol > 0: the iteration stops when the recursive residual (read back every 8 iterations) is <= tol * |b|; the TRUE
 * residual b - Mhat x is then recomputed with one more operator application and put into the history, and while it is
 * still above tol * |b| and iterations are left the solver is restarted on Mhat e = b - Mhat x and x += e (defect
 * correction), until a round no longer halves the true residual (the working precision's limit, ~1e-6 in fp32):
 * the last history entry is always the true |b - Mhat x| / |b|, so a reported convergence is real.  Exact zeros in a
 * denominator of the recurrence (b = 0, breakdown) give a zero step, never NaN.  *iters_out (may be NULL) receives
 * the iterations done; hist_host (HOST, max_iter + 1 doubles, may be NULL) the relative residuals, k = 0..iters.
 * Workspace (five half fields) is owned by the gauge handle (allocated on first use, reused, released by
 * wd_destroy_gauge; not re-entrant for one handle); the call synchronises the gauge's stream before returning.
 */
int wd_cgnr_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4],
                  int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host);

/* wd_cgnr_schur_block -- the same CGNR for nrhs right-hand sides at once (the set-up and the propagator calculation solve
 * for many sources with the same links): x and b hold nrhs native half fields, the iterations advance in
 * lock step, every operator application is ONE batched launch pair in which a block of links serves all right-hand
 * sides, every right-hand side has its own scalars.  Per right-hand side the arithmetic is that of wd_cgnr_schur with
 * tol = 0 (bit-identical iterates).  tol > 0 stops when EVERY right-hand side's recursive residual is <= tol * |b_r|
 * (no true-residual restarts here).  hist_host: HOST, nrhs * (max_iter + 1) doubles, row r = history of right-hand side r.
 * Workspace 5 * nrhs half fields in the gauge handle. */
int wd_cgnr_schur_block(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int nrhs,
                        int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host);

/* wd_bicgstab_schur -- BiCGstab (van der Vorst) for Mhat x = b, x_0 = 0: the paper's other solver around the
 * even-odd matvec (Table 2).  Same arguments, execution model and workspace as wd_cgnr_schur;
 * one iteration = two Mhat applications; complex inner products summed deterministically in fp64. */
int wd_bicgstab_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4],
                      int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host);

/* wd_gcr_schur -- restarted GCR(restart) for Mhat x = b, x_0 = 0, no preconditioner: the paper's outer Krylov solver
 * ("GCR(8)"), one Mhat application per iteration, modified Gram-Schmidt against the directions of the
 * current cycle.  1 <= restart <= 32.  Otherwise as wd_cgnr_schur (workspace: 2*restart + 2 half fields). */
int wd_gcr_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int precision,
                 int parity, int max_iter, int restart, double tol, int *iters_out, double *hist_host);

/* The preconditioner slot of GCR (the multigrid cycle "is used as a preconditioner for a GCR(8) outer
 * Krylov solver").  precond(ctx, z, r, stream) must enqueue z = K r on `stream` (the gauge's stream, a cudaStream_t as
 * void*) for native half fields z, r of `parity` and return 0; K may differ from call to call (GCR is flexible: the
 * search direction is p_j = K r_j, then q_j = Mhat p_j is orthogonalised as before).  It may call wd_apply_*,
 * wd_restrict / wd_prolong / wd_apply_coarse, but not the wd_*_schur solvers of this gauge (shared workspace).
 * precond == NULL is wd_gcr_schur.  A non-zero return aborts the solve with WD_ERR_CUDA. */
typedef int (*wd_precond_fn)(void *ctx, void *z_half_dev, const void *r_half_dev, void *stream);
int wd_gcr_schur_precond(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int precision,
                         int parity, int max_iter, int restart, double tol, int *iters_out, double *hist_host,
                         wd_precond_fn precond, void *precond_ctx);

/*
 * ---- transfer operators of the adaptive multigrid set-up: eq. (2.7), on 4^4 space-time blocks with
 * the gamma5 = +-1 (sigma3) split of PAPER.md:116; SURVEY.md 8(f) row f3.  Every extent must be a multiple of 4.
 * The nv vectors are nv right-hand sides of ONE native buffer (wd_spinor_bytes(lat, nv, precision)).  Coarse vectors:
 * [bt][bz][by][bx][sigma 0..1][alpha 0..nv-1][re, im] reals of the working precision, wd_coarse_reals(lat, nv) of them.
 */
long long wd_coarse_reals(const wd_lattice *lat, int nv);
/* In place: vecs_native_dev <- orthonormal basis of its restrictions to every (block, chirality), modified
 * Gram-Schmidt in the order alpha = 0..nv-1 (the columns P_{x; xhat, alpha} of eq. (2.7)). */
int wd_block_orthonormalise(const wd_lattice *lat, void *vecs_native_dev, int nv, int precision, void *stream);
/* coarse = P^dagger psi   (psi: one native field). */
int wd_restrict(const wd_lattice *lat, void *coarse_dev, const void *basis_native_dev, const void *psi_native_dev, int nv,
                int precision, void *stream);
/* psi = P coarse. */
int wd_prolong(const wd_lattice *lat, void *psi_native_dev, const void *basis_native_dev, const void *coarse_dev, int nv,
               int precision, void *stream);

/*
 * The coarse operator as an explicit stencil (PAPER.md:82-88 Galerkin form Dhat = P^dagger D P; PAPER.md:116 4^4 blocks
 * x chirality; "the N_V x N_V complex matrix operations needed for the coarse operators").  D couples
 * nearest neighbours, so Dhat couples a block b to itself and its 8 neighbour blocks; with the coarse index
 * i = sigma * nv + alpha (n = 2 nv per block, as in wd_restrict's output) there are nine n x n complex matrices per block
 *   k = 0: A(b);  k = 1 + mu: F_mu(b) (acts on c(b + mu));  k = 5 + mu: B_mu(b) (acts on c(b - mu)),  mu = 0..3 = x,y,z,t
 *   (Dhat c)(b) = A(b) c(b) + sum_mu [ F_mu(b) c(b+mu) + B_mu(b) c(b-mu) ]        periodic coarse lattice of L/4 blocks
 * A hop belongs to F_mu / B_mu when it leaves the block through its +mu / -mu face, whatever block it lands in (coarse
 * extent 1 or 2: coincident neighbour blocks simply add; reading S4).  Device layout of the stencil:
 *   S[block][k][column j][row i][re, im]   (column major) in the working precision; wd_coarse_stencil_reals() reals.
 *
 * wd_build_coarse: stencil from the columns of P (`basis_native_dev`: nv vectors as nv right-hand sides of one native
 * buffer, orthonormalised per block and chirality by wd_block_orthonormalise) and the gauge's links and mass.  The
 * Galerkin products are formed as written (the diagonal term as (4+m) W^dag W, not assumed to be (4+m) 1).  `scratch_dev`:
 * caller-owned, same size as the stencil, overwritten.  Launches on the gauge's stream; deterministic (no atomics).
 * nv <= 32, at most 65535 blocks.  wd_apply_coarse: out[r] = Dhat in[r] for nrhs coarse vectors
 * [rhs][block][sigma][alpha][re, im] (wd_coarse_reals() reals each); out must not overlap in; nv <= 56.
 */
long long wd_coarse_stencil_reals(const wd_lattice *lat, int nv);
int wd_build_coarse(const wd_gauge *gauge, void *stencil_dev, void *scratch_dev, const void *basis_native_dev, double mass,
                    const int dims[4], int nv, int precision);
int wd_apply_coarse(const wd_lattice *lat, void *out_coarse_dev, const void *in_coarse_dev, const void *stencil_dev, int nv,
                    int nrhs, int precision, void *stream);

/* Number of CUDA kernels the library has launched in this process (all handles). */
long long wd_launch_count(void);

/* Message for the last error on this thread ("" if none); static storage, never NULL. */
const char *wd_last_error(void);

/* Release handles.  NULL is a no-op.  A gauge must be destroyed before its lattice is
 * only in the sense that it keeps its own copy of the extents: order does not matter. */
void wd_destroy_gauge(wd_gauge *gauge);
void wd_destroy(wd_lattice *lat);

#ifdef __cplusplus
}
#endif
#endif /* WD_H */
