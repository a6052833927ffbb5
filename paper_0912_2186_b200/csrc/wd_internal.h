// wd_internal.h -- host-side structures shared by the translation units of libwd.so.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

namespace wd {
// Tuning variables: read from the environment ONCE, at wd_load_gauge, into the gauge handle;
// wd_set_tuning changes one of them later.  A negative value means "not set: use the launcher's default".
struct Tuning {
    int tile_ty = -1, tile_tz = -1; // WD_TILE_SHAPE=ty,tz
    int tile_tc = -1;               // WD_TILE_TC      slices per t-chunk
    int tile_nchunk = -1;           // WD_TILE_NCHUNK  t-chunks (overrides tile_tc)
    int tile_nrb = -1;              // WD_TILE_NRB     right-hand sides per CTA of the multi-RHS kernel
    int mrhs_patch = -1;            // WD_MRHS_PATCH   side of the tile-column patch of the multi-RHS block order (0 = off)
    int stage_no_mrhs = -1;         // WD_STAGE_NO_MRHS  1 = run several right-hand sides through the single-RHS staged kernel
    int site_slab_mb = -1;          // WD_SITE_SLAB_MB  link slab of the site kernel's multi-RHS block order
    int host_no_pipeline = -1;      // WD_HOST_NO_PIPELINE  1 = one-stream wd_apply_host
    int mrhs_no_tail = -1;          // WD_MRHS_NO_TAIL  1 = no shortened t-chunks in the last wave of the multi-RHS kernel
    int mrhs_bulk = -1;             // WD_MRHS_BULK     1 = stage the links of the multi-RHS kernel by cp.async.bulk (A/B variant)
    int host_nslab = -1;            // WD_HOST_NSLAB    slabs of the pipelined wd_apply_host (3..32, default 16)
    int stage_bulk = -1;            // WD_STAGE_BULK    staged kernel on Lx = 32: 1 = bulk-copy member (wd_dslash_stage_bulk.cu), 0 = per-thread cp.async
    int mrhs_reg = -1;              // WD_MRHS_REG      multi-RHS member with the links in registers (wd_dslash_rloop.cu): 0 = never, 1 = plain-load
                                    //                  member, 2 = ring member (Lx = 32; else plain-load), 3 = ring member with uniform roles;
                                    //                  unset: 8-real links on Lx = 32 only (uniform-role ring)
    int mrhs_rgrp = -1;             // WD_MRHS_RGRP     right-hand sides per group of that member (default: what two CTAs per SM allow)
};
void tuning_from_env(Tuning &t);
int tuning_set(Tuning &t, const char *name, int value); // 0 = ok, -1 = unknown name
const Tuning &default_tuning();
} // namespace wd

struct wd_lattice {
    unsigned magic;
    int dims[4];      // Lx, Ly, Lz, Lt
    long long V;
};

struct wd_gauge {
    unsigned magic;
    int dims[4];
    long long V;
    int precision;    // 32 / 64
    int recon;        // 18 / 12
    int kernel;       // wd_kernel selector
    int tgauge;       // wd_set_temporal_gauge: U_t(x,t) = 1 for t < Lt-1 (verified when set)
    wd::Tuning tune;  // tuning variables, read once at wd_load_gauge
    int pipe_ready;   // the three streams and 34 events of the pipelined host path all exist
    void *links;      // native links, device (cudaMalloc)
    size_t links_bytes;
    void *links_eo;   // the same link records ordered by parity (even sites, then odd sites; record index lex / 2): what the
                      // red/black kernels read; built from `links` on the first red/black call, NULL until then
    cudaStream_t stream;
    // staging for wd_apply_host (allocated on first use)
    void *stage_canon;   // canonical spinor buffer (input), device
    void *stage_canon_out; // canonical spinor buffer (result), device
    void *stage_in;      // native in
    void *stage_out;     // native out
    size_t stage_bytes;
    // workspace of wd_cgnr_schur (five half fields + reduction scalars), allocated on first use, reused
    void *rf_ws;         // workspace of the true-residual control around the solvers (three half fields), on first use
    size_t rf_ws_bytes;
    void *cg_ws;
    size_t cg_ws_bytes;
    double *cg_sc;
    size_t cg_sc_count;
    cudaStream_t pipe_stream[3]; // copy-in, compute, copy-out streams of the pipelined host path
    cudaEvent_t pipe_event[2 * 32 + 2];
};

namespace wd {

struct ApplyArgs {
    void *out;
    const void *in;
    const void *links;
    const void *links_eo;           // red/black kernels: parity-ordered copy of the links (wd_gauge::links_eo)
    int dims[4];
    long long V;
    double mass;
    int nrhs;
    int precision;
    int recon;
    cudaStream_t stream;
    const Tuning *tune;             // never null inside the launchers (default_tuning() when the caller has none)
    int dagger;                     // apply D^dagger = gamma5 D gamma5 instead of D (site and single-RHS staged kernels)
    int tgauge;                     // links are in temporal gauge (U_t = 1 for t < Lt-1): kernels may skip them
    long long site_begin, site_end; // site kernel only: apply on [site_begin, site_end); 0,0 = whole lattice
};

void count_launch(int n = 1);

// one thread per site, any extents >= 1
cudaError_t launch_site(const ApplyArgs &a);
// t-marching tile kernel with every global read staged through shared memory by cp.async (fp32 and fp64);
// stage_supported() is a pure host-side predicate
bool stage_supported(const ApplyArgs &a);
cudaError_t launch_stage(const ApplyArgs &a);
// cudaFuncAttributeMaxDynamicSharedMemorySize is per device: set it once per (kernel, device), thread-safe
cudaError_t ensure_dynamic_smem(const void *kernel, size_t bytes, size_t *per_device_cache);
int sm_count(); // multiprocessors of the current device (cached per device)

// site range [site0, site0 + nsites) of every right-hand side; site0 a multiple of 128; nsites < 0 = all
cudaError_t launch_pack_spinor(void *native, const void *canonical, long long V, int nrhs, int precision,
                               cudaStream_t s, long long site0 = 0, long long nsites = -1);
cudaError_t launch_unpack_spinor(void *canonical, const void *native, long long V, int nrhs, int precision,
                                 cudaStream_t s, long long site0 = 0, long long nsites = -1);
// red/black blocks (wd_dslash_eo.cu): out_p = alpha * xin_p + beta * hops(in_q); half-field <-> canonical copies
// the same in half storage (wd_half.cu): fields of one parity in the half layout over lex / 2; no epilogues
cudaError_t launch_eo_half(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger);
cudaError_t launch_parity_copy_half(void *native, void *canon, const int dims[4], long long V, int nrhs, int parity, bool to_native,
                                    cudaStream_t s);
// wd_noalloc.cu: Mhat with its intermediate field in a static device array (no allocation anywhere)
size_t schur_static_need(const ApplyArgs &a);
cudaError_t launch_schur_static(const ApplyArgs &a, int parity);
// parity-ordered link records: record cb of parity p sits at p * eo_links_half_bytes + native position of `cb`
size_t eo_links_half_bytes(long long V, int precision, int recon);
cudaError_t launch_links_to_eo(void *links_eo, const void *links, const int dims[4], long long V, int precision, int recon,
                               cudaStream_t s);
cudaError_t launch_eo(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger = false,
                      double *norm_part = nullptr, const void *dot_y = nullptr, double *dot_part = nullptr);
// CGNR for Mhat x = b on one parity (wd_cg.cu); shape carries dims, V, precision, recon, links, stream
int cgnr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
               double tol, int *iters_out, double *hist_host, cudaError_t *err);
int bicgstab_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
                   double tol, int *iters_out, double *hist_host, cudaError_t *err);
int cgnr_schur_block(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int nrhs, int max_iter,
                     double tol, int *iters_out, double *hist_host, cudaError_t *err);
// preconditioner slot of GCR: z = K r, enqueued on `stream` (same type as wd_precond_fn in wd.h)
typedef int (*precond_fn)(void *ctx, void *z_half_dev, const void *r_half_dev, void *stream);
int gcr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter, int restart,
              double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond = nullptr, void *ctx = nullptr);
// the public solvers: kind 0 = CGNR, 1 = BiCGstab, 2 = GCR(restart); tol > 0 adds true-residual control (wd_cg.cu)
int solve_schur(wd_gauge *g, const ApplyArgs &shape, int kind, void *x, const void *b, double mass, int parity, int max_iter,
                int restart, double tol, int *iters_out, double *hist_host, cudaError_t *err, precond_fn precond = nullptr,
                void *ctx = nullptr);
// transfer operators of the multigrid set-up (wd_transfer.cu)
cudaError_t launch_transfer(int what, void *a, const void *b, const void *c, const int dims[4], long long V, int nv,
                            int precision, cudaStream_t s);
// explicit coarse operator (wd_coarse.cu): build the 9-point stencil from the basis and the links; apply it
cudaError_t launch_coarse_build(void *S, void *part, const void *W, const void *links, const int dims[4], long long V, int nv,
                                double mass, int precision, int recon, cudaStream_t s);
cudaError_t launch_coarse_apply(void *out, const void *in, const void *S, const int dims[4], int nv, int nrhs, int precision,
                                cudaStream_t s);
// half-precision storage (wd_half.cu): fp32 arithmetic on binary16 fields; canonical side is float32
cudaError_t launch_half(const ApplyArgs &a);
bool half_stage_supported(const ApplyArgs &a); // staged member (wd_half_stage.cu): Lx a power of two, tiles of <= 128 sites
cudaError_t launch_half_stage(const ApplyArgs &a);
cudaError_t launch_spinor_half(void *native, void *canonical, long long V, int nrhs, bool to_native, cudaStream_t s);
cudaError_t launch_pack_links_half(void *native, const void *canonical, long long V, int recon, cudaStream_t s, int *bad_dev);
cudaError_t launch_parity_copy(void *native, void *canon, const int dims[4], long long V, int nrhs, int precision,
                               int parity, bool to_native, cudaStream_t s);
cudaError_t launch_pack_links(void *native, const void *canonical, long long V, int precision, int recon,
                              cudaStream_t s, int *bad_dev = nullptr);
cudaError_t launch_check_temporal_gauge(const void *links, const int dims[4], long long V, int precision, int recon,
                                        int *flag_dev, cudaStream_t s);
size_t native_link_bytes(long long V, int precision, int recon);

} // namespace wd
