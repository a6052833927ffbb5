// wd_internal.h -- host-side structures shared by the translation units of libwd.so.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

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
    void *links;      // native links, device (cudaMalloc)
    size_t links_bytes;
    cudaStream_t stream;
    // staging for wd_apply_host (allocated on first use)
    void *stage_canon;   // canonical spinor buffer (input), device
    void *stage_canon_out; // canonical spinor buffer (result), device
    void *stage_in;      // native in
    void *stage_out;     // native out
    size_t stage_bytes;
    // workspace of wd_cgnr_schur (five half fields + reduction scalars), allocated on first use, reused
    void *cg_ws;
    size_t cg_ws_bytes;
    double *cg_sc;
    size_t cg_sc_count;
    cudaStream_t pipe_stream[3]; // copy-in, compute, copy-out streams of the pipelined host path
    cudaEvent_t pipe_event[2 * 16 + 2];
};

namespace wd {

struct ApplyArgs {
    void *out;
    const void *in;
    const void *links;
    int dims[4];
    long long V;
    double mass;
    int nrhs;
    int precision;
    int recon;
    cudaStream_t stream;
    int dagger;                     // site kernel only: apply D^dagger = gamma5 D gamma5 instead of D
    int tgauge;                     // links are in temporal gauge (U_t = 1 for t < Lt-1): kernels may skip them
    long long site_begin, site_end; // site kernel only: apply on [site_begin, site_end); 0,0 = whole lattice
};

void count_launch(int n = 1);

// one thread per site, any extents >= 1
cudaError_t launch_site(const ApplyArgs &a);
// shared-memory tiled kernel; supported() is a pure host-side predicate
bool tile_supported(const ApplyArgs &a);
cudaError_t launch_tile(const ApplyArgs &a);
// tile kernel with every global read staged through shared memory by cp.async (fp32)
bool stage_supported(const ApplyArgs &a);
cudaError_t launch_stage(const ApplyArgs &a);

// site range [site0, site0 + nsites) of every right-hand side; site0 a multiple of 128; nsites < 0 = all
cudaError_t launch_pack_spinor(void *native, const void *canonical, long long V, int nrhs, int precision,
                               cudaStream_t s, long long site0 = 0, long long nsites = -1);
cudaError_t launch_unpack_spinor(void *canonical, const void *native, long long V, int nrhs, int precision,
                                 cudaStream_t s, long long site0 = 0, long long nsites = -1);
// red/black blocks (wd_dslash_eo.cu): out_p = alpha * xin_p + beta * hops(in_q); half-field <-> canonical copies
cudaError_t launch_eo(const ApplyArgs &a, const void *xin, double alpha, double beta, int parity, bool dagger = false,
                      double *norm_part = nullptr);
// CGNR for Mhat x = b on one parity (wd_cg.cu); shape carries dims, V, precision, recon, links, stream
int cgnr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
               double tol, int *iters_out, double *hist_host, cudaError_t *err);
int bicgstab_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter,
                   double tol, int *iters_out, double *hist_host, cudaError_t *err);
int gcr_schur(wd_gauge *g, const ApplyArgs &shape, void *x, const void *b, double mass, int parity, int max_iter, int restart,
              double tol, int *iters_out, double *hist_host, cudaError_t *err);
// transfer operators of the multigrid set-up (wd_transfer.cu)
cudaError_t launch_transfer(int what, void *a, const void *b, const void *c, const int dims[4], long long V, int nv,
                            int precision, cudaStream_t s);
cudaError_t launch_parity_copy(void *native, void *canon, const int dims[4], long long V, int nrhs, int precision,
                               int parity, bool to_native, cudaStream_t s);
cudaError_t launch_pack_links(void *native, const void *canonical, long long V, int precision, int recon,
                              cudaStream_t s);
cudaError_t launch_check_temporal_gauge(const void *links, const int dims[4], long long V, int precision, int recon,
                                        int *flag_dev, cudaStream_t s);
size_t native_link_bytes(long long V, int precision, int recon);

} // namespace wd
