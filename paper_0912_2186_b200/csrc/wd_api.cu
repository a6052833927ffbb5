// wd_api.cu -- the extern "C" boundary declared in include/wd.h: argument validation, handle
// management and kernel dispatch.  No arithmetic of the method lives here.
#include <atomic>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/wd.h"
#include "wd_internal.h"
#include "wd_layout.cuh"

namespace {

constexpr unsigned LATTICE_MAGIC = 0x57444c41u; // "WDLA"
constexpr unsigned GAUGE_MAGIC = 0x57444741u;   // "WDGA"

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    return fail(WD_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

bool valid_precision(int p) { return p == WD_FP32 || p == WD_FP64; }                  // arithmetic precisions
bool valid_storage(int p) { return p == WD_FP16 || p == WD_FP32 || p == WD_FP64; }    // + half-precision storage
// bytes of one real of the CANONICAL arrays (half-precision storage exchanges float32 canonical fields)
size_t canon_real_bytes(int p) { return p == WD_FP64 ? 8 : 4; }
// bytes per site and right-hand side of a NATIVE spinor field (half: 24 binary16 ratios + one float32 scale)
size_t native_site_bytes(int p) { return p == WD_FP16 ? 52 : p == WD_FP32 ? 96 : 192; }
bool valid_recon(int r) { return r == WD_RECON_18 || r == WD_RECON_12 || r == WD_RECON_8; }

// volume with overflow guard; returns -1 on bad extents
long long checked_volume(const int dims[4])
{
    long long v = 1;
    for (int d = 0; d < 4; ++d) {
        if (dims[d] < 1) return -1;
        v *= dims[d];
        if (v > (1LL << 40)) return -1;
    }
    return v;
}

bool overlap(const void *a, size_t abytes, const void *b, size_t bbytes)
{
    const uintptr_t pa = (uintptr_t)a, pb = (uintptr_t)b;
    return pa < pb + bbytes && pb < pa + abytes;
}

int check_apply_args(const void *out, const void *in, const wd_gauge *g, const int dims[4], int nrhs, int precision,
                     bool allow_half = false)
{
    if (!out || !in || !g || !dims) return fail(WD_ERR_NULL, "wd_apply: NULL argument");
    if (g->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_apply: not a live wd_gauge handle");
    if (!valid_storage(precision)) return fail(WD_ERR_PRECISION, "wd_apply: precision %d is not 16, 32 or 64", precision);
    if (precision == WD_FP16 && !allow_half)
        return fail(WD_ERR_PRECISION, "half-precision storage is taken by wd_apply, wd_apply_dagger, wd_apply_hop and wd_apply_schur* only");
    if (precision != g->precision)
        return fail(WD_ERR_PRECISION, "wd_apply: precision %d but gauge was loaded in %d", precision, g->precision);
    for (int d = 0; d < 4; ++d)
        if (dims[d] != g->dims[d])
            return fail(WD_ERR_DIMS, "wd_apply: dims[%d]=%d but gauge lattice has %d", d, dims[d], g->dims[d]);
    if (nrhs < 1) return fail(WD_ERR_NRHS, "wd_apply: nrhs=%d", nrhs);
    return WD_OK;
}

} // namespace

namespace wd {
void count_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

static int env_int(const char *name)
{
    const char *e = getenv(name);
    if (!e || !*e) return -1;
    const int v = atoi(e);
    return v < 0 ? -1 : v;
}

void tuning_from_env(Tuning &t)
{
    t = Tuning();
    if (const char *e = getenv("WD_TILE_SHAPE")) {
        int ty = 0, tz = 0;
        if (sscanf(e, "%d,%d", &ty, &tz) == 2 && ty >= 1 && tz >= 1) {
            t.tile_ty = ty;
            t.tile_tz = tz;
        }
    }
    t.tile_tc = env_int("WD_TILE_TC");
    t.tile_nchunk = env_int("WD_TILE_NCHUNK");
    t.tile_nrb = env_int("WD_TILE_NRB");
    t.mrhs_patch = env_int("WD_MRHS_PATCH");
    t.stage_no_mrhs = env_int("WD_STAGE_NO_MRHS");
    t.site_slab_mb = env_int("WD_SITE_SLAB_MB");
    t.host_no_pipeline = env_int("WD_HOST_NO_PIPELINE");
    t.mrhs_no_tail = env_int("WD_MRHS_NO_TAIL");
    t.host_nslab = env_int("WD_HOST_NSLAB");
    t.mrhs_bulk = env_int("WD_MRHS_BULK");
    t.stage_bulk = env_int("WD_STAGE_BULK");
    t.mrhs_reg = env_int("WD_MRHS_REG");
    t.mrhs_rgrp = env_int("WD_MRHS_RGRP");
}

int tuning_set(Tuning &t, const char *name, int value)
{
    struct { const char *n; int Tuning::*f; } tab[] = {
        {"tile_ty", &Tuning::tile_ty}, {"tile_tz", &Tuning::tile_tz}, {"tile_tc", &Tuning::tile_tc},
        {"tile_nchunk", &Tuning::tile_nchunk}, {"tile_nrb", &Tuning::tile_nrb}, {"mrhs_patch", &Tuning::mrhs_patch},
        {"stage_no_mrhs", &Tuning::stage_no_mrhs}, {"site_slab_mb", &Tuning::site_slab_mb},
        {"host_no_pipeline", &Tuning::host_no_pipeline}, {"mrhs_no_tail", &Tuning::mrhs_no_tail},
        {"host_nslab", &Tuning::host_nslab}, {"mrhs_bulk", &Tuning::mrhs_bulk},
        {"mrhs_reg", &Tuning::mrhs_reg}, {"stage_bulk", &Tuning::stage_bulk}, {"mrhs_rgrp", &Tuning::mrhs_rgrp}};
    for (auto &e : tab)
        if (!strcmp(name, e.n)) {
            t.*(e.f) = value < 0 ? -1 : value;
            return 0;
        }
    return -1;
}

const Tuning &default_tuning()
{
    static const Tuning t;
    return t;
}
} // namespace wd

extern "C" {

int wd_create_lattice(const int dims[4], wd_lattice **lat)
{
    if (!dims || !lat) return fail(WD_ERR_NULL, "wd_create_lattice: NULL argument");
    *lat = nullptr;
    const long long V = checked_volume(dims);
    if (V < 0) return fail(WD_ERR_DIMS, "wd_create_lattice: bad extents %d %d %d %d", dims[0], dims[1], dims[2], dims[3]);
    wd_lattice *l = new (std::nothrow) wd_lattice;
    if (!l) return fail(WD_ERR_ALLOC, "wd_create_lattice: out of host memory");
    l->magic = LATTICE_MAGIC;
    for (int d = 0; d < 4; ++d) l->dims[d] = dims[d];
    l->V = V;
    *lat = l;
    return WD_OK;
}

int wd_lattice_dims(const wd_lattice *lat, int dims_out[4])
{
    if (!lat || !dims_out) return fail(WD_ERR_NULL, "wd_lattice_dims: NULL argument");
    if (lat->magic != LATTICE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_lattice_dims: not a live wd_lattice handle");
    for (int d = 0; d < 4; ++d) dims_out[d] = lat->dims[d];
    return WD_OK;
}

long long wd_lattice_volume(const wd_lattice *lat)
{
    if (!lat || lat->magic != LATTICE_MAGIC) return -1;
    return lat->V;
}

size_t wd_spinor_bytes(const wd_lattice *lat, int nrhs, int precision)
{
    if (!lat || lat->magic != LATTICE_MAGIC || nrhs < 1 || !valid_storage(precision)) return 0;
    return (size_t)nrhs * (size_t)wd::padded_volume(lat->V) * native_site_bytes(precision);
}

int wd_load_gauge(const wd_lattice *lat, const void *links_canonical_dev, int precision, int recon, void *stream,
                  wd_gauge **gauge)
{
    if (!lat || !links_canonical_dev || !gauge) return fail(WD_ERR_NULL, "wd_load_gauge: NULL argument");
    *gauge = nullptr;
    if (lat->magic != LATTICE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_load_gauge: not a live wd_lattice handle");
    if (!valid_storage(precision)) return fail(WD_ERR_PRECISION, "wd_load_gauge: precision %d is not 16, 32 or 64", precision);
    if (!valid_recon(recon)) return fail(WD_ERR_RECON, "wd_load_gauge: recon %d is not 18, 12 or 8", recon);
    wd_gauge *g = new (std::nothrow) wd_gauge;
    if (!g) return fail(WD_ERR_ALLOC, "wd_load_gauge: out of host memory");
    memset(g, 0, sizeof(*g));
    g->magic = GAUGE_MAGIC;
    for (int d = 0; d < 4; ++d) g->dims[d] = lat->dims[d];
    g->V = lat->V;
    g->precision = precision;
    g->recon = recon;
    g->kernel = WD_KERNEL_AUTO;
    g->tune = wd::Tuning();
    wd::tuning_from_env(g->tune); // the one place the environment is read
    g->stream = (cudaStream_t)stream;
    g->links_bytes = wd::native_link_bytes(g->V, precision, recon);
    cudaError_t e = cudaMalloc(&g->links, g->links_bytes);
    if (e != cudaSuccess) {
        delete g;
        return e == cudaErrorMemoryAllocation ? fail(WD_ERR_ALLOC, "wd_load_gauge: cudaMalloc failed")
                                              : cuda_fail(e, "wd_load_gauge: cudaMalloc");
    }
    int *bad = nullptr, hbad = 0;
    if (recon == WD_RECON_8) { // the 8-real parametrisation cannot hold a link with U01 = U02 = 0: checked (one sync)
        e = cudaMalloc(&bad, sizeof(int));
        if (e == cudaSuccess) e = cudaMemsetAsync(bad, 0, sizeof(int), g->stream);
    }
    if (e == cudaSuccess)
        e = precision == WD_FP16 ? wd::launch_pack_links_half(g->links, links_canonical_dev, g->V, recon, g->stream, bad)
                                 : wd::launch_pack_links(g->links, links_canonical_dev, g->V, precision, recon, g->stream, bad);
    if (e == cudaSuccess && bad) {
        e = cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, g->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
    }
    cudaFree(bad);
    if (e != cudaSuccess || hbad) {
        cudaFree(g->links);
        delete g;
        if (hbad) return fail(WD_ERR_RECON, "wd_load_gauge: a link with U[0][1] = U[0][2] = 0 cannot be stored in 8 reals");
        return cuda_fail(e, "wd_load_gauge: pack kernel");
    }
    *gauge = g;
    return WD_OK;
}

int wd_set_stream(wd_gauge *gauge, void *stream)
{
    if (!gauge) return fail(WD_ERR_NULL, "wd_set_stream: NULL gauge");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_set_stream: not a live wd_gauge handle");
    // work already queued on the old stream (the link conversion of wd_load_gauge, earlier applies) comes first
    if ((cudaStream_t)stream != gauge->stream) {
        cudaEvent_t ev;
        cudaError_t e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventRecord(ev, gauge->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent((cudaStream_t)stream, ev, 0);
        if (e == cudaSuccess) e = cudaEventDestroy(ev);
        if (e != cudaSuccess) return cuda_fail(e, "wd_set_stream");
    }
    gauge->stream = (cudaStream_t)stream;
    return WD_OK;
}

int wd_set_tuning(wd_gauge *gauge, const char *name, int value)
{
    if (!gauge || !name) return fail(WD_ERR_NULL, "wd_set_tuning: NULL argument");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_set_tuning: not a live wd_gauge handle");
    if (wd::tuning_set(gauge->tune, name, value)) return fail(WD_ERR_MISMATCH, "wd_set_tuning: unknown variable '%s'", name);
    return WD_OK;
}

int wd_set_temporal_gauge(wd_gauge *gauge, int on)
{
    if (!gauge) return fail(WD_ERR_NULL, "wd_set_temporal_gauge: NULL gauge");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_set_temporal_gauge: not a live wd_gauge handle");
    if (!on) {
        gauge->tgauge = 0;
        return WD_OK;
    }
    if (gauge->precision == WD_FP16) return fail(WD_ERR_PRECISION, "wd_set_temporal_gauge: not for half-precision storage");
    if (gauge->recon == WD_RECON_8)
        return fail(WD_ERR_RECON, "wd_set_temporal_gauge: unit links cannot be stored in 8 reals (load the gauge with recon 18 or 12)");
    int *flag = nullptr, h = 0;
    cudaError_t e = cudaMalloc(&flag, sizeof(int));
    if (e != cudaSuccess) return cuda_fail(e, "wd_set_temporal_gauge: cudaMalloc");
    e = cudaMemsetAsync(flag, 0, sizeof(int), gauge->stream);
    if (e == cudaSuccess) e = wd::launch_check_temporal_gauge(gauge->links, gauge->dims, gauge->V, gauge->precision, gauge->recon, flag, gauge->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, gauge->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(gauge->stream);
    cudaFree(flag);
    if (e != cudaSuccess) return cuda_fail(e, "wd_set_temporal_gauge");
    if (h) return fail(WD_ERR_MISMATCH, "wd_set_temporal_gauge: some U_t(x,t), t < Lt-1, is not the unit matrix");
    gauge->tgauge = 1;
    return WD_OK;
}

int wd_set_kernel(wd_gauge *gauge, int kernel)
{
    if (!gauge) return fail(WD_ERR_NULL, "wd_set_kernel: NULL gauge");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_set_kernel: not a live wd_gauge handle");
    if (kernel != WD_KERNEL_AUTO && kernel != WD_KERNEL_SITE && kernel != WD_KERNEL_STAGE)
        return fail(WD_ERR_MISMATCH, "wd_set_kernel: unknown kernel %d", kernel);
    if (kernel == WD_KERNEL_STAGE && gauge->precision == WD_FP16) {
        wd::ApplyArgs a{};
        for (int d = 0; d < 4; ++d) a.dims[d] = gauge->dims[d];
        a.V = gauge->V;
        if (!wd::half_stage_supported(a))
            return fail(WD_ERR_MISMATCH, "wd_set_kernel: the staged half-precision kernel does not support this lattice");
        gauge->kernel = kernel;
        return WD_OK;
    }
    if (kernel == WD_KERNEL_STAGE) {
        wd::ApplyArgs a{};
        for (int d = 0; d < 4; ++d) a.dims[d] = gauge->dims[d];
        a.V = gauge->V;
        a.nrhs = 1;
        a.precision = gauge->precision;
        a.recon = gauge->recon;
        a.tune = &gauge->tune;
        if (!wd::stage_supported(a))
            return fail(WD_ERR_MISMATCH, "wd_set_kernel: staged kernel does not support lattice %d %d %d %d", a.dims[0],
                        a.dims[1], a.dims[2], a.dims[3]);
    }
    gauge->kernel = kernel;
    return WD_OK;
}

// native: wd_spinor_bytes() bytes (padded volume); canonical: nrhs * V * 24 reals
static int check_pack_args(const char *who, const wd_lattice *lat, const void *native, const void *canonical, int nrhs,
                           int precision)
{
    const void *a = native, *b = canonical;
    if (!lat || !a || !b) return fail(WD_ERR_NULL, "%s: NULL argument", who);
    if (lat->magic != LATTICE_MAGIC) return fail(WD_ERR_MISMATCH, "%s: not a live wd_lattice handle", who);
    if (!valid_storage(precision)) return fail(WD_ERR_PRECISION, "%s: precision %d is not 16, 32 or 64", who, precision);
    if (nrhs < 1) return fail(WD_ERR_NRHS, "%s: nrhs=%d", who, nrhs);
    const size_t cbytes = (size_t)nrhs * (size_t)lat->V * 24 * canon_real_bytes(precision);
    if (overlap(native, wd_spinor_bytes(lat, nrhs, precision), canonical, cbytes))
        return fail(WD_ERR_ALIAS, "%s: buffers overlap", who);
    return WD_OK;
}

int wd_pack_spinor(const wd_lattice *lat, void *native_dev, const void *canonical_dev, int nrhs, int precision,
                   void *stream)
{
    int rc = check_pack_args("wd_pack_spinor", lat, native_dev, canonical_dev, nrhs, precision);
    if (rc) return rc;
    cudaError_t e = precision == WD_FP16
                        ? wd::launch_spinor_half(native_dev, const_cast<void *>(canonical_dev), lat->V, nrhs, true, (cudaStream_t)stream)
                        : wd::launch_pack_spinor(native_dev, canonical_dev, lat->V, nrhs, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_pack_spinor");
}

int wd_unpack_spinor(const wd_lattice *lat, void *canonical_dev, const void *native_dev, int nrhs, int precision,
                     void *stream)
{
    int rc = check_pack_args("wd_unpack_spinor", lat, native_dev, canonical_dev, nrhs, precision);
    if (rc) return rc;
    cudaError_t e = precision == WD_FP16
                        ? wd::launch_spinor_half(const_cast<void *>(native_dev), canonical_dev, lat->V, nrhs, false, (cudaStream_t)stream)
                        : wd::launch_unpack_spinor(canonical_dev, native_dev, lat->V, nrhs, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_unpack_spinor");
}

// which kernel WD_KERNEL_AUTO resolves to, by measurement (profiles/): the staged kernels (single- and multi-RHS
// members) on every lattice they can tile that has at least one wave of tiles; everything else -> site kernel
static int auto_kernel(const wd::ApplyArgs &a)
{
    if (a.precision == WD_FP16) // half-precision storage: wd_half_stage.cu on large lattices it can tile, else wd_half.cu
        return (a.V >= (1LL << 18) && wd::half_stage_supported(a)) ? WD_KERNEL_STAGE : WD_KERNEL_SITE;
    const bool big = a.V >= (1LL << 18);
    if (big && wd::stage_supported(a)) return WD_KERNEL_STAGE;
    return WD_KERNEL_SITE;
}

static wd::ApplyArgs shape_args(const wd_gauge *g, int nrhs)
{
    wd::ApplyArgs a{};
    for (int d = 0; d < 4; ++d) a.dims[d] = g->dims[d];
    a.V = g->V;
    a.nrhs = nrhs;
    a.precision = g->precision;
    a.recon = g->recon;
    a.tgauge = g->tgauge;
    a.tune = &g->tune;
    a.links_eo = g->links_eo;
    return a;
}

static int dispatch_apply(void *out, const void *in, const wd_gauge *g, double mass, int nrhs, int dagger = 0)
{
    wd::ApplyArgs a{};
    a.out = out;
    a.in = in;
    a.links = g->links;
    for (int d = 0; d < 4; ++d) a.dims[d] = g->dims[d];
    a.V = g->V;
    a.mass = mass;
    a.nrhs = nrhs;
    a.precision = g->precision;
    a.recon = g->recon;
    a.tgauge = g->tgauge;
    a.tune = &g->tune;
    a.stream = g->stream;
    a.dagger = dagger;
    cudaError_t e;
    if (g->precision == WD_FP16) {
        const int k = g->kernel == WD_KERNEL_AUTO ? auto_kernel(a) : g->kernel;
        if (k == WD_KERNEL_STAGE && !wd::half_stage_supported(a)) return fail(WD_ERR_MISMATCH, "wd_apply: staged kernel cannot take this call");
        e = k == WD_KERNEL_STAGE ? wd::launch_half_stage(a) : wd::launch_half(a);
    }
    else if (g->kernel == WD_KERNEL_SITE)
        e = wd::launch_site(a);
    else if (g->kernel == WD_KERNEL_STAGE) {
        if (!wd::stage_supported(a)) return fail(WD_ERR_MISMATCH, "wd_apply: staged kernel cannot take this call");
        e = wd::launch_stage(a);
    } else
        e = auto_kernel(a) == WD_KERNEL_STAGE ? wd::launch_stage(a) : wd::launch_site(a);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_apply: kernel launch");
}

int wd_apply(void *out_native_dev, const void *in_native_dev, const wd_gauge *gauge, double mass, const int dims[4],
             int nrhs, int precision)
{
    int rc = check_apply_args(out_native_dev, in_native_dev, gauge, dims, nrhs, precision, true);
    if (rc) return rc;
    const size_t bytes = (size_t)nrhs * (size_t)wd::padded_volume(gauge->V) * native_site_bytes(precision);
    if (overlap(out_native_dev, bytes, in_native_dev, bytes)) return fail(WD_ERR_ALIAS, "wd_apply: out and in overlap");
    if (((uintptr_t)out_native_dev | (uintptr_t)in_native_dev) & 15)
        return fail(WD_ERR_MISMATCH, "wd_apply: buffers must be 16-byte aligned");
    return dispatch_apply(out_native_dev, in_native_dev, gauge, mass, nrhs);
}

int wd_apply_dagger(void *out_native_dev, const void *in_native_dev, const wd_gauge *gauge, double mass, const int dims[4],
                    int nrhs, int precision)
{
    int rc = check_apply_args(out_native_dev, in_native_dev, gauge, dims, nrhs, precision, true);
    if (rc) return rc;
    const size_t bytes = (size_t)nrhs * (size_t)wd::padded_volume(gauge->V) * native_site_bytes(precision);
    if (overlap(out_native_dev, bytes, in_native_dev, bytes)) return fail(WD_ERR_ALIAS, "wd_apply_dagger: out and in overlap");
    if (((uintptr_t)out_native_dev | (uintptr_t)in_native_dev) & 15)
        return fail(WD_ERR_MISMATCH, "wd_apply_dagger: buffers must be 16-byte aligned");
    return dispatch_apply(out_native_dev, in_native_dev, gauge, mass, nrhs, 1);
}

// the same `width` bytes of each of `rows` right-hand sides (pitch `pitch` on both sides); one right-hand side is a plain
// linear copy
static cudaError_t copy_rows(char *dst, const char *src, size_t pitch, size_t width, int rows, cudaMemcpyKind kind,
                             cudaStream_t st)
{
    if (rows == 1) return cudaMemcpyAsync(dst, src, width, kind, st);
    return cudaMemcpy2DAsync(dst, pitch, src, pitch, width, rows, kind, st);
}

int wd_apply_host(void *out_canonical_host, const void *in_canonical_host, wd_gauge *gauge, double mass,
                  const int dims[4], int nrhs, int precision)
{
    int rc = check_apply_args(out_canonical_host, in_canonical_host, gauge, dims, nrhs, precision);
    if (rc) return rc;
    wd_gauge *g = gauge;
    const size_t bytes = (size_t)nrhs * (size_t)g->V * 24 * (precision == WD_FP32 ? 4 : 8); // canonical
    const size_t nbytes = (size_t)nrhs * (size_t)wd::padded_volume(g->V) * 24 * (precision == WD_FP32 ? 4 : 8); // native
    if (g->stage_bytes < nbytes) {
        void **bufs[4] = {&g->stage_canon, &g->stage_canon_out, &g->stage_in, &g->stage_out};
        for (void **b : bufs) {
            cudaFree(*b);
            *b = nullptr;
        }
        g->stage_bytes = 0;
        cudaError_t e = cudaSuccess;
        for (void **b : bufs)
            if (e == cudaSuccess) e = cudaMalloc(b, nbytes);
        if (e != cudaSuccess) {
            for (void **b : bufs) {
                cudaFree(*b);
                *b = nullptr;
            }
            cudaGetLastError();
            return fail(WD_ERR_ALLOC, "wd_apply_host: cudaMalloc of %zu staging bytes failed", 4 * nbytes);
        }
        g->stage_bytes = nbytes;
    }
    cudaStream_t s = g->stream;
    const size_t w = precision == WD_FP32 ? 4 : 8;
    const long long S3 = (long long)g->dims[0] * g->dims[1] * g->dims[2];
    const int Lt = g->dims[3];
    cudaError_t e;

    // ---- pipelined path: the lattice is cut into up to 32 slabs of whole time slices; the slabs are copied in on one
    // stream; packing, D (site kernel on a range of time slices) and unpacking run on a second as the slabs land; the
    // results go home on a third, so the host->device and device->host transfers overlap (PCIe is full duplex) ----
    // (the event arrays of wd_gauge hold 32; more slabs = shorter pipeline fill and drain but more launches: measured 16 best)
    int nslab = g->tune.host_nslab >= 3 ? g->tune.host_nslab : 16;
    if (nslab > 32) nslab = 32;
    if (nslab > Lt) nslab = Lt;
    const bool pipelined = nslab >= 3 && S3 % 128 == 0 && bytes >= (8u << 20) && g->tune.host_no_pipeline <= 0;
    if (pipelined) {
        if (!g->pipe_ready) { // all 3 streams and 34 events, or none
            e = cudaSuccess;
            for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaStreamCreateWithFlags(&g->pipe_stream[i], cudaStreamNonBlocking);
            for (auto &ev : g->pipe_event)
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e != cudaSuccess) {
                for (auto &st : g->pipe_stream) {
                    if (st) cudaStreamDestroy(st);
                    st = nullptr;
                }
                for (auto &ev : g->pipe_event) {
                    if (ev) cudaEventDestroy(ev);
                    ev = nullptr;
                }
                return cuda_fail(e, "wd_apply_host: stream / event create");
            }
            g->pipe_ready = 1;
        }
        // on any error below: drain the three private streams before returning, so that no copy or kernel still
        // touches the caller's host buffers after the call has failed
        auto bail = [&](cudaError_t err, const char *what) {
            for (auto &st : g->pipe_stream) cudaStreamSynchronize(st);
            return cuda_fail(err, what);
        };
        cudaStream_t s_in = g->pipe_stream[0], s_cmp = g->pipe_stream[1], s_out = g->pipe_stream[2];
        cudaEvent_t *ev_in = g->pipe_event, *ev_cmp = g->pipe_event + 32, ev_start = g->pipe_event[64], ev_end = g->pipe_event[65];
        // everything enqueued on the gauge's stream so far (e.g. the link conversion) comes first
        if ((e = cudaEventRecord(ev_start, s)) != cudaSuccess) return bail(e, "wd_apply_host: event record");
        for (int i = 0; i < 3; ++i) cudaStreamWaitEvent(g->pipe_stream[i], ev_start, 0);
        // Slab boundaries in time slices.  Only one direction of the link is busy until the first result leaves and after
        // the last slab has landed, so the slabs at either end are thin when Lt allows it (Lt >= 4 nslab, nslab >= 8:
        // 2, 3 slices at the head; 2, 1, 1 at the tail) and the rest share what is left evenly.
        long long bnd[33];
        {
            for (int k = 0; k <= nslab; ++k) bnd[k] = (long long)Lt * k / nslab;
            if (Lt >= 4 * nslab && nslab >= 8) {
                bnd[1] = 2;
                bnd[2] = 5;
                bnd[nslab - 1] = Lt - 1;
                bnd[nslab - 2] = Lt - 2;
                bnd[nslab - 3] = Lt - 4;
                const int mid = nslab - 5; // evenly sized slabs 2 .. nslab-4
                for (int j = 1; j < mid; ++j) bnd[2 + j] = 5 + (Lt - 9) * j / mid;
            }
        }
        const size_t row = (size_t)g->V * 24 * w; // bytes of one right-hand side, canonical
        // Copy streams carry ONLY copies (back to back, nothing between two transfers); pack, apply and unpack all run on
        // the compute stream.  Arrival order: the LAST slab first (it holds slice 0's backward neighbour), then 0, 1, ...,
        // nslab-2.  The computed ranges are the slabs shifted back by one slice, so that a range needs nothing beyond the
        // slab that has just landed:
        //   after slabs nslab-1 and 0:  [bnd[nslab-1]+1, Lt)  and  [0, bnd[1]-1)
        //   after slab k = 1..nslab-3:  [bnd[k]-1, bnd[k+1]-1)
        //   after slab nslab-2 (last):  [bnd[nslab-2]-1, bnd[nslab-1]+1)
        // and only that last range (the last slab landed plus two slices) is left to compute at the end.  `hold` = the slab
        // whose arrival releases a range's copy home (see below), -1 = none.
        for (int i = 0; i < nslab; ++i) {
            const int k = i == 0 ? nslab - 1 : i - 1;
            const long long s0 = bnd[k] * S3, ns = (bnd[k + 1] - bnd[k]) * S3;
            e = copy_rows((char *)g->stage_canon + (size_t)s0 * 24 * w, (const char *)in_canonical_host + (size_t)s0 * 24 * w,
                          row, (size_t)ns * 24 * w, nrhs, cudaMemcpyHostToDevice, s_in);
            if (e != cudaSuccess) return bail(e, "wd_apply_host: H2D copy");
            cudaEventRecord(ev_in[k], s_in);
        }
        auto pack_slab = [&](int k) {
            cudaStreamWaitEvent(s_cmp, ev_in[k], 0);
            return wd::launch_pack_spinor(g->stage_in, g->stage_canon, g->V, nrhs, precision, s_cmp, bnd[k] * S3,
                                          (bnd[k + 1] - bnd[k]) * S3);
        };
        int n_ev = 0;
        const char *what = nullptr;
        // D on the time slices [ta, tb), its result unpacked and sent home
        auto range = [&](long long ta, long long tb, int hold) {
            if (tb <= ta) return cudaSuccess;
            wd::ApplyArgs a = shape_args(g, nrhs);
            a.out = g->stage_out;
            a.in = g->stage_in;
            a.links = g->links;
            a.mass = mass;
            a.stream = s_cmp;
            a.site_begin = ta * S3;
            a.site_end = tb * S3;
            what = "wd_apply_host: kernel launch";
            cudaError_t er = wd::launch_site(a);
            if (er != cudaSuccess) return er;
            what = "wd_apply_host: unpack";
            er = wd::launch_unpack_spinor(g->stage_canon_out, g->stage_out, g->V, nrhs, precision, s_cmp, a.site_begin,
                                          a.site_end - a.site_begin);
            if (er != cudaSuccess) return er;
            cudaEventRecord(ev_cmp[n_ev], s_cmp);
            cudaStreamWaitEvent(s_out, ev_cmp[n_ev], 0);
            // Measured on B200 (PCIe 5 x16): a host->device copy that STARTS while a device->host copy is in flight loses
            // about 40 us (16 pieces against one long copy out: 4.89 ms; one piece against 13 out: 4.34 ms for 201 MB
            // each way), while a copy out may start at any time.  So a result leaves when the NEXT slab has landed: both
            // directions then start their pieces together and the copy in never starts under a copy out (4.96 -> 4.76 ms)
            if (hold >= 0) cudaStreamWaitEvent(s_out, ev_in[hold], 0);
            ++n_ev;
            what = "wd_apply_host: D2H copy";
            return copy_rows((char *)out_canonical_host + (size_t)a.site_begin * 24 * w,
                             (const char *)g->stage_canon_out + (size_t)a.site_begin * 24 * w, row,
                             (size_t)(a.site_end - a.site_begin) * 24 * w, nrhs, cudaMemcpyDeviceToHost, s_out);
        };
        if ((e = pack_slab(nslab - 1)) != cudaSuccess || (e = pack_slab(0)) != cudaSuccess) return bail(e, "wd_apply_host: pack");
        if ((e = range(0, bnd[1] - 1, 1)) != cudaSuccess) return bail(e, what);
        if ((e = range(bnd[nslab - 1] + 1, Lt, 1)) != cudaSuccess) return bail(e, what);
        for (int k = 1; k <= nslab - 2; ++k) {
            if ((e = pack_slab(k)) != cudaSuccess) return bail(e, "wd_apply_host: pack");
            const long long tb = k == nslab - 2 ? bnd[nslab - 1] + 1 : bnd[k + 1] - 1;
            if ((e = range(bnd[k] - 1, tb, k + 1 <= nslab - 2 ? k + 1 : -1)) != cudaSuccess) return bail(e, what);
        }
        if ((e = cudaEventRecord(ev_end, s_out)) != cudaSuccess) return bail(e, "wd_apply_host: event record");
        cudaStreamWaitEvent(s, ev_end, 0);
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return bail(e, "wd_apply_host: stream synchronize");
        return WD_OK;
    }

    // ---- small or oddly shaped lattices: one stream, whole field at a time ----
    e = cudaMemcpyAsync(g->stage_canon, in_canonical_host, bytes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_host: H2D copy");
    e = wd::launch_pack_spinor(g->stage_in, g->stage_canon, g->V, nrhs, precision, s);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_host: pack");
    rc = dispatch_apply(g->stage_out, g->stage_in, g, mass, nrhs);
    if (rc) return rc;
    e = wd::launch_unpack_spinor(g->stage_canon_out, g->stage_out, g->V, nrhs, precision, s);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_host: unpack");
    e = cudaMemcpyAsync(out_canonical_host, g->stage_canon_out, bytes, cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_host: D2H copy");
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_host: stream synchronize");
    return WD_OK;
}

int wd_selected_kernel(const wd_gauge *gauge, int nrhs)
{
    if (!gauge) return fail(WD_ERR_NULL, "wd_selected_kernel: NULL gauge");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_selected_kernel: not a live wd_gauge handle");
    if (nrhs < 1) return fail(WD_ERR_NRHS, "wd_selected_kernel: nrhs=%d", nrhs);
    if (gauge->kernel != WD_KERNEL_AUTO) return gauge->kernel;
    return auto_kernel(shape_args(gauge, nrhs));
}

// ---- red/black blocks ----------------------------------------------------------------------------
static bool all_even(const int dims[4])
{
    for (int d = 0; d < 4; ++d)
        if (dims[d] % 2) return false;
    return true;
}

static size_t half_bytes(long long V, int nrhs, int precision)
{
    if (precision == WD_FP16) return (size_t)nrhs * (size_t)wd::padded_volume(V / 2) * 52; // 3 vectors of 8 halves + a float scale
    return (size_t)nrhs * (size_t)wd::padded_volume(V / 2) * 24 * (precision == WD_FP32 ? 4 : 8);
}

size_t wd_spinor_bytes_parity(const wd_lattice *lat, int nrhs, int precision)
{
    if (!lat || lat->magic != LATTICE_MAGIC || nrhs < 1 || !valid_storage(precision) || !all_even(lat->dims)) return 0;
    return half_bytes(lat->V, nrhs, precision);
}

static int parity_copy(const char *who, const wd_lattice *lat, void *native, void *canon, int nrhs, int precision,
                       int parity, bool to_native, void *stream)
{
    if (!lat || !native || !canon) return fail(WD_ERR_NULL, "%s: NULL argument", who);
    if (lat->magic != LATTICE_MAGIC) return fail(WD_ERR_MISMATCH, "%s: not a live wd_lattice handle", who);
    if (!valid_storage(precision)) return fail(WD_ERR_PRECISION, "%s: precision %d is not 16, 32 or 64", who, precision);
    if (nrhs < 1) return fail(WD_ERR_NRHS, "%s: nrhs=%d", who, nrhs);
    if (!all_even(lat->dims)) return fail(WD_ERR_DIMS, "%s: red/black fields need even extents", who);
    if (parity != 0 && parity != 1) return fail(WD_ERR_MISMATCH, "%s: parity %d is not 0 or 1", who, parity);
    const size_t cbytes = (size_t)nrhs * (size_t)lat->V * 24 * canon_real_bytes(precision);
    if (overlap(native, half_bytes(lat->V, nrhs, precision), canon, cbytes)) return fail(WD_ERR_ALIAS, "%s: buffers overlap", who);
    cudaError_t e = precision == WD_FP16
                        ? wd::launch_parity_copy_half(native, canon, lat->dims, lat->V, nrhs, parity, to_native, (cudaStream_t)stream)
                        : wd::launch_parity_copy(native, canon, lat->dims, lat->V, nrhs, precision, parity, to_native,
                                                 (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, who);
}

int wd_pack_spinor_parity(const wd_lattice *lat, void *native_half_dev, const void *canonical_dev, int nrhs, int precision,
                          int parity, void *stream)
{
    return parity_copy("wd_pack_spinor_parity", lat, native_half_dev, const_cast<void *>(canonical_dev), nrhs, precision,
                       parity, true, stream);
}

int wd_unpack_spinor_parity(const wd_lattice *lat, void *canonical_dev, const void *native_half_dev, int nrhs,
                            int precision, int parity, void *stream)
{
    return parity_copy("wd_unpack_spinor_parity", lat, const_cast<void *>(native_half_dev), canonical_dev, nrhs, precision,
                       parity, false, stream);
}

static int check_eo_args(const char *who, const void *out, const void *in, const wd_gauge *g, const int dims[4], int nrhs,
                         int precision, int parity, bool allow_half = false)
{
    int rc = check_apply_args(out, in, g, dims, nrhs, precision, allow_half);
    if (rc) return rc;
    if (!all_even(g->dims)) return fail(WD_ERR_DIMS, "%s: red/black blocks need even extents", who);
    if (parity != 0 && parity != 1) return fail(WD_ERR_MISMATCH, "%s: parity %d is not 0 or 1", who, parity);
    const size_t hb = half_bytes(g->V, nrhs, precision);
    if (overlap(out, hb, in, hb)) return fail(WD_ERR_ALIAS, "%s: out and in overlap", who);
    if (((uintptr_t)out | (uintptr_t)in) & 15) return fail(WD_ERR_MISMATCH, "%s: buffers must be 16-byte aligned", who);
    // the red/black kernels read a parity-ordered copy of the link records (wd_dslash_eo.cu); it is made here, on the
    // gauge's stream, by the first red/black call on the handle (the handle is opaque to the caller: the copy is a cache)
    if (!g->links_eo) {
        wd_gauge *gm = const_cast<wd_gauge *>(g);
        const size_t nb = 2 * wd::eo_links_half_bytes(g->V, g->precision, g->recon);
        if (cudaMalloc(&gm->links_eo, nb) != cudaSuccess) {
            gm->links_eo = nullptr;
            cudaGetLastError();
            return fail(WD_ERR_ALLOC, "%s: cudaMalloc of %zu bytes for the parity-ordered links failed", who, nb);
        }
        cudaError_t e = cudaMemsetAsync(gm->links_eo, 0, nb, g->stream); // padding lanes of the last blocks
        if (e == cudaSuccess) e = wd::launch_links_to_eo(gm->links_eo, g->links, g->dims, g->V, g->precision, g->recon, g->stream);
        if (e != cudaSuccess) {
            cudaFree(gm->links_eo);
            gm->links_eo = nullptr;
            return cuda_fail(e, "parity-ordered links");
        }
    }
    return WD_OK;
}

int wd_apply_hop(void *out_half_dev, const void *in_half_dev, const wd_gauge *gauge, const int dims[4], int nrhs,
                 int precision, int parity_out)
{
    int rc = check_eo_args("wd_apply_hop", out_half_dev, in_half_dev, gauge, dims, nrhs, precision, parity_out, true);
    if (rc) return rc;
    wd::ApplyArgs a = shape_args(gauge, nrhs);
    a.out = out_half_dev;
    a.in = in_half_dev;
    a.links = gauge->links;
    a.stream = gauge->stream;
    cudaError_t e = wd::launch_eo(a, nullptr, 0.0, -0.5, parity_out);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_apply_hop: kernel launch");
}

static int apply_schur(void *out_half_dev, const void *in_half_dev, void *tmp_half_dev, const wd_gauge *gauge, double mass,
                       const int dims[4], int nrhs, int precision, int parity, bool dagger)
{
    int rc = check_eo_args("wd_apply_schur", out_half_dev, in_half_dev, gauge, dims, nrhs, precision, parity, true);
    if (rc) return rc;
    if (!tmp_half_dev) return fail(WD_ERR_NULL, "wd_apply_schur: NULL tmp");
    const size_t hb = half_bytes(gauge->V, nrhs, precision);
    if (overlap(tmp_half_dev, hb, in_half_dev, hb) || overlap(tmp_half_dev, hb, out_half_dev, hb) || ((uintptr_t)tmp_half_dev & 15))
        return fail(WD_ERR_ALIAS, "wd_apply_schur: tmp overlaps out or in, or is not 16-byte aligned");
    const double a0 = 4.0 + mass;
    if (a0 == 0.0) return fail(WD_ERR_MISMATCH, "wd_apply_schur: 4 + mass = 0, the diagonal block is not invertible");
    wd::ApplyArgs a = shape_args(gauge, nrhs);
    a.links = gauge->links;
    a.stream = gauge->stream;
    a.out = tmp_half_dev; // tmp_q = H_qp in_p
    a.in = in_half_dev;
    cudaError_t e = wd::launch_eo(a, nullptr, 0.0, -0.5, 1 - parity, dagger);
    if (e != cudaSuccess) return cuda_fail(e, "wd_apply_schur: kernel launch");
    a.out = out_half_dev; // out_p = (4+m) in_p - H_pq tmp_q / (4+m) = (4+m) in_p + hops(tmp_q) / (2 (4+m))
    a.in = tmp_half_dev;
    e = wd::launch_eo(a, in_half_dev, a0, 0.5 / a0, parity, dagger);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_apply_schur: kernel launch");
}

int wd_apply_schur(void *out_half_dev, const void *in_half_dev, void *tmp_half_dev, const wd_gauge *gauge, double mass,
                   const int dims[4], int nrhs, int precision, int parity)
{
    return apply_schur(out_half_dev, in_half_dev, tmp_half_dev, gauge, mass, dims, nrhs, precision, parity, false);
}

int wd_apply_schur_dagger(void *out_half_dev, const void *in_half_dev, void *tmp_half_dev, const wd_gauge *gauge,
                          double mass, const int dims[4], int nrhs, int precision, int parity)
{
    return apply_schur(out_half_dev, in_half_dev, tmp_half_dev, gauge, mass, dims, nrhs, precision, parity, true);
}

int wd_apply_schur_static(void *out_half_dev, const void *in_half_dev, const wd_gauge *gauge, double mass, const int dims[4],
                          int nrhs, int precision, int parity)
{
    // (not check_eo_args: that one builds the parity-ordered link copy with cudaMalloc; nothing below allocates)
    int rc = check_apply_args(out_half_dev, in_half_dev, gauge, dims, nrhs, precision);
    if (rc) return rc;
    if (!all_even(gauge->dims)) return fail(WD_ERR_DIMS, "wd_apply_schur_static: red/black blocks need even extents");
    if (parity != 0 && parity != 1) return fail(WD_ERR_MISMATCH, "wd_apply_schur_static: parity %d is not 0 or 1", parity);
    const size_t hb = half_bytes(gauge->V, nrhs, precision);
    if (overlap(out_half_dev, hb, in_half_dev, hb)) return fail(WD_ERR_ALIAS, "wd_apply_schur_static: out and in overlap");
    if (((uintptr_t)out_half_dev | (uintptr_t)in_half_dev) & 15)
        return fail(WD_ERR_MISMATCH, "wd_apply_schur_static: buffers must be 16-byte aligned");
    if (4.0 + mass == 0.0) return fail(WD_ERR_MISMATCH, "wd_apply_schur_static: 4 + mass = 0, the diagonal block is not invertible");
    wd::ApplyArgs a = shape_args(gauge, nrhs);
    a.out = out_half_dev;
    a.in = in_half_dev;
    a.links = gauge->links;
    a.mass = mass;
    a.stream = gauge->stream;
    const size_t need = wd::schur_static_need(a);
    if (need > (size_t)WD_STATIC_SCRATCH_BYTES)
        return fail(WD_ERR_DIMS, "wd_apply_schur_static: the intermediate field needs %zu bytes, the static scratch array holds %zu",
                    need, (size_t)WD_STATIC_SCRATCH_BYTES);
    cudaError_t e = wd::launch_schur_static(a, parity);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_apply_schur_static");
}

int wd_cgnr_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4],
                  int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host)
{
    int rc = check_eo_args("wd_cgnr_schur", x_half_dev, b_half_dev, gauge, dims, 1, precision, parity);
    if (rc) return rc;
    if (max_iter < 0 || tol < 0.0) return fail(WD_ERR_MISMATCH, "wd_cgnr_schur: max_iter=%d tol=%g", max_iter, tol);
    if (4.0 + mass == 0.0) return fail(WD_ERR_MISMATCH, "wd_cgnr_schur: 4 + mass = 0");
    wd::ApplyArgs a = shape_args(gauge, 1);
    a.links = gauge->links;
    a.stream = gauge->stream;
    cudaError_t e = cudaSuccess;
    if (wd::solve_schur(gauge, a, 0, x_half_dev, b_half_dev, mass, parity, max_iter, 0, tol, iters_out, hist_host, &e))
        return e == cudaErrorMemoryAllocation ? fail(WD_ERR_ALLOC, "wd_cgnr_schur: workspace allocation failed")
                                              : cuda_fail(e, "wd_cgnr_schur");
    return WD_OK;
}

int wd_cgnr_schur_block(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int nrhs,
                        int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host)
{
    int rc = check_eo_args("wd_cgnr_schur_block", x_half_dev, b_half_dev, gauge, dims, nrhs, precision, parity);
    if (rc) return rc;
    if (max_iter < 0 || tol < 0.0) return fail(WD_ERR_MISMATCH, "wd_cgnr_schur_block: max_iter=%d tol=%g", max_iter, tol);
    if (4.0 + mass == 0.0) return fail(WD_ERR_MISMATCH, "wd_cgnr_schur_block: 4 + mass = 0");
    wd::ApplyArgs a = shape_args(gauge, 1);
    a.links = gauge->links;
    a.stream = gauge->stream;
    cudaError_t e = cudaSuccess;
    if (wd::cgnr_schur_block(gauge, a, x_half_dev, b_half_dev, mass, parity, nrhs, max_iter, tol, iters_out, hist_host, &e))
        return e == cudaErrorMemoryAllocation ? fail(WD_ERR_ALLOC, "wd_cgnr_schur_block: workspace allocation failed")
                                              : cuda_fail(e, "wd_cgnr_schur_block");
    return WD_OK;
}

int wd_bicgstab_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4],
                      int precision, int parity, int max_iter, double tol, int *iters_out, double *hist_host)
{
    int rc = check_eo_args("wd_bicgstab_schur", x_half_dev, b_half_dev, gauge, dims, 1, precision, parity);
    if (rc) return rc;
    if (max_iter < 0 || tol < 0.0) return fail(WD_ERR_MISMATCH, "wd_bicgstab_schur: max_iter=%d tol=%g", max_iter, tol);
    if (4.0 + mass == 0.0) return fail(WD_ERR_MISMATCH, "wd_bicgstab_schur: 4 + mass = 0");
    wd::ApplyArgs a = shape_args(gauge, 1);
    a.links = gauge->links;
    a.stream = gauge->stream;
    cudaError_t e = cudaSuccess;
    if (wd::solve_schur(gauge, a, 1, x_half_dev, b_half_dev, mass, parity, max_iter, 0, tol, iters_out, hist_host, &e))
        return e == cudaErrorMemoryAllocation ? fail(WD_ERR_ALLOC, "wd_bicgstab_schur: workspace allocation failed")
                                              : cuda_fail(e, "wd_bicgstab_schur");
    return WD_OK;
}

int wd_gcr_schur(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int precision,
                 int parity, int max_iter, int restart, double tol, int *iters_out, double *hist_host)
{
    return wd_gcr_schur_precond(x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, restart, tol, iters_out,
                                hist_host, nullptr, nullptr);
}

int wd_gcr_schur_precond(void *x_half_dev, const void *b_half_dev, wd_gauge *gauge, double mass, const int dims[4], int precision,
                         int parity, int max_iter, int restart, double tol, int *iters_out, double *hist_host,
                         wd_precond_fn precond, void *precond_ctx)
{
    int rc = check_eo_args("wd_gcr_schur", x_half_dev, b_half_dev, gauge, dims, 1, precision, parity);
    if (rc) return rc;
    if (max_iter < 0 || tol < 0.0 || restart < 1 || restart > 32)
        return fail(WD_ERR_MISMATCH, "wd_gcr_schur: max_iter=%d restart=%d tol=%g", max_iter, restart, tol);
    if (4.0 + mass == 0.0) return fail(WD_ERR_MISMATCH, "wd_gcr_schur: 4 + mass = 0");
    wd::ApplyArgs a = shape_args(gauge, 1);
    a.links = gauge->links;
    a.stream = gauge->stream;
    cudaError_t e = cudaSuccess;
    if (wd::solve_schur(gauge, a, 2, x_half_dev, b_half_dev, mass, parity, max_iter, restart, tol, iters_out, hist_host, &e, precond,
                        precond_ctx))
        return e == cudaErrorMemoryAllocation ? fail(WD_ERR_ALLOC, "wd_gcr_schur: workspace allocation failed")
                                              : cuda_fail(e, "wd_gcr_schur");
    return WD_OK;
}

// ---- transfer operators ------------------------------------------------------------------------------
static int check_transfer(const char *who, const wd_lattice *lat, int nv, int precision)
{
    if (!lat) return fail(WD_ERR_NULL, "%s: NULL lattice", who);
    if (lat->magic != LATTICE_MAGIC) return fail(WD_ERR_MISMATCH, "%s: not a live wd_lattice handle", who);
    if (!valid_precision(precision)) return fail(WD_ERR_PRECISION, "%s: precision %d is not 32 or 64", who, precision);
    if (nv < 1) return fail(WD_ERR_NRHS, "%s: nv=%d", who, nv);
    for (int d = 0; d < 4; ++d)
        if (lat->dims[d] % 4) return fail(WD_ERR_DIMS, "%s: extents must be multiples of the 4^4 block", who);
    return WD_OK;
}

long long wd_coarse_reals(const wd_lattice *lat, int nv)
{
    if (check_transfer("wd_coarse_reals", lat, nv, WD_FP32)) return -1;
    return lat->V / 256 * 2 * nv * 2;
}

int wd_block_orthonormalise(const wd_lattice *lat, void *vecs_native_dev, int nv, int precision, void *stream)
{
    int rc = check_transfer("wd_block_orthonormalise", lat, nv, precision);
    if (rc) return rc;
    if (!vecs_native_dev) return fail(WD_ERR_NULL, "wd_block_orthonormalise: NULL argument");
    cudaError_t e = wd::launch_transfer(0, vecs_native_dev, nullptr, nullptr, lat->dims, lat->V, nv, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_block_orthonormalise");
}

int wd_restrict(const wd_lattice *lat, void *coarse_dev, const void *basis_native_dev, const void *psi_native_dev, int nv,
                int precision, void *stream)
{
    int rc = check_transfer("wd_restrict", lat, nv, precision);
    if (rc) return rc;
    if (!coarse_dev || !basis_native_dev || !psi_native_dev) return fail(WD_ERR_NULL, "wd_restrict: NULL argument");
    cudaError_t e = wd::launch_transfer(1, coarse_dev, basis_native_dev, psi_native_dev, lat->dims, lat->V, nv, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_restrict");
}

int wd_prolong(const wd_lattice *lat, void *psi_native_dev, const void *basis_native_dev, const void *coarse_dev, int nv,
               int precision, void *stream)
{
    int rc = check_transfer("wd_prolong", lat, nv, precision);
    if (rc) return rc;
    if (!psi_native_dev || !basis_native_dev || !coarse_dev) return fail(WD_ERR_NULL, "wd_prolong: NULL argument");
    if (overlap(psi_native_dev, wd_spinor_bytes(lat, 1, precision), basis_native_dev, wd_spinor_bytes(lat, nv, precision)))
        return fail(WD_ERR_ALIAS, "wd_prolong: psi overlaps the basis");
    cudaError_t e = wd::launch_transfer(2, psi_native_dev, basis_native_dev, coarse_dev, lat->dims, lat->V, nv, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_prolong");
}

long long wd_coarse_stencil_reals(const wd_lattice *lat, int nv)
{
    if (check_transfer("wd_coarse_stencil_reals", lat, nv, WD_FP32)) return -1;
    return lat->V / 256 * 9 * (2LL * nv) * (2LL * nv) * 2;
}

int wd_build_coarse(const wd_gauge *gauge, void *stencil_dev, void *scratch_dev, const void *basis_native_dev, double mass,
                    const int dims[4], int nv, int precision)
{
    if (!gauge || !stencil_dev || !scratch_dev || !basis_native_dev || !dims) return fail(WD_ERR_NULL, "wd_build_coarse: NULL argument");
    if (gauge->magic != GAUGE_MAGIC) return fail(WD_ERR_MISMATCH, "wd_build_coarse: not a live wd_gauge handle");
    if (!valid_precision(precision) || precision != gauge->precision)
        return fail(WD_ERR_PRECISION, "wd_build_coarse: precision %d, gauge was loaded in %d", precision, gauge->precision);
    for (int d = 0; d < 4; ++d) {
        if (dims[d] != gauge->dims[d]) return fail(WD_ERR_DIMS, "wd_build_coarse: dims[%d]=%d but gauge lattice has %d", d, dims[d], gauge->dims[d]);
        if (dims[d] % 4) return fail(WD_ERR_DIMS, "wd_build_coarse: extents must be multiples of the 4^4 block");
    }
    if (nv < 1 || nv > 32) return fail(WD_ERR_NRHS, "wd_build_coarse: nv=%d (1..32)", nv);
    if (gauge->V / 256 > 65535) return fail(WD_ERR_DIMS, "wd_build_coarse: more than 65535 blocks");
    const size_t sb = (size_t)(gauge->V / 256) * 9 * (2 * nv) * (2 * nv) * 2 * (precision == WD_FP32 ? 4 : 8);
    if (overlap(stencil_dev, sb, scratch_dev, sb)) return fail(WD_ERR_ALIAS, "wd_build_coarse: stencil and scratch overlap");
    cudaError_t e = wd::launch_coarse_build(stencil_dev, scratch_dev, basis_native_dev, gauge->links, gauge->dims, gauge->V, nv,
                                            mass, precision, gauge->recon, gauge->stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_build_coarse");
}

int wd_apply_coarse(const wd_lattice *lat, void *out_coarse_dev, const void *in_coarse_dev, const void *stencil_dev, int nv,
                    int nrhs, int precision, void *stream)
{
    int rc = check_transfer("wd_apply_coarse", lat, nv, precision);
    if (rc) return rc;
    if (!out_coarse_dev || !in_coarse_dev || !stencil_dev) return fail(WD_ERR_NULL, "wd_apply_coarse: NULL argument");
    if (nrhs < 1) return fail(WD_ERR_NRHS, "wd_apply_coarse: nrhs=%d", nrhs);
    if (nv > 56) return fail(WD_ERR_NRHS, "wd_apply_coarse: nv=%d (9 * 2 nv threads must fit one CTA)", nv);
    const size_t cb = (size_t)nrhs * (size_t)(lat->V / 256) * 2 * nv * 2 * (precision == WD_FP32 ? 4 : 8);
    if (overlap(out_coarse_dev, cb, in_coarse_dev, cb)) return fail(WD_ERR_ALIAS, "wd_apply_coarse: out and in overlap");
    cudaError_t e = wd::launch_coarse_apply(out_coarse_dev, in_coarse_dev, stencil_dev, lat->dims, nv, nrhs, precision, (cudaStream_t)stream);
    return e == cudaSuccess ? WD_OK : cuda_fail(e, "wd_apply_coarse");
}

long long wd_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char *wd_last_error(void) { return g_err; }

void wd_destroy_gauge(wd_gauge *gauge)
{
    if (!gauge || gauge->magic != GAUGE_MAGIC) return;
    gauge->magic = 0;
    cudaFree(gauge->links);
    cudaFree(gauge->links_eo);
    cudaFree(gauge->stage_canon);
    cudaFree(gauge->stage_canon_out);
    cudaFree(gauge->cg_ws);
    cudaFree(gauge->rf_ws);
    cudaFree(gauge->cg_sc);
    cudaFree(gauge->stage_in);
    cudaFree(gauge->stage_out);
    if (gauge->pipe_ready) {
        for (auto &st : gauge->pipe_stream) cudaStreamDestroy(st);
        for (auto &ev : gauge->pipe_event) cudaEventDestroy(ev);
    }
    delete gauge;
}

void wd_destroy(wd_lattice *lat)
{
    if (!lat || lat->magic != LATTICE_MAGIC) return;
    lat->magic = 0;
    delete lat;
}

} // extern "C"
