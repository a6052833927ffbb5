"""Thin ctypes binding of libwd.so -- same names as include/wd.h, argument marshalling only.

Every step of the Wilson-Dirac hot path (eq. (2.2)) runs in the CUDA kernels
behind the C ABI; nothing here computes.  PyTorch appears only as the owner of device memory and
streams: a "device pointer" argument may be a torch tensor (its data_ptr() is passed) or an int.

There is NO CPU fallback: if libwd.so has not been built (python -m paper_0912_2186_b200.build)
the first call raises WdError, loudly.
"""
import ctypes
import os

WD_OK = 0
WD_FP16, WD_FP32, WD_FP64 = 16, 32, 64
WD_RECON_18, WD_RECON_12, WD_RECON_8 = 18, 12, 8
WD_KERNEL_AUTO, WD_KERNEL_SITE, WD_KERNEL_STAGE = 0, 1, 3

STATUS_NAMES = {
    0: "WD_OK", -1: "WD_ERR_NULL", -2: "WD_ERR_DIMS", -3: "WD_ERR_PRECISION", -4: "WD_ERR_RECON",
    -5: "WD_ERR_NRHS", -6: "WD_ERR_ALIAS", -7: "WD_ERR_MISMATCH", -8: "WD_ERR_CUDA", -9: "WD_ERR_ALLOC",
}

# every symbol include/wd.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "wd_create_lattice", "wd_lattice_dims", "wd_lattice_volume", "wd_load_gauge", "wd_set_stream",
    "wd_set_kernel", "wd_set_tuning", "wd_set_temporal_gauge", "wd_selected_kernel", "wd_spinor_bytes", "wd_spinor_bytes_parity", "wd_pack_spinor_parity",
    "wd_unpack_spinor_parity", "wd_apply_hop", "wd_apply_schur", "wd_apply_schur_dagger", "wd_apply_schur_static", "wd_cgnr_schur", "wd_bicgstab_schur", "wd_gcr_schur", "wd_gcr_schur_precond", "wd_cgnr_schur_block", "wd_coarse_reals", "wd_coarse_stencil_reals", "wd_build_coarse", "wd_apply_coarse",
    "wd_block_orthonormalise", "wd_restrict", "wd_prolong", "wd_pack_spinor", "wd_unpack_spinor", "wd_apply", "wd_apply_dagger", "wd_apply_host",
    "wd_launch_count", "wd_last_error", "wd_destroy_gauge", "wd_destroy",
)

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libwd.so")
_lib = None


class WdError(RuntimeError):
    def __init__(self, code, where, msg=""):
        self.code = int(code)
        super().__init__(f"{where}: {STATUS_NAMES.get(self.code, self.code)} {msg}".rstrip())


def lib():
    """Load libwd.so once.  Raises WdError if it is missing -- there is no other code path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise WdError(-8, "binding.lib", f"{LIB_PATH} not built; run `python -m paper_0912_2186_b200.build`")
    L = ctypes.CDLL(LIB_PATH)
    vp, ip, i, d = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int), ctypes.c_int, ctypes.c_double
    L.wd_create_lattice.argtypes = [ip, ctypes.POINTER(vp)]
    L.wd_lattice_dims.argtypes = [vp, ip]
    L.wd_lattice_volume.argtypes = [vp]
    L.wd_lattice_volume.restype = ctypes.c_longlong
    L.wd_load_gauge.argtypes = [vp, vp, i, i, vp, ctypes.POINTER(vp)]
    L.wd_set_stream.argtypes = [vp, vp]
    L.wd_set_kernel.argtypes = [vp, i]
    L.wd_set_tuning.argtypes = [vp, ctypes.c_char_p, i]
    L.wd_set_temporal_gauge.argtypes = [vp, i]
    L.wd_selected_kernel.argtypes = [vp, i]
    L.wd_spinor_bytes.argtypes = [vp, i, i]
    L.wd_spinor_bytes.restype = ctypes.c_size_t
    L.wd_pack_spinor.argtypes = [vp, vp, vp, i, i, vp]
    L.wd_unpack_spinor.argtypes = [vp, vp, vp, i, i, vp]
    L.wd_apply.argtypes = [vp, vp, vp, d, ip, i, i]
    L.wd_apply_dagger.argtypes = [vp, vp, vp, d, ip, i, i]
    L.wd_apply_host.argtypes = [vp, vp, vp, d, ip, i, i]
    L.wd_spinor_bytes_parity.argtypes = [vp, i, i]
    L.wd_spinor_bytes_parity.restype = ctypes.c_size_t
    L.wd_pack_spinor_parity.argtypes = [vp, vp, vp, i, i, i, vp]
    L.wd_unpack_spinor_parity.argtypes = [vp, vp, vp, i, i, i, vp]
    L.wd_apply_hop.argtypes = [vp, vp, vp, ip, i, i, i]
    L.wd_apply_schur.argtypes = [vp, vp, vp, vp, d, ip, i, i, i]
    L.wd_apply_schur_dagger.argtypes = [vp, vp, vp, vp, d, ip, i, i, i]
    L.wd_apply_schur_static.argtypes = [vp, vp, vp, d, ip, i, i, i]
    L.wd_cgnr_schur.argtypes = [vp, vp, vp, d, ip, i, i, i, d, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)]
    L.wd_bicgstab_schur.argtypes = L.wd_cgnr_schur.argtypes
    L.wd_gcr_schur.argtypes = [vp, vp, vp, d, ip, i, i, i, i, d, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double)]
    L.wd_coarse_reals.argtypes = [vp, i]
    L.wd_coarse_reals.restype = ctypes.c_longlong
    L.wd_coarse_stencil_reals.argtypes = [vp, i]
    L.wd_coarse_stencil_reals.restype = ctypes.c_longlong
    L.wd_build_coarse.argtypes = [vp, vp, vp, vp, d, ip, i, i]
    L.wd_build_coarse.restype = i
    L.wd_apply_coarse.argtypes = [vp, vp, vp, vp, i, i, i, vp]
    L.wd_apply_coarse.restype = i
    L.wd_block_orthonormalise.argtypes = [vp, vp, i, i, vp]
    L.wd_restrict.argtypes = [vp, vp, vp, vp, i, i, vp]
    L.wd_prolong.argtypes = [vp, vp, vp, vp, i, i, vp]
    L.wd_launch_count.argtypes = []
    L.wd_launch_count.restype = ctypes.c_longlong
    L.wd_last_error.argtypes = []
    L.wd_last_error.restype = ctypes.c_char_p
    L.wd_destroy_gauge.argtypes = [vp]
    L.wd_destroy_gauge.restype = None
    L.wd_destroy.argtypes = [vp]
    L.wd_destroy.restype = None
    for name in ("wd_create_lattice", "wd_lattice_dims", "wd_load_gauge", "wd_set_stream", "wd_set_kernel",
                 "wd_set_tuning", "wd_set_temporal_gauge",
                 "wd_selected_kernel", "wd_pack_spinor", "wd_unpack_spinor", "wd_apply", "wd_apply_dagger", "wd_apply_host",
                 "wd_pack_spinor_parity", "wd_unpack_spinor_parity", "wd_apply_hop", "wd_apply_schur",
                 "wd_apply_schur_dagger", "wd_cgnr_schur", "wd_bicgstab_schur", "wd_gcr_schur",
                 "wd_block_orthonormalise", "wd_restrict", "wd_prolong"):
        getattr(L, name).restype = i
    _lib = L
    return L


def _ptr(x):
    """torch tensor / numpy array / int / None -> integer address (no copies, no checks on content)."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "cuda_stream"):  # torch.cuda.Stream
        return int(x.cuda_stream)
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _dims(dims):
    if dims is None:
        return None
    return (ctypes.c_int * 4)(*[int(v) for v in dims])


def _check(rc, where):
    if rc != WD_OK:
        raise WdError(rc, where, wd_last_error())


def wd_last_error():
    return lib().wd_last_error().decode()


def wd_launch_count():
    return int(lib().wd_launch_count())


def wd_create_lattice(dims):
    h = ctypes.c_void_p()
    _check(lib().wd_create_lattice(_dims(dims), ctypes.byref(h)), "wd_create_lattice")
    return h


def wd_lattice_dims(lat):
    out = (ctypes.c_int * 4)()
    _check(lib().wd_lattice_dims(lat, out), "wd_lattice_dims")
    return tuple(out)


def wd_lattice_volume(lat):
    return int(lib().wd_lattice_volume(lat))


def wd_load_gauge(lat, links_canonical_dev, precision, recon, stream=None):
    h = ctypes.c_void_p()
    _check(lib().wd_load_gauge(lat, _ptr(links_canonical_dev), int(precision), int(recon), _ptr(stream),
                               ctypes.byref(h)), "wd_load_gauge")
    return h


def wd_set_stream(gauge, stream):
    _check(lib().wd_set_stream(gauge, _ptr(stream)), "wd_set_stream")


def wd_set_kernel(gauge, kernel):
    _check(lib().wd_set_kernel(gauge, int(kernel)), "wd_set_kernel")


def wd_set_tuning(gauge, name, value):
    _check(lib().wd_set_tuning(gauge, name.encode(), int(value)), "wd_set_tuning")


def wd_selected_kernel(gauge, nrhs=1):
    k = int(lib().wd_selected_kernel(gauge, int(nrhs)))
    if k < 0:
        _check(k, "wd_selected_kernel")
    return k


KERNEL_NAMES = {WD_KERNEL_SITE: "site", WD_KERNEL_STAGE: "stage"}


def wd_set_temporal_gauge(gauge, on=True):
    _check(lib().wd_set_temporal_gauge(gauge, int(bool(on))), "wd_set_temporal_gauge")


def wd_spinor_bytes(lat, nrhs, precision):
    return int(lib().wd_spinor_bytes(lat, int(nrhs), int(precision)))


def wd_pack_spinor(lat, native_dev, canonical_dev, nrhs, precision, stream=None):
    _check(lib().wd_pack_spinor(lat, _ptr(native_dev), _ptr(canonical_dev), int(nrhs), int(precision),
                                _ptr(stream)), "wd_pack_spinor")


def wd_unpack_spinor(lat, canonical_dev, native_dev, nrhs, precision, stream=None):
    _check(lib().wd_unpack_spinor(lat, _ptr(canonical_dev), _ptr(native_dev), int(nrhs), int(precision),
                                  _ptr(stream)), "wd_unpack_spinor")


def wd_apply(out_native_dev, in_native_dev, gauge, mass, dims, nrhs, precision):
    _check(lib().wd_apply(_ptr(out_native_dev), _ptr(in_native_dev), gauge, float(mass), _dims(dims), int(nrhs),
                          int(precision)), "wd_apply")


def wd_apply_dagger(out_native_dev, in_native_dev, gauge, mass, dims, nrhs, precision):
    _check(lib().wd_apply_dagger(_ptr(out_native_dev), _ptr(in_native_dev), gauge, float(mass), _dims(dims), int(nrhs),
                                 int(precision)), "wd_apply_dagger")


def wd_apply_host(out_canonical_host, in_canonical_host, gauge, mass, dims, nrhs, precision):
    _check(lib().wd_apply_host(_ptr(out_canonical_host), _ptr(in_canonical_host), gauge, float(mass), _dims(dims),
                               int(nrhs), int(precision)), "wd_apply_host")


def wd_spinor_bytes_parity(lat, nrhs, precision):
    return int(lib().wd_spinor_bytes_parity(lat, int(nrhs), int(precision)))


def wd_pack_spinor_parity(lat, native_half_dev, canonical_dev, nrhs, precision, parity, stream=None):
    _check(lib().wd_pack_spinor_parity(lat, _ptr(native_half_dev), _ptr(canonical_dev), int(nrhs), int(precision),
                                       int(parity), _ptr(stream)), "wd_pack_spinor_parity")


def wd_unpack_spinor_parity(lat, canonical_dev, native_half_dev, nrhs, precision, parity, stream=None):
    _check(lib().wd_unpack_spinor_parity(lat, _ptr(canonical_dev), _ptr(native_half_dev), int(nrhs), int(precision),
                                         int(parity), _ptr(stream)), "wd_unpack_spinor_parity")


def wd_apply_hop(out_half_dev, in_half_dev, gauge, dims, nrhs, precision, parity_out):
    _check(lib().wd_apply_hop(_ptr(out_half_dev), _ptr(in_half_dev), gauge, _dims(dims), int(nrhs), int(precision),
                              int(parity_out)), "wd_apply_hop")


def wd_apply_schur(out_half_dev, in_half_dev, tmp_half_dev, gauge, mass, dims, nrhs, precision, parity):
    _check(lib().wd_apply_schur(_ptr(out_half_dev), _ptr(in_half_dev), _ptr(tmp_half_dev), gauge, float(mass),
                                _dims(dims), int(nrhs), int(precision), int(parity)), "wd_apply_schur")


def wd_apply_schur_dagger(out_half_dev, in_half_dev, tmp_half_dev, gauge, mass, dims, nrhs, precision, parity):
    _check(lib().wd_apply_schur_dagger(_ptr(out_half_dev), _ptr(in_half_dev), _ptr(tmp_half_dev), gauge, float(mass),
                                       _dims(dims), int(nrhs), int(precision), int(parity)), "wd_apply_schur_dagger")


WD_STATIC_SCRATCH_BYTES = 16 << 20  # include/wd.h


def wd_apply_schur_static(out_half_dev, in_half_dev, gauge, mass, dims, nrhs, precision, parity):
    """wd_apply_schur without a caller-supplied intermediate field and without any device allocation (static scratch)."""
    _check(lib().wd_apply_schur_static(_ptr(out_half_dev), _ptr(in_half_dev), gauge, float(mass), _dims(dims), int(nrhs),
                                       int(precision), int(parity)), "wd_apply_schur_static")


def _solve(name, x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, tol):
    it = ctypes.c_int(0)
    hist = (ctypes.c_double * (int(max_iter) + 1))()
    _check(getattr(lib(), name)(_ptr(x_half_dev), _ptr(b_half_dev), gauge, float(mass), _dims(dims), int(precision),
                                int(parity), int(max_iter), float(tol), ctypes.byref(it), hist), name)
    return it.value, [hist[i] for i in range(it.value + 1)]


def wd_cgnr_schur(x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, tol=0.0):
    """Returns (iterations done, relative residual history as a list of floats)."""
    return _solve("wd_cgnr_schur", x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, tol)


def wd_bicgstab_schur(x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, tol=0.0):
    """Returns (iterations done, relative residual history as a list of floats)."""
    return _solve("wd_bicgstab_schur", x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, tol)


def wd_gcr_schur(x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, restart=8, tol=0.0):
    """Returns (iterations done, relative residual history as a list of floats)."""
    it = ctypes.c_int(0)
    hist = (ctypes.c_double * (int(max_iter) + 1))()
    _check(lib().wd_gcr_schur(_ptr(x_half_dev), _ptr(b_half_dev), gauge, float(mass), _dims(dims), int(precision),
                              int(parity), int(max_iter), int(restart), float(tol), ctypes.byref(it), hist), "wd_gcr_schur")
    return it.value, [hist[i] for i in range(it.value + 1)]


def wd_cgnr_schur_block(x_half_dev, b_half_dev, gauge, mass, dims, nrhs, precision, parity, max_iter, tol=0.0):
    """Returns (iterations done, [history of right-hand side r as a list of floats for r < nrhs])."""
    it = ctypes.c_int(0)
    hs = int(max_iter) + 1
    hist = (ctypes.c_double * (int(nrhs) * hs))()
    fn = lib().wd_cgnr_schur_block
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.POINTER(ctypes.c_int), ctypes.c_int,
                   ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_int),
                   ctypes.POINTER(ctypes.c_double)]
    fn.restype = ctypes.c_int
    _check(fn(_ptr(x_half_dev), _ptr(b_half_dev), gauge, float(mass), _dims(dims), int(nrhs), int(precision), int(parity),
              int(max_iter), float(tol), ctypes.byref(it), hist), "wd_cgnr_schur_block")
    return it.value, [[hist[r * hs + i] for i in range(it.value + 1)] for r in range(int(nrhs))]


PRECOND_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p)


def wd_gcr_schur_precond(x_half_dev, b_half_dev, gauge, mass, dims, precision, parity, max_iter, restart, tol, precond):
    """GCR with the preconditioner slot: precond(z_ptr, r_ptr, stream_ptr) is a Python callable that enqueues z = K r on the
    given stream for the two device addresses (native half fields) and returns 0.  Marshalling only."""
    it = ctypes.c_int(0)
    hist = (ctypes.c_double * (int(max_iter) + 1))()
    cb = PRECOND_FN(lambda ctx, z, r, s: int(precond(z, r, s) or 0))
    fn = lib().wd_gcr_schur_precond
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.POINTER(ctypes.c_int), ctypes.c_int,
                   ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_int),
                   ctypes.POINTER(ctypes.c_double), PRECOND_FN, ctypes.c_void_p]
    fn.restype = ctypes.c_int
    _check(fn(_ptr(x_half_dev), _ptr(b_half_dev), gauge, float(mass), _dims(dims), int(precision), int(parity), int(max_iter),
              int(restart), float(tol), ctypes.byref(it), hist, cb, None), "wd_gcr_schur_precond")
    return it.value, [hist[i] for i in range(it.value + 1)]


def wd_coarse_reals(lat, nv):
    return int(lib().wd_coarse_reals(lat, int(nv)))


def wd_block_orthonormalise(lat, vecs_native_dev, nv, precision, stream=None):
    _check(lib().wd_block_orthonormalise(lat, _ptr(vecs_native_dev), int(nv), int(precision), _ptr(stream)),
           "wd_block_orthonormalise")


def wd_restrict(lat, coarse_dev, basis_native_dev, psi_native_dev, nv, precision, stream=None):
    _check(lib().wd_restrict(lat, _ptr(coarse_dev), _ptr(basis_native_dev), _ptr(psi_native_dev), int(nv), int(precision),
                             _ptr(stream)), "wd_restrict")


def wd_prolong(lat, psi_native_dev, basis_native_dev, coarse_dev, nv, precision, stream=None):
    _check(lib().wd_prolong(lat, _ptr(psi_native_dev), _ptr(basis_native_dev), _ptr(coarse_dev), int(nv), int(precision),
                            _ptr(stream)), "wd_prolong")


def wd_coarse_stencil_reals(lat, nv):
    return int(lib().wd_coarse_stencil_reals(lat, int(nv)))


def wd_build_coarse(gauge, stencil_dev, scratch_dev, basis_native_dev, mass, dims, nv, precision):
    _check(lib().wd_build_coarse(gauge, _ptr(stencil_dev), _ptr(scratch_dev), _ptr(basis_native_dev), float(mass), _dims(dims),
                                 int(nv), int(precision)), "wd_build_coarse")


def wd_apply_coarse(lat, out_coarse_dev, in_coarse_dev, stencil_dev, nv, nrhs, precision, stream=None):
    _check(lib().wd_apply_coarse(lat, _ptr(out_coarse_dev), _ptr(in_coarse_dev), _ptr(stencil_dev), int(nv), int(nrhs),
                                 int(precision), _ptr(stream)), "wd_apply_coarse")


def wd_destroy_gauge(gauge):
    lib().wd_destroy_gauge(gauge)


def wd_destroy(lat):
    lib().wd_destroy(lat)


class WilsonDirac:
    """Handle bundle for one gauge field: lattice + native links (+ the stream to launch on).

    Marshalling only.  `links_canonical_dev` is a torch CUDA tensor [4,Lt,Lz,Ly,Lx,3,3,2] of
    float32/float64; spinors passed to apply() are NATIVE-layout torch CUDA tensors (use pack()).
    """

    def __init__(self, dims, links_canonical_dev, precision, recon=WD_RECON_18, stream=None, kernel=WD_KERNEL_AUTO):
        self.dims = tuple(int(v) for v in dims)
        self.precision = int(precision)
        self.recon = int(recon)
        self.stream = stream
        self.lat = wd_create_lattice(self.dims)
        self.gauge = None
        self.gauge = wd_load_gauge(self.lat, links_canonical_dev, self.precision, self.recon, stream)
        self.volume = wd_lattice_volume(self.lat)
        self._cdims = _dims(self.dims)          # marshalled once: wd_apply is called in launch-bound loops
        self._apply = lib().wd_apply
        self._apply_dagger = lib().wd_apply_dagger
        if kernel != WD_KERNEL_AUTO:
            wd_set_kernel(self.gauge, kernel)

    def set_stream(self, stream):
        wd_set_stream(self.gauge, stream)
        self.stream = stream

    def set_kernel(self, kernel):
        wd_set_kernel(self.gauge, kernel)

    def set_tuning(self, name, value):
        wd_set_tuning(self.gauge, name, value)

    def pack(self, native_dev, canonical_dev, nrhs, stream=None):
        wd_pack_spinor(self.lat, native_dev, canonical_dev, nrhs, self.precision, stream or self.stream)

    def unpack(self, canonical_dev, native_dev, nrhs, stream=None):
        wd_unpack_spinor(self.lat, canonical_dev, native_dev, nrhs, self.precision, stream or self.stream)

    def set_temporal_gauge(self, on=True):
        wd_set_temporal_gauge(self.gauge, on)

    def selected_kernel(self, nrhs=1):
        """Name of the kernel wd_apply will launch for nrhs right-hand sides ("site", "stage")."""
        return KERNEL_NAMES[wd_selected_kernel(self.gauge, nrhs)]

    def apply_dagger(self, out_native_dev, in_native_dev, mass, nrhs=1):
        rc = self._apply_dagger(_ptr(out_native_dev), _ptr(in_native_dev), self.gauge, mass, self._cdims, nrhs, self.precision)
        if rc != WD_OK:
            _check(rc, "wd_apply_dagger")

    def native_numel(self, nrhs=1):
        """Elements (float16 / float32 / float64 by precision) of a NATIVE spinor buffer of nrhs fields (the volume is
        padded to 32-site blocks; half-precision storage: 26 two-byte elements per site = 24 ratios + a float32 scale)."""
        return wd_spinor_bytes(self.lat, nrhs, self.precision) // {16: 2, 32: 4, 64: 8}[self.precision]

    def apply(self, out_native_dev, in_native_dev, mass, nrhs=1):
        rc = self._apply(_ptr(out_native_dev), _ptr(in_native_dev), self.gauge, mass, self._cdims, nrhs, self.precision)
        if rc != WD_OK:
            _check(rc, "wd_apply")

    # ---- red/black (even-odd) blocks: half fields of one parity ----
    def half_numel(self, nrhs=1):
        """Elements (float16 / float32 / float64 by precision) of a native HALF field (one parity) of nrhs right-hand
        sides; 0 if an extent is odd."""
        return wd_spinor_bytes_parity(self.lat, nrhs, self.precision) // {16: 2, 32: 4, 64: 8}[self.precision]

    def pack_parity(self, native_half_dev, canonical_dev, nrhs, parity, stream=None):
        wd_pack_spinor_parity(self.lat, native_half_dev, canonical_dev, nrhs, self.precision, parity, stream or self.stream)

    def unpack_parity(self, canonical_dev, native_half_dev, nrhs, parity, stream=None):
        wd_unpack_spinor_parity(self.lat, canonical_dev, native_half_dev, nrhs, self.precision, parity,
                                stream or self.stream)

    def apply_hop(self, out_half_dev, in_half_dev, parity_out, nrhs=1):
        wd_apply_hop(out_half_dev, in_half_dev, self.gauge, self.dims, nrhs, self.precision, parity_out)

    def apply_schur(self, out_half_dev, in_half_dev, tmp_half_dev, mass, parity, nrhs=1):
        wd_apply_schur(out_half_dev, in_half_dev, tmp_half_dev, self.gauge, mass, self.dims, nrhs, self.precision, parity)

    def apply_schur_static(self, out_half_dev, in_half_dev, mass, parity, nrhs=1):
        wd_apply_schur_static(out_half_dev, in_half_dev, self.gauge, mass, self.dims, nrhs, self.precision, parity)

    def apply_schur_dagger(self, out_half_dev, in_half_dev, tmp_half_dev, mass, parity, nrhs=1):
        wd_apply_schur_dagger(out_half_dev, in_half_dev, tmp_half_dev, self.gauge, mass, self.dims, nrhs, self.precision,
                              parity)

    def cgnr_schur(self, x_half_dev, b_half_dev, mass, parity, max_iter, tol=0.0):
        return wd_cgnr_schur(x_half_dev, b_half_dev, self.gauge, mass, self.dims, self.precision, parity, max_iter, tol)

    def bicgstab_schur(self, x_half_dev, b_half_dev, mass, parity, max_iter, tol=0.0):
        return wd_bicgstab_schur(x_half_dev, b_half_dev, self.gauge, mass, self.dims, self.precision, parity, max_iter, tol)

    def gcr_schur(self, x_half_dev, b_half_dev, mass, parity, max_iter, restart=8, tol=0.0):
        return wd_gcr_schur(x_half_dev, b_half_dev, self.gauge, mass, self.dims, self.precision, parity, max_iter, restart,
                            tol)

    def cgnr_schur_block(self, x_half_dev, b_half_dev, mass, parity, nrhs, max_iter, tol=0.0):
        return wd_cgnr_schur_block(x_half_dev, b_half_dev, self.gauge, mass, self.dims, nrhs, self.precision, parity, max_iter, tol)

    def gcr_schur_precond(self, x_half_dev, b_half_dev, mass, parity, max_iter, restart, tol, precond):
        return wd_gcr_schur_precond(x_half_dev, b_half_dev, self.gauge, mass, self.dims, self.precision, parity, max_iter,
                                    restart, tol, precond)

    def apply_host(self, out_canonical_host, in_canonical_host, mass, nrhs=1):
        wd_apply_host(out_canonical_host, in_canonical_host, self.gauge, mass, self.dims, nrhs, self.precision)

    def close(self):
        if self.gauge is not None:
            wd_destroy_gauge(self.gauge)
            self.gauge = None
        if self.lat is not None:
            wd_destroy(self.lat)
            self.lat = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
