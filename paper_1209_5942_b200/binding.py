"""ctypes binding of liblqcd.so -- same names as include/lqcd.h, marshalling only.

Device buffers are torch CUDA tensors (PyTorch is used for device memory and
streams only); every ``lqcd_*`` function below passes ``tensor.data_ptr()``
straight to the C ABI and raises ``LqcdError`` on a negative status.
"""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liblqcd.so")

LQCD_OK, LQCD_NOT_CONVERGED = 0, 1
LQCD_NOT_INITIALISED, LQCD_BAD_DIMS, LQCD_BAD_ARG, LQCD_CUDA_ERROR, LQCD_BREAKDOWN = -1, -2, -3, -4, -5
LQCD_DOUBLE, LQCD_SINGLE = 0, 1
LQCD_HEATBATH, LQCD_OVERRELAX = 0, 1
LQCD_ELEM_FLOAT, LQCD_ELEM_DOUBLE, LQCD_ELEM_VEC16, LQCD_ELEM_SU3_AOS, LQCD_ELEM_SPINOR_AOS = 0, 1, 2, 3, 4
LQCD_STREAM_COPY, LQCD_STREAM_READ, LQCD_STREAM_MIX71 = 0, 1, 2
LQCD_STREAM_PROBE_BLOCKS = 1184

SYMBOLS = [
    "lqcd_last_error", "lqcd_init", "lqcd_finalize", "lqcd_set_stream", "lqcd_set_format",
    "lqcd_gauge_bytes", "lqcd_spinor_bytes", "lqcd_pack_gauge", "lqcd_pack_spinor",
    "lqcd_unpack_spinor", "lqcd_dslash_eo", "lqcd_mtm", "lqcd_mtm_full", "lqcd_solve_full", "lqcd_cg_mdagm", "lqcd_cg_setup",
    "lqcd_cg_iterate", "lqcd_cg_finish", "lqcd_cg_stats", "lqcd_cg_mdagm_mixed", "lqcd_cg_outer_iterations", "lqcd_bicgstab_mhat", "lqcd_force_bytes", "lqcd_unpack_force", "lqcd_fermion_force", "lqcd_force_tm", "lqcd_mtm_host", "lqcd_cg_mdagm_host",
    "lqcd_launch_count", "lqcd_set_block_size", "lqcd_set_hop_variant", "lqcd_profile", "lqcd_profile_read",
    "lqcd_gauge_update", "lqcd_gauge_sweep", "lqcd_plaquette", "lqcd_plaquette_static", "lqcd_unpack_gauge", "lqcd_stream_probe", "lqcd_fp64_probe",
    "lqcd_select_context", "lqcd_slab_init", "lqcd_slab_spinor_halo", "lqcd_slab_gauge_halo", "lqcd_slab_dslash",
    "lqcd_slab_mhat_stage", "lqcd_slab_cg_begin", "lqcd_slab_cg_stage", "lqcd_slab_cg_halo_field",
    "lqcd_slab_sum_ptr", "lqcd_slab_cg_poll", "lqcd_slab_cg_end",
]


class LqcdError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"liblqcd status {status}: {text}")
        self.status = status


def _load():
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, dbl, i32, u64 = ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.c_ulonglong
    lib.lqcd_last_error.restype = ctypes.c_char_p
    lib.lqcd_gauge_bytes.restype = ctypes.c_size_t
    lib.lqcd_spinor_bytes.restype = ctypes.c_size_t
    lib.lqcd_force_bytes.restype = ctypes.c_size_t
    lib.lqcd_launch_count.restype = ctypes.c_longlong
    sig = {
        "lqcd_init": [ctypes.POINTER(i32), ctypes.POINTER(dbl)],
        "lqcd_finalize": [],
        "lqcd_set_stream": [vp],
        "lqcd_set_format": [i32, i32],
        "lqcd_pack_gauge": [vp, vp],
        "lqcd_pack_spinor": [vp, vp, i32],
        "lqcd_unpack_spinor": [vp, vp, i32],
        "lqcd_dslash_eo": [vp, vp, vp, i32, dbl],
        "lqcd_mtm": [vp, vp, vp, dbl, dbl, i32],
        "lqcd_mtm_full": [vp, vp, vp, vp, vp, dbl, dbl],
        "lqcd_solve_full": [vp, vp, vp, vp, vp, dbl, dbl, dbl, i32],
        "lqcd_cg_mdagm": [vp, vp, vp, dbl, dbl, dbl, i32],
        "lqcd_bicgstab_mhat": [vp, vp, vp, dbl, dbl, dbl, i32],
        "lqcd_unpack_force": [vp, vp],
        "lqcd_fermion_force": [vp, vp, vp, vp, vp, vp, dbl],
        "lqcd_force_tm": [vp, vp, vp, dbl, dbl, dbl, i32],
        "lqcd_cg_setup": [vp, vp, vp, dbl, dbl, dbl],
        "lqcd_cg_mdagm_mixed": [vp, i32, vp, i32, vp, vp, dbl, dbl, dbl, i32, dbl],
        "lqcd_cg_outer_iterations": [],
        "lqcd_cg_iterate": [i32],
        "lqcd_cg_finish": [],
        "lqcd_cg_stats": [ctypes.POINTER(i32), ctypes.POINTER(dbl), ctypes.POINTER(dbl)],
        "lqcd_mtm_host": [vp, vp, vp, dbl, dbl, i32],
        "lqcd_cg_mdagm_host": [vp, vp, vp, dbl, dbl, dbl, i32],
        "lqcd_set_block_size": [i32],
        "lqcd_set_hop_variant": [i32],
        "lqcd_gauge_update": [vp, i32, i32, i32, dbl, u64, u64],
        "lqcd_gauge_sweep": [vp, i32, dbl, u64, u64],
        "lqcd_plaquette": [vp, ctypes.POINTER(dbl)],
        "lqcd_plaquette_static": [vp, vp],
        "lqcd_unpack_gauge": [vp, vp],
        "lqcd_stream_probe": [i32, i32, vp, vp, ctypes.c_size_t],
        "lqcd_fp64_probe": [dbl, dbl, i32, vp],
        "lqcd_select_context": [i32],
        "lqcd_slab_init": [ctypes.POINTER(i32), ctypes.POINTER(dbl), i32, i32],
        "lqcd_slab_spinor_halo": [ctypes.POINTER(ctypes.c_size_t)] * 5,
        "lqcd_slab_gauge_halo": [i32] + [ctypes.POINTER(ctypes.c_size_t)] * 3,
        "lqcd_slab_dslash": [vp, vp, vp, i32, dbl, i32],
        "lqcd_slab_mhat_stage": [vp, vp, vp, vp, dbl, dbl, i32, i32, i32],
        "lqcd_slab_cg_begin": [vp, vp, vp, dbl, dbl, dbl],
        "lqcd_slab_cg_stage": [i32, i32],
        "lqcd_slab_cg_poll": [ctypes.POINTER(i32), ctypes.POINTER(i32)],
        "lqcd_slab_cg_end": [i32],
        "lqcd_profile": [i32],
        "lqcd_profile_read": [i32, ctypes.POINTER(dbl), ctypes.POINTER(i32)],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = i32
    lib.lqcd_slab_cg_halo_field.argtypes = [i32]
    lib.lqcd_slab_cg_halo_field.restype = vp
    lib.lqcd_slab_sum_ptr.argtypes = []
    lib.lqcd_slab_sum_ptr.restype = vp
    return lib


_lib = _load()
# mirrors format and sites per parity of each context (lqcd_select_context), for buffer helpers only
_fmts = [{"precision": LQCD_DOUBLE, "vh": 0} for _ in range(8)]
_fmt = _fmts[0]
_cur_ctx = [0]        # the selected context (lqcd_select_context)


def _check(status):
    if status < 0:
        raise LqcdError(status, _lib.lqcd_last_error().decode())
    return status


def _ptr(t):
    """Device (torch CUDA tensor) or host (numpy array / CPU tensor) pointer, or a raw int."""
    if isinstance(t, int):
        return ctypes.c_void_p(t)
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return ctypes.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return ctypes.c_void_p(t.data_ptr())


def lqcd_last_error():
    return _lib.lqcd_last_error().decode()


def lqcd_init(dims, bc_phase):
    d = (ctypes.c_int * 4)(*[int(v) for v in dims])
    ph = np.asarray(bc_phase, dtype=np.complex128)
    p = (ctypes.c_double * 8)(*[float(v) for z in ph for v in (z.real, z.imag)])
    rc = _check(_lib.lqcd_init(d, p))
    _lib_streams.pop(_cur_ctx[0], None)      # lqcd_init resets the library's stream to the legacy default
    _fmt["precision"] = LQCD_DOUBLE
    _fmt["vh"] = int(np.prod([int(v) for v in dims])) // 2
    return rc


def lqcd_finalize():
    return _check(_lib.lqcd_finalize())


_lib_streams = {}     # context id -> the torch stream handed to lqcd_set_stream (None: never set = legacy default)


def lqcd_set_stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    rc = _check(_lib.lqcd_set_stream(ctypes.c_void_p(s.cuda_stream)))
    _lib_streams[_cur_ctx[0]] = s
    return rc


def library_stream():
    """The torch stream the library launches on in the selected context (None before lqcd_set_stream)."""
    return _lib_streams.get(_cur_ctx[0])


def check_same_stream(library_handle, current_handle):
    """The slab driver's ordering rule: torch.distributed orders its NCCL point-to-point operations and
    all-reduces against torch's CURRENT stream, the library's kernels run on the stream of
    lqcd_set_stream.  With two different streams a send could read a boundary slice before the hopping
    kernel that produces it has finished, and a boundary launch could read ghosts before the receive has
    landed -- so the two must be one stream (raw cudaStream_t handles compared)."""
    if int(library_handle or 0) != int(current_handle or 0):
        raise RuntimeError(f"slab exchange: torch's current stream ({int(current_handle or 0):#x}) is not the library's "
                           f"stream ({int(library_handle or 0):#x}); run under torch.cuda.stream(<the stream given to "
                           f"lqcd_set_stream>) or call lqcd_set_stream() for the current stream")


class _OnLibraryStream:
    """Makes the library's stream torch's current stream for the communication calls inside, then checks it."""

    def __init__(self, tensor=None):
        self.cuda = torch.cuda.is_available() and (tensor is None or (torch.is_tensor(tensor) and tensor.is_cuda))
        self.cm = None

    def __enter__(self):
        if not self.cuda:
            return self
        s = library_stream()
        if s is not None:
            self.cm = torch.cuda.stream(s)
            self.cm.__enter__()
        check_same_stream(s.cuda_stream if s is not None else 0, torch.cuda.current_stream().cuda_stream)
        return self

    def __exit__(self, *a):
        if self.cm is not None:
            self.cm.__exit__(*a)
        return False


def lqcd_set_format(precision, recon):
    rc = _check(_lib.lqcd_set_format(precision, recon))
    _fmt["precision"] = precision
    return rc


def lqcd_set_block_size(threads):
    return _check(_lib.lqcd_set_block_size(threads))


def lqcd_set_hop_variant(variant):
    return _check(_lib.lqcd_set_hop_variant(variant))


def lqcd_gauge_bytes():
    return int(_lib.lqcd_gauge_bytes())


def lqcd_spinor_bytes():
    return int(_lib.lqcd_spinor_bytes())


def lqcd_launch_count():
    return int(_lib.lqcd_launch_count())


def lqcd_profile(enable):
    return _check(_lib.lqcd_profile(int(enable)))


def lqcd_profile_read(category):
    """(total_ms, launches) of one kernel category since lqcd_profile(1)."""
    ms = ctypes.c_double(0.0)
    n = ctypes.c_int(0)
    _check(_lib.lqcd_profile_read(category, ctypes.byref(ms), ctypes.byref(n)))
    return ms.value, n.value


def lqcd_pack_gauge(canon_dev, internal_dev):
    return _check(_lib.lqcd_pack_gauge(_ptr(canon_dev), _ptr(internal_dev)))


def lqcd_pack_spinor(canon_dev, internal_dev, parity):
    return _check(_lib.lqcd_pack_spinor(_ptr(canon_dev), _ptr(internal_dev), parity))


def lqcd_unpack_spinor(internal_dev, canon_dev, parity):
    return _check(_lib.lqcd_unpack_spinor(_ptr(internal_dev), _ptr(canon_dev), parity))


def lqcd_dslash_eo(gauge, inp, out, parity, kappa):
    return _check(_lib.lqcd_dslash_eo(_ptr(gauge), _ptr(inp), _ptr(out), parity, kappa))


def lqcd_mtm(gauge, inp, out, kappa, mu, dagger):
    return _check(_lib.lqcd_mtm(_ptr(gauge), _ptr(inp), _ptr(out), kappa, mu, dagger))


def lqcd_mtm_full(gauge, in_even, in_odd, out_even, out_odd, kappa, mu):
    return _check(_lib.lqcd_mtm_full(_ptr(gauge), _ptr(in_even), _ptr(in_odd), _ptr(out_even), _ptr(out_odd),
                                     kappa, mu))


def lqcd_solve_full(gauge, eta_even, eta_odd, psi_even, psi_odd, kappa, mu, tol, maxit):
    return _check(_lib.lqcd_solve_full(_ptr(gauge), _ptr(eta_even), _ptr(eta_odd), _ptr(psi_even), _ptr(psi_odd),
                                       kappa, mu, tol, maxit))


def lqcd_cg_mdagm(gauge, b, x, kappa, mu, tol, maxit):
    return _check(_lib.lqcd_cg_mdagm(_ptr(gauge), _ptr(b), _ptr(x), kappa, mu, tol, maxit))


def lqcd_bicgstab_mhat(gauge, b, x, kappa, mu, tol, maxit):
    return _check(_lib.lqcd_bicgstab_mhat(_ptr(gauge), _ptr(b), _ptr(x), kappa, mu, tol, maxit))


def lqcd_force_bytes():
    return int(_lib.lqcd_force_bytes())


def lqcd_unpack_force(force_internal_dev, canon_dev):
    return _check(_lib.lqcd_unpack_force(_ptr(force_internal_dev), _ptr(canon_dev)))


def lqcd_fermion_force(gauge, x_even, x_odd, y_even, y_odd, force, kappa):
    return _check(_lib.lqcd_fermion_force(_ptr(gauge), _ptr(x_even), _ptr(x_odd), _ptr(y_even), _ptr(y_odd),
                                          _ptr(force), kappa))


def lqcd_force_tm(gauge, phi, force, kappa, mu, tol, maxit):
    return _check(_lib.lqcd_force_tm(_ptr(gauge), _ptr(phi), _ptr(force), kappa, mu, tol, maxit))


def lqcd_cg_mdagm_mixed(gauge_double, recon_double, gauge_single, recon_single, b, x, kappa, mu, tol, maxit,
                        inner_tol=0.0):
    return _check(_lib.lqcd_cg_mdagm_mixed(_ptr(gauge_double), recon_double, _ptr(gauge_single), recon_single,
                                           _ptr(b), _ptr(x), kappa, mu, tol, maxit, inner_tol))


def lqcd_cg_outer_iterations():
    return int(_lib.lqcd_cg_outer_iterations())


def lqcd_cg_setup(gauge, b, x, kappa, mu, tol):
    return _check(_lib.lqcd_cg_setup(_ptr(gauge), _ptr(b), _ptr(x), kappa, mu, tol))


def lqcd_cg_iterate(n):
    return _check(_lib.lqcd_cg_iterate(n))


def lqcd_cg_finish():
    return _check(_lib.lqcd_cg_finish())


def lqcd_cg_stats():
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0.0)
    rt = ctypes.c_double(0.0)
    _check(_lib.lqcd_cg_stats(ctypes.byref(it), ctypes.byref(rr), ctypes.byref(rt)))
    return it.value, rr.value, rt.value


def lqcd_mtm_host(gauge_canon_host, in_canon_host, out_canon_host, kappa, mu, dagger):
    return _check(_lib.lqcd_mtm_host(_ptr(gauge_canon_host), _ptr(in_canon_host), _ptr(out_canon_host),
                                     kappa, mu, dagger))


def lqcd_cg_mdagm_host(gauge_canon_host, b_canon_host, x_canon_host, kappa, mu, tol, maxit):
    return _check(_lib.lqcd_cg_mdagm_host(_ptr(gauge_canon_host), _ptr(b_canon_host), _ptr(x_canon_host),
                                          kappa, mu, tol, maxit))


def lqcd_gauge_update(gauge, mu, parity, mode, beta, seed, tag):
    return _check(_lib.lqcd_gauge_update(_ptr(gauge), mu, parity, mode, beta, seed, tag))


def lqcd_gauge_sweep(gauge, mode, beta, seed, tag):
    return _check(_lib.lqcd_gauge_sweep(_ptr(gauge), mode, beta, seed, tag))


def lqcd_plaquette(gauge):
    p = ctypes.c_double(0.0)
    _check(_lib.lqcd_plaquette(_ptr(gauge), ctypes.byref(p)))
    return p.value


def lqcd_plaquette_static(gauge, plaquette_dev):
    """No-allocation variant: the result goes to plaquette_dev, one double in device memory (include/lqcd.h)."""
    return _check(_lib.lqcd_plaquette_static(_ptr(gauge), _ptr(plaquette_dev)))


def lqcd_unpack_gauge(internal_dev, canon_dev):
    return _check(_lib.lqcd_unpack_gauge(_ptr(internal_dev), _ptr(canon_dev)))


def lqcd_stream_probe(elem, mode, src_dev, dst_dev, nbytes):
    return _check(_lib.lqcd_stream_probe(elem, mode, _ptr(src_dev), _ptr(dst_dev), nbytes))


def lqcd_fp64_probe(a, b, iters, out_dev):
    return _check(_lib.lqcd_fp64_probe(a, b, iters, _ptr(out_dev)))


# ---------------------------------------------------------------------------- buffer helpers
def alloc_gauge(device="cuda"):
    """Uninitialised device buffer for one internal gauge field (current format)."""
    return torch.empty(lqcd_gauge_bytes(), dtype=torch.uint8, device=device)


def alloc_spinor(device="cuda"):
    """Uninitialised device buffer for one internal half-spinor field (current format)."""
    return torch.empty(lqcd_spinor_bytes(), dtype=torch.uint8, device=device)


def alloc_force(device="cuda"):
    """Uninitialised device buffer for one internal force field (8 reals per link, double)."""
    return torch.empty(lqcd_force_bytes(), dtype=torch.uint8, device=device)


def download_force(f_internal):
    """internal force field -> numpy (V,4,8) float64."""
    canon = torch.empty((2 * _fmt["vh"], 4, 8), dtype=torch.float64, device=f_internal.device)
    lqcd_unpack_force(f_internal, canon)
    return canon.cpu().numpy()


def upload_gauge(U_canon, device="cuda"):
    """numpy (V,4,3,3) complex128 -> packed internal device buffer."""
    canon = torch.from_numpy(np.ascontiguousarray(U_canon)).to(device)
    g = alloc_gauge(device)
    lqcd_pack_gauge(canon, g)
    return g


def download_gauge(g_internal):
    """packed internal gauge buffer -> numpy (V,4,3,3) complex128."""
    canon = torch.empty((2 * _fmt["vh"], 4, 3, 3), dtype=torch.complex128, device=g_internal.device)
    lqcd_unpack_gauge(g_internal, canon)
    return canon.cpu().numpy()


def upload_spinor(psi_canon, parity, device="cuda"):
    """numpy (V/2,4,3) complex128 -> packed internal device buffer."""
    canon = torch.from_numpy(np.ascontiguousarray(psi_canon)).to(device)
    s = alloc_spinor(device)
    lqcd_pack_spinor(canon, s, parity)
    return s


def download_spinor(s_internal, parity):
    """packed internal device buffer -> numpy (V/2,4,3) complex128."""
    canon = torch.empty((_fmt["vh"], 4, 3), dtype=torch.complex128, device=s_internal.device)
    lqcd_unpack_spinor(s_internal, canon, parity)
    return canon.cpu().numpy()


# ---------------------------------------------------------------------------- slab decomposition
# Several ranks, one GPU each, each owning a slab of time slices (include/lqcd.h "Slab
# decomposition").  The library computes; what follows only moves halos and sums scalars with
# torch.distributed (NCCL between GPUs; the same code runs on CPU tensors over gloo in the tests).
def lqcd_select_context(ctx_id):
    global _fmt
    rc = _check(_lib.lqcd_select_context(int(ctx_id)))
    _fmt = _fmts[int(ctx_id)]
    _cur_ctx[0] = int(ctx_id)
    return rc


def lqcd_slab_init(dims_global, bc_phase, rank, nranks):
    d = (ctypes.c_int * 4)(*[int(v) for v in dims_global])
    ph = np.asarray(bc_phase, dtype=np.complex128)
    p = (ctypes.c_double * 8)(*[float(v) for z in ph for v in (z.real, z.imag)])
    rc = _check(_lib.lqcd_slab_init(d, p, int(rank), int(nranks)))
    _lib_streams.pop(_cur_ctx[0], None)
    _fmt["precision"] = LQCD_DOUBLE
    _fmt["vh"] = int(np.prod([int(v) for v in dims_global])) // (2 * int(nranks))
    return rc


def lqcd_slab_spinor_halo():
    v = [ctypes.c_size_t() for _ in range(5)]
    _check(_lib.lqcd_slab_spinor_halo(*[ctypes.byref(x) for x in v]))
    return dict(zip(("send_lo", "send_hi", "ghost_fwd", "ghost_bwd", "bytes"), (int(x.value) for x in v)))


def lqcd_slab_gauge_halo(parity):
    v = [ctypes.c_size_t() for _ in range(3)]
    _check(_lib.lqcd_slab_gauge_halo(int(parity), *[ctypes.byref(x) for x in v]))
    return dict(zip(("send_hi", "ghost_bwd", "bytes"), (int(x.value) for x in v)))


def lqcd_slab_dslash(gauge, inp, out, parity, kappa, part=0):
    return _check(_lib.lqcd_slab_dslash(_ptr(gauge), _ptr(inp), _ptr(out), parity, kappa, part))


def lqcd_slab_mhat_stage(gauge, inp, tmp_odd, out, kappa, mu, dagger, stage, part=0):
    return _check(_lib.lqcd_slab_mhat_stage(_ptr(gauge), _ptr(inp), _ptr(tmp_odd), _ptr(out), kappa, mu, dagger,
                                            stage, part))


def lqcd_slab_cg_begin(gauge, b, x, kappa, mu, tol):
    return _check(_lib.lqcd_slab_cg_begin(_ptr(gauge), _ptr(b), _ptr(x), kappa, mu, tol))


def lqcd_slab_cg_stage(stage, part=0):
    return _check(_lib.lqcd_slab_cg_stage(stage, part))


def lqcd_slab_cg_halo_field(stage):
    """Raw device pointer (int) of the field whose ghosts `stage` reads, or None."""
    return _lib.lqcd_slab_cg_halo_field(stage)


def lqcd_slab_sum_ptr():
    return _lib.lqcd_slab_sum_ptr()


def lqcd_slab_cg_poll():
    done, iters = ctypes.c_int(0), ctypes.c_int(0)
    _check(_lib.lqcd_slab_cg_poll(ctypes.byref(done), ctypes.byref(iters)))
    return bool(done.value), iters.value


def lqcd_slab_cg_end(with_true_resid=True):
    return _check(_lib.lqcd_slab_cg_end(1 if with_true_resid else 0))


class _DevMem:
    """A raw device allocation as a CUDA-array-interface object (uint8), for torch.as_tensor."""

    def __init__(self, ptr, nbytes):
        self.__cuda_array_interface__ = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False),
                                         "version": 2}


def device_bytes(ptr, nbytes, device="cuda"):
    """uint8 tensor view of `nbytes` of device memory at raw pointer `ptr` (no copy)."""
    return torch.as_tensor(_DevMem(ptr, nbytes), device=device)


def slab_exchange_blocks(buf, sends, recvs, rank, world, group=None):
    """The halo exchange of one field: `buf` is the field as a flat uint8 tensor (device or CPU);
    sends = [(offset, nbytes, 'prev'|'next'), ...], recvs likewise, posted in order as ONE batch of
    point-to-point operations (rank r: prev = r-1, next = r+1, cyclically).  Returns the requests;
    the caller waits on them (or lets later work on the same stream wait, NCCL) before the ghosts
    are read.  world = 1: the rank is its own neighbour, plain copies."""
    import torch.distributed as dist
    if world == 1:
        for (so, n, _), (ro, _, _) in zip(sends, recvs):
            buf[ro:ro + n].copy_(buf[so:so + n])
        return []
    peer = {"prev": (rank - 1) % world, "next": (rank + 1) % world}
    ops = []
    for tag, (off, n, to) in enumerate(sends):
        ops.append(dist.P2POp(dist.isend, buf[off:off + n], peer[to], group=group, tag=tag))
    for tag, (off, n, frm) in enumerate(recvs):
        ops.append(dist.P2POp(dist.irecv, buf[off:off + n], peer[frm], group=group, tag=tag))
    return dist.batch_isend_irecv(ops)


def slab_exchange_spinor(field, rank, world, group=None, wait=True):
    """Fill the two ghost time slices of an internal half-spinor field (tensor or raw pointer).  Device
    fields: issued on the library's stream (check_same_stream), so the sends are ordered after the kernel
    that wrote the boundary slices and later launches after the receives."""
    h = lqcd_slab_spinor_halo()
    if not torch.is_tensor(field):
        field = device_bytes(field, lqcd_spinor_bytes())
    n = h["bytes"]
    with _OnLibraryStream(field):
        # first slice -> forward ghost of the previous rank; last slice -> backward ghost of the next
        reqs = slab_exchange_blocks(field, [(h["send_lo"], n, "prev"), (h["send_hi"], n, "next")],
                                    [(h["ghost_fwd"], n, "next"), (h["ghost_bwd"], n, "prev")], rank, world, group)
        if wait:
            for r in reqs:
                r.wait()
            return []
    return reqs


def slab_exchange_gauge(gauge, rank, world, group=None):
    """Once, after lqcd_pack_gauge: receive the time-like links of the previous rank's last slice."""
    with _OnLibraryStream(gauge):
        for parity in (0, 1):
            h = lqcd_slab_gauge_halo(parity)
            for r in slab_exchange_blocks(gauge, [(h["send_hi"], h["bytes"], "next")],
                                          [(h["ghost_bwd"], h["bytes"], "prev")], rank, world, group):
                r.wait()


def slab_cg(gauge, b, x, kappa, mu, tol, maxit, rank, world, group=None, overlap=False, check_every=4):
    """CG on Mhat^dag Mhat across `world` ranks (one process per GPU, torch.distributed initialised):
    the stages of lqcd_slab_cg_stage with the halo exchanges and the three all-reduces between
    them.  Everything -- kernels, NCCL point-to-point operations, all-reduces -- is issued on ONE
    stream, the library's (check_same_stream).  overlap: a hopping stage runs its interior sites while
    its halos are in flight; off by default, because on one GPU the split launch costs 4-16% of the
    kernel time against a wire time of ~3.5 us (profiles/r01f_slab.md) and no two-GPU measurement says
    otherwise yet.  Returns the solve status; lqcd_cg_stats() gives iterations and residuals."""
    import torch.distributed as dist
    with _OnLibraryStream():
        lqcd_slab_cg_begin(gauge, b, x, kappa, mu, tol)
        total = device_bytes(lqcd_slab_sum_ptr(), 8).view(torch.float64)

        def allreduce():
            if world > 1:
                dist.all_reduce(total, group=group)

        def hop(stage):
            f = lqcd_slab_cg_halo_field(stage)
            if overlap:
                reqs = slab_exchange_spinor(f, rank, world, group, wait=False)
                lqcd_slab_cg_stage(stage, 1)
                for r in reqs:
                    r.wait()
                lqcd_slab_cg_stage(stage, 2)
            else:
                slab_exchange_spinor(f, rank, world, group)
                lqcd_slab_cg_stage(stage, 0)

        lqcd_slab_cg_stage(0); allreduce(); lqcd_slab_cg_stage(1)
        it = 0
        while it < maxit:
            hop(2); hop(3)
            lqcd_slab_cg_stage(4); allreduce(); lqcd_slab_cg_stage(5)
            hop(6); hop(7)
            lqcd_slab_cg_stage(8); allreduce(); lqcd_slab_cg_stage(9)
            it += 1
            if it % check_every == 0 or it == maxit:
                done, _ = lqcd_slab_cg_poll()
                if done:
                    break
        for stage in (11, 12, 13, 14):
            hop(stage)
        lqcd_slab_cg_stage(15); allreduce(); lqcd_slab_cg_stage(16)
        return lqcd_slab_cg_end(True)
