"""ctypes binding of include/tm.h.  Function names and argument order follow the header one to one."""
import ctypes
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtm_b200.so")

TM_PREC_F64, TM_PREC_F32, TM_PREC_F16 = 8, 4, 2
TM_RECON_18, TM_RECON_12, TM_RECON_8 = 18, 12, 8
TM_RECON_18_TG, TM_RECON_12_TG = 218, 212  # field declared in temporal gauge (tm.h)
TM_RECON_18_FIX16, TM_RECON_12_FIX16 = 118, 112  # 16-bit fixed-point link words for TM_PREC_F16 fields (tm.h)
TM_KIND_PLAIN, TM_KIND_TWIST_INV, TM_KIND_XPAY_TWIST = 0, 1, 2
TM_CG_HP_MIXED, TM_CG_LP_TRUNCATED, TM_CG_HP_DEFECT = 0, 1, 2
TM_ONEEND_TAU3, TM_ONEEND_GENERAL = 0, 1
TM_OK, TM_ERR_ARG, TM_ERR_LAYOUT, TM_ERR_NOT_SU3, TM_ERR_CUDA, TM_ERR_BREAKDOWN, TM_ERR_MAXITER, TM_ERR_RECON8 = 0, -1, -2, -3, -4, -5, -6, -7
TM_ERR_NOT_TGAUGE = -8
TM_ERR_STATIC_LIMIT = -9
TM_LOOP_STATIC_BYTES = 8388608
TM_MAX_NRHS = 16

ABI_SYMBOLS = [
    "tm_version", "tm_strerror", "tm_last_cuda_error", "tm_lattice_create", "tm_lattice_destroy", "tm_gauge_bytes",
    "tm_spinor_bytes", "tm_gauge_pack", "tm_spinor_pack", "tm_spinor_unpack", "tm_spinor_pack_z4", "tm_dslash",
    "tm_dslash_general", "tm_MdagM", "tm_cg_workspace_bytes", "tm_cg_multi", "tm_cg", "tm_loop_workspace_bytes",
    "tm_loop_contract", "tm_loop_contract_ex", "tm_M", "tm_oneend_workspace_bytes", "tm_oneend_loops", "tm_tsm_combine",
    "tm_tsm_workspace_bytes", "tm_tsm_batch_host", "tm_launch_count", "tm_kernel_timing_enable",
    "tm_kernel_timing_read", "tm_covdev", "tm_contract_field", "tm_loop_momentum_workspace_bytes", "tm_loop_momentum",
    "tm_time_dilute", "tm_loop_contract_slice", "tm_hpe_remainder", "tm_hpe_local_traces", "tm_spinor_pack_z4_bits",
    "tm_tsm_batch_host_bits", "tm_noise_z4", "tm_gauge_fix_temporal", "tm_kernel_signature", "tm_gauge_synthetic", "tm_loop_contract_static",
]


class tm_cg_params(ctypes.Structure):
    _fields_ = [("kappa", ctypes.c_double), ("mu", ctypes.c_double), ("tol", ctypes.c_double), ("max_iter", ctypes.c_int),
                ("mode", ctypes.c_int), ("reliable_delta", ctypes.c_double), ("check_every", ctypes.c_int),
                ("skip_true_resid", ctypes.c_int)]


class tm_cg_info(ctypes.Structure):
    _fields_ = [("iters", ctypes.c_int), ("status", ctypes.c_int), ("reliable_updates", ctypes.c_int),
                ("iterated_resid", ctypes.c_double), ("true_resid", ctypes.c_double)]


class TmError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = "%s: %s" % (where, tm_strerror(status))
        if status == TM_ERR_CUDA:
            msg += " [" + tm_last_cuda_error() + "]"
        super().__init__(msg)


_lib = None


def load():
    """Load libtm_b200.so (built in-tree on first use if missing); fails loudly if it cannot be built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        # a fresh checkout (built artefacts are not in the history): compile once with nvcc; still no CPU fallback
        try:
            from . import build as _build
            _build.build()
        except Exception as e:
            raise ImportError("libtm_b200.so is missing and could not be built (python -m paper_1309_2256_b200.build): %s; "
                              "there is no CPU fallback" % e) from e
    lib = ctypes.CDLL(LIB_PATH)
    vp, i, d, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    P = ctypes.POINTER
    sig = {
        "tm_version": (i, []),
        "tm_strerror": (ctypes.c_char_p, [i]),
        "tm_last_cuda_error": (ctypes.c_char_p, []),
        "tm_lattice_create": (i, [P(vp), P(i), i]),
        "tm_lattice_destroy": (None, [vp]),
        "tm_gauge_bytes": (sz, [vp, i, i]),
        "tm_spinor_bytes": (sz, [vp, i, i, i]),
        "tm_gauge_pack": (i, [vp, vp, i, i, vp, d, vp]),
        "tm_spinor_pack": (i, [vp, vp, i, i, vp, vp]),
        "tm_spinor_unpack": (i, [vp, vp, i, i, vp, vp]),
        "tm_spinor_pack_z4": (i, [vp, vp, i, i, vp, vp]),
        "tm_dslash": (i, [vp, vp, i, i, vp, vp, vp, i, i, i, d, d, i, vp]),
        "tm_dslash_general": (i, [vp, vp, i, i, vp, vp, vp, i, i, P(d), i, vp]),
        "tm_MdagM": (i, [vp, vp, i, i, vp, vp, vp, i, d, d, i, vp]),
        "tm_cg_workspace_bytes": (sz, [vp, i, i, i, i]),
        "tm_cg_multi": (i, [vp, vp, i, vp, i, i, vp, vp, P(tm_cg_params), i, P(tm_cg_info), vp, sz, vp]),
        "tm_cg": (i, [vp, vp, i, vp, i, i, vp, vp, P(tm_cg_params), P(tm_cg_info), vp, sz, vp]),
        "tm_loop_workspace_bytes": (sz, [vp, i]),
        "tm_loop_contract": (i, [vp, vp, vp, i, i, vp, vp, vp]),
        "tm_loop_contract_ex": (i, [vp, vp, vp, i, i, i, i, d, d, vp, vp, vp]),
        "tm_M": (i, [vp, vp, i, i, vp, vp, d, d, i, i, vp]),
        "tm_oneend_workspace_bytes": (sz, [vp, i, i]),
        "tm_oneend_loops": (i, [vp, vp, i, i, vp, i, d, d, i, vp, vp, sz, vp]),
        "tm_tsm_combine": (i, [i, vp, vp, i, vp, i, vp, vp]),
        "tm_tsm_workspace_bytes": (sz, [vp, i, i]),
        "tm_tsm_batch_host": (i, [vp, vp, i, i, vp, P(tm_cg_params), i, P(tm_cg_info), vp, vp, sz, vp]),
        "tm_launch_count": (ctypes.c_ulonglong, []),
        "tm_kernel_timing_enable": (i, [i]),
        "tm_kernel_timing_read": (i, [P(d), P(ctypes.c_longlong), i]),
        "tm_kernel_signature": (ctypes.c_char_p, []),
        "tm_loop_contract_static": (i, [vp, vp, vp, i, i, vp, vp]),
        "tm_gauge_synthetic": (i, [vp, ctypes.c_ulonglong, d, d, vp, vp]),
        "tm_covdev": (i, [vp, vp, i, i, vp, vp, i, i, vp]),
        "tm_contract_field": (i, [vp, vp, vp, i, i, vp, vp]),
        "tm_loop_momentum_workspace_bytes": (sz, [vp, i, i, i]),
        "tm_loop_momentum": (i, [vp, vp, vp, i, i, P(i), i, vp, vp, sz, vp]),
        "tm_time_dilute": (i, [vp, vp, i, i, ctypes.c_char_p, vp, vp]),
        "tm_loop_contract_slice": (i, [vp, vp, vp, i, i, i, vp, vp, vp]),
        "tm_hpe_remainder": (i, [vp, vp, i, i, vp, vp, vp, d, d, i, vp]),
        "tm_hpe_local_traces": (i, [d, d, P(d)]),
        "tm_spinor_pack_z4_bits": (i, [vp, vp, i, i, vp, vp]),
        "tm_noise_z4": (i, [vp, ctypes.c_ulonglong, ctypes.c_ulonglong, i, i, vp, vp]),
        "tm_gauge_fix_temporal": (i, [vp, vp, vp, vp]),
        "tm_tsm_batch_host_bits": (i, [vp, vp, i, i, vp, P(tm_cg_params), i, P(tm_cg_info), vp, vp, sz, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype = res
        f.argtypes = args
    _lib = lib
    return lib


def _ptr(t):
    """Device/host pointer of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        return ctypes.c_void_p(t.data_ptr())
    if isinstance(t, np.ndarray):
        return ctypes.c_void_p(t.ctypes.data)
    return ctypes.c_void_p(int(t))


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _check(rc, where, allow=()):
    if rc != TM_OK and rc not in allow:
        raise TmError(rc, where)
    return rc


def tm_version():
    return load().tm_version()


def tm_strerror(status):
    return load().tm_strerror(status).decode()


def tm_last_cuda_error():
    return load().tm_last_cuda_error().decode()


class Lattice:
    """Owns a tm_lattice* (host-side geometry descriptor)."""

    def __init__(self, dims, antiperiodic_t=True):
        self.dims = tuple(int(d) for d in dims)
        self.antiperiodic_t = bool(antiperiodic_t)
        h = ctypes.c_void_p()
        arr = (ctypes.c_int * 4)(*self.dims)
        _check(load().tm_lattice_create(ctypes.byref(h), arr, int(antiperiodic_t)), "tm_lattice_create")
        self.handle = h
        X, Y, Z, T = self.dims
        self.V = X * Y * Z * T
        self.T = T

    def __del__(self):
        try:
            if getattr(self, "handle", None):
                load().tm_lattice_destroy(self.handle)
                self.handle = None
        except Exception:
            pass


def tm_lattice_create(dims, antiperiodic_t=True):
    return Lattice(dims, antiperiodic_t)


def tm_gauge_bytes(L, prec, recon):
    return load().tm_gauge_bytes(L.handle, prec, recon)


def tm_spinor_bytes(L, prec, full, nrhs=1):
    return load().tm_spinor_bytes(L.handle, prec, int(full), nrhs)


def tm_gauge_pack(L, U_canonical, prec, recon, packed_out, su3_tol=1e-10, stream=None):
    return _check(load().tm_gauge_pack(L.handle, _ptr(U_canonical), prec, recon, _ptr(packed_out), su3_tol, _stream(stream)),
                  "tm_gauge_pack")


def tm_spinor_pack(L, psi_canonical, prec, nrhs, packed_out, stream=None):
    return _check(load().tm_spinor_pack(L.handle, _ptr(psi_canonical), prec, nrhs, _ptr(packed_out), _stream(stream)), "tm_spinor_pack")


def tm_spinor_unpack(L, packed, prec, nrhs, psi_canonical, stream=None):
    return _check(load().tm_spinor_unpack(L.handle, _ptr(packed), prec, nrhs, _ptr(psi_canonical), _stream(stream)), "tm_spinor_unpack")


def tm_spinor_pack_z4(L, codes, prec, nrhs, packed_out, stream=None):
    return _check(load().tm_spinor_pack_z4(L.handle, _ptr(codes), prec, nrhs, _ptr(packed_out), _stream(stream)), "tm_spinor_pack_z4")


def tm_dslash(L, gauge, prec, recon, out, inp, x, out_parity, dagger, kind, kappa, mu, nrhs=1, stream=None):
    return _check(load().tm_dslash(L.handle, _ptr(gauge), prec, recon, _ptr(out), _ptr(inp), _ptr(x), out_parity, int(dagger), kind,
                                   kappa, mu, nrhs, _stream(stream)), "tm_dslash")


def tm_dslash_general(L, gauge, prec, recon, out, inp, x, out_parity, dagger, pq, nrhs=1, stream=None):
    arr = (ctypes.c_double * 4)(*pq)
    return _check(load().tm_dslash_general(L.handle, _ptr(gauge), prec, recon, _ptr(out), _ptr(inp), _ptr(x), out_parity, int(dagger),
                                           arr, nrhs, _stream(stream)), "tm_dslash_general")


def tm_MdagM(L, gauge, prec, recon, out, inp, tmp, parity, kappa, mu, nrhs=1, stream=None):
    return _check(load().tm_MdagM(L.handle, _ptr(gauge), prec, recon, _ptr(out), _ptr(inp), _ptr(tmp), parity, kappa, mu, nrhs,
                                  _stream(stream)), "tm_MdagM")


def tm_cg_workspace_bytes(L, prec_hp, prec_lp, mode, nrhs=1):
    return load().tm_cg_workspace_bytes(L.handle, prec_hp, prec_lp, mode, nrhs)


def make_cg_params(kappa, mu, tol, max_iter, mode, reliable_delta=0.1, check_every=0, skip_true_resid=0):
    return tm_cg_params(kappa, mu, tol, max_iter, mode, reliable_delta, check_every, skip_true_resid)


_SOFT = (TM_ERR_MAXITER, TM_ERR_BREAKDOWN)


def tm_cg_multi(L, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, s_full, eta_full, params, nrhs, workspace, stream=None):
    """Returns (status, [tm_cg_info]*nrhs); MAXITER / BREAKDOWN are returned, not raised."""
    info = (tm_cg_info * nrhs)()
    ws_bytes = workspace.numel() * workspace.element_size()
    rc = load().tm_cg_multi(L.handle, _ptr(gauge_hp), prec_hp, _ptr(gauge_lp), prec_lp, recon, _ptr(s_full), _ptr(eta_full),
                            ctypes.byref(params), nrhs, info, _ptr(workspace), ws_bytes, _stream(stream))
    _check(rc, "tm_cg_multi", allow=_SOFT)
    return rc, list(info)


def tm_cg(L, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, s_full, eta_full, params, workspace, stream=None):
    rc, info = tm_cg_multi(L, gauge_hp, prec_hp, gauge_lp, prec_lp, recon, s_full, eta_full, params, 1, workspace, stream)
    return rc, info[0]


def tm_loop_workspace_bytes(L, nrhs=1):
    return load().tm_loop_workspace_bytes(L.handle, nrhs)


def tm_loop_contract(L, a_full, b_full, prec, nrhs, out, workspace, stream=None):
    return _check(load().tm_loop_contract(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs, _ptr(out), _ptr(workspace), _stream(stream)),
                  "tm_loop_contract")


def tm_loop_contract_ex(L, a_full, b_full, prec, nrhs, g5_left, g5_right, scale, out, workspace, stream=None):
    scale = complex(scale)
    return _check(load().tm_loop_contract_ex(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs, int(g5_left), int(g5_right), scale.real,
                                             scale.imag, _ptr(out), _ptr(workspace), _stream(stream)), "tm_loop_contract_ex")


def tm_M(L, gauge, prec, recon, out_full, in_full, kappa, mu, dagger=0, nrhs=1, stream=None):
    return _check(load().tm_M(L.handle, _ptr(gauge), prec, recon, _ptr(out_full), _ptr(in_full), kappa, mu, int(dagger), nrhs,
                              _stream(stream)), "tm_M")


def tm_oneend_workspace_bytes(L, prec, nrhs=1):
    return load().tm_oneend_workspace_bytes(L.handle, prec, nrhs)


def tm_oneend_loops(L, gauge, prec, recon, s_full, kind, kappa, mu, nrhs, out, workspace, stream=None):
    ws_bytes = workspace.numel() * workspace.element_size()
    return _check(load().tm_oneend_loops(L.handle, _ptr(gauge), prec, recon, _ptr(s_full), kind, kappa, mu, nrhs, _ptr(out),
                                         _ptr(workspace), ws_bytes, _stream(stream)), "tm_oneend_loops")


def tm_tsm_combine(T, loops_hp, loops_lp_same, n_hp, loops_lp, n_lp, out, stream=None):
    return _check(load().tm_tsm_combine(T, _ptr(loops_hp), _ptr(loops_lp_same), n_hp, _ptr(loops_lp), n_lp, _ptr(out),
                                        _stream(stream)), "tm_tsm_combine")


def tm_tsm_workspace_bytes(L, prec_lp, nrhs):
    return load().tm_tsm_workspace_bytes(L.handle, prec_lp, nrhs)


def tm_tsm_batch_host(L, gauge_lp, prec_lp, recon, codes_host, params, nrhs, loops_host, workspace, stream=None):
    info = (tm_cg_info * nrhs)()
    ws_bytes = workspace.numel() * workspace.element_size()
    rc = load().tm_tsm_batch_host(L.handle, _ptr(gauge_lp), prec_lp, recon, _ptr(codes_host), ctypes.byref(params), nrhs, info,
                                  _ptr(loops_host), _ptr(workspace), ws_bytes, _stream(stream))
    _check(rc, "tm_tsm_batch_host", allow=_SOFT)
    return rc, list(info)


def tm_covdev(L, gauge, prec, recon, out_full, in_full, mu, nrhs=1, stream=None):
    return _check(load().tm_covdev(L.handle, _ptr(gauge), prec, recon, _ptr(out_full), _ptr(in_full), mu, nrhs, _stream(stream)),
                  "tm_covdev")


def tm_contract_field(L, a_full, b_full, prec, nrhs, out, stream=None):
    return _check(load().tm_contract_field(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs, _ptr(out), _stream(stream)),
                  "tm_contract_field")


def tm_loop_momentum_workspace_bytes(L, nrhs, n_momenta, pmax):
    return load().tm_loop_momentum_workspace_bytes(L.handle, nrhs, n_momenta, pmax)


def tm_loop_momentum(L, a_full, b_full, prec, nrhs, momenta, out, workspace, stream=None):
    """momenta: host int array [K][3]."""
    m = np.ascontiguousarray(momenta, dtype=np.int32)
    ws_bytes = workspace.numel() * workspace.element_size()
    return _check(load().tm_loop_momentum(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs,
                                          m.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), int(m.shape[0]), _ptr(out), _ptr(workspace),
                                          ws_bytes, _stream(stream)), "tm_loop_momentum")


def tm_time_dilute(L, in_full, prec, nrhs, keep_slice, out_full, stream=None):
    """keep_slice: host sequence of T flags."""
    k = bytes(bytearray(1 if v else 0 for v in keep_slice))
    return _check(load().tm_time_dilute(L.handle, _ptr(in_full), prec, nrhs, k, _ptr(out_full), _stream(stream)), "tm_time_dilute")


def tm_loop_contract_slice(L, a_full, b_full, prec, nrhs, t0, out, workspace, stream=None):
    return _check(load().tm_loop_contract_slice(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs, int(t0), _ptr(out), _ptr(workspace),
                                                _stream(stream)), "tm_loop_contract_slice")


def tm_hpe_remainder(L, gauge, prec, recon, out_full, s_full, tmp_full, kappa, mu, nrhs=1, stream=None):
    return _check(load().tm_hpe_remainder(L.handle, _ptr(gauge), prec, recon, _ptr(out_full), _ptr(s_full), _ptr(tmp_full), kappa, mu,
                                          nrhs, _stream(stream)), "tm_hpe_remainder")


def tm_hpe_local_traces(kappa, mu):
    """Per-site exact HPE terms, complex [16] (host arithmetic in the library)."""
    out = (ctypes.c_double * 32)()
    _check(load().tm_hpe_local_traces(kappa, mu, out), "tm_hpe_local_traces")
    return np.array(out[:]).view(np.complex128)


def tm_spinor_pack_z4_bits(L, codes3, prec, nrhs, packed_out, stream=None):
    return _check(load().tm_spinor_pack_z4_bits(L.handle, _ptr(codes3), prec, nrhs, _ptr(packed_out), _stream(stream)),
                  "tm_spinor_pack_z4_bits")


def tm_gauge_fix_temporal(L, U_canonical, g_out, stream=None):
    return _check(load().tm_gauge_fix_temporal(L.handle, _ptr(U_canonical), _ptr(g_out), _stream(stream)), "tm_gauge_fix_temporal")


def tm_gauge_synthetic(L, seed, w, eps, U_canonical_out, stream=None):
    return _check(load().tm_gauge_synthetic(L.handle, int(seed), float(w), float(eps), _ptr(U_canonical_out), _stream(stream)), "tm_gauge_synthetic")


def tm_noise_z4(L, seed, seed_stride, prec, nrhs, packed_out, stream=None):
    return _check(load().tm_noise_z4(L.handle, int(seed), int(seed_stride), prec, nrhs, _ptr(packed_out), _stream(stream)), "tm_noise_z4")


def tm_tsm_batch_host_bits(L, gauge_lp, prec_lp, recon, codes3_host, params, nrhs, loops_host, workspace, stream=None):
    info = (tm_cg_info * nrhs)()
    ws_bytes = workspace.numel() * workspace.element_size()
    rc = load().tm_tsm_batch_host_bits(L.handle, _ptr(gauge_lp), prec_lp, recon, _ptr(codes3_host), ctypes.byref(params), nrhs, info,
                                       _ptr(loops_host), _ptr(workspace), ws_bytes, _stream(stream))
    _check(rc, "tm_tsm_batch_host_bits", allow=_SOFT)
    return rc, list(info)


def tm_launch_count():
    return int(load().tm_launch_count())


def tm_kernel_timing_enable(on):
    return _check(load().tm_kernel_timing_enable(int(on)), "tm_kernel_timing_enable")


def tm_kernel_timing_read(reset=True):
    ms = ctypes.c_double()
    n = ctypes.c_longlong()
    _check(load().tm_kernel_timing_read(ctypes.byref(ms), ctypes.byref(n), int(reset)), "tm_kernel_timing_read")
    return ms.value, n.value


def tm_loop_contract_static(L, a_full, b_full, prec, nrhs, out, stream=None):
    return _check(load().tm_loop_contract_static(L.handle, _ptr(a_full), _ptr(b_full), prec, nrhs, _ptr(out), _stream(stream)),
                  "tm_loop_contract_static")


def tm_kernel_signature():
    return load().tm_kernel_signature().decode()


def device_buffer(nbytes, device="cuda"):
    """Plumbing: a 256-byte aligned uint8 device buffer owned by PyTorch."""
    t = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=device)
    off = (-t.data_ptr()) % 256
    return t[off:off + int(nbytes)]


__all__ = [n for n in dir() if n.startswith(("tm_", "TM_"))] + ["Lattice", "TmError", "make_cg_params", "device_buffer", "load",
                                                                 "LIB_PATH", "ABI_SYMBOLS"]
