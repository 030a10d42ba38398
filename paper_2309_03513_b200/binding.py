"""Thin ctypes binding of libtddft_b200.so: argument marshalling only, same names as include/tddft.h.

Every numerical step runs inside the CUDA library.  PyTorch supplies device memory and streams only.
Importing this module never falls back to a CPU implementation: if the shared library is missing the
import raises, and if no CUDA device is present `tddft_init` returns TDDFT_ECUDA.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtddft_b200.so")

TDDFT_SPIN_CONSERVING, TDDFT_SPIN_FLIP, TDDFT_SPIN_FLIP_DOWN_UP = 0, 1, 2
TDDFT_OK, TDDFT_EINVAL, TDDFT_ENOMEM, TDDFT_ECUDA, TDDFT_ENOTCONVERGED, TDDFT_EUNSUPPORTED = range(6)

EXPORTS = [
    "tddft_enumerate_gvectors", "tddft_init", "tddft_npw_half", "tddft_gvectors", "tddft_vector_len",
    "tddft_workspace_bytes", "tddft_apply_liouville", "tddft_apply_liouville_host", "tddft_davidson",
    "tddft_set_timing", "tddft_get_stats", "tddft_pair_potentials", "tddft_project", "tddft_gram",
    "tddft_orbital_real_space", "tddft_last_error", "tddft_destroy", "tddft_apply_coupling", "tddft_orbital_overlap",
    "tddft_exchange_apply", "tddft_fp64_peak", "tddft_stream_probe", "tddft_gram_static",
]


class tddft_options(C.Structure):
    _fields_ = [
        ("struct_size", C.c_int), ("use_hartree_fxc", C.c_int), ("rho_floor", C.c_double),
        ("vloc_up", C.c_void_p), ("vloc_dn", C.c_void_p), ("cuda_stream", C.c_void_p),
        ("workspace_gb", C.c_double), ("pair_tile", C.c_int), ("fft_batch", C.c_int),
        ("max_subspace", C.c_int), ("max_iter", C.c_int), ("tol", C.c_double),
        ("x0", C.c_void_p), ("n_x0", C.c_int), ("seed", C.c_ulonglong), ("fft_path", C.c_int),
        ("block", C.c_int), ("precond", C.c_int), ("verbose", C.c_int),
        ("sf_xc_kernel", C.c_int), ("sf_cut", C.c_double),
        ("wannier_u_up", C.c_void_p), ("wannier_u_dn", C.c_void_p), ("s_thr", C.c_double),
        ("pair_list_up", C.c_void_p), ("n_pairs_up", C.c_long), ("pair_list_dn", C.c_void_p), ("n_pairs_dn", C.c_long),
        ("ace", C.c_int), ("psi_ace_up", C.c_void_p), ("n_ace_extra_up", C.c_int),
        ("psi_ace_dn", C.c_void_p), ("n_ace_extra_dn", C.c_int),
        ("work_l2_mb", C.c_double), ("tile_width", C.c_int), ("plan", C.c_int), ("shard_rank", C.c_int), ("shard_count", C.c_int),
    ]


class tddft_stats(C.Structure):
    _fields_ = [("kernel_launches", C.c_longlong), ("pair_ffts", C.c_longlong), ("ms_total", C.c_double),
                ("ms_s1_to_real", C.c_double), ("ms_s23_hxc", C.c_double), ("ms_s4_pair_fft", C.c_double),
                ("ms_s5_contract", C.c_double), ("ms_s6_to_sphere", C.c_double), ("ms_s8_project", C.c_double),
                ("ms_s7_rotate_ace", C.c_double),
                ("fft_batch", C.c_int), ("fft_path", C.c_int), ("pair_batch", C.c_int), ("pair_tile", C.c_int),
                ("k_chunk", C.c_int), ("blocks_resident", C.c_int), ("tile_width", C.c_int)]


def load_library():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libtddft_b200.so is not built: run `python -m paper_2309_03513_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.tddft_last_error.restype = C.c_char_p
    lib.tddft_last_error.argtypes = [C.c_void_p]
    return lib


_lib = load_library()


class TddftError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("tddft status %d: %s" % (status, msg))
        self.status = status


def _check(rc, ctx=None):
    if rc != TDDFT_OK:
        msg = _lib.tddft_last_error(ctx)
        raise TddftError(rc, msg.decode() if msg else "")


def _ptr(t):
    """Device (torch tensor) or raw integer pointer."""
    if t is None:
        return None
    if isinstance(t, int):
        return C.c_void_p(t)
    return C.c_void_p(t.data_ptr())


def tddft_enumerate_gvectors(lattice, ecut_wfc_ry):
    """Returns (miller[npwh,3] int32, g2[npwh] float64)."""
    lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
    n = C.c_long(0)
    rc = _lib.tddft_enumerate_gvectors(lat.ctypes.data_as(C.c_void_p), C.c_double(ecut_wfc_ry), C.c_long(0), None, None, C.byref(n))
    _check(rc)
    miller = np.zeros((n.value, 3), dtype=np.int32)
    g2 = np.zeros(n.value, dtype=np.float64)
    rc = _lib.tddft_enumerate_gvectors(lat.ctypes.data_as(C.c_void_p), C.c_double(ecut_wfc_ry), C.c_long(n.value),
                                       miller.ctypes.data_as(C.c_void_p), g2.ctypes.data_as(C.c_void_p), C.byref(n))
    _check(rc)
    return miller, g2


class Context:
    """Owns a tddft_ctx*.  Keeps references to the borrowed device tensors (psi, vloc, x0) alive."""

    def __init__(self, handle, keep):
        self._h = handle
        self._keep = keep

    def destroy(self):
        if self._h:
            _lib.tddft_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def tddft_init(lattice, grid, ecut_wfc_ry, nspin, nocc, psi_up, psi_dn, eig_up, eig_dn, alpha, **opt):
    """psi_*: CUDA torch tensors complex128 [nocc, npwh]; eig_*: host arrays; opt: fields of tddft_options."""
    lat = np.ascontiguousarray(lattice, dtype=np.float64).reshape(9)
    g = (C.c_int * 3)(*[int(x) for x in grid])
    no = (C.c_int * 2)(int(nocc[0]), int(nocc[1]) if len(nocc) > 1 else 0)
    eu = np.ascontiguousarray(eig_up, dtype=np.float64)
    ed = None if eig_dn is None else np.ascontiguousarray(eig_dn, dtype=np.float64)
    o = tddft_options()
    o.struct_size = C.sizeof(tddft_options)
    o.use_hartree_fxc = -1
    keep = [psi_up, psi_dn]
    for k, v in opt.items():
        if k in ("vloc_up", "vloc_dn", "x0", "psi_ace_up", "psi_ace_dn"):        # device tensors
            keep.append(v)
            setattr(o, k, None if v is None else v.data_ptr())
            if k.startswith("psi_ace") and v is not None:
                setattr(o, "n_ace_extra_" + k[-2:], int(v.shape[0]))
        elif k in ("wannier_u_up", "wannier_u_dn"):                               # host matrices, read during init
            if v is not None:
                u = np.ascontiguousarray(v, dtype=np.float64)
                keep.append(u)
                setattr(o, k, u.ctypes.data)
        elif k in ("pair_list_up", "pair_list_dn"):                               # host int pairs, read during init
            if v is not None:
                pl = np.ascontiguousarray(v, dtype=np.int32).reshape(-1, 2)
                keep.append(pl)
                setattr(o, k, pl.ctypes.data if len(pl) else np.zeros(2, dtype=np.int32).ctypes.data)
                if not len(pl):
                    keep.append(np.zeros(2, dtype=np.int32)); setattr(o, k, keep[-1].ctypes.data)
                setattr(o, "n_pairs_" + k[-2:], len(pl))
        elif k == "cuda_stream":
            o.cuda_stream = v
        else:
            setattr(o, k, v)
    h = C.c_void_p(None)
    rc = _lib.tddft_init(C.byref(h), lat.ctypes.data_as(C.c_void_p), g, C.c_double(ecut_wfc_ry), C.c_int(nspin), no,
                         _ptr(psi_up), _ptr(psi_dn), eu.ctypes.data_as(C.c_void_p),
                         None if ed is None else ed.ctypes.data_as(C.c_void_p), C.c_double(alpha), C.byref(o))
    _check(rc)
    return Context(h, keep)


def tddft_npw_half(ctx):
    n = C.c_long(0)
    _check(_lib.tddft_npw_half(ctx._h, C.byref(n)), ctx._h)
    return n.value


def tddft_gvectors(ctx):
    m = np.zeros((tddft_npw_half(ctx), 3), dtype=np.int32)
    _check(_lib.tddft_gvectors(ctx._h, m.ctypes.data_as(C.c_void_p)), ctx._h)
    return m


def tddft_vector_len(ctx, mode):
    n = C.c_long(0)
    _check(_lib.tddft_vector_len(ctx._h, C.c_int(mode), C.byref(n)), ctx._h)
    return n.value


def tddft_workspace_bytes(ctx):
    n = C.c_longlong(0)
    _check(_lib.tddft_workspace_bytes(ctx._h, C.byref(n)), ctx._h)
    return n.value


def tddft_apply_liouville(ctx, X, AX, nvec, mode=TDDFT_SPIN_CONSERVING):
    """X, AX: CUDA torch tensors complex128 [nvec, vector_len] (AX is written)."""
    _check(_lib.tddft_apply_liouville(ctx._h, _ptr(X), _ptr(AX), C.c_int(nvec), C.c_int(mode)), ctx._h)


def allreduce_sum_(t, group=None):
    """Sum a tensor over the ranks of a torch.distributed group, in place (NCCL on CUDA tensors, gloo on CPU tensors)."""
    import torch
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(torch.view_as_real(t) if t.is_complex() else t, op=dist.ReduceOp.SUM, group=group)
    return t


def tddft_apply_liouville_sharded(ctx, X, AX, nvec, mode, group=None):
    """One apply sharded over the ranks of `group`: every rank holds a context created with shard_rank = its rank and
    shard_count = the group size, the same orbitals and the same X; each applies the exchange tiles it owns and the partial results
    are summed by ONE all-reduce of AX (NCCL over NVLink).  Argument marshalling + the collective only."""
    tddft_apply_liouville(ctx, X, AX, nvec, mode)
    return allreduce_sum_(AX, group)


def tddft_apply_liouville_host(ctx, X_host, AX_host, nvec, mode=TDDFT_SPIN_CONSERVING):
    """X_host, AX_host: numpy complex128 arrays or (pinned) CPU torch tensors."""
    def hp(a):
        return C.c_void_p(a.ctypes.data) if isinstance(a, np.ndarray) else C.c_void_p(a.data_ptr())
    _check(_lib.tddft_apply_liouville_host(ctx._h, hp(X_host), hp(AX_host), C.c_int(nvec), C.c_int(mode)), ctx._h)


def tddft_davidson(ctx, nroots, mode=TDDFT_SPIN_CONSERVING, evecs=None, allow_unconverged=False):
    """Returns (evals[nroots], iters, resnorms[nroots]); evecs: optional CUDA tensor [nroots, vector_len]."""
    ev = np.zeros(nroots, dtype=np.float64)
    rn = np.zeros(nroots, dtype=np.float64)
    it = C.c_int(0)
    rc = _lib.tddft_davidson(ctx._h, C.c_int(nroots), C.c_int(mode), ev.ctypes.data_as(C.c_void_p), _ptr(evecs),
                             C.byref(it), rn.ctypes.data_as(C.c_void_p))
    if not (allow_unconverged and rc == TDDFT_ENOTCONVERGED):
        _check(rc, ctx._h)
    return ev, it.value, rn


def tddft_set_timing(ctx, enabled):
    _check(_lib.tddft_set_timing(ctx._h, C.c_int(1 if enabled else 0)), ctx._h)


def tddft_get_stats(ctx):
    s = tddft_stats()
    _check(_lib.tddft_get_stats(ctx._h, C.byref(s)), ctx._h)
    return {k: getattr(s, k) for k, _ in tddft_stats._fields_}


def tddft_pair_potentials(ctx, spin, pairs, tau):
    p = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    _check(_lib.tddft_pair_potentials(ctx._h, C.c_int(spin), p.ctypes.data_as(C.c_void_p), C.c_long(len(p)), _ptr(tau)), ctx._h)


def tddft_project(ctx, spin, Y, nfun):
    _check(_lib.tddft_project(ctx._h, C.c_int(spin), _ptr(Y), C.c_long(nfun)), ctx._h)


def tddft_gram(ctx, V, W, m, n_complex):
    G = np.zeros((m, m), dtype=np.float64)
    _check(_lib.tddft_gram(ctx._h, _ptr(V), _ptr(W), C.c_int(m), C.c_long(n_complex), G.ctypes.data_as(C.c_void_p)), ctx._h)
    return G


TDDFT_GRAM_STATIC_MAX_M = 256


def tddft_gram_static(ctx, V, W, m, n_complex, G):
    """G (DEVICE float64 [m][m]) = <V_i|W_j> with the partial sums in the library's static device array: no allocation, no
    synchronisation; G is valid once the context's stream has passed the call (include/tddft.h)."""
    _check(_lib.tddft_gram_static(ctx._h, _ptr(V), _ptr(W), C.c_int(m), C.c_long(n_complex), _ptr(G)), ctx._h)


def tddft_orbital_real_space(ctx, spin, v, out):
    _check(_lib.tddft_orbital_real_space(ctx._h, C.c_int(spin), C.c_int(v), _ptr(out)), ctx._h)


def tddft_apply_coupling(ctx, X, BX, nvec, mode=TDDFT_SPIN_CONSERVING):
    """BX = (K2e - K2d) X; spin flip: X in the layout of the opposite flip direction (include/tddft.h)."""
    _check(_lib.tddft_apply_coupling(ctx._h, _ptr(X), _ptr(BX), C.c_int(nvec), C.c_int(mode)), ctx._h)


def tddft_orbital_overlap(ctx, spin, nocc):
    S = np.zeros((nocc, nocc), dtype=np.float64)
    _check(_lib.tddft_orbital_overlap(ctx._h, C.c_int(spin), S.ctypes.data_as(C.c_void_p)), ctx._h)
    return S


def tddft_exchange_apply(ctx, spin, Y, VY, nfun, use_ace=False):
    _check(_lib.tddft_exchange_apply(ctx._h, C.c_int(spin), _ptr(Y), _ptr(VY), C.c_long(nfun), C.c_int(1 if use_ace else 0)), ctx._h)


def tddft_fp64_peak(ctx):
    """(DFMA TFLOP/s, DMMA TFLOP/s) measured on the context's device."""
    a = C.c_double(0.0); b = C.c_double(0.0)
    _check(_lib.tddft_fp64_peak(ctx._h, C.byref(a), C.byref(b)), ctx._h)
    return a.value, b.value


def tddft_stream_probe(ctx, piece_bytes):
    g = C.c_double(0)
    _check(_lib.tddft_stream_probe(ctx._h, C.c_int(piece_bytes), C.byref(g)), ctx._h)
    return g.value


def tddft_last_error(ctx=None):
    msg = _lib.tddft_last_error(None if ctx is None else ctx._h)
    return msg.decode() if msg else ""


def tddft_destroy(ctx):
    ctx.destroy()
