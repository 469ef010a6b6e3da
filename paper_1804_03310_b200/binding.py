"""Thin ctypes binding of include/afqmc.h (argument marshalling only).

Every arithmetic step runs in the CUDA kernels of libafqmc_b200.so; torch is used for
device memory and the stream handle only.  The library must be built (build.py); if it is
missing or cannot be loaded this module raises -- there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafqmc_b200.so")

AFQMC_OK, AFQMC_EINVAL, AFQMC_EUNSUPPORTED, AFQMC_ECUDA, AFQMC_ENOMEM = range(5)
FLAG_SINGULAR, FLAG_NONFINITE, FLAG_KILLED = 1, 2, 4

SYMBOLS = ["afqmc_query_bytes", "afqmc_init", "afqmc_destroy", "afqmc_last_error", "afqmc_overlap_green",
           "afqmc_force_bias", "afqmc_propagate", "afqmc_local_energy", "afqmc_step", "afqmc_step_host",
           "afqmc_launch_count", "afqmc_gemm_path", "afqmc_profile_enable", "afqmc_profile_read",
           "afqmc_orthonormalize", "afqmc_population_control", "afqmc_run", "afqmc_comb_record_bytes",
           "afqmc_comb_map", "afqmc_comb_pack", "afqmc_comb_unpack", "afqmc_mixed_sums", "afqmc_mixed_energy", "afqmc_peak_probe", "afqmc_peak_mma_table", "afqmc_set_stream", "afqmc_comb_map_noalloc"]

STAGES = ["shift", "assemble", "taylor", "green", "force_bias", "energy", "symmetrize", "ortho", "popctl"]


class AfqmcParams(C.Structure):
    _fields_ = [("M", C.c_int32), ("n_alpha", C.c_int32), ("n_beta", C.c_int32), ("n_chol", C.c_int32),
                ("n_walkers", C.c_int32), ("precision", C.c_int32), ("taylor_order", C.c_int32),
                ("weight_mode", C.c_int32), ("n_det", C.c_int32), ("n_act", C.c_int32), ("max_exc", C.c_int32),
                ("gemm_path", C.c_int32), ("dt", C.c_double), ("E0", C.c_double)]


class AfqmcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"afqmc status {status}: {msg}")
        self.status = status


_lib = None


def load_library():
    """dlopen the C-ABI library; raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: run `python -m paper_1804_03310_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp, i32p, szp = C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)
    pp = C.POINTER(AfqmcParams)
    lib.afqmc_query_bytes.argtypes = [pp, szp, szp]
    lib.afqmc_init.argtypes = [C.POINTER(vp), pp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.afqmc_set_stream.argtypes = [vp, vp]
    lib.afqmc_set_stream.restype = C.c_int
    lib.afqmc_destroy.argtypes = [vp]
    lib.afqmc_destroy.restype = None
    lib.afqmc_last_error.argtypes = [vp]
    lib.afqmc_last_error.restype = C.c_char_p
    lib.afqmc_overlap_green.argtypes = [vp, vp, vp, vp, vp, i32p]
    lib.afqmc_force_bias.argtypes = [vp, vp, vp, vp]
    lib.afqmc_propagate.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32p]
    lib.afqmc_local_energy.argtypes = [vp, vp, vp, vp]
    lib.afqmc_step.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int32, vp, i32p]
    lib.afqmc_step_host.argtypes = [vp, vp, vp, vp, vp, C.c_int32, vp, i32p, szp, szp]
    lib.afqmc_orthonormalize.argtypes = [vp, vp, vp, i32p]
    lib.afqmc_population_control.argtypes = [vp, vp, vp, vp, vp, vp, C.c_double, i32p]
    lib.afqmc_run.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, vp, vp, i32p, i32p]
    lib.afqmc_mixed_sums.argtypes = [vp, vp, vp, vp]
    lib.afqmc_mixed_sums.restype = C.c_int
    dp_ = C.POINTER(C.c_double)
    lib.afqmc_peak_probe.argtypes = [C.c_int32, C.c_int32, C.c_int32, vp, C.c_size_t, vp, dp_, dp_, dp_]
    lib.afqmc_peak_probe.restype = C.c_int
    lib.afqmc_peak_mma_table.argtypes = [vp, C.c_int32, vp, vp, dp_]
    lib.afqmc_peak_mma_table.restype = C.c_int
    lib.afqmc_mixed_energy.argtypes = [vp, vp, C.c_int32, vp]
    lib.afqmc_mixed_energy.restype = C.c_int
    lib.afqmc_comb_record_bytes.argtypes = [vp]
    lib.afqmc_comb_record_bytes.restype = C.c_size_t
    lib.afqmc_comb_map.argtypes = [vp, vp, C.c_int64, C.c_double, vp, i32p, vp]
    lib.afqmc_comb_map_noalloc.argtypes = [vp, vp, C.c_int64, C.c_double, i32p, vp]
    lib.afqmc_comb_map_noalloc.restype = C.c_int
    lib.afqmc_comb_pack.argtypes = [vp, vp, vp, vp, vp, i32p, C.c_int64, C.c_int64, C.c_int64, vp]
    lib.afqmc_comb_unpack.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp]
    lib.afqmc_launch_count.argtypes = [vp]
    lib.afqmc_launch_count.restype = C.c_int64
    lib.afqmc_gemm_path.argtypes = [vp]
    lib.afqmc_gemm_path.restype = C.c_int32
    lib.afqmc_profile_enable.argtypes = [vp, C.c_int32]
    lib.afqmc_profile_read.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_int32)]
    lib.afqmc_profile_enable.restype = C.c_int
    lib.afqmc_profile_read.restype = C.c_int
    for name in ("afqmc_query_bytes", "afqmc_init", "afqmc_overlap_green", "afqmc_force_bias", "afqmc_propagate",
                 "afqmc_local_energy", "afqmc_step", "afqmc_step_host", "afqmc_orthonormalize", "afqmc_population_control",
                 "afqmc_run", "afqmc_comb_map", "afqmc_comb_pack", "afqmc_comb_unpack"):
        getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def make_params(M, n_alpha, n_beta, n_chol, n_walkers, precision, dt, taylor_order=6, weight_mode=0, E0=0.0,
                n_det=1, n_act=0, max_exc=2, gemm_path=0) -> AfqmcParams:
    prec = {"c64": 0, "c128": 1, 0: 0, 1: 1}[precision]
    return AfqmcParams(M, n_alpha, n_beta, n_chol, n_walkers, prec, taylor_order, weight_mode, n_det, n_act,
                       max_exc, gemm_path, float(dt), float(E0))


def afqmc_query_bytes(params: AfqmcParams):
    lib = load_library()
    cb, wb = C.c_size_t(0), C.c_size_t(0)
    st = lib.afqmc_query_bytes(C.byref(params), C.byref(cb), C.byref(wb))
    if st:
        raise AfqmcError(st, lib.afqmc_last_error(None).decode())
    return cb.value, wb.value


def afqmc_peak_probe(kind, n, iters, scratch, stream=None):
    """(ms, units, clk_per_mma) of one peak microbenchmark; scratch = CUDA uint8 tensor (>= 1 MiB)."""
    import torch
    lib = load_library()
    ms, units, clk = C.c_double(0), C.c_double(0), C.c_double(0)
    st = stream if stream is not None else torch.cuda.current_stream(scratch.device)
    with torch.cuda.device(scratch.device):
        rc = lib.afqmc_peak_probe(int(kind), int(n), int(iters), C.c_void_p(scratch.data_ptr()), scratch.numel(),
                                  C.c_void_p(st.cuda_stream), C.byref(ms), C.byref(units), C.byref(clk))
    if rc:
        raise AfqmcError(rc, "afqmc_peak_probe failed")
    return ms.value, units.value, clk.value


def afqmc_peak_mma_table(mmas, iters, scratch, stream=None):
    """mmas: list of (a_offset, b_offset, N, d_column); returns clocks per MMA."""
    import torch
    lib = load_library()
    tab = np.zeros(1 + 4 * 64, dtype=np.int32)
    tab[0] = len(mmas)
    for i, (a, b, n, d) in enumerate(mmas):
        tab[1 + i], tab[65 + i], tab[129 + i], tab[193 + i] = a, b, n, d
    clk = C.c_double(0)
    st = stream if stream is not None else torch.cuda.current_stream(scratch.device)
    rc = lib.afqmc_peak_mma_table(tab.ctypes.data_as(C.c_void_p), int(iters), C.c_void_p(scratch.data_ptr()),
                                  C.c_void_p(st.cuda_stream), C.byref(clk))
    if rc:
        raise AfqmcError(rc, "afqmc_peak_mma_table failed")
    return clk.value


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t):
    """device pointer of a torch tensor (or None)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensor required"
    return C.c_void_p(t.data_ptr())


class AfqmcContext:
    """Owns the opaque afqmc_ctx plus the two device arenas (torch uint8 tensors)."""

    def __init__(self, params: AfqmcParams, h1, L_chol, psiT_a=None, psiT_b=None, C_act=None, det_coeff=None,
                 det_exc=None, device="cuda:0", stream=None):
        import torch
        self._lib = load_library()
        self.params = params
        self.device = torch.device(device)
        cb, wb = afqmc_query_bytes(params)
        self.const_bytes, self.work_bytes = cb, wb
        self.const_mem = torch.empty(cb + 256, dtype=torch.uint8, device=self.device)
        self.work_mem = torch.empty(wb + 256, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.rdtype = torch.float64 if params.precision else torch.float32
        self.cdtype = torch.complex128 if params.precision else torch.complex64
        al = lambda t: (t.data_ptr() + 255) // 256 * 256
        h1, L_chol, psiT_a, psiT_b = _f64(h1), _f64(L_chol), _f64(psiT_a), _f64(psiT_b)
        C_act, det_coeff = _f64(C_act), _f64(det_coeff)
        det_exc = None if det_exc is None else np.ascontiguousarray(det_exc, dtype=np.int32)
        ctx = C.c_void_p(None)
        with torch.cuda.device(self.device):
            st = self._lib.afqmc_init(C.byref(ctx), C.byref(params), _hp(h1), _hp(L_chol), _hp(psiT_a), _hp(psiT_b),
                                      _hp(C_act), _hp(det_coeff), _hp(det_exc), C.c_void_p(al(self.const_mem)),
                                      C.c_void_p(al(self.work_mem)), C.c_void_p(self.stream.cuda_stream))
        if st:
            raise AfqmcError(st, self._lib.afqmc_last_error(None).decode())
        self._ctx = ctx

    def use_stream(self, stream):
        """Enqueue all further work of this context on `stream` (a torch.cuda.Stream), e.g. a CUDA-graph capture stream."""
        st = self._lib.afqmc_set_stream(self._ctx, C.c_void_p(stream.cuda_stream))
        self._chk(st)
        self.stream = stream

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.afqmc_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, st):
        if st:
            raise AfqmcError(st, self._lib.afqmc_last_error(self._ctx).decode())

    @property
    def launch_count(self) -> int:
        return int(self._lib.afqmc_launch_count(self._ctx))

    @property
    def gemm_path(self) -> int:
        return int(self._lib.afqmc_gemm_path(self._ctx))

    def afqmc_profile_enable(self, enable=True):
        self._chk(self._lib.afqmc_profile_enable(self._ctx, 1 if enable else 0))

    def afqmc_profile_read(self):
        """{stage name: (total_ms, recorded executions)}; synchronise the stream first."""
        out = {}
        for i, name in enumerate(STAGES):
            ms, n = C.c_double(0), C.c_int32(0)
            self._chk(self._lib.afqmc_profile_read(self._ctx, i, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, n.value)
        return out

    # ---- same names as the C ABI; tensors are torch CUDA tensors ----
    def afqmc_overlap_green(self, phi, ovlp, theta, G=None, flags=None):
        self._chk(self._lib.afqmc_overlap_green(self._ctx, _dp(phi), _dp(ovlp), _dp(theta), _dp(G), _dp(flags)))

    def afqmc_force_bias(self, phi, theta, fb):
        self._chk(self._lib.afqmc_force_bias(self._ctx, _dp(phi), _dp(theta), _dp(fb)))

    def afqmc_propagate(self, phi, x, fb, ovlp, weight, theta, eloc_pre=None, flags=None):
        self._chk(self._lib.afqmc_propagate(self._ctx, _dp(phi), _dp(x), _dp(fb), _dp(ovlp), _dp(weight), _dp(theta),
                                            _dp(eloc_pre), _dp(flags)))

    def afqmc_local_energy(self, phi, theta, eloc):
        self._chk(self._lib.afqmc_local_energy(self._ctx, _dp(phi), _dp(theta), _dp(eloc)))

    def afqmc_step(self, phi, weight, ovlp, theta, fb, x, n_steps, eloc, flags=None):
        self._chk(self._lib.afqmc_step(self._ctx, _dp(phi), _dp(weight), _dp(ovlp), _dp(theta), _dp(fb), _dp(x),
                                       int(n_steps), _dp(eloc), _dp(flags)))

    def afqmc_orthonormalize(self, phi, ovlp, flags=None):
        self._chk(self._lib.afqmc_orthonormalize(self._ctx, _dp(phi), _dp(ovlp), _dp(flags)))

    def afqmc_population_control(self, phi, weight, ovlp, theta, fb, u, parent=None):
        self._chk(self._lib.afqmc_population_control(self._ctx, _dp(phi), _dp(weight), _dp(ovlp), _dp(theta), _dp(fb),
                                                     float(u), _dp(parent)))

    def afqmc_run(self, phi, weight, ovlp, theta, fb, x, n_steps, energy_every=1, ortho_every=0, pc_every=0, u=None,
                  eloc=None, w_meas=None, parents=None, flags=None):
        """u: host sequence of comb offsets in [0, 1), one per population-control event."""
        ua = None if u is None else np.ascontiguousarray(u, dtype=np.float64)
        self._chk(self._lib.afqmc_run(self._ctx, _dp(phi), _dp(weight), _dp(ovlp), _dp(theta), _dp(fb), _dp(x),
                                      int(n_steps), int(energy_every), int(ortho_every), int(pc_every), _hp(ua),
                                      _dp(eloc), _dp(w_meas), _dp(parents), _dp(flags)))

    def afqmc_mixed_sums(self, weight, eloc, out3):
        self._chk(self._lib.afqmc_mixed_sums(self._ctx, _dp(weight), _dp(eloc), _dp(out3)))

    def afqmc_mixed_energy(self, sums, n, e_mix):
        self._chk(self._lib.afqmc_mixed_energy(self._ctx, _dp(sums), int(n), _dp(e_mix)))

    @property
    def afqmc_comb_record_bytes(self) -> int:
        return int(self._lib.afqmc_comb_record_bytes(self._ctx))

    def afqmc_comb_map(self, weight_all, u, cum_scratch, parent_all, w_new):
        self._chk(self._lib.afqmc_comb_map(self._ctx, _dp(weight_all), int(weight_all.numel()), float(u), _dp(cum_scratch),
                                           _dp(parent_all), _dp(w_new)))

    def afqmc_comb_map_noalloc(self, weight_all, u, parent_all, w_new):
        self._chk(self._lib.afqmc_comb_map_noalloc(self._ctx, _dp(weight_all), int(weight_all.numel()), float(u), _dp(parent_all),
                                                   _dp(w_new)))

    def afqmc_comb_pack(self, phi, ovlp, theta, fb, parent_all, slot_lo, count, first_local, sendbuf):
        self._chk(self._lib.afqmc_comb_pack(self._ctx, _dp(phi), _dp(ovlp), _dp(theta), _dp(fb), _dp(parent_all),
                                            int(slot_lo), int(count), int(first_local), _dp(sendbuf)))

    def afqmc_comb_unpack(self, recvbuf, phi, weight, ovlp, theta, fb, w_new):
        self._chk(self._lib.afqmc_comb_unpack(self._ctx, _dp(recvbuf), _dp(phi), _dp(weight), _dp(ovlp), _dp(theta),
                                              _dp(fb), _dp(w_new)))

    def afqmc_step_host(self, phi_h, weight_h, ovlp_h, x_h, n_steps, eloc_h, flags_h=None):
        """HOST buffers: numpy arrays or CPU (pinned) torch tensors, updated in place. Returns (h2d, d2h) bytes."""
        def hp(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.flags["C_CONTIGUOUS"]
                return a.ctypes.data_as(C.c_void_p)
            assert (not a.is_cuda) and a.is_contiguous()
            return C.c_void_p(a.data_ptr())
        up, down = C.c_size_t(0), C.c_size_t(0)
        self._chk(self._lib.afqmc_step_host(self._ctx, hp(phi_h), hp(weight_h), hp(ovlp_h), hp(x_h), int(n_steps),
                                            hp(eloc_h), hp(flags_h), C.byref(up), C.byref(down)))
        return up.value, down.value
