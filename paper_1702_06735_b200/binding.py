"""Thin ctypes binding of the C-ABI in include/tddp4.h (csrc/libtddp4.so).

Argument marshalling only: every arithmetic step runs in the CUDA kernels behind the C-ABI.  PyTorch is
used for device memory and streams.  There is no CPU fallback: if the library is missing or no CUDA
device is usable the calls raise.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libtddp4.so")

OK, ERR_ARG, ERR_CUDA, ERR_CAPACITY, ERR_DOMAIN, ERR_NONFINITE, ERR_STATE = 0, -1, -2, -3, -4, -5, -6
GET_S, GET_SHAPE, GET_STATIC, GET_COLUMNS, GET_TERMS = range(5)
K_KIN, K_COLUMNS, K_GRAM, K_NLL, K_GEN_RATIO, K_GEN_EMIT, K_COLNLL, K_TRES, K_GRAD = range(9)
PROJECT_STATIC_MAX_BINS = 512   # TDDP4_PROJECT_STATIC_MAX_BINS: size of the static scratch of tddp4_project_static
KERNEL_NAMES = ["kin", "columns", "gram", "nll", "gen_ratio", "gen_emit", "columns_nll", "time_rows", "nll_grad"]

# every symbol include/tddp4.h declares
SYMBOLS = ["tddp4_create", "tddp4_destroy", "tddp4_set_stream", "tddp4_last_error", "tddp4_version",
           "tddp4_load_events", "tddp4_set_params", "tddp4_nll", "tddp4_nll_async", "tddp4_nll_result",
           "tddp4_nll_parts", "tddp4_nll_grad", "tddp4_param_stride", "tddp4_nll_batch", "tddp4_gram", "tddp4_gram_override", "tddp4_norm", "tddp4_generate", "tddp4_weight_bound",
           "tddp4_candidates", "tddp4_get", "tddp4_layout", "tddp4_profile", "tddp4_profile_read",
           "tddp4_profile_reset", "tddp4_launch_count", "tddp4_gram_enqueue", "tddp4_gram_reduce", "tddp4_nll_enqueue",
           "tddp4_gram_state", "tddp4_fp64_peak", "tddp4_project", "tddp4_jit_source", "tddp4_math_probe", "tddp4_set_gram_mode", "tddp4_profile_in_kernel",
           "tddp4_project_static", "tddp4_profile_in_kernel_of"]


class Tddp4Error(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"tddp4 error {code}: {text}")
        self.code = code


class _Res(C.Structure):
    _fields_ = [("L", C.c_int), ("lineshape", C.c_int), ("r", C.c_double)]


class _Term(C.Structure):
    _fields_ = [("spin_factor", C.c_int), ("res", C.c_int * 2), ("perm", C.c_int * 4), ("coupling", C.c_int)]


class _Desc(C.Structure):
    _fields_ = [("m_parent", C.c_double), ("m_final", C.c_double * 4), ("r_res", C.c_double),
                ("r_parent", C.c_double), ("n_res", C.c_int), ("res", C.POINTER(_Res)), ("n_terms", C.c_int),
                ("terms", C.POINTER(_Term)), ("n_couplings", C.c_int), ("t_lo", C.c_double), ("t_hi", C.c_double),
                ("use_resolution", C.c_int)]


_lib = None


def load_library():
    """dlopen csrc/libtddp4.so; raises if it has not been built (python -m paper_1702_06735_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1702_06735_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, dbl, dp = C.c_void_p, C.c_int64, C.c_double, C.POINTER(C.c_double)
    L.tddp4_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
    L.tddp4_destroy.argtypes = [vp]
    L.tddp4_set_stream.argtypes = [vp, vp]
    L.tddp4_last_error.argtypes = [vp]
    L.tddp4_last_error.restype = C.c_char_p
    L.tddp4_version.restype = C.c_char_p
    L.tddp4_load_events.argtypes = [vp, C.c_int, i64, i64, vp, vp, vp, vp, C.c_int]
    L.tddp4_set_params.argtypes = [vp, vp, vp, vp, dbl, dbl, dbl]
    L.tddp4_nll.argtypes = [vp, dp, vp]
    L.tddp4_nll_grad.argtypes = [vp, dp, vp]
    L.tddp4_nll_async.argtypes = [vp, C.c_int]
    L.tddp4_nll_result.argtypes = [vp, C.c_int, dp]
    L.tddp4_nll_parts.argtypes = [vp, C.c_int, dp]
    L.tddp4_param_stride.argtypes = [vp]
    L.tddp4_nll_batch.argtypes = [vp, i64, vp, vp, vp]
    L.tddp4_gram.argtypes = [vp, vp, C.POINTER(i64)]
    L.tddp4_gram_override.argtypes = [vp, vp, i64]
    L.tddp4_norm.argtypes = [vp, dp]
    L.tddp4_generate.argtypes = [vp, C.c_uint64, C.c_uint32, i64, i64, i64, dbl, i64, vp, vp, vp,
                                 C.POINTER(i64), C.POINTER(i64), dp]
    L.tddp4_weight_bound.argtypes = [vp, dp]
    L.tddp4_candidates.argtypes = [vp, C.c_uint64, C.c_uint32, i64, i64, vp, vp, vp, vp, vp]
    L.tddp4_get.argtypes = [vp, C.c_int, C.c_int, vp]
    L.tddp4_layout.argtypes = [vp] + [C.POINTER(C.c_int)] * 6
    L.tddp4_profile.argtypes = [vp, C.c_int]
    L.tddp4_profile_read.argtypes = [vp, C.c_int, dp, C.POINTER(i64), dp]
    L.tddp4_profile_reset.argtypes = [vp]
    L.tddp4_launch_count.argtypes = [vp]
    L.tddp4_launch_count.restype = i64
    L.tddp4_gram_enqueue.argtypes = [vp, vp]
    L.tddp4_gram_reduce.argtypes = [vp, vp, C.c_int, i64]
    L.tddp4_nll_enqueue.argtypes = [vp, vp]
    L.tddp4_gram_state.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.tddp4_fp64_peak.argtypes = [vp, dp]
    L.tddp4_jit_source.argtypes = [C.POINTER(_Desc), C.c_int, C.c_int, C.c_int, C.c_char_p, i64]
    L.tddp4_jit_source.restype = i64
    L.tddp4_math_probe.argtypes = [vp, C.c_int, i64, vp, vp, vp]
    L.tddp4_set_gram_mode.argtypes = [vp, C.c_int, C.POINTER(i64)]
    L.tddp4_profile_in_kernel.argtypes = [vp, dp, C.POINTER(i64)]
    L.tddp4_profile_in_kernel_of.argtypes = [vp, C.c_int, dp, C.POINTER(i64)]
    L.tddp4_project.argtypes = [vp, i64, i64, vp, C.c_int, vp, vp, vp]
    L.tddp4_project_static.argtypes = [vp, i64, i64, vp, C.c_int, vp, vp, vp]
    _lib = L
    return L


def _ptr(t):
    """Device (torch) or host (numpy) buffer -> raw address; None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _make_desc(model):
    """workloads.Model-like object -> (tddp4_model_desc, the ctypes arrays it points to)."""
    res = (_Res * max(1, model.n_res))()
    radii = getattr(model, "res_r", None) or [0.0] * model.n_res
    kinds = getattr(model, "res_lineshape", None) or [0] * model.n_res
    for r, L in enumerate(model.res_L):
        res[r].L, res[r].lineshape, res[r].r = L, kinds[r], radii[r]
    terms = (_Term * model.n_terms)()
    for k in range(model.n_terms):
        terms[k].spin_factor = model.term_sf[k]
        terms[k].res[0], terms[k].res[1] = model.term_res[k]
        for r in range(4):
            terms[k].perm[r] = model.term_perm[k][r]
        terms[k].coupling = model.term_coupling[k]
    d = _Desc()
    d.m_parent = model.m_parent
    for i in range(4):
        d.m_final[i] = model.m_final[i]
    d.r_res, d.r_parent = model.r_res, model.r_parent
    d.n_res, d.res, d.n_terms, d.terms = model.n_res, res, model.n_terms, terms
    d.n_couplings, d.t_lo, d.t_hi, d.use_resolution = model.n_couplings, model.t_lo, model.t_hi, model.use_resolution
    return d, (res, terms)


def jit_source(model, what, weighted=False, mode=0):
    """tddp4_jit_source: the CUDA text the library hands to NVRTC for this model (what = 0 Gram pass, 1 data pass) or one
    of the headers it includes (2 jit_shared.cuh, 3 nll_shared.cuh).  Needs no GPU."""
    lib = load_library()
    d, keep = _make_desc(model)
    need = lib.tddp4_jit_source(C.byref(d), what, int(weighted), mode, None, 0)
    if need < 0:
        raise Tddp4Error(int(need), "tddp4_jit_source")
    buf = C.create_string_buffer(int(need))
    lib.tddp4_jit_source(C.byref(d), what, int(weighted), mode, buf, need)
    return buf.value.decode()


class Tddp4:
    """One handle of the C-ABI library.  `model` is a workloads.Model-like plain-data object."""

    def __init__(self, model, device="cuda:0"):
        import torch

        self._torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("tddp4 needs a CUDA device; there is no CPU fallback")
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        torch.cuda.init()
        torch.zeros(1, device=self.device)           # make sure the primary context exists
        self.model = model
        self.n_res, self.n_terms, self.kc = model.n_res, model.n_terms, model.n_couplings
        d, self._desc_keep = _make_desc(model)
        self._h = C.c_void_p()
        rc = self.lib.tddp4_create(C.byref(d), C.byref(self._h))
        if rc != OK:
            text = self.lib.tddp4_last_error(self._h).decode() if self._h else "create failed"
            if self._h:
                self.lib.tddp4_destroy(self._h)
            self._h = None
            raise Tddp4Error(rc, text)
        self.n = [0, 0]
        self.stream = None
        c, cb = np.empty(self.kc, np.complex128), np.empty(self.kc, np.complex128)
        mw = np.zeros((max(1, self.n_res), 2))
        self._pbuf = (c, cb, mw, c.ctypes.data, cb.ctypes.data, mw.ctypes.data)
        self.h2d_bytes_per_call = c.nbytes + cb.nbytes + (mw.nbytes if self.n_res else 0) + 24
        self._nll_out = C.c_double()
        self._nll_ref = C.byref(self._nll_out)

    @property
    def n_data(self):
        return self.n[0]

    # -- plumbing ---------------------------------------------------------------------------------
    def _check(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise Tddp4Error(rc, self.lib.tddp4_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self.lib.tddp4_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_stream(self, stream):
        """stream: torch.cuda.Stream (or None for the legacy default stream)."""
        self._check(self.lib.tddp4_set_stream(self._h, stream.cuda_stream if stream is not None else None))
        self.stream = stream

    def empty(self, *shape, dtype=None):
        return self._torch.empty(*shape, dtype=dtype or self._torch.float64, device=self.device)

    # -- tddp4_load_events ------------------------------------------------------------------------
    def load_events(self, which, p4, t=None, sigma_t=None, weight=None):
        """p4: [16][n] fp64, torch CUDA tensor (read in place) or numpy array (copied from the host)."""
        on_device = not isinstance(p4, np.ndarray)
        if on_device:
            assert p4.is_cuda and p4.dtype == self._torch.float64 and p4.dim() == 2 and p4.shape[0] == 16
            assert p4.stride(1) == 1
            n, ld = p4.shape[1], (p4.stride(0) if p4.shape[1] > 1 else max(1, p4.shape[1]))
            self._torch.cuda.current_stream(self.device).synchronize()
        else:
            p4 = np.ascontiguousarray(p4, dtype=np.float64)
            n, ld = p4.shape[1], p4.shape[1]
            t = None if t is None else np.ascontiguousarray(t, dtype=np.float64)
            sigma_t = None if sigma_t is None else np.ascontiguousarray(sigma_t, dtype=np.float64)
            weight = None if weight is None else np.ascontiguousarray(weight, dtype=np.float64)
        self._keep = (p4, t, sigma_t, weight)
        self._check(self.lib.tddp4_load_events(self._h, which, n, ld, _ptr(p4), _ptr(t), _ptr(sigma_t), _ptr(weight),
                                               1 if on_device else 0))
        self._keep = None
        self.n[which] = n

    # -- tddp4_set_params -------------------------------------------------------------------------
    def set_params(self, par, dbar=False):
        """par: workloads.Params-like (c, cbar complex arrays; mass, width; x, y, tau).  dbar: this handle holds a
        D0bar-tagged sample, for which the two amplitudes of eq. (1) exchange their roles: the coupling vectors are
        handed over in the opposite order (marshalling only)."""
        b = self._pbuf                                   # preallocated marshalling buffers: no allocation per call
        b[0][:] = par.cbar if dbar else par.c
        b[1][:] = par.c if dbar else par.cbar
        if self.n_res:
            b[2][:, 0] = par.mass
            b[2][:, 1] = par.width
        self._check(self.lib.tddp4_set_params(self._h, b[3], b[4], b[5], par.x, par.y, par.tau))

    # -- tddp4_nll and friends --------------------------------------------------------------------
    def nll(self, prob_out=None, strict=True):
        rc = self.lib.tddp4_nll(self._h, self._nll_ref, None if prob_out is None else _ptr(prob_out))
        if rc != OK and (strict or rc != ERR_NONFINITE):
            self._check(rc)
        return self._nll_out.value if rc == OK else math.inf

    def nll_grad(self):
        """(NLL, gradient[4 K_c + 2]) for the current parameters; layout as tddp4_nll_grad."""
        out = C.c_double()
        g = np.empty(4 * self.kc + 2)
        self._check(self.lib.tddp4_nll_grad(self._h, C.byref(out), g.ctypes.data))
        return out.value, g

    def nll_async(self, slot):
        self._check(self.lib.tddp4_nll_async(self._h, slot))

    def nll_result(self, slot, strict=True):
        out = C.c_double()
        rc = self._check(self.lib.tddp4_nll_result(self._h, slot, C.byref(out)), allow=() if strict else (ERR_NONFINITE,))
        return out.value if rc == OK else math.inf

    def nll_parts(self, slot=0):
        out = (C.c_double * 5)()
        self._check(self.lib.tddp4_nll_parts(self._h, slot, out))
        return dict(sum_log_B=out[0], sum_t=out[1], norm=out[2], nll=out[3], n_bad=out[4])

    def pack_params(self, points):
        """[Params-like] -> host array [n_points][stride] in the layout tddp4_nll_batch reads."""
        stride = self.lib.tddp4_param_stride(self._h)
        out = np.empty((len(points), stride))
        kc, nr = self.kc, self.n_res
        for i, p in enumerate(points):
            out[i, 0:2 * kc] = np.asarray(p.c, dtype=np.complex128).view(np.float64)
            out[i, 2 * kc:4 * kc] = np.asarray(p.cbar, dtype=np.complex128).view(np.float64)
            out[i, 4 * kc:4 * kc + 2 * nr:2] = p.mass
            out[i, 4 * kc + 1:4 * kc + 2 * nr:2] = p.width
            out[i, -3:] = (p.x, p.y, p.tau)
        return out

    def nll_batch(self, packed, strict=True):
        """packed: pack_params() output.  Returns (nll[n_points], status[n_points])."""
        packed = np.ascontiguousarray(packed, dtype=np.float64)
        n = packed.shape[0]
        out = np.empty(n)
        st = np.zeros(n, dtype=np.int32)
        rc = self.lib.tddp4_nll_batch(self._h, n, packed.ctypes.data, out.ctypes.data, st.ctypes.data)
        if strict:
            self._check(rc)
        return out, st

    def gram(self):
        G = np.empty((self.kc, self.kc, 2))
        n = C.c_int64()
        self._check(self.lib.tddp4_gram(self._h, G.ctypes.data, C.byref(n)))
        return G[..., 0] + 1j * G[..., 1], n.value

    def gram_override(self, G_sum, n_norm):
        G = np.ascontiguousarray(np.stack([np.real(G_sum), np.imag(G_sum)], axis=-1), dtype=np.float64)
        self._check(self.lib.tddp4_gram_override(self._h, G.ctypes.data, int(n_norm)))

    # -- event-sharded evaluation: everything stays on the handle's stream --------------------------------
    def gram_enqueue(self, G_dev):
        """G_dev: CUDA tensor [2 K_c^2 + 1] <- this rank's Gram sums and its normalisation event count."""
        self._check(self.lib.tddp4_gram_enqueue(self._h, _ptr(G_dev)))

    def gram_reduce(self, gathered_dev, world, n_norm_total):
        """gathered_dev: CUDA tensor [world][2 K_c^2 + 1]; the rank-ordered sum becomes the Gram matrix in force."""
        self._check(self.lib.tddp4_gram_reduce(self._h, _ptr(gathered_dev), int(world), int(n_norm_total)))

    def nll_enqueue(self, result_dev):
        """result_dev: CUDA tensor [8] <- (sum log B, sum t, N, NLL term, #bad, stamp, -, -) of this rank."""
        self._check(self.lib.tddp4_nll_enqueue(self._h, _ptr(result_dev)))

    def gram_state(self):
        v, o = C.c_int(), C.c_int()
        self._check(self.lib.tddp4_gram_state(self._h, C.byref(v), C.byref(o)))
        return bool(v.value), bool(o.value)

    def fp64_peak(self):
        out = C.c_double()
        self._check(self.lib.tddp4_fp64_peak(self._h, C.byref(out)))
        return out.value

    def set_gram_mode(self, mode):
        """tddp4_set_gram_mode: 0 full Gram passes (default), 1 stored normalisation columns + incremental passes, -1 query;
        returns the number of incremental passes run so far."""
        out = C.c_int64()
        self._check(self.lib.tddp4_set_gram_mode(self._h, mode, C.byref(out)))
        return out.value

    def math_probe(self, what, x, y=None):
        """tddp4_math_probe: 0 1/x, 1 sqrt(x), 2 1/sqrt(x), 3 x/y with the kernels' branch-free primitives; device tensors."""
        out = self._torch.empty_like(x)
        self._check(self.lib.tddp4_math_probe(self._h, what, x.numel(), _ptr(x), _ptr(y), _ptr(out)))
        return out

    def norm(self):
        out = C.c_double()
        self._check(self.lib.tddp4_norm(self._h, C.byref(out)))
        return out.value

    # -- tddp4_generate / tddp4_candidates --------------------------------------------------------
    def generate(self, seed, stream_id, first, n_candidates, n_pilot, envelope_scale, capacity, want_index=False,
                 strict=True):
        T = self._torch
        p4 = self.empty(16, max(1, capacity))
        t = self.empty(max(1, capacity))
        idx = self.empty(max(1, capacity), dtype=T.int64) if want_index else None
        na, no, env = C.c_int64(), C.c_int64(), C.c_double()
        rc = self._check(self.lib.tddp4_generate(self._h, seed, stream_id, first, n_candidates, n_pilot, envelope_scale,
                                                 capacity, _ptr(p4), _ptr(t), _ptr(idx), C.byref(na), C.byref(no),
                                                 C.byref(env)), allow=() if strict else (ERR_CAPACITY,))
        k = min(na.value, capacity)
        return dict(p4=p4[:, :k], t=t[:k], index=None if idx is None else idx[:k], n_accepted=na.value,
                    n_overflow=no.value, envelope=env.value, status=rc)

    def weight_bound(self):
        out = C.c_double()
        self._check(self.lib.tddp4_weight_bound(self._h, C.byref(out)))
        return out.value

    def generate_n(self, seed, stream_id, n_events, n_pilot, envelope_scale, chunk=1 << 24, want_index=False):
        """Loop tddp4_generate over consecutive candidate ranges until n_events are accepted (orchestration
        only).  The envelope is fixed by the first call's pilot.  Returns p4[16][n_events], t, index, info."""
        T = self._torch
        p4 = self.empty(16, n_events)
        t = self.empty(n_events)
        idx = self.empty(n_events, dtype=T.int64) if want_index else None
        got, first, env, over = 0, 0, None, 0
        while got < n_events:
            g = self.generate(seed, stream_id, first, chunk, n_pilot if env is None else 0,
                              envelope_scale if env is None else env, chunk, want_index=want_index)
            env = g["envelope"]
            k = min(g["n_accepted"], n_events - got)
            p4[:, got:got + k] = g["p4"][:, :k]
            t[got:got + k] = g["t"][:k]
            if want_index:
                idx[got:got + k] = g["index"][:k]
            got += k
            first += chunk
            over += g["n_overflow"]
            if g["n_accepted"] == 0 and first > 400 * chunk:
                raise RuntimeError("accept-reject makes no progress")
        return p4, t, idx, dict(envelope=env, n_candidates=first, n_overflow=over)

    def candidates(self, seed, stream_id, first, n):
        p4, t, w, r, u = self.empty(16, n), self.empty(n), self.empty(n), self.empty(n), self.empty(n)
        self._check(self.lib.tddp4_candidates(self._h, seed, stream_id, first, n, _ptr(p4), _ptr(t), _ptr(w), _ptr(r),
                                              _ptr(u)))
        return p4, t, w, r, u

    # -- tddp4_project ----------------------------------------------------------------------------
    def project(self, p4, n_bins, ranges, want_values=False):
        """p4: CUDA tensor [16][n].  Returns (hist int64 [5][n_bins], values CUDA [5][n] or None)."""
        assert p4.is_cuda and p4.dim() == 2 and p4.shape[0] == 16 and p4.stride(1) == 1
        n, ld = p4.shape[1], (p4.stride(0) if p4.shape[1] > 1 else max(1, p4.shape[1]))
        self._torch.cuda.current_stream(self.device).synchronize()
        rng = np.ascontiguousarray(ranges, dtype=np.float64)
        hist = np.zeros((5, n_bins), dtype=np.int64)
        values = self.empty(5, max(1, n)) if want_values else None
        self._check(self.lib.tddp4_project(self._h, n, ld, _ptr(p4), n_bins, rng.ctypes.data, hist.ctypes.data, _ptr(values)))
        return hist, (values[:, :n] if want_values else None)

    def project_static(self, p4, n_bins, ranges, hist_out, values_out=None):
        """tddp4_project_static: the projection with the library's static device scratch, no allocation inside the call.
        p4: CUDA tensor [16][n]; hist_out: the caller's CUDA int64 tensor [5][n_bins]; values_out: the caller's CUDA fp64
        tensor [5][n] or None.  Enqueues on the handle's stream and returns; hist_out is valid once that stream (set_stream) or the device has been synchronised."""
        assert p4.is_cuda and p4.dim() == 2 and p4.shape[0] == 16 and p4.stride(1) == 1
        n, ld = p4.shape[1], (p4.stride(0) if p4.shape[1] > 1 else max(1, p4.shape[1]))
        assert hist_out.is_cuda and hist_out.dtype == self._torch.int64 and hist_out.is_contiguous() and hist_out.numel() >= 5 * max(0, n_bins)
        assert values_out is None or (values_out.is_cuda and values_out.is_contiguous() and tuple(values_out.shape) == (5, n))
        self._torch.cuda.current_stream(self.device).synchronize()
        rng = np.ascontiguousarray(ranges, dtype=np.float64)
        self._check(self.lib.tddp4_project_static(self._h, n, ld, _ptr(p4), n_bins, rng.ctypes.data, _ptr(hist_out), _ptr(values_out)))

    # -- inspection -------------------------------------------------------------------------------
    def layout(self):
        ns, ni = C.c_int(), C.c_int()
        sm, ir, isys, isub = (C.c_int * 16)(), (C.c_int * 32)(), (C.c_int * 32)(), (C.c_int * 32)()
        self._check(self.lib.tddp4_layout(self._h, C.byref(ns), sm, C.byref(ni), ir, isys, isub))
        return dict(sys_mask=list(sm[:ns.value]), inst_res=list(ir[:ni.value]), inst_sys=list(isys[:ni.value]),
                    inst_sub=list(isub[:ni.value]))

    def get(self, which, what):
        n = self.n[which]
        lay = self.layout()
        rows = {GET_S: len(lay["sys_mask"]), GET_SHAPE: len(lay["inst_res"]), GET_STATIC: self.n_terms,
                GET_COLUMNS: self.kc, GET_TERMS: self.n_terms}[what]
        cplx = what in (GET_COLUMNS, GET_TERMS)
        out = self.empty(max(1, rows), n, 2) if cplx else self.empty(max(1, rows), n)
        self._check(self.lib.tddp4_get(self._h, which, what, _ptr(out)))
        out = out[:rows]
        return self._torch.view_as_complex(out) if cplx else out

    def profile(self, enable=True):
        self._check(self.lib.tddp4_profile(self._h, 1 if enable else 0))

    def profile_reset(self):
        self._check(self.lib.tddp4_profile_reset(self._h))

    def profile_read(self):
        """{kernel: (total_ms, launches, algorithmic bytes)} since the last reset."""
        out = {}
        for k, name in enumerate(KERNEL_NAMES):
            ms, n, by = C.c_double(), C.c_int64(), C.c_double()
            self._check(self.lib.tddp4_profile_read(self._h, k, C.byref(ms), C.byref(n), C.byref(by)))
            out[name] = (ms.value, n.value, by.value)
        return out

    def profile_in_kernel(self):
        """tddp4_profile_in_kernel: (sum of in-kernel durations of the coupling-only NLL kernel in us, launches)."""
        us, n = C.c_double(), C.c_int64()
        self._check(self.lib.tddp4_profile_in_kernel(self._h, C.byref(us), C.byref(n)))
        return us.value, n.value

    def profile_in_kernel_of(self, kernel_id):
        """tddp4_profile_in_kernel_of: the same for K_NLL or K_GRAD (the gradient kernel without resolution)."""
        us, n = C.c_double(), C.c_int64()
        self._check(self.lib.tddp4_profile_in_kernel_of(self._h, int(kernel_id), C.byref(us), C.byref(n)))
        return us.value, n.value

    def launch_count(self):
        return int(self.lib.tddp4_launch_count(self._h))
