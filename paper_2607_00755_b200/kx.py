"""ctypes binding of libkx (include/kx.h).  Argument marshalling only: every step of the path runs in
the CUDA kernels.  torch is used for device memory (`Tensor.data_ptr()`) and streams, nothing else.

The method names mirror the C entry points: kx_build -> Handle(...), kx_collide -> Handle.collide, ...
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import warnings

import numpy as np

from . import build as _build

INTERP_LOG, INTERP_LINEAR = 0, 1
STORE_SYM_ROWS, STORE_TILED = 0, 1
STAT_CLASSICAL, STAT_BOSE, STAT_FERMI = 0, 1, -1
FP64 = 0
FP32 = 1
EXP_TABLE, EXP_LIBM = 0, 1
PROJECT, DIAG = 1, 2
EULER, HEUN, RK4 = 0, 1, 2

_STATUS = {0: "KX_OK", 1: "KX_ERR_INVALID_ARG", 2: "KX_ERR_ALLOC", 3: "KX_ERR_CUDA",
           4: "KX_ERR_UNSUPPORTED", 5: "KX_ERR_NONFINITE"}

_dp = C.POINTER(C.c_double)


class KxError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int32), ("p", _dp), ("dp", _dp)]


class _Species(C.Structure):
    _fields_ = [("m", C.c_double), ("g_chi", C.c_double)]


class _Msq(C.Structure):
    _fields_ = [("M2_0", C.c_double), ("m_med", C.c_double)]


class _Opts(C.Structure):
    _fields_ = [("interp", C.c_int32), ("storage", C.c_int32), ("precision", C.c_int32),
                ("exp_impl", C.c_int32), ("loss_nodes", C.c_int32), ("statistics", C.c_int32), ("n_mu", C.c_int32), ("reserved", C.c_int32),
                ("f_floor", C.c_double), ("eps_supp", C.c_double)]


class _Source(C.Structure):
    _fields_ = [("nsrc", C.c_int32), ("G", C.c_void_p), ("amp", _dp)]


class _Evolve(C.Structure):
    _fields_ = [("method", C.c_int32), ("S", C.c_int32), ("tau", _dp), ("rate", _dp), ("mass", _dp),
                ("kappa", _dp), ("flags", C.c_uint32), ("diag", C.c_void_p)]


class _Adaptive(C.Structure):
    _fields_ = [("u0", C.c_double), ("u1", C.c_double), ("du0", C.c_double), ("rtol", C.c_double), ("atol", C.c_double),
                ("safety", C.c_double), ("rate0", C.c_double), ("rate_slope", C.c_double), ("kappa", _dp), ("amp", _dp),
                ("max_steps", C.c_int32), ("flags", C.c_uint32), ("mass_slope", C.c_double), ("du_fixed", C.c_double),
                ("eps_switch", C.c_double)]


class _AdaptiveResult(C.Structure):
    _fields_ = [("u", C.c_double), ("du", C.c_double), ("accepted", C.c_int64), ("rejected", C.c_int64),
                ("done", C.c_int32), ("switched", C.c_int32), ("u_switch", C.c_double), ("fixed_steps", C.c_int64),
                ("ratio", C.c_double)]


# every symbol include/kx.h declares
SYMBOLS = ["kx_build", "kx_set_mass", "kx_collide", "kx_collide_static", "kx_collide_parts", "kx_collide_ex",
           "kx_collide_host", "kx_moments", "kx_evolve", "kx_evolve_adaptive", "kx_delta_source", "kx_info", "kx_tensor_export",
           "kx_kinematics_export", "kx_reserve", "kx_fallback_members", "kx_profile", "kx_profile_read", "kx_trace", "kx_trace_read",
           "kx_probe_flops", "kx_plan_probe", "kx_last_error", "kx_destroy", "kx_version"]
TRACE_CTAS, TRACE_SLOTS = 160, 32

_lib = None


def library_path() -> str:
    return _build.LIB


def build_library(force: bool = False) -> str:
    return _build.build(force=force)


def _load():
    """Load libkx.so.  Fails loudly when it is missing and cannot be built: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_build.LIB):
        _build.build()
    elif _build.needs_build():       # a source is newer than the library: never run a stale build silently
        try:
            _build.build()
        except (OSError, subprocess.CalledProcessError) as e:
            warnings.warn(f"libkx.so is older than its sources and could not be rebuilt ({e}); loading it as it is",
                          RuntimeWarning)
    lib = C.CDLL(_build.LIB)
    vp, i32, u32, i64p = C.c_void_p, C.c_int32, C.c_uint32, C.POINTER(C.c_int64)
    lib.kx_build.argtypes = [C.POINTER(_Grid), C.POINTER(_Species), C.POINTER(_Msq), C.POINTER(_Opts),
                             C.c_int, vp, C.POINTER(vp)]
    lib.kx_set_mass.argtypes = [vp, C.c_double, vp]
    lib.kx_collide.argtypes = [vp, vp, vp, i32, u32, vp]
    lib.kx_collide_static.argtypes = [vp, vp, vp, i32, u32, vp]
    lib.kx_collide_parts.argtypes = [vp, vp, vp, vp, i32, vp]
    lib.kx_collide_ex.argtypes = [vp, vp, vp, vp, vp, vp, i32, u32, vp]
    lib.kx_collide_host.argtypes = [vp, vp, vp, i32, u32, vp]
    lib.kx_moments.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp]
    lib.kx_evolve.argtypes = [vp, vp, i32, C.POINTER(_Source), C.POINTER(_Evolve), vp]
    lib.kx_evolve_adaptive.argtypes = [vp, vp, i32, C.POINTER(_Source), C.POINTER(_Adaptive),
                                       C.POINTER(_AdaptiveResult), vp]
    lib.kx_delta_source.argtypes = [vp, C.c_double, vp, vp]
    lib.kx_info.argtypes = [vp, i64p, i64p, C.POINTER(i32)]
    lib.kx_tensor_export.argtypes = [vp, C.c_int64, i64p, _dp, _dp, C.POINTER(C.c_uint32)]
    lib.kx_kinematics_export.argtypes = [vp, _dp, _dp, _dp]
    lib.kx_reserve.argtypes = [vp, i32, vp]
    lib.kx_fallback_members.argtypes = [vp, i64p]
    lib.kx_trace.argtypes = [vp, i32]
    lib.kx_trace_read.argtypes = [vp, C.POINTER(C.c_uint64)]
    lib.kx_profile.argtypes = [vp, i32]
    lib.kx_profile_read.argtypes = [vp, _dp, i64p]
    lib.kx_probe_flops.argtypes = [C.c_int, i32, _dp]
    lib.kx_plan_probe.argtypes = [i32, i32, i32, i32, C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
    lib.kx_last_error.argtypes = [vp]
    lib.kx_last_error.restype = C.c_char_p
    lib.kx_destroy.argtypes = [vp]
    lib.kx_destroy.restype = None
    lib.kx_version.restype = i32
    for name in SYMBOLS:
        if name not in ("kx_last_error", "kx_destroy", "kx_version"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def plan_probe(N: int, B: int, groups_per_tile, Q: int = 24, sm_count: int = 148) -> dict:
    """kx_plan_probe: the host-side launch plan of the tensor-core kernel (no device needed)."""
    lib = _load()
    g = np.ascontiguousarray(groups_per_tile, dtype=np.uint32)
    NT = (N + 15) // 16
    if g.size != NT:
        raise ValueError("groups_per_tile must have ceil(N/16) entries")
    head = (C.c_int32 * 8)()
    wstart = (C.c_uint32 * (NT + 1))()
    ld = (C.c_uint32 * 8)()
    rc = lib.kx_plan_probe(N, B, Q, sm_count, g.ctypes.data_as(C.POINTER(C.c_uint32)), head, wstart, ld)
    if rc != 0:
        raise KxError(rc, "kx_plan_probe")
    return dict(GG=head[0], GL=head[1], nbt=head[2], WC=head[3], NT=head[4], RS=head[5], LC=head[6], smem=head[7],
                wstart=np.array(wstart[:], dtype=np.int64), ld0=np.array(ld[:4], dtype=np.int64), ld1=np.array(ld[4:], dtype=np.int64))


def exported_symbols() -> list[str]:
    """Names from include/kx.h that libkx.so really exports (used by the CPU-side ABI test)."""
    lib = _load()
    return [s for s in SYMBOLS if hasattr(lib, s)]


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _stream(stream):
    import torch
    if stream is None:
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev(t, B=None, N=None):
    """Check a device tensor and return its pointer."""
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


class Handle:
    """kx_build: kinematics, index map and kernel tensor on the device for one (grid, species, |M|^2)."""

    def __init__(self, p, dp, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, *, interp=INTERP_LOG,
                 exp_impl=EXP_TABLE, storage=STORE_TILED, loss_nodes=0, statistics=STAT_CLASSICAL, n_mu=0, f_floor=1e-300,
                 eps_supp=1e-12, precision=FP64, device=0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise KxError(3, "no CUDA device: libkx has no CPU fallback")
        lib = _load()
        self._lib = lib
        self._h = C.c_void_p()
        p, dp = _f64(p), _f64(dp)
        if p.shape != dp.shape or p.ndim != 1:
            raise ValueError("p and dp must be 1-D arrays of the same length")
        self.N = int(p.size)
        self.device = int(device)
        grid = _Grid(self.N, _ptr(p), _ptr(dp))
        sp = _Species(float(m), float(g_chi))
        msq = _Msq(float(M2_0), float(m_med))
        opts = _Opts(int(interp), int(storage), int(precision), int(exp_impl), int(loss_nodes), int(statistics), int(n_mu), 0, float(f_floor),
                     float(eps_supp))
        with torch.cuda.device(self.device):
            rc = lib.kx_build(C.byref(grid), C.byref(sp), C.byref(msq), C.byref(opts), self.device,
                              _stream(stream), C.byref(self._h))
        if rc != 0:
            raise KxError(rc, (lib.kx_last_error(None) or b"").decode())

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc):
        if rc != 0:
            raise KxError(rc, (self._lib.kx_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.kx_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _batch(self, f):
        if f.dim() != 2 or f.shape[1] != self.N:
            raise ValueError(f"f must be [B, {self.N}]")
        return int(f.shape[0])

    # ------------------------------------------------------------------ the C entry points
    def set_mass(self, m, stream=None):
        self._check(self._lib.kx_set_mass(self._h, float(m), _stream(stream)))

    def collide(self, f, flags=0, out=None, stream=None):
        """kx_collide: C[B,N] (raw, or projected with PROJECT)."""
        import torch
        B = self._batch(f)
        out = torch.empty_like(f) if out is None else out
        self._check(self._lib.kx_collide(self._h, _dev(f), _dev(out), B, int(flags), _stream(stream)))
        return out

    def collide_static(self, f, flags=0, out=None, stream=None):
        """kx_collide_static: the operator through the entry point that allocates nothing (static device scratch).  `out`
        must be given by callers that may not allocate; it is created here only as a convenience when omitted."""
        import torch
        B = self._batch(f)
        if out is None:
            out = torch.empty_like(f)
        self._check(self._lib.kx_collide_static(self._h, _dev(f), _dev(out), B, int(flags), _stream(stream)))
        return out

    def collide_parts(self, f, stream=None):
        """kx_collide_parts: gain[B,N], loss[B,N]."""
        import torch
        B = self._batch(f)
        g, l = torch.empty_like(f), torch.empty_like(f)
        self._check(self._lib.kx_collide_parts(self._h, _dev(f), _dev(g), _dev(l), B, _stream(stream)))
        return g, l

    def collide_ex(self, f, flags=0, want=("C", "gain", "loss", "diag"), stream=None):
        """kx_collide_ex: dict with any of C, gain, loss [B,N] and diag [B,4]."""
        import torch
        B = self._batch(f)
        o = {k: (torch.empty((B, 4), dtype=torch.float64, device=f.device) if k == "diag" else torch.empty_like(f))
             for k in want}
        self._check(self._lib.kx_collide_ex(self._h, _dev(f), _dev(o.get("C")), _dev(o.get("gain")),
                                            _dev(o.get("loss")), _dev(o.get("diag")), B, int(flags),
                                            _stream(stream)))
        return o

    def collide_host(self, f_host, C_host, flags=0, stream=None):
        """kx_collide_host: HOST buffers (numpy arrays or pinned CPU tensors), copies inside the call."""
        B = int(f_host.shape[0])
        fp = f_host.data_ptr() if hasattr(f_host, "data_ptr") else f_host.ctypes.data
        cp = C_host.data_ptr() if hasattr(C_host, "data_ptr") else C_host.ctypes.data
        self._check(self._lib.kx_collide_host(self._h, C.c_void_p(fp), C.c_void_p(cp), B, int(flags),
                                              _stream(stream)))
        return C_host

    def moments(self, f, stream=None):
        """kx_moments: tensor [4,B] = n, rho, <p>, <p^2>."""
        import torch
        B = self._batch(f)
        out = torch.empty((4, B), dtype=torch.float64, device=f.device)
        ptrs = [C.c_void_p(out[k].data_ptr()) for k in range(4)]
        self._check(self._lib.kx_moments(self._h, _dev(f), B, *ptrs, _stream(stream)))
        return out

    def evolve(self, f, tau, *, method=RK4, rate=None, mass=None, kappa=None, project=True,
               G=None, amp=None, want_diag=False, stream=None):
        """kx_evolve: advances f [B,N] in place over the steps tau[0..S]; returns diag [S,B,6] or None."""
        import torch
        B = self._batch(f)
        tau = _f64(tau)
        S = int(tau.size) - 1
        rate = None if rate is None else _f64(rate)
        mass = None if mass is None else _f64(mass)
        kappa = None if kappa is None else _f64(kappa)
        if rate is not None and rate.size != 2 * S + 1:
            raise ValueError("rate must have 2S+1 entries")
        if mass is not None and mass.size != 2 * S + 1:
            raise ValueError("mass must have 2S+1 entries")
        if kappa is not None and kappa.size != B:
            raise ValueError("kappa must have B entries")
        src = None
        if G is not None:
            if G.dim() != 2 or G.shape[1] != self.N:
                raise ValueError("G must be [nsrc, N]")
            amp = _f64(amp)
            if amp.shape != (G.shape[0], S):
                raise ValueError("amp must be [nsrc, S]")
            src = _Source(int(G.shape[0]), _dev(G), _ptr(amp))
        diag = torch.zeros((S, B, 6), dtype=torch.float64, device=f.device) if want_diag else None
        flags = (PROJECT if project else 0) | (DIAG if want_diag else 0)
        ctl = _Evolve(int(method), S, _ptr(tau), _ptr(rate), _ptr(mass), _ptr(kappa), flags,
                      _dev(diag) if diag is not None else None)
        self._check(self._lib.kx_evolve(self._h, _dev(f), B, C.byref(src) if src is not None else None,
                                        C.byref(ctl), _stream(stream)))
        return diag

    def evolve_adaptive(self, f, u0, u1, *, du0=1e-4, rtol=1e-2, atol=2e-8, safety=0.9, rate0=1.0, rate_slope=0.0,
                        mass_slope=0.0, du_fixed=0.0, eps_switch=0.0, kappa=None, project=True, G=None, amp=None,
                        max_steps=100000, stream=None):
        """kx_evolve_adaptive: the time integration of Sec. 4.2 in u (sources only on fixed intervals until
        Gamma_2->2/H > eps_switch when eps_switch > 0, then adaptive Heun; kinematic mass m exp(mass_slope (u - u0)));
        f [B,N] in place; returns dict(u, du, accepted, rejected, done, switched, u_switch, fixed_steps, ratio)."""
        B = self._batch(f)
        kappa = None if kappa is None else _f64(kappa)
        if kappa is not None and kappa.size != B:
            raise ValueError("kappa must have B entries")
        src = None
        if G is not None and amp is not None:
            if G.dim() != 2 or G.shape[1] != self.N:
                raise ValueError("G must be [nsrc, N]")
            amp = _f64(amp)
            if amp.shape != (G.shape[0],):
                raise ValueError("amp must be [nsrc]")
            src = _Source(int(G.shape[0]), _dev(G), None)
        else:
            amp = None
        ctl = _Adaptive(float(u0), float(u1), float(du0), float(rtol), float(atol), float(safety), float(rate0),
                        float(rate_slope), _ptr(kappa), _ptr(amp), int(max_steps), PROJECT if project else 0,
                        float(mass_slope), float(du_fixed), float(eps_switch))
        res = _AdaptiveResult()
        self._check(self._lib.kx_evolve_adaptive(self._h, _dev(f), B, C.byref(src) if src is not None else None,
                                                 C.byref(ctl), C.byref(res), _stream(stream)))
        return dict(u=res.u, du=res.du, accepted=int(res.accepted), rejected=int(res.rejected), done=bool(res.done),
                    switched=bool(res.switched), u_switch=res.u_switch, fixed_steps=int(res.fixed_steps), ratio=res.ratio)

    def delta_source(self, p0, stream=None):
        """kx_delta_source: shape [N] of a monoenergetic source at p0 for the current mass."""
        import torch
        G = torch.empty(self.N, dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._lib.kx_delta_source(self._h, float(p0), C.c_void_p(G.data_ptr()), _stream(stream)))
        return G

    def reserve(self, B, stream=None):
        """kx_reserve: allocate workspaces and launch plan for batches up to B now (later calls only enqueue work)."""
        self._check(self._lib.kx_reserve(self._h, int(B), _stream(stream)))

    def fallback_members(self):
        """kx_fallback_members: (member, evaluation) pairs that took the exact fallback since the last call."""
        n = C.c_int64()
        self._check(self._lib.kx_fallback_members(self._h, C.byref(n)))
        return int(n.value)

    def trace(self, enable=True):
        self._check(self._lib.kx_trace(self._h, int(bool(enable))))

    def trace_read(self):
        """kx_trace_read: %globaltimer stamps [160 CTAs, 32 slots] (ns, 0 = not written) of the last launches."""
        out = np.zeros((TRACE_CTAS, TRACE_SLOTS), dtype=np.uint64)
        self._check(self._lib.kx_trace_read(self._h, out.ctypes.data_as(C.POINTER(C.c_uint64))))
        return out

    def profile(self, enable=True):
        self._check(self._lib.kx_profile(self._h, int(bool(enable))))

    def profile_read(self):
        """kx_profile_read: (summed contraction-kernel milliseconds, launches) since the last read."""
        ms, n = C.c_double(), C.c_int64()
        self._check(self._lib.kx_profile_read(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def probe_flops(self, kind=1):
        """kx_probe_flops: measured peak TFLOP/s of the handle's device (0 = DFMA, 1 = DMMA.8x8x4)."""
        v = C.c_double()
        self._check(self._lib.kx_probe_flops(self.device, int(kind), C.byref(v)))
        return v.value

    def info(self):
        nnz, tb, n = C.c_int64(), C.c_int64(), C.c_int32()
        self._check(self._lib.kx_info(self._h, C.byref(nnz), C.byref(tb), C.byref(n)))
        return dict(nnz=nnz.value, tensor_bytes=tb.value, N=n.value)

    def tensor_export(self):
        """kx_tensor_export: rowptr[N+1], W[nnz], omega[nnz], n[nnz], m[nnz], jL[nnz] as numpy arrays."""
        nnz = self.info()["nnz"]
        rowptr = np.empty(self.N + 1, dtype=np.int64)
        W, om = np.empty(nnz), np.empty(nnz)
        nmj = np.empty(nnz, dtype=np.uint32)
        self._check(self._lib.kx_tensor_export(self._h, nnz, rowptr.ctypes.data_as(C.POINTER(C.c_int64)),
                                               _ptr(W), _ptr(om), nmj.ctypes.data_as(C.POINTER(C.c_uint32))))
        return dict(rowptr=rowptr, W=W, omega=om, n=(nmj & 1023).astype(np.int64),
                    m=((nmj >> 10) & 1023).astype(np.int64), jL=(nmj >> 20).astype(np.int64))

    def kinematics_export(self):
        E, K, h = np.empty(self.N), np.empty(self.N), np.empty(self.N)
        self._check(self._lib.kx_kinematics_export(self._h, _ptr(E), _ptr(K), _ptr(h)))
        return E, K, h
