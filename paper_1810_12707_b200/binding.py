"""Thin ctypes binding of libmhd.so (include/mhd.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of `csrc/`; this module only loads the shared library,
declares the C signatures under the same names, and offers `MHD`, a convenience class that lets torch own
the device workspace and the stream (plumbing, not arithmetic).  There is no CPU fallback: if the library
is missing or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmhd.so")

MHD_OK = 0
MHD_HOST, MHD_DEVICE = 0, 1
MHD_CONSERVATIVE, MHD_PRIMITIVE = 0, 1
MHD_OPT_FUSED, MHD_OPT_PRUNE, MHD_OPT_INTEGRATOR, MHD_OPT_FUSE_CURRENT, MHD_OPT_OOC_BRICK, MHD_OPT_OOC_SLAB = 1, 2, 3, 4, 5, 6
MHD_OPT_FUSE_ASSEMBLE = 14
MHD_OPT_TMA = 13
MHD_FLAG_OUT_OF_CORE, MHD_FLAG_STATE_ON_HOST, MHD_FLAG_WORK_ON_HOST = 1, 2, 4
MHD_FLAG_STAGE_STORAGE = 8


def MHD_FLAG_BUDGET_MIB(m):
    return int(m) << 8


ERRORS = {-1: "MHD_ERR_INVALID_ARG", -2: "MHD_ERR_NOT_BOUND", -3: "MHD_ERR_NO_FIELDS", -4: "MHD_ERR_CUDA",
          -5: "MHD_ERR_NOMEM"}

# every symbol include/mhd.h declares (checked by tests/test_abi.py)
SYMBOLS = ["mhd_init", "mhd_workspace_bytes", "mhd_pinned_bytes", "mhd_bind", "mhd_set_option", "mhd_set_fields",
           "mhd_rhs", "mhd_step", "mhd_get_fields", "mhd_diagnostics", "mhd_nspec", "mhd_fft3d_r2c",
           "mhd_fft3d_c2r", "mhd_launch_count", "mhd_transfer_bytes", "mhd_profile_enable", "mhd_profile_get", "mhd_last_error",
           "mhd_destroy", "mhd_tracers_bytes", "mhd_tracers_field_bytes", "mhd_tracers_bind", "mhd_tracers_set", "mhd_tracers_get",
           "mhd_tracers_push", "mhd_set_param", "mhd_probe_fp64", "mhd_dist_config", "mhd_dist_phase",
           "mhd_dist_counts", "mhd_dist_pack", "mhd_dist_unpack", "mhd_dist_ranges", "mhd_dist_peers",
           "mhd_dist_enable_peer_access", "mhd_energy_means_noalloc", "mhd_alt_launch_count"]


class MhdDiag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("ke", C.c_double), ("me", C.c_double),
                ("ie", C.c_double), ("mass", C.c_double), ("mom", C.c_double * 3), ("etot", C.c_double),
                ("max_divb", C.c_double), ("rho_min", C.c_double), ("p_min", C.c_double)]


_lib = None


def lib():
    """Load libmhd.so (fails loudly if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libmhd.so is missing (%s): run `python -m paper_1810_12707_b200.build` "
                           "(or __graft_entry__.build()); the product path has no CPU fallback" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    P8 = C.POINTER(C.c_void_p)
    L.mhd_init.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double]
    L.mhd_workspace_bytes.argtypes = [C.c_int, C.c_uint]
    L.mhd_workspace_bytes.restype = C.c_size_t
    L.mhd_pinned_bytes.argtypes = [C.c_int, C.c_uint]
    L.mhd_pinned_bytes.restype = C.c_size_t
    L.mhd_bind.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_uint, C.c_void_p, C.c_size_t]
    L.mhd_set_option.argtypes = [C.c_void_p, C.c_int, C.c_int]
    L.mhd_set_param.argtypes = [C.c_void_p, C.c_int, C.c_double]
    L.mhd_set_fields.argtypes = [C.c_void_p, C.c_int, C.c_int, P8]
    L.mhd_rhs.argtypes = [C.c_void_p, C.c_int, P8]
    L.mhd_step.argtypes = [C.c_void_p, C.c_int]
    L.mhd_get_fields.argtypes = [C.c_void_p, C.c_int, C.c_int, P8]
    L.mhd_diagnostics.argtypes = [C.c_void_p, C.POINTER(MhdDiag), C.c_void_p, C.c_void_p, C.c_int]
    L.mhd_nspec.argtypes = [C.c_int]
    L.mhd_fft3d_r2c.argtypes = [C.c_void_p, C.c_int, P8, P8, P8, C.c_int]
    L.mhd_fft3d_c2r.argtypes = [C.c_void_p, C.c_int, P8, P8, C.c_int]
    L.mhd_tracers_bytes.argtypes = [C.c_longlong]
    L.mhd_tracers_bytes.restype = C.c_size_t
    L.mhd_tracers_field_bytes.argtypes = [C.c_void_p]
    L.mhd_tracers_field_bytes.restype = C.c_size_t
    L.mhd_tracers_bind.argtypes = [C.c_void_p, C.c_longlong, C.c_void_p, C.c_size_t]
    L.mhd_tracers_set.argtypes = [C.c_void_p, C.c_int, P8, P8]
    L.mhd_tracers_get.argtypes = [C.c_void_p, C.c_int, P8, P8]
    L.mhd_tracers_push.argtypes = [C.c_void_p, C.c_int]
    L.mhd_probe_fp64.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    L.mhd_launch_count.argtypes = [C.c_void_p]
    L.mhd_launch_count.restype = C.c_longlong
    L.mhd_transfer_bytes.argtypes = [C.c_void_p, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]
    L.mhd_profile_enable.argtypes = [C.c_void_p, C.c_int]
    L.mhd_profile_get.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_double),
                                  C.POINTER(C.c_longlong)]
    L.mhd_last_error.argtypes = [C.c_void_p]
    L.mhd_last_error.restype = C.c_char_p
    L.mhd_destroy.argtypes = [C.c_void_p]
    L.mhd_alt_launch_count.argtypes = [C.c_void_p, C.c_int]
    L.mhd_alt_launch_count.restype = C.c_longlong
    L.mhd_energy_means_noalloc.argtypes = [C.c_longlong, C.c_double, P8, C.c_void_p, C.c_void_p, C.c_char_p, C.c_size_t]
    _lib = L
    return L


def _ptr_array(ptrs):
    a = (C.c_void_p * len(ptrs))()
    for i, p in enumerate(ptrs):
        a[i] = p
    return a


NOALLOC_MAX_POINTS = 1 << 30
NOALLOC_KEYS = ("ke", "me", "ie", "mass", "momx", "momy", "momz", "etot", "rho_min", "p_min")


def energy_means_noalloc(fields, gamma, out, stream=None):
    """mhd_energy_means_noalloc (include/mhd.h): scalar diagnostics of 8 real-space conservative fields for callers that
    cannot allocate device memory.  `fields`: 8 contiguous float64 CUDA tensors of equal size; `out`: a float64 CUDA tensor
    of 10 elements that the caller already owns (this wrapper allocates nothing on the device either); `stream`: a
    torch.cuda.Stream or None for the current one.  Asynchronous: read `out` after synchronising the stream."""
    import torch
    assert len(fields) == 8 and all(f.is_cuda and f.dtype == torch.float64 and f.is_contiguous() for f in fields)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 10
    st = stream if stream is not None else torch.cuda.current_stream(fields[0].device)
    err = C.create_string_buffer(256)
    with torch.cuda.device(fields[0].device):
        rc = lib().mhd_energy_means_noalloc(fields[0].numel(), float(gamma), _ptr_array([f.data_ptr() for f in fields]),
                                            out.data_ptr(), st.cuda_stream, err, len(err))
    if rc != MHD_OK:
        raise RuntimeError("libmhd: %s: %s" % (ERRORS.get(rc, rc), err.value.decode()))


class MHD:
    """One solver context on the current CUDA device; torch owns the workspace and the stream."""

    def __init__(self, N, L=2 * math.pi, gamma=5.0 / 3.0, mu=0.0, eta=0.0, dt=1e-3, device="cuda:0", stream=None,
                 flags=0):
        """flags: 0 = in-core; MHD_FLAG_OUT_OF_CORE [| MHD_FLAG_STATE_ON_HOST | MHD_FLAG_WORK_ON_HOST |
        MHD_FLAG_BUDGET_MIB(m)] = the chunked pipeline (include/mhd.h); torch then also owns the pinned host block."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the product path has no CPU fallback")
        self._L = lib()
        self.N = int(N)
        self.torch = torch
        self.device = torch.device(device)
        self._h = C.c_void_p()
        rc = self._L.mhd_init(C.byref(self._h), self.N, L, gamma, mu, eta, dt)
        if rc != MHD_OK:
            raise ValueError("mhd_init: %s" % ERRORS.get(rc, rc))
        self.flags = int(flags)
        nbytes = int(self._L.mhd_workspace_bytes(self.N, self.flags))
        if nbytes == 0:
            self.close()
            raise ValueError("mhd_workspace_bytes: flags 0x%x / device budget not usable for N = %d" % (self.flags, self.N))
        npinned = int(self._L.mhd_pinned_bytes(self.N, self.flags))
        self.workspace_bytes, self.pinned_bytes = nbytes, npinned
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._base = (base + 255) // 256 * 256
            self.pinned = None
            hbase = None
            if npinned:
                self.pinned = torch.empty(npinned + 256, dtype=torch.uint8, pin_memory=True)
                hbase = (self.pinned.data_ptr() + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self._check(self._L.mhd_bind(self._h, self._base, nbytes, self.stream.cuda_stream, self.flags, hbase, npinned))

    # -- helpers ----------------------------------------------------------------------------------------
    def _check(self, rc):
        if rc != MHD_OK:
            raise RuntimeError("libmhd: %s: %s" % (ERRORS.get(rc, rc), self._L.mhd_last_error(self._h).decode()))

    def close(self):
        if getattr(self, "_h", None):
            self._L.mhd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _marshal(self, fields):
        """-> (where, pointer array, keep-alive list) for 8 numpy (host) or torch cuda (device) arrays."""
        torch = self.torch
        n3 = self.N ** 3
        if all(isinstance(f, np.ndarray) for f in fields):
            keep = [np.ascontiguousarray(f, dtype=np.float64) for f in fields]
            assert all(k.size == n3 for k in keep)
            return MHD_HOST, _ptr_array([k.ctypes.data for k in keep]), keep
        assert all(isinstance(f, torch.Tensor) for f in fields)
        keep = [f.contiguous() for f in fields]
        assert all(k.dtype == torch.float64 and k.numel() == n3 for k in keep)
        if all(k.is_cuda for k in keep):
            return MHD_DEVICE, _ptr_array([k.data_ptr() for k in keep]), keep
        assert all(not k.is_cuda for k in keep)      # host tensors (e.g. pinned)
        return MHD_HOST, _ptr_array([k.data_ptr() for k in keep]), keep

    def _new_out(self, where, out):
        torch = self.torch
        shape = (self.N,) * 3
        if out is not None:
            # the library writes through these pointers: a silently made contiguous / float64 copy would receive the
            # result instead of the caller's arrays, so outputs must already be C-contiguous float64 in the right place
            for f in out:
                if isinstance(f, np.ndarray):
                    ok = f.dtype == np.float64 and f.flags["C_CONTIGUOUS"] and f.flags["WRITEABLE"]
                else:
                    ok = f.dtype == torch.float64 and f.is_contiguous()
                if not ok:
                    raise ValueError("output fields must be C-contiguous float64 arrays")
            w, ptrs, _ = self._marshal(out)
            if w != where:
                raise ValueError("output arrays live on the %s but where=%s was requested"
                                 % ("host" if w == MHD_HOST else "device", "host" if where == MHD_HOST else "device"))
            return ptrs, out
        if where == MHD_HOST:
            arrs = [np.empty(shape, dtype=np.float64) for _ in range(8)]
            return _ptr_array([a.ctypes.data for a in arrs]), arrs
        arrs = [torch.empty(shape, dtype=torch.float64, device=self.device) for _ in range(8)]
        return _ptr_array([a.data_ptr() for a in arrs]), arrs

    # -- the ABI calls ------------------------------------------------------------------------------------
    def set_option(self, option, value):
        self._check(self._L.mhd_set_option(self._h, int(option), int(value)))

    def set_param(self, param, value):
        self._check(self._L.mhd_set_param(self._h, int(param), float(value)))

    def set_variant(self, cs2=0.0, f0=0.0, kf=1, evolve=3):
        """Equation-set variants (include/mhd.h MHD_PARAM_CS2, MHD_PARAM_FORCE_AMP, MHD_OPT_FORCE_K, MHD_OPT_EVOLVE)."""
        self.set_param(1, cs2)
        self.set_option(9, kf)
        self.set_param(2, f0)
        self.set_option(8, evolve)

    def set_stress(self, on=True):
        """MHD_OPT_STRESS: viscous terms of Eq. 11-12 (2 nu rho S) instead of mu lap(u)."""
        self.set_option(12, 1 if on else 0)

    def set_fields(self, fields, kind="primitive"):
        where, ptrs, keep = self._marshal(fields)
        self._check(self._L.mhd_set_fields(self._h, MHD_PRIMITIVE if kind == "primitive" else MHD_CONSERVATIVE, where, ptrs))

    def rhs(self, where="host", out=None):
        w = MHD_HOST if where == "host" else MHD_DEVICE
        ptrs, arrs = self._new_out(w, out)
        self._check(self._L.mhd_rhs(self._h, w, ptrs))
        return arrs

    def step(self, n=1):
        self._check(self._L.mhd_step(self._h, int(n)))

    def get_fields(self, kind="conservative", where="host", out=None):
        w = MHD_HOST if where == "host" else MHD_DEVICE
        ptrs, arrs = self._new_out(w, out)
        self._check(self._L.mhd_get_fields(self._h, MHD_PRIMITIVE if kind == "primitive" else MHD_CONSERVATIVE, w, ptrs))
        return arrs

    def nspec(self):
        return int(self._L.mhd_nspec(self.N))

    def diagnostics(self, spectra=False):
        d = MhdDiag()
        if spectra:
            ns = self.nspec()
            sk, sm = np.zeros(ns), np.zeros(ns)
            self._check(self._L.mhd_diagnostics(self._h, C.byref(d), sk.ctypes.data, sm.ctypes.data, ns))
        else:
            sk = sm = None
            self._check(self._L.mhd_diagnostics(self._h, C.byref(d), None, None, 0))
        out = {k: getattr(d, k) for k in ("t", "step", "ke", "me", "ie", "mass", "etot", "max_divb", "rho_min", "p_min")}
        out["mom"] = [d.mom[0], d.mom[1], d.mom[2]]
        if spectra:
            out["spec_kin"], out["spec_mag"] = sk, sm
        return out

    def fft3d_r2c(self, real, spec, nyq=None, prune=False):
        """real/spec/nyq: lists of torch cuda float64 tensors (N^3 / N*N*(N/2)*2 / N*N*8*2 doubles)."""
        n = len(real)
        r = _ptr_array([t.data_ptr() for t in real])
        s = _ptr_array([t.data_ptr() for t in spec])
        q = _ptr_array([t.data_ptr() for t in nyq]) if nyq is not None else None
        self._check(self._L.mhd_fft3d_r2c(self._h, n, r, s, q, int(prune)))

    def fft3d_c2r(self, spec, real, prune=False):
        n = len(real)
        r = _ptr_array([t.data_ptr() for t in real])
        s = _ptr_array([t.data_ptr() for t in spec])
        self._check(self._L.mhd_fft3d_c2r(self._h, n, s, r, int(prune)))

    # -- tracer particles (Sec. VI) ------------------------------------------------------------
    def _marshal3(self, arrs, n):
        torch = self.torch
        if all(isinstance(a, np.ndarray) for a in arrs):
            keep = [np.ascontiguousarray(a, dtype=np.float64) for a in arrs]
            assert all(k.size == n for k in keep)
            return MHD_HOST, _ptr_array([k.ctypes.data for k in keep]), keep
        keep = [a.contiguous() for a in arrs]
        assert all(k.dtype == torch.float64 and k.numel() == n for k in keep)
        where = MHD_DEVICE if keep[0].is_cuda else MHD_HOST
        assert all(k.is_cuda == keep[0].is_cuda for k in keep)
        return where, _ptr_array([k.data_ptr() for k in keep]), keep

    def tracers_set(self, pos, vel=None):
        """Attach len(pos[0]) tracers (torch owns their device storage); vel=None: v0 = CIC of u = m/rho."""
        torch = self.torch
        n = int(pos[0].numel() if isinstance(pos[0], torch.Tensor) else np.asarray(pos[0]).size)
        if getattr(self, "_ntr", 0) != n:
            nbytes = int(self._L.mhd_tracers_bytes(n)) + int(self._L.mhd_tracers_field_bytes(self._h))
            with torch.cuda.device(self.device):
                self._trbuf = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._trbuf.data_ptr() + 255) // 256 * 256
            self._check(self._L.mhd_tracers_bind(self._h, n, base, nbytes))
            self._ntr = n
        where, pp, keep_p = self._marshal3(pos, n)
        if vel is None:
            self._check(self._L.mhd_tracers_set(self._h, where, pp, None))
        else:
            wv, vp, keep_v = self._marshal3(vel, n)
            assert wv == where
            self._check(self._L.mhd_tracers_set(self._h, where, pp, vp))

    def tracers_get(self, where="host"):
        n = self._ntr
        if where == "host":
            pos = [np.empty(n) for _ in range(3)]
            vel = [np.empty(n) for _ in range(3)]
            pp, vp = _ptr_array([a.ctypes.data for a in pos]), _ptr_array([a.ctypes.data for a in vel])
            self._check(self._L.mhd_tracers_get(self._h, MHD_HOST, pp, vp))
        else:
            pos = [self.torch.empty(n, dtype=self.torch.float64, device=self.device) for _ in range(3)]
            vel = [self.torch.empty(n, dtype=self.torch.float64, device=self.device) for _ in range(3)]
            pp, vp = _ptr_array([a.data_ptr() for a in pos]), _ptr_array([a.data_ptr() for a in vel])
            self._check(self._L.mhd_tracers_get(self._h, MHD_DEVICE, pp, vp))
        return pos, vel

    def tracers_push(self, nsteps=1):
        """nsteps Boris pushes in the B of the current state (fields do not advance)."""
        self._check(self._L.mhd_tracers_push(self._h, int(nsteps)))

    def probe_fp64(self):
        """fp64 instructions / s of a register-only DFMA kernel (the fp64 issue ceiling of this GPU)."""
        v = C.c_double()
        self._check(self._L.mhd_probe_fp64(self._h, C.byref(v)))
        return v.value

    def transfer_bytes(self):
        """(host->device, device->host) bytes the chunked pipeline has copied so far."""
        a, b = C.c_longlong(0), C.c_longlong(0)
        self._check(self._L.mhd_transfer_bytes(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def launch_count(self):
        return int(self._L.mhd_launch_count(self._h))

    def alt_launch_count(self, which):
        """Launches of an opt-in alternative kernel so far (which = MHD_OPT_TMA or MHD_OPT_FUSE_ASSEMBLE)."""
        return int(self._L.mhd_alt_launch_count(self._h, int(which)))

    def profile_enable(self, on=True):
        self._check(self._L.mhd_profile_enable(self._h, int(on)))

    def profile_get(self):
        n = 32
        names = (C.c_char_p * n)()
        ms = (C.c_double * n)()
        cnt = (C.c_longlong * n)()
        k = self._L.mhd_profile_get(self._h, n, names, ms, cnt)
        return {names[i].decode(): {"ms": ms[i], "launches": int(cnt[i])} for i in range(k)}
