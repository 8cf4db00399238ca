"""Thin ctypes binding of the C-ABI library (include/alegb.h): argument marshalling only.

Every function has the name of the C entry point it calls.  Device arrays are passed as torch CUDA tensors (their
``data_ptr()`` is handed to the library) or as raw integer device addresses; host arrays as numpy arrays.  Nothing
here computes: if libalegb.so is missing or fails to load, importing this module raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libalegb.so")

OK, INVALID_ARG, BAD_MESH, NOT_READY, UNSUPPORTED, CUDA_ERROR = 0, -1, -2, -3, -4, -5
MOTION_NONE, MOTION_SINES_PRODUCT, MOTION_SINES_CROSS, MOTION_PLUNGE_BLEND, MOTION_CARANGIFORM, MOTION_USER = range(6)
COORDS_CLOSED_FORM, COORDS_RK = 0, 1
RELAX_COLLOCATION, RELAX_CUBATURE = 0, 1
STATUS_NAMES = {0: "OK", -1: "INVALID_ARG", -2: "BAD_MESH", -3: "NOT_READY", -4: "UNSUPPORTED", -5: "CUDA_ERROR"}

if not os.path.exists(LIB_PATH):
    raise ImportError("libalegb.so is not built (run `python -m paper_2607_00199_b200.build`); "
                      "the library has no fallback path")
_lib = ctypes.CDLL(LIB_PATH)

_c = ctypes
_P = _c.c_void_p
_SIGNATURES = {
    "alegb_create": (_c.c_int, [_c.POINTER(_P), _c.c_int, _c.c_int, _c.c_int]),
    "alegb_destroy": (_c.c_int, [_P]),
    "alegb_mesh_upload": (_c.c_int, [_P, _c.c_int64, _P, _c.c_int64, _P, _P, _P, _P]),
    "alegb_set_params": (_c.c_int, [_P, _c.c_double, _c.c_double, _P]),
    "alegb_set_motion": (_c.c_int, [_P, _c.c_int, _P, _c.c_int]),
    "alegb_set_motion_user": (_c.c_int, [_P, _P, _P]),
    "alegb_set_motion_user_stages": (_c.c_int, [_P, _P, _P]),
    "alegb_set_coordinate_mode": (_c.c_int, [_P, _c.c_int, _c.c_double]),
    "alegb_set_relaxation": (_c.c_int, [_P, _c.c_int]),
    "alegb_set_geometry_overlap": (_c.c_int, [_P, _c.c_int]),
    "alegb_set_layer_fusion": (_c.c_int, [_P, _c.c_int]),
    "alegb_wall_forces": (_c.c_int, [_P, _c.c_double, _P, _c.c_int, _P, _P, _P]),
    "alegb_wall_forces_static": (_c.c_int, [_P, _c.c_double, _P, _c.c_int, _c.c_int, _P, _P]),
    "alegb_get_cubature": (_c.c_int, [_P, _c.POINTER(_c.c_int), _c.POINTER(_c.c_int), _P, _P, _P, _P]),
    "alegb_get_positions": (_c.c_int, [_P, _P, _P]),
    "alegb_rhs": (_c.c_int, [_P, _c.c_double, _P, _P, _P]),
    "alegb_rhs_pml": (_c.c_int, [_P, _c.c_double, _P, _P, _P, _P, _P]),
    "alegb_step": (_c.c_int, [_P, _P, _c.c_double, _c.c_double, _c.c_int, _P]),
    "alegb_step_debug": (_c.c_int, [_P, _P, _c.c_double, _c.c_double, _P, _P]),
    "alegb_step_host": (_c.c_int, [_P, _P, _c.c_double, _c.c_double, _c.c_int]),
    "alegb_geometry": (_c.c_int, [_P, _c.c_double, _P, _P, _P, _P, _P]),
    "alegb_pml_count": (_c.c_int64, [_P]),
    "alegb_pml_elements": (_c.c_int, [_P, _P]),
    "alegb_pml_reset": (_c.c_int, [_P, _P]),
    "alegb_pml_get": (_c.c_int, [_P, _P, _P]),
    "alegb_pml_set": (_c.c_int, [_P, _P, _P]),
    "alegb_get_sizes": (_c.c_int, [_P] + [_c.POINTER(_c.c_int)] * 6 + [_c.POINTER(_c.c_int64)] * 2),
    "alegb_get_operators": (_c.c_int, [_P] * 10),
    "alegb_get_reference": (_c.c_int, [_P, _P, _P, _P]),
    "alegb_sark_coefficients": (_c.c_int, [_c.c_double, _P, _P]),
    "alegb_workspace_bytes": (_c.c_int64, [_P]),
    "alegb_last_error": (_c.c_char_p, [_P]),
    "alegb_launch_count": (_c.c_int64, [_P]),
    "alegb_set_kernel": (_c.c_int, [_P, _c.c_int]),
    "alegb_set_max_ctas": (_c.c_int, [_P, _c.c_int]),
    "alegb_pipe_config": (_c.c_int, [_c.c_int, _c.c_int, _P]),
    "alegb_pipe_config_layer": (_c.c_int, [_c.c_int, _c.c_int, _P]),
    "alegb_set_graph": (_c.c_int, [_P, _c.c_int]),
    "alegb_profile_enable": (_c.c_int, [_P, _c.c_int]),
    "alegb_profile_read": (_c.c_int, [_P, _c.POINTER(_c.c_int64), _c.POINTER(_c.c_double)]),
    "alegb_measure_fp64_peak": (_c.c_int, [_P, _c.POINTER(_c.c_double), _c.POINTER(_c.c_double)]),
}
for _name, (_res, _args) in _SIGNATURES.items():
    _fn = getattr(_lib, _name)          # AttributeError here = the library does not export a declared symbol
    _fn.restype, _fn.argtypes = _res, _args
EXPORTED = sorted(_SIGNATURES)


class AlegbError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), message))
        self.status = status


def _dev(x):
    """Device address of a torch CUDA tensor / raw int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if not x.is_cuda or not x.is_contiguous():
        raise ValueError("device arrays must be contiguous CUDA tensors")
    if str(x.dtype) != "torch.float64":
        raise ValueError("device arrays must be float64 (got %s)" % x.dtype)
    return x.data_ptr()


def _host(x, dtype):
    if x is None:
        return None, None
    a = np.ascontiguousarray(x, dtype=dtype)
    return a, a.ctypes.data


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


class Context:
    """Owns one ``alegb_ctx``.  Methods are the C entry points without the ``alegb_`` prefix handling errors."""

    def __init__(self, dim, N, cuda_device=0):
        h = _P()
        rc = _lib.alegb_create(ctypes.byref(h), dim, N, cuda_device)
        if rc != OK:
            raise AlegbError(rc, "alegb_create(dim=%d, N=%d, device=%d) failed" % (dim, N, cuda_device))
        self._h = h
        self.device = cuda_device
        self.dim, self.N, self.Np, self.Nfp, self.Nfaces, self.Nf, self.K, self.Nverts = self.alegb_get_sizes()

    def close(self):
        if getattr(self, "_h", None):
            _lib.alegb_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != OK:
            raise AlegbError(rc, (_lib.alegb_last_error(self._h) or b"").decode())

    # ---- setup
    def alegb_mesh_upload(self, X0, EToV, vertex_equiv=None, EToB=None, pml_sigma=None):
        X0a, X0p = _host(X0, np.float64)
        Ea, Ep = _host(EToV, np.int32)
        va, vp = _host(vertex_equiv, np.int32)
        ba, bp = _host(EToB, np.int8)
        sa, sp = _host(pml_sigma, np.float64)
        if X0a.ndim != 2 or X0a.shape[1] != self.dim or Ea.ndim != 2 or Ea.shape[1] != self.dim + 1:
            raise ValueError("X0 must be [Nverts, dim] and EToV [K, dim+1]")
        self._check(_lib.alegb_mesh_upload(self._h, X0a.shape[0], X0p, Ea.shape[0], Ep, vp, bp, sp))
        self.dim, self.N, self.Np, self.Nfp, self.Nfaces, self.Nf, self.K, self.Nverts = self.alegb_get_sizes()

    def alegb_set_params(self, RT, tau, q_inf=None):
        qa, qp = _host(q_inf, np.float64)
        self._check(_lib.alegb_set_params(self._h, float(RT), float(tau), qp))

    def alegb_set_motion(self, kind, params=None):
        pa, pp = _host(params, np.float64)
        self._check(_lib.alegb_set_motion(self._h, int(kind), pp, 0 if pa is None else pa.size))

    def alegb_set_motion_user(self, d_xv, d_vv):
        self._check(_lib.alegb_set_motion_user(self._h, _dev(d_xv), _dev(d_vv)))

    def alegb_set_motion_user_stages(self, d_xv4, d_vv4):
        """d_xv4 (or None), d_vv4: CUDA tensors [4, Nverts, dim] -- the data of the four RK stages of the next step."""
        self._check(_lib.alegb_set_motion_user_stages(self._h, _dev(d_xv4), _dev(d_vv4)))

    def alegb_wall_forces(self, t, d_q, tag=1, stream=None):
        """-> (F_p[dim], F_v[dim]) host arrays."""
        Fp, Fv = np.zeros(self.dim), np.zeros(self.dim)
        self._check(_lib.alegb_wall_forces(self._h, float(t), _dev(d_q), int(tag), Fp.ctypes.data, Fv.ctypes.data, _stream(stream)))
        return Fp, Fv

    def alegb_wall_forces_static(self, t, d_q, d_F, tag=1, nblocks=0, stream=None):
        """The wall forces for callers that cannot allocate where they need them (see include/alegb.h): d_F is the
        caller's CUDA tensor of 2 dim doubles, filled with (F_p, F_v) on `stream`; the call allocates nothing, copies
        nothing to the host and does not wait.  nblocks = 0 reproduces alegb_wall_forces bit for bit."""
        self._check(_lib.alegb_wall_forces_static(self._h, float(t), _dev(d_q), int(tag), int(nblocks), _dev(d_F), _stream(stream)))

    def alegb_measure_fp64_peak(self):
        """-> (DMMA TFLOP/s, DFMA TFLOP/s) measured on the context's device."""
        a, b = _c.c_double(0.0), _c.c_double(0.0)
        self._check(_lib.alegb_measure_fp64_peak(self._h, _c.byref(a), _c.byref(b)))
        return a.value, b.value

    def alegb_set_geometry_overlap(self, on):
        self._check(_lib.alegb_set_geometry_overlap(self._h, int(bool(on))))

    def alegb_set_layer_fusion(self, on):
        self._check(_lib.alegb_set_layer_fusion(self._h, int(bool(on))))

    def alegb_set_relaxation(self, mode):
        self._check(_lib.alegb_set_relaxation(self._h, int(mode)))

    def alegb_get_cubature(self):
        """-> dict(degree, Nc, rst[dim, Nc], w[Nc], I[Nc, Np], P[Np, Nc]) (host arrays)."""
        deg, nc = _c.c_int(0), _c.c_int(0)
        self._check(_lib.alegb_get_cubature(self._h, _c.byref(deg), _c.byref(nc), None, None, None, None))
        dim, Np, Nc = self.dim, self.Np, nc.value
        rst, w = np.empty((dim, Nc)), np.empty(Nc)
        I, P = np.empty((Nc, Np)), np.empty((Np, Nc))
        self._check(_lib.alegb_get_cubature(self._h, None, None, rst.ctypes.data, w.ctypes.data, I.ctypes.data, P.ctypes.data))
        return dict(degree=deg.value, Nc=Nc, rst=rst, w=w, I=I, P=P)

    def alegb_set_coordinate_mode(self, mode, t_start=0.0):
        self._check(_lib.alegb_set_coordinate_mode(self._h, int(mode), float(t_start)))

    def alegb_get_positions(self, d_x, stream=None):
        self._check(_lib.alegb_get_positions(self._h, _dev(d_x), _stream(stream)))

    # ---- compute (device arrays)
    def alegb_rhs(self, t, d_q, d_F, stream=None):
        self._check(_lib.alegb_rhs(self._h, float(t), _dev(d_q), _dev(d_F), _stream(stream)))

    def alegb_rhs_pml(self, t, d_q, d_aux, d_F, d_Faux, stream=None):
        self._check(_lib.alegb_rhs_pml(self._h, float(t), _dev(d_q), _dev(d_aux), _dev(d_F), _dev(d_Faux), _stream(stream)))

    def alegb_step(self, d_q, t0, dt, nsteps, stream=None):
        self._check(_lib.alegb_step(self._h, _dev(d_q), float(t0), float(dt), int(nsteps), _stream(stream)))

    def alegb_step_debug(self, d_q, t0, dt, d_stages, stream=None):
        self._check(_lib.alegb_step_debug(self._h, _dev(d_q), float(t0), float(dt), _dev(d_stages), _stream(stream)))

    def alegb_step_host(self, h_q, t0, dt, nsteps):
        """h_q: C-contiguous float64 numpy array or CPU torch tensor (pinned or not), updated in place."""
        ptr = h_q.ctypes.data if isinstance(h_q, np.ndarray) else h_q.data_ptr()
        self._check(_lib.alegb_step_host(self._h, ptr, float(t0), float(dt), int(nsteps)))

    def alegb_geometry(self, t, d_vgeo=None, d_sgeo=None, d_xv=None, d_vv=None, stream=None):
        self._check(_lib.alegb_geometry(self._h, float(t), _dev(d_vgeo), _dev(d_sgeo), _dev(d_xv), _dev(d_vv), _stream(stream)))

    # ---- absorbing layer state
    def alegb_pml_count(self):
        return int(_lib.alegb_pml_count(self._h))

    def alegb_pml_elements(self):
        out = np.empty(self.alegb_pml_count(), dtype=np.int32)
        self._check(_lib.alegb_pml_elements(self._h, out.ctypes.data))
        return out

    def alegb_pml_reset(self, stream=None):
        self._check(_lib.alegb_pml_reset(self._h, _stream(stream)))

    def alegb_pml_get(self, d_aux, stream=None):
        self._check(_lib.alegb_pml_get(self._h, _dev(d_aux), _stream(stream)))

    def alegb_pml_set(self, d_aux, stream=None):
        self._check(_lib.alegb_pml_set(self._h, _dev(d_aux), _stream(stream)))

    # ---- introspection (host)
    def alegb_get_sizes(self):
        ints = [_c.c_int() for _ in range(6)]
        longs = [_c.c_int64() for _ in range(2)]
        rc = _lib.alegb_get_sizes(self._h, *[ctypes.byref(v) for v in ints + longs])
        if rc != OK:
            raise AlegbError(rc, "alegb_get_sizes")
        return tuple(int(v.value) for v in ints + longs)

    def alegb_get_operators(self, with_maps=False):
        Np, ncol = self.Np, self.Nfaces * self.Nfp
        out = dict(r=np.empty(Np), s=np.empty(Np), t=np.empty(Np) if self.dim == 3 else None,
                   Dr=np.empty((Np, Np)), Ds=np.empty((Np, Np)), Dt=np.empty((Np, Np)) if self.dim == 3 else None,
                   LIFT=np.empty((Np, ncol)))
        maps = dict(vmapM=None, vmapP=None)
        if with_maps:
            maps = dict(vmapM=np.empty((self.K, self.Nfaces, self.Nfp), dtype=np.int32),
                        vmapP=np.empty((self.K, self.Nfaces, self.Nfp), dtype=np.int32))
        ptr = lambda a: None if a is None else a.ctypes.data
        self._check(_lib.alegb_get_operators(self._h, ptr(out["r"]), ptr(out["s"]), ptr(out["t"]), ptr(out["Dr"]),
                                             ptr(out["Ds"]), ptr(out["Dt"]), ptr(out["LIFT"]), ptr(maps["vmapM"]),
                                             ptr(maps["vmapP"])))
        out.update(maps)
        return out

    def alegb_get_reference(self):
        w = np.empty(self.Np)
        lam = np.empty((self.Np, self.dim + 1))
        fmask = np.empty((self.Nfaces, self.Nfp), dtype=np.int32)
        self._check(_lib.alegb_get_reference(self._h, w.ctypes.data, lam.ctypes.data, fmask.ctypes.data))
        return dict(w=w, lam=lam, fmask=fmask)

    def alegb_workspace_bytes(self):
        return int(_lib.alegb_workspace_bytes(self._h))

    def alegb_launch_count(self):
        return int(_lib.alegb_launch_count(self._h))

    def alegb_set_kernel(self, kind):
        self._check(_lib.alegb_set_kernel(self._h, int(kind)))

    def alegb_set_max_ctas(self, max_ctas):
        self._check(_lib.alegb_set_max_ctas(self._h, int(max_ctas)))

    def alegb_set_graph(self, on):
        self._check(_lib.alegb_set_graph(self._h, int(bool(on))))

    def alegb_profile_enable(self, on):
        self._check(_lib.alegb_profile_enable(self._h, int(bool(on))))

    def alegb_profile_read(self):
        n, ms = _c.c_int64(), _c.c_double()
        self._check(_lib.alegb_profile_read(self._h, ctypes.byref(n), ctypes.byref(ms)))
        return int(n.value), float(ms.value)

    def alegb_last_error(self):
        return (_lib.alegb_last_error(self._h) or b"").decode()


def alegb_sark_coefficients(gamma):
    a = np.empty(6)
    b = np.empty(4)
    rc = _lib.alegb_sark_coefficients(float(gamma), a.ctypes.data, b.ctypes.data)
    if rc != OK:
        raise AlegbError(rc, "alegb_sark_coefficients")
    return a, b


PIPE_CONFIG_FIELDS = ("producer_groups", "slots", "items_per_quad", "consumer_warps", "warps_per_group",
                      "producer_warps", "elements_per_quad", "smem_bytes")


def alegb_pipe_config(dim, N):
    """-> dict of the hand-over parameters of the pipelined stage kernel for (dim, N); raises UNSUPPORTED if none."""
    out = (_c.c_int * 8)()
    rc = _lib.alegb_pipe_config(int(dim), int(N), out)
    if rc != OK:
        raise AlegbError(rc, "alegb_pipe_config(dim=%d, N=%d)" % (dim, N))
    return dict(zip(PIPE_CONFIG_FIELDS, (int(v) for v in out)))


def alegb_pipe_config_layer(dim, N):
    """The same for the instantiation with the absorbing layer fused in (alegb_set_layer_fusion)."""
    out = (_c.c_int * 8)()
    rc = _lib.alegb_pipe_config_layer(int(dim), int(N), out)
    if rc != OK:
        raise AlegbError(rc, "alegb_pipe_config_layer(dim=%d, N=%d)" % (dim, N))
    return dict(zip(PIPE_CONFIG_FIELDS, (int(v) for v in out)))


def context_from_config(cfg, cuda_device=0):
    """Create a context and apply mesh / params / motion from a workload dict (workloads/configs.py)."""
    ctx = Context(cfg["dim"], cfg["N"], cuda_device)
    ctx.alegb_mesh_upload(cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"), cfg.get("pml_sigma"))
    ctx.alegb_set_params(cfg["RT"], cfg["tau"], cfg.get("q_inf"))
    ctx.alegb_set_motion(cfg["motion_kind"], cfg.get("motion_params"))
    return ctx
