"""Thin Python binding of the C ABI in include/gh.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libgh.so.  PyTorch is used for device memory
(the workspace and I/O tensors) and the CUDA stream, nothing else.  There is no CPU fallback: if
libgh.so is missing the import of the library fails loudly (``GHError``), and without a CUDA
device ``gh_domain_create`` returns GH_ERR_CUDA.

The module-level functions carry the names of the C entry points; ``Domain`` is a convenience
wrapper that owns the workspace tensor and the handle.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgh.so")

GH_NCOMP = 50
GH_SHELL, GH_BLOCK, GH_CYLINDER = range(3)
GH_NUM_KERNELS = 13
GH_T_A, GH_T_AA, GH_T_AB, GH_T_ABB = range(4)
GH_FILTER_NONE, GH_FILTER_HEAVISIDE, GH_FILTER_EXP = range(3)
GH_OPT_RK_OUT_OF_PLACE, GH_OPT_NO_GRAPH = 0, 1
GH_OK, GH_ERR_ARG, GH_ERR_WORKSPACE, GH_ERR_CUDA, GH_ERR_STATE, GH_ERR_SINGULAR = range(6)
STATUS_NAMES = ["GH_OK", "GH_ERR_ARG", "GH_ERR_WORKSPACE", "GH_ERR_CUDA", "GH_ERR_STATE", "GH_ERR_SINGULAR"]

# every symbol include/gh.h declares (checked by tests/test_abi.py)
EXPORTS = [
    "gh_workspace_bytes", "gh_domain_create", "gh_domain_destroy", "gh_domain_layout", "gh_domain_coords",
    "gh_set_fields", "gh_get_fields", "gh_set_gauge_source", "gh_rhs", "gh_gradient", "gh_rk_step",
    "gh_constraint_norms", "gh_set_profiling", "gh_profile_read", "gh_profile_reset", "gh_kernel_name",
    "gh_launch_count", "gh_last_error", "gh_basis_cheb", "gh_basis_gauss_legendre", "gh_basis_shell",
    "gh_set_filter", "gh_apply_filter", "gh_filter_sigma",
    "gh_dp5_workspace_bytes", "gh_dp5_attach", "gh_dp5_step", "gh_set_option",
    "gh_rk_step_norms", "gh_set_frame_map", "gh_set_jacobian", "gh_spatial_coord_jac", "gh_spatial_coord_jac_state", "gh_fp64_peak",
    "gh_constraint_norms_static",
]


class GHError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {message}")
        self.status = status


class gh_filter_desc(C.Structure):
    _fields_ = [("kind", C.c_int32), ("cut", C.c_int32), ("alpha", C.c_double), ("p", C.c_int32), ("pad_", C.c_int32)]


def make_filter(f):
    """None | {'kind': 'heaviside', 'cut': n} | {'kind': 'exp', 'alpha': a, 'p': p} -> gh_filter_desc or None."""
    if f is None:
        return None
    d = gh_filter_desc()
    kind = f.get("kind", "none")
    d.kind = {"none": GH_FILTER_NONE, "heaviside": GH_FILTER_HEAVISIDE, "exp": GH_FILTER_EXP}[kind]
    d.cut = int(f.get("cut", 0))
    d.alpha = float(f.get("alpha", 0.0))
    d.p = int(f.get("p", 1))
    return d


class gh_subdomain_desc(C.Structure):
    _fields_ = [
        ("kind", C.c_int32),
        ("n", C.c_int32 * 3),
        ("lo", C.c_double * 3),
        ("hi", C.c_double * 3),
        ("center", C.c_double * 3),
        ("face", C.c_int32 * 6),
        ("gamma", C.c_double * 3),
    ]


_lib = None


def lib() -> C.CDLL:
    """Load libgh.so (built in-tree by paper_1804_09101_b200.build).  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise GHError(GH_ERR_STATE, f"{LIB_PATH} is missing: run `python -m paper_1804_09101_b200.build` "
                                    "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_int
    descp = C.POINTER(gh_subdomain_desc)
    L.gh_workspace_bytes.restype = C.c_size_t
    L.gh_workspace_bytes.argtypes = [descp, C.c_int32]
    L.gh_domain_create.argtypes = [descp, C.c_int32, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.gh_domain_destroy.restype = None
    L.gh_domain_destroy.argtypes = [vp]
    L.gh_domain_layout.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.gh_domain_coords.argtypes = [vp, dp, ip]
    L.gh_set_fields.argtypes = [vp, dp, ip, C.c_double]
    L.gh_get_fields.argtypes = [vp, dp, ip, C.POINTER(C.c_double)]
    L.gh_set_gauge_source.argtypes = [vp, dp, dp, ip]
    L.gh_rhs.argtypes = [vp, dp, ip]
    L.gh_gradient.argtypes = [vp, dp, ip]
    L.gh_rk_step.argtypes = [vp, C.c_double]
    L.gh_constraint_norms.argtypes = [vp, dp, dp]
    L.gh_constraint_norms_static.argtypes = [vp, dp, dp]
    L.gh_rk_step_norms.argtypes = [vp, C.c_double, dp, dp]
    L.gh_set_profiling.argtypes = [vp, ip]
    L.gh_profile_read.argtypes = [vp, dp, dp]
    L.gh_profile_reset.argtypes = [vp]
    L.gh_kernel_name.restype = C.c_char_p
    L.gh_kernel_name.argtypes = [ip]
    L.gh_launch_count.restype = C.c_int64
    L.gh_launch_count.argtypes = [vp]
    L.gh_last_error.restype = C.c_char_p
    L.gh_last_error.argtypes = [vp]
    L.gh_basis_cheb.argtypes = [C.c_int32, dp, dp]
    L.gh_basis_gauss_legendre.argtypes = [C.c_int32, dp, dp]
    L.gh_basis_shell.argtypes = [C.c_int32, dp, dp, dp, dp]
    fp = C.POINTER(gh_filter_desc)
    L.gh_set_filter.argtypes = [vp, fp, fp]
    L.gh_apply_filter.argtypes = [vp]
    L.gh_filter_sigma.argtypes = [fp, C.c_int32, dp]
    L.gh_dp5_workspace_bytes.restype = C.c_size_t
    L.gh_dp5_workspace_bytes.argtypes = [vp]
    L.gh_dp5_attach.argtypes = [vp, vp, C.c_size_t]
    L.gh_dp5_step.argtypes = [vp, C.c_double, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    L.gh_set_option.argtypes = [vp, ip, ip]
    L.gh_set_frame_map.argtypes = [vp, dp, dp, ip]
    L.gh_set_jacobian.argtypes = [vp, dp, ip]
    L.gh_spatial_coord_jac.argtypes = [vp, ip, dp, dp, ip]
    L.gh_spatial_coord_jac_state.argtypes = [vp]
    L.gh_fp64_peak.argtypes = [vp, dp]
    _lib = L
    return L


def make_descs(descs):
    """list of descriptor dicts (configs.py) -> ctypes array of gh_subdomain_desc."""
    arr = (gh_subdomain_desc * len(descs))()
    for s, d in enumerate(descs):
        e = arr[s]
        e.kind = {"shell": GH_SHELL, "block": GH_BLOCK, "cylinder": GH_CYLINDER}[d["kind"]]
        n = list(d["n"]) + [0] * (3 - len(d["n"]))
        lo = list(d["lo"]) + [0.0] * (3 - len(d["lo"]))
        hi = list(d["hi"]) + [0.0] * (3 - len(d["hi"]))
        ce = list(d.get("center", [0.0, 0.0, 0.0]))
        fa = list(d.get("face", [])) + [0] * (6 - len(d.get("face", [])))
        ga = list(d.get("gamma", [1.0, -1.0, 1.0]))
        for i in range(3):
            e.n[i], e.lo[i], e.hi[i], e.center[i], e.gamma[i] = int(n[i]), float(lo[i]), float(hi[i]), float(ce[i]), float(ga[i])
        for i in range(6):
            e.face[i] = int(fa[i])
    return arr


def _ptr(a):
    """Raw address + on_device flag of a numpy array (HOST) or a torch CUDA tensor (DEVICE)."""
    if a is None:
        return None, 0
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"]:
            raise ValueError("host buffers must be C-contiguous float64")
        return a.ctypes.data, 0
    import torch

    if isinstance(a, torch.Tensor):
        if a.dtype != torch.float64 or not a.is_contiguous():
            raise ValueError("tensors must be contiguous float64")
        return a.data_ptr(), (1 if a.is_cuda else 0)
    raise TypeError(type(a))


def _check(status: int, handle=None):
    if status != GH_OK:
        msg = lib().gh_last_error(handle)
        raise GHError(status, msg.decode() if msg else "")


# ---- same-name wrappers of the C entry points ---------------------------------------------------
def gh_workspace_bytes(descs) -> int:
    arr = make_descs(descs)
    n = lib().gh_workspace_bytes(arr, len(descs))
    if n == 0:
        _check(GH_ERR_ARG, None)
    return int(n)


def gh_domain_create(descs, workspace_ptr: int, nbytes: int, stream: int):
    arr = make_descs(descs)
    h = C.c_void_p()
    _check(lib().gh_domain_create(arr, len(descs), workspace_ptr, nbytes, stream, C.byref(h)), None)
    return h


def gh_domain_destroy(h):
    lib().gh_domain_destroy(h)


def gh_domain_layout(h, n_sub: int):
    P, S = C.c_int64(), C.c_int64()
    off = (C.c_int64 * (n_sub + 1))()
    _check(lib().gh_domain_layout(h, C.byref(P), C.byref(S), off), h)
    return int(P.value), int(S.value), [int(v) for v in off]


def gh_domain_coords(h, xyz):
    p, dev = _ptr(xyz)
    _check(lib().gh_domain_coords(h, p, dev), h)


def gh_set_fields(h, u, t: float = 0.0):
    p, dev = _ptr(u)
    _check(lib().gh_set_fields(h, p, dev, float(t)), h)


def gh_get_fields(h, u) -> float:
    p, dev = _ptr(u)
    t = C.c_double()
    _check(lib().gh_get_fields(h, p, dev, C.byref(t)), h)
    return float(t.value)


def gh_set_gauge_source(h, H, dH=None):
    p, dev = _ptr(H)
    q, dev2 = _ptr(dH)
    if dH is not None and dev != dev2:
        raise ValueError("H and dH must live on the same side")
    _check(lib().gh_set_gauge_source(h, p, q, dev), h)


def gh_rhs(h, dtu):
    p, dev = _ptr(dtu)
    _check(lib().gh_rhs(h, p, dev), h)


def gh_gradient(h, du):
    p, dev = _ptr(du)
    _check(lib().gh_gradient(h, p, dev), h)


def gh_rk_step(h, dt: float):
    _check(lib().gh_rk_step(h, float(dt)), h)


def gh_constraint_norms(h, n_sub: int, per_sub: bool = False):
    out = np.zeros((3, 2))
    ps = np.zeros((n_sub, 3, 2)) if per_sub else None
    _check(lib().gh_constraint_norms(h, out.ctypes.data, ps.ctypes.data if per_sub else None), h)
    return (out, ps) if per_sub else out


def gh_constraint_norms_static(h, n_sub: int, per_sub: bool = False):
    """gh_constraint_norms with its reduction scratch in the library's static device array: no allocation on the call path."""
    out = np.zeros((3, 2))
    ps = np.zeros((n_sub, 3, 2)) if per_sub else None
    _check(lib().gh_constraint_norms_static(h, out.ctypes.data, ps.ctypes.data if per_sub else None), h)
    return (out, ps) if per_sub else out


def gh_rk_step_norms(h, dt: float, n_sub: int, per_sub: bool = False):
    out = np.zeros((3, 2))
    ps = np.zeros((n_sub, 3, 2)) if per_sub else None
    _check(lib().gh_rk_step_norms(h, float(dt), out.ctypes.data, ps.ctypes.data if per_sub else None), h)
    return (out, ps) if per_sub else out


def gh_set_filter(h, block_axes=None, shell_angular=None):
    fb, fs = make_filter(block_axes), make_filter(shell_angular)
    _check(lib().gh_set_filter(h, C.byref(fb) if fb is not None else None, C.byref(fs) if fs is not None else None), h)


def gh_apply_filter(h):
    _check(lib().gh_apply_filter(h), h)


def gh_filter_sigma(f, kmax: int) -> np.ndarray:
    d = make_filter(f)
    out = np.empty(kmax + 1)
    st = lib().gh_filter_sigma(C.byref(d), int(kmax), out.ctypes.data)
    if st != GH_OK:
        raise GHError(st, "gh_filter_sigma: bad descriptor")
    return out


def gh_dp5_workspace_bytes(h) -> int:
    return int(lib().gh_dp5_workspace_bytes(h))


def gh_dp5_attach(h, workspace_ptr: int, nbytes: int):
    _check(lib().gh_dp5_attach(h, C.c_void_p(workspace_ptr), nbytes), h)


def gh_dp5_step(h, dt: float, tol: float = 0.0):
    """-> (err_rms, err_max, accepted)"""
    err = (C.c_double * 2)()
    acc = C.c_int(0)
    _check(lib().gh_dp5_step(h, float(dt), float(tol), err, C.byref(acc)), h)
    return float(err[0]), float(err[1]), bool(acc.value)


def gh_set_frame_map(h, Jm=None, v=None):
    p, dev = _ptr(Jm)
    q, dev2 = _ptr(v)
    if Jm is not None and v is not None and dev != dev2:
        raise ValueError("Jm and v must live on the same side")
    _check(lib().gh_set_frame_map(h, p, q, dev), h)


def gh_set_jacobian(h, J):
    p, dev = _ptr(J)
    _check(lib().gh_set_jacobian(h, p, dev), h)


def gh_spatial_coord_jac(h, structure: int, T, out):
    p, dev = _ptr(T)
    q, dev2 = _ptr(out)
    if dev != dev2:
        raise ValueError("T and out must live on the same side")
    _check(lib().gh_spatial_coord_jac(h, int(structure), p, q, dev), h)


def gh_spatial_coord_jac_state(h):
    _check(lib().gh_spatial_coord_jac_state(h), h)


def gh_fp64_peak(h):
    """-> (DMMA TFLOP/s, DFMA TFLOP/s) measured now on the domain's device"""
    out = np.zeros(2)
    _check(lib().gh_fp64_peak(h, out.ctypes.data), h)
    return float(out[0]), float(out[1])


def gh_basis_cheb(N: int):
    x, D = np.zeros(N), np.zeros((N, N))
    _check(lib().gh_basis_cheb(N, x.ctypes.data, D.ctypes.data), None)
    return x, D


def gh_basis_gauss_legendre(L: int):
    th, w = np.zeros(L + 1), np.zeros(L + 1)
    _check(lib().gh_basis_gauss_legendre(L, th.ctypes.data, w.ctypes.data), None)
    return th, w


def gh_basis_shell(L: int):
    nt, npp, nq = L + 1, 2 * L + 2, 2 * L + 1
    Fa, Fs = np.zeros((nq, npp)), np.zeros((npp, nq))
    Th, Pr = np.zeros((L + 1, nt, nt)), np.zeros((L + 1, nt, nt))
    _check(lib().gh_basis_shell(L, Fa.ctypes.data, Fs.ctypes.data, Th.ctypes.data, Pr.ctypes.data), None)
    return Fa, Fs, Th, Pr


# ---- convenience wrapper -------------------------------------------------------------------------
def _ordered(fn):
    """Stream plumbing of a Domain method: the library works on the domain's own stream, torch on its current one; make each see
    what the other enqueued before (two event waits, no host synchronisation)."""
    import functools

    @functools.wraps(fn)
    def wrapper(self, *a, **kw):
        cur = self.torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)
        try:
            return fn(self, *a, **kw)
        finally:
            if cur != self.stream:
                cur.wait_stream(self.stream)
    return wrapper


class Domain:
    """Owns the device workspace (a torch uint8 tensor), the CUDA stream the library works on and the gh_domain handle.

    stream: a torch.cuda.Stream, or None for a stream of the domain's own (not torch's default stream: the legacy default stream
    cannot be captured into a CUDA graph, and the library replays each step as one graph launch)."""

    def __init__(self, descs, device: str = "cuda:0", stream=None):
        import torch

        self.torch = torch
        self.descs = list(descs)
        self.n_sub = len(self.descs)
        self.device = torch.device(device)
        nbytes = gh_workspace_bytes(self.descs)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            self.stream.wait_stream(torch.cuda.current_stream(self.device))
            self.h = gh_domain_create(self.descs, aligned, nbytes, self.stream.cuda_stream)
        self.P, self.S, self.offsets = gh_domain_layout(self.h, self.n_sub)
        self.sizes = [self._npts(d) for d in self.descs]

    @staticmethod
    def _npts(d):
        if d["kind"] == "shell":
            return d["n"][0] * (d["n"][1] + 1) * (2 * d["n"][1] + 2)
        return d["n"][0] * d["n"][1] * d["n"][2]

    def close(self):
        if getattr(self, "h", None) is not None:
            self.stream.synchronize()
            gh_domain_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # layout helpers (host, numpy): per-subdomain lists <-> the padded [C][S] store
    def pack(self, parts) -> np.ndarray:
        ncomp = parts[0].shape[0]
        out = np.zeros((ncomp, self.S))
        for s, a in enumerate(parts):
            out[:, self.offsets[s]:self.offsets[s] + self.sizes[s]] = a
        return out

    def unpack(self, arr):
        arr = np.asarray(arr)
        return [np.ascontiguousarray(arr[..., self.offsets[s]:self.offsets[s] + self.sizes[s]]) for s in range(self.n_sub)]

    def coords(self):
        xyz = np.zeros((3, self.S))
        gh_domain_coords(self.h, xyz)
        return self.unpack(xyz)

    def empty(self, *lead):
        return self.torch.empty(*lead, self.S, dtype=self.torch.float64, device=self.device)

    @_ordered
    def set_fields(self, u, t: float = 0.0):
        gh_set_fields(self.h, u, t)

    @_ordered
    def get_fields(self, out=None):
        out = np.zeros((GH_NCOMP, self.S)) if out is None else out
        gh_get_fields(self.h, out)
        return out

    @_ordered
    def set_gauge_source(self, H, dH=None):
        gh_set_gauge_source(self.h, H, dH)

    @_ordered
    def rhs(self, out=None):
        out = np.zeros((GH_NCOMP, self.S)) if out is None else out
        gh_rhs(self.h, out)
        return out

    @_ordered
    def gradient(self, out=None):
        out = np.zeros((3, GH_NCOMP, self.S)) if out is None else out
        gh_gradient(self.h, out)
        return out

    @_ordered
    def rk_step(self, dt: float):
        gh_rk_step(self.h, dt)

    @_ordered
    def rk_step_norms(self, dt: float, per_sub: bool = False):
        return gh_rk_step_norms(self.h, dt, self.n_sub, per_sub)

    @_ordered
    def constraint_norms(self, per_sub: bool = False):
        return gh_constraint_norms(self.h, self.n_sub, per_sub)

    @_ordered
    def constraint_norms_static(self, per_sub: bool = False):
        return gh_constraint_norms_static(self.h, self.n_sub, per_sub)

    @_ordered
    def dp5_attach(self):
        """Allocate (torch) and attach the workspace of the Dormand-Prince stepper."""
        import torch

        n = gh_dp5_workspace_bytes(self.h)
        self._dp_ws = torch.empty(n + 256, dtype=torch.uint8, device=self.device)
        gh_dp5_attach(self.h, (self._dp_ws.data_ptr() + 255) // 256 * 256, n)

    @_ordered
    def dp5_step(self, dt: float, tol: float = 0.0):
        return gh_dp5_step(self.h, dt, tol)

    @_ordered
    def set_filter(self, block_axes=None, shell_angular=None):
        gh_set_filter(self.h, block_axes, shell_angular)

    @_ordered
    def apply_filter(self):
        gh_apply_filter(self.h)

    @_ordered
    def set_frame_map(self, Jm=None, v=None):
        gh_set_frame_map(self.h, Jm, v)

    @_ordered
    def set_jacobian(self, J):
        gh_set_jacobian(self.h, J)

    @_ordered
    def spatial_coord_jac(self, structure: int, T, out=None):
        out = (np.empty_like(T) if isinstance(T, np.ndarray) else self.torch.empty_like(T)) if out is None else out
        gh_spatial_coord_jac(self.h, structure, T, out)
        return out

    @_ordered
    def spatial_coord_jac_state(self):
        gh_spatial_coord_jac_state(self.h)

    @_ordered
    def fp64_peak(self):
        return gh_fp64_peak(self.h)

    def set_option(self, option: int, value: int):
        _check(lib().gh_set_option(self.h, int(option), int(value)), self.h)

    def set_profiling(self, on: bool):
        _check(lib().gh_set_profiling(self.h, int(on)), self.h)

    def profile_reset(self):
        _check(lib().gh_profile_reset(self.h), self.h)

    def profile_read(self):
        ms = np.zeros(GH_NUM_KERNELS)
        cnt = np.zeros(GH_NUM_KERNELS, dtype=np.int64)
        _check(lib().gh_profile_read(self.h, ms.ctypes.data, cnt.ctypes.data), self.h)
        names = [lib().gh_kernel_name(k).decode() for k in range(GH_NUM_KERNELS)]
        return {names[k]: (float(ms[k]), int(cnt[k])) for k in range(GH_NUM_KERNELS)}

    def launch_count(self) -> int:
        return int(lib().gh_launch_count(self.h))
