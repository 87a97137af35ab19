"""ctypes front end of the CPU oracle (oracle/gh_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this.  It imports nothing from paper_1804_09101_b200.

Two builds of the same C source: ``real = long double`` (parity; default) and
``real = double`` (``precision="double"``, the timed CPU baseline).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gh_oracle.c")
_LOCK = threading.Lock()


def build(force: bool = False) -> dict:
    """Compile liboracle_ld.so (long double) and liboracle_d.so (double) with gcc."""
    out = {}
    for tag, flags in (("ld", []), ("d", ["-DORA_DOUBLE"])):
        so = os.path.join(_HERE, f"liboracle_{tag}.so")
        if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
            tmp = so + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", *flags, _SRC, "-o", tmp, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, so)
        out[tag] = so
    return out


class Subdomain(C.Structure):
    _fields_ = [
        ("kind", C.c_int32),
        ("n", C.c_int32 * 3),
        ("lo", C.c_double * 3),
        ("hi", C.c_double * 3),
        ("center", C.c_double * 3),
        ("face", C.c_int32 * 6),
        ("gamma", C.c_double * 3),
    ]


def make_subdomain(d: dict) -> Subdomain:
    """d: {'kind': 'shell'|'block'|'cylinder', 'n': [..], 'lo': [..], 'hi': [..], 'center': [..], 'face': [..], 'gamma': [..]}"""
    s = Subdomain()
    s.kind = {"shell": 0, "block": 1, "cylinder": 2}[d["kind"]]
    n = list(d["n"]) + [0] * (3 - len(d["n"]))
    lo = list(d["lo"]) + [0.0] * (3 - len(d["lo"]))
    hi = list(d["hi"]) + [0.0] * (3 - len(d["hi"]))
    face = list(d.get("face", [])) + [0] * (6 - len(d.get("face", [])))
    for i in range(3):
        s.n[i] = int(n[i])
        s.lo[i] = float(lo[i])
        s.hi[i] = float(hi[i])
        s.center[i] = float(d.get("center", [0, 0, 0])[i])
        s.gamma[i] = float(d.get("gamma", [1.0, -1.0, 1.0])[i])
    for i in range(6):
        s.face[i] = int(face[i])
    return s


_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")


class Oracle:
    def __init__(self, precision: str = "long double", threads: int | None = None):
        with _LOCK:
            libs = build()
        self.precision = precision
        self.lib = C.CDLL(libs["ld" if precision == "long double" else "d"])
        L = self.lib
        L.ora_real_bytes.restype = C.c_int
        L.ora_num_points.restype = C.c_int64
        L.ora_num_points.argtypes = [C.POINTER(Subdomain)]
        L.ora_cheb_nodes.argtypes = [C.c_int, _dp]
        L.ora_gl_nodes.argtypes = [C.c_int, _dp, _dp]
        L.ora_coords.argtypes = [C.POINTER(Subdomain), _dp]
        L.ora_cheb_derivative_line.argtypes = [C.c_int, _dp, _dp]
        L.ora_fourier_derivative_line.argtypes = [C.c_int, _dp, _dp]
        L.ora_pbar.argtypes = [C.c_int, C.c_double, _dp, _dp]
        L.ora_shell_angular.argtypes = [C.c_int, _dp, _dp, _dp]
        L.ora_shell_project.argtypes = [C.c_int, _dp, _dp]
        L.ora_gradient.argtypes = [C.POINTER(Subdomain), C.c_int, _dp, _dp]
        L.ora_geometry_point.argtypes = [_dp, _dp, _dp, _dp, _dp]
        L.ora_geometry_point.restype = C.c_int
        L.ora_rhs_point.argtypes = [_dp] * 12
        L.ora_rhs_point.restype = C.c_int
        L.ora_constraints_point.argtypes = [_dp] * 9
        L.ora_constraints_point.restype = C.c_int
        L.ora_rhs_subdomain.argtypes = [C.POINTER(Subdomain), _dp, _dp, C.c_void_p, _dp]
        L.ora_rhs_subdomain.restype = C.c_int
        L.ora_rhs_subdomain_full.argtypes = [C.POINTER(Subdomain), _dp, _dp, C.c_void_p, _dp]
        L.ora_rhs_subdomain_full.restype = C.c_int
        L.ora_rk3_subdomain.argtypes = [C.POINTER(Subdomain), _dp, _dp, C.c_void_p, C.c_double, C.c_int]
        L.ora_rk3_subdomain.restype = C.c_int
        L.ora_constraints_subdomain.argtypes = [C.POINTER(Subdomain), _dp, _dp, _dp, _dp, C.c_void_p]
        L.ora_constraints_subdomain.restype = C.c_int
        L.ora_rhs_subdomain_ifc.argtypes = [C.POINTER(Subdomain), _dp, _dp, C.c_void_p, C.c_void_p, C.c_void_p, _dp]
        L.ora_rhs_subdomain_ifc.restype = C.c_int
        L.ora_dp5_tableau.argtypes = [_dp] * 4
        L.ora_dp5_tableau.restype = None
        L.ora_dp5_subdomain.argtypes = [C.POINTER(Subdomain), _dp, _dp, C.c_void_p, C.c_double, _dp]
        L.ora_dp5_subdomain.restype = C.c_int
        L.ora_char_bc_point.argtypes = [_dp] * 7
        L.ora_char_bc_point.restype = C.c_int
        L.ora_filter_subdomain.argtypes = [C.POINTER(Subdomain), C.c_int, _dp, _dp, _dp, _dp]
        L.ora_filter_subdomain.restype = C.c_int
        L.ora_rhs_point_map.argtypes = [_dp] * 14
        L.ora_rhs_point_map.restype = C.c_int
        L.ora_rhs_subdomain_map.argtypes = [C.POINTER(Subdomain), _dp, _dp, _dp, _dp, _dp, C.c_double, C.c_int, _dp]
        L.ora_rhs_subdomain_map.restype = C.c_int
        L.ora_shell_interp.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.ora_scj_point.argtypes = [C.c_int, _dp, _dp, _dp]
        L.ora_scj_point.restype = C.c_double
        L.ora_scj_eq12.argtypes = [C.c_int]
        L.ora_scj_eq12.restype = C.c_double
        L.ora_scj_subdomain.argtypes = [C.c_int, C.c_int64, _dp, _dp, _dp]
        L.ora_scj_subdomain.restype = C.c_int
        L.ora_scj_state.argtypes = [C.c_int64, _dp, _dp, _dp]
        L.ora_scj_state.restype = C.c_int
        self.threads = threads
        if threads is not None:
            try:
                omp = C.CDLL("libgomp.so.1")
                omp.omp_set_num_threads(int(threads))
            except OSError:
                pass

    # ---- grids -------------------------------------------------------
    def num_points(self, sd: dict) -> int:
        return int(self.lib.ora_num_points(C.byref(make_subdomain(sd))))

    def cheb_nodes(self, N: int) -> np.ndarray:
        x = np.empty(N)
        self.lib.ora_cheb_nodes(N, x)
        return x

    def gl_nodes(self, L: int):
        th, w = np.empty(L + 1), np.empty(L + 1)
        self.lib.ora_gl_nodes(L, th, w)
        return th, w

    def coords(self, sd: dict) -> np.ndarray:
        s = make_subdomain(sd)
        P = int(self.lib.ora_num_points(C.byref(s)))
        xyz = np.empty((3, P))
        self.lib.ora_coords(C.byref(s), xyz)
        return xyz

    # ---- O1 / O2 / O3 ------------------------------------------------
    def cheb_derivative_line(self, u: np.ndarray) -> np.ndarray:
        u = np.ascontiguousarray(u, dtype=np.float64)
        du = np.empty_like(u)
        self.lib.ora_cheb_derivative_line(u.shape[0], u, du)
        return du

    def fourier_derivative_line(self, u: np.ndarray) -> np.ndarray:
        """O15: d/dphi of one periodic line sampled at phi_k = 2 pi k / N."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        du = np.empty_like(u)
        self.lib.ora_fourier_derivative_line(u.shape[0], u, du)
        return du

    def pbar(self, L: int, theta: float):
        n = L + 1
        pb, dpb = np.empty((n, n)), np.empty((n, n))
        self.lib.ora_pbar(L, float(theta), pb, dpb)
        return pb, dpb

    def shell_angular(self, L: int, u: np.ndarray):
        u = np.ascontiguousarray(u, dtype=np.float64)
        assert u.shape == (L + 1, 2 * L + 2)
        a, b = np.empty_like(u), np.empty_like(u)
        self.lib.ora_shell_angular(L, u, a, b)
        return a, b

    def shell_project(self, L: int, u: np.ndarray) -> np.ndarray:
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.empty_like(u)
        self.lib.ora_shell_project(L, u, out)
        return out

    def shell_interp(self, Ls: int, Ld: int, u: np.ndarray) -> np.ndarray:
        """O12b: planes u[..., Ls+1, 2Ls+2] on the grid of band limit Ls -> the same series summed at the nodes of band limit Ld."""
        u = np.ascontiguousarray(u, dtype=np.float64)
        lead = u.shape[:-2]
        assert u.shape[-2:] == (Ls + 1, 2 * Ls + 2)
        flat = u.reshape(-1, Ls + 1, 2 * Ls + 2)
        out = np.empty((flat.shape[0], Ld + 1, 2 * Ld + 2))
        for i in range(flat.shape[0]):
            self.lib.ora_shell_interp(Ls, Ld, np.ascontiguousarray(flat[i]), out[i])
        return out.reshape(*lead, Ld + 1, 2 * Ld + 2)

    def spectral_filter(self, sd: dict, u: np.ndarray, sigmas) -> np.ndarray:
        """O9: filtered copy of u[ncomp][P].  sigmas: blocks [sigma_x, sigma_y, sigma_z] (one value per Chebyshev mode);
        shells [sigma_l] (l = 0..L; no radial filter)."""
        s = make_subdomain(sd)
        out = np.array(u, dtype=np.float64, order="C", copy=True)
        sg = [np.ascontiguousarray(x, dtype=np.float64) for x in sigmas]
        while len(sg) < 3:
            sg.append(sg[0])
        self.lib.ora_filter_subdomain(C.byref(s), out.shape[0], out, sg[0], sg[1], sg[2])
        return out

    def gradient(self, sd: dict, u: np.ndarray) -> np.ndarray:
        """u[ncomp,P] -> g[3,ncomp,P] (Cartesian d/dx, d/dy, d/dz)."""
        s = make_subdomain(sd)
        u = np.ascontiguousarray(u, dtype=np.float64)
        g = np.empty((3,) + u.shape)
        self.lib.ora_gradient(C.byref(s), u.shape[0], u, g)
        return g

    # ---- O4 / O5 / O8 at a point (full arrays) ------------------------
    def geometry_point(self, psi: np.ndarray):
        ginv, lapse, shift, psiinv = np.empty((3, 3)), np.empty(1), np.empty(3), np.empty((4, 4))
        bad = self.lib.ora_geometry_point(np.ascontiguousarray(psi, dtype=np.float64), ginv, lapse, shift, psiinv)
        if bad:
            raise ValueError("non-physical metric")
        return ginv, float(lapse[0]), shift, psiinv

    def rhs_point(self, psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, gamma):
        c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        o1, o2, o3 = np.empty((4, 4)), np.empty((4, 4)), np.empty((3, 4, 4))
        bad = self.lib.ora_rhs_point(c(psi), c(Pi), c(Phi), c(dpsi), c(dPi), c(dPhi), c(H), c(dH), c(gamma), o1, o2, o3)
        if bad:
            raise ValueError("non-physical metric")
        return o1, o2, o3

    def rhs_point_map(self, psi, Pi, Phi, dpsi, dPi, dPhi, H, dH, gamma, Jm, v):
        """O14 at a point: derivative inputs in the GRID frame, Jm[3,3] = d xbar^k / d x^i, v[3] the grid velocity; dH inertial."""
        c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        o1, o2, o3 = np.empty((4, 4)), np.empty((4, 4)), np.empty((3, 4, 4))
        bad = self.lib.ora_rhs_point_map(c(psi), c(Pi), c(Phi), c(dpsi), c(dPi), c(dPhi), c(H), c(dH), c(gamma), c(Jm), c(v), o1, o2, o3)
        if bad:
            raise ValueError("non-physical metric")
        return o1, o2, o3

    def rhs_map(self, sd: dict, u, H, dH, Jm, v, dt: float = 0.0, nsteps: int = 0) -> np.ndarray:
        """O14 on a subdomain: nsteps = 0 -> the dual-frame RHS; nsteps > 0 -> the state after that many RK3 steps (map frozen)."""
        s = make_subdomain(sd)
        uu = np.array(u, dtype=np.float64, order="C", copy=True)
        out = np.empty_like(uu)
        c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        bad = self.lib.ora_rhs_subdomain_map(C.byref(s), uu, c(H), c(dH), c(Jm), c(v), float(dt), int(nsteps), out)
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return uu if nsteps > 0 else out

    def char_bc_point(self, psi, gamma, s, dtpsi, dtPi, dtPhi):
        """O10 at one point: freeze the incoming characteristic fields.  psi[4,4]; s[3] outward direction;
        dtpsi[4,4], dtPi[4,4], dtPhi[3,4,4] -> (dtpsi', dtPi', dtPhi', speeds[v0, v1+, v1-, v2])."""
        c = lambda a: np.array(a, dtype=np.float64, order="C", copy=True)
        a, b, d3, sp = c(dtpsi), c(dtPi), c(dtPhi), np.empty(4)
        if self.lib.ora_char_bc_point(c(psi), c(gamma), c(s), a, b, d3, sp):
            raise ValueError("non-physical metric")
        return a, b, d3, sp

    def constraints_point(self, psi, Pi, Phi, dpsi, dPhi, H):
        c = lambda a: np.ascontiguousarray(a, dtype=np.float64)
        o1, o2, o3 = np.empty(4), np.empty((3, 4, 4)), np.empty((3, 3, 4, 4))
        bad = self.lib.ora_constraints_point(c(psi), c(Pi), c(Phi), c(dpsi), c(dPhi), c(H), o1, o2, o3)
        if bad:
            raise ValueError("non-physical metric")
        return o1, o2, o3

    # ---- subdomain level (packed 50-component storage) ---------------
    @staticmethod
    def _opt(a):
        if a is None:
            return None, None
        a = np.ascontiguousarray(a, dtype=np.float64)
        return a, a.ctypes.data_as(C.c_void_p)

    def rhs(self, sd: dict, u, H, dH=None) -> np.ndarray:
        s = make_subdomain(sd)
        u = np.ascontiguousarray(u, dtype=np.float64)
        H = np.ascontiguousarray(H, dtype=np.float64)
        keep, ptr = self._opt(dH)
        out = np.empty_like(u)
        bad = self.lib.ora_rhs_subdomain(C.byref(s), u, H, ptr, out)
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return out

    def rhs_full(self, sd: dict, u, H, dH=None) -> np.ndarray:
        s = make_subdomain(sd)
        u = np.ascontiguousarray(u, dtype=np.float64)
        H = np.ascontiguousarray(H, dtype=np.float64)
        keep, ptr = self._opt(dH)
        out = np.zeros((80, u.shape[1]))
        bad = self.lib.ora_rhs_subdomain_full(C.byref(s), u, H, ptr, out)
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return out

    def rk3(self, sd: dict, u, H, dt: float, nsteps: int = 1, dH=None) -> np.ndarray:
        s = make_subdomain(sd)
        u = np.array(u, dtype=np.float64, order="C", copy=True)
        H = np.ascontiguousarray(H, dtype=np.float64)
        keep, ptr = self._opt(dH)
        bad = self.lib.ora_rk3_subdomain(C.byref(s), u, H, ptr, float(dt), int(nsteps))
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return u

    def rhs_ifc(self, sd: dict, u, H, nbr_in=None, nbr_out=None) -> np.ndarray:
        """O12: RHS of one shell whose INTERFACE faces (flag 3) see the neighbour's face state nbr_*[50, n_theta*n_phi]."""
        s = make_subdomain(sd)
        u = np.ascontiguousarray(u, dtype=np.float64)
        H = np.ascontiguousarray(H, dtype=np.float64)
        keep = [None if a is None else np.ascontiguousarray(a, dtype=np.float64) for a in (nbr_in, nbr_out)]
        ptr = [None if a is None else a.ctypes.data for a in keep]
        out = np.empty_like(u)
        bad = self.lib.ora_rhs_subdomain_ifc(C.byref(s), u, H, None, ptr[0], ptr[1], out)
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return out

    def dp5_tableau(self):
        c, a, b, bh = np.empty(7), np.empty((7, 6)), np.empty(7), np.empty(7)
        self.lib.ora_dp5_tableau(c, a, b, bh)
        return c, a, b, bh

    def dp5(self, sd: dict, u, H, dt: float, dH=None):
        """O11: one Dormand-Prince 5(4) step -> (u_new[50,P], err[50,P])."""
        s = make_subdomain(sd)
        out = np.array(u, dtype=np.float64, order="C", copy=True)
        err = np.empty_like(out)
        Hc = np.ascontiguousarray(H, dtype=np.float64)
        dHc = None if dH is None else np.ascontiguousarray(dH, dtype=np.float64)
        bad = self.lib.ora_dp5_subdomain(C.byref(s), out, Hc, None if dHc is None else dHc.ctypes.data, float(dt), err)
        if bad:
            raise ValueError("non-physical metric")
        return out, err

    # ---- O13: SpatialCoordJac (NEXT-4) -----------------------------------
    SCJ = {"a": 0, "aa": 1, "ab": 2, "abb": 3}

    def scj_point(self, structure: str, J, T):
        """One point, FULL arrays (shape (4,), (4,4), (4,4), (4,4,4)); J[3,3] = J_i^k -> (T', flop count of the evaluation)."""
        T = np.ascontiguousarray(T, dtype=np.float64)
        out = np.empty_like(T)
        fl = self.lib.ora_scj_point(self.SCJ[structure], np.ascontiguousarray(J, dtype=np.float64), T, out)
        return out, float(fl)

    def scj_eq12(self, structure: str) -> float:
        return float(self.lib.ora_scj_eq12(self.SCJ[structure]))

    def scj(self, structure: str, J, T) -> np.ndarray:
        """Packed arrays: J[9,P], T[N_e,P] (N_e = 4, 10, 16, 40) -> T'[N_e,P]."""
        J = np.ascontiguousarray(J, dtype=np.float64)
        T = np.ascontiguousarray(T, dtype=np.float64)
        out = np.empty_like(T)
        self.lib.ora_scj_subdomain(self.SCJ[structure], T.shape[1], J, T, out)
        return out

    def scj_state(self, J, u) -> np.ndarray:
        J = np.ascontiguousarray(J, dtype=np.float64)
        u = np.ascontiguousarray(u, dtype=np.float64)
        out = np.empty_like(u)
        if self.lib.ora_scj_state(u.shape[1], J, u, out):
            raise ValueError("SpatialCoordJac mixed a timelike first index into Phi")
        return out

    def constraints(self, sd: dict, u, H, fields: bool = False):
        """-> (sums[3], maxs[3], Cfield[64,P] or None) for one subdomain."""
        s = make_subdomain(sd)
        u = np.ascontiguousarray(u, dtype=np.float64)
        H = np.ascontiguousarray(H, dtype=np.float64)
        sums, maxs = np.empty(3), np.empty(3)
        Cf = np.zeros((64, u.shape[1])) if fields else None
        ptr = Cf.ctypes.data_as(C.c_void_p) if fields else None
        bad = self.lib.ora_constraints_subdomain(C.byref(s), u, H, sums, maxs, ptr)
        if bad:
            raise ValueError(f"{bad} non-physical points")
        return sums, maxs, Cf

    def constraint_norms(self, sds, us, Hs) -> np.ndarray:
        """Domain norms [3][2] = (rms, max) for C_a, C_iab, C_ijab (unweighted)."""
        S = np.zeros(3)
        M = np.zeros(3)
        P = 0
        for sd, u, H in zip(sds, us, Hs):
            s, m, _ = self.constraints(sd, u, H)
            S += s
            M = np.maximum(M, m)
            P += u.shape[1]
        ncomp = np.array([4.0, 30.0, 30.0])
        return np.stack([np.sqrt(S / (P * ncomp)), M], axis=1)
