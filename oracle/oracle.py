"""ctypes wrapper around oracle/trimeg_oracle.c (plain C, gcc) -- TEST INFRASTRUCTURE.

Argument marshalling only; all arithmetic is in the C file, whose header lists the
passages of /root/reference/PAPER.md each step follows.  Builds the shared object
next to the source on first use (gcc -O2 -fopenmp -ffp-contract=off).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "trimeg_oracle.c")
_LIB = os.path.join(_HERE, "libtrimeg_oracle.so")
_lock = threading.Lock()
_lib = None

_d = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")


def build_oracle(force: bool = False) -> str:
    """Compile the C oracle (idempotent). Returns the path of the shared object."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
                   "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build_oracle())
        lib.orc_create.restype = C.c_void_p
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_num_threads.restype = C.c_int
        lib.orc_set_num_threads.argtypes = [C.c_int]
        lib.orc_equilibrium_set.argtypes = [C.c_void_p] + [C.c_double] * 6 + [C.c_int]
        lib.orc_equilibrium_set_numeric.argtypes = [C.c_void_p, C.c_int, C.c_int] + [C.c_double] * 7 + [_d]
        lib.orc_species_set.argtypes = [C.c_void_p] + [C.c_double] * 6 + [C.c_int, C.c_int]
        lib.orc_mesh_load.argtypes = [C.c_void_p, C.c_int64, _d, C.c_int64, _i, C.c_int32, C.c_double]
        lib.orc_fields_set.argtypes = [C.c_void_p, C.c_int, _d]
        lib.orc_element_coeffs.argtypes = [C.c_void_p, C.c_int64, _d, _d]
        lib.orc_poly_eval.argtypes = [C.c_void_p, C.c_int64, _d, C.c_double, C.c_double, _d]
        lib.orc_locate.argtypes = [C.c_void_p, C.c_int64, _d, _d, _i, C.c_int]
        lib.orc_bspline.argtypes = [C.c_void_p, C.c_double, C.POINTER(C.c_int), _d, _d]
        lib.orc_gather.argtypes = [C.c_void_p, C.c_int64, _d, _d, _d, _d, _i, C.c_int]
        lib.orc_equil_eval.argtypes = [C.c_void_p, C.c_double, C.c_double, _d]
        lib.orc_ln_f0.argtypes = [C.c_void_p] + [C.c_double] * 4
        lib.orc_ln_f0.restype = C.c_double
        lib.orc_grad_ln_f0.argtypes = [C.c_void_p] + [C.c_double] * 4 + [_d]
        lib.orc_rhs.argtypes = [C.c_void_p, C.c_int64] + [_d] * 7 + [_d, _i]
        lib.orc_pullback.argtypes = [C.c_void_p, C.c_int64] + [_d] * 7 + [_i]
        lib.orc_density_g2p.argtypes = [C.c_void_p, C.c_int, C.c_int64, _d, _d, _d, _d]
        lib.orc_f_interp.argtypes = [C.c_void_p, C.c_int64] + [_d] * 6
        lib.orc_gather_gyro.argtypes = [C.c_void_p, C.c_int64, _d, _d, _d, _d, C.c_int, _d, _i]
        lib.orc_deposit.argtypes = [C.c_void_p, C.c_int64, _d, _d, _d, _d, _d]
        lib.orc_push_rk4.argtypes = [C.c_void_p, C.c_int64] + [_d] * 7 + [_i, C.c_double, C.c_int32]
        _lib = lib
    return _lib


def oracle_threads(n: int | None = None) -> int:
    """Get (and optionally set) the OpenMP thread count the oracle uses."""
    lib = _load()
    if n is not None:
        lib.orc_set_num_threads(int(n))
    return int(lib.orc_num_threads())


def _f(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """One oracle context (mesh + equilibrium + species + fields)."""

    EQ_FIELDS = ("r", "q", "qbar", "psi1", "psi2", "B_R", "B_phi", "B_Z", "B", "b_R", "b_phi", "b_Z",
                 "gradB_R", "gradB_phi", "gradB_Z", "curlb_R", "curlb_phi", "curlb_Z", "F")

    def __init__(self):
        self._lib = _load()
        self._h = C.c_void_p(self._lib.orc_create())
        self.n_tri = 0
        self.n_planes = 0

    def __del__(self):
        try:
            self._lib.orc_destroy(self._h)
        except Exception:
            pass

    def _ck(self, rc, what):
        if rc != 0:
            raise RuntimeError(f"oracle {what} failed rc={rc}")

    def equilibrium_set(self, R0, a, B0, q0, q1, q2, qbar_sqrt=1):
        self._ck(self._lib.orc_equilibrium_set(self._h, R0, a, B0, q0, q1, q2, int(qbar_sqrt)), "equilibrium_set")

    def equilibrium_set_numeric(self, nR, nZ, Rmin, Rmax, Zmin, Zmax, F, R0, a, coef):
        """psi as tensor-product cubic B-spline coefficients coef[nR+3][nZ+3]; F = R B_phi; R0, a for the Eq.(8) profiles."""
        coef = _f(coef)
        assert coef.shape == (nR + 3, nZ + 3), coef.shape
        self._ck(self._lib.orc_equilibrium_set_numeric(self._h, int(nR), int(nZ), Rmin, Rmax, Zmin, Zmax, F, R0, a, coef), "equilibrium_set_numeric")

    def species_set(self, qom, kappa_n=0.0, kappa_T=0.0, w_n=0.3, w_T=0.3, r0=0.0, bstar_exact=1, weight_mode=0):
        self._ck(self._lib.orc_species_set(self._h, qom, kappa_n, kappa_T, w_n, w_T, r0, int(bstar_exact),
                                           int(weight_mode)), "species_set")

    def mesh_load(self, RZ, tri, n_planes, phi_period=2 * np.pi):
        RZ = _f(RZ)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        rc = self._lib.orc_mesh_load(self._h, RZ.shape[0], RZ, tri.shape[0], tri, int(n_planes), float(phi_period))
        self._ck(rc, "mesh_load")
        self.n_tri, self.n_planes, self.n_nodes = tri.shape[0], int(n_planes), RZ.shape[0]

    def fields_set(self, which, dof):
        dof = _f(dof)
        assert dof.shape == (self.n_planes, self.n_nodes, 6), dof.shape
        self._ck(self._lib.orc_fields_set(self._h, int(which), dof), "fields_set")

    def element_coeffs(self, t, dof18):
        out = np.zeros(21)
        self._ck(self._lib.orc_element_coeffs(self._h, int(t), _f(dof18), out), "element_coeffs")
        return out

    def poly_eval(self, t, coef21, R, Z):
        out = np.zeros(6)
        self._ck(self._lib.orc_poly_eval(self._h, int(t), _f(coef21), float(R), float(Z), out), "poly_eval")
        return out

    def locate(self, R, Z, brute=False):
        R, Z = _f(R), _f(Z)
        out = np.zeros(R.shape[0], dtype=np.int32)
        self._ck(self._lib.orc_locate(self._h, R.shape[0], R, Z, out, int(brute)), "locate")
        return out

    def bspline(self, phi):
        k = C.c_int(0)
        w, dw = np.zeros(4), np.zeros(4)
        self._ck(self._lib.orc_bspline(self._h, float(phi), C.byref(k), w, dw), "bspline")
        return k.value, w, dw

    def gather(self, R, Z, phi, brute=False):
        """-> (out[8][n], tri[n]); rows: Phi, dR, dZ, dphi, Apar, dR, dZ, dphi (dphi = raw d/dphi)."""
        R, Z, phi = _f(R), _f(Z), _f(phi)
        n = R.shape[0]
        out = np.zeros((8, n))
        tri = np.zeros(n, dtype=np.int32)
        self._ck(self._lib.orc_gather(self._h, n, R, Z, phi, out, tri, int(brute)), "gather")
        return out, tri

    def equil(self, R, Z):
        out = np.zeros(19)
        self._ck(self._lib.orc_equil_eval(self._h, float(R), float(Z), out), "equil_eval")
        return dict(zip(self.EQ_FIELDS, out))

    def ln_f0(self, R, Z, u, mu):
        return float(self._lib.orc_ln_f0(self._h, R, Z, u, mu))

    def grad_ln_f0(self, R, Z, u, mu):
        out = np.zeros(3)
        self._lib.orc_grad_ln_f0(self._h, R, Z, u, mu, out)
        return out

    def rhs(self, R, Z, phi, u, w, mu, p):
        """-> (d[5][n] = dR, dZ, dphi, du, dw ; outside[n])."""
        a = [_f(x) for x in (R, Z, phi, u, w, mu, p)]
        n = a[0].shape[0]
        out = np.zeros((5, n))
        outside = np.zeros(n, dtype=np.int32)
        self._ck(self._lib.orc_rhs(self._h, n, *a, out, outside), "rhs")
        return out, outside

    def pullback(self, R, Z, phi, u, w, mu, p):
        """-> new (u, w, status); the other inputs are unchanged by the map."""
        R, Z, phi, mu, p = [_f(x) for x in (R, Z, phi, mu, p)]
        u, w = _f(u).copy(), _f(w).copy()
        st = np.zeros(R.shape[0], dtype=np.int32)
        self._ck(self._lib.orc_pullback(self._h, R.shape[0], R, Z, phi, u, w, mu, p, st), "pullback")
        return u, w, st

    def density_g2p(self, which, R, Z, phi):
        R, Z, phi = _f(R), _f(Z), _f(phi)
        out = np.zeros(R.shape[0])
        self._ck(self._lib.orc_density_g2p(self._h, int(which), R.shape[0], R, Z, phi, out), "density_g2p")
        return out

    def f_interp(self, R, Z, phi, u, mu):
        R, Z, phi, u, mu = [_f(x) for x in (R, Z, phi, u, mu)]
        out = np.zeros(R.shape[0])
        self._ck(self._lib.orc_f_interp(self._h, R.shape[0], R, Z, phi, u, mu, out), "f_interp")
        return out

    def gather_gyro(self, R, Z, phi, rho, npts):
        """N-point gyro-average of the gather -> (out[8][n], tri[n] of the gyrocentres)."""
        R, Z, phi, rho = [_f(x) for x in (R, Z, phi, rho)]
        n = R.shape[0]
        out = np.zeros((8, n))
        tri = np.zeros(n, dtype=np.int32)
        self._ck(self._lib.orc_gather_gyro(self._h, n, R, Z, phi, rho, int(npts), out, tri), "gather_gyro")
        return out, tri

    def deposit(self, R, Z, phi, q):
        """P2G: -> b[n_planes][n_nodes][6], the transpose of the gather applied to the marker charges q."""
        R, Z, phi, q = [_f(x) for x in (R, Z, phi, q)]
        out = np.zeros((self.n_planes, self.n_nodes, 6))
        self._ck(self._lib.orc_deposit(self._h, R.shape[0], R, Z, phi, q, out), "deposit")
        return out

    def push_rk4(self, R, Z, phi, u, w, mu, p, dt, nsteps, status=None):
        """Returns new (R, Z, phi, u, w, status); inputs are not modified."""
        R, Z, phi, u, w = [_f(x).copy() for x in (R, Z, phi, u, w)]
        mu, p = _f(mu), _f(p)
        n = R.shape[0]
        st = np.zeros(n, dtype=np.int32) if status is None else np.ascontiguousarray(status, dtype=np.int32).copy()
        self._ck(self._lib.orc_push_rk4(self._h, n, R, Z, phi, u, w, mu, p, st, float(dt), int(nsteps)), "push_rk4")
        return R, Z, phi, u, w, st
