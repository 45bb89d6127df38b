"""Thin Python binding of include/trimeg.h: argument marshalling only.

Every step of the path runs inside libtrimeg_b200.so (hand-written CUDA, sm_100a).  PyTorch appears here
for two things: device memory (tensors as buffers) and the CUDA stream.  There is no CPU fallback: if the
shared library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtrimeg_b200.so")
HOST, DEVICE = 0, 1
PHI, APAR = 0, 1

EXPORTS = [
    "trimeg_create", "trimeg_destroy", "trimeg_sync", "trimeg_last_error", "trimeg_equilibrium_set",
    "trimeg_species_set", "trimeg_mesh_load", "trimeg_fields_set", "trimeg_gather", "trimeg_scratch_bytes",
    "trimeg_markers_bind", "trimeg_markers_get", "trimeg_sort", "trimeg_set_sort_interval", "trimeg_push_rk4",
    "trimeg_rhs", "trimeg_set_push_variant", "trimeg_push_variant_used", "trimeg_bench_dfma", "trimeg_push_stats", "trimeg_push_kernel_ms",
    "trimeg_fields_bytes", "trimeg_fields_export", "trimeg_fields_import", "trimeg_build_info", "trimeg_set_gather_mode", "trimeg_gather_kernel_ms",
    "trimeg_pullback", "trimeg_density_g2p", "trimeg_f_interp", "trimeg_deposit", "trimeg_gather_gyro", "trimeg_equilibrium_set_numeric", "trimeg_gather_noalloc", "trimeg_bench_dfma_mix",
]


class TrimegError(RuntimeError):
    pass


class _Equil(C.Structure):
    _fields_ = [("R0", C.c_double), ("a", C.c_double), ("B0", C.c_double), ("q0", C.c_double), ("q1", C.c_double),
                ("q2", C.c_double), ("qbar_sqrt", C.c_int32)]


class _EquilGrid(C.Structure):
    _fields_ = [("nR", C.c_int32), ("nZ", C.c_int32), ("Rmin", C.c_double), ("Rmax", C.c_double), ("Zmin", C.c_double),
                ("Zmax", C.c_double), ("F", C.c_double), ("R0", C.c_double), ("a", C.c_double)]


class _Species(C.Structure):
    _fields_ = [("qom", C.c_double), ("kappa_n", C.c_double), ("kappa_T", C.c_double), ("w_n", C.c_double),
                ("w_T", C.c_double), ("r0", C.c_double), ("bstar_exact", C.c_int32), ("weight_mode", C.c_int32)]


_lib = None


def build_library(force: bool = False, verbose: bool = False) -> str:
    from . import build as _b
    return _b.build(force=force, verbose=verbose)


def load_library():
    """dlopen libtrimeg_b200.so (built in-tree by build.py / __graft_entry__.build()).  Raises if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise TrimegError(f"{LIB_PATH} not found: run `python -m paper_2606_24327_b200.build` (nvcc, sm_100a). "
                          "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.trimeg_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    lib.trimeg_destroy.argtypes = [vp]
    lib.trimeg_sync.argtypes = [vp]
    lib.trimeg_last_error.argtypes = [vp]
    lib.trimeg_last_error.restype = C.c_char_p
    lib.trimeg_equilibrium_set.argtypes = [vp, C.POINTER(_Equil)]
    lib.trimeg_equilibrium_set_numeric.argtypes = [vp, C.POINTER(_EquilGrid), vp]
    lib.trimeg_species_set.argtypes = [vp, C.POINTER(_Species)]
    lib.trimeg_mesh_load.argtypes = [vp, i64, vp, i64, vp, i32, dbl]
    lib.trimeg_fields_set.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.trimeg_gather.argtypes = [vp, i64, vp, vp, vp, vp, vp, C.c_int]
    lib.trimeg_gather_noalloc.argtypes = [vp, i64, vp, vp, vp, vp, vp]
    lib.trimeg_set_gather_mode.argtypes = [vp, i32]
    lib.trimeg_gather_kernel_ms.argtypes = [vp, C.POINTER(dbl)]
    lib.trimeg_pullback.argtypes = [vp]
    lib.trimeg_density_g2p.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.trimeg_f_interp.argtypes = [vp, vp, C.c_int]
    lib.trimeg_gather_gyro.argtypes = [vp, i64, vp, vp, vp, vp, i32, vp, vp, C.c_int]
    lib.trimeg_deposit.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.trimeg_build_info.argtypes = []
    lib.trimeg_build_info.restype = C.c_char_p
    lib.trimeg_fields_bytes.argtypes = [vp]
    lib.trimeg_fields_bytes.restype = C.c_size_t
    lib.trimeg_fields_export.argtypes = [vp, vp, C.c_size_t]
    lib.trimeg_fields_import.argtypes = [vp, vp, C.c_size_t]
    lib.trimeg_scratch_bytes.argtypes = [vp, i64]
    lib.trimeg_scratch_bytes.restype = C.c_size_t
    lib.trimeg_markers_bind.argtypes = [vp, i64] + [vp] * 7 + [C.c_int, vp, C.c_size_t]
    lib.trimeg_markers_get.argtypes = [vp] + [vp] * 6 + [C.c_int]
    lib.trimeg_sort.argtypes = [vp]
    lib.trimeg_set_sort_interval.argtypes = [vp, i32]
    lib.trimeg_push_rk4.argtypes = [vp, dbl, i32]
    lib.trimeg_rhs.argtypes = [vp, vp, C.c_int]
    lib.trimeg_set_push_variant.argtypes = [vp, i32]
    lib.trimeg_push_variant_used.argtypes = [vp, C.POINTER(i32)]
    lib.trimeg_bench_dfma.argtypes = [vp, C.POINTER(dbl)]
    lib.trimeg_bench_dfma_mix.argtypes = [vp, i32, C.POINTER(dbl)]
    lib.trimeg_push_stats.argtypes = [vp, C.POINTER(i64)]
    lib.trimeg_push_kernel_ms.argtypes = [vp, C.POINTER(dbl)]
    _lib = lib
    return lib


def _ptr(x):
    """(address, memspace) of a numpy array (HOST) or torch tensor (HOST or DEVICE); None -> (None, HOST)."""
    if x is None:
        return None, HOST
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data, HOST
    assert x.is_contiguous()
    return x.data_ptr(), (DEVICE if x.is_cuda else HOST)


def build_info() -> str:
    """-D options of a tuning build ("" for the shipped configuration)."""
    return load_library().trimeg_build_info().decode()


class Trimeg:
    """One library context.  Method names follow the C calls (trimeg_<name>)."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise TrimegError("no CUDA device: the marker push has no CPU fallback")
        self._torch = torch
        self._lib = load_library()
        self.device = torch.device("cuda", device)
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        rc = self._lib.trimeg_create(C.byref(h), device, C.c_void_p(self._stream.cuda_stream))
        if rc != 0:
            raise TrimegError(f"trimeg_create failed rc={rc}")
        self._h = h
        self._scratch = None
        self.n = 0
        self.n_tri = self.n_nodes = self.n_planes = 0

    def close(self):
        if getattr(self, "_h", None):
            self._lib.trimeg_destroy(self._h)
            self._h = None
            self._scratch = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc, what):
        if rc != 0:
            msg = self._lib.trimeg_last_error(self._h)
            raise TrimegError(f"{what}: rc={rc}: {msg.decode() if msg else ''}")

    # ---- setup
    def equilibrium_set(self, R0, a, B0, q0, q1, q2, qbar_sqrt=1):
        e = _Equil(R0, a, B0, q0, q1, q2, int(qbar_sqrt))
        self._ck(self._lib.trimeg_equilibrium_set(self._h, C.byref(e)), "trimeg_equilibrium_set")

    def equilibrium_set_numeric(self, nR, nZ, Rmin, Rmax, Zmin, Zmax, F, R0, a, coef):
        coef = np.ascontiguousarray(coef, dtype=np.float64)
        assert coef.shape == (nR + 3, nZ + 3), coef.shape
        gs = _EquilGrid(int(nR), int(nZ), Rmin, Rmax, Zmin, Zmax, F, R0, a)
        self._ck(self._lib.trimeg_equilibrium_set_numeric(self._h, C.byref(gs), coef.ctypes.data), "trimeg_equilibrium_set_numeric")

    def species_set(self, qom, kappa_n=0.0, kappa_T=0.0, w_n=0.3, w_T=0.3, r0=0.0, bstar_exact=1, weight_mode=0):
        s = _Species(qom, kappa_n, kappa_T, w_n, w_T, r0, int(bstar_exact), int(weight_mode))
        self._ck(self._lib.trimeg_species_set(self._h, C.byref(s)), "trimeg_species_set")

    def mesh_load(self, RZ, tri, n_planes, phi_period=2 * np.pi):
        RZ = np.ascontiguousarray(RZ, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        rc = self._lib.trimeg_mesh_load(self._h, RZ.shape[0], RZ.ctypes.data, tri.shape[0], tri.ctypes.data,
                                        int(n_planes), float(phi_period))
        self.n_nodes = self.n_tri = self.n_planes = 0
        self._ck(rc, "trimeg_mesh_load")
        self.n_nodes, self.n_tri, self.n_planes = RZ.shape[0], tri.shape[0], int(n_planes)

    def fields_set(self, which, dof):
        if isinstance(dof, np.ndarray):
            dof = np.ascontiguousarray(dof, dtype=np.float64)
        if self.n_planes:  # without a mesh the C call reports BAD_STATE itself
            assert tuple(dof.shape) == (self.n_planes, self.n_nodes, 6), tuple(dof.shape)
        p, ms = _ptr(dof)
        self._ck(self._lib.trimeg_fields_set(self._h, int(which), p, ms), "trimeg_fields_set")

    @staticmethod
    def build_info():
        return build_info()

    def fields_bytes(self):
        return int(self._lib.trimeg_fields_bytes(self._h))

    def fields_export(self, out=None):
        """-> uint8 CUDA tensor holding the coefficient table (opaque; for a broadcast to other ranks)."""
        n = self.fields_bytes()
        if out is None:
            out = self._torch.empty(n, dtype=self._torch.uint8, device=self.device)
        assert out.is_cuda and out.is_contiguous() and out.numel() * out.element_size() == n
        self._ck(self._lib.trimeg_fields_export(self._h, out.data_ptr(), n), "trimeg_fields_export")
        return out

    def fields_import(self, buf):
        assert buf.is_cuda and buf.is_contiguous()
        self._ck(self._lib.trimeg_fields_import(self._h, buf.data_ptr(), buf.numel() * buf.element_size()), "trimeg_fields_import")

    def set_gather_mode(self, mode):
        """0 automatic, 1 direct kernel, 2 staged path."""
        self._ck(self._lib.trimeg_set_gather_mode(self._h, int(mode)), "trimeg_set_gather_mode")

    def gather_kernel_ms(self):
        a = (C.c_double * 6)()
        self._ck(self._lib.trimeg_gather_kernel_ms(self._h, a), "trimeg_gather_kernel_ms")
        return dict(keys=a[0], scan=a[1], scatter=a[2], staged=a[3], unsort=a[4], direct=a[5])

    # ---- gather
    def gather(self, R, Z, phi, out=None, tri_out=None, want_tri=True):
        """R, Z, phi: all numpy (HOST) or all CUDA tensors (DEVICE). Returns (out[8,n], tri[n] or None) of the same kind."""
        pR, ms = _ptr(R)
        pZ, ms2 = _ptr(Z)
        pP, ms3 = _ptr(phi)
        assert ms == ms2 == ms3
        n = int(R.shape[0])
        if ms == HOST:
            assert all(a.dtype == np.float64 for a in (R, Z, phi))
            out = np.empty((8, n)) if out is None else out
            tri_out = np.empty(n, dtype=np.int32) if (tri_out is None and want_tri) else tri_out
        else:
            t = self._torch
            out = t.empty((8, n), dtype=t.float64, device=self.device) if out is None else out
            tri_out = t.empty(n, dtype=t.int32, device=self.device) if (tri_out is None and want_tri) else tri_out
        po, _ = _ptr(out)
        pt, _ = _ptr(tri_out)
        self._ck(self._lib.trimeg_gather(self._h, n, pR, pZ, pP, po, pt, ms), "trimeg_gather")
        return out, tri_out

    GATHER_NOALLOC_MAX = 131072

    def gather_noalloc(self, R, Z, phi, out, tri_out=None):
        """trimeg_gather_noalloc: CUDA tensors only, caller-provided out [8, n] (and tri_out [n] or None); the library allocates
        nothing (static scratch array, at most GATHER_NOALLOC_MAX points per call)."""
        ptrs = [_ptr(a) for a in (R, Z, phi, out)]
        assert all(q[1] == DEVICE for q in ptrs), "gather_noalloc takes DEVICE buffers"
        pt = _ptr(tri_out)[0] if tri_out is not None else None
        self._ck(self._lib.trimeg_gather_noalloc(self._h, int(R.shape[0]), *[q[0] for q in ptrs], pt), "trimeg_gather_noalloc")
        return out, tri_out

    def gather_gyro(self, R, Z, phi, rho, npts):
        """N-point gyro-average of the gather; all numpy (HOST) or all CUDA tensors (DEVICE) -> (out[8,n], tri[n])."""
        ptrs = [_ptr(a) for a in (R, Z, phi, rho)]
        ms = ptrs[0][1]
        assert all(q[1] == ms for q in ptrs)
        n = int(R.shape[0])
        if ms == HOST:
            out, tri = np.empty((8, n)), np.empty(n, dtype=np.int32)
        else:
            t = self._torch
            out, tri = t.empty((8, n), dtype=t.float64, device=self.device), t.empty(n, dtype=t.int32, device=self.device)
        self._ck(self._lib.trimeg_gather_gyro(self._h, n, *[q[0] for q in ptrs], int(npts), _ptr(out)[0], _ptr(tri)[0], ms), "trimeg_gather_gyro")
        return out, tri

    # ---- markers
    def scratch_bytes(self, n):
        return int(self._lib.trimeg_scratch_bytes(self._h, int(n)))

    def markers_bind(self, R, Z, phi, u, w, mu, p):
        """Seven arrays [n], all numpy float64 (HOST) or all CUDA float64 tensors (DEVICE)."""
        arrs = [R, Z, phi, u, w, mu, p]
        ptrs = [_ptr(a) for a in arrs]
        ms = ptrs[0][1]
        assert all(q[1] == ms for q in ptrs)
        n = int(R.shape[0])
        nbytes = self.scratch_bytes(n)
        if self._scratch is None or self._scratch.numel() < nbytes:
            self._scratch = None
            self._scratch = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
        self._hold = arrs  # HOST inputs must outlive the async copies
        rc = self._lib.trimeg_markers_bind(self._h, n, *[q[0] for q in ptrs], ms, self._scratch.data_ptr(), nbytes)
        self._ck(rc, "trimeg_markers_bind")
        self.n = n

    def markers_get(self, host=False, pinned=None):
        """-> dict R, Z, phi, u, w (float64), status (int32) in the caller's order; CUDA tensors or numpy arrays."""
        t = self._torch
        if host:
            if pinned is not None:
                out = pinned
            else:
                out = {k: np.empty(self.n) for k in ("R", "Z", "phi", "u", "w")}
                out["status"] = np.empty(self.n, dtype=np.int32)
            ms = HOST
        else:
            out = {k: t.empty(self.n, dtype=t.float64, device=self.device) for k in ("R", "Z", "phi", "u", "w")}
            out["status"] = t.empty(self.n, dtype=t.int32, device=self.device)
            ms = DEVICE
        ptrs = [_ptr(out[k])[0] for k in ("R", "Z", "phi", "u", "w", "status")]
        self._ck(self._lib.trimeg_markers_get(self._h, *ptrs, ms), "trimeg_markers_get")
        return out

    def sort(self):
        self._ck(self._lib.trimeg_sort(self._h), "trimeg_sort")

    def set_sort_interval(self, every_n_steps):
        self._ck(self._lib.trimeg_set_sort_interval(self._h, int(every_n_steps)), "trimeg_set_sort_interval")

    def set_push_variant(self, variant):
        self._ck(self._lib.trimeg_set_push_variant(self._h, int(variant)), "trimeg_set_push_variant")

    def push_variant_used(self):
        v = C.c_int32(-1)
        self._ck(self._lib.trimeg_push_variant_used(self._h, C.byref(v)), "trimeg_push_variant_used")
        return v.value

    def push_rk4(self, dt, nsteps):
        self._ck(self._lib.trimeg_push_rk4(self._h, float(dt), int(nsteps)), "trimeg_push_rk4")

    def rhs(self, host=False):
        t = self._torch
        out = np.empty((5, self.n)) if host else t.empty((5, self.n), dtype=t.float64, device=self.device)
        p, ms = _ptr(out)
        self._ck(self._lib.trimeg_rhs(self._h, p, ms), "trimeg_rhs")
        return out

    def pullback(self):
        self._ck(self._lib.trimeg_pullback(self._h), "trimeg_pullback")

    def _scalar_out(self, host):
        t = self._torch
        return np.empty(self.n) if host else t.empty(self.n, dtype=t.float64, device=self.device)

    def density_g2p(self, which, host=False):
        out = self._scalar_out(host)
        p, ms = _ptr(out)
        self._ck(self._lib.trimeg_density_g2p(self._h, int(which), p, ms), "trimeg_density_g2p")
        return out

    def f_interp(self, host=False):
        out = self._scalar_out(host)
        p, ms = _ptr(out)
        self._ck(self._lib.trimeg_f_interp(self._h, p, ms), "trimeg_f_interp")
        return out

    def deposit(self, quantity=0, host=False):
        """P2G: -> b[n_planes][n_nodes][6]; quantity 0: charges w, 1: w * u."""
        t = self._torch
        shape = (self.n_planes, self.n_nodes, 6)
        out = np.empty(shape) if host else t.empty(shape, dtype=t.float64, device=self.device)
        p, ms = _ptr(out)
        self._ck(self._lib.trimeg_deposit(self._h, int(quantity), p, ms), "trimeg_deposit")
        return out

    def sync(self):
        self._ck(self._lib.trimeg_sync(self._h), "trimeg_sync")

    def bench_dfma(self):
        v = C.c_double(0)
        self._ck(self._lib.trimeg_bench_dfma(self._h, C.byref(v)), "trimeg_bench_dfma")
        return v.value

    def bench_dfma_mix(self, kind):
        v = C.c_double(0)
        self._ck(self._lib.trimeg_bench_dfma_mix(self._h, int(kind), C.byref(v)), "trimeg_bench_dfma_mix")
        return v.value

    def push_stats(self):
        a = (C.c_int64 * 4)()
        self._ck(self._lib.trimeg_push_stats(self._h, a), "trimeg_push_stats")
        return dict(launches=a[0], slow_path=a[1], retired=a[2], sorts=a[3])

    def push_kernel_ms(self):
        a = (C.c_double * 3)()
        self._ck(self._lib.trimeg_push_kernel_ms(self._h, a), "trimeg_push_kernel_ms")
        return dict(sort=a[0], push=a[1], finish=a[2])
