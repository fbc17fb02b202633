"""ctypes marshalling for pasta_oracle.c (TEST INFRASTRUCTURE ONLY; no arithmetic lives here)."""
import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pasta_oracle.c")
_LIB = os.path.join(_HERE, "libpasta_oracle.so")
_lib = None


class _CParams(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("a", "b", "c", "Lambda", "alpha", "lambda_", "r_c", "mass", "r_nuc", "coul_nocut")]


@dataclass
class Params:
    """Table I, Eq. 1c alpha*hbar*c and lambda, M."""

    a: float = 110.0
    b: float = -26.0
    c: float = 24.0
    Lambda: float = 1.25
    alpha: float = 1.44
    lambda_: float = 10.0
    r_c: float = 20.0
    mass: float = 939.0
    r_nuc: float = 0.0  # > 0: the paper's separate nuclear cut-off (11.5 fm); 0: none (reading D1)
    coul_nocut: float = 0.0  # != 0: Coulomb between every proton pair at the nearest image, no radial cut-off

    def _c(self):
        if self.coul_nocut and not self.r_nuc > 0.0:
            raise ValueError("coul_nocut needs r_nuc > 0: without r_c the nuclear terms have no other cut-off (PAPER.md:98)")
        return _CParams(self.a, self.b, self.c, self.Lambda, self.alpha, self.lambda_, self.r_c, self.mass, self.r_nuc, self.coul_nocut)


def build(force=False):
    """Compile the oracle with gcc: FP64, no FMA contraction (pinned predicates), OpenMP for timing."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
             _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_ncell.restype = C.c_int32
        _lib.orc_ncell.argtypes = [C.c_double, C.c_double, C.c_int32]
        _lib.orc_kinetic.restype = C.c_double
        _lib.orc_kinetic.argtypes = [C.c_int64, C.c_void_p, C.c_double]
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_forces_cells.restype = C.c_int
        _lib.orc_clusters_cells.restype = C.c_int
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _u8(a):
    return np.ascontiguousarray(a, dtype=np.uint8)


def num_threads():
    return int(_load().orc_num_threads())


def set_num_threads(n):
    _load().orc_set_num_threads(C.c_int(int(n)))


def pair(params, r, pi, pj):
    V, F = C.c_double(), C.c_double()
    _load().orc_pair(C.byref(params._c()), C.c_double(r), C.c_int(int(pi)), C.c_int(int(pj)), C.byref(V), C.byref(F))
    return V.value, F.value


def forces(x, is_p, L, params, targets=None):
    """O1. Returns (F[nt,3], e[nt], PE over the targets, diag dict)."""
    x = _f64(x, (-1, 3))
    is_p = _u8(is_p)
    N = x.shape[0]
    if targets is None:
        nt, tp = N, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = targets.shape[0], _p(targets)
    F = np.zeros((nt, 3))
    e = np.zeros(nt)
    PE = C.c_double()
    diag = np.zeros(3)
    _load().orc_forces(C.c_int64(N), _p(x), _p(is_p), C.c_double(L), C.byref(params._c()), C.c_int64(nt), tp,
                       _p(F), _p(e), C.byref(PE), _p(diag))
    return F, e, PE.value, {"ordered_pairs": diag[0], "boundary_pairs": diag[1], "boundary_absV": diag[2]}


def forces_cells(x, is_p, L, params):
    """P7 helper: same definition through the 27-cell grid. Returns (F, e, PE, ordered_pairs)."""
    x = _f64(x, (-1, 3))
    is_p = _u8(is_p)
    N = x.shape[0]
    F = np.zeros((N, 3))
    e = np.zeros(N)
    PE, npairs = C.c_double(), C.c_double()
    rc = _load().orc_forces_cells(C.c_int64(N), _p(x), _p(is_p), C.c_double(L), C.byref(params._c()), _p(F), _p(e),
                                  C.byref(PE), C.byref(npairs))
    if rc != 0:
        raise ValueError("orc_forces_cells needs floor(L/r_c) >= 3")
    return F, e, PE.value, npairs.value


def wrap(x, L):
    x = _f64(x, (-1, 3)).copy()
    _load().orc_wrap(C.c_int64(x.shape[0]), _p(x), C.c_double(L))
    return x


def ncell(L, r_c, k):
    return int(_load().orc_ncell(C.c_double(L), C.c_double(r_c), C.c_int32(k)))


def cells(x, L, n_cell):
    """O3. Returns (cell_id[N] int32, cell_start[n_cell^3+1] int32)."""
    x = _f64(x, (-1, 3))
    N = x.shape[0]
    cid = np.zeros(N, dtype=np.int32)
    start = np.zeros(n_cell ** 3 + 1, dtype=np.int32)
    _load().orc_cells(C.c_int64(N), _p(x), C.c_double(L), C.c_int32(n_cell), _p(cid), _p(start))
    return cid, start


def cell_coords(x, L, n):
    """O3 per axis: c = min(n-1, floor(x n / L)) for every coordinate; returns int32 array of x's shape."""
    x = _f64(x)
    c = np.zeros(x.shape, dtype=np.int32)
    lib = _load()
    lib.orc_cell_coords.restype = None
    lib.orc_cell_coords(C.c_int64(x.size), _p(x), C.c_double(L), C.c_int32(n), _p(c))
    return c


def kinetic(v, mass):
    v = _f64(v, (-1, 3))
    return float(_load().orc_kinetic(C.c_int64(v.shape[0]), _p(v), C.c_double(mass)))


def step(x, v, is_p, L, params, T, interval, scale_per_step, dt, nsteps, step_count=0, F=None):
    """O2. Returns (x, v, L, step_count, F, PE) after nsteps; inputs are not modified."""
    x = _f64(x, (-1, 3)).copy()
    v = _f64(v, (-1, 3)).copy()
    is_p = _u8(is_p)
    N = x.shape[0]
    if F is None:
        F = forces(x, is_p, L, params)[0]
    F = _f64(F, (-1, 3)).copy()
    Lc, cnt, PE = C.c_double(L), C.c_int64(step_count), C.c_double(0.0)
    _load().orc_step(C.c_int64(N), _p(x), _p(v), _p(is_p), C.byref(Lc), C.byref(params._c()), C.c_double(T),
                     C.c_int32(interval), C.c_double(scale_per_step), C.c_double(dt), C.c_int64(nsteps),
                     C.byref(cnt), _p(F), C.byref(PE))
    return x, v, Lc.value, cnt.value, F, PE.value


def step_linear(x, v, is_p, L0, xi_dot, params, T, interval, dt, nsteps, n_exp=0, step_count=0, F=None):
    """O2': the paper's linear box-only expansion (Eq. 3a; reading D25).
    Returns (x, v, L, n_exp, step_count, F, PE) after nsteps; inputs are not modified."""
    x = _f64(x, (-1, 3)).copy()
    v = _f64(v, (-1, 3)).copy()
    is_p = _u8(is_p)
    N = x.shape[0]
    L = L0 * (1.0 + xi_dot * (dt * float(n_exp)))
    if F is None:
        F = forces(x, is_p, L, params)[0]
    F = _f64(F, (-1, 3)).copy()
    Lc, ne, cnt, PE = C.c_double(L), C.c_int64(n_exp), C.c_int64(step_count), C.c_double(0.0)
    _load().orc_step_linear(C.c_int64(N), _p(x), _p(v), _p(is_p), C.c_double(L0), C.c_double(xi_dot), C.byref(ne),
                            C.byref(Lc), C.byref(params._c()), C.c_double(T), C.c_int32(interval), C.c_double(dt),
                            C.c_int64(nsteps), C.byref(cnt), _p(F), C.byref(PE))
    return x, v, Lc.value, ne.value, cnt.value, F, PE.value


def expand(x, L, s):
    x = _f64(x, (-1, 3)).copy()
    Lc = C.c_double(L)
    _load().orc_expand(C.c_int64(x.shape[0]), _p(x), C.byref(Lc), C.c_double(s))
    return x, Lc.value


def _clusters(fn, x, is_p, L, r_cl):
    x = _f64(x, (-1, 3))
    is_p = _u8(is_p)
    N = x.shape[0]
    label = np.zeros(N, dtype=np.int32)
    A = np.zeros(N, dtype=np.int32)
    Z = np.zeros(N, dtype=np.int32)
    n = C.c_int64()
    rc = fn(C.c_int64(N), _p(x), _p(is_p), C.c_double(L), C.c_double(r_cl), _p(label), _p(A), _p(Z), C.byref(n))
    if rc not in (None, 0):
        raise ValueError("orc_clusters_cells needs floor(L/r_cl) >= 3")
    return label, A, Z, n.value


def clusters(x, is_p, L, r_cl):
    """O4 by brute force. Returns (label[N], A[N], Z[N], n_clusters)."""
    lib = _load()
    lib.orc_clusters.restype = None
    return _clusters(lib.orc_clusters, x, is_p, L, r_cl)


def clusters_mst(x, is_p, L, r_pp=4.5, r_np=3.0):
    """O4': the paper's two-radius MST clusters (reading D24). Returns (label, A, Z, n_clusters)."""
    x = _f64(x, (-1, 3))
    is_p = _u8(is_p)
    N = x.shape[0]
    label = np.zeros(N, dtype=np.int32)
    A = np.zeros(N, dtype=np.int32)
    Z = np.zeros(N, dtype=np.int32)
    n = C.c_int64()
    lib = _load()
    lib.orc_clusters_mst.restype = None
    lib.orc_clusters_mst(C.c_int64(N), _p(x), _p(is_p), C.c_double(L), C.c_double(r_pp), C.c_double(r_np), _p(label),
                         _p(A), _p(Z), C.byref(n))
    return label, A, Z, n.value


def clusters_cells(x, is_p, L, r_cl):
    return _clusters(_load().orc_clusters_cells, x, is_p, L, r_cl)


def composition(A, Z, a_min=12):
    A = np.ascontiguousarray(A, dtype=np.int32)
    Z = np.ascontiguousarray(Z, dtype=np.int32)
    out = np.zeros(6)
    _load().orc_composition(C.c_int64(A.shape[0]), _p(A), _p(Z), C.c_int32(a_min), _p(out))
    return dict(zip(("free_n_fraction", "n_heavy", "mean_A", "sigma_A", "mean_Z", "sigma_Z"), out.tolist()))
