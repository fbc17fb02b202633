"""Thin Python binding of include/pasta.h: argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch supplies device memory (the library's
internal buffers are torch tensors handed out through pasta_env.alloc), the stream, and the
tensors results are returned in.  There is no CPU fallback: if the library cannot be built or
loaded, or no CUDA device is usable, the calls raise.
"""
import ctypes as C
import os

from . import build as _build

_lib = None


class PastaError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("pasta error %d: %s" % (code, text))
        self.code = code


class Params(C.Structure):
    """pasta_params (include/pasta.h)."""

    _fields_ = [
        ("struct_size", C.c_uint32), ("reserved0", C.c_uint32),
        ("a", C.c_double), ("b", C.c_double), ("c", C.c_double), ("Lambda", C.c_double),
        ("alpha_hbarc", C.c_double), ("lambda_", C.c_double), ("r_c", C.c_double), ("mass", C.c_double),
        ("scale_per_step", C.c_double),
        ("thermostat_interval", C.c_int32), ("cell_subdiv", C.c_int32), ("energy_every_step", C.c_int32),
        ("skip_exact_zeros", C.c_int32), ("list_reuse", C.c_int32),
        ("list_halo", C.c_double), ("r_nuc", C.c_double), ("xi_dot", C.c_double),
        ("coulomb_all_pairs", C.c_int32), ("reserved1", C.c_int32),
    ]


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
_ALLREDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_int64, C.c_void_p)


class Env(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("device", C.c_int32), ("stream", C.c_void_p),
                ("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


# name -> (restype, argtypes); the ABI test checks that the library exports exactly these.
SIGNATURES = {
    "pasta_params_default": (C.c_int, [C.POINTER(Params)]),
    "pasta_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int64, C.c_double, C.c_double, C.c_double,
                               C.POINTER(Params), C.c_uint64, C.POINTER(Env)]),
    "pasta_destroy": (C.c_int, [C.c_void_p]),
    "pasta_forces": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]),
    "pasta_step": (C.c_int, [C.c_void_p, C.c_int64, C.c_double]),
    "pasta_expand": (C.c_int, [C.c_void_p, C.c_double]),
    "pasta_clusters": (C.c_int, [C.c_void_p, C.c_double, C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_clusters_mst": (C.c_int, [C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_clusters_noalloc": (C.c_int, [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.c_void_p, C.c_void_p,
                                         C.c_int32, C.c_void_p]),
    "pasta_cluster_sizes": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pasta_composition": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(C.c_double)]),
    "pasta_get_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double),
                                  C.POINTER(C.c_int64)]),
    "pasta_set_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]),
    "pasta_get_state_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double),
                                       C.POINTER(C.c_int64)]),
    "pasta_set_state_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]),
    "pasta_set_state_host_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]),
    "pasta_get_state_host_async": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double),
                                             C.POINTER(C.c_int64)]),
    "pasta_host_sync": (C.c_int, [C.c_void_p]),
    "pasta_cells": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)]),
    "pasta_ncell": (C.c_int, [C.c_void_p, C.POINTER(C.c_int32)]),
    "pasta_force_grid": (C.c_int, [C.c_void_p, C.POINTER(C.c_int32)]),
    "pasta_force_cells": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pasta_list_stats": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_energy": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "pasta_particle_energies": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pasta_pair_count": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_pair_counts": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_force_stats": (C.c_int, [C.c_void_p, C.POINTER(C.c_int64)]),
    "pasta_set_timing": (C.c_int, [C.c_void_p, C.c_int32]),
    "pasta_get_timing": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
    "pasta_launch_count": (C.c_int64, [C.c_void_p]),
    "pasta_graph_replays": (C.c_int64, [C.c_void_p]),
    "pasta_set_shard": (C.c_int, [C.c_void_p, C.c_int32, C.c_int32, _ALLREDUCE_FN, C.c_void_p]),
    "pasta_shard_bounds": (C.c_int, [C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_int32, C.POINTER(C.c_int64)]),
    "pasta_shard_costs": (C.c_int, [C.c_void_p, C.POINTER(C.c_double)]),
    "pasta_last_error": (C.c_char_p, []),
    "pasta_version": (C.c_char_p, []),
}


def library_path():
    return _build.LIB


def load():
    """Build (if stale) and load the C-ABI library; raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        lib = C.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _check(rc):
    if rc != 0:
        raise PastaError(rc, load().pasta_last_error().decode())


def shard_bounds(N, Np, cost_p, cost_n, world):
    """pasta_shard_bounds: the sorted-slot stretch of every rank (host arithmetic only, no GPU needed)."""
    out = (C.c_int64 * (int(world) + 1))()
    _check(load().pasta_shard_bounds(int(N), int(Np), float(cost_p), float(cost_n), int(world), out))
    return [int(b) for b in out]


CLUSTERS_NOALLOC_MAX_N = 65536  # PASTA_CLUSTERS_NOALLOC_MAX_N of include/pasta.h


def clusters_noalloc(x, L, r_cl, label_out, n_clusters_out=None, stream=None):
    """pasta_clusters_noalloc: friends-of-friends labels of the positions x ([N,3] float64 cuda tensor, box side L)
    written into label_out ([N] int32 cuda) and the number of clusters into n_clusters_out ([1] int64 cuda, optional).

    For callers that cannot allocate device memory when they need the labels -- the free memory of the GPU belongs to
    someone else's pool, or a cudaMalloc would stall a simulation stepping on other streams.  Neither this wrapper nor
    the library call behind it allocates on the device: the outputs are the caller's tensors and the working memory is
    a fixed array inside the library, which limits N to CLUSTERS_NOALLOC_MAX_N (a larger N raises PastaError, code -1).
    Nothing is synchronised; the results are ordered with `stream` (default: torch's current stream of x's device).
    All calls on one GPU share that working array: do not let two of them overlap on the device."""
    import torch

    if not (x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.dim() == 2 and x.shape[1] == 3):
        raise ValueError("x must be a contiguous [N,3] float64 cuda tensor")
    N = x.shape[0]
    if not (label_out.is_cuda and label_out.dtype == torch.int32 and label_out.is_contiguous()
            and label_out.numel() == N and label_out.device == x.device):
        raise ValueError("label_out must be a contiguous [N] int32 tensor on x's device")
    if n_clusters_out is not None and not (n_clusters_out.dtype == torch.int64 and n_clusters_out.numel() == 1
                                           and n_clusters_out.device == x.device):
        raise ValueError("n_clusters_out must be one int64 on x's device")
    st = torch.cuda.current_stream(x.device) if stream is None else stream
    _check(load().pasta_clusters_noalloc(
        C.c_void_p(x.data_ptr()), N, float(L), float(r_cl), C.c_void_p(label_out.data_ptr()),
        None if n_clusters_out is None else C.c_void_p(n_clusters_out.data_ptr()), x.device.index,
        C.c_void_p(st.cuda_stream)))


def default_params(**overrides):
    p = Params()
    _check(load().pasta_params_default(C.byref(p)))
    for k, v in overrides.items():
        if k == "lambda":
            k = "lambda_"
        if not hasattr(p, k):
            raise AttributeError("pasta_params has no field %r" % k)
        setattr(p, k, v)
    return p


class Sim:
    """One simulation on one GPU (an opaque pasta_sim handle plus the torch tensors backing it)."""

    def __init__(self, N, Y_P, density, T, params=None, seed=0, device=None, stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("pasta: no CUDA device is available and there is no CPU fallback")
        self._torch = torch
        self.lib = load()
        self.device = torch.device("cuda", torch.cuda.current_device() if device is None else device)
        self.params = params if params is not None else default_params()
        self.N = int(N)
        self._pool = {}
        torch_dev = self.device

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=torch_dev)
            except Exception:  # out of memory -> NULL -> PASTA_ENOMEM
                return None
            self._pool[t.data_ptr()] = t
            return t.data_ptr()

        def _free(ptr, _user):
            self._pool.pop(ptr, None)

        self._alloc_cb = _ALLOC_FN(_alloc)
        self._free_cb = _FREE_FN(_free)
        with torch.cuda.device(self.device):
            st = torch.cuda.current_stream() if stream is None else stream
        self.stream = st
        self._env = Env(C.sizeof(Env), self.device.index, C.c_void_p(st.cuda_stream), self._alloc_cb, self._free_cb, None)
        h = C.c_void_p()
        _check(self.lib.pasta_create(C.byref(h), self.N, float(Y_P), float(density), float(T), C.byref(self.params),
                                     int(seed), C.byref(self._env)))
        self._h = h

    # -- lifetime ------------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self.lib.pasta_destroy(self._h)
            self._h = None
            self._pool.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _empty(self, shape, dtype):
        return self._torch.empty(shape, dtype=dtype, device=self.device)

    def _dev(self, t, dtype, numel):
        torch = self._torch
        if t is None:
            return None, None
        t = torch.as_tensor(t)
        t = t.to(device=self.device, dtype=dtype).contiguous()
        if t.numel() != numel:
            raise ValueError("expected %d elements, got %d" % (numel, t.numel()))
        return t, C.c_void_p(t.data_ptr())

    # -- the five calls of the north star -------------------------------------------------------------
    def forces(self, want_pe=True):
        """pasta_forces -> (F [N,3] float64 cuda tensor, PE float or None)."""
        F = self._empty((self.N, 3), self._torch.float64)
        pe = C.c_double()
        _check(self.lib.pasta_forces(self._h, C.c_void_p(F.data_ptr()), C.byref(pe) if want_pe else None))
        return F, (pe.value if want_pe else None)

    def step(self, n, dt):
        _check(self.lib.pasta_step(self._h, int(n), float(dt)))

    def expand(self, scale):
        _check(self.lib.pasta_expand(self._h, float(scale)))

    def clusters(self, r_cl):
        """pasta_clusters -> (label [N] int32 cuda tensor, n_clusters)."""
        label = self._empty((self.N,), self._torch.int32)
        n = C.c_int64()
        _check(self.lib.pasta_clusters(self._h, float(r_cl), C.c_void_p(label.data_ptr()), C.byref(n)))
        return label, n.value

    # -- accessors --------------------------------------------------------------------------------------
    def clusters_mst(self, r_pp=4.5, r_np=3.0):
        """The paper's two-radius MST clusters: (label[N] int32 tensor, number of clusters)."""
        label = self._empty((self.N,), self._torch.int32)
        n = C.c_int64()
        _check(self.lib.pasta_clusters_mst(self._h, r_pp, r_np, C.c_void_p(label.data_ptr()), C.byref(n)))
        return label, n.value

    def cluster_sizes(self):
        A = self._empty((self.N,), self._torch.int32)
        Z = self._empty((self.N,), self._torch.int32)
        _check(self.lib.pasta_cluster_sizes(self._h, C.c_void_p(A.data_ptr()), C.c_void_p(Z.data_ptr())))
        return A, Z

    def composition(self, a_min=12):
        out = (C.c_double * 6)()
        _check(self.lib.pasta_composition(self._h, int(a_min), out))
        return dict(zip(("free_n_fraction", "n_heavy", "mean_A", "sigma_A", "mean_Z", "sigma_Z"), list(out)))

    def get_state(self):
        """-> x [N,3], v [N,3] (float64 cuda), is_proton [N] (uint8 cuda), L, step."""
        torch = self._torch
        x = self._empty((self.N, 3), torch.float64)
        v = self._empty((self.N, 3), torch.float64)
        p = self._empty((self.N,), torch.uint8)
        L, step = C.c_double(), C.c_int64()
        _check(self.lib.pasta_get_state(self._h, C.c_void_p(x.data_ptr()), C.c_void_p(v.data_ptr()),
                                        C.c_void_p(p.data_ptr()), C.byref(L), C.byref(step)))
        return x, v, p, L.value, step.value

    def set_state(self, x, v, is_proton=None, F=None, L=None):
        torch = self._torch
        if L is None:
            L = self.box_length()
        keep = []
        ptrs = []
        for t, dt, n in ((x, torch.float64, 3 * self.N), (v, torch.float64, 3 * self.N),
                         (is_proton, torch.uint8, self.N), (F, torch.float64, 3 * self.N)):
            tt, ptr = self._dev(t, dt, n)
            keep.append(tt)
            ptrs.append(ptr)
        _check(self.lib.pasta_set_state(self._h, ptrs[0], ptrs[1], ptrs[2], ptrs[3], float(L)))
        self.stream.synchronize()  # `keep` may be temporaries
        del keep

    def set_state_host(self, x, v, is_proton=None, F=None, L=None):
        """Host (ideally pinned) torch CPU tensors -> device, asynchronously on the stream."""
        if L is None:
            L = self.box_length()

        def hp(t):
            return None if t is None else C.c_void_p(t.data_ptr())

        _check(self.lib.pasta_set_state_host(self._h, hp(x), hp(v), hp(is_proton), hp(F), float(L)))

    def get_state_host(self, x=None, v=None, F=None):
        def hp(t):
            return None if t is None else C.c_void_p(t.data_ptr())

        L, step = C.c_double(), C.c_int64()
        _check(self.lib.pasta_get_state_host(self._h, hp(x), hp(v), hp(F), C.byref(L), C.byref(step)))
        return L.value, step.value

    def set_state_host_async(self, x, v, F=None, L=None):
        """Pipelined upload (pinned torch CPU tensors): returns at once; see pasta_set_state_host_async."""
        if L is None:
            L = self.box_length()
        hp = lambda t: None if t is None else C.c_void_p(t.data_ptr())  # noqa: E731
        _check(self.lib.pasta_set_state_host_async(self._h, hp(x), hp(v), hp(F), float(L)))

    def get_state_host_async(self, x=None, v=None, F=None):
        """Pipelined download: returns (L, step) at once; the buffers are valid after host_sync()."""
        hp = lambda t: None if t is None else C.c_void_p(t.data_ptr())  # noqa: E731
        L, step = C.c_double(), C.c_int64()
        _check(self.lib.pasta_get_state_host_async(self._h, hp(x), hp(v), hp(F), C.byref(L), C.byref(step)))
        return L.value, step.value

    def host_sync(self):
        _check(self.lib.pasta_host_sync(self._h))

    def box_length(self):
        L = C.c_double()
        _check(self.lib.pasta_get_state(self._h, None, None, None, C.byref(L), None))
        return L.value

    def step_count(self):
        n = C.c_int64()
        _check(self.lib.pasta_get_state(self._h, None, None, None, None, C.byref(n)))
        return n.value

    def ncell(self):
        n = C.c_int32()
        _check(self.lib.pasta_ncell(self._h, C.byref(n)))
        return n.value

    def cells(self):
        """-> cell_id [N] int32, cell_start [ncell^3+1] int32 (cuda), ncell per side."""
        nc = self.ncell()
        cid = self._empty((self.N,), self._torch.int32)
        start = self._empty((nc ** 3 + 1,), self._torch.int32)
        n = C.c_int32()
        _check(self.lib.pasta_cells(self._h, C.c_void_p(cid.data_ptr()), C.c_void_p(start.data_ptr()), C.byref(n)))
        assert n.value == nc
        return cid, start, nc

    def force_grid(self):
        """{'ncell': (protons, neutrons), 'ncx': (protons, neutrons)} of the force path's per-species grids."""
        out = (C.c_int32 * 4)()
        _check(self.lib.pasta_force_grid(self._h, out))
        return {"ncell": (out[0], out[2]), "ncx": (out[1], out[3])}

    def force_cells(self):
        """The force path's own cell list of the current positions: bin [N], bin_start [bins + 1], perm [N] (int32 cuda)."""
        g = self.force_grid()
        nbins = sum(nc * nc * ncx for nc, ncx in zip(g["ncell"], g["ncx"]))
        i32 = self._torch.int32
        b, start, perm = self._empty((self.N,), i32), self._empty((nbins + 1,), i32), self._empty((self.N,), i32)
        _check(self.lib.pasta_force_cells(self._h, C.c_void_p(b.data_ptr()), C.c_void_p(start.data_ptr()),
                                          C.c_void_p(perm.data_ptr())))
        return b, start, perm, g

    def list_stats(self):
        out = (C.c_int64 * 2)()
        _check(self.lib.pasta_list_stats(self._h, out))
        return {"force_evals": int(out[0]), "list_builds": int(out[1])}

    def energy(self):
        ke, pe = C.c_double(), C.c_double()
        _check(self.lib.pasta_energy(self._h, C.byref(ke), C.byref(pe)))
        return ke.value, pe.value

    def kinetic(self):
        ke = C.c_double()
        _check(self.lib.pasta_energy(self._h, C.byref(ke), None))
        return ke.value

    def particle_energies(self):
        e = self._empty((self.N,), self._torch.float64)
        _check(self.lib.pasta_particle_energies(self._h, C.c_void_p(e.data_ptr())))
        return e

    def pair_count(self):
        n = C.c_int64()
        _check(self.lib.pasta_pair_count(self._h, C.byref(n)))
        return n.value

    def pair_counts(self):
        """(ordered in-range pairs, those with a term that is not exactly zero in FP32)."""
        out = (C.c_int64 * 2)()
        _check(self.lib.pasta_pair_counts(self._h, out))
        return int(out[0]), int(out[1])

    def force_stats(self):
        out = (C.c_int64 * 3)()
        _check(self.lib.pasta_force_stats(self._h, out))
        return {"sources_streamed": out[0], "tiles": out[1], "pair_evaluations": out[2]}

    def set_timing(self, enable=True):
        _check(self.lib.pasta_set_timing(self._h, 1 if enable else 0))

    def get_timing(self):
        ms = (C.c_double * 3)()
        n = C.c_int64()
        _check(self.lib.pasta_get_timing(self._h, ms, C.byref(n)))
        return {"cells_ms": ms[0], "force_ms": ms[1], "integrate_ms": ms[2], "force_evals": n.value}

    def launch_count(self):
        return int(self.lib.pasta_launch_count(self._h))

    def graph_replays(self):
        return int(self.lib.pasta_graph_replays(self._h))

    # -- target sharding over several GPUs (pasta_set_shard) -------------------------------------------
    def _f64_view(self, ptr, n):
        """The n doubles at device address ptr as a torch tensor (ptr lies inside one of the library's buffers,
        which are torch tensors handed out through pasta_env.alloc)."""
        for base, t in self._pool.items():
            if base <= ptr and ptr + 8 * n <= base + t.numel():
                return t[ptr - base: ptr - base + 8 * n].view(self._torch.float64)
        raise ValueError("pasta: allreduce on a pointer that is not inside a library buffer")

    def set_shard(self, rank, world, group=None, allreduce=None):
        """pasta_set_shard: this process evaluates the targets of stretch `rank` of `world` of the cell-sorted order;
        the partial forces/energies are summed over the ranks with torch.distributed.all_reduce on `group` (NCCL over
        NVLink on a multi-GPU node), ordered with the simulation's stream.  `allreduce` (a callable taking the tensor)
        replaces the collective -- the tests use it to play the ranks one after another on a single GPU."""
        torch = self._torch

        def _cb(ptr, n, _user):
            try:
                t = self._f64_view(int(ptr), int(n))
                with torch.cuda.stream(self.stream):
                    if allreduce is not None:
                        allreduce(t)
                    else:
                        import torch.distributed as dist

                        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
                return 0
            except Exception:  # no exception crosses the ABI
                import traceback

                traceback.print_exc()
                return 1

        self._shard_cb = _ALLREDUCE_FN(_cb) if int(world) > 1 else _ALLREDUCE_FN()
        _check(self.lib.pasta_set_shard(self._h, int(rank), int(world), self._shard_cb, None))

    def shard_costs(self):
        out = (C.c_double * 2)()
        _check(self.lib.pasta_shard_costs(self._h, out))
        return float(out[0]), float(out[1])
