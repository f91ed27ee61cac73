"""ctypes binding of the C ABI in include/pdn.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels behind libpdn.so; this file only builds the C
structs and passes pointers.  torch is used for device memory and streams, nothing else.  There is
no fallback: if libpdn.so is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdn.so")

PDN_OK = 0
PDN_TIERS_ON_HOST = 1
PDN_SKIP_CONNECTIVITY_CHECK = 2
PDN_TIME_KERNELS = 4
PDN_NO_UNIFORM_FAST_PATH = 8
PDN_TERMINAL_PAIRS = 16
PDN_PRECOND_F32 = 32
PDN_NO_INITIAL_GUESS = 64
PDN_STATIC_MAX_LOADS = 512     # pdn.h: largest n_loads pdn_load_voltages_static accepts
KERNEL_CLASSES = ("pq", "down0", "up0", "down_coarse", "up_coarse", "small", "dense", "pair")


class PdnTier(C.Structure):
    _fields_ = [("n", C.c_int32), ("gx", C.c_void_p), ("gy", C.c_void_p)]


class PdnTsv(C.Structure):
    _fields_ = [("iface", C.c_int32), ("y", C.c_int32), ("x", C.c_int32), ("r_ohm", C.c_double)]


class PdnSite(C.Structure):
    _fields_ = [("y", C.c_int32), ("x", C.c_int32)]


class PdnOpts(C.Structure):
    _fields_ = [("rtol", C.c_double), ("max_iter", C.c_int32), ("rhs_batch", C.c_int32),
                ("cuda_stream", C.c_void_p), ("flags", C.c_int32), ("nu", C.c_int32), ("cheb_ratio", C.c_double),
                ("shard_rank", C.c_int32), ("shard_world", C.c_int32)]


class PdnStats(C.Structure):
    _fields_ = [("n_tiers", C.c_int32), ("n_ports_total", C.c_int32), ("n_levels", C.c_int32),
                ("n_uniform_tiers", C.c_int32), ("kernel_launches", C.c_int64), ("stencil_launches", C.c_int64),
                ("pcg_iters_max", C.c_int32), ("pcg_iters_sum", C.c_int32), ("rhs_iterations", C.c_int64),
                ("worst_rel_residual", C.c_double), ("ms_upload", C.c_double), ("ms_stencil", C.c_double),
                ("ms_dense", C.c_double), ("ms_total", C.c_double), ("stencil_bytes", C.c_double),
                ("ms_update_stencil", C.c_double), ("ms_update_dense", C.c_double), ("update_solves", C.c_int64),
                ("class_ms", C.c_double * 8), ("class_bytes", C.c_double * 8),
                ("class_launches", C.c_int64 * 8), ("n_guess_tiers", C.c_int32), ("n_guess_rejected", C.c_int32)]


EXPORTS = ("pdn_create", "pdn_reff", "pdn_reff_host", "pdn_destroy", "pdn_strerror", "pdn_last_error",
           "pdn_get_stats", "pdn_port_count", "pdn_get_port_matrix", "pdn_release_cache", "pdn_update_tsvs",
           "pdn_reff_same_side", "pdn_load_voltages", "pdn_reff_nodes", "pdn_shard_slice", "pdn_shard_buffers",
           "pdn_finish", "pdn_set_solver_opts", "pdn_reff_from", "pdn_load_voltages_static")

_lib = None


def load_library() -> C.CDLL:
    """dlopen libpdn.so (built in-tree by __graft_entry__.build()); fails loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.pdn_create.restype = C.c_int
    lib.pdn_create.argtypes = [C.POINTER(C.c_void_p), C.c_int32, C.POINTER(PdnTier), C.c_int32, C.POINTER(PdnTsv),
                               C.c_int32, C.POINTER(PdnSite), C.c_int32, C.POINTER(PdnSite), C.POINTER(PdnOpts)]
    for name in ("pdn_reff", "pdn_reff_host"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.pdn_destroy.restype = None
    lib.pdn_destroy.argtypes = [C.c_void_p]
    lib.pdn_strerror.restype = C.c_char_p
    lib.pdn_strerror.argtypes = [C.c_int]
    lib.pdn_last_error.restype = C.c_char_p
    lib.pdn_last_error.argtypes = []
    lib.pdn_update_tsvs.restype = C.c_int
    lib.pdn_update_tsvs.argtypes = [C.c_void_p, C.c_int32, C.POINTER(PdnTsv)]
    lib.pdn_set_solver_opts.restype = C.c_int
    lib.pdn_set_solver_opts.argtypes = [C.c_void_p, C.c_double, C.c_int32]
    lib.pdn_reff_same_side.restype = C.c_int
    lib.pdn_reff_same_side.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    for name in ("pdn_load_voltages", "pdn_load_voltages_static"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_double, C.c_void_p]
    lib.pdn_reff_nodes.restype = C.c_int
    lib.pdn_reff_nodes.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.pdn_reff_from.restype = C.c_int
    lib.pdn_reff_from.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.pdn_shard_slice.restype = C.c_int
    lib.pdn_shard_slice.argtypes = [C.c_void_p, C.c_int32, C.c_int32] + [C.POINTER(C.c_int32)] * 4
    lib.pdn_shard_buffers.restype = C.c_int
    lib.pdn_shard_buffers.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_int64),
                                      C.POINTER(C.c_int32), C.POINTER(C.c_void_p)]
    lib.pdn_finish.restype = C.c_int
    lib.pdn_finish.argtypes = [C.c_void_p]
    lib.pdn_release_cache.restype = None
    lib.pdn_release_cache.argtypes = []
    lib.pdn_get_stats.restype = C.c_int
    lib.pdn_get_stats.argtypes = [C.c_void_p, C.POINTER(PdnStats)]
    lib.pdn_port_count.restype = C.c_int32
    lib.pdn_port_count.argtypes = [C.c_void_p, C.c_int32]
    lib.pdn_get_port_matrix.restype = C.c_int
    lib.pdn_get_port_matrix.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    _lib = lib
    return lib


class PdnError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = load_library()
        self.status = status
        msg = lib.pdn_strerror(status).decode()
        detail = lib.pdn_last_error().decode()
        super().__init__(f"{where}: status {status} ({msg}){': ' + detail if detail else ''}")


_TSV_DTYPE = np.dtype([("iface", np.int32), ("y", np.int32), ("x", np.int32), ("r_ohm", np.float64)], align=True)
_SITE_DTYPE = np.dtype([("y", np.int32), ("x", np.int32)], align=True)
assert _TSV_DTYPE.itemsize == C.sizeof(PdnTsv) and _SITE_DTYPE.itemsize == C.sizeof(PdnSite)


def _sites(arr) -> np.ndarray:
    """(k, 2) rows (y, x) -> array of pdn_site (numpy structured array with the C layout)."""
    a = np.ascontiguousarray(arr, dtype=np.int32).reshape(-1, 2)
    out = np.zeros(max(len(a), 1), dtype=_SITE_DTYPE)
    out["y"][: len(a)] = a[:, 0]
    out["x"][: len(a)] = a[:, 1]
    return out


def _tsvs(tsv_site, tsv_r) -> tuple:
    """Per-interface site / resistance lists -> (array of pdn_tsv, count)."""
    n = sum(len(np.asarray(s).reshape(-1, 2)) for s in tsv_site)
    out = np.zeros(max(n, 1), dtype=_TSV_DTYPE)
    k = 0
    for i, (s, r) in enumerate(zip(tsv_site, tsv_r)):
        s = np.asarray(s, dtype=np.int32).reshape(-1, 2)
        out["iface"][k:k + len(s)] = i
        out["y"][k:k + len(s)] = s[:, 0]
        out["x"][k:k + len(s)] = s[:, 1]
        out["r_ohm"][k:k + len(s)] = np.asarray(r, dtype=np.float64)
        k += len(s)
    return out, n


def _ptr(t, kind: str, what: str, count=None) -> int:
    """Address of a torch tensor (device or host) or a numpy array after checking what the C side assumes about
    it: contiguous, dtype `kind` ("f8" = float64, "i4" = int32) and, if given, exactly `count` elements.  The
    library reads / writes raw doubles and int32s: a float32 `out` or an int64 index tensor would be misread
    silently, so they are refused here."""
    if isinstance(t, np.ndarray):
        ok_dtype = t.dtype == (np.float64 if kind == "f8" else np.int32)
        contiguous, n, addr = t.flags["C_CONTIGUOUS"], t.size, t.ctypes.data
    else:
        import torch
        ok_dtype = t.dtype == (torch.float64 if kind == "f8" else torch.int32)
        contiguous, n, addr = t.is_contiguous(), t.numel(), t.data_ptr()
    if not ok_dtype:
        raise TypeError(f"{what} must be {'float64' if kind == 'f8' else 'int32'}, got {t.dtype}")
    if not contiguous:
        raise ValueError(f"{what} must be contiguous")
    if count is not None and n != count:
        raise ValueError(f"{what} must have {count} elements, got {n}")
    return addr


def _on_cuda(t) -> bool:
    return bool(getattr(t, "is_cuda", False))


class _CudaArray:
    """Minimal __cuda_array_interface__ carrier so that torch can alias library-owned device memory."""

    def __init__(self, ptr: int, n: int):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2}


def _device_view(ptr: int, n: int):
    import torch
    return torch.as_tensor(_CudaArray(ptr, n), device=f"cuda:{torch.cuda.current_device()}")


def shard_bounds(k: int, world: int):
    """Rank r owns [floor(r k / world), floor((r+1) k / world)) of k sources (the rule pdn_create applies)."""
    return [(r * k // world, (r + 1) * k // world) for r in range(world)]


class Pdn:
    """Owns one pdn_ctx.  `gx`, `gy`: per-tier (n, n) FP64 planes, torch CUDA tensors (device path)
    or numpy / torch CPU arrays (host path: PDN_TIERS_ON_HOST is set and the library uploads)."""

    def __init__(self, n, gx, gy, tsv_site, tsv_r, bumps, loads, rtol=0.0, max_iter=0, rhs_batch=0,
                 nu=0, flags=0, stream=None, cheb_ratio=0.0, shard_rank=0, shard_world=0):
        lib = load_library()
        d = len(gx)
        on_host = isinstance(gx[0], np.ndarray) or (hasattr(gx[0], "is_cuda") and not gx[0].is_cuda)
        tiers = (PdnTier * d)()
        self._keep = (gx, gy)
        for t in range(d):
            if tuple(gx[t].shape) != (n, n) or tuple(gy[t].shape) != (n, n):
                raise ValueError(f"tier {t}: gx / gy must have shape ({n}, {n})")
            if _on_cuda(gx[t]) == on_host or _on_cuda(gy[t]) == on_host:
                raise ValueError("all conductance planes must live on the same side (all CUDA tensors or all host arrays)")
            tiers[t].n = n
            tiers[t].gx = _ptr(gx[t], "f8", f"gx[{t}]")
            tiers[t].gy = _ptr(gy[t], "f8", f"gy[{t}]")
        tsvs, ntsv = _tsvs(tsv_site, tsv_r)
        self.m = len(np.asarray(bumps).reshape(-1, 2))
        self.nl = len(np.asarray(loads).reshape(-1, 2))
        opts = PdnOpts(rtol=rtol, max_iter=max_iter, rhs_batch=rhs_batch,
                       cuda_stream=C.c_void_p(stream) if stream else None,
                       flags=flags | (PDN_TIERS_ON_HOST if on_host else 0), nu=nu, cheb_ratio=cheb_ratio,
                       shard_rank=shard_rank, shard_world=shard_world)
        self.d = d
        self.n = n
        h = C.c_void_p()
        b_arr, l_arr = _sites(bumps), _sites(loads)
        st = lib.pdn_create(C.byref(h), d, tiers, ntsv, tsvs.ctypes.data_as(C.POINTER(PdnTsv)), self.m,
                            b_arr.ctypes.data_as(C.POINTER(PdnSite)), self.nl,
                            l_arr.ctypes.data_as(C.POINTER(PdnSite)), C.byref(opts))
        if st != PDN_OK:
            raise PdnError(st, "pdn_create")
        self._h = h
        self._lib = lib
        self._terminal_rows = bool(flags & PDN_TERMINAL_PAIRS)
        # the CUDA device the context lives on (the one current at pdn_create): buffers made here go there
        self._device = None
        if not on_host:
            self._device = gx[0].device
        else:
            try:
                import torch
                if torch.cuda.is_available():
                    self._device = torch.device("cuda", torch.cuda.current_device())
            except ImportError:
                pass

    @classmethod
    def from_network(cls, net, device=None, **kw):
        """Convenience: a pdn_inputs.Network; device='cuda' uploads the planes with torch first."""
        gx, gy = net.gx, net.gy
        if device is not None:
            import torch
            gx = [torch.from_numpy(np.ascontiguousarray(g)).to(device) for g in gx]
            gy = [torch.from_numpy(np.ascontiguousarray(g)).to(device) for g in gy]
        return cls(net.n, gx, gy, net.tsv_site, net.tsv_r, net.bumps, net.loads, **kw)

    def _pair_args(self, out, bump_idx, load_idx, device: bool):
        npairs = out.size if isinstance(out, np.ndarray) else out.numel()
        if (bump_idx is None) != (load_idx is None):
            raise ValueError("bump_idx and load_idx must both be given or both be None")
        for t, what in ((out, "out"), (bump_idx, "bump_idx"), (load_idx, "load_idx")):
            if t is not None and _on_cuda(t) != device:
                raise ValueError(f"{what} must be a {'CUDA tensor' if device else 'host array'}")
        if bump_idx is None and npairs != self.m * self.nl:
            raise ValueError(f"the full cross product needs out of {self.m * self.nl} elements, got {npairs}")
        return (npairs, _ptr(bump_idx, "i4", "bump_idx", npairs) if bump_idx is not None else None,
                _ptr(load_idx, "i4", "load_idx", npairs) if load_idx is not None else None, _ptr(out, "f8", "out"))

    def reff(self, out, bump_idx=None, load_idx=None):
        """pdn_reff: `out` (float64) and the index arrays (int32, one entry per pair) are torch CUDA tensors."""
        st = self._lib.pdn_reff(self._h, *self._pair_args(out, bump_idx, load_idx, True))
        if st != PDN_OK:
            raise PdnError(st, "pdn_reff")
        return out

    def reff_host(self, out: np.ndarray, bump_idx=None, load_idx=None):
        """pdn_reff_host: `out` (float64) / index arrays (int32) are numpy (or pinned torch CPU) buffers."""
        st = self._lib.pdn_reff_host(self._h, *self._pair_args(out, bump_idx, load_idx, False))
        if st != PDN_OK:
            raise PdnError(st, "pdn_reff_host")
        return out

    def update_tsvs(self, tsv_site, tsv_r):
        """pdn_update_tsvs: re-plan the TSVs (per-interface site / resistance lists, as in the constructor)."""
        tsvs, ntsv = _tsvs(tsv_site, tsv_r)
        st = self._lib.pdn_update_tsvs(self._h, ntsv, tsvs.ctypes.data_as(C.POINTER(PdnTsv)))
        if st != PDN_OK:
            # A failure before the library's commit point leaves the context valid for the OLD plan; one after it
            # poisons the context (every later call returns PDN_E_ARG).  Either way the caller is told.
            raise PdnError(st, "pdn_update_tsvs")

    def set_solver_opts(self, rtol: float = 0.0, max_iter: int = 0):
        """pdn_set_solver_opts: stopping rule of the port solves later calls run (0 keeps the current value)."""
        st = self._lib.pdn_set_solver_opts(self._h, float(rtol), int(max_iter))
        if st != PDN_OK:
            raise PdnError(st, "pdn_set_solver_opts")

    def reff_same_side(self, side: int, out):
        """pdn_reff_same_side: `out` is a torch CUDA tensor of nt*nt doubles (side 0: bumps, 1: loads)."""
        nt = self.m if side == 0 else self.nl
        st = self._lib.pdn_reff_same_side(self._h, side, _ptr(out, "f8", "out", nt * nt))
        if st != PDN_OK:
            raise PdnError(st, "pdn_reff_same_side")
        return out

    def load_voltages(self, bump: int, i_load, v_bump: float, v_out):
        """pdn_load_voltages (Eq. 4): `i_load`, `v_out` are torch CUDA tensors of n_loads doubles."""
        st = self._lib.pdn_load_voltages(self._h, bump, _ptr(i_load, "f8", "i_load", self.nl), float(v_bump),
                                         _ptr(v_out, "f8", "v_out", self.nl))
        if st != PDN_OK:
            raise PdnError(st, "pdn_load_voltages")
        return v_out

    def load_voltages_static(self, bump: int, i_load, v_bump: float, v_out):
        """pdn_load_voltages_static: Eq. 4 with the scratch in the library's static device array (no allocation;
        at most PDN_STATIC_MAX_LOADS loads).  Same arguments and result as load_voltages."""
        st = self._lib.pdn_load_voltages_static(self._h, bump, _ptr(i_load, "f8", "i_load", self.nl), float(v_bump),
                                                _ptr(v_out, "f8", "v_out", self.nl))
        if st != PDN_OK:
            raise PdnError(st, "pdn_load_voltages_static")
        return v_out

    def reff_nodes(self, nodes, out):
        """pdn_reff_nodes: `nodes` is an (k, 3) integer array of (tier, y, x) probes on the host, `out` a torch CUDA
        tensor of k*k doubles that receives R_eff between every two of them."""
        nd = np.ascontiguousarray(np.asarray(nodes, dtype=np.int32).reshape(-1, 3))
        k = int(nd.shape[0])
        st = self._lib.pdn_reff_nodes(self._h, k, nd.ctypes.data, _ptr(out, "f8", "out", k * k))
        if st != PDN_OK:
            raise PdnError(st, "pdn_reff_nodes")
        return out

    def reff_from(self, src, nodes, out):
        """pdn_reff_from: `src` = (tier, y, x); `nodes` an (k, 3) integer array of (tier, y, x) probes on the host; `out`
        a torch CUDA tensor of k doubles that receives R_eff(src, node) for every probe."""
        sr = np.ascontiguousarray(np.asarray(src, dtype=np.int32).reshape(1, 3))
        nd = np.ascontiguousarray(np.asarray(nodes, dtype=np.int32).reshape(-1, 3))
        k = int(nd.shape[0])
        st = self._lib.pdn_reff_from(self._h, sr.ctypes.data, k, nd.ctypes.data, _ptr(out, "f8", "out", k))
        if st != PDN_OK:
            raise PdnError(st, "pdn_reff_from")
        return out

    def reff_map(self, src, tier: int, stride: int = 1):
        """R_eff map (Fig. 6(d) of the paper): effective resistance from the node `src` = (tier, y, x)
        to every `stride`-th node (rows and columns 0, stride, 2*stride, ...) of tier `tier`, as a 2-D numpy array.
        One pdn_reff_from call with the grid nodes as probes; only marshalling and reshaping here."""
        import torch
        ys = np.arange(0, self.n, stride, dtype=np.int32)
        yy, xx = np.meshgrid(ys, ys, indexing="ij")
        nodes = np.stack([np.full(yy.size, tier, dtype=np.int32), yy.ravel(), xx.ravel()], axis=1)
        out = torch.empty(nodes.shape[0], dtype=torch.float64, device=self._device)
        self.reff_from(src, nodes, out)
        return out.cpu().numpy().reshape(ys.size, ys.size)

    # ---- NEXT-4: one network sharded over several GPUs (argument marshalling + the exchange plumbing only)
    def shard_pieces(self, rank: int):
        """The device pieces rank `rank` owns, as (tier, torch CUDA tensor view) pairs: its rows of every tier's
        port matrix and its slice of zdiag.  The views alias library memory (no copy)."""
        import torch
        out = []
        for t in range(self.d):
            v = [C.c_int32() for _ in range(4)]
            st = self._lib.pdn_shard_slice(self._h, t, rank, *[C.byref(x) for x in v])
            if st != PDN_OK:
                raise PdnError(st, "pdn_shard_slice")
            tsv0, ntsv, term0, nterm = [x.value for x in v]
            zt, ld, ntot, zd = C.c_void_p(), C.c_int64(), C.c_int32(), C.c_void_p()
            st = self._lib.pdn_shard_buffers(self._h, t, C.byref(zt), C.byref(ld), C.byref(ntot), C.byref(zd))
            if st != PDN_OK:
                raise PdnError(st, "pdn_shard_buffers")
            if ntsv:
                out.append((t, _device_view(zt.value + 8 * tsv0 * ld.value, ntsv * ld.value)))
            if nterm:
                out.append((t, _device_view(zd.value + 8 * term0, nterm)))
                if self._terminal_rows:
                    out.append((t, _device_view(zt.value + 8 * (ntot.value + term0) * ld.value, nterm * ld.value)))
        return out

    def exchange_and_finish(self, dist, world: int):
        """Every rank broadcasts its pieces (torch.distributed, NCCL over NVLink on GPUs), then S2-S3 run."""
        for r in range(world):
            for _, piece in self.shard_pieces(r):
                dist.broadcast(piece, src=r)
        self.finish()

    def finish(self):
        st = self._lib.pdn_finish(self._h)
        if st != PDN_OK:
            raise PdnError(st, "pdn_finish")

    def stats(self) -> dict:
        s = PdnStats()
        st = self._lib.pdn_get_stats(self._h, C.byref(s))
        if st != PDN_OK:
            raise PdnError(st, "pdn_get_stats")
        out = {name: getattr(s, name) for name, _ in PdnStats._fields_ if not name.startswith("class_")}
        for key in ("class_ms", "class_bytes", "class_launches"):
            out[key] = {k: getattr(s, key)[i] for i, k in enumerate(KERNEL_CLASSES)}
        return out

    def port_matrix(self, tier: int) -> np.ndarray:
        q = self._lib.pdn_port_count(self._h, tier)
        out = np.empty((q, q))
        st = self._lib.pdn_get_port_matrix(self._h, tier, out.ctypes.data)
        if st != PDN_OK:
            raise PdnError(st, "pdn_get_port_matrix")
        return out

    def close(self):
        if getattr(self, "_h", None):
            self._lib.pdn_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
