"""paper_2301_04642_b200 -- B200-native recursive Fermi-operator expansion (RFOE, arXiv 2301.04642).

Thin Python binding over the C-ABI library ``librfoe.so`` (``include/rfoe.h``): argument marshalling
only -- every step of the path (Gershgorin bounds, affine map, symmetric squarings on the FP64 tensor
cores with the fused update / mirror / reductions, device-side branch decisions, output pass) runs in
the CUDA kernels under ``csrc/``.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: importing works anywhere, but any call without the built library or without
an sm_100 GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

__all__ = ["Rfoe", "RfoeError", "ExpandResult", "load_library", "shard_range", "torch_distributed_allgather", "gather_ipc_handles", "SP2", "MCWEENY", "SP2_MIXED", "SP2_ACCEL",
           "TRUNC", "TRUNC_MIXED", "RULE_A", "RULE_B", "EXPORTS", "bounds_static", "STATIC_MAX_K"]

SP2, MCWEENY, SP2_MIXED, SP2_ACCEL, TRUNC, TRUNC_MIXED = 0, 1, 2, 3, 4, 5
RULE_A, RULE_B = 0, 1
MAX_STEPS = 256

(OPT_STOP_RULE, OPT_MAX_ITER, OPT_EPS_MIN, OPT_EPS_MAX, OPT_CHECK_SYMMETRY, OPT_MIXED_HEAD, OPT_MIXED_RELTR,
 OPT_HOMO, OPT_LUMO, OPT_LANCZOS_STEPS, OPT_TRUNC_STEPS, OPT_RESIDENT, OPT_REDUCED_PAIR) = range(13)

(OK, ERR_INVALID_ARG, ERR_ALLOC, ERR_CUDA, ERR_BAD_BOUNDS, ERR_NOT_SYMMETRIC, ERR_UNSUPPORTED, ERR_NOT_CONVERGED,
 ERR_NO_PEER_ACCESS, ERR_STATIC_LIMIT) = range(10)
STATIC_MAX_K = 32768      # RFOE_STATIC_MAX_K

# every symbol include/rfoe.h declares
EXPORTS = ("rfoe_create", "rfoe_bounds", "rfoe_bounds_static", "rfoe_bounds_lanczos", "rfoe_expand", "rfoe_expand_host", "rfoe_square", "rfoe_square_reduced",
           "rfoe_symm_product", "rfoe_probe_fp64_peak", "rfoe_project", "rfoe_apply", "rfoe_expand_sharded", "rfoe_shard_range", "rfoe_plan_squaring", "rfoe_plan_resident",
           "rfoe_shard_local_ptrs", "rfoe_shard_set_peers", "rfoe_shard_ipc_export", "rfoe_shard_ipc_import",
           "rfoe_expand_sharded_p2p", "rfoe_expand_many",
           "rfoe_estimate_homo_lumo", "rfoe_set_option", "rfoe_get_stats", "rfoe_destroy", "rfoe_strerror", "rfoe_version")


# int allgather(void* user, const void* send, void* recv, int64_t bytes, stream)  -- see include/rfoe.h
ALLGATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)


# int barrier(void* user, stream)  -- see include/rfoe.h
BARRIER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p)
IPC_HANDLE_BYTES = 64


class RfoeError(RuntimeError):
    def __init__(self, status: int, msg: str, cuda_error: int = 0):
        super().__init__(f"librfoe: {msg} (status {status}" + (f", cudaError {cuda_error})" if cuda_error else ")"))
        self.status = status
        self.cuda_error = cuda_error


class _Stats(C.Structure):
    _fields_ = [
        ("status", C.c_int32), ("cuda_error", C.c_int32), ("variant", C.c_int32), ("stop_rule", C.c_int32),
        ("iterations", C.c_int32), ("multiplications", C.c_int32), ("mcweeny_steps", C.c_int32),
        ("fp32_steps", C.c_int32), ("converged", C.c_int32), ("square_launches", C.c_int32),
        ("trunc_steps", C.c_int32), ("resident", C.c_int32),
        ("k", C.c_int64), ("nocc", C.c_int64), ("gpu_launches", C.c_int64),
        ("tol", C.c_double), ("eps_min", C.c_double), ("eps_max", C.c_double), ("tr_PH", C.c_double),
        ("device_ms", C.c_double), ("square_ms", C.c_double), ("resident_phase_ms", C.c_double * 5),
        ("t", C.c_double * (MAX_STEPS + 1)), ("s", C.c_double * (MAX_STEPS + 1)),
        ("e", C.c_double * MAX_STEPS), ("reltr", C.c_double * MAX_STEPS),
        ("branch", C.c_char * (MAX_STEPS + 8)),
    ]


_lib = None


def load_library(path: str | None = None):
    """dlopen librfoe.so (building it first if the sources are newer) and declare the prototypes."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or _build.LIB
    if path is None and _build.stale():
        _build.build()
    if not os.path.exists(p):
        raise RfoeError(ERR_UNSUPPORTED, f"{p} is missing: run `python -m paper_2301_04642_b200.build`")
    L = C.CDLL(p)
    vp, i64, dbl, dp = C.c_void_p, C.c_int64, C.c_double, C.POINTER(C.c_double)
    L.rfoe_create.argtypes = [C.POINTER(vp), C.c_int, i64]
    L.rfoe_bounds.argtypes = [vp, vp, i64, dp, dp, vp]
    L.rfoe_bounds_static.argtypes = [vp, i64, vp, vp, C.POINTER(C.c_int)]
    L.rfoe_bounds_lanczos.argtypes = [vp, vp, i64, C.c_int, dp, dp, vp]
    L.rfoe_expand.argtypes = [vp, vp, i64, i64, C.c_int, dbl, vp, vp]
    L.rfoe_expand_host.argtypes = [vp, vp, i64, i64, C.c_int, dbl, vp, vp]
    L.rfoe_square.argtypes = [vp, vp, i64, dbl, dbl, dbl, vp, dp, C.POINTER(C.c_float), vp]
    L.rfoe_square_reduced.argtypes = [vp, vp, i64, dbl, dbl, dbl, vp, dp, C.POINTER(C.c_float), vp]
    L.rfoe_symm_product.argtypes = [vp, vp, vp, i64, dbl, dbl, dbl, vp, dp, C.POINTER(C.c_float), vp]
    L.rfoe_probe_fp64_peak.argtypes = [vp, dbl, dp, vp]
    L.rfoe_project.argtypes = [vp, vp, vp, i64, i64, i64, vp, dp, C.POINTER(C.c_float), vp]
    L.rfoe_apply.argtypes = [vp, vp, vp, i64, i64, i64, vp, i64, vp, C.POINTER(C.c_float), vp]
    L.rfoe_expand_sharded.argtypes = [vp, vp, i64, i64, C.c_int, dbl, vp, C.c_int, C.c_int, ALLGATHER_FN, vp, vp]
    L.rfoe_shard_local_ptrs.argtypes = [vp, C.POINTER(vp)]
    L.rfoe_shard_set_peers.argtypes = [vp, C.c_int, C.c_int, C.POINTER(vp)]
    L.rfoe_shard_ipc_export.argtypes = [vp, vp]
    L.rfoe_shard_ipc_import.argtypes = [vp, C.c_int, C.c_int, vp]
    L.rfoe_expand_sharded_p2p.argtypes = [vp, vp, i64, i64, C.c_int, dbl, vp, BARRIER_FN, vp, vp]
    L.rfoe_expand_many.argtypes = [C.POINTER(vp), C.POINTER(vp), C.c_int, C.c_int, C.POINTER(vp), C.POINTER(i64), C.POINTER(i64),
                                   C.c_int, dp, C.POINTER(vp), C.POINTER(C.c_int), C.POINTER(_Stats)]
    L.rfoe_plan_squaring.argtypes = [i64, C.c_int, C.POINTER(i64), C.POINTER(i64), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.rfoe_plan_resident.argtypes = [i64, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(i64),
                                     C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.rfoe_shard_range.argtypes = [i64, C.c_int, C.c_int, C.POINTER(i64), C.POINTER(i64)]
    L.rfoe_set_option.argtypes = [vp, C.c_int, dbl]
    L.rfoe_get_stats.argtypes = [vp, C.POINTER(_Stats)]
    L.rfoe_estimate_homo_lumo.argtypes = [C.POINTER(_Stats), dp, dp]
    L.rfoe_destroy.argtypes = [vp]
    L.rfoe_strerror.argtypes = [C.c_int]
    L.rfoe_strerror.restype = C.c_char_p
    L.rfoe_version.argtypes = []
    for name in EXPORTS:
        if name != "rfoe_strerror":
            getattr(L, name).restype = C.c_int
    if path is None:
        _lib = L
    return L


@dataclass
class ExpandResult:
    P: object              # torch tensor (device) or numpy array (host entry point)
    status: int
    converged: bool
    iterations: int
    multiplications: int
    mcweeny_steps: int
    fp32_steps: int
    branch: str
    eps_min: float
    eps_max: float
    tr_PH: float
    device_ms: float
    square_ms: float
    square_launches: int
    gpu_launches: int
    trunc_steps: int
    resident: bool
    resident_phase_ms: tuple
    t: np.ndarray
    s: np.ndarray
    e: np.ndarray
    reltr: np.ndarray


def _stream_ptr(stream):
    import torch

    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _check_dev(x, name):
    import torch

    if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float64 and x.dim() == 2
            and x.shape[0] == x.shape[1] and x.is_contiguous()):
        raise ValueError(f"{name}: contiguous square float64 CUDA tensor expected")


def _check_rect(x, name):
    import torch

    if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float64 and x.dim() == 2 and x.stride(1) == 1
            and x.stride(0) >= x.shape[1]):
        raise ValueError(f"{name}: row-major float64 CUDA matrix (k x M, unit column stride) expected")


def _result_from(st: _Stats, P, rc) -> "ExpandResult":
    n = st.iterations
    return ExpandResult(
        P=P, status=rc, converged=bool(st.converged), iterations=n, multiplications=st.multiplications,
        mcweeny_steps=st.mcweeny_steps, fp32_steps=st.fp32_steps, branch=st.branch.decode()[:n],
        eps_min=st.eps_min, eps_max=st.eps_max, tr_PH=st.tr_PH, device_ms=st.device_ms, square_ms=st.square_ms,
        square_launches=st.square_launches, gpu_launches=st.gpu_launches, trunc_steps=st.trunc_steps,
        resident=bool(st.resident), resident_phase_ms=tuple(st.resident_phase_ms), t=np.array(st.t[: n + 1]),
        s=np.array(st.s[: n + 1]), e=np.array(st.e[:n]), reltr=np.array(st.reltr[:n]))


def expand_many(handles, problems, variant: int = SP2, streams=None):
    """rfoe_expand_many: independent problems side by side on one GPU.  ``handles``: Rfoe objects (one host thread and
    one stream each, inside the library); ``problems``: list of (Hp, nocc, tol) or (Hp, nocc, tol, P) with CUDA tensors.
    Returns one ExpandResult per problem, in order; raises on any status other than OK / NOT_CONVERGED."""
    import torch

    L = load_library()
    nh, n = len(handles), len(problems)
    if streams is None:
        streams = [torch.cuda.Stream() for _ in handles]
    torch.cuda.current_stream().synchronize()              # every Hp complete before the call (rfoe.h)
    Ps = []
    for pr in problems:
        _check_dev(pr[0], "Hp")
        Ps.append(pr[3] if len(pr) > 3 and pr[3] is not None else torch.empty_like(pr[0]))
        _check_dev(Ps[-1], "P")
    vp = C.c_void_p
    hs = (vp * nh)(*[h._h.value for h in handles])
    ss = (vp * nh)(*[s.cuda_stream for s in streams])
    Hp = (vp * n)(*[pr[0].data_ptr() for pr in problems])
    Pp = (vp * n)(*[p.data_ptr() for p in Ps])
    ks = (C.c_int64 * n)(*[pr[0].shape[0] for pr in problems])
    no = (C.c_int64 * n)(*[int(pr[1]) for pr in problems])
    tl = (C.c_double * n)(*[float(pr[2]) for pr in problems])
    status = (C.c_int * n)()
    stats = (_Stats * n)()
    rc = L.rfoe_expand_many(hs, ss, nh, n, Hp, ks, no, int(variant), tl, Pp, status, stats)
    out = []
    for j in range(n):
        if status[j] not in (OK, ERR_NOT_CONVERGED):
            raise RfoeError(status[j], f"rfoe_expand_many, problem {j}: " + L.rfoe_strerror(status[j]).decode(),
                            stats[j].cuda_error)
        out.append(_result_from(stats[j], Ps[j], status[j]))
    if rc not in (OK, ERR_NOT_CONVERGED):
        raise RfoeError(rc, "rfoe_expand_many: " + L.rfoe_strerror(rc).decode())
    return out


def estimate_homo_lumo(stats: _Stats):
    """rfoe_estimate_homo_lumo on a raw stats structure (host only, no device needed)."""
    L = load_library()
    ho, lu = C.c_double(), C.c_double()
    rc = L.rfoe_estimate_homo_lumo(C.byref(stats), C.byref(ho), C.byref(lu))
    if rc != OK:
        raise RfoeError(rc, "rfoe_estimate_homo_lumo: " + L.rfoe_strerror(rc).decode())
    return ho.value, lu.value


def bounds_static(Hp, out, stream=None):
    """rfoe_bounds_static: Gershgorin bounds with no handle and no allocation anywhere below this call (scratch in a fixed
    device array, k <= STATIC_MAX_K).  `out`: float64 CUDA tensor of >= 2 elements on Hp's device, receives
    (eps_min, eps_max).  Asynchronous on `stream`; calls that overlap on one GPU race on the shared scratch."""
    import torch

    _check_dev(Hp, "Hp")
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.is_contiguous()
            and out.numel() >= 2 and out.device == Hp.device):
        raise ValueError("out: contiguous float64 CUDA tensor of >= 2 elements on Hp's device expected")
    L = load_library()
    err = C.c_int(0)
    with torch.cuda.device(Hp.device):
        rc = L.rfoe_bounds_static(C.c_void_p(Hp.data_ptr()), Hp.shape[0], C.c_void_p(out.data_ptr()), _stream_ptr(stream), C.byref(err))
    if rc != OK:
        raise RfoeError(rc, "rfoe_bounds_static: " + L.rfoe_strerror(rc).decode(), err.value)
    return out


def plan_squaring(k: int, sm_count: int = 148):
    """(n_tiles, n_main, slices, kt_per_slice): how one squaring at size k is launched (host-only C call)."""
    nt, nm, sl, per = C.c_int64(), C.c_int64(), C.c_int(), C.c_int()
    rc = load_library().rfoe_plan_squaring(int(k), int(sm_count), C.byref(nt), C.byref(nm), C.byref(sl), C.byref(per))
    if rc != OK:
        raise RfoeError(rc, "rfoe_plan_squaring: invalid argument")
    return nt.value, nm.value, sl.value, per.value


def plan_resident(k: int, sm_count: int = 148):
    """rfoe_plan_resident (host-only C call): dict(path, grid, kt, n_tiles, n_split, boundaries, split_tiles)."""
    path, grid, kt, ns = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    nt = C.c_int64()
    bounds = (C.c_int * (sm_count + 2))()
    split = (C.c_int * (3 * sm_count + 6))()
    rc = load_library().rfoe_plan_resident(int(k), int(sm_count), C.byref(path), C.byref(grid), C.byref(kt), C.byref(nt), C.byref(ns),
                                           bounds, split)
    if rc != OK:
        raise RfoeError(rc, "rfoe_plan_resident: invalid argument")
    g = grid.value
    return dict(path=path.value, grid=g, kt=kt.value, n_tiles=nt.value, n_split=ns.value,
                boundaries=list(bounds[: g + 1]) if path.value == 3 else [],
                split_tiles=[tuple(split[3 * i: 3 * i + 3]) for i in range(ns.value)] if path.value == 3 else [])


def shard_range(n_tiles: int, rank: int, world: int):
    """(begin, count) of the upper-triangle tile range `rank` of `world` squares (host-only C call)."""
    b, c = C.c_int64(), C.c_int64()
    rc = load_library().rfoe_shard_range(int(n_tiles), int(rank), int(world), C.byref(b), C.byref(c))
    if rc != OK:
        raise RfoeError(rc, "rfoe_shard_range: invalid argument")
    return b.value, c.value


def gather_ipc_handles(mine: bytes, group=None) -> bytes:
    """The layout rfoe_shard_ipc_import expects: every rank's 4 x 64-byte CUDA IPC handles (W0, W1, records of even /
    odd steps), concatenated in RANK order.  Any torch.distributed backend (the handles are host bytes)."""
    import torch.distributed as dist

    if len(mine) != 4 * IPC_HANDLE_BYTES:
        raise ValueError("4 x 64 bytes of IPC handles expected")
    world = dist.get_world_size(group)
    gathered = [None] * world
    dist.all_gather_object(gathered, bytes(mine), group=group)
    out = b"".join(gathered)
    assert len(out) == 4 * IPC_HANDLE_BYTES * world
    return out


class _DevBytes:
    """A raw device range as a __cuda_array_interface__ object (so torch can wrap it without copying)."""

    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False), "version": 2}


def torch_distributed_allgather(group=None):
    """The exchange step of rfoe_expand_sharded through torch.distributed (NCCL over NVLink): an all-gather of the
    library's send buffer into its receive buffer, issued under the library's stream."""
    import torch
    import torch.distributed as dist

    def allgather(send_ptr: int, recv_ptr: int, nbytes: int, stream_ptr) -> int:
        world = dist.get_world_size(group)
        ext = torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.default_stream()
        with torch.cuda.stream(ext):
            send = torch.as_tensor(_DevBytes(send_ptr, nbytes), device="cuda")
            recv = torch.as_tensor(_DevBytes(recv_ptr, nbytes * world), device="cuda")
            dist.all_gather_into_tensor(recv, send, group=group)
        return 0

    return allgather


class Rfoe:
    """One librfoe handle (same names as the C ABI: bounds / expand / expand_host / square / symm_product)."""

    def __init__(self, k_max: int, device: int = 0):
        self._L = load_library()
        self._h = C.c_void_p()
        self.k_max = int(k_max)
        self.device = int(device)
        rc = self._L.rfoe_create(C.byref(self._h), self.device, self.k_max)
        if rc != OK:
            self._h = C.c_void_p()
            raise RfoeError(rc, self._L.rfoe_strerror(rc).decode())

    def close(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value:
            self._h = None
            self._L.rfoe_destroy(h)

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- helpers
    def _raise(self, rc):
        st = self.stats_raw()
        raise RfoeError(rc, self._L.rfoe_strerror(rc).decode(), st.cuda_error)

    def stats_raw(self) -> _Stats:
        st = _Stats()
        self._L.rfoe_get_stats(self._h, C.byref(st))
        return st

    def estimate_homo_lumo(self):
        """(homo, lumo) estimates from the history of the last plain SP2 run of this handle (rfoe_estimate_homo_lumo)."""
        return estimate_homo_lumo(self.stats_raw())

    def set_option(self, key: int, value: float):
        rc = self._L.rfoe_set_option(self._h, key, float(value))
        if rc != OK:
            raise RfoeError(rc, self._L.rfoe_strerror(rc).decode())

    def configure(self, *, stop_rule=None, max_iter=None, bounds=None, check_symmetry=None, mixed_head=None,
                  mixed_reltr=None, homo=None, lumo=None, lanczos_steps=None, trunc_steps=None, resident=None, reduced_pair=None):
        if lanczos_steps is not None: self.set_option(OPT_LANCZOS_STEPS, lanczos_steps)
        if trunc_steps is not None: self.set_option(OPT_TRUNC_STEPS, trunc_steps)
        if resident is not None: self.set_option(OPT_RESIDENT, float(int(resident)))      # True / False, or 2: band form only (rfoe.h)
        if reduced_pair is not None: self.set_option(OPT_REDUCED_PAIR, 1.0 if reduced_pair else 0.0)
        if stop_rule is not None: self.set_option(OPT_STOP_RULE, stop_rule)
        if max_iter is not None: self.set_option(OPT_MAX_ITER, max_iter)
        if bounds is not None:
            lo, hi = (float("nan"), float("nan")) if bounds is False else bounds
            self.set_option(OPT_EPS_MIN, lo)
            self.set_option(OPT_EPS_MAX, hi)
        if check_symmetry is not None: self.set_option(OPT_CHECK_SYMMETRY, 1.0 if check_symmetry else 0.0)
        if mixed_head is not None: self.set_option(OPT_MIXED_HEAD, mixed_head)
        if mixed_reltr is not None: self.set_option(OPT_MIXED_RELTR, mixed_reltr)
        if homo is not None: self.set_option(OPT_HOMO, homo)
        if lumo is not None: self.set_option(OPT_LUMO, lumo)
        return self

    def _result(self, P, rc) -> ExpandResult:
        return _result_from(self.stats_raw(), P, rc)

    # ---- the C-ABI calls
    def bounds(self, Hp, stream=None):
        _check_dev(Hp, "Hp")
        lo, hi = C.c_double(), C.c_double()
        rc = self._L.rfoe_bounds(self._h, C.c_void_p(Hp.data_ptr()), Hp.shape[0], C.byref(lo), C.byref(hi), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return lo.value, hi.value

    def bounds_lanczos(self, Hp, m: int = 24, stream=None):
        """m-step Lanczos spectral bounds (theta_min - beta_m, theta_max + beta_m)."""
        _check_dev(Hp, "Hp")
        lo, hi = C.c_double(), C.c_double()
        rc = self._L.rfoe_bounds_lanczos(self._h, C.c_void_p(Hp.data_ptr()), Hp.shape[0], int(m), C.byref(lo), C.byref(hi),
                                         _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return lo.value, hi.value

    def expand(self, Hp, nocc: int, variant: int = SP2, tol: float = 1e-12, P=None, stream=None) -> ExpandResult:
        import torch

        _check_dev(Hp, "Hp")
        if P is None:
            P = torch.empty_like(Hp)
        _check_dev(P, "P")
        rc = self._L.rfoe_expand(self._h, C.c_void_p(Hp.data_ptr()), Hp.shape[0], int(nocc), int(variant), float(tol),
                                 C.c_void_p(P.data_ptr()), _stream_ptr(stream))
        if rc not in (OK, ERR_NOT_CONVERGED):
            self._raise(rc)
        return self._result(P, rc)

    def expand_host(self, Hp: np.ndarray, nocc: int, variant: int = SP2, tol: float = 1e-12, P=None, stream=None) -> ExpandResult:
        """Host buffers in, host buffers out (numpy arrays or pinned CPU torch tensors)."""
        def ptr(a):
            return a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr()
        k = Hp.shape[0]
        if P is None:
            P = np.empty((k, k), dtype=np.float64)
        rc = self._L.rfoe_expand_host(self._h, C.c_void_p(ptr(Hp)), k, int(nocc), int(variant), float(tol),
                                      C.c_void_p(ptr(P)), _stream_ptr(stream))
        if rc not in (OK, ERR_NOT_CONVERGED):
            self._raise(rc)
        return self._result(P, rc)

    def square(self, X, c2=1.0, c1=0.0, c0=0.0, out=None, stream=None, reduced=False):
        """out = c2 X X + c1 X + c0 I; returns (out, scalars[5], kernel_ms).  reduced=True: rfoe_square_reduced."""
        import torch

        _check_dev(X, "X")
        out = torch.empty_like(X) if out is None else out
        sc = (C.c_double * 5)()
        ms = C.c_float()
        fn = self._L.rfoe_square_reduced if reduced else self._L.rfoe_square
        rc = fn(self._h, C.c_void_p(X.data_ptr()), X.shape[0], c2, c1, c0, C.c_void_p(out.data_ptr()),
                                 sc, C.byref(ms), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return out, np.array(sc[:]), ms.value

    def probe_fp64_peak(self, ms: float = 200.0, stream=None) -> float:
        """rfoe_probe_fp64_peak: TFLOP/s of a register-only DMMA.8x8x4 issue loop on every SM for about ``ms`` ms."""
        tf = C.c_double()
        rc = self._L.rfoe_probe_fp64_peak(self._h, float(ms), C.byref(tf), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return tf.value

    def symm_product(self, A, B, c2=1.0, c1=0.0, c0=0.0, out=None, stream=None):
        """out = c2 A B + c1 A + c0 I (upper triangle mirrored); returns (out, scalars[5], kernel_ms)."""
        import torch

        _check_dev(A, "A")
        _check_dev(B, "B")
        out = torch.empty_like(A) if out is None else out
        sc = (C.c_double * 5)()
        ms = C.c_float()
        rc = self._L.rfoe_symm_product(self._h, C.c_void_p(A.data_ptr()), C.c_void_p(B.data_ptr()), A.shape[0], c2, c1, c0,
                                       C.c_void_p(out.data_ptr()), sc, C.byref(ms), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return out, np.array(sc[:]), ms.value

    def project(self, Psi, HPsi, out=None, stream=None):
        """Rayleigh-Ritz step: Hp = Psi HPsi^T (upper triangle mirrored); returns (Hp, (Tr Hp, ||Hp||_F^2), kernel_ms)."""
        import torch

        _check_rect(Psi, "Psi")
        _check_rect(HPsi, "HPsi")
        if HPsi.shape != Psi.shape or HPsi.stride(0) != Psi.stride(0):
            raise ValueError("Psi and HPsi must have the same shape and row pitch")
        k, M = Psi.shape
        out = torch.empty((k, k), dtype=torch.float64, device=Psi.device) if out is None else out
        _check_dev(out, "Hp")
        sc = (C.c_double * 2)()
        ms = C.c_float()
        rc = self._L.rfoe_project(self._h, C.c_void_p(Psi.data_ptr()), C.c_void_p(HPsi.data_ptr()), k, M, Psi.stride(0),
                                  C.c_void_p(out.data_ptr()), sc, C.byref(ms), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return out, (sc[0], sc[1]), ms.value

    def apply(self, P, Psi, out=None, density=True, stream=None):
        """Y = P Psi and (density=True) rho_m = sum_i Psi_im Y_im; returns (Y, rho or None, kernel_ms)."""
        import torch

        _check_dev(P, "P")
        _check_rect(Psi, "Psi")
        k, M = Psi.shape
        if P.shape[0] != k:
            raise ValueError("P must be k x k with k = Psi.shape[0]")
        out = torch.empty((k, M), dtype=torch.float64, device=Psi.device) if out is None else out
        _check_rect(out, "Y")
        rho = torch.empty((M,), dtype=torch.float64, device=Psi.device) if density else None
        ms = C.c_float()
        rc = self._L.rfoe_apply(self._h, C.c_void_p(P.data_ptr()), C.c_void_p(Psi.data_ptr()), k, M, Psi.stride(0),
                                C.c_void_p(out.data_ptr()), out.stride(0), C.c_void_p(rho.data_ptr() if density else None),
                                C.byref(ms), _stream_ptr(stream))
        if rc != OK:
            self._raise(rc)
        return out, rho, ms.value

    def expand_sharded(self, Hp, nocc: int, variant: int = SP2, tol: float = 1e-12, P=None, *, rank: int, world: int,
                       allgather=None, stream=None) -> ExpandResult:
        """One expansion sharded over `world` ranks (one process per GPU); every rank passes the same H^p and gets
        the whole P.  `allgather(send_ptr, recv_ptr, nbytes, stream_ptr) -> int` performs the exchange step; the
        default is torch.distributed's all_gather_into_tensor on the default process group."""
        import torch

        _check_dev(Hp, "Hp")
        if P is None:
            P = torch.empty_like(Hp)
        _check_dev(P, "P")
        fn = allgather if allgather is not None else torch_distributed_allgather()
        err = []

        def _cb(user, send, recv, nbytes, stream_ptr):
            try:
                return int(fn(send, recv, nbytes, stream_ptr))
            except BaseException as e:  # an exception must not unwind through the C frames
                err.append(e)
                return 1

        cb = ALLGATHER_FN(_cb)
        rc = self._L.rfoe_expand_sharded(self._h, C.c_void_p(Hp.data_ptr()), Hp.shape[0], int(nocc), int(variant), float(tol),
                                         C.c_void_p(P.data_ptr()), int(rank), int(world), cb, None, _stream_ptr(stream))
        if err:
            raise err[0]
        if rc not in (OK, ERR_NOT_CONVERGED):
            self._raise(rc)
        return self._result(P, rc)

    # ---- sharded expansion with the exchange fused into the squaring kernel (peer memory)
    def shard_local_ptrs(self):
        """The four device pointers (work matrices W0, W1, tile records of even / odd steps) peers must be able to write."""
        out = (C.c_void_p * 4)()
        rc = self._L.rfoe_shard_local_ptrs(self._h, out)
        if rc != OK:
            self._raise(rc)
        return [int(p) for p in out]

    def shard_set_peers(self, rank: int, world: int, ptrs):
        """ptrs: 4 * world device pointers, rank d's four at [4 d, 4 d + 4) (same process; P2P enabled by the caller)."""
        arr = (C.c_void_p * (4 * world))(*[C.c_void_p(int(p)) for p in ptrs])
        rc = self._L.rfoe_shard_set_peers(self._h, int(rank), int(world), arr)
        if rc != OK:
            self._raise(rc)

    def shard_ipc_export(self) -> bytes:
        buf = C.create_string_buffer(4 * IPC_HANDLE_BYTES)
        rc = self._L.rfoe_shard_ipc_export(self._h, buf)
        if rc != OK:
            self._raise(rc)
        return buf.raw

    def shard_ipc_import(self, rank: int, world: int, handles: bytes):
        assert len(handles) == 4 * IPC_HANDLE_BYTES * world
        rc = self._L.rfoe_shard_ipc_import(self._h, int(rank), int(world), C.create_string_buffer(handles, len(handles)))
        if rc != OK:
            self._raise(rc)

    def shard_connect(self, group=None):
        """One process per GPU: exchange CUDA IPC handles of the work buffers over torch.distributed and map the peers.
        Raises RfoeError(ERR_NO_PEER_ACCESS) when a peer's buffers cannot be reached (fall back to expand_sharded)."""
        import torch.distributed as dist

        world, rank = dist.get_world_size(group), dist.get_rank(group)
        self.shard_ipc_import(rank, world, gather_ipc_handles(self.shard_ipc_export(), group))
        return rank, world

    def expand_sharded_p2p(self, Hp, nocc: int, variant: int = SP2, tol: float = 1e-12, P=None, *, barrier=None,
                           stream=None) -> ExpandResult:
        """rfoe_expand_sharded_p2p after shard_set_peers / shard_connect.  `barrier(stream_ptr) -> int` must return once
        every rank's enqueued work has completed; default: stream synchronize + torch.distributed.barrier()."""
        import torch

        _check_dev(Hp, "Hp")
        if P is None:
            P = torch.empty_like(Hp)
        _check_dev(P, "P")
        if barrier is None:
            import torch.distributed as dist

            def barrier(stream_ptr):
                (torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.default_stream()).synchronize()
                dist.barrier()
                return 0
        err = []

        def _cb(user, stream_ptr):
            try:
                return int(barrier(stream_ptr))
            except BaseException as e:  # an exception must not unwind through the C frames
                err.append(e)
                return 1

        cb = BARRIER_FN(_cb)
        rc = self._L.rfoe_expand_sharded_p2p(self._h, C.c_void_p(Hp.data_ptr()), Hp.shape[0], int(nocc), int(variant), float(tol),
                                             C.c_void_p(P.data_ptr()), cb, None, _stream_ptr(stream))
        if err:
            raise err[0]
        if rc not in (OK, ERR_NOT_CONVERGED):
            self._raise(rc)
        return self._result(P, rc)
