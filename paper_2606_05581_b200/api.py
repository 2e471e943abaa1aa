"""Thin ctypes binding of include/mcdtn.h: argument marshalling only.

Every step of the path runs in the CUDA library (libmcdtn.so, built in-tree by
paper_2606_05581_b200/build.py).  PyTorch supplies device memory and streams,
nothing else.  There is no CPU fallback: loading fails loudly if the library is
missing, and every call raises McsError on a non-zero return code.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("MCDTN_LIB") or os.path.join(HERE, "libmcdtn.so")     # MCDTN_LIB: another build of the same library

MCS_OK, MCS_EINVAL, MCS_EDEGENERATE, MCS_ENOMEM, MCS_ECUDA = 0, -1, -2, -3, -4
MCS_WNOTCONVERGED = 1


class McsError(RuntimeError):
    def __init__(self, code: int, where: str, msg: str):
        super().__init__(f"{where}: {msg} (code {code})")
        self.code = code


class _BuildOpts(C.Structure):
    _fields_ = [("no_split", C.c_int32), ("max_pieces", C.c_int32), ("split_length", C.c_float), ("split_budget", C.c_float)]


class BvhInfo(C.Structure):
    _fields_ = [("V", C.c_int64), ("F", C.c_int64), ("n_nodes", C.c_int64), ("max_depth", C.c_int32),
                ("n_degenerate", C.c_int32), ("aabb_lo", C.c_float * 3), ("aabb_hi", C.c_float * 3),
                ("area", C.c_double), ("device_bytes", C.c_size_t), ("n_leaves", C.c_int64), ("sah_cost", C.c_double)]


class _Samples(C.Structure):
    _fields_ = [("tri", C.c_void_p), ("bary", C.c_void_p), ("weight", C.c_void_p), ("normal", C.c_void_p),
                ("n_s", C.c_int64)]


class _Basis(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad_", C.c_int32), ("K", C.c_int64), ("points", C.c_void_p),
                ("normals", C.c_void_p), ("k", C.c_int32), ("sigma", C.c_float), ("tau_n", C.c_float),
                ("pad2_", C.c_int32)]


class _Params(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("walks_per_sample", C.c_int32), ("max_steps", C.c_int32),
                ("eps", C.c_float), ("cap_half_angle_deg", C.c_float), ("rmax_scale", C.c_float),
                ("rmax_override", C.c_float), ("bisection_iters", C.c_int32), ("importance_sample", C.c_int32),
                ("antithetic", C.c_int32), ("include_killing", C.c_int32), ("n_kill_walks", C.c_int64),
                ("kelvin_origin", C.c_float * 3), ("output_kind", C.c_int32), ("coo_capacity", C.c_int64),
                ("estimator", C.c_int32), ("inset", C.c_float), ("far_alpha", C.c_float), ("far_near_factor", C.c_float),
                ("exterior_query", C.c_int32), ("nonblocking", C.c_int32)]


class _Matrix(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad_", C.c_int32), ("K", C.c_int64), ("dense", C.c_void_p),
                ("coo_capacity", C.c_int64), ("coo_row", C.c_void_p), ("coo_col", C.c_void_p), ("coo_val", C.c_void_p),
                ("coo_nnz", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [("n_samples", C.c_int64), ("n_discarded", C.c_int64), ("n_walks", C.c_int64),
                ("n_truncated", C.c_int64), ("n_steps", C.c_int64), ("n_queries", C.c_int64),
                ("n_nodes_visited", C.c_int64), ("n_tris_tested", C.c_int64), ("n_prep_queries", C.c_int64),
                ("n_prep_nodes", C.c_int64), ("n_prep_tris", C.c_int64), ("n_entries", C.c_int64),
                ("n_unique", C.c_int64), ("workspace_needed", C.c_int64), ("n_far_queries", C.c_int64), ("nodes_hist", C.c_int64 * 16),
                ("cuda_error", C.c_int32),
                ("pad_", C.c_int32)]

    def as_dict(self):
        return {k: (list(getattr(self, k)) if k == "nodes_hist" else getattr(self, k)) for k, _ in self._fields_ if k != "pad_"}


_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built: no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_05581_b200.build` "
                              "(there is no CPU or PyTorch fallback for this path)")
        L = C.CDLL(LIB_PATH)
        L.mcs_error_string.restype = C.c_char_p
        L.mcs_version.restype = C.c_char_p
        for name in ("mcs_workspace_bytes", "mcs_walk_workspace_bytes", "mcs_accumulate_workspace_bytes",
                     "mcs_sort_workspace_bytes"):
            getattr(L, name).restype = C.c_size_t
        L.mcs_free_bvh.restype = None
        _lib = L
    return _lib


def _check(rc: int, where: str):
    if rc != MCS_OK:
        raise McsError(rc, where, lib().mcs_error_string(rc).decode())


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _stream(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _dev(t, dtype, name):
    if not isinstance(t, torch.Tensor):
        t = torch.as_tensor(t)
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (this path has no CPU implementation)")
    return t.to(dtype).contiguous()


@dataclass
class Params:
    seed: int = 0
    walks_per_sample: int = 1
    max_steps: int = 4096
    eps: float = 1e-3
    cap_half_angle_deg: float = 2.5
    rmax_scale: float = 1.0
    rmax_override: float = 0.0
    bisection_iters: int = 10
    importance_sample: bool = True
    antithetic: bool = False
    include_killing: bool = False
    n_kill_walks: int = 0
    kelvin_origin: tuple = (0.0, 0.0, 0.0)
    output_kind: int = 0                 # 0 dense, 1 sparse COO (upper triangle)
    coo_capacity: int = 0
    estimator: int = 0                   # 0: Alg. 2; 1: Alg. 1 (naive finite difference, interior only)
    inset: float = 0.0                   # Alg. 1: walks start at s - inset * n_s
    far_alpha: float = 0.0               # > 0: far-field queries return a lower bound of the distance (mcs_params.far_alpha)
    far_near_factor: float = 0.0         # boxes closer than this many eps are always descended (0: 16)
    exterior_query: int = 0              # exterior: 0 conservative radius on flat faces (E3); 1 exact inverted faces (E4)

    def c(self) -> _Params:
        p = _Params(seed=self.seed, walks_per_sample=self.walks_per_sample, max_steps=self.max_steps,
                    eps=self.eps, cap_half_angle_deg=self.cap_half_angle_deg, rmax_scale=self.rmax_scale,
                    rmax_override=self.rmax_override, bisection_iters=self.bisection_iters,
                    importance_sample=int(self.importance_sample), antithetic=int(self.antithetic),
                    include_killing=int(self.include_killing), n_kill_walks=int(self.n_kill_walks),
                    output_kind=int(self.output_kind), coo_capacity=int(self.coo_capacity),
                    estimator=int(self.estimator), inset=float(self.inset), far_alpha=float(self.far_alpha),
                    far_near_factor=float(self.far_near_factor), exterior_query=int(self.exterior_query))
        p.kelvin_origin[:] = [float(x) for x in self.kelvin_origin]
        return p


@dataclass
class Samples:
    """Boundary samples on the device."""
    tri: torch.Tensor
    bary: torch.Tensor
    weight: torch.Tensor
    normal: torch.Tensor | None = None
    _keep: list = field(default_factory=list, repr=False)

    @classmethod
    def from_arrays(cls, tri, bary, weight, normal=None, device="cuda"):
        tri = torch.as_tensor(tri).to(device=device, dtype=torch.int32).contiguous()
        bary = torch.as_tensor(bary).to(device=device, dtype=torch.float32).contiguous()
        weight = torch.as_tensor(weight).to(device=device, dtype=torch.float32).contiguous()
        if normal is not None:
            normal = torch.as_tensor(normal).to(device=device, dtype=torch.float32).contiguous()
        return cls(tri, bary, weight, normal)

    @property
    def n_s(self):
        return int(self.tri.shape[0])

    def c(self) -> _Samples:
        assert self.bary.shape == (self.n_s, 3) and self.weight.shape == (self.n_s,)
        return _Samples(tri=self.tri.data_ptr(), bary=self.bary.data_ptr(), weight=self.weight.data_ptr(),
                        normal=self.normal.data_ptr() if self.normal is not None else None, n_s=self.n_s)


class Bvh:
    """Opaque LBVH handle (mcs_build_bvh / mcs_free_bvh)."""

    def __init__(self, verts, faces, split=True, max_pieces=0, split_length=0.0, split_budget=0.0):
        self.verts = _dev(verts, torch.float32, "verts")
        self.faces = _dev(faces, torch.int32, "faces")
        if self.verts.ndim != 2 or self.verts.shape[1] != 3 or self.faces.ndim != 2 or self.faces.shape[1] != 3:
            raise ValueError("verts must be [V,3], faces [F,3]")
        self.device = self.verts.device
        self._h = C.c_void_p(0)
        with torch.cuda.device(self.device):
            opts = _BuildOpts(no_split=int(not split), max_pieces=int(max_pieces), split_length=float(split_length),
                              split_budget=float(split_budget))
            rc = lib().mcs_build_bvh(_ptr(self.verts), C.c_int64(self.verts.shape[0]), _ptr(self.faces),
                                     C.c_int64(self.faces.shape[0]), C.byref(opts), _stream(self.device), C.byref(self._h))
        _check(rc, "mcs_build_bvh")

    def __del__(self):
        h = getattr(self, "_h", None)
        if h is not None and h.value and _lib is not None:       # _lib is None at interpreter shutdown
            _lib.mcs_free_bvh(h)
            self._h = C.c_void_p(0)

    @property
    def handle(self):
        return self._h

    @property
    def V(self):
        return int(self.verts.shape[0])

    @property
    def F(self):
        return int(self.faces.shape[0])

    def info(self) -> BvhInfo:
        o = BvhInfo()
        _check(lib().mcs_bvh_info(self._h, C.byref(o)), "mcs_bvh_info")
        return o

    def dump(self):
        info = self.info()
        nodes = torch.empty((info.n_nodes, 16), dtype=torch.int32, device=self.device)
        leaf_tri = torch.empty(info.n_leaves, dtype=torch.int32, device=self.device)
        morton = torch.empty(info.n_leaves, dtype=torch.int64, device=self.device)
        with torch.cuda.device(self.device):
            _check(lib().mcs_bvh_dump(self._h, _ptr(nodes), _ptr(leaf_tri), _ptr(morton), _stream(self.device)),
                   "mcs_bvh_dump")
        return nodes, leaf_tri, morton


def build_bvh(verts, faces, split=True, max_pieces=0, split_length=0.0, split_budget=0.0) -> Bvh:
    """LBVH over the triangle soup (mcs_build_bvh).  split: long thin faces enter the tree as several leaf references
    (mcs_build_opts); the query results do not depend on it."""
    return Bvh(verts, faces, split, max_pieces, split_length, split_budget)


def _closest(fn, name, bvh: Bvh, q):
    q = _dev(q, torch.float32, "q")
    n = q.shape[0]
    dist = torch.empty(n, dtype=torch.float32, device=bvh.device)
    tri = torch.empty(n, dtype=torch.int32, device=bvh.device)
    bary = torch.empty((n, 3), dtype=torch.float32, device=bvh.device)
    with torch.cuda.device(bvh.device):
        _check(fn(bvh.handle, _ptr(q), C.c_int64(n), _ptr(dist), _ptr(tri), _ptr(bary), _stream(bvh.device)), name)
    return dist, tri, bary


def closest_point(bvh: Bvh, q):
    return _closest(lib().mcs_closest_point, "mcs_closest_point", bvh, q)


def closest_point_bruteforce(bvh: Bvh, q):
    return _closest(lib().mcs_closest_point_bruteforce, "mcs_closest_point_bruteforce", bvh, q)


@dataclass
class PointBasis:
    """Point-based function space (mcs_basis.kind 1; App. B): device tensors points [K,3], unit normals
    [K,3]; k neighbours, sigma, tau_n."""
    points: torch.Tensor
    normals: torch.Tensor
    k: int = 8
    sigma: float = 0.025
    tau_n: float = 0.8

    @classmethod
    def from_arrays(cls, points, normals, k=8, sigma=0.025, tau_n=0.8, device="cuda"):
        p = torch.as_tensor(points).to(device=device, dtype=torch.float32).contiguous()
        n = torch.as_tensor(normals).to(device=device, dtype=torch.float32).contiguous()
        return cls(p, n, k, sigma, tau_n)

    @property
    def K(self):
        return int(self.points.shape[0])

    def c(self) -> _Basis:
        assert self.points.is_cuda and self.normals.is_cuda and self.points.shape == self.normals.shape
        return _Basis(kind=1, K=self.K, points=self.points.data_ptr(), normals=self.normals.data_ptr(), k=int(self.k),
                      sigma=float(self.sigma), tau_n=float(self.tau_n))


def _basis(bvh: Bvh, basis=None) -> _Basis:
    return basis.c() if basis is not None else _Basis(kind=0, K=bvh.V)


def knn_weights(basis: PointBasis, q, nq):
    """(idx [Q,k] int32, w [Q,k] fp32) of the k-NN bilateral interpolator (mcs_knn_weights)."""
    q, nq = _dev(q, torch.float32, "q"), _dev(nq, torch.float32, "nq")
    Q = int(q.shape[0])
    idx = torch.empty((Q, basis.k), dtype=torch.int32, device=q.device)
    w = torch.empty((Q, basis.k), dtype=torch.float32, device=q.device)
    cb = basis.c()
    with torch.cuda.device(q.device):
        _check(lib().mcs_knn_weights(C.byref(cb), _ptr(q), _ptr(nq), C.c_int64(Q), _ptr(idx), _ptr(w), _stream(q.device)),
               "mcs_knn_weights")
    return idx, w


def workspace_bytes(bvh: Bvh, samples: Samples, params: Params, exterior: bool, basis=None) -> int:
    cs, cb, cp = samples.c(), _basis(bvh, basis), params.c()
    return int(lib().mcs_workspace_bytes(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), C.c_int(int(exterior))))


def _estimate(fn, name, bvh, samples, params, exterior, want_stats, out, workspace, _exact_workspace=False, basis=None,
              nonblocking=False):
    cs, cb, cp = samples.c(), _basis(bvh, basis), params.c()
    K = basis.K if basis is not None else bvh.V
    if nonblocking:
        # mcs_params.nonblocking: the library only enqueues work (no read-back, no allocation), so the call may sit in
        # a CUDA graph.  The caller owns `out` and `workspace` for as long as the work may run.
        if want_stats or basis is not None or out is None or workspace is None:
            raise ValueError("nonblocking=True needs out= and workspace= from the caller, the hat basis and want_stats=False")
        if workspace.numel() < workspace_bytes(bvh, samples, params, exterior, basis):
            raise ValueError("workspace too small")
    if out is None:
        out = torch.empty((K, K), dtype=torch.float32, device=bvh.device)
    elif not (isinstance(out, torch.Tensor) and out.is_cuda and out.device == bvh.device and out.dtype == torch.float32
              and out.is_contiguous() and tuple(out.shape) == (K, K)):
        raise ValueError(f"out must be a contiguous CUDA float32 tensor of shape ({K}, {K}) on {bvh.device}")
    if workspace is not None and not (isinstance(workspace, torch.Tensor) and workspace.is_cuda and workspace.device == bvh.device
                                      and workspace.dtype == torch.uint8 and workspace.is_contiguous()):
        raise ValueError(f"workspace must be a contiguous CUDA uint8 tensor on {bvh.device}")
    need = workspace_bytes(bvh, samples, params, exterior, basis)
    if workspace is None or (workspace.numel() < need and not _exact_workspace):
        workspace = torch.empty(need, dtype=torch.uint8, device=bvh.device)
    m = _Matrix(kind=0, K=K, dense=out.data_ptr())
    st = Stats() if want_stats else None
    cp.nonblocking = 1 if nonblocking else 0
    with torch.cuda.device(bvh.device):
        rc = fn(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), _ptr(workspace), C.c_size_t(workspace.numel()),
                C.byref(m), C.byref(st) if st is not None else None, _stream(bvh.device))
    _check(rc, name)
    return (out, st) if want_stats else out


def estimate_dtn_interior(bvh: Bvh, samples: Samples, params: Params, want_stats=False, out=None, workspace=None,
                          _exact_workspace=False, basis=None, nonblocking=False):
    """Interior DtN matrix, Alg. 2: dense [K,K] fp32 on the device (K = V, or the number of
    points of a PointBasis).  nonblocking=True (hat basis, caller's out and workspace): only enqueues work on the
    current stream -- capturable in a CUDA graph; input errors only the device can see then turn the output into NaN."""
    return _estimate(lib().mcs_estimate_dtn_interior, "mcs_estimate_dtn_interior", bvh, samples, params, False,
                     want_stats, out, workspace, _exact_workspace, basis, nonblocking)


def estimate_dtn_exterior(bvh: Bvh, samples: Samples, params: Params, want_stats=False, out=None, workspace=None,
                          _exact_workspace=False, basis=None, nonblocking=False):
    """Exterior DtN matrix, Eq. 32.  nonblocking: see estimate_dtn_interior."""
    return _estimate(lib().mcs_estimate_dtn_exterior, "mcs_estimate_dtn_exterior", bvh, samples, params, True,
                     want_stats, out, workspace, _exact_workspace, basis, nonblocking)


def workspace_bytes_both(bvh: Bvh, samples: Samples, params_interior: Params, params_exterior: Params, basis=None) -> int:
    cs, cb = samples.c(), _basis(bvh, basis)
    ci, ce = params_interior.c(), params_exterior.c()
    fn = lib().mcs_workspace_bytes_both
    fn.restype = C.c_size_t
    return int(fn(bvh.handle, C.byref(cs), C.byref(cb), C.byref(ci), C.byref(ce)))


def estimate_dtn_both(bvh: Bvh, samples: Samples, params_interior: Params, params_exterior: Params, want_stats=False,
                      out_interior=None, out_exterior=None, workspace=None, basis=None, nonblocking=False):
    """Interior and exterior DtN matrices of one mesh in one call (mcs_estimate_dtn_both): the same results as the
    two single calls, bit for bit, with the two walk kernels overlapped on two streams.  nonblocking: see
    estimate_dtn_interior (caller's outputs and workspace, hat basis, no statistics)."""
    cs, cb = samples.c(), _basis(bvh, basis)
    ci, ce = params_interior.c(), params_exterior.c()
    if nonblocking:
        if want_stats or basis is not None or out_interior is None or out_exterior is None or workspace is None:
            raise ValueError("nonblocking=True needs out_interior=, out_exterior= and workspace= from the caller, the hat basis and want_stats=False")
        if workspace.numel() < workspace_bytes_both(bvh, samples, params_interior, params_exterior, basis):
            raise ValueError("workspace too small")
        ci.nonblocking = ce.nonblocking = 1
    K = basis.K if basis is not None else bvh.V
    if out_interior is None:
        out_interior = torch.empty((K, K), dtype=torch.float32, device=bvh.device)
    if out_exterior is None:
        out_exterior = torch.empty((K, K), dtype=torch.float32, device=bvh.device)
    need = workspace_bytes_both(bvh, samples, params_interior, params_exterior, basis)
    if workspace is None or workspace.numel() < need:
        workspace = torch.empty(need, dtype=torch.uint8, device=bvh.device)
    mi = _Matrix(kind=0, K=K, dense=out_interior.data_ptr())
    me = _Matrix(kind=0, K=K, dense=out_exterior.data_ptr())
    si = Stats() if want_stats else None
    se = Stats() if want_stats else None
    with torch.cuda.device(bvh.device):
        rc = lib().mcs_estimate_dtn_both(bvh.handle, C.byref(cs), C.byref(cb), C.byref(ci), C.byref(ce), _ptr(workspace),
                                         C.c_size_t(workspace.numel()), C.byref(mi), C.byref(me),
                                         C.byref(si) if si is not None else None, C.byref(se) if se is not None else None,
                                         _stream(bvh.device))
    _check(rc, "mcs_estimate_dtn_both")
    return (out_interior, out_exterior, si, se) if want_stats else (out_interior, out_exterior)


def estimate_dtn_host(verts, faces, tri, bary, weight, params: Params, interior=True, exterior=True,
                      out_interior=None, out_exterior=None, normal=None, want_stats=False, device=None):
    """The whole path from HOST tensors (mcs_estimate_dtn_host): upload, LBVH build, estimators,
    download.  Inputs are CPU tensors (pinned memory makes the copies asynchronous); the results are
    written into CPU tensors [V,V] (allocated pinned when not given)."""
    def host(t, dtype, name):
        t = torch.as_tensor(t)
        if t.is_cuda:
            raise ValueError(f"{name} must be a CPU tensor for the host entry point")
        return t.to(dtype).contiguous()
    verts, faces = host(verts, torch.float32, "verts"), host(faces, torch.int32, "faces")
    tri, bary, weight = host(tri, torch.int32, "tri"), host(bary, torch.float32, "bary"), host(weight, torch.float32, "weight")
    normal = host(normal, torch.float32, "normal") if normal is not None else None
    V, F, n_s = int(verts.shape[0]), int(faces.shape[0]), int(tri.shape[0])
    ops = (1 if interior else 0) | (2 if exterior else 0)
    if interior and out_interior is None:
        out_interior = torch.empty((V, V), dtype=torch.float32, pin_memory=True)
    if exterior and out_exterior is None:
        out_exterior = torch.empty((V, V), dtype=torch.float32, pin_memory=True)
    cs = _Samples(tri=tri.data_ptr(), bary=bary.data_ptr(), weight=weight.data_ptr(),
                  normal=normal.data_ptr() if normal is not None else None, n_s=n_s)
    cp = params.c()
    st = Stats() if want_stats else None
    dev = torch.device("cuda" if device is None else device)
    with torch.cuda.device(dev):
        rc = lib().mcs_estimate_dtn_host(_ptr(verts), C.c_int64(V), _ptr(faces), C.c_int64(F), C.byref(cs), C.byref(cp),
                                         C.c_int(ops), _ptr(out_interior) if interior else None,
                                         _ptr(out_exterior) if exterior else None,
                                         C.byref(st) if st is not None else None, _stream(dev))
    _check(rc, "mcs_estimate_dtn_host")
    h2d = verts.numel() * 4 + faces.numel() * 4 + n_s * 20 + (n_s * 12 if normal is not None else 0)
    d2h = (int(interior) + int(exterior)) * V * V * 4
    res = dict(interior=out_interior if interior else None, exterior=out_exterior if exterior else None,
               h2d_bytes=h2d, d2h_bytes=d2h)
    if want_stats:
        res["stats"] = st
    return res


class _HostCoo(C.Structure):
    _fields_ = [("capacity", C.c_int64), ("row", C.c_void_p), ("col", C.c_void_p), ("val", C.c_void_p), ("nnz", C.c_int64)]


def estimate_dtn_host_coo(verts, faces, tri, bary, weight, params_interior: Params, params_exterior: Params,
                          out_interior, out_exterior, orient_h_scale=0.0, orient_beta=0.0, normal=None, want_stats=False,
                          device=None):
    """The whole path from HOST tensors with sparse output (mcs_estimate_dtn_host_coo): upload, LBVH build, optional
    sidedness pre-pass, both estimators, download.  out_*: (row int32, col int32, val fp32) CPU tensors of equal
    length = capacity (pinned memory makes the copies asynchronous).  Returns dict(nnz_interior, nnz_exterior,
    h2d_bytes, d2h_bytes[, stats_interior, stats_exterior]); raises McsError(MCS_ENOMEM) with .need = (ni, ne) when a
    capacity is too small."""
    def host(t, dtype, name):
        t = torch.as_tensor(t)
        if t.is_cuda:
            raise ValueError(f"{name} must be a CPU tensor for the host entry point")
        return t.to(dtype).contiguous()
    verts, faces = host(verts, torch.float32, "verts"), host(faces, torch.int32, "faces")
    tri, bary, weight = host(tri, torch.int32, "tri"), host(bary, torch.float32, "bary"), host(weight, torch.float32, "weight")
    normal = host(normal, torch.float32, "normal") if normal is not None else None
    V, F, n_s = int(verts.shape[0]), int(faces.shape[0]), int(tri.shape[0])
    outs = []
    for name, o in (("out_interior", out_interior), ("out_exterior", out_exterior)):
        r, c, v = o
        if r.is_cuda or c.is_cuda or v.is_cuda or r.dtype != torch.int32 or c.dtype != torch.int32 or v.dtype != torch.float32:
            raise ValueError(f"{name} must be CPU tensors (int32, int32, float32)")
        if not (r.is_contiguous() and c.is_contiguous() and v.is_contiguous()) or not (r.numel() == c.numel() == v.numel() > 0):
            raise ValueError(f"{name}: three contiguous tensors of equal, non-zero length")
        outs.append(_HostCoo(capacity=r.numel(), row=r.data_ptr(), col=c.data_ptr(), val=v.data_ptr(), nnz=0))
    cs = _Samples(tri=tri.data_ptr(), bary=bary.data_ptr(), weight=weight.data_ptr(),
                  normal=normal.data_ptr() if normal is not None else None, n_s=n_s)
    ci, ce = params_interior.c(), params_exterior.c()
    si = Stats() if want_stats else None
    se = Stats() if want_stats else None
    dev = torch.device("cuda" if device is None else device)
    with torch.cuda.device(dev):
        rc = lib().mcs_estimate_dtn_host_coo(_ptr(verts), C.c_int64(V), _ptr(faces), C.c_int64(F), C.byref(cs), C.byref(ci),
                                             C.byref(ce), C.c_float(float(orient_h_scale)), C.c_float(float(orient_beta)),
                                             C.byref(outs[0]), C.byref(outs[1]),
                                             C.byref(si) if si is not None else None, C.byref(se) if se is not None else None,
                                             _stream(dev))
    ni, ne = int(outs[0].nnz), int(outs[1].nnz)
    if rc == MCS_ENOMEM and (ni > outs[0].capacity or ne > outs[1].capacity):
        err = McsError(rc, "mcs_estimate_dtn_host_coo", "sparse output capacity too small")
        err.need = (ni, ne)
        raise err
    _check(rc, "mcs_estimate_dtn_host_coo")
    h2d = verts.numel() * 4 + faces.numel() * 4 + n_s * 20 + (n_s * 12 if (normal is not None and not orient_h_scale > 0) else 0)
    res = dict(nnz_interior=ni, nnz_exterior=ne, h2d_bytes=h2d, d2h_bytes=12 * (ni + ne) + 16)
    if want_stats:
        res["stats_interior"], res["stats_exterior"] = si, se
    return res


class _BatchItem(C.Structure):
    _fields_ = [("verts", C.c_void_p), ("V", C.c_int64), ("faces", C.c_void_p), ("F", C.c_int64), ("samples", _Samples),
                ("basis", _Basis), ("kelvin_origin", C.c_float * 3), ("rc", C.c_int32), ("out_interior", C.c_void_p),
                ("out_exterior", C.c_void_p), ("normal_out", C.c_void_p)]


def estimate_dtn_batch(meshes, params_interior: Params, params_exterior: Params, out_interior, out_exterior,
                       orient_h_scale=1.0, orient_beta=2.5, n_workers=4):
    """Interior and exterior dense DtN matrices of many meshes in one call (mcs_estimate_dtn_batch).
    meshes: list of dicts with CUDA tensors verts [V,3] fp32, faces [F,3] int32, samples (Samples), optional basis
    (PointBasis; default hat basis K = V), origin (3 floats).  out_interior / out_exterior: lists of (or a stacked
    tensor of) CUDA fp32 [K,K] matrices, one per mesh.  Returns the list of sidedness normals (or None)."""
    n = len(meshes)
    items = (_BatchItem * n)()
    keep, normals = [], []
    dev = meshes[0]["verts"].device
    for i, m in enumerate(meshes):
        v, f, S = _dev(m["verts"], torch.float32, "verts"), _dev(m["faces"], torch.int32, "faces"), m["samples"]
        basis = m.get("basis")
        cb = basis.c() if basis is not None else _Basis(kind=0, K=int(v.shape[0]))
        K = int(cb.K)
        oi, oe = out_interior[i], out_exterior[i]
        for o in (oi, oe):
            if not (o.is_cuda and o.dtype == torch.float32 and o.is_contiguous() and tuple(o.shape) == (K, K)):
                raise ValueError("batch outputs must be contiguous CUDA float32 [K, K] matrices")
        nrm = torch.empty((S.n_s, 3), dtype=torch.float32, device=dev) if orient_h_scale > 0 else None
        normals.append(nrm)
        keep.append((v, f, S, basis, nrm))
        it = items[i]
        it.verts, it.V, it.faces, it.F = v.data_ptr(), int(v.shape[0]), f.data_ptr(), int(f.shape[0])
        it.samples, it.basis = S.c(), cb
        it.kelvin_origin[:] = [float(x) for x in m.get("origin", (0.0, 0.0, 0.0))]
        it.out_interior, it.out_exterior = oi.data_ptr(), oe.data_ptr()
        it.normal_out = nrm.data_ptr() if nrm is not None else None
    ci, ce = params_interior.c(), params_exterior.c()
    with torch.cuda.device(dev):
        rc = lib().mcs_estimate_dtn_batch(items, C.c_int64(n), C.byref(ci), C.byref(ce), C.c_float(float(orient_h_scale)),
                                          C.c_float(float(orient_beta)), C.c_int32(int(n_workers)), _stream(dev))
    if rc != MCS_OK:
        bad = [(i, items[i].rc) for i in range(n) if items[i].rc != MCS_OK]
        raise McsError(rc, "mcs_estimate_dtn_batch", f"{lib().mcs_error_string(rc).decode()}; failing items {bad[:8]}")
    return normals if orient_h_scale > 0 else None


def tangent_balls(bvh: Bvh, samples: Samples, params: Params, exterior: bool):
    cs, cp = samples.c(), params.c()
    balls = torch.empty((samples.n_s, 8), dtype=torch.float32, device=bvh.device)
    with torch.cuda.device(bvh.device):
        _check(lib().mcs_tangent_balls(bvh.handle, C.byref(cs), C.byref(cp), C.c_int(int(exterior)), _ptr(balls),
                                       _stream(bvh.device)), "mcs_tangent_balls")
    return balls


def num_records(samples: Samples, params: Params, exterior: bool) -> int:
    n = samples.n_s * params.walks_per_sample
    if exterior and params.include_killing:
        n += params.n_kill_walks
    return n


def run_walks(bvh: Bvh, samples: Samples, params: Params, exterior: bool, want_stats=False):
    """Records [n,4] fp32 (column 0 holds tri_t as int32 bits) and steps [n] int32."""
    cs, cp = samples.c(), params.c()
    n = num_records(samples, params, exterior)
    rec = torch.empty((n, 4), dtype=torch.float32, device=bvh.device)
    steps = torch.empty(n, dtype=torch.int32, device=bvh.device)
    need = int(lib().mcs_walk_workspace_bytes(C.byref(cs)))
    ws = torch.empty(need, dtype=torch.uint8, device=bvh.device)
    st = Stats() if want_stats else None
    with torch.cuda.device(bvh.device):
        rc = lib().mcs_run_walks(bvh.handle, C.byref(cs), C.byref(cp), C.c_int(int(exterior)), _ptr(ws),
                                 C.c_size_t(need), _ptr(rec), _ptr(steps),
                                 C.byref(st) if st is not None else None, _stream(bvh.device))
    _check(rc, "mcs_run_walks")
    return (rec, steps, st) if want_stats else (rec, steps)


def accumulate(bvh: Bvh, samples: Samples, params: Params, records, want_stats=False, basis=None):
    cs, cb, cp = samples.c(), _basis(bvh, basis), params.c()
    records = _dev(records, torch.float32, "records")
    n = records.shape[0]
    K = basis.K if basis is not None else bvh.V
    out = torch.empty((K, K), dtype=torch.float32, device=bvh.device)
    need = int(lib().mcs_accumulate_workspace_bytes(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), C.c_int64(n)))
    ws = torch.empty(need, dtype=torch.uint8, device=bvh.device)
    m = _Matrix(kind=0, K=K, dense=out.data_ptr())
    st = Stats() if want_stats else None
    with torch.cuda.device(bvh.device):
        rc = lib().mcs_accumulate(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), _ptr(records), C.c_int64(n),
                                  _ptr(ws), C.c_size_t(need), C.byref(m),
                                  C.byref(st) if st is not None else None, _stream(bvh.device))
    _check(rc, "mcs_accumulate")
    return (out, st) if want_stats else out


def philox4x32_10(counters, key):
    counters = _dev(counters, torch.int32, "counters")
    n = counters.shape[0]
    out = torch.empty((n, 4), dtype=torch.int32, device=counters.device)
    k = (C.c_uint32 * 2)(int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF)
    with torch.cuda.device(counters.device):
        _check(lib().mcs_philox4x32_10(_ptr(counters), C.c_int64(n), k, _ptr(out), _stream(counters.device)),
               "mcs_philox4x32_10")
    return out


def sort_pairs_u64(keys, vals, key_bits=64):
    """In-place stable radix sort of int64 keys (as unsigned) with int32 payloads."""
    assert keys.is_cuda and vals.is_cuda and keys.dtype == torch.int64 and vals.dtype == torch.int32
    n = keys.numel()
    need = int(lib().mcs_sort_workspace_bytes(C.c_int64(n)))
    ws = torch.empty(need, dtype=torch.uint8, device=keys.device)
    with torch.cuda.device(keys.device):
        _check(lib().mcs_sort_pairs_u64(_ptr(keys), _ptr(vals), C.c_int64(n), C.c_int32(key_bits), _ptr(ws),
                                        C.c_size_t(need), _stream(keys.device)), "mcs_sort_pairs_u64")
    return keys, vals


def sort_static_max_n() -> int:
    f = lib().mcs_sort_static_max_n
    f.restype = C.c_int64
    return int(f())


def sort_pairs_u64_static(keys, vals, key_bits=64):
    """mcs_sort_pairs_u64_static: the same in-place sort with the workspace in a static device array of the library
    (no allocation in the call; n <= sort_static_max_n(); calls that overlap on the GPU race on the shared array)."""
    assert keys.is_cuda and vals.is_cuda and keys.dtype == torch.int64 and vals.dtype == torch.int32
    n = keys.numel()
    with torch.cuda.device(keys.device):
        _check(lib().mcs_sort_pairs_u64_static(_ptr(keys), _ptr(vals), C.c_int64(n), C.c_int32(key_bits),
                                               _stream(keys.device)), "mcs_sort_pairs_u64_static")
    return keys, vals


class PhaseTimes(C.Structure):
    _fields_ = [("prep_ms", C.c_float), ("walk_ms", C.c_float), ("accumulate_ms", C.c_float),
                ("total_ms", C.c_float), ("walk_interior_ms", C.c_float), ("walk_exterior_ms", C.c_float)]


def launch_count() -> int:
    f = lib().mcs_launch_count
    f.restype = C.c_ulonglong
    return int(f())


def profile_enable(on: bool):
    _check(lib().mcs_profile_enable(C.c_int(int(on))), "mcs_profile_enable")


def profile_last() -> PhaseTimes:
    o = PhaseTimes()
    _check(lib().mcs_profile_last(C.byref(o)), "mcs_profile_last")
    return o


def version() -> str:
    return lib().mcs_version().decode()


def measure_fp32_tflops(device="cuda") -> float:
    o = C.c_double(0.0)
    with torch.cuda.device(device):
        _check(lib().mcs_measure_fp32_tflops(C.byref(o), _stream(torch.device(device))), "mcs_measure_fp32_tflops")
    return o.value


def measure_l2_gbs(device="cuda") -> float:
    o = C.c_double(0.0)
    with torch.cuda.device(device):
        _check(lib().mcs_measure_l2_gbs(C.byref(o), _stream(torch.device(device))), "mcs_measure_l2_gbs")
    return o.value


# ------------------------------------------------------------------------------
# sparse output (output_kind 1)
# ------------------------------------------------------------------------------
@dataclass
class CooMatrix:
    """Upper triangle (row <= col) of the symmetric DtN matrix, sorted by (row, col)."""
    K: int
    row: torch.Tensor
    col: torch.Tensor
    val: torch.Tensor

    @property
    def nnz(self):
        return int(self.row.numel())

    def to_dense(self):
        S = torch.zeros((self.K, self.K), dtype=torch.float32, device=self.val.device)
        r, c = self.row.long(), self.col.long()
        S[r, c] = self.val
        S[c, r] = self.val
        return S


def _coo_buffers(K, capacity, device):
    row = torch.empty(capacity, dtype=torch.int32, device=device)
    col = torch.empty(capacity, dtype=torch.int32, device=device)
    val = torch.empty(capacity, dtype=torch.float32, device=device)
    nnz = torch.zeros(1, dtype=torch.int64, device=device)
    m = _Matrix(kind=1, K=K, dense=None, coo_capacity=capacity, coo_row=row.data_ptr(), coo_col=col.data_ptr(),
                coo_val=val.data_ptr(), coo_nnz=nnz.data_ptr())
    return row, col, val, nnz, m


def estimate_dtn_coo(bvh: Bvh, samples: Samples, params: Params, exterior: bool, capacity: int | None = None,
                     want_stats=False, max_retries=6):
    """DtN matrix in sparse COO form (any K): mcs_estimate_dtn_* with output_kind 1.  When the capacity guess is too
    small the library reports MCS_ENOMEM with a lower bound of the need; the walks are NOT repeated: their records are
    still at the head of the workspace, and only the accumulation (mcs_accumulate) is run again with a larger buffer."""
    import dataclasses
    K = bvh.V
    n_rec = num_records(samples, params, exterior)
    cap = int(capacity) if capacity else max(4096, min(K * (K + 1) // 2, 4 * n_rec))
    fn = lib().mcs_estimate_dtn_exterior if exterior else lib().mcs_estimate_dtn_interior
    p = dataclasses.replace(params, output_kind=1, coo_capacity=cap)
    cs, cb, cp = samples.c(), _basis(bvh), p.c()
    need = int(lib().mcs_workspace_bytes(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), C.c_int(int(exterior))))
    ws = torch.empty(need, dtype=torch.uint8, device=bvh.device)
    row, col, val, nnz, m = _coo_buffers(K, cap, bvh.device)
    st = Stats()
    with torch.cuda.device(bvh.device):
        rc = fn(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), _ptr(ws), C.c_size_t(need), C.byref(m),
                C.byref(st), _stream(bvh.device))
    if rc == MCS_ENOMEM and int(nnz.item()) > cap:
        if max_retries <= 1:
            raise McsError(MCS_ENOMEM, "estimate_dtn_coo", "capacity retries exhausted")
        # records: [n_rec][4] fp32 at offset 0 of the workspace (capi.cu make_layout); the walk counters are already in st
        records = ws[: n_rec * 16].view(torch.float32).view(n_rec, 4).clone()
        del ws, row, col, val
        out = accumulate_coo(bvh, samples, params, records, capacity=max(2 * cap, 2 * int(nnz.item())), max_retries=max_retries - 1)
        st.n_unique = out.nnz
        return (out, st) if want_stats else out
    _check(rc, "mcs_estimate_dtn (coo)")
    n = int(nnz.item())
    out = CooMatrix(K, row[:n], col[:n], val[:n])
    return (out, st) if want_stats else out


def accumulate_coo(bvh: Bvh, samples: Samples, params: Params, records, capacity: int | None = None, max_retries=6):
    """A7 alone with sparse output (mcs_accumulate, output_kind 1): records [n,4] fp32 as run_walks returns them."""
    import dataclasses
    records = _dev(records, torch.float32, "records")
    n = int(records.shape[0])
    K = bvh.V
    cap = int(capacity) if capacity else max(4096, min(K * (K + 1) // 2, 21 * n))
    for _ in range(max_retries):
        p = dataclasses.replace(params, output_kind=1, coo_capacity=cap)
        cs, cb, cp = samples.c(), _basis(bvh), p.c()
        need = int(lib().mcs_accumulate_workspace_bytes(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), C.c_int64(n)))
        ws = torch.empty(need, dtype=torch.uint8, device=bvh.device)
        row, col, val, nnz, m = _coo_buffers(K, cap, bvh.device)
        with torch.cuda.device(bvh.device):
            rc = lib().mcs_accumulate(bvh.handle, C.byref(cs), C.byref(cb), C.byref(cp), _ptr(records), C.c_int64(n),
                                      _ptr(ws), C.c_size_t(need), C.byref(m), None, _stream(bvh.device))
        if rc == MCS_ENOMEM and int(nnz.item()) > cap:
            cap = min(K * (K + 1) // 2, max(2 * cap, 2 * int(nnz.item())))
            continue
        _check(rc, "mcs_accumulate (coo)")
        k = int(nnz.item())
        return CooMatrix(K, row[:k], col[:k], val[:k])
    raise McsError(MCS_ENOMEM, "accumulate_coo", "capacity retries exhausted")


def estimate_dtn_coo_both(bvh: Bvh, samples: Samples, params_interior: Params, params_exterior: Params,
                          capacity: int | None = None, max_retries=6, scratch: dict | None = None):
    """Interior and exterior DtN matrices in sparse COO form from one mcs_estimate_dtn_both call (walk kernels
    overlapped).  Same entries as two estimate_dtn_coo calls; one capacity for both, grown on MCS_ENOMEM.
    scratch: a dict the caller keeps between calls; the workspace and the output buffers are kept in it and reused
    while they are large enough (the returned matrices are then views into it, valid until the next call)."""
    import dataclasses
    K = bvh.V
    n_rec = max(num_records(samples, params_interior, False), num_records(samples, params_exterior, True))
    cap = int(capacity) if capacity else max(4096, min(K * (K + 1) // 2, 4 * n_rec))
    for _ in range(max_retries):
        pi = dataclasses.replace(params_interior, output_kind=1, coo_capacity=cap)
        pe = dataclasses.replace(params_exterior, output_kind=1, coo_capacity=cap)
        need = workspace_bytes_both(bvh, samples, pi, pe)
        ws = scratch.get("ws") if scratch is not None else None
        if ws is None or ws.numel() < need or ws.device != bvh.device:
            ws = None
            if scratch is not None:
                scratch.pop("ws", None)
            ws = torch.empty(need, dtype=torch.uint8, device=bvh.device)
            if scratch is not None:
                scratch["ws"] = ws
        bufs = scratch.get("bufs") if scratch is not None else None
        if bufs is None or bufs[0] != (K, cap):
            bufs = ((K, cap), _coo_buffers(K, cap, bvh.device), _coo_buffers(K, cap, bvh.device))
            if scratch is not None:
                scratch["bufs"] = bufs
        bi, be = bufs[1], bufs[2]
        cs, cb, ci, ce = samples.c(), _basis(bvh), pi.c(), pe.c()
        with torch.cuda.device(bvh.device):
            rc = lib().mcs_estimate_dtn_both(bvh.handle, C.byref(cs), C.byref(cb), C.byref(ci), C.byref(ce), _ptr(ws),
                                             C.c_size_t(ws.numel()), C.byref(bi[4]), C.byref(be[4]), None, None,
                                             _stream(bvh.device))
            torch.cuda.current_stream(bvh.device).synchronize()
        worst = max(int(bi[3].item()), int(be[3].item()))
        if rc == MCS_ENOMEM and worst > cap:
            if max_retries <= 1:
                raise McsError(MCS_ENOMEM, "estimate_dtn_coo_both", "capacity retries exhausted")
            # The walks are not repeated: both operators' records sit at the head of their halves of the workspace
            # (capi.cu estimate_both: interior at 0, exterior behind the interior's layout); only A7 runs again.
            n_i, n_e = num_records(samples, pi, False), num_records(samples, pe, True)
            off = workspace_bytes(bvh, samples, pi, False)
            rec_i = ws[: n_i * 16].view(torch.float32).view(n_i, 4).clone()
            rec_e = ws[off: off + n_e * 16].view(torch.float32).view(n_e, 4).clone()
            del ws, bi, be, bufs
            if scratch is not None:
                scratch.clear()
            big = max(2 * cap, 2 * worst)
            return (accumulate_coo(bvh, samples, params_interior, rec_i, capacity=big, max_retries=max_retries - 1),
                    accumulate_coo(bvh, samples, params_exterior, rec_e, capacity=big, max_retries=max_retries - 1))
        _check(rc, "mcs_estimate_dtn_both (coo)")
        ni, ne = int(bi[3].item()), int(be[3].item())
        return (CooMatrix(K, bi[0][:ni], bi[1][:ni], bi[2][:ni]), CooMatrix(K, be[0][:ne], be[1][:ne], be[2][:ne]))
    raise McsError(MCS_ENOMEM, "estimate_dtn_coo_both", "capacity retries exhausted")


def steklov_eigs(S, mass, n_eig, want_vectors=True, method="auto"):
    """Smallest n_eig eigenpairs of S psi = lambda diag(mass) psi (mcs_steklov_eigs).  S: [K,K] or [B,K,K] CUDA fp32;
    mass: [K] or [B,K].  Returns (evals [B,n_eig] or [n_eig], evecs [B,n_eig,K] or [n_eig,K] or None, sweeps).
    method: "auto" (subspace iteration for few eigenpairs of a large matrix, else Jacobi), "jacobi", "subspace"."""
    method_code = {"auto": 0, "jacobi": 1, "subspace": 2}[method]
    S = _dev(S, torch.float32, "S")
    mass = _dev(mass, torch.float32, "mass")
    single = S.ndim == 2
    if single:
        S, mass = S[None], mass[None]
    B, K = int(S.shape[0]), int(S.shape[1])
    f = lib().mcs_steklov_eigs_workspace_bytes
    f.restype = C.c_size_t
    need = int(f(C.c_int64(K), C.c_int64(B)))
    ws = torch.empty(need, dtype=torch.uint8, device=S.device)
    evals = torch.empty((B, n_eig), dtype=torch.float32, device=S.device)
    evecs = torch.empty((B, n_eig, K), dtype=torch.float32, device=S.device) if want_vectors else None
    sweeps = C.c_int32(0)
    with torch.cuda.device(S.device):
        rc = lib().mcs_steklov_eigs_method(_ptr(S), _ptr(mass), C.c_int64(K), C.c_int64(B), C.c_int32(n_eig), C.c_int32(method_code),
                                           _ptr(evals), _ptr(evecs), _ptr(ws), C.c_size_t(need), C.byref(sweeps), _stream(S.device))
    if rc == MCS_WNOTCONVERGED:
        import warnings
        warnings.warn("mcs_steklov_eigs: iteration cap reached before convergence (input not positive semi-definite, or "
                      "method='subspace' on a spectrum crowded at its low end?)")
    else:
        _check(rc, "mcs_steklov_eigs")
    if single:
        return evals[0], (evecs[0] if evecs is not None else None), sweeps.value
    return evals, evecs, sweeps.value


def _winding_ws(bvh, n, device):
    f = lib().mcs_winding_workspace_bytes
    f.restype = C.c_size_t
    need = int(f(bvh.handle, C.c_int64(n)))
    return torch.empty(need, dtype=torch.uint8, device=device), need


def winding_number(bvh, points, exclude=None):
    """Generalised winding number of the mesh at points [n,3] (mcs_winding_number); exclude [n] int32: face left out."""
    points = _dev(points, torch.float32, "points").reshape(-1, 3)
    n = int(points.shape[0])
    ex = _dev(exclude, torch.int32, "exclude") if exclude is not None else None
    w = torch.empty(n, dtype=torch.float32, device=points.device)
    with torch.cuda.device(points.device):
        ws, need = _winding_ws(bvh, n, points.device)
        _check(lib().mcs_winding_number(bvh.handle, _ptr(points), _ptr(ex), C.c_int64(n), _ptr(w), _ptr(ws),
                                        C.c_size_t(need), _stream(points.device)), "mcs_winding_number")
    return w


def orient_samples(bvh, samples, h_scale=1.0):
    """(normal [n_s,3] pointing out of the solid, d [n_s]) by the winding-number rule G-R1 (mcs_orient_samples).
    Pass the normals back as Samples(..., normal=...) to draw the tangent balls on the right side of flipped faces."""
    dev = samples.tri.device
    n = int(samples.tri.shape[0])
    nrm = torch.empty((n, 3), dtype=torch.float32, device=dev)
    d = torch.empty(n, dtype=torch.float32, device=dev)
    cs = samples.c()
    with torch.cuda.device(dev):
        ws, need = _winding_ws(bvh, n, dev)
        _check(lib().mcs_orient_samples(bvh.handle, C.byref(cs), C.c_float(h_scale), _ptr(nrm), _ptr(d), _ptr(ws),
                                        C.c_size_t(need), _stream(dev)), "mcs_orient_samples")
    return nrm, d


def orient_samples_fast(bvh, samples, h_scale=1.0, beta=2.5):
    """(normal [n_s,3], d [n_s]) as orient_samples, from the hierarchical evaluation (mcs_orient_samples_fast)."""
    dev = samples.tri.device
    n = int(samples.tri.shape[0])
    nrm = torch.empty((n, 3), dtype=torch.float32, device=dev)
    d = torch.empty(n, dtype=torch.float32, device=dev)
    cs = samples.c()
    with torch.cuda.device(dev):
        _check(lib().mcs_orient_samples_fast(bvh.handle, C.byref(cs), C.c_float(h_scale), C.c_float(beta), _ptr(nrm), _ptr(d),
                                             _stream(dev)), "mcs_orient_samples_fast")
    return nrm, d


def project_galerkin(S, Phi):
    """Reduced Ritz-Galerkin matrix Phi^T S Phi (mcs_project_galerkin).  S [V,V], Phi [V,K] CUDA fp32 -> [K,K]."""
    S = _dev(S, torch.float32, "S")
    Phi = _dev(Phi, torch.float32, "Phi")
    V, K = int(Phi.shape[0]), int(Phi.shape[1])
    if tuple(S.shape) != (V, V):
        raise ValueError("S must be [V, V] with V = Phi.shape[0]")
    f = lib().mcs_project_workspace_bytes
    f.restype = C.c_size_t
    need = int(f(C.c_int64(V), C.c_int64(K)))
    ws = torch.empty(need, dtype=torch.uint8, device=S.device)
    out = torch.empty((K, K), dtype=torch.float32, device=S.device)
    with torch.cuda.device(S.device):
        _check(lib().mcs_project_galerkin(_ptr(S), _ptr(Phi), C.c_int64(V), C.c_int64(K), _ptr(out), _ptr(ws),
                                          C.c_size_t(need), _stream(S.device)), "mcs_project_galerkin")
    return out


def project_galerkin_coo(coo, Phi):
    """Reduced Ritz-Galerkin matrix Phi^T S Phi from the sparse output (CooMatrix of estimate_dtn_coo); Phi [V,K]."""
    Phi = _dev(Phi, torch.float32, "Phi")
    V, K = int(Phi.shape[0]), int(Phi.shape[1])
    if V != coo.K:
        raise ValueError("Phi must have one row per basis function of the sparse matrix")
    row, col, val = _dev(coo.row, torch.int32, "row"), _dev(coo.col, torch.int32, "col"), _dev(coo.val, torch.float32, "val")
    f = lib().mcs_project_coo_workspace_bytes
    f.restype = C.c_size_t
    need = int(f(C.c_int64(V), C.c_int64(K)))
    ws = torch.empty(need, dtype=torch.uint8, device=Phi.device)
    out = torch.empty((K, K), dtype=torch.float32, device=Phi.device)
    with torch.cuda.device(Phi.device):
        _check(lib().mcs_project_galerkin_coo(_ptr(row), _ptr(col), _ptr(val), C.c_int64(int(row.numel())), _ptr(Phi),
                                              C.c_int64(V), C.c_int64(K), _ptr(out), _ptr(ws), C.c_size_t(need),
                                              _stream(Phi.device)), "mcs_project_galerkin_coo")
    return out
