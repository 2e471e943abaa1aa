"""ctypes front end of oracle/dtn_oracle.c (argument marshalling only).

TEST INFRASTRUCTURE: see the package docstring for who may import this.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass, field

import numpy as np

from .build import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_u01.restype = C.c_double
        _lib.orc_u01.argtypes = [C.c_uint32]
        _lib.orc_closest_point_triangle.restype = C.c_double
        _lib.orc_closest_point_triangle_alt.restype = C.c_double
        _lib.orc_inverted_ratio2_triangle.restype = C.c_double
        _lib.orc_rmax.restype = C.c_double
        _lib.orc_aabb_diagonal.restype = C.c_double
        _lib.orc_max_vertex_norm.restype = C.c_double
        _lib.orc_total_area.restype = C.c_double
        _lib.orc_run_walks.restype = C.c_int64
        _lib.orc_run_walks_subset.restype = C.c_int64
        _lib.orc_walk_query_points.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
        for f in ("orc_sizeof_record", "orc_sizeof_params", "orc_sizeof_geom"):
            getattr(_lib, f).restype = C.c_size_t
        assert _lib.orc_sizeof_record() == RECORD_DTYPE.itemsize
        assert _lib.orc_sizeof_params() == C.sizeof(_Params)
        assert _lib.orc_sizeof_geom() == C.sizeof(_Geom)
        _lib.orc_sizeof_point_basis.restype = C.c_size_t
        assert _lib.orc_sizeof_point_basis() == C.sizeof(_PointBasis)
    return _lib


class _Geom(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pad_", C.c_int32),
                ("verts", C.c_void_p), ("V", C.c_int64),
                ("faces", C.c_void_p), ("F", C.c_int64),
                ("centre", C.c_double * 3), ("radius", C.c_double)]


class _Params(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("walks_per_sample", C.c_int32), ("max_steps", C.c_int32),
                ("eps", C.c_double), ("cap_half_angle_deg", C.c_double), ("rmax", C.c_double),
                ("bisection_iters", C.c_int32), ("importance_sample", C.c_int32),
                ("antithetic", C.c_int32), ("include_killing", C.c_int32),
                ("n_kill_walks", C.c_int64), ("origin", C.c_double * 3), ("Rmax_norm", C.c_double),
                ("escape_radius", C.c_double), ("estimator", C.c_int32), ("pad_", C.c_int32), ("inset", C.c_double),
                ("exterior_query", C.c_int32), ("pad2_", C.c_int32)]


class _PointBasis(C.Structure):
    _fields_ = [("points", C.c_void_p), ("normals", C.c_void_p), ("K", C.c_int64), ("k", C.c_int32),
                ("pad_", C.c_int32), ("sigma", C.c_double), ("tau_n", C.c_double)]


@dataclass
class PointBasis:
    """Point-based function space: points, unit normals, k, sigma, tau_n."""
    points: np.ndarray
    normals: np.ndarray
    k: int = 8
    sigma: float = 0.025
    tau_n: float = 0.8

    def c(self):
        self._p = np.ascontiguousarray(self.points, np.float32)
        self._n = np.ascontiguousarray(self.normals, np.float32)
        return _PointBasis(points=self._p.ctypes.data, normals=self._n.ctypes.data, K=len(self._p), k=int(self.k),
                           sigma=float(self.sigma), tau_n=float(self.tau_n))


RECORD_DTYPE = np.dtype([("sample", np.int64), ("tri_t", np.int64), ("bary_t", np.float64, 3),
                         ("t", np.float64, 3), ("z", np.float64, 3), ("weight", np.float64),
                         ("steps", np.int32), ("pad_", np.int32)])


@dataclass
class OracleParams:
    seed: int = 0
    walks_per_sample: int = 1
    eps: float = 1e-3
    max_steps: int = 4096
    cap_half_angle_deg: float = 2.5
    rmax_scale: float = 1.0
    bisection_iters: int = 10
    importance_sample: bool = True
    antithetic: bool = False
    include_killing: bool = False
    n_kill_walks: int = 0
    origin: tuple = (0.0, 0.0, 0.0)
    estimator: int = 0                   # 0: Alg. 2; 1: Alg. 1 (naive finite difference, interior only)
    inset: float = 0.0                   # Alg. 1: x = s - inset * n_s
    exterior_query: int = 0              # 0: flat-triangle query + conservative radius (E3); 1: exact inverted faces (E4)
    rmax: float | None = None            # overrides the AABB rule (analytic sphere pins)
    Rmax_norm: float | None = None


@dataclass
class _GeomHandle:
    c: _Geom
    keep: list = field(default_factory=list)
    verts: np.ndarray | None = None
    faces: np.ndarray | None = None


def mesh_geom(verts, faces) -> _GeomHandle:
    v = np.ascontiguousarray(verts, np.float32)
    f = np.ascontiguousarray(faces, np.int32)
    g = _Geom(kind=0, verts=v.ctypes.data, V=len(v), faces=f.ctypes.data, F=len(f))
    return _GeomHandle(g, [v, f], v, f)


def sphere_geom(centre=(0.0, 0.0, 0.0), radius=1.0) -> _GeomHandle:
    g = _Geom(kind=1, verts=None, V=0, faces=None, F=0, radius=float(radius))
    g.centre[:] = [float(x) for x in centre]
    return _GeomHandle(g)


def philox4x32_10(counter, key):
    lib = _load()
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in counter])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib.orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def u01(x: int) -> float:
    return _load().orc_u01(int(x) & 0xFFFFFFFF)


def _d3(x):
    return (C.c_double * 3)(*[float(v) for v in x])


def closest_point_triangle(p, a, b, c):
    lib = _load()
    cp, bary = (C.c_double * 3)(), (C.c_double * 3)()
    d2 = lib.orc_closest_point_triangle(_d3(p), _d3(a), _d3(b), _d3(c), cp, bary)
    return d2, np.array(cp), np.array(bary)


def closest_point_triangle_alt(p, a, b, c):
    lib = _load()
    cp = (C.c_double * 3)()
    d2 = lib.orc_closest_point_triangle_alt(_d3(p), _d3(a), _d3(b), _d3(c), cp)
    return d2, np.array(cp)


def inverted_ratio2_triangle(x, a, b, c):
    """min over the flat triangle (a, b, c) of |x - p|^2 / |p|^2 (coordinates about the inversion centre) and the
    barycentrics of the minimiser: the exact distance to the Kelvin image of the face is sqrt(.) / |x| (reading E4)."""
    lib = _load()
    bary = (C.c_double * 3)()
    r2 = lib.orc_inverted_ratio2_triangle(_d3(x), _d3(a), _d3(b), _d3(c), bary)
    return r2, np.array(bary)


class Oracle:
    """Brute-force CPU estimator over one geometry (mesh or analytic sphere)."""

    def __init__(self, geom: _GeomHandle):
        self.lib = _load()
        self.geom = geom

    # -- geometry --------------------------------------------------------
    def closest_points(self, queries, want_second=False):
        q = np.ascontiguousarray(queries, np.float32)
        n = len(q)
        dist = np.empty(n)
        tri = np.empty(n, np.int64)
        cp = np.empty((n, 3))
        bary = np.empty((n, 3))
        second = np.empty(n) if want_second else None
        self.lib.orc_closest_points(C.byref(self.geom.c), q.ctypes.data_as(C.c_void_p), C.c_int64(n),
                                    dist.ctypes.data_as(C.c_void_p), tri.ctypes.data_as(C.c_void_p),
                                    cp.ctypes.data_as(C.c_void_p), bary.ctypes.data_as(C.c_void_p),
                                    second.ctypes.data_as(C.c_void_p) if want_second else None)
        out = dict(dist=dist, tri=tri, cp=cp, bary=bary)
        if want_second:
            out["second"] = second
        return out

    def runner_up(self, queries, tri):
        """Distance to the nearest face other than `tri` (and its exact copies): tie filter."""
        q = np.ascontiguousarray(queries, np.float32)
        t = np.ascontiguousarray(tri, np.int64)
        out = np.empty(len(q))
        self.lib.orc_runner_up(C.byref(self.geom.c), q.ctypes.data_as(C.c_void_p), C.c_int64(len(q)),
                               t.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
        return out

    def closest_point_inverted(self, x, origin=(0, 0, 0)):
        """(ratio, face, closest primal point, barycentrics): min over the mesh of |x - p| / |p - o| (reading E4)."""
        class _Hit(C.Structure):
            _fields_ = [("dist", C.c_double), ("cp", C.c_double * 3), ("bary", C.c_double * 3), ("tri", C.c_int64)]
        h = _Hit()
        self.lib.orc_closest_point_inverted(C.byref(self.geom.c), _d3(x), _d3(origin), C.byref(h))
        return h.dist, int(h.tri), np.array(h.cp), np.array(h.bary)

    def rmax(self, exterior=False, origin=(0, 0, 0)):
        return self.lib.orc_rmax(C.byref(self.geom.c), C.c_int(int(exterior)), _d3(origin))

    def max_vertex_norm(self, origin=(0, 0, 0)):
        return self.lib.orc_max_vertex_norm(C.byref(self.geom.c), _d3(origin))

    def total_area(self):
        return self.lib.orc_total_area(C.byref(self.geom.c))

    def mass_matrix(self):
        V = self.geom.c.V
        M = np.zeros((V, V))
        self.lib.orc_mass_matrix_p1(C.byref(self.geom.c), M.ctypes.data_as(C.c_void_p))
        return M

    # -- estimator -------------------------------------------------------
    def _params(self, p: OracleParams, exterior: bool) -> _Params:
        cp = _Params(seed=p.seed, walks_per_sample=p.walks_per_sample, max_steps=p.max_steps,
                     eps=p.eps, cap_half_angle_deg=p.cap_half_angle_deg,
                     bisection_iters=p.bisection_iters, importance_sample=int(p.importance_sample),
                     antithetic=int(p.antithetic), include_killing=int(p.include_killing),
                     n_kill_walks=int(p.n_kill_walks), estimator=int(p.estimator), inset=float(p.inset),
                     exterior_query=int(p.exterior_query))
        cp.origin[:] = [float(x) for x in p.origin]
        if p.rmax is not None:
            cp.rmax = float(p.rmax)
        else:
            cp.rmax = float(np.float32(p.rmax_scale)) * self.rmax(exterior, p.origin)
        cp.escape_radius = 0.0 if exterior else float(np.float32(self.lib.orc_aabb_diagonal(C.byref(self.geom.c))))
        if p.Rmax_norm is not None:
            cp.Rmax_norm = float(p.Rmax_norm)
        elif self.geom.c.kind == 0:
            cp.Rmax_norm = self.max_vertex_norm(p.origin)
        return cp

    def run_walks(self, params: OracleParams, exterior: bool, tri=None, bary=None, weight=None,
                  normal=None, pos=None):
        """One record per walk (slot sample*W + walk, then killing walks) and the
        tangent balls [r, c(3), |s*|] per sample."""
        weight = np.ascontiguousarray(weight, np.float32)
        n_s = len(weight)
        if self.geom.c.kind == 0:
            tri = np.ascontiguousarray(tri, np.int32)
            bary = np.ascontiguousarray(bary, np.float32)
        else:
            pos = np.ascontiguousarray(pos, np.float64)
        if normal is not None:
            normal = np.ascontiguousarray(normal, np.float32)
        cp = self._params(params, exterior)
        n_kill = params.n_kill_walks if (exterior and params.include_killing) else 0
        rec = np.zeros(n_s * params.walks_per_sample + n_kill, RECORD_DTYPE)
        balls = np.zeros((n_s, 5))
        ptr = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        n = self.lib.orc_run_walks(C.byref(self.geom.c), C.byref(cp), C.c_int(int(exterior)),
                                   ptr(tri), ptr(bary), ptr(weight), ptr(normal), ptr(pos),
                                   C.c_int64(n_s), ptr(rec), ptr(balls))
        assert n == len(rec)
        return rec, balls

    def run_walks_subset(self, params: OracleParams, exterior: bool, tri, bary, weight, ids, n_w,
                         n_kill_first=0, normal=None):
        """Records of walks 0..n_w-1 of the samples `ids` of the FULL arrays (same Philox
        counters as the full run), then of the first n_kill_first killing walks."""
        tri = np.ascontiguousarray(tri, np.int32)
        bary = np.ascontiguousarray(bary, np.float32)
        weight = np.ascontiguousarray(weight, np.float32)
        ids = np.ascontiguousarray(ids, np.int64)
        if normal is not None:
            normal = np.ascontiguousarray(normal, np.float32)
        cp = self._params(params, exterior)
        nk = int(n_kill_first) if (exterior and params.include_killing) else 0
        rec = np.zeros(len(ids) * n_w + nk, RECORD_DTYPE)
        ptr = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        n = self.lib.orc_run_walks_subset(C.byref(self.geom.c), C.byref(cp), C.c_int(int(exterior)),
                                          ptr(tri), ptr(bary), ptr(weight), ptr(normal), ptr(ids),
                                          C.c_int64(len(ids)), C.c_int(int(n_w)), C.c_int64(nk), ptr(rec))
        assert n == len(rec)
        return rec

    def walk_query_points(self, params: OracleParams, exterior: bool, tri, bary, weight, ids, n_w, max_pos=64, normal=None):
        """(points [n,3], exact distances [n]): the primal query points of the closest-point queries made by walks
        0..n_w-1 of the samples `ids` (measurement helper of bench.py: the population on which the ideal traversal
        counts of a tree are taken)."""
        tri = np.ascontiguousarray(tri, np.int32)
        bary = np.ascontiguousarray(bary, np.float32)
        weight = np.ascontiguousarray(weight, np.float32)
        ids = np.ascontiguousarray(ids, np.int64)
        if normal is not None:
            normal = np.ascontiguousarray(normal, np.float32)
        cp = self._params(params, exterior)
        cap = len(ids) * n_w * max_pos
        pos = np.zeros((cap, 3))
        dist = np.zeros(cap)
        count = np.zeros(len(ids) * n_w, np.int32)
        ptr = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        self.lib.orc_walk_query_points(C.byref(self.geom.c), C.byref(cp), C.c_int(int(exterior)), ptr(tri), ptr(bary), ptr(weight),
                                       ptr(normal), ptr(ids), C.c_int64(len(ids)), C.c_int(int(n_w)), C.c_int(int(max_pos)),
                                       ptr(pos), ptr(dist), ptr(count))
        keep = (np.arange(max_pos)[None, :] < count[:, None]).ravel()
        return pos[keep], dist[keep]

    def accumulate_hat(self, rec, tri, bary, want_var=False, naive=False):
        K = self.geom.c.V
        tri = np.ascontiguousarray(tri, np.int32)
        bary = np.ascontiguousarray(bary, np.float32)
        rec = np.ascontiguousarray(rec)
        S = np.zeros((K, K))
        S2 = np.zeros((K, K)) if want_var else None
        fn = self.lib.orc_accumulate_hat_naive if naive else self.lib.orc_accumulate_hat
        fn(C.byref(self.geom.c), rec.ctypes.data_as(C.c_void_p),
                                    C.c_int64(len(rec)), tri.ctypes.data_as(C.c_void_p),
                                    bary.ctypes.data_as(C.c_void_p), C.c_int64(K),
                                    S.ctypes.data_as(C.c_void_p),
                                    S2.ctypes.data_as(C.c_void_p) if want_var else None)
        return (S, S2) if want_var else S

    def accumulate_reduced(self, rec, tri, bary, Phi):
        """Reduced Ritz-Galerkin DtN matrix: basis functions phi_k = sum_v Phi[v,k] hat_v,
        so b(p) = Phi^T iota(p) with iota(p) the hat-basis vector of p (3 non-zeros), and every walk adds
        weight * d d^T with d = b(s) - b(t) (Alg. 2; killing walks add weight * b(t) b(t)^T, Eq. 32).
        Written as the deferred batched outer product D^T diag(w) D over all records.  Phi: [V, K] fp64."""
        Phi = np.asarray(Phi, np.float64)
        faces = np.ctypeslib.as_array(C.cast(self.geom.c.faces, C.POINTER(C.c_int32)), shape=(self.geom.c.F, 3))
        rec = rec[(rec["tri_t"] >= 0) & (rec["weight"] != 0)]
        bt = np.einsum("qk,qkc->qc", rec["bary_t"], Phi[faces[rec["tri_t"]]])                 # b(t)
        main = rec["sample"] >= 0
        smp = rec["sample"][main]
        bs = np.einsum("qk,qkc->qc", np.asarray(bary, np.float64)[smp], Phi[faces[np.asarray(tri)[smp]]])
        D = bt.copy()
        D[main] = bs - bt[main]
        return (D * rec["weight"][:, None]).T @ D

    def winding_number(self, p, exclude=None):
        """Generalised winding number of the mesh at points p [n,3]; exclude [n]: face left out (-1: none)."""
        p = np.ascontiguousarray(p, np.float64).reshape(-1, 3)
        w = np.empty(len(p))
        ex = None if exclude is None else np.ascontiguousarray(exclude, np.int64)
        self.lib.orc_winding_number(C.byref(self.geom.c), p.ctypes.data_as(C.c_void_p), C.c_int64(len(p)),
                                    ex.ctypes.data_as(C.c_void_p) if ex is not None else None, w.ctypes.data_as(C.c_void_p))
        return w

    def orient_samples(self, tri, bary, h_scale=1.0):
        """(outward normal [n,3], d [n]) of boundary samples by the winding-number rule G-R1."""
        tri = np.ascontiguousarray(tri, np.int32)
        bary = np.ascontiguousarray(bary, np.float32)
        nrm = np.empty((len(tri), 3))
        d = np.empty(len(tri))
        self.lib.orc_orient_samples(C.byref(self.geom.c), tri.ctypes.data_as(C.c_void_p), bary.ctypes.data_as(C.c_void_p),
                                    C.c_int64(len(tri)), C.c_double(h_scale), nrm.ctypes.data_as(C.c_void_p),
                                    d.ctypes.data_as(C.c_void_p))
        return nrm, d

    def knn_weights(self, basis: "PointBasis", q, nq):
        """(idx [n,k], w [n,k]) of the k-NN bilateral interpolator at points q with normals nq (Eq. 44-45)."""
        pb = basis.c()
        q = np.ascontiguousarray(q, np.float64).reshape(-1, 3)
        nq = np.ascontiguousarray(nq, np.float64).reshape(-1, 3)
        idx = np.empty((len(q), basis.k), np.int64)
        w = np.empty((len(q), basis.k))
        for i in range(len(q)):
            self.lib.orc_knn_weights(C.byref(pb), q[i].ctypes.data_as(C.c_void_p), nq[i].ctypes.data_as(C.c_void_p),
                                     idx[i].ctypes.data_as(C.c_void_p), w[i].ctypes.data_as(C.c_void_p))
        return idx, w

    def accumulate_points(self, basis: "PointBasis", rec, tri=None, bary=None, weight=None, normal=None, pos=None,
                          want_var=False):
        pb = basis.c()
        K = len(basis.points)
        rec = np.ascontiguousarray(rec)
        weight = np.ascontiguousarray(weight, np.float32)
        if self.geom.c.kind == 0:
            tri = np.ascontiguousarray(tri, np.int32)
            bary = np.ascontiguousarray(bary, np.float32)
        else:
            pos = np.ascontiguousarray(pos, np.float64)
        if normal is not None:
            normal = np.ascontiguousarray(normal, np.float32)
        S = np.zeros((K, K))
        S2 = np.zeros((K, K)) if want_var else None
        ptr = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        self.lib.orc_accumulate_points(C.byref(self.geom.c), C.byref(pb), ptr(rec), C.c_int64(len(rec)), ptr(tri), ptr(bary),
                                       ptr(weight), ptr(normal), ptr(pos), ptr(S), ptr(S2))
        return (S, S2) if want_var else S

    def estimate_dtn_points(self, basis: "PointBasis", params: OracleParams, exterior: bool, tri, bary, weight,
                            normal=None, want_var=False):
        """Dense DtN matrix in the point basis (K = number of points) plus records."""
        rec, balls = self.run_walks(params, exterior, tri, bary, weight, normal)
        out = self.accumulate_points(basis, rec, tri, bary, weight, normal, want_var=want_var)
        S, var = out if want_var else (out, None)
        return dict(S=S, var=var, records=rec, balls=balls)

    def estimate_dtn(self, params: OracleParams, exterior: bool, tri, bary, weight, normal=None,
                     want_var=False):
        """Dense hat-basis DtN matrix (Alg. 2 / Eq. 32) plus records and balls."""
        rec, balls = self.run_walks(params, exterior, tri, bary, weight, normal)
        out = self.accumulate_hat(rec, tri, bary, want_var, naive=(params.estimator == 1 and not exterior))
        S, var = out if want_var else (out, None)
        return dict(S=S, var=var, records=rec, balls=balls)

    @property
    def num_threads(self):
        return self.lib.orc_num_threads()


def steklov_eigs(S, M, k):
    """Smallest k generalised eigenvalues of S psi = lambda M psi.
    A library routine (LAPACK through scipy) serves as this step."""
    import scipy.linalg as sla
    Ssym = 0.5 * (S + S.T)
    w = sla.eigh(Ssym, M, eigvals_only=True, subset_by_index=[0, min(k, len(S)) - 1])
    return w


def steklov_eigpairs(S, mass, k):
    """Smallest k eigenpairs of S psi = lambda diag(mass) psi (lumped boundary mass), fp64.
    Returns (lambda [k] ascending, psi [k][K] with psi_i^T M psi_j = delta_ij).  LAPACK (scipy) serves as the step."""
    import scipy.linalg as sla
    S = np.asarray(S, dtype=np.float64)
    mass = np.asarray(mass, dtype=np.float64)
    w, V = sla.eigh(0.5 * (S + S.T), np.diag(mass), subset_by_index=[0, min(k, len(S)) - 1])
    return w, V.T.copy()

