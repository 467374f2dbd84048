"""ctypes marshalling for oracle/pct_oracle.c (argument conversion only; no arithmetic here)."""
import ctypes as C
import hashlib
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pct_oracle.c")
_SO = os.path.join(_HERE, "libpct_oracle.so")
_STAMP = _SO + ".stamp"


def _flags():
    flags = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11"]
    try:
        with open("/proc/cpuinfo") as f:
            if " fma " in f.read().replace("\n", " "):
                flags.append("-mfma")  # fmaf() -> one vfmadd; without it glibc's exact fmaf is called
    except OSError:
        pass
    # ORACLE_SANITIZE=1: AddressSanitizer + UndefinedBehaviorSanitizer build of the checker (run the CPU tests with
    # LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0; profiles/r2_sanitizers.md)
    if os.environ.get("ORACLE_SANITIZE"):
        flags += ["-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"]
    return flags


def build(force=False):
    """Compile pct_oracle.c -> libpct_oracle.so with gcc (rebuilds when source or flags change)."""
    flags = _flags()
    with open(_SRC, "rb") as f:
        tag = hashlib.sha256(f.read() + " ".join(flags).encode()).hexdigest()
    if not force and os.path.exists(_SO) and os.path.exists(_STAMP):
        with open(_STAMP) as f:
            if f.read().strip() == tag:
                return _SO
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.run(["gcc", *flags, "-o", tmp, _SRC, "-lm"], check=True)
    os.replace(tmp, _SO)
    with open(_STAMP, "w") as f:
        f.write(tag)
    return _SO


class _Geom(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("h", C.c_float),
                ("u_in", C.c_float), ("u_out", C.c_float)]


class _Hist(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("t_in", "v_in", "t_out", "v_out", "tht_in", "thv_in",
                                         "tht_out", "thv_out", "cs", "sn")]


_FP = C.POINTER(C.c_float)


class _Histories(C.Structure):
    _fields_ = [(n, _FP) for n in ("t_in", "v_in", "t_out", "v_out", "tht_in", "thv_in", "tht_out",
                                   "thv_out", "wepl")] + [
        ("proj", C.POINTER(C.c_uint16)), ("proj_cos", _FP), ("proj_sin", _FP), ("n_proj", C.c_int)]


@dataclass
class Geometry:
    nx: int
    ny: int
    nz: int
    h: float
    u_in: float
    u_out: float

    def c(self):
        return _Geom(self.nx, self.ny, self.nz, self.h, self.u_in, self.u_out)

    @property
    def nmin(self):
        return min(self.nx, self.ny)

    @property
    def n_voxels(self):
        return self.nx * self.ny * self.nz


_FIELDS = ("t_in", "v_in", "t_out", "v_out", "tht_in", "thv_in", "tht_out", "thv_out", "wepl")


class Histories:
    """Host SoA histories: dict of float32 arrays (+ uint16 proj, float32 cos/sin tables)."""

    def __init__(self, arrays):
        self.a = {k: np.ascontiguousarray(arrays[k], dtype=np.float32) for k in _FIELDS}
        self.proj = np.ascontiguousarray(arrays["proj"], dtype=np.uint16)
        self.proj_cos = np.ascontiguousarray(arrays["proj_cos"], dtype=np.float32)
        self.proj_sin = np.ascontiguousarray(arrays["proj_sin"], dtype=np.float32)
        self.n = int(self.proj.shape[0])

    def c(self):
        s = _Histories()
        for k in _FIELDS:
            setattr(s, k, self.a[k].ctypes.data_as(_FP))
        s.proj = self.proj.ctypes.data_as(C.POINTER(C.c_uint16))
        s.proj_cos = self.proj_cos.ctypes.data_as(_FP)
        s.proj_sin = self.proj_sin.ctypes.data_as(_FP)
        s.n_proj = int(self.proj_cos.shape[0])
        return s

    def hist(self, i):
        p = min(int(self.proj[i]), int(self.proj_cos.shape[0]) - 1)  # DESIGN.md R24: clamped, as load_hist does in C
        return _Hist(*[float(self.a[k][i]) for k in _FIELDS[:8]], float(self.proj_cos[p]),
                     float(self.proj_sin[p]))


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        L.orc_mlp_matrix_f64.argtypes = [C.c_double, C.c_double, dp, dp, dp, C.c_int, dp]
        L.orc_mlp_chi2_f64.argtypes = [C.c_double, C.c_double, dp, dp, dp, C.c_int]
        L.orc_mlp_chi2_f64.restype = C.c_double
        L.orc_scatter_f.argtypes = [C.c_double]
        L.orc_scatter_f.restype = C.c_double
        L.orc_sigma_f64.argtypes = [C.c_double, C.c_double, dp, dp]
        L.orc_sigma_f64.restype = None
        L.orc_path_f64.argtypes = [C.POINTER(_Geom), C.POINTER(_Hist), C.c_int, dp, dp]
        L.orc_sigma1_table.argtypes = [C.c_float, C.c_int, _FP, _FP, _FP]
        L.orc_rule_log.argtypes = [C.c_float]
        L.orc_rule_log.restype = C.c_float
        L.orc_row_f32.argtypes = [C.POINTER(_Geom), C.POINTER(_Hist), _FP, _FP, _FP, C.c_int, ip, _FP,
                                  ip, _FP, _FP, _FP, C.POINTER(C.c_int)]
        L.orc_block_accumulate.argtypes = [C.POINTER(_Geom), C.POINTER(_Histories), C.c_int64,
                                           C.c_int64, dp, dp, ip, C.POINTER(C.c_int64), C.c_int]
        L.orc_drop_iterate.argtypes = [C.POINTER(_Geom), C.POINTER(_Histories), C.c_int64, C.c_double,
                                       C.c_int64, C.c_int, dp, C.POINTER(C.c_int64), C.c_int]
        L.orc_carp_iterate.argtypes = [C.POINTER(_Geom), C.POINTER(_Histories), C.c_int64, C.c_double,
                                       C.c_int64, C.c_int, C.c_int, dp, C.c_int]
        L.orc_num_threads.restype = C.c_int
        L.orc_set_path_model.argtypes = [C.c_int]
        L.orc_set_path_model.restype = None
        L.orc_get_path_model.restype = C.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def mlp_matrix_f64(s1, L, y0, y2, a_mm=None, use_log=True):
    y0 = np.asarray(y0, dtype=np.float64)
    y2 = np.asarray(y2, dtype=np.float64)
    out = np.zeros(2)
    ap = None
    if a_mm is not None:
        a = np.ascontiguousarray(a_mm, dtype=np.float64)
        assert a.shape == (6,)
        ap = _dp(a)
    rc = lib().orc_mlp_matrix_f64(float(s1), float(L), _dp(y0), _dp(y2), ap, int(bool(use_log)), _dp(out))
    if rc:
        raise ValueError("s1 must lie strictly inside (0, L)")
    return out


def mlp_chi2_f64(s1, L, y0, y2, y1, use_log=True):
    y0, y2, y1 = (np.asarray(v, dtype=np.float64) for v in (y0, y2, y1))
    return lib().orc_mlp_chi2_f64(float(s1), float(L), _dp(y0), _dp(y2), _dp(y1), int(bool(use_log)))


def scatter_f(s_mm):
    return lib().orc_scatter_f(float(s_mm))


def sigma_f64(s1, L):
    a, b = np.zeros(3), np.zeros(3)
    lib().orc_sigma_f64(float(s1), float(L), _dp(a), _dp(b))
    return a, b


def rule_log(x):
    return float(lib().orc_rule_log(float(np.float32(x))))


def sigma1_table(h, kmax):
    p = [np.zeros(kmax + 1, dtype=np.float32) for _ in range(3)]
    lib().orc_sigma1_table(float(h), int(kmax), *[a.ctypes.data_as(_FP) for a in p])
    return p


def path_f64(geom, hist):
    """T64 nodes (n,3) float64 in the object frame and hull tuple (u0,t0,v0,u2,t2,v2,L); (None, None) if skipped."""
    n = get_substeps() * geom.nmin + 3
    nodes = np.zeros((n, 3))
    hull = np.zeros(7)
    g, h = geom.c(), hist
    rc = lib().orc_path_f64(C.byref(g), C.byref(h), n, _dp(nodes), _dp(hull))
    if rc < 0:
        raise RuntimeError("node buffer too small: need %d" % -rc)
    if rc == 0:
        return None, None
    return nodes[:rc].copy(), hull


def row_f32(geom, hist, table=None):
    """One history through the fp32 rule.  Returns dict(nnz,row_idx,row_len,seg_idx,seg_len,nodes,coefs)."""
    if table is None:
        table = sigma1_table(geom.h / get_substeps(), get_substeps() * geom.nmin)
    ms = get_substeps() * geom.nmin + 2
    cap = ms if get_walk_mode() == 0 else 8 * ms
    row_idx = np.zeros(cap, dtype=np.int32)
    row_len = np.zeros(cap, dtype=np.float32)
    seg_idx = np.zeros(cap, dtype=np.int32)
    seg_len = np.zeros(cap, dtype=np.float32)
    nodes = np.zeros((ms + 1, 3), dtype=np.float32)
    coefs = np.zeros((ms + 1, 2), dtype=np.float32)
    nseg = C.c_int(0)
    ip = C.POINTER(C.c_int32)
    g, h = geom.c(), hist
    rc = lib().orc_row_f32(C.byref(g), C.byref(h), *[a.ctypes.data_as(_FP) for a in table], cap,
                           row_idx.ctypes.data_as(ip), row_len.ctypes.data_as(_FP),
                           seg_idx.ctypes.data_as(ip), seg_len.ctypes.data_as(_FP),
                           nodes.ctypes.data_as(_FP), coefs.ctypes.data_as(_FP), C.byref(nseg))
    if rc < 0:
        raise RuntimeError("segment buffer too small: need %d" % -rc)
    ns = nseg.value  # items of the row before merging: segments (midpoint rule) or pieces (exact traversal)
    nn = int(lib().orc_node_count(C.byref(g), C.byref(h))) if ns else 0
    return dict(nnz=rc, nseg=ns, row_idx=row_idx[:rc].copy(), row_len=row_len[:rc].copy(),
                seg_idx=seg_idx[:ns].copy(), seg_len=seg_len[:ns].copy(),
                nodes=nodes[:nn].copy(), coefs=coefs[:nn].copy())


def block_accumulate(geom, hists, first, count, x, nthreads=0):
    """Delta (float64[M]) and c (int32[M]) of one DROP block against image x; stats=(rows,nnz,segments)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    M = geom.n_voxels
    assert x.shape == (M,)
    delta = np.zeros(M)
    cnt = np.zeros(M, dtype=np.int32)
    stats = (C.c_int64 * 3)()
    g, hs = geom.c(), hists.c()
    rc = lib().orc_block_accumulate(C.byref(g), C.byref(hs), int(first), int(count), _dp(x), _dp(delta),
                                    cnt.ctypes.data_as(C.POINTER(C.c_int32)), stats, int(nthreads))
    if rc:
        raise RuntimeError("orc_block_accumulate failed: %d" % rc)
    return delta, cnt, tuple(stats)


def drop_iterate(geom, hists, lam, block_size, n_iter, x, n=None, nthreads=0):
    """n_iter DROP sweeps in place on x (float64[M]); returns (x, (rows, nnz) of the last sweep)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.shape == (geom.n_voxels,)
    stats = (C.c_int64 * 2)()
    g, hs = geom.c(), hists.c()
    rc = lib().orc_drop_iterate(C.byref(g), C.byref(hs), int(hists.n if n is None else n), float(lam),
                                int(block_size), int(n_iter), _dp(x), stats, int(nthreads))
    if rc:
        raise RuntimeError("orc_drop_iterate failed: %d" % rc)
    return x, tuple(stats)


def carp_iterate(geom, hists, lam, block_size, n_iter, n_strings, x, n=None, nthreads=0):
    """n_iter CARP iterations in place on x (float64[M]): n_strings strings from a common
    x0, each one DROP sweep over its own histories, then the mean of the string solutions."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    assert x.shape == (geom.n_voxels,)
    g, hs = geom.c(), hists.c()
    rc = lib().orc_carp_iterate(C.byref(g), C.byref(hs), int(hists.n if n is None else n), float(lam),
                                int(block_size), int(n_iter), int(n_strings), _dp(x), int(nthreads))
    if rc:
        raise RuntimeError("orc_carp_iterate failed: %d" % rc)
    return x


def set_path_model(model):
    """0: most-likely path (default), 1: cubic spline through the hull points (R30).  Process-wide."""
    lib().orc_set_path_model(int(model))


def get_path_model():
    return int(lib().orc_get_path_model())


def num_threads():
    return int(lib().orc_num_threads())


def xyz_to_beam_f32(u_pl, x, y, z, tht, thv, proj, proj_cos, proj_sin):
    """Object-frame tracker hits -> (t, v) at the tracker plane u_pl, fp32 rule (R32)."""
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    x, y, z, tht, thv, pc, ps = (f32(a) for a in (x, y, z, tht, thv, proj_cos, proj_sin))
    proj = np.ascontiguousarray(proj, dtype=np.uint16)
    n = x.shape[0]
    t = np.zeros(n, dtype=np.float32)
    v = np.zeros(n, dtype=np.float32)
    fp = lambda a: a.ctypes.data_as(_FP)
    L = lib()
    L.orc_xyz_to_beam_f32.argtypes = [C.c_float, C.c_int] + [_FP] * 5 + [C.POINTER(C.c_uint16), _FP, _FP, C.c_int, _FP, _FP]
    L.orc_xyz_to_beam_f32.restype = None
    L.orc_xyz_to_beam_f32(float(u_pl), n, fp(x), fp(y), fp(z), fp(tht), fp(thv), proj.ctypes.data_as(C.POINTER(C.c_uint16)),
                          fp(pc), fp(ps), int(pc.shape[0]), fp(t), fp(v))
    return t, v


def xyz_to_beam_f64(u_pl, x, y, z, tht, thv, cs, sn):
    out = np.zeros(2)
    L = lib()
    L.orc_xyz_to_beam_f64.argtypes = [C.c_double] * 8 + [C.POINTER(C.c_double)]
    L.orc_xyz_to_beam_f64.restype = None
    L.orc_xyz_to_beam_f64(float(u_pl), float(x), float(y), float(z), float(tht), float(thv), float(cs), float(sn), _dp(out))
    return out


def set_substeps(n):
    """1: depth step = one voxel edge (R9, default); 2: half-voxel step (R33).  Process-wide, like the path model."""
    lib().orc_set_substeps(int(n))


def get_substeps():
    return int(lib().orc_get_substeps())


def set_walk_mode(mode):
    """0: midpoint rule (R10, default); 1: exact traversal of the polyline (R34).  Process-wide."""
    lib().orc_set_walk_mode(int(mode))


def get_walk_mode():
    return int(lib().orc_get_walk_mode())
