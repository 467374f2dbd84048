"""ctypes binding of libpct.so with the names of include/pct.h.

Argument marshalling only: every step of the path (hull, MLP, voxel walk, DROP update) runs in the
CUDA kernels of the library.  There is no CPU fallback: if the library cannot be built or loaded
the import fails loudly.  torch appears only as the provider of device memory and streams
(``tensor.data_ptr()``, ``torch.cuda.current_stream().cuda_stream``).
"""
import ctypes as C
import os

from . import _build

PCT_OK, PCT_EINVAL, PCT_ENOMEM, PCT_ECUDA, PCT_ESTATE, PCT_EINTERNAL = 0, -1, -2, -3, -4, -5
_STATUS = {0: "PCT_OK", -1: "PCT_EINVAL", -2: "PCT_ENOMEM", -3: "PCT_ECUDA", -4: "PCT_ESTATE", -5: "PCT_EINTERNAL"}

FIELDS = ("entry_t", "entry_v", "exit_t", "exit_v", "entry_dt", "entry_dv", "exit_dt", "exit_dv", "wepl")

_FP = C.POINTER(C.c_float)
_IP = C.POINTER(C.c_int32)


class pct_histories(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in FIELDS] + [("proj", C.c_void_p), ("proj_cos", C.c_void_p),
                                                     ("proj_sin", C.c_void_p), ("n_proj", C.c_int32)]


XYZ_FIELDS = ("entry_x", "entry_y", "entry_z", "exit_x", "exit_y", "exit_z", "entry_dt", "entry_dv", "exit_dt", "exit_dv", "wepl")


class pct_histories_xyz(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in XYZ_FIELDS] + [("proj", C.c_void_p), ("proj_cos", C.c_void_p),
                                                         ("proj_sin", C.c_void_p), ("n_proj", C.c_int32)]


class PctError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("%s: %s" % (_STATUS.get(code, code), msg))
        self.code = code


_lib = None


def lib():
    """Load (building first if needed) libpct.so.  Raises if that is impossible -- no fallback."""
    global _lib
    if _lib is None:
        # always through the stamp check (a cheap no-op when sources and flags are unchanged): a stale
        # binary next to newer sources is rebuilt, never silently loaded
        path = _build.build(force=bool(os.environ.get("PCT_REBUILD")))
        L = C.CDLL(path)
        vp, i64 = C.c_void_p, C.c_int64
        L.pct_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_float, C.c_float, C.c_float, vp]
        L.pct_set_histories.argtypes = [vp, i64, C.POINTER(pct_histories)]
        L.pct_set_histories_host.argtypes = [vp, i64, C.POINTER(pct_histories)]
        L.pct_set_histories_xyz.argtypes = [vp, i64, C.POINTER(pct_histories_xyz)]
        L.pct_iterate.argtypes = [vp, C.c_float, i64, C.c_int]
        L.pct_iterate_carp.argtypes = [vp, C.c_float, i64, C.c_int, C.c_int]
        L.pct_set_path_model.argtypes = [vp, C.c_int]
        L.pct_get_image.argtypes = [vp, vp, i64]
        L.pct_set_image.argtypes = [vp, vp, i64]
        L.pct_synchronize.argtypes = [vp]
        L.pct_get_stats.argtypes = [vp, C.POINTER(i64)]
        L.pct_destroy.argtypes = [vp]
        L.pct_destroy.restype = None
        L.pct_last_error.argtypes = [vp]
        L.pct_last_error.restype = C.c_char_p
        L.pct_version.restype = C.c_char_p
        L.pct_debug_rows.argtypes = [vp, i64, i64, C.c_int32, vp, vp, vp, vp, vp, vp]
        L.pct_debug_block.argtypes = [vp, i64, i64, vp, vp]
        L.pct_profile_sweep.argtypes = [vp, C.c_float, i64, C.POINTER(C.c_float)]
        L.pct_measure_peaks.argtypes = [vp, i64, C.POINTER(C.c_double)]
        L.pct_set_tvs.argtypes = [vp, C.c_float, C.c_float, C.c_int]
        L.pct_set_step.argtypes = [vp, C.c_int]
        L.pct_set_walk.argtypes = [vp, C.c_int]
        L.pct_set_option.argtypes = [vp, C.c_int, C.c_int]
        L.pct_debug_rule_sweep.argtypes = [C.c_int, C.c_uint32, C.c_uint32, C.POINTER(C.c_uint64), vp]
        L.pct_image_storage.argtypes = [vp, C.POINTER(vp), C.POINTER(i64)]
        L.pct_tvs_step.argtypes = [vp]
        L.pct_get_tvs_state.argtypes = [vp, C.POINTER(C.c_double)]
        L.pct_tvs_step_static.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int, vp, vp]
        L.pct_tvs_step_static_error.restype = C.c_char_p
        _lib = L
    return _lib


EXPORTS = ("pct_create", "pct_set_histories", "pct_set_histories_host", "pct_set_histories_xyz", "pct_iterate", "pct_iterate_carp", "pct_set_path_model", "pct_get_image",
           "pct_set_image", "pct_synchronize", "pct_get_stats", "pct_destroy", "pct_last_error", "pct_version",
           "pct_debug_rows", "pct_debug_block", "pct_profile_sweep", "pct_measure_peaks", "pct_set_tvs", "pct_tvs_step", "pct_set_step", "pct_set_walk", "pct_image_storage",
           "pct_get_tvs_state", "pct_tvs_step_static", "pct_tvs_step_static_error", "pct_set_option", "pct_debug_rule_sweep")


def _ptr(a):
    """Address of a torch tensor / numpy array / int / None."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    return a.ctypes.data


def _check(ctx, rc):
    if rc != PCT_OK:
        raise PctError(rc, lib().pct_last_error(ctx).decode())


def pct_version():
    return lib().pct_version().decode()


def pct_create(nx, ny, nz, voxel_mm, tracker_u_in_mm, tracker_u_out_mm, cuda_stream=None):
    """-> opaque context handle (include/pct.h: pct_create)."""
    h = C.c_void_p()
    rc = lib().pct_create(C.byref(h), nx, ny, nz, voxel_mm, tracker_u_in_mm, tracker_u_out_mm, cuda_stream)
    _check(None, rc)
    return h


def _hist_struct(arrays):
    s = pct_histories()
    keep = []
    for k in FIELDS + ("proj", "proj_cos", "proj_sin"):
        a = arrays[k]
        keep.append(a)
        setattr(s, k, _ptr(a))
    s.n_proj = int(arrays["proj_cos"].shape[0])
    return s, keep


def pct_set_histories(ctx, n, arrays):
    """arrays: mapping of CUDA tensors (float32 fields, uint16/int16 proj, float32 cos/sin tables), borrowed."""
    s, _ = _hist_struct(arrays)
    _check(ctx, lib().pct_set_histories(ctx, int(n), C.byref(s)))


def pct_set_histories_host(ctx, n, arrays):
    """arrays: mapping of host arrays (numpy or CPU tensors, ideally pinned); the library copies them."""
    s, _ = _hist_struct(arrays)
    _check(ctx, lib().pct_set_histories_host(ctx, int(n), C.byref(s)))


def pct_set_histories_xyz(ctx, n, arrays):
    """arrays: mapping of CUDA tensors keyed as pct_histories_xyz (object-frame tracker hits + beam-frame slopes)."""
    s = pct_histories_xyz()
    for k in XYZ_FIELDS + ("proj", "proj_cos", "proj_sin"):
        setattr(s, k, _ptr(arrays[k]))
    s.n_proj = int(arrays["proj_cos"].shape[0])
    _check(ctx, lib().pct_set_histories_xyz(ctx, int(n), C.byref(s)))


def pct_iterate(ctx, lam, block_size, n_iter):
    _check(ctx, lib().pct_iterate(ctx, float(lam), int(block_size), int(n_iter)))


def pct_iterate_carp(ctx, lam, block_size, n_iter, n_strings):
    _check(ctx, lib().pct_iterate_carp(ctx, float(lam), int(block_size), int(n_iter), int(n_strings)))


PCT_PATH_MLP, PCT_PATH_SPLINE = 0, 1


def pct_set_path_model(ctx, model):
    _check(ctx, lib().pct_set_path_model(ctx, int(model)))


def pct_get_image(ctx, dst, n_voxels):
    _check(ctx, lib().pct_get_image(ctx, _ptr(dst), int(n_voxels)))


def pct_set_image(ctx, src, n_voxels):
    _check(ctx, lib().pct_set_image(ctx, _ptr(src), int(n_voxels)))


def pct_synchronize(ctx):
    _check(ctx, lib().pct_synchronize(ctx))


def pct_get_stats(ctx):
    out = (C.c_int64 * 4)()
    _check(ctx, lib().pct_get_stats(ctx, out))
    return dict(rows=out[0], nnz=out[1], segments=out[2], histories=out[3])


def pct_destroy(ctx):
    lib().pct_destroy(ctx)


def pct_debug_rows(ctx, first, count, max_seg, nseg, nnz, seg_idx=None, seg_len=None, row_len=None, nodes=None):
    _check(ctx, lib().pct_debug_rows(ctx, int(first), int(count), int(max_seg), _ptr(nseg), _ptr(nnz), _ptr(seg_idx),
                                     _ptr(seg_len), _ptr(row_len), _ptr(nodes)))


def pct_debug_block(ctx, first, count, delta, cnt):
    _check(ctx, lib().pct_debug_block(ctx, int(first), int(count), _ptr(delta), _ptr(cnt)))


def pct_debug_rule_sweep(which, first_bits, last_bits, cuda_stream=None):
    """The rule's 1/a (which=0) or sqrt(a) (which=1) against the IEEE intrinsic on every fp32 bit pattern of the range
    -> (number of mismatches, lowest mismatching pattern)."""
    out = (C.c_uint64 * 2)()
    _check(None, lib().pct_debug_rule_sweep(int(which), int(first_bits), int(last_bits), out, cuda_stream))
    return int(out[0]), int(out[1])


def pct_profile_sweep(ctx, lam, block_size):
    """One sweep with CUDA events around every launch -> dict of device times (include/pct.h)."""
    out = (C.c_float * 6)()
    _check(ctx, lib().pct_profile_sweep(ctx, float(lam), int(block_size), out))
    return dict(accumulate_ms=out[0], update_ms=out[1], sweep_ms=out[2], blocks=int(out[3]), tvs_ms=out[4])


def pct_measure_peaks(footprint_bytes, cuda_stream=None):
    """Micro-benchmarks behind the roofline (include/pct.h: pct_measure_peaks) -> dict."""
    out = (C.c_double * 12)()
    rc = lib().pct_measure_peaks(cuda_stream, int(footprint_bytes), out)
    if rc != PCT_OK:
        raise PctError(rc, "pct_measure_peaks failed")
    return dict(gather_random_per_s=out[0], gather_path_per_s=out[1], red_v2_random_per_s=out[2], stream_read_bytes_per_s=out[3],
                ffma_inst_per_s=out[4], ffma2_inst_per_s=out[5], red_v2_path_per_s=out[6], footprint_bytes=int(out[7]),
                gather_path_tiled_per_s=out[8], red_v2_path_tiled_per_s=out[9], mixed_pairs_tiled_per_s=out[10])


def pct_set_tvs(ctx, beta0, gamma=1.0, n_halvings=4):
    """Total-variation superiorization step before every DROP block / CARP iteration (include/pct.h); beta0 = 0: off."""
    _check(ctx, lib().pct_set_tvs(ctx, float(beta0), float(gamma), int(n_halvings)))


def pct_tvs_step(ctx):
    _check(ctx, lib().pct_tvs_step(ctx))


def pct_get_tvs_state(ctx):
    out = (C.c_double * 6)()
    _check(ctx, lib().pct_get_tvs_state(ctx, out))
    return dict(beta=out[0], tv_before=out[1], tv_after=out[2], level=int(out[3]), steps=int(out[4]), accepted=int(out[5]))


PCT_TVS_STATIC_MAX_SLOTS = 1 << 20


def pct_tvs_step_static(image, nx, ny, nz, beta, n_halvings=4, info=None, cuda_stream=None):
    """One TVS step on a caller-owned CUDA tensor without any device allocation (include/pct.h: pct_tvs_step_static).

    For callers that cannot cudaMalloc while running (all device memory in their own pool, a latency-bound loop, a fixed
    memory budget): the step's working memory is a fixed array inside the library.  image: float32 CUDA tensor of
    nx*ny*nz values, overwritten; info: None or a float64 CUDA tensor of 4 (step used, TV before, TV after, level).
    Calls that may overlap on the GPU share that array and race: keep them on one stream."""
    rc = lib().pct_tvs_step_static(_ptr(image), int(nx), int(ny), int(nz), float(beta), int(n_halvings), _ptr(info), cuda_stream)
    if rc != PCT_OK:
        raise PctError(rc, lib().pct_tvs_step_static_error().decode())


def pct_set_step(ctx, substeps):
    """Depth step of the path: 1 = one voxel edge (default), 2 = half a voxel edge (include/pct.h)."""
    _check(ctx, lib().pct_set_step(ctx, int(substeps)))


def pct_image_storage(ctx):
    """-> (device address, length) of the library's own image array, in its storage order (include/pct.h)."""
    p, n = C.c_void_p(), C.c_int64()
    _check(ctx, lib().pct_image_storage(ctx, C.byref(p), C.byref(n)))
    return int(p.value), int(n.value)


PCT_WALK_MIDPOINT, PCT_WALK_EXACT = 0, 1
PCT_OPT_ORDER, PCT_OPT_ROWS_PAIR = 0, 1


def pct_set_option(ctx, key, value):
    """PCT_OPT_ORDER 0/1/2 (depth-slab order inside a block: never / by footprint / always), PCT_OPT_ROWS_PAIR 0/1."""
    _check(ctx, lib().pct_set_option(ctx, int(key), int(value)))


def pct_set_walk(ctx, mode):
    """PCT_WALK_MIDPOINT (default) or PCT_WALK_EXACT: exact traversal of the path polyline (include/pct.h)."""
    _check(ctx, lib().pct_set_walk(ctx, int(mode)))
