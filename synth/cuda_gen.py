"""CUDA generator of the synthetic histories (same recipe as generate.py, DESIGN.md "Synthetic
inputs"), for the workloads too large for numpy.  Input generation only -- no reconstruction
arithmetic.  Fills torch CUDA tensors in place; returns a dict keyed like generate_numpy."""
import ctypes as C
import hashlib
import os
import shutil
import subprocess

import numpy as np

from .generate import FIELDS, angle_table

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "csrc", "synth_gen.cu")
_SO = os.path.join(_HERE, "libpct_synth.so")
_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
          "-shared", "-cudart", "static"]
_lib = None


def build(force=False):
    with open(_SRC, "rb") as f:
        tag = hashlib.sha256(f.read() + " ".join(_FLAGS).encode()).hexdigest()
    stamp = _SO + ".stamp"
    if not force and os.path.exists(_SO) and os.path.exists(stamp) and open(stamp).read().strip() == tag:
        return _SO
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.run([nvcc, *_FLAGS, "-o", tmp, _SRC], check=True)
    os.replace(tmp, _SO)
    with open(stamp, "w") as f:
        f.write(tag)
    return _SO


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            build()
        _lib = C.CDLL(_SO)
        _lib.synth_generate.argtypes = [C.c_longlong, C.c_longlong, C.c_ulonglong, C.c_int, C.c_int, C.c_int, C.c_float,
                                        C.c_float, C.c_float, C.c_float, C.c_void_p, C.POINTER(C.c_void_p), C.c_void_p,
                                        C.c_void_p]
    return _lib


def generate_cuda(cfg, n=None, noise=True, device="cuda", first=0):
    """Histories [first, first+n) of cfg as CUDA tensors (float32 fields, int16-viewed uint16 proj) + fp32 tables."""
    import torch

    n = cfg.n if n is None else int(n)
    lib = _load()
    out = {k: torch.empty(n, dtype=torch.float32, device=device) for k in FIELDS}
    proj = torch.empty(n, dtype=torch.int16, device=device)
    shapes = np.minimum(np.asarray(cfg.shapes, dtype=np.float64), 1.0e30).astype(np.float32)
    shapes_dev = torch.from_numpy(shapes).to(device)
    ptrs = (C.c_void_p * 9)(*[out[k].data_ptr() for k in FIELDS])
    stream = torch.cuda.current_stream().cuda_stream
    chunk = 1 << 26
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        sub = (C.c_void_p * 9)(*[ptrs[j] + 4 * s for j in range(9)])
        rc = lib.synth_generate(first + s, m, cfg.seed, cfg.n_angles, shapes.shape[0], int(round(cfg.u_out - cfg.u_in)),
                                0.5 * cfg.nx * cfg.h, 0.5 * cfg.nz * cfg.h, cfg.u_in, cfg.wepl_noise if noise else 0.0,
                                shapes_dev.data_ptr(), sub, proj.data_ptr() + 2 * s, stream)
        if rc:
            raise RuntimeError("synth_generate failed: %d" % rc)
    torch.cuda.synchronize()
    cs, sn = angle_table(cfg.n_angles)
    out["proj"] = proj
    out["proj_cos"] = torch.from_numpy(cs).to(device)
    out["proj_sin"] = torch.from_numpy(sn).to(device)
    return out
