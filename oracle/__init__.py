"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front-end of ``oracle/nbody_oracle.c`` (plain FP64 CPU direct summation written from the
definition; see that file's header for the passages it follows and its pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference`` legs may import
this package.  It imports nothing from ``paper_1504_03687_b200`` and vice versa.

The shared object is compiled with gcc (-O3 -march=native -fopenmp) on the host it runs on; its
file name carries a hash of the host's CPU flags so that a build made on another machine (the
repo snapshot travels to the GPU box) is never loaded by mistake.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "nbody_oracle.c"
_lib = None


def _host_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    h = hashlib.sha1((flags + _SRC.read_text()).encode()).hexdigest()[:12]
    return h


def lib_path() -> Path:
    return _HERE / f"liboracle_{_host_tag()}.so"


def build(force: bool = False) -> Path:
    out = lib_path()
    if out.exists() and not force:
        return out
    tmp = out.with_suffix(f".tmp{os.getpid()}.so")
    cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, out)
    return out


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(str(build()))
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int32)
    lib.orc_num_threads.restype = ctypes.c_int
    lib.orc_predict.restype = None
    lib.orc_predict.argtypes = [ctypes.c_int64, dp, dp, dp, dp, dp, ctypes.c_double, dp, dp]
    lib.orc_regular.restype = ctypes.c_int
    lib.orc_regular.argtypes = [ctypes.c_int64, dp, dp, dp, ctypes.c_int32, ip, dp, ctypes.c_int32,
                                dp, dp, dp, dp, dp, dp, ip, ip, ip]
    lib.orc_band_pairs.restype = ctypes.c_int64
    lib.orc_band_pairs.argtypes = [ctypes.c_int64, dp, dp, dp, ctypes.c_int32, ip, dp, ctypes.c_double,
                                   ctypes.c_int64, ip, ip, dp, dp]
    lib.orc_irregular.restype = ctypes.c_int
    lib.orc_irregular.argtypes = [ctypes.c_int64, dp, dp, dp, dp, dp, dp, ctypes.c_double, ctypes.c_int32, ip, ip, ip,
                                  ctypes.c_int32, dp, dp, dp]
    _lib = lib
    return lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def num_threads() -> int:
    return int(_load().orc_num_threads())


def predict(x0, v0, a0, j0, t0, t: float):
    """All-particle Hermite prediction to time t. Returns xp, vp as [N,3] float64."""
    lib = _load()
    x0, px = _d(x0); v0, pv = _d(v0); a0, pa = _d(a0); j0, pj = _d(j0); t0, pt = _d(t0)
    N = t0.shape[0]
    assert x0.shape == (N, 3) and v0.shape == (N, 3) and a0.shape == (N, 3) and j0.shape == (N, 3)
    xp = np.empty((N, 3)); vp = np.empty((N, 3))
    lib.orc_predict(N, px, pv, pa, pj, pt, float(t), _d(xp)[1], _d(vp)[1])
    return xp, vp


def regular(m, xp, vp, idx_i, h2_i, cap: int, want_list: bool = True) -> dict:
    """Regular force / jerk / potential + neighbour list for the active block."""
    lib = _load()
    m, pm = _d(m); xp, pxp = _d(xp); vp, pvp = _d(vp)
    idx_i, pidx = _i(idx_i); h2_i, ph2 = _d(h2_i)
    N = m.shape[0]; n = idx_i.shape[0]
    assert xp.shape == (N, 3) and vp.shape == (N, 3) and h2_i.shape == (n,)
    out = dict(acc=np.zeros((n, 3)), jerk=np.zeros((n, 3)), pot=np.zeros(n),
               acc_nb=np.zeros((n, 3)), jerk_nb=np.zeros((n, 3)), pot_nb=np.zeros(n),
               nnb=np.zeros(n, np.int32), overflow=np.zeros(n, np.int32),
               nblist=np.full((n, cap), -1, np.int32) if want_list else None)
    pl = _i(out["nblist"])[1] if want_list else None
    rc = lib.orc_regular(N, pm, pxp, pvp, n, pidx, ph2, int(cap),
                         _d(out["acc"])[1], _d(out["jerk"])[1], _d(out["pot"])[1],
                         _d(out["acc_nb"])[1], _d(out["jerk_nb"])[1], _d(out["pot_nb"])[1],
                         _i(out["nnb"])[1], pl, _i(out["overflow"])[1])
    assert rc == 0
    return out


def band_pairs(m, xp, vp, idx_i, h2_i, band: float = 1e-5, max_pairs: int = 1 << 20) -> dict:
    """Pairs with |r2 - h2| < band*h2 and their seven pair terms (north_star: "reported separately")."""
    lib = _load()
    m, pm = _d(m); xp, pxp = _d(xp); vp, pvp = _d(vp)
    idx_i, pidx = _i(idx_i); h2_i, ph2 = _d(h2_i)
    k = np.zeros(max_pairs, np.int32); j = np.zeros(max_pairs, np.int32)
    r2 = np.zeros(max_pairs); terms = np.zeros((max_pairs, 7))
    n = lib.orc_band_pairs(m.shape[0], pm, pxp, pvp, idx_i.shape[0], pidx, ph2, float(band),
                           max_pairs, _i(k)[1], _i(j)[1], _d(r2)[1], _d(terms)[1])
    if n > max_pairs:
        raise RuntimeError(f"{n} band pairs exceed max_pairs={max_pairs}")
    order = np.lexsort((j[:n], k[:n]))
    return dict(k=k[:n][order], j=j[:n][order], r2=r2[:n][order], terms=terms[:n][order])


def irregular(m, x0, v0, a0, j0, t0, t: float, idx_i, nnb, nblist, cap: int) -> dict:
    """Neighbour (irregular) force / jerk / potential over the listed neighbours, each predicted to t
    from the state at its own t0."""
    lib = _load()
    m, pm = _d(m); x0, px = _d(x0); v0, pv = _d(v0); a0, pa = _d(a0); j0, pj = _d(j0); t0, pt = _d(t0)
    idx_i, pidx = _i(idx_i); nnb, pn = _i(nnb); nblist, pl = _i(nblist)
    n = idx_i.shape[0]
    assert nblist.shape == (n, cap) and nnb.shape == (n,)
    out = dict(acc=np.zeros((n, 3)), jerk=np.zeros((n, 3)), pot=np.zeros(n))
    rc = lib.orc_irregular(m.shape[0], pm, px, pv, pa, pj, pt, float(t), n, pidx, pn, pl, int(cap),
                           _d(out["acc"])[1], _d(out["jerk"])[1], _d(out["pot"])[1])
    assert rc == 0
    return out


def regular_step(cfg: dict, want_list: bool = True) -> dict:
    """predict_all(t) + regular for a config dict from nbgen (one pass of the hot path)."""
    xp, vp = predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    out = regular(cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cfg["cap"], want_list)
    out["xp"], out["vp"] = xp, vp
    return out
