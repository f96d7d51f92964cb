"""ctypes binding of libnbreg (same names as include/nbreg.h; marshalling only)."""
from __future__ import annotations

import ctypes
import re
from pathlib import Path

from .build import LIB, build_lib

NB_OK, NB_EINVAL, NB_ESTATE, NB_ENOMEM, NB_ECUDA, NB_EOVERFLOW, NB_ELIMIT = 0, 1, 2, 3, 4, 5, 6
NB_STATIC_MAX_N = 16777216      # include/nbreg.h
INFO = dict(kernel_launches=0, last_jsplit=1, last_iblock=2, last_grid=3, sm_count=4, n_padded=5,
            force_jsplit=16, force_variant=17, last_variant=18, profile=19, force_kernel_ns=20,
            force_kernel_count=21, step_chunks=22, fuse_predict=23, local_g_milli=24, stats=25,
            local_warps=26, total_warps=27, last_fused=28, reorder_min=29, last_reordered=30, speculate=31, spec_hits=32, spec_misses=33, select_chunks=34, irr_pred_min=35, last_block_n=36, select_grid=37,
            force_kernel_ns_at=1000)

_lib = None
_vp = ctypes.c_void_p


class NbregError(RuntimeError):
    def __init__(self, code: int, where: str, detail: str = ""):
        self.code = code
        super().__init__(f"{where}: nbreg status {code} ({detail})")


def declared_symbols() -> list[str]:
    """Every function include/nbreg.h declares (parsed from the header text)."""
    text = (Path(__file__).resolve().parent.parent / "include" / "nbreg.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nb_[a-z_0-9]+)\s*\(", text)))


def load_library(build: bool = True) -> ctypes.CDLL:
    """Load libnbreg.so (building it in-tree with nvcc if stale).  Fails loudly -- no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if build:
        build_lib()
    if not LIB.exists():
        raise RuntimeError(f"{LIB} is missing: the CUDA library was not built and there is no CPU fallback")
    lib = ctypes.CDLL(str(LIB))
    i32, i64, dbl = ctypes.c_int32, ctypes.c_int64, ctypes.c_double
    lib.nb_open.argtypes = [i64, i32, ctypes.POINTER(_vp)]
    lib.nb_close.argtypes = [_vp]
    lib.nb_set_stream.argtypes = [_vp, _vp]
    lib.nb_synchronize.argtypes = [_vp]
    lib.nb_set_j.argtypes = [_vp] + [_vp] * 6
    lib.nb_set_j_host.argtypes = [_vp] + [_vp] * 6
    lib.nb_predict_all.argtypes = [_vp, dbl]
    lib.nb_get_predicted.argtypes = [_vp, _vp, _vp]
    lib.nb_regular.argtypes = [_vp, i32] + [_vp] * 8
    lib.nb_regular_host.argtypes = [_vp, i32] + [_vp] * 8
    lib.nb_regular_all.argtypes = [_vp] + [_vp] * 7
    lib.nb_step_host.argtypes = [_vp] + [_vp] * 6 + [dbl, i32] + [_vp] * 8
    lib.nb_update_j.argtypes = [_vp, i32] + [_vp] * 7
    lib.nb_irregular.argtypes = [_vp, dbl, i32] + [_vp] * 6
    lib.nb_set_steps.argtypes = [_vp, _vp]
    lib.nb_init_steps.argtypes = [_vp, dbl, dbl]
    lib.nb_next_block.argtypes = [_vp, ctypes.POINTER(dbl), ctypes.POINTER(i32), _vp]
    lib.nb_next_block_static.argtypes = [i64, _vp, _vp, _vp, _vp, _vp]
    lib.nb_correct.argtypes = [_vp, dbl, i32, _vp, _vp, _vp, dbl, dbl]
    lib.nb_get_state.argtypes = [_vp] + [_vp] * 7
    lib.nb_block_step.argtypes = [_vp, _vp, dbl, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(i32)]
    lib.nb_get_block.argtypes = [_vp, i32] + [_vp] * 7
    lib.nb_ac_init.argtypes = [_vp, dbl, _vp, dbl, dbl, ctypes.POINTER(i32)]
    lib.nb_ac_step.argtypes = [_vp, dbl, dbl, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(i32), ctypes.POINTER(i32)]
    lib.nb_ac_get.argtypes = [_vp] + [_vp] * 10
    lib.nb_ac_set_radii.argtypes = [_vp, i32, _vp, _vp]
    lib.nb_ac_get_failed.argtypes = [_vp, i32, ctypes.POINTER(i32), _vp, _vp]
    lib.nb_ac_run.argtypes = [_vp, dbl, dbl, dbl, dbl, i64, ctypes.POINTER(dbl)] + [ctypes.POINTER(i64)] * 3
    lib.nb_run_blocks.argtypes = [_vp, _vp, dbl, dbl, dbl, i64, ctypes.POINTER(dbl)] + [ctypes.POINTER(i64)] * 2
    lib.nb_set_j_offset.argtypes = [_vp, i64]
    lib.nb_regular_shard.argtypes = [_vp, dbl, i32] + [_vp] * 9
    lib.nb_plan_regular.argtypes = [i64, i64, i32, i32] + [ctypes.POINTER(i32)] * 4
    lib.nb_plan_chunks.argtypes = [i64, i32, ctypes.POINTER(i64), ctypes.POINTER(i32)]
    lib.nb_get_info.argtypes = [_vp, i32, ctypes.POINTER(i64)]
    lib.nb_set_tuning.argtypes = [_vp, i32, i64]
    lib.nb_last_cuda_error.argtypes = [_vp]
    lib.nb_strerror.argtypes = [ctypes.c_int]
    lib.nb_strerror.restype = ctypes.c_char_p
    for name in declared_symbols():
        fn = getattr(lib, name)             # AttributeError if the .so does not export it
        if name != "nb_strerror":
            fn.restype = ctypes.c_int
    _lib = lib
    return lib


def exported_symbols() -> list[str]:
    lib = load_library()
    return [n for n in declared_symbols() if hasattr(lib, n)]


def _check(rc: int, where: str, ctx=None):
    if rc != NB_OK:
        lib = load_library()
        detail = lib.nb_strerror(rc).decode()
        if ctx is not None and rc == NB_ECUDA:
            detail += f"; cudaError={lib.nb_last_cuda_error(ctx)}"
        raise NbregError(rc, where, detail)


def _dev_ptr(t, dtype, numel, name):
    import torch
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise ValueError(f"{name}: need contiguous {dtype} with {numel} elements, got {t.dtype} {tuple(t.shape)}")
    return _vp(t.data_ptr())


def _host_ptr(a, dtype, numel, name):
    import numpy as np
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda:
            raise TypeError(f"{name}: expected host memory")
        a = a.numpy()
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous or a.size != numel:
        raise ValueError(f"{name}: need C-contiguous {dtype} with {numel} elements")
    return _vp(a.ctypes.data)


class NbContext:
    """Owns one nb_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, N: int, nb_cap: int, stream=None):
        self._lib = load_library()
        self._ctx = _vp()
        self.N, self.cap = int(N), int(nb_cap)
        rc = self._lib.nb_open(self.N, self.cap, ctypes.byref(self._ctx))
        if rc != NB_OK:
            ctx, self._ctx = self._ctx, _vp()
            err = self._lib.nb_last_cuda_error(ctx) if ctx else 0
            if ctx:
                self._lib.nb_close(ctx)
            raise NbregError(rc, "nb_open", self._lib.nb_strerror(rc).decode() + f"; cudaError={err}")
        if stream is not None:
            self.set_stream(stream)

    # -- lifetime
    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.nb_close(self._ctx)
            self._ctx = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- plumbing
    def set_stream(self, stream):
        handle = stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)
        _check(self._lib.nb_set_stream(self._ctx, _vp(handle)), "nb_set_stream", self._ctx)

    def synchronize(self):
        _check(self._lib.nb_synchronize(self._ctx), "nb_synchronize", self._ctx)

    def info(self, key: str, index: int = 0) -> int:
        v = ctypes.c_int64()
        _check(self._lib.nb_get_info(self._ctx, INFO[key] + int(index), ctypes.byref(v)), "nb_get_info")
        return v.value

    def tune(self, key: str, value: int):
        _check(self._lib.nb_set_tuning(self._ctx, INFO[key], int(value)), "nb_set_tuning")

    # -- the path (device tensors)
    def set_j(self, m, x0, v0, a0, j0, t0):
        import torch
        N, f8 = self.N, torch.float64
        args = [_dev_ptr(m, f8, N, "m"), _dev_ptr(x0, f8, 3 * N, "x0"), _dev_ptr(v0, f8, 3 * N, "v0"),
                _dev_ptr(a0, f8, 3 * N, "a0"), _dev_ptr(j0, f8, 3 * N, "j0"), _dev_ptr(t0, f8, N, "t0")]
        _check(self._lib.nb_set_j(self._ctx, *args), "nb_set_j", self._ctx)

    def update_j(self, idx, m, x0, v0, a0, j0, t0):
        import torch
        n, f8 = int(idx.numel()), torch.float64
        if n == 0:
            return
        args = [_dev_ptr(idx, torch.int32, n, "idx"), _dev_ptr(m, f8, n, "m"), _dev_ptr(x0, f8, 3 * n, "x0"),
                _dev_ptr(v0, f8, 3 * n, "v0"), _dev_ptr(a0, f8, 3 * n, "a0"), _dev_ptr(j0, f8, 3 * n, "j0"),
                _dev_ptr(t0, f8, n, "t0")]
        _check(self._lib.nb_update_j(self._ctx, n, *args), "nb_update_j", self._ctx)

    def irregular(self, t: float, idx_i, nnb, nblist, acc, jerk, pot=None):
        import torch
        n, f8, i4 = int(idx_i.numel()), torch.float64, torch.int32
        if n == 0:
            return
        args = [_dev_ptr(idx_i, i4, n, "idx_i"), _dev_ptr(nnb, i4, n, "nnb"),
                _dev_ptr(nblist, i4, n * self.cap, "nblist"), _dev_ptr(acc, f8, 3 * n, "acc"),
                _dev_ptr(jerk, f8, 3 * n, "jerk"), _vp() if pot is None else _dev_ptr(pot, f8, n, "pot")]
        _check(self._lib.nb_irregular(self._ctx, float(t), n, *args), "nb_irregular", self._ctx)

    def predict_all(self, t: float):
        _check(self._lib.nb_predict_all(self._ctx, float(t)), "nb_predict_all", self._ctx)

    def get_predicted(self, xp, vp):
        import torch
        _check(self._lib.nb_get_predicted(self._ctx, _dev_ptr(xp, torch.float64, 3 * self.N, "xp"),
                                          _dev_ptr(vp, torch.float64, 3 * self.N, "vp")),
               "nb_get_predicted", self._ctx)

    def regular(self, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow):
        import torch
        n = int(idx_i.numel())
        f8, i4 = torch.float64, torch.int32
        if n == 0:
            _check(self._lib.nb_regular(self._ctx, 0, *([_vp()] * 8)), "nb_regular", self._ctx)
            return
        args = [_dev_ptr(idx_i, i4, n, "idx_i"), _dev_ptr(h2_i, f8, n, "h2_i"), _dev_ptr(acc, f8, 3 * n, "acc"),
                _dev_ptr(jerk, f8, 3 * n, "jerk"), _dev_ptr(pot, f8, n, "pot"), _dev_ptr(nnb, i4, n, "nnb"),
                _dev_ptr(nblist, i4, n * self.cap, "nblist"), _dev_ptr(overflow, i4, n, "overflow")]
        _check(self._lib.nb_regular(self._ctx, n, *args), "nb_regular", self._ctx)

    def regular_all(self, h2, acc, jerk, pot, nnb, nblist, overflow):
        """Full-N pass (identity block); nblist may be None: neighbours are counted, not stored."""
        import torch
        n, f8, i4 = self.N, torch.float64, torch.int32
        args = [_dev_ptr(h2, f8, n, "h2"), _dev_ptr(acc, f8, 3 * n, "acc"), _dev_ptr(jerk, f8, 3 * n, "jerk"),
                _dev_ptr(pot, f8, n, "pot"), _dev_ptr(nnb, i4, n, "nnb"),
                _vp() if nblist is None else _dev_ptr(nblist, i4, n * self.cap, "nblist"),
                _dev_ptr(overflow, i4, n, "overflow")]
        _check(self._lib.nb_regular_all(self._ctx, *args), "nb_regular_all", self._ctx)

    # -- block loop
    def set_steps(self, dt):
        import torch
        _check(self._lib.nb_set_steps(self._ctx, _dev_ptr(dt, torch.float64, self.N, "dt")), "nb_set_steps", self._ctx)

    def init_steps(self, eta_s: float, dt_max: float):
        _check(self._lib.nb_init_steps(self._ctx, float(eta_s), float(dt_max)), "nb_init_steps", self._ctx)

    def next_block(self, idx_act):
        """-> (t_next, n_act); idx_act (int32 CUDA tensor with room for N) receives the active indices."""
        import torch
        t, n = ctypes.c_double(), ctypes.c_int32()
        _check(self._lib.nb_next_block(self._ctx, ctypes.byref(t), ctypes.byref(n),
                                       _dev_ptr(idx_act, torch.int32, self.N, "idx_act")), "nb_next_block", self._ctx)
        return t.value, n.value

    def correct(self, t: float, idx, acc1, jerk1, eta: float, dt_max: float):
        import torch
        n, f8 = int(idx.numel()), torch.float64
        if n == 0:
            return
        _check(self._lib.nb_correct(self._ctx, float(t), n, _dev_ptr(idx, torch.int32, n, "idx"),
                                    _dev_ptr(acc1, f8, 3 * n, "acc1"), _dev_ptr(jerk1, f8, 3 * n, "jerk1"),
                                    float(eta), float(dt_max)), "nb_correct", self._ctx)

    def block_step(self, h2_all, eta: float, dt_max: float, t_stop: float = float("inf")):
        """nb_block_step -> (t_next, n_act); h2_all: float64 CUDA tensor [N] indexed by body, or None."""
        import torch
        t, n = ctypes.c_double(), ctypes.c_int32()
        h2 = _vp() if h2_all is None else _dev_ptr(h2_all, torch.float64, self.N, "h2_all")
        t_stop = min(float(t_stop), 1.7976931348623157e308)
        _check(self._lib.nb_block_step(self._ctx, h2, float(eta), float(dt_max), t_stop, ctypes.byref(t),
                                       ctypes.byref(n)), "nb_block_step", self._ctx)
        return t.value, n.value

    def get_block(self, n: int, want_list: bool = False) -> dict:
        """nb_get_block: the last block's results (n = the n_act block_step returned) as new CUDA tensors."""
        import torch
        f8, i4, dev = torch.float64, torch.int32, "cuda"
        out = dict(idx_act=torch.empty(n, dtype=i4, device=dev), acc=torch.empty((n, 3), dtype=f8, device=dev),
                   jerk=torch.empty((n, 3), dtype=f8, device=dev), pot=torch.empty(n, dtype=f8, device=dev),
                   nnb=torch.empty(n, dtype=i4, device=dev), overflow=torch.empty(n, dtype=i4, device=dev))
        if want_list:
            out["nblist"] = torch.empty((n, self.cap), dtype=i4, device=dev)
        if n:
            ptr = lambda k: _vp(out[k].data_ptr()) if k in out else _vp()
            _check(self._lib.nb_get_block(self._ctx, int(n), *(ptr(k) for k in ("idx_act", "acc", "jerk", "pot", "nnb", "nblist",
                                                                          "overflow"))), "nb_get_block", self._ctx)
        return out

    # -- two-level Ahmad-Cohen stepping
    def ac_init(self, t_start: float, h2_all, eta_s: float, dt_max: float) -> int:
        """nb_ac_init -> number of overflowed lists (raises NbregError(NB_EOVERFLOW) if any)."""
        import torch
        n = ctypes.c_int32()
        rc = self._lib.nb_ac_init(self._ctx, float(t_start), _dev_ptr(h2_all, torch.float64, self.N, "h2_all"),
                                  float(eta_s), float(dt_max), ctypes.byref(n))
        _check(rc, "nb_ac_init", self._ctx)
        return n.value

    def ac_step(self, eta_I: float, eta_R: float, dt_max: float, t_stop: float = float("inf")):
        """nb_ac_step -> (t_next, n_irr, n_reg)."""
        t, ni, nr = ctypes.c_double(), ctypes.c_int32(), ctypes.c_int32()
        t_stop = min(float(t_stop), 1.7976931348623157e308)
        _check(self._lib.nb_ac_step(self._ctx, float(eta_I), float(eta_R), float(dt_max), t_stop, ctypes.byref(t),
                                    ctypes.byref(ni), ctypes.byref(nr)), "nb_ac_step", self._ctx)
        return t.value, ni.value, nr.value

    def ac_run(self, eta_I: float, eta_R: float, dt_max: float, t_stop: float = float("inf"), max_blocks: int = 1 << 62):
        """nb_ac_run -> (t_next, blocks, irregular_steps, regular_steps)."""
        t = ctypes.c_double()
        nb_, ni, nr = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64()
        t_stop = min(float(t_stop), 1.7976931348623157e308)
        _check(self._lib.nb_ac_run(self._ctx, float(eta_I), float(eta_R), float(dt_max), t_stop, int(max_blocks),
                                   ctypes.byref(t), ctypes.byref(nb_), ctypes.byref(ni), ctypes.byref(nr)), "nb_ac_run", self._ctx)
        return t.value, nb_.value, ni.value, nr.value

    def run_blocks(self, h2_all, eta: float, dt_max: float, t_stop: float = float("inf"), max_blocks: int = 1 << 62):
        """nb_run_blocks -> (t_next, blocks, particle_steps)."""
        import torch
        t = ctypes.c_double()
        nb_, ns = ctypes.c_int64(), ctypes.c_int64()
        h2 = _vp() if h2_all is None else _dev_ptr(h2_all, torch.float64, self.N, "h2_all")
        t_stop = min(float(t_stop), 1.7976931348623157e308)
        _check(self._lib.nb_run_blocks(self._ctx, h2, float(eta), float(dt_max), t_stop, int(max_blocks), ctypes.byref(t),
                                       ctypes.byref(nb_), ctypes.byref(ns)), "nb_run_blocks", self._ctx)
        return t.value, nb_.value, ns.value

    def ac_set_radii(self, idx, h2):
        """nb_ac_set_radii: new squared radii h2 for the bodies idx (int32 CUDA tensor), or for all N if idx is None."""
        import torch
        n = self.N if idx is None else int(idx.numel())
        _check(self._lib.nb_ac_set_radii(self._ctx, n, _vp() if idx is None else _dev_ptr(idx, torch.int32, n, "idx"),
                                         _dev_ptr(h2, torch.float64, n, "h2")), "nb_ac_set_radii", self._ctx)

    def ac_get_failed(self):
        """nb_ac_get_failed -> (idx, nnb): the regular steps of the block that returned NB_EOVERFLOW and the true size
        of each new list (empty tensors if the last step did not overflow)."""
        import torch
        n = ctypes.c_int32()
        _check(self._lib.nb_ac_get_failed(self._ctx, 0, ctypes.byref(n), _vp(), _vp()), "nb_ac_get_failed", self._ctx)
        idx = torch.empty(n.value, dtype=torch.int32, device="cuda")
        nnb = torch.empty(n.value, dtype=torch.int32, device="cuda")
        if n.value:
            _check(self._lib.nb_ac_get_failed(self._ctx, n.value, ctypes.byref(n), _vp(idx.data_ptr()), _vp(nnb.data_ptr())),
                   "nb_ac_get_failed", self._ctx)
        return idx, nnb

    def ac_get(self, with_lists: bool = False) -> dict:
        import torch
        N, f8, i4, dev = self.N, torch.float64, torch.int32, "cuda"
        out = dict(idx_act=torch.empty(N, dtype=i4, device=dev), idx_reg=torch.empty(N, dtype=i4, device=dev),
                   aI=torch.empty((N, 3), dtype=f8, device=dev), jI=torch.empty((N, 3), dtype=f8, device=dev),
                   aR=torch.empty((N, 3), dtype=f8, device=dev), jR=torch.empty((N, 3), dtype=f8, device=dev),
                   tR=torch.empty(N, dtype=f8, device=dev), dtR=torch.empty(N, dtype=f8, device=dev),
                   nnb=torch.empty(N, dtype=i4, device=dev))
        if with_lists:
            out["nblist"] = torch.empty((N, self.cap), dtype=i4, device=dev)
        ptr = lambda k: _vp(out[k].data_ptr()) if k in out else _vp()
        _check(self._lib.nb_ac_get(self._ctx, *(ptr(k) for k in ("idx_act", "idx_reg", "aI", "jI", "aR", "jR", "tR", "dtR",
                                                                  "nnb", "nblist"))), "nb_ac_get", self._ctx)
        return out

    def get_state(self, with_steps: bool = True):
        import torch
        N, kw = self.N, dict(dtype=torch.float64, device="cuda")
        st = dict(m=torch.empty(N, **kw), x0=torch.empty((N, 3), **kw), v0=torch.empty((N, 3), **kw),
                  a0=torch.empty((N, 3), **kw), j0=torch.empty((N, 3), **kw), t0=torch.empty(N, **kw))
        if with_steps:
            st["dt"] = torch.empty(N, **kw)
        args = [_vp(st[k].data_ptr()) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
        args.append(_vp(st["dt"].data_ptr()) if with_steps else _vp())
        _check(self._lib.nb_get_state(self._ctx, *args), "nb_get_state", self._ctx)
        return st

    # -- j-sharding
    def set_j_offset(self, j_offset: int):
        _check(self._lib.nb_set_j_offset(self._ctx, int(j_offset)), "nb_set_j_offset", self._ctx)

    def regular_shard(self, t: float, idx_i, istate, h2_i, acc, jerk, pot, nnb, nblist, overflow):
        """This shard's partial sums / local neighbours for a block given by GLOBAL indices and the active
        particles' gathered FP64 state istate[14][n_i]."""
        import torch
        n, f8, i4 = int(idx_i.numel()), torch.float64, torch.int32
        if n == 0:
            return
        args = [_dev_ptr(idx_i, i4, n, "idx_i"), _dev_ptr(istate, f8, 14 * n, "istate"), _dev_ptr(h2_i, f8, n, "h2_i"),
                _dev_ptr(acc, f8, 3 * n, "acc"), _dev_ptr(jerk, f8, 3 * n, "jerk"), _dev_ptr(pot, f8, n, "pot"),
                _dev_ptr(nnb, i4, n, "nnb"), _dev_ptr(nblist, i4, n * self.cap, "nblist"),
                _dev_ptr(overflow, i4, n, "overflow")]
        _check(self._lib.nb_regular_shard(self._ctx, float(t), n, *args), "nb_regular_shard", self._ctx)

    # -- the path (host buffers: numpy arrays or CPU tensors, pinned or not)
    def set_j_host(self, m, x0, v0, a0, j0, t0):
        import numpy as np
        N, f8 = self.N, np.float64
        args = [_host_ptr(m, f8, N, "m"), _host_ptr(x0, f8, 3 * N, "x0"), _host_ptr(v0, f8, 3 * N, "v0"),
                _host_ptr(a0, f8, 3 * N, "a0"), _host_ptr(j0, f8, 3 * N, "j0"), _host_ptr(t0, f8, N, "t0")]
        _check(self._lib.nb_set_j_host(self._ctx, *args), "nb_set_j_host", self._ctx)

    def regular_host(self, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow):
        import numpy as np
        n = int(idx_i.size if isinstance(idx_i, np.ndarray) else idx_i.numel())
        f8, i4 = np.float64, np.int32
        args = [_host_ptr(idx_i, i4, n, "idx_i"), _host_ptr(h2_i, f8, n, "h2_i"), _host_ptr(acc, f8, 3 * n, "acc"),
                _host_ptr(jerk, f8, 3 * n, "jerk"), _host_ptr(pot, f8, n, "pot"), _host_ptr(nnb, i4, n, "nnb"),
                _vp() if nblist is None else _host_ptr(nblist, i4, n * self.cap, "nblist"),
                _host_ptr(overflow, i4, n, "overflow")]
        _check(self._lib.nb_regular_host(self._ctx, n, *args), "nb_regular_host", self._ctx)

    def step_host(self, m, x0, v0, a0, j0, t0, t, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow):
        """nb_step_host: set_j + predict_all(t) + regular through host buffers, copies pipelined."""
        import numpy as np
        N, f8, i4 = self.N, np.float64, np.int32
        n = int(idx_i.size if isinstance(idx_i, np.ndarray) else idx_i.numel())
        jargs = [_host_ptr(m, f8, N, "m"), _host_ptr(x0, f8, 3 * N, "x0"), _host_ptr(v0, f8, 3 * N, "v0"),
                 _host_ptr(a0, f8, 3 * N, "a0"), _host_ptr(j0, f8, 3 * N, "j0"), _host_ptr(t0, f8, N, "t0")]
        if n == 0:
            oargs = [_vp()] * 8
        else:
            oargs = [_host_ptr(idx_i, i4, n, "idx_i"), _host_ptr(h2_i, f8, n, "h2_i"),
                     _host_ptr(acc, f8, 3 * n, "acc"), _host_ptr(jerk, f8, 3 * n, "jerk"),
                     _host_ptr(pot, f8, n, "pot"), _host_ptr(nnb, i4, n, "nnb"),
                     _vp() if nblist is None else _host_ptr(nblist, i4, n * self.cap, "nblist"),
                     _host_ptr(overflow, i4, n, "overflow")]
        _check(self._lib.nb_step_host(self._ctx, *jargs, float(t), n, *oargs), "nb_step_host", self._ctx)

    # -- convenience: allocate outputs with torch and run one block
    def regular_alloc(self, idx_i, h2_i):
        import torch
        n = int(idx_i.numel())
        dev = idx_i.device
        out = dict(acc=torch.empty((n, 3), dtype=torch.float64, device=dev),
                   jerk=torch.empty((n, 3), dtype=torch.float64, device=dev),
                   pot=torch.empty(n, dtype=torch.float64, device=dev),
                   nnb=torch.empty(n, dtype=torch.int32, device=dev),
                   nblist=torch.full((n, self.cap), -1, dtype=torch.int32, device=dev),
                   overflow=torch.empty(n, dtype=torch.int32, device=dev))
        self.regular(idx_i, h2_i, **out)
        return out


def nb_plan_regular(N: int, n_i: int, sm_count: int = 148, ctas_per_sm: int = 2) -> dict:
    """Pure host planning (no GPU needed): variant, i-block, j-splits, tiles per split."""
    lib = load_library()
    v = [ctypes.c_int32() for _ in range(4)]
    _check(lib.nb_plan_regular(N, n_i, sm_count, ctas_per_sm, *(ctypes.byref(x) for x in v)), "nb_plan_regular")
    return dict(variant=v[0].value, iblock=v[1].value, jsplit=v[2].value, tiles_per_split=v[3].value)


def nb_plan_chunks(N: int, chunks: int = 0) -> list[int]:
    """Pure host planning: body boundaries of the chunks nb_step_host sends the j-state in."""
    lib = load_library()
    fb = (ctypes.c_int64 * 9)()
    n = ctypes.c_int32()
    _check(lib.nb_plan_chunks(N, chunks, fb, ctypes.byref(n)), "nb_plan_chunks")
    return [fb[q] for q in range(n.value + 1)]


def nb_next_block_static(t0, dt, idx_act, block, stream=None):
    """nb_next_block_static: the next block's time and members from t0 and dt alone, for callers that cannot
    allocate GPU memory where they run (a plug-in under an application whose pool owns the device, a hook that must
    not stall other streams with cudaMalloc's device-wide synchronisation).  No context: t0, dt (float64 CUDA
    tensors [N]), idx_act (int32 CUDA tensor [N]) and block (float64 CUDA tensor [2] <- {t_next, n}) are the
    caller's; the working memory is a fixed array inside the library, so N <= NB_STATIC_MAX_N (NbregError with
    NB_ELIMIT beyond).  Enqueues on `stream` (a torch stream; None = the legacy default stream) and returns without
    synchronising.  Calls whose GPU work overlaps share that array and race: keep them on one stream."""
    import torch
    N = int(t0.numel())
    handle = _vp() if stream is None else _vp(stream.cuda_stream)
    rc = load_library().nb_next_block_static(N, _dev_ptr(t0, torch.float64, N, "t0"), _dev_ptr(dt, torch.float64, N, "dt"),
                                             _dev_ptr(idx_act, torch.int32, N, "idx_act"),
                                             _dev_ptr(block, torch.float64, 2, "block"), handle)
    _check(rc, "nb_next_block_static")


# Function-style aliases with the C names (north_star: nb_open / nb_set_j / nb_predict_all / nb_regular)
def nb_open(N: int, nb_cap: int, stream=None) -> NbContext:
    return NbContext(N, nb_cap, stream)


def nb_close(ctx: NbContext):
    ctx.close()


def nb_set_j(ctx: NbContext, m, x0, v0, a0, j0, t0):
    ctx.set_j(m, x0, v0, a0, j0, t0)


def nb_predict_all(ctx: NbContext, t: float):
    ctx.predict_all(t)


def nb_regular(ctx: NbContext, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow):
    ctx.regular(idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow)


def nb_update_j(ctx: NbContext, idx, m, x0, v0, a0, j0, t0):
    ctx.update_j(idx, m, x0, v0, a0, j0, t0)


def nb_irregular(ctx: NbContext, t: float, idx_i, nnb, nblist, acc, jerk, pot=None):
    ctx.irregular(t, idx_i, nnb, nblist, acc, jerk, pot)


def nb_step_host(ctx: NbContext, m, x0, v0, a0, j0, t0, t, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow):
    ctx.step_host(m, x0, v0, a0, j0, t0, t, idx_i, h2_i, acc, jerk, pot, nnb, nblist, overflow)


def nb_regular_all(ctx: NbContext, h2, acc, jerk, pot, nnb, nblist, overflow):
    ctx.regular_all(h2, acc, jerk, pot, nnb, nblist, overflow)
