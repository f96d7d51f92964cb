"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/nbreg.h declares; without a GPU the product path fails loudly (no fallback)."""
import ctypes

import numpy as np
import pytest


def test_library_builds_and_exports_every_declared_symbol():
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200.binding import declared_symbols
    decl = declared_symbols()
    assert {"nb_open", "nb_close", "nb_set_j", "nb_predict_all", "nb_regular", "nb_set_j_host",
            "nb_regular_host", "nb_strerror", "nb_set_stream"} <= set(decl)
    assert nb.exported_symbols() == decl
    lib = nb.load_library()
    assert lib.nb_strerror(0) == b"ok" and b"invalid" in lib.nb_strerror(1)


def test_argument_validation_without_compute():
    import paper_1504_03687_b200 as nb
    lib = nb.load_library()
    ctx = ctypes.c_void_p()
    assert lib.nb_open(0, 8, ctypes.byref(ctx)) == nb.NB_EINVAL and not ctx
    assert lib.nb_open(8, 0, ctypes.byref(ctx)) == nb.NB_EINVAL and not ctx
    assert lib.nb_open(8, 8, None) == nb.NB_EINVAL
    assert lib.nb_close(None) == nb.NB_EINVAL
    assert lib.nb_predict_all(None, 0.0) == nb.NB_EINVAL


def test_product_path_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_1504_03687_b200 as nb
    with pytest.raises(nb.NbregError) as e:
        nb.nb_open(1024, 64)
    assert e.value.code == nb.NB_ECUDA


def test_sass_is_blackwell_native():
    """The force kernel stages j-tiles with TMA bulk copies (UBLKCP) and mbarriers (SYNCS) and uses the
    SFU rsqrt (MUFU.RSQ); no tensor-core or FP64-convert instructions in its inner loop."""
    import subprocess
    from paper_1504_03687_b200.build import LIB, build_lib
    build_lib()
    sass = subprocess.run(["cuobjdump", "-sass", str(LIB)], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass and "SYNCS" in sass and "MUFU.RSQ" in sass
    assert "HMMA" not in sass and "sm_100a" in sass


def test_i_sharding_covers_block_exactly_once():
    import nbgen
    idx = np.arange(1000, dtype=np.int32)[::-1].copy()
    h2 = np.linspace(0, 1, 1000)
    for world in (1, 2, 3, 8):
        parts = [nbgen.shard_active_block(idx, h2, r, world) for r in range(world)]
        assert np.array_equal(np.concatenate([p[0] for p in parts]), idx)
        assert np.array_equal(np.concatenate([p[1] for p in parts]), h2)
        sizes = [p[0].size for p in parts]
        assert max(sizes) - min(sizes) <= 1
