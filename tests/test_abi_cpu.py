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


def test_binding_keys_match_the_header_enum():
    """nb_get_info / nb_set_tuning keys: the binding's table carries the numbers include/nbreg.h defines."""
    import re
    from pathlib import Path
    from paper_1504_03687_b200.binding import INFO
    text = (Path(__file__).resolve().parent.parent / "include" / "nbreg.h").read_text()
    enum = {m.group(2).lower(): int(m.group(3)) for m in re.finditer(r"\b(NB_INFO|NB_TUNE)_([A-Z_]+)\s*=\s*(\d+)", text)}
    assert len(enum) >= 20
    for key, val in INFO.items():
        assert enum.get(key) == val, key
    assert set(enum) == set(INFO)


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


# ----------------------------------------------------------------------------- host logic: launch planning

def test_plan_regular_fills_the_chip_and_covers_the_j_range():
    """nb_plan_regular (pure host function of the library): the split covers every j-tile, pads the
    block as little as any variant can, and its modelled cost -- (waves + 0.13) x (tiles per split + per-CTA
    overhead) + finalize cost per split, DESIGN.md section 7 -- is within 1.5 % of the best over all splits,
    with no smaller split count inside that window."""
    import paper_1504_03687_b200 as nb
    sm, per_sm = 148, 2
    conc = sm * per_sm
    tile_us = lambda ib: ib * 256 / 3.6e9 * 1e6
    rate = {512: 1.0, 256: 1.01, 128: 1.025, 64: 1.03, 32: 1.11}     # cost per padded i-slot
    for N in (1024, 65536, 262144, 1048576, 1000003):
        ntiles = -(-N // 256)
        for n_i in (1, 32, 64, 100, 128, 257, 512, 1000, 4096, 8192, 65536, 131072):
            if n_i > N:
                continue
            p = nb.nb_plan_regular(N, n_i, sm, per_sm)
            ib, S, tps = p["iblock"], p["jsplit"], p["tiles_per_split"]
            assert ib == (512, 256, 128, 64, 32)[p["variant"]]
            pad = -(-n_i // ib) * ib
            assert abs(pad * rate[ib] - min(-(-n_i // b) * b * rate[b] for b in rate)) < 1e-9 * pad   # least rate-weighted padded work
            assert 1 <= S <= ntiles and tps == -(-ntiles // S) and (S - 1) * tps < ntiles <= S * tps
            n_ib = pad // ib

            def cost(s):
                t = -(-ntiles // s)
                seff = -(-ntiles // t)
                waves = -(-(n_ib * seff) // conc)
                return (waves + 0.13) * (t + 5.0 / tile_us(ib)) + 0.005 * seff / tile_us(ib)

            costs = {s: cost(s) for s in range(1, min(ntiles, 8192) + 1)}
            best = min(costs.values())
            assert costs[S] <= 1.0151 * best
            assert all(costs[s] > 1.0149 * best for s in range(1, S) if -(-ntiles // -(-ntiles // s)) != S)
    p = nb.nb_plan_regular(1048576, 8192, sm, per_sm)
    assert p["iblock"] == 512 and p["jsplit"] * (8192 // p["iblock"]) % conc == 0   # the headline block: whole waves
    assert nb.nb_plan_regular(1048576, 32)["iblock"] == 32 and nb.nb_plan_regular(1048576, 64)["iblock"] == 64
    assert nb.nb_plan_regular(1048576, 8256)["iblock"] == 64           # a ragged block takes the variant that pads least
    assert nb.nb_plan_regular(1048576, 131072)["iblock"] == 512
    with pytest.raises(nb.NbregError):
        nb.nb_plan_regular(1024, 2048)


def test_plan_chunks_partition_the_bodies_and_grow():
    import paper_1504_03687_b200 as nb
    for N in (1, 255, 10000, 131072, 140000, 600000, 1048576, 3000001):
        for want in (0, 1, 2, 3, 5, 8):
            b = nb.nb_plan_chunks(N, want)
            assert b[0] == 0 and b[-1] == N and all(x < y for x, y in zip(b, b[1:]))
            assert all(x % 256 == 0 for x in b[:-1])                   # whole j-tiles
            sizes = np.diff(b)
            assert len(sizes) <= 8 and (want == 0 or len(sizes) <= want)
            if len(sizes) > 2:       # first copy short, later ones double; the last takes the rounding remainder
                assert sizes[0] == sizes[1] and all(y == 2 * x for x, y in zip(sizes[1:-2], sizes[2:-1]))
                assert sizes[-1] <= 2 * sizes[-2] + 256 * 2 ** (len(sizes) - 1)
    assert nb.nb_plan_chunks(1048576) == [0, 65536, 131072, 262144, 524288, 1048576]
    assert nb.nb_plan_chunks(1048576, 1) == [0, 1048576]
