"""CPU-side checks of the product library: it loads, exports every symbol include/gp_b200.h
declares, validates arguments without touching a GPU, and its static tile-task schedules (a6)
replay correctly against the device's dependency rules.  No compute calls: there is no GPU here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def gp():
    from paper_2602_19683_b200 import build
    build.build()
    from paper_2602_19683_b200 import binding
    binding.load()
    return binding


def test_exports_match_header(gp):
    hdr = open(os.path.join(ROOT, "include", "gp_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(gp_[a-z0-9_]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    lib = ctypes.CDLL(gp.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in gp_b200.h but not exported"
    assert declared == set(gp.EXPORTS), declared ^ set(gp.EXPORTS)


def test_no_library_linear_algebra_linked(gp):
    import subprocess
    out = subprocess.run(["ldd", gp.LIB_PATH], capture_output=True, text=True).stdout
    assert "cublas" not in out.lower() and "cusolver" not in out.lower(), out


def test_strerror_and_block_size(gp):
    assert gp.strerror(0) == "ok"
    for code in gp.ERR.values():
        assert gp.strerror(code) not in ("ok", "unknown error code")
    assert gp.gp_block_size(32) == 32 and gp.gp_block_size(64) == 64 and gp.gp_block_size(160) == 32
    assert gp.gp_block_size(256) == 128 and gp.gp_block_size(1024) == 128
    assert gp.gp_block_size(48) == gp.ERR["TILE"]


def test_workspace_sizes_and_argument_errors(gp):
    c, s, f = gp.gp_workspace_bytes(32768, 4096, 8, 1024)
    assert f >= 32768 * 4096 * 8                     # holds V^T (m x n)
    assert c < 64 << 20 and s < 64 << 20
    c0, s0, f0 = gp.gp_workspace_bytes(128, 0, 8, 32)
    assert f0 == 0 and c0 > 0 and s0 > 0
    for bad in ((100, 0, 8, 32), (128, 100, 8, 32), (128, 0, 8, 0), (128, 0, 8, 48)):
        with pytest.raises(gp.GpError) as e:
            gp.gp_workspace_bytes(*bad)
        assert e.value.code == gp.ERR["TILE"]
    with pytest.raises(gp.GpError) as e:
        gp.gp_workspace_bytes(0, 0, 8, 32)
    assert e.value.code == gp.ERR["SIZE"]
    total = gp.gp_pipeline_workspace_bytes(1024, 1024, 8, 256)
    assert total >= (10 * 256 * 256 + 1024 * 1024 + 1024 * 1024) * 8


def test_task_counts_match_paper_dag(gp):
    # M POTRF + M(M-1)/2 TRSM + M(M-1)/2 SYRK + M(M-1)(M-2)/6 GEMM
    for M, want in ((4, 20), (8, 120), (16, 816), (32, 5984)):
        tasks, items = gp.gp_cholesky_task_counts(M * 128, 128)
        assert tasks == want
        # a work item is a block-level piece of a tile task or (trailing updates) of up to 4 merged tile tasks
        assert items > 0 and 4 * items >= tasks


@pytest.mark.parametrize("n,m,tile", [
    (128, 0, 32), (128, 128, 32), (1024, 0, 256), (1024, 1024, 256), (1536, 384, 384), (320, 320, 160),
    (8192, 0, 512), (8192, 1024, 1024), (2048, 0, 2048), (4096, 1024, 128),
])
@pytest.mark.parametrize("workers", [1, 7, 148])
def test_schedule_is_a_valid_topological_order(gp, n, m, tile, workers):
    rc, st = gp.gp_schedule_selfcheck(n, m, tile, workers)
    assert rc == 0
    assert st["items"] > 0 and st["makespan_us"] >= st["critical_path_us"] * 0.999
    assert st["makespan_us"] >= st["work_us"] / workers * 0.999


@pytest.mark.parametrize("n,m,tile", [(128, 128, 32), (1024, 1024, 256), (1536, 384, 384), (8192, 1024, 1024), (4096, 1024, 128)])
def test_variance_only_schedule_is_a_valid_topological_order(gp, n, m, tile):
    rc, st = gp.gp_schedule_selfcheck_variance(n, m, tile, 148)
    rc_full, st_full = gp.gp_schedule_selfcheck(n, m, tile, 148)
    assert rc == 0 and rc_full == 0
    assert 0 < st["items"] < st_full["items"]          # the W = V^T V items are gone


def test_schedule_headline_config(gp):
    rc, st = gp.gp_schedule_selfcheck(32768, 0, 1024, 148)
    assert rc == 0
    # list-scheduling simulation must keep 148 workers busy: makespan within 10 % of work/148
    assert st["makespan_us"] <= 1.10 * st["work_us"] / 148


def test_schedule_fingerprint_is_stable_and_shape_dependent(gp):
    a = gp.gp_schedule_fingerprint(1024, 0, 256)
    assert a == gp.gp_schedule_fingerprint(1024, 0, 256) and a != 0
    assert a == gp.gp_schedule_fingerprint(1024, 0, 512)      # same blocks, same scheduling tile: the storage tile does not matter
    assert a != gp.gp_schedule_fingerprint(2048, 0, 256)
    assert a != gp.gp_schedule_fingerprint(1024, 1024, 256)
    assert gp.gp_schedule_fingerprint(1024, 1024, 256, with_sigma=True) != gp.gp_schedule_fingerprint(1024, 1024, 256, with_sigma=False)
    with pytest.raises(gp.GpError) as e:
        gp.gp_schedule_fingerprint(1000, 0, 256)
    assert e.value.code == gp.ERR["TILE"]


def test_schedule_granularity_auto_and_override(gp):
    # block edge: 64 up to n = 8192 (when the tile admits it), 128 beyond; independent of the storage tile
    assert gp.gp_block_size_for(1024, 256) == 64 and gp.gp_block_size_for(8192, 1024) == 64
    assert gp.gp_block_size_for(16384, 1024) == 128 and gp.gp_block_size_for(32768, 1024) == 128
    assert gp.gp_block_size_for(128, 32) == 32 and gp.gp_block_size_for(32768, 64) == 64 and gp.gp_block_size_for(320, 160) == 32
    # auto granularity: 1 scheduling block up to 96 block columns, then about 32 scheduling tiles per dimension
    assert gp.gp_schedule_granularity(1024, 1024, 256) == 1
    assert gp.gp_schedule_granularity(4096, 1024, 512) == 1
    assert gp.gp_schedule_granularity(8192, 1024, 512) == 4       # 128 block columns of 64
    assert gp.gp_schedule_granularity(32768, 4096, 1024) == 8
    assert gp.gp_schedule_granularity(65536, 8192, 2048) == 16
    assert gp.gp_schedule_granularity(32768, 0, 128) == 8        # independent of the storage tile
    try:
        gp.gp_set_block_edge(128)
        assert gp.gp_block_size_for(1024, 256) == 128 and gp.gp_block_size_for(1024, 64) == 64
        for g in (1, 2, 4, 8):
            gp.gp_set_schedule_granularity(g)
            assert gp.gp_schedule_granularity(8192, 1024, 512) == g
            for (n, m) in ((8192, 0), (8192, 1024)):
                rc, st = gp.gp_schedule_selfcheck(n, m, 512, 148)
                assert rc == 0 and st["items"] > 0
        gp.gp_set_schedule_granularity(3)                          # not a divisor of 64: the largest divisor below it
        assert gp.gp_schedule_granularity(8192, 1024, 512) == 2
        gp.gp_set_block_edge(32)
        assert gp.gp_block_size_for(32768, 1024) == 32
    finally:
        gp.gp_set_schedule_granularity(0)
        gp.gp_set_block_edge(0)
    with pytest.raises(gp.GpError):
        gp.gp_set_schedule_granularity(-1)
    with pytest.raises(gp.GpError):
        gp.gp_set_block_edge(48)


def test_prepare_validates_arguments_before_touching_the_device(gp):
    for bad, code in (((1000, 0, 256, 1), "TILE"), ((1024, 1000, 256, 2), "TILE"), ((1024, 0, 256, 2), "SIZE"),
                      ((1024, 0, 256, 0), "MODE"), ((1024, 0, 256, 8), "MODE"), ((0, 0, 256, 1), "SIZE")):
        with pytest.raises(gp.GpError) as e:
            gp.gp_prepare(*bad)
        assert e.value.code == gp.ERR[code], bad


def test_ncu_traffic_record_matches_the_schedule_the_library_builds(gp):
    """profiles/ncu_traffic.json must describe the CURRENT schedule, otherwise bench.py prints traffic = null."""
    import json
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        pytest.skip("no ncu traffic record committed yet")
    for key, rec in json.load(open(path)).items():
        n, tile = (int(x.split("=")[1]) for x in key.split(","))
        assert rec["schedule_fingerprint"] == "%016x" % gp.gp_schedule_fingerprint(n, 0, tile, 148), key
        assert rec["dram_bytes"] > 0 and rec["source"].startswith("profiles/")
        assert os.path.exists(os.path.join(ROOT, rec["source"].split(" ")[0]))


@pytest.mark.parametrize("n,tile", [(512, 128), (1024, 256), (4096, 1024), (32768, 1024)])
def test_panel_schedules_of_the_mixed_factorisation_replay(gp, n, tile):
    """gp_cholesky_tiled_mixed runs step J's FP64 half (POTRF + TRSM tile tasks) on blocks that already carry J versions."""
    M = n // tile
    for J in sorted({0, 1, M // 2, M - 1}):
        items = gp.gp_panel_schedule_selfcheck(n, tile, J)
        nbt = tile // 128
        # diagonal tile: POTRF + TRSM + update blocks; below it every block row is nbt solves and nbt - 1 in-tile updates
        want = nbt + nbt * (nbt - 1) // 2 + sum((nbt - kk) for jj in range(nbt) for kk in range(jj + 1, nbt)) + (M - J - 1) * nbt * (2 * nbt - 1)
        assert items == want, (J, items, want)
    assert gp.gp_panel_schedule_selfcheck(n, tile, M) == gp.ERR["SIZE"]
    assert gp.gp_mixed_workspace_bytes(n, tile) >= gp.gp_ozaki_planes() * n * n
    with pytest.raises(gp.GpError):
        gp.gp_mixed_workspace_bytes(n, 96)


def test_binding_refuses_cpu_tensors(gp):
    import torch
    X = torch.zeros(32, 2, dtype=torch.float64)
    with pytest.raises(ValueError):
        gp.gp_assemble_tiles(X, X, gp.Hyper(), 32, gp.GP_SYM_LOWER, torch.zeros(32 * 32, dtype=torch.float64))
