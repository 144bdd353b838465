"""Thin ctypes binding over libgp_b200.so (include/gp_b200.h): argument marshalling only.

Every step of the pipeline runs in the library's CUDA kernels; PyTorch supplies device
memory and the current stream.  There is NO CPU fallback: importing this module without the
built library, or calling it without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgp_b200.so")

GP_OK = 0
GP_SYM_LOWER, GP_GENERAL = 0, 1
ERR = {"NULL": -1, "SIZE": -2, "TILE": -3, "HYPER": -4, "WORKSPACE": -5, "CUDA": -6, "MODE": -7, "LIMIT": -8}

EXPORTS = ("gp_assemble_tiles", "gp_cholesky_tiled", "gp_solve", "gp_solve_noalloc", "gp_predict_mean", "gp_predict_full_cov",
           "gp_workspace_bytes", "gp_tiles_to_dense", "gp_cholesky_task_counts", "gp_release_cached_schedules",
           "gp_block_size", "gp_strerror", "gp_pipeline_workspace_bytes", "gp_pipeline_host", "gp_pipeline_mixed_workspace_bytes", "gp_pipeline_host_mixed", "gp_fp64_peak_launch", "gp_schedule_selfcheck", "gp_exec_stats",
           "gp_contraction_bench_launch", "gp_predict_variance", "gp_log_marginal_likelihood",
           "gp_schedule_selfcheck_variance", "gp_prepare", "gp_schedule_fingerprint",
           "gp_set_schedule_granularity", "gp_schedule_granularity", "gp_block_size_for", "gp_set_block_edge",
           "gp_ozaki_planes", "gp_ozaki_digit_bits", "gp_mixed_panel_bcast", "gp_predict_variance_mixed", "gp_int8_mma_peak_launch", "gp_ozaki_probe_launch", "gp_ozaki_probe_stamps", "gp_ozaki_plane_bytes", "gp_ozaki_slice", "gp_ozaki_contract",
           "gp_mixed_workspace_bytes", "gp_cholesky_tiled_mixed", "gp_panel_schedule_selfcheck",
           "gp_mixed_begin", "gp_mixed_update_column", "gp_mixed_panel", "gp_mixed_slice_column",
           "gp_predict_vt", "gp_cov_rows_workspace_bytes", "gp_predict_cov_rows", "gp_set_ozaki_tile_n",
           "gp_mixed_predict_workspace_bytes", "gp_predict_full_cov_mixed")


class gp_hyper(ctypes.Structure):
    _fields_ = [("lengthscale", ctypes.c_double), ("vertical", ctypes.c_double), ("noise", ctypes.c_double),
                ("ell_squared", ctypes.c_int)]


@dataclass(frozen=True)
class Hyper:
    lengthscale: float = 1.0
    vertical: float = 1.0
    noise: float = 0.1
    ell_squared: bool = False

    def c(self) -> gp_hyper:
        return gp_hyper(float(self.lengthscale), float(self.vertical), float(self.noise), int(bool(self.ell_squared)))


class GpError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {strerror(code)} ({code})")


_lib = None


def load() -> ctypes.CDLL:
    """Load the C-ABI library; fails loudly if it has not been built (python -m paper_2602_19683_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2602_19683_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, ci, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_size_t
    psz = ctypes.POINTER(ctypes.c_size_t)
    lib.gp_assemble_tiles.argtypes = [vp, i64, vp, i64, ci, gp_hyper, ci, ci, vp, vp]
    lib.gp_cholesky_tiled.argtypes = [vp, i64, ci, ci, vp, vp, sz, vp]
    lib.gp_solve.argtypes = [vp, i64, ci, vp, vp, vp, vp, sz, vp]
    lib.gp_solve_noalloc.argtypes = [vp, i64, ci, vp, vp, vp, vp]
    lib.gp_predict_mean.argtypes = [vp, i64, ci, vp, vp, i64, gp_hyper, vp, vp]
    lib.gp_predict_full_cov.argtypes = [vp, vp, i64, ci, vp, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_predict_variance.argtypes = [vp, vp, i64, ci, vp, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_log_marginal_likelihood.argtypes = [vp, i64, ci, vp, vp, vp, vp]
    lib.gp_predict_vt.argtypes = [vp, vp, i64, ci, vp, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_cov_rows_workspace_bytes.argtypes = [i64, i64, i64, ci, psz]
    lib.gp_predict_cov_rows.argtypes = [vp, vp, i64, i64, ci, i64, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_workspace_bytes.argtypes = [i64, i64, ci, ci, psz, psz, psz]
    lib.gp_tiles_to_dense.argtypes = [vp, i64, i64, ci, ci, vp, vp]
    lib.gp_cholesky_task_counts.argtypes = [i64, ci, ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.gp_release_cached_schedules.argtypes = []
    lib.gp_release_cached_schedules.restype = None
    lib.gp_block_size.argtypes = [ci]
    lib.gp_strerror.argtypes = [ci]
    lib.gp_pipeline_workspace_bytes.argtypes = [i64, i64, ci, ci, psz]
    lib.gp_pipeline_host.argtypes = [vp, vp, vp, i64, i64, ci, gp_hyper, ci, ci, vp, vp, vp, vp, vp, sz, vp]
    lib.gp_pipeline_host_mixed.argtypes = [vp, vp, vp, i64, i64, ci, gp_hyper, ci, ci, vp, vp, vp, vp, vp, sz, vp]
    lib.gp_pipeline_mixed_workspace_bytes.argtypes = [i64, i64, ci, ci, psz]
    lib.gp_schedule_selfcheck.argtypes = [i64, i64, ci, ci, ctypes.POINTER(ctypes.c_double)]
    lib.gp_schedule_selfcheck_variance.argtypes = [i64, i64, ci, ci, ctypes.POINTER(ctypes.c_double)]
    lib.gp_exec_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_uint64), ci, vp]
    lib.gp_fp64_peak_launch.argtypes = [ci, ci, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.gp_contraction_bench_launch.argtypes = [ci, ci, vp, sz, ctypes.POINTER(ctypes.c_double), psz, vp]
    lib.gp_prepare.argtypes = [i64, i64, ci, ci, ctypes.POINTER(ctypes.c_double)]
    lib.gp_schedule_fingerprint.argtypes = [i64, i64, ci, ci, ci, ctypes.POINTER(ctypes.c_uint64)]
    lib.gp_mixed_workspace_bytes.argtypes = [i64, ci, psz]
    lib.gp_cholesky_tiled_mixed.argtypes = [vp, i64, ci, ci, vp, vp, sz, vp]
    lib.gp_panel_schedule_selfcheck.argtypes = [i64, ci, ci]
    lib.gp_mixed_begin.argtypes = [vp, i64, ci, vp, vp, sz, vp]
    lib.gp_mixed_update_column.argtypes = [vp, i64, ci, ci, ci, ci, vp, sz, vp]
    lib.gp_mixed_panel.argtypes = [vp, i64, ci, ci, ci, vp, vp, sz, vp]
    lib.gp_mixed_slice_column.argtypes = [vp, i64, ci, ci, vp, sz, vp]
    lib.gp_mixed_panel_bcast.argtypes = [vp, i64, ci, ci, ci, vp, vp, sz, ctypes.POINTER(ctypes.c_void_p), ci, vp]
    lib.gp_ozaki_plane_bytes.argtypes = [i64, i64, psz]
    lib.gp_int8_mma_peak_launch.argtypes = [ci, ci, vp, ctypes.POINTER(ctypes.c_double), vp]
    lib.gp_ozaki_probe_launch.argtypes = [ci, vp, i64, vp, i64, i64, vp, i64, vp]
    lib.gp_ozaki_probe_stamps.argtypes = [ctypes.POINTER(ctypes.c_longlong)]
    lib.gp_set_ozaki_tile_n.argtypes = [ci]
    lib.gp_mixed_predict_workspace_bytes.argtypes = [i64, i64, ci, psz]
    lib.gp_predict_full_cov_mixed.argtypes = [vp, vp, i64, ci, vp, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_predict_variance_mixed.argtypes = [vp, vp, i64, ci, vp, i64, gp_hyper, ci, ci, vp, vp, sz, vp]
    lib.gp_ozaki_slice.argtypes = [vp, i64, i64, i64, ctypes.c_double, vp, vp, vp]
    lib.gp_ozaki_contract.argtypes = [vp, i64, vp, i64, i64, ctypes.c_double, ctypes.c_double, vp, i64, vp]
    lib.gp_block_size_for.argtypes = [i64, ci]
    lib.gp_set_block_edge.argtypes = [ci]
    lib.gp_set_schedule_granularity.argtypes = [ci]
    lib.gp_schedule_granularity.argtypes = [i64, i64, ci]
    lib.gp_strerror.restype = ctypes.c_char_p
    for name in EXPORTS:
        if name not in ("gp_release_cached_schedules", "gp_strerror"):
            getattr(lib, name).restype = ci
    _lib = lib
    return lib


def strerror(code: int) -> str:
    return load().gp_strerror(int(code)).decode()


def _check(rc: int, where: str) -> None:
    if rc != GP_OK:
        raise GpError(rc, where)


def _ptr(t: torch.Tensor | None, dtype=torch.float64):
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError("gp_b200 needs CUDA tensors (there is no CPU path)")
    if t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"expected a contiguous {dtype} tensor, got {t.dtype} contiguous={t.is_contiguous()}")
    return ctypes.c_void_p(t.data_ptr())


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def num_lower_tiles(n: int, tile: int) -> int:
    M = n // tile
    return M * (M + 1) // 2


def gp_block_size(tile: int) -> int:
    return int(load().gp_block_size(int(tile)))


def gp_workspace_bytes(n: int, m: int, D: int, tile: int):
    c, s, f = ctypes.c_size_t(0), ctypes.c_size_t(0), ctypes.c_size_t(0)
    _check(load().gp_workspace_bytes(n, m, D, tile, ctypes.byref(c), ctypes.byref(s), ctypes.byref(f)), "gp_workspace_bytes")
    return int(c.value), int(s.value), int(f.value)


def gp_cholesky_task_counts(n: int, tile: int):
    a, b = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(load().gp_cholesky_task_counts(n, tile, ctypes.byref(a), ctypes.byref(b)), "gp_cholesky_task_counts")
    return int(a.value), int(b.value)


def gp_assemble_tiles(A: torch.Tensor, B: torch.Tensor, h: Hyper, tile: int, mode: int, out: torch.Tensor) -> torch.Tensor:
    na, D = A.shape
    nb = B.shape[0]
    _check(load().gp_assemble_tiles(_ptr(A), na, _ptr(B), nb, D, h.c(), tile, mode, _ptr(out), _stream()), "gp_assemble_tiles")
    return out


def gp_cholesky_tiled(KL: torch.Tensor, n: int, tile: int, sched_width: int, info: torch.Tensor, work: torch.Tensor) -> None:
    _check(load().gp_cholesky_tiled(_ptr(KL), n, tile, sched_width, _ptr(info, torch.int32), _ptr(work, torch.uint8),
                                    work.numel(), _stream()), "gp_cholesky_tiled")


def gp_solve(L: torch.Tensor, n: int, tile: int, y: torch.Tensor, alpha: torch.Tensor, beta: torch.Tensor | None,
             work: torch.Tensor) -> None:
    _check(load().gp_solve(_ptr(L), n, tile, _ptr(y), _ptr(alpha), _ptr(beta), _ptr(work, torch.uint8), work.numel(), _stream()),
           "gp_solve")


def gp_solve_noalloc(L: torch.Tensor, n: int, tile: int, y: torch.Tensor, alpha: torch.Tensor, beta: torch.Tensor | None = None) -> None:
    """gp_solve on the library's static device scratch (n <= 8192): allocates nothing; calls that overlap on the GPU race."""
    _check(load().gp_solve_noalloc(_ptr(L), n, tile, _ptr(y), _ptr(alpha), _ptr(beta), _stream()), "gp_solve_noalloc")


def gp_predict_mean(X: torch.Tensor, alpha: torch.Tensor, Xs: torch.Tensor, h: Hyper, mean: torch.Tensor) -> None:
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_mean(_ptr(X), n, D, _ptr(alpha), _ptr(Xs), m, h.c(), _ptr(mean), _stream()), "gp_predict_mean")


def gp_predict_full_cov(L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, h: Hyper, tile: int, sched_width: int,
                        Sigma: torch.Tensor, work: torch.Tensor) -> None:
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_full_cov(_ptr(L), _ptr(X), n, D, _ptr(Xs), m, h.c(), tile, sched_width, _ptr(Sigma),
                                      _ptr(work, torch.uint8), work.numel(), _stream()), "gp_predict_full_cov")


def gp_predict_variance(L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, h: Hyper, tile: int, sched_width: int,
                        var: torch.Tensor, work: torch.Tensor) -> None:
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_variance(_ptr(L), _ptr(X), n, D, _ptr(Xs), m, h.c(), tile, sched_width, _ptr(var),
                                      _ptr(work, torch.uint8), work.numel(), _stream()), "gp_predict_variance")


def gp_predict_variance_mixed(L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, h: Hyper, tile: int, sched_width: int,
                              var: torch.Tensor, work: torch.Tensor) -> None:
    """gp_predict_variance with the V^T solve on the int8-emulated contraction (work: gp_mixed_predict_workspace_bytes)."""
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_variance_mixed(_ptr(L), _ptr(X), n, D, _ptr(Xs), m, h.c(), tile, sched_width, _ptr(var),
                                            _ptr(work, torch.uint8), work.numel(), _stream()), "gp_predict_variance_mixed")


def gp_predict_vt(L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, h: Hyper, tile: int, sched_width: int, Vt: torch.Tensor,
                  work: torch.Tensor) -> None:
    """Vt [m x n, GP_GENERAL tiles, flat] <- K_{X^,X} L^-T for the m test points of Xs."""
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_vt(_ptr(L), _ptr(X), n, D, _ptr(Xs), m, h.c(), tile, sched_width, _ptr(Vt), _ptr(work, torch.uint8),
                                work.numel(), _stream()), "gp_predict_vt")


def gp_predict_cov_rows(Vt_all: torch.Tensor, Xs_all: torch.Tensor, n: int, row0: int, rows: int, h: Hyper, tile: int, sched_width: int,
                        Sigma_rows: torch.Tensor, work: torch.Tensor) -> None:
    """Sigma_rows [rows x m] <- K_{X^_r,X^} - V_r^T (V^T)^T for the test points [row0, row0 + rows)."""
    m, D = Xs_all.shape
    need = ctypes.c_size_t(0)
    _check(load().gp_cov_rows_workspace_bytes(n, m, rows, tile, ctypes.byref(need)), "gp_cov_rows_workspace_bytes")
    if work.numel() < need.value:
        raise GpError(ERR["WORKSPACE"], "gp_predict_cov_rows")
    _check(load().gp_predict_cov_rows(_ptr(Vt_all), _ptr(Xs_all), n, m, D, row0, rows, h.c(), tile, sched_width, _ptr(Sigma_rows),
                                      _ptr(work, torch.uint8), work.numel(), _stream()), "gp_predict_cov_rows")


def gp_log_marginal_likelihood(L: torch.Tensor, n: int, tile: int, y: torch.Tensor, alpha: torch.Tensor, out: torch.Tensor) -> None:
    _check(load().gp_log_marginal_likelihood(_ptr(L), n, tile, _ptr(y), _ptr(alpha), _ptr(out), _stream()),
           "gp_log_marginal_likelihood")


def gp_tiles_to_dense(tiles: torch.Tensor, n: int, nb: int, tile: int, lower_packed: bool, dense: torch.Tensor) -> torch.Tensor:
    _check(load().gp_tiles_to_dense(_ptr(tiles), n, nb, tile, int(lower_packed), _ptr(dense), _stream()), "gp_tiles_to_dense")
    return dense


def gp_pipeline_workspace_bytes(n: int, m: int, D: int, tile: int) -> int:
    b = ctypes.c_size_t(0)
    _check(load().gp_pipeline_workspace_bytes(n, m, D, tile, ctypes.byref(b)), "gp_pipeline_workspace_bytes")
    return int(b.value)


def gp_pipeline_mixed_workspace_bytes(n: int, m: int, D: int, tile: int) -> int:
    b = ctypes.c_size_t(0)
    _check(load().gp_pipeline_mixed_workspace_bytes(n, m, D, tile, ctypes.byref(b)), "gp_pipeline_mixed_workspace_bytes")
    return int(b.value)


def _hptr(t: torch.Tensor | None, dtype=torch.float64):
    if t is None:
        return None
    if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise ValueError(f"expected a contiguous host {dtype} tensor")
    return ctypes.c_void_p(t.data_ptr())


def gp_pipeline_host(hX: torch.Tensor, hY: torch.Tensor, hXs: torch.Tensor, h: Hyper, tile: int, sched_width: int,
                     hMean: torch.Tensor, hSigma: torch.Tensor | None, hAlpha: torch.Tensor | None, work: torch.Tensor, mixed: bool = False) -> int:
    """HOST tensors in, HOST tensors out (pinned recommended); `work` is device scratch. Returns info.  mixed: the int8-emulated
    factorisation and covariance (gp_pipeline_host_mixed; `work` from gp_pipeline_mixed_workspace_bytes)."""
    n, D = hX.shape
    m = hXs.shape[0]
    info = ctypes.c_int(0)
    fn = load().gp_pipeline_host_mixed if mixed else load().gp_pipeline_host
    _check(fn(_hptr(hX), _hptr(hY), _hptr(hXs), n, m, D, h.c(), tile, sched_width, _hptr(hMean),
                                   _hptr(hSigma), _hptr(hAlpha), ctypes.byref(info), _ptr(work, torch.uint8), work.numel(),
                                   _stream()), "gp_pipeline_host")
    return int(info.value)


def gp_fp64_peak_launch(mode: int, iters: int, sink: torch.Tensor) -> float:
    """Enqueue one FP64 peak microbenchmark launch (0 = DMMA, 1 = DFMA); returns its flop count."""
    f = ctypes.c_double(0.0)
    _check(load().gp_fp64_peak_launch(mode, iters, _ptr(sink), ctypes.byref(f), _stream()), "gp_fp64_peak_launch")
    return float(f.value)


def gp_contraction_bench_bytes(K: int, reps: int) -> int:
    need = ctypes.c_size_t(0)
    _check(load().gp_contraction_bench_launch(K, reps, None, 0, None, ctypes.byref(need), None), "gp_contraction_bench_launch")
    return int(need.value)


def gp_contraction_bench_launch(K: int, reps: int, buf: torch.Tensor) -> float:
    """Enqueue one launch of the contraction steady-state microbenchmark; returns its flop count."""
    f = ctypes.c_double(0.0)
    _check(load().gp_contraction_bench_launch(K, reps, _ptr(buf, torch.uint8), buf.numel(), ctypes.byref(f), None, _stream()),
           "gp_contraction_bench_launch")
    return float(f.value)


def gp_schedule_selfcheck(n: int, m: int, tile: int, workers: int = 148):
    """(rc, stats) of the host-only schedule replay; stats = items, edges, makespan_us, work_us, critical_path_us."""
    st = (ctypes.c_double * 5)()
    rc = int(load().gp_schedule_selfcheck(n, m, tile, workers, st))
    return rc, dict(zip(("items", "edges", "makespan_us", "work_us", "critical_path_us"), list(st)))


def gp_schedule_selfcheck_variance(n: int, m: int, tile: int, workers: int = 148):
    st = (ctypes.c_double * 5)()
    rc = int(load().gp_schedule_selfcheck_variance(n, m, tile, workers, st))
    return rc, dict(zip(("items", "edges", "makespan_us", "work_us", "critical_path_us"), list(st)))


def gp_exec_stats(work: torch.Tensor, max_workers: int = 148):
    """Per-worker (producer_poll_cycles, total_cycles, items, sm_id, consumer_job_wait_cycles, 0, jobs, 0) of the
    last executor launch that used `work`."""
    buf = (ctypes.c_uint64 * (8 * max_workers))()
    w = int(load().gp_exec_stats(_ptr(work, torch.uint8), buf, max_workers, _stream()))
    if w < 0:
        raise GpError(w, "gp_exec_stats")
    return [tuple(buf[8 * i:8 * i + 8]) for i in range(w)]


GP_PREPARE_CHOLESKY, GP_PREPARE_FULL_COV, GP_PREPARE_VARIANCE = 1, 2, 4


def gp_prepare(n: int, m: int, tile: int, what: int = GP_PREPARE_CHOLESKY | GP_PREPARE_FULL_COV) -> float:
    """Build + upload the schedules for this shape on the current device; returns the host time in ms."""
    ms = ctypes.c_double(0.0)
    _check(load().gp_prepare(n, m, tile, what, ctypes.byref(ms)), "gp_prepare")
    return float(ms.value)


def gp_schedule_fingerprint(n: int, m: int, tile: int, workers: int = 148, with_sigma: bool = True) -> int:
    fp = ctypes.c_uint64(0)
    _check(load().gp_schedule_fingerprint(n, m, tile, workers, int(with_sigma), ctypes.byref(fp)), "gp_schedule_fingerprint")
    return int(fp.value)


def gp_mixed_workspace_bytes(n: int, tile: int) -> int:
    b = ctypes.c_size_t(0)
    _check(load().gp_mixed_workspace_bytes(n, tile, ctypes.byref(b)), "gp_mixed_workspace_bytes")
    return int(b.value)


def gp_cholesky_tiled_mixed(KL: torch.Tensor, n: int, tile: int, sched_width: int, info: torch.Tensor, work: torch.Tensor) -> None:
    """gp_cholesky_tiled with the trailing updates emulated on the int8 tensor cores (opt-in)."""
    _check(load().gp_cholesky_tiled_mixed(_ptr(KL), n, tile, sched_width, _ptr(info, torch.int32), _ptr(work, torch.uint8),
                                          work.numel(), _stream()), "gp_cholesky_tiled_mixed")


def gp_mixed_begin(KL: torch.Tensor, n: int, tile: int, info: torch.Tensor, work: torch.Tensor) -> None:
    _check(load().gp_mixed_begin(_ptr(KL), n, tile, _ptr(info, torch.int32), _ptr(work, torch.uint8), work.numel(), _stream()), "gp_mixed_begin")


def gp_mixed_update_column(KL: torch.Tensor, n: int, tile: int, J: int, k0: int, k1: int, work: torch.Tensor) -> None:
    _check(load().gp_mixed_update_column(_ptr(KL), n, tile, J, k0, k1, _ptr(work, torch.uint8), work.numel(), _stream()),
           "gp_mixed_update_column")


def gp_mixed_panel(KL: torch.Tensor, n: int, tile: int, J: int, sched_width: int, info: torch.Tensor, work: torch.Tensor) -> None:
    _check(load().gp_mixed_panel(_ptr(KL), n, tile, J, sched_width, _ptr(info, torch.int32), _ptr(work, torch.uint8), work.numel(),
                                 _stream()), "gp_mixed_panel")


def gp_mixed_panel_bcast(KL: torch.Tensor, n: int, tile: int, J: int, sched_width: int, info: torch.Tensor, work: torch.Tensor, peers) -> None:
    """gp_mixed_panel whose finished blocks are also stored into the other ranks' copies of the tile array: `peers` = their
    device addresses as seen from this GPU (ints; at most 7)."""
    arr = (ctypes.c_void_p * max(len(peers), 1))(*[ctypes.c_void_p(int(a)) for a in peers])
    _check(load().gp_mixed_panel_bcast(_ptr(KL), n, tile, J, sched_width, _ptr(info, torch.int32), _ptr(work, torch.uint8), work.numel(),
                                       arr, len(peers), _stream()), "gp_mixed_panel_bcast")


def gp_mixed_slice_column(KL: torch.Tensor, n: int, tile: int, J: int, work: torch.Tensor) -> None:
    _check(load().gp_mixed_slice_column(_ptr(KL), n, tile, J, _ptr(work, torch.uint8), work.numel(), _stream()), "gp_mixed_slice_column")


def gp_panel_schedule_selfcheck(n: int, tile: int, J: int) -> int:
    return int(load().gp_panel_schedule_selfcheck(n, tile, J))


def gp_mixed_predict_workspace_bytes(n: int, m: int, tile: int) -> int:
    b = ctypes.c_size_t(0)
    _check(load().gp_mixed_predict_workspace_bytes(n, m, tile, ctypes.byref(b)), "gp_mixed_predict_workspace_bytes")
    return int(b.value)


def gp_predict_full_cov_mixed(L: torch.Tensor, X: torch.Tensor, Xs: torch.Tensor, h: Hyper, tile: int, sched_width: int,
                              Sigma: torch.Tensor, work: torch.Tensor) -> None:
    n, D = X.shape
    m = Xs.shape[0]
    _check(load().gp_predict_full_cov_mixed(_ptr(L), _ptr(X), n, D, _ptr(Xs), m, h.c(), tile, sched_width, _ptr(Sigma),
                                            _ptr(work, torch.uint8), work.numel(), _stream()), "gp_predict_full_cov_mixed")


def gp_int8_mma_peak_launch(n_cols: int, iters: int, cycles: torch.Tensor) -> float:
    """Enqueue the bare tcgen05.mma kind::i8 issue loop (128 x n_cols x 32) on every SM; returns its int8 operation count."""
    ops = ctypes.c_double(0.0)
    _check(load().gp_int8_mma_peak_launch(int(n_cols), int(iters), _ptr(cycles, torch.int64), ctypes.byref(ops), _stream()), "gp_int8_mma_peak_launch")
    return float(ops.value)


def gp_ozaki_probe_launch(probe: int, Aplanes: torch.Tensor, Bplanes: torch.Tensor, C: torch.Tensor) -> None:
    _, ma, k = Aplanes.shape
    _, nb, _ = Bplanes.shape
    _check(load().gp_ozaki_probe_launch(int(probe), _ptr(Aplanes, torch.int8), ma, _ptr(Bplanes, torch.int8), nb, k, _ptr(C), nb, _stream()),
           "gp_ozaki_probe_launch")


def gp_ozaki_probe_stamps():
    buf = (ctypes.c_longlong * 8)()
    _check(load().gp_ozaki_probe_stamps(buf), "gp_ozaki_probe_stamps")
    return list(buf)


def gp_ozaki_planes() -> int:
    return int(load().gp_ozaki_planes())


def gp_ozaki_digit_bits() -> int:
    return int(load().gp_ozaki_digit_bits())


def gp_set_ozaki_tile_n(n: int) -> None:
    _check(load().gp_set_ozaki_tile_n(int(n)), "gp_set_ozaki_tile_n")


def gp_ozaki_slice(X: torch.Tensor, scale: float) -> torch.Tensor:
    """FP64 [rows, k] (row-major, contiguous) -> int8 digit planes [8, rows, k]; raises if an entry exceeds scale / 2."""
    rows, k = X.shape
    need = ctypes.c_size_t(0)
    _check(load().gp_ozaki_plane_bytes(rows, k, ctypes.byref(need)), "gp_ozaki_plane_bytes")
    planes = torch.empty(int(need.value), dtype=torch.int8, device=X.device)
    overflow = torch.zeros(1, dtype=torch.int32, device=X.device)
    _check(load().gp_ozaki_slice(_ptr(X), rows, k, k, float(scale), _ptr(planes, torch.int8), _ptr(overflow, torch.int32), _stream()),
           "gp_ozaki_slice")
    if int(overflow.item()) != 0:
        raise ValueError("gp_ozaki_slice: an entry exceeds scale / 2")
    return planes.view(int(load().gp_ozaki_planes()), rows, k)


def gp_ozaki_contract(Aplanes: torch.Tensor, Bplanes: torch.Tensor, scaleA: float, scaleB: float, C: torch.Tensor) -> None:
    """C [ma, nb] (FP64, contiguous) -= A B^T from the digit planes of A [ma, k] and B [nb, k]."""
    _, ma, k = Aplanes.shape
    _, nb, kb = Bplanes.shape
    assert k == kb and C.shape == (ma, nb)
    _check(load().gp_ozaki_contract(_ptr(Aplanes, torch.int8), ma, _ptr(Bplanes, torch.int8), nb, k, float(scaleA), float(scaleB),
                                    _ptr(C), nb, _stream()), "gp_ozaki_contract")


def gp_block_size_for(n: int, tile: int) -> int:
    return int(load().gp_block_size_for(int(n), int(tile)))


def gp_set_block_edge(b: int) -> None:
    """Override the cap on the block edge (0 = auto, 32, 64, 128); call before allocating workspaces."""
    _check(load().gp_set_block_edge(int(b)), "gp_set_block_edge")


def gp_set_schedule_granularity(blocks: int) -> None:
    """Override the scheduling-tile edge in blocks for later calls (0 = auto); measurement support."""
    _check(load().gp_set_schedule_granularity(int(blocks)), "gp_set_schedule_granularity")


def gp_schedule_granularity(n: int, m: int, tile: int) -> int:
    g = int(load().gp_schedule_granularity(n, m, tile))
    if g < 0:
        raise GpError(g, "gp_schedule_granularity")
    return g


def gp_release_cached_schedules() -> None:
    load().gp_release_cached_schedules()


# ------------------------------------------------------------------------------------------------
# Convenience driver: the whole pipeline of PAPER.md section 4.1 on device tensors (allocation and
# call sequencing only).
# ------------------------------------------------------------------------------------------------
@dataclass
class GpResult:
    L_tiles: torch.Tensor
    alpha: torch.Tensor
    beta: torch.Tensor
    info: torch.Tensor
    mean: torch.Tensor | None = None
    Sigma: torch.Tensor | None = None


class GpPipeline:
    """Pre-allocates every device buffer for one (n, m, D, tile) shape so that run() only launches."""

    def __init__(self, n: int, m: int, D: int, tile: int, h: Hyper, sched_width: int = 0, device="cuda"):
        self.n, self.m, self.D, self.tile, self.h, self.width = n, m, D, tile, h, sched_width
        dev = torch.device(device)
        cb, sb, fb = gp_workspace_bytes(n, m, D, tile)
        self.KL = torch.empty(num_lower_tiles(n, tile) * tile * tile, dtype=torch.float64, device=dev)
        self.work = torch.empty(max(cb, sb, fb), dtype=torch.uint8, device=dev)
        self.info = torch.zeros(1, dtype=torch.int32, device=dev)
        self.alpha = torch.empty(n, dtype=torch.float64, device=dev)
        self.beta = torch.empty(n, dtype=torch.float64, device=dev)
        self.mean = torch.empty(m, dtype=torch.float64, device=dev) if m > 0 else None
        self.Sigma = torch.empty(m, m, dtype=torch.float64, device=dev) if m > 0 else None

    def assemble(self, X):
        gp_assemble_tiles(X, X, self.h, self.tile, GP_SYM_LOWER, self.KL)

    def cholesky(self):
        gp_cholesky_tiled(self.KL, self.n, self.tile, self.width, self.info, self.work)

    def solve(self, y):
        gp_solve(self.KL, self.n, self.tile, y, self.alpha, self.beta, self.work)

    def predict(self, X, Xs, full_cov=True):
        gp_predict_mean(X, self.alpha, Xs, self.h, self.mean)
        if full_cov:
            gp_predict_full_cov(self.KL, X, Xs, self.h, self.tile, self.width, self.Sigma, self.work)

    def run(self, X, y, Xs, full_cov=True) -> GpResult:
        self.assemble(X)
        self.cholesky()
        self.solve(y)
        self.predict(X, Xs, full_cov)
        return GpResult(self.KL, self.alpha, self.beta, self.info, self.mean, self.Sigma if full_cov else None)

    def dense_L(self) -> torch.Tensor:
        out = torch.empty(self.n, self.n, dtype=torch.float64, device=self.KL.device)
        return gp_tiles_to_dense(self.KL, self.n, self.n, self.tile, True, out)
