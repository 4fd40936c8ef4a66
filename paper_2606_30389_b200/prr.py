"""Thin ctypes binding over libprr.so (include/prr.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  Names mirror the C ABI.  torch is used for device
memory and streams.  There is no CPU fallback: a missing library raises at first use.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libprr.so")

OK, E_INVALID, E_UNSUPPORTED, E_STATE, E_CUDA, E_NOMEM = range(6)
DROP, RETAIN = 0, 1
OPT_PDL, OPT_CLUSTER, OPT_CUT, OPT_SUBTILE, OPT_KERNEL, OPT_PACE = 0, 1, 2, 3, 4, 5
OPT_SUMMARY = 6
SUMMARY_MEAN, SUMMARY_QUEST = 0, 1
OPT_LAST_CLUSTER, OPT_LAST_RING, OPT_LAST_GRID, OPT_LAST_KERNEL = 16, 17, 18, 19
KERNEL_AUTO, KERNEL_PERSISTENT, KERNEL_CLUSTER = 0, 1, 2
MODE_S3, MODE_S2, MODE_S1 = 0, 1, 2
FUSED, STREAMS = 0, 1
BF16, FP8_E4M3 = 0, 1

SYMBOLS = [
    "prr_create", "prr_destroy", "prr_last_error", "prr_version", "prr_build_summaries", "prr_append",
    "prr_set_ema_params", "prr_reset_ema", "prr_calibrate", "prr_predict", "prr_ema_update", "prr_score",
    "prr_set_mode", "prr_set_budget", "prr_get_budget", "prr_profile_budget", "prr_budget_fit", "prr_budget_for",
    "prr_topk", "prr_speculate", "prr_repair", "prr_attend", "prr_decode_step", "prr_step_append",
    "prr_decode_step_host",
    "prr_get_sets", "prr_get_scores", "prr_get_ema", "prr_get_stats", "prr_check", "prr_launch_count",
    "prr_timeline_enable", "prr_timeline_read", "prr_timeline_peek", "prr_set_option", "prr_get_option",
    "prr_graph_begin", "prr_graph_end", "prr_graph_launch", "prr_graph_destroy",
    "prr_static_scratch_bytes", "prr_attend_blocks_static", "prr_quantize_kv_fp8", "prr_set_kv_scales",
    "prr_set_budget_seq", "prr_get_budget_seq",
]


class Layout(C.Structure):
    _fields_ = [("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("max_batch", C.c_int32), ("max_blocks_per_seq", C.c_int32), ("n_layers", C.c_int32),
                ("kv_dtype", C.c_int32), ("overpredict_policy", C.c_int32), ("sm_scale", C.c_float),
                ("orchestration", C.c_int32)]


class PagedKV(C.Structure):
    _fields_ = [("k_pages", C.c_void_p), ("v_pages", C.c_void_p), ("block_table", C.c_void_p),
                ("seq_lens", C.c_void_p), ("batch", C.c_int32), ("layer", C.c_int32)]


class PrrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"prr error {code}: {msg}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Loads libprr.so (built by `python -m paper_2606_30389_b200.build`); raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_30389_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.prr_last_error.restype = C.c_char_p
        L.prr_last_error.argtypes = [C.c_void_p]
        L.prr_version.restype = C.c_char_p
        L.prr_launch_count.restype = C.c_int64
        L.prr_static_scratch_bytes.restype = C.c_int64
        L.prr_launch_count.argtypes = [C.c_void_p]
        L.prr_set_ema_params.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                         C.c_double, C.c_void_p]
        L.prr_decode_step_host.argtypes = [C.c_void_p, C.POINTER(PagedKV)] + [C.c_void_p] * 6  # (plain ints pass as is)
        L.prr_decode_step_host.restype = C.c_int32
        _lib = L
    return _lib


def _p(t) -> Optional[int]:
    """Device (or host) address of a tensor / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    assert t.is_contiguous(), "prr binding: tensors must be contiguous"
    return t.data_ptr()


def _stream(stream=None) -> int:
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


class Graph:
    def __init__(self, handle):
        self._h = handle

    def launch(self, stream=None):
        r = lib().prr_graph_launch(self._h, C.c_void_p(_stream(stream)))
        if r:
            raise PrrError(r, "prr_graph_launch failed")

    def destroy(self):
        if self._h:
            lib().prr_graph_destroy(self._h)
            self._h = None


class Context:
    """prr_ctx handle.  Methods take torch CUDA tensors with the layouts of include/prr.h."""

    def __init__(self, n_q_heads, n_kv_heads, head_dim, block_size, K, budget, max_batch=1,
                 max_blocks_per_seq=1, n_layers=1, policy=DROP, sm_scale=0.0, orchestration=FUSED, kv_dtype=BF16):
        self.layout = Layout(n_q_heads, n_kv_heads, head_dim, max_batch, max_blocks_per_seq, n_layers,
                             kv_dtype, policy, sm_scale, orchestration)
        self.block_size, self.K, self.budget = block_size, K, budget
        self._h = C.c_void_p()
        r = lib().prr_create(C.byref(self.layout), block_size, K, budget, C.byref(self._h))
        if r:
            raise PrrError(r, lib().prr_last_error(None).decode())

    # -- plumbing ---------------------------------------------------------------------------
    def _chk(self, r):
        if r:
            raise PrrError(r, lib().prr_last_error(self._h).decode())

    def destroy(self):
        if self._h:
            lib().prr_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @staticmethod
    def kv(k_pages, v_pages, block_table, seq_lens, layer=0) -> PagedKV:
        assert block_table.dtype == torch.int32 and seq_lens.dtype == torch.int32
        kv = PagedKV(_p(k_pages), _p(v_pages), _p(block_table), _p(seq_lens), seq_lens.shape[0], layer)
        kv._keep = (k_pages, v_pages, block_table, seq_lens)
        return kv

    # -- cache maintenance ------------------------------------------------------------------
    def build_summaries(self, kv, summaries, stream=None):
        self._chk(lib().prr_build_summaries(self._h, C.byref(kv), C.c_void_p(_p(summaries)),
                                            C.c_void_p(_stream(stream))))

    def append(self, kv, k_new, v_new, summaries, stream=None):
        self._chk(lib().prr_append(self._h, C.byref(kv), C.c_void_p(_p(k_new)), C.c_void_p(_p(v_new)),
                                   C.c_void_p(_p(summaries)), C.c_void_p(_stream(stream))))

    # -- predictor ---------------------------------------------------------------------------
    def set_ema_params(self, layer, seq, alpha, beta, gamma, stream=None):
        self._chk(lib().prr_set_ema_params(self._h, layer, seq, alpha, beta, gamma,
                                           C.c_void_p(_stream(stream))))

    def reset_ema(self, layer, stream=None):
        self._chk(lib().prr_reset_ema(self._h, layer, C.c_void_p(_stream(stream))))

    def calibrate(self, layer, seq, prefill_scores, n_valid=None, want_host=True, stream=None):
        """prefill_scores: fp32 [n_kv_heads, T, N].  Returns (theta*, H*, H_all[80]) if want_host."""
        assert prefill_scores.dtype == torch.float32 and prefill_scores.dim() == 3
        _, T, N = prefill_scores.shape
        th = (C.c_double * 3)()
        H = C.c_double()
        Ha = (C.c_double * 80)()
        self._chk(lib().prr_calibrate(self._h, layer, seq, C.c_void_p(_p(prefill_scores)), T, N,
                                      C.c_void_p(_p(n_valid)), th if want_host else None,
                                      C.byref(H) if want_host else None, Ha if want_host else None,
                                      C.c_void_p(_stream(stream))))
        return (tuple(th), H.value, list(Ha)) if want_host else None

    def predict(self, layer, batch, P_out, count_out=None, stream=None):
        self._chk(lib().prr_predict(self._h, layer, batch, C.c_void_p(_p(P_out)), C.c_void_p(_p(count_out)),
                                    C.c_void_p(_stream(stream))))

    def ema_update(self, layer, batch, scores, n_blocks, stream=None):
        self._chk(lib().prr_ema_update(self._h, layer, batch, C.c_void_p(_p(scores)),
                                       C.c_void_p(_p(n_blocks)), C.c_void_p(_stream(stream))))

    # -- selection ---------------------------------------------------------------------------
    def score(self, kv, q, summaries, scores_out, stream=None):
        self._chk(lib().prr_score(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(summaries)),
                                  C.c_void_p(_p(scores_out)), C.c_void_p(_stream(stream))))

    def topk(self, scores, n_blocks, batch, k, idx_out, count_out=None, stream=None):
        self._chk(lib().prr_topk(self._h, C.c_void_p(_p(scores)), C.c_void_p(_p(n_blocks)), batch, k,
                                 C.c_void_p(_p(idx_out)), C.c_void_p(_p(count_out)),
                                 C.c_void_p(_stream(stream))))

    # -- attention ---------------------------------------------------------------------------
    def speculate(self, kv, q, P, O_part, m_part, l_part, stream=None):
        self._chk(lib().prr_speculate(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(P)),
                                      C.c_void_p(_p(O_part)), C.c_void_p(_p(m_part)),
                                      C.c_void_p(_p(l_part)), C.c_void_p(_stream(stream))))

    def repair(self, kv, q, A, P, O_part, m_part, l_part, out, m_out=None, l_out=None, stream=None):
        self._chk(lib().prr_repair(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(A)),
                                   C.c_void_p(_p(P)), C.c_void_p(_p(O_part)), C.c_void_p(_p(m_part)),
                                   C.c_void_p(_p(l_part)), C.c_void_p(_p(out)), C.c_void_p(_p(m_out)),
                                   C.c_void_p(_p(l_out)), C.c_void_p(_stream(stream))))

    def set_budget_seq(self, layer, seq, budget, stream=None):
        self._chk(lib().prr_set_budget_seq(self._h, C.c_int32(layer), C.c_int32(seq), C.c_int32(budget), C.c_void_p(_stream(stream))))

    def get_budget_seq(self, layer, seq) -> int:
        v = C.c_int32()
        self._chk(lib().prr_get_budget_seq(self._h, C.c_int32(layer), C.c_int32(seq), C.byref(v)))
        return v.value

    def quantize_kv_fp8(self, kv, k8_pages, v8_pages, k_scale, v_scale, stream=None):
        self._chk(lib().prr_quantize_kv_fp8(self._h, C.byref(kv), C.c_void_p(_p(k8_pages)), C.c_void_p(_p(v8_pages)),
                                            C.c_void_p(_p(k_scale)), C.c_void_p(_p(v_scale)), C.c_void_p(_stream(stream))))

    def set_kv_scales(self, layer, k_scale, v_scale):
        self._keep_scales = getattr(self, "_keep_scales", {})
        self._keep_scales[layer] = (k_scale, v_scale)
        self._chk(lib().prr_set_kv_scales(self._h, C.c_int32(layer), C.c_void_p(_p(k_scale)), C.c_void_p(_p(v_scale))))

    def attend_blocks_static(self, kv, q, blocks, width, out, m_out=None, l_out=None, stream=None):
        """prr_attend_blocks_static: attention over given block lists; partial states in the library's static scratch."""
        self._chk(lib().prr_attend_blocks_static(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(blocks)),
                                                 C.c_int32(int(width)), C.c_void_p(_p(out)), C.c_void_p(_p(m_out)),
                                                 C.c_void_p(_p(l_out)), C.c_void_p(_stream(stream))))

    def attend(self, kv, q, summaries, out, stream=None):
        self._chk(lib().prr_attend(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(summaries)),
                                   C.c_void_p(_p(out)), C.c_void_p(_stream(stream))))

    def decode_step(self, kv, q, summaries, out, stream=None):
        self._chk(lib().prr_decode_step(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(summaries)),
                                        C.c_void_p(_p(out)), C.c_void_p(_stream(stream))))

    def step_append(self, kv, q, k_new, v_new, summaries, out, sequential=False, stream=None):
        """prr_append + prr_decode_step (or prr_attend) as one call: one launch when fused."""
        self._chk(lib().prr_step_append(self._h, C.byref(kv), C.c_void_p(_p(q)), C.c_void_p(_p(k_new)),
                                        C.c_void_p(_p(v_new)), C.c_void_p(_p(summaries)), C.c_void_p(_p(out)),
                                        C.c_int32(int(bool(sequential))), C.c_void_p(_stream(stream))))

    def decode_step_host(self, kv, q_host, k_new_host, v_new_host, summaries, out_host, stream=None):
        if type(q_host) is int and type(stream) is int:  # addresses taken by the caller: marshalling only
            r = lib().prr_decode_step_host(self._h, kv, q_host, k_new_host, v_new_host, summaries, out_host, stream)
            if r:
                self._chk(r)
            return
        self._chk(lib().prr_decode_step_host(self._h, C.byref(kv), _p(q_host), _p(k_new_host), _p(v_new_host),
                                             _p(summaries), _p(out_host), _stream(stream)))

    # -- introspection -----------------------------------------------------------------------
    def get_sets(self, layer, batch, A=None, P=None, M=None, counts=None, stream=None):
        self._chk(lib().prr_get_sets(self._h, layer, batch, C.c_void_p(_p(A)), C.c_void_p(_p(P)),
                                     C.c_void_p(_p(M)), C.c_void_p(_p(counts)), C.c_void_p(_stream(stream))))

    def get_scores(self, layer, batch, scores, stream=None):
        self._chk(lib().prr_get_scores(self._h, layer, batch, C.c_void_p(_p(scores)),
                                       C.c_void_p(_stream(stream))))

    def get_ema(self, layer, seq, level=None, trend=None, n_state=None, want_theta=False, stream=None):
        th = (C.c_double * 3)()
        self._chk(lib().prr_get_ema(self._h, layer, seq, C.c_void_p(_p(level)), C.c_void_p(_p(trend)),
                                    C.c_void_p(_p(n_state)), th if want_theta else None,
                                    C.c_void_p(_stream(stream))))
        return tuple(th) if want_theta else None

    def get_stats(self, reset=False, stream=None):
        """(sum|A|, sum|A n P|, sum|M|, sum|P|) since create / last reset."""
        st = (C.c_int64 * 4)()
        self._chk(lib().prr_get_stats(self._h, st, int(reset), C.c_void_p(_stream(stream))))
        return tuple(st)

    def check(self, stream=None):
        """Synchronises; raises if a fused step timed out on a dependency or a CUDA error is pending."""
        self._chk(lib().prr_check(self._h, C.c_void_p(_stream(stream))))

    def launch_count(self) -> int:
        return int(lib().prr_launch_count(self._h))

    def set_mode(self, mode: int, stream=None):
        self._chk(lib().prr_set_mode(self._h, int(mode), C.c_void_p(_stream(stream))))

    # -- profiling-guided budget ------------------------------------------------------------
    def set_budget(self, layer: int, budget: int, stream=None):
        self._chk(lib().prr_set_budget(self._h, int(layer), int(budget), C.c_void_p(_stream(stream))))

    def get_budget(self, layer: int) -> int:
        v = C.c_int32(0)
        self._chk(lib().prr_get_budget(self._h, int(layer), C.byref(v)))
        return int(v.value)

    def profile_budget(self, kv, q_traj, summaries, budgets, cold_l2=True, stream=None):
        """-> (us per step for each budget, us per step of the sequential path, best budget)."""
        n = len(budgets)
        b = (C.c_int32 * n)(*[int(x) for x in budgets])
        us = (C.c_float * n)()
        seq = C.c_float(0.0)
        best = C.c_int32(0)
        self._chk(lib().prr_profile_budget(self._h, C.byref(kv), C.c_void_p(_p(q_traj)), int(q_traj.shape[0]),
                                           C.c_void_p(_p(summaries)), b, n, int(bool(cold_l2)), us, C.byref(seq),
                                           C.byref(best), C.c_void_p(_stream(stream))))
        return list(us), float(seq.value), int(best.value)

    def budget_fit(self, ctx_lens, budgets, degree=2):
        n = len(ctx_lens)
        self._chk(lib().prr_budget_fit(self._h, n, (C.c_int32 * n)(*[int(x) for x in ctx_lens]),
                                       (C.c_int32 * n)(*[int(x) for x in budgets]), int(degree)))

    def budget_for(self, ctx_len: int) -> int:
        v = C.c_int32(0)
        self._chk(lib().prr_budget_for(self._h, int(ctx_len), C.byref(v)))
        return int(v.value)

    def set_option(self, option: int, value: int):
        self._chk(lib().prr_set_option(self._h, int(option), int(value)))

    def get_option(self, option: int) -> int:
        v = C.c_int32(0)
        self._chk(lib().prr_get_option(self._h, int(option), C.byref(v)))
        return int(v.value)

    def timeline_enable(self, on=True):
        self._chk(lib().prr_timeline_enable(self._h, int(on)))

    def timeline_read(self, max_warps=8192, stream=None):
        """uint64 numpy [n_warps, 16]: %globaltimer stamps (ns) of the last fused step's warps."""
        import numpy as np
        buf = np.zeros((max_warps, 16), dtype=np.uint64)
        n = C.c_int32(0)
        self._chk(lib().prr_timeline_read(self._h, buf.ctypes.data_as(C.c_void_p), max_warps, C.byref(n),
                                          C.c_void_p(_stream(stream))))
        return buf[:n.value]

    def timeline_peek(self, max_warps=8192):
        """timeline_read without synchronising (the stamps live in pinned host memory)."""
        import numpy as np
        buf = np.zeros((max_warps, 16), dtype=np.uint64)
        n = C.c_int32(0)
        self._chk(lib().prr_timeline_peek(self._h, buf.ctypes.data_as(C.c_void_p), max_warps, C.byref(n)))
        return buf[:n.value]

    # -- graphs ------------------------------------------------------------------------------
    def graph_begin(self, stream=None):
        self._chk(lib().prr_graph_begin(self._h, C.c_void_p(_stream(stream))))

    def graph_end(self, stream=None) -> Graph:
        g = C.c_void_p()
        self._chk(lib().prr_graph_end(self._h, C.c_void_p(_stream(stream)), C.byref(g)))
        return Graph(g)
